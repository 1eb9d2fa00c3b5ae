// sso_inst.cu -- explicit instantiations of the pass kernel for one (precision, line length).
// Compiled once per pair with -DSSO_T=<float|double> -DSSO_TNAME=<f32|f64> -DSSO_N=<n>
// (see paper_1012_3911_b200/build.py); each object exports one lookup function that the
// dispatcher in sso_api.cu calls.
#include <atomic>

#include "sso_pass.cuh"
#include "sso_ring.cuh"
#include "sso_sring.cuh"
#include "sso_line1d.cuh"
#include "sso_line1d_cluster.cuh"
#include "sso_dispatch.h"

#ifndef SSO_T
#error "compile with -DSSO_T=float|double -DSSO_TNAME=f32|f64 -DSSO_N=<line length>"
#endif

namespace sso {

// cudaFuncSetAttribute is per device: opt a kernel in to large dynamic shared memory once per device (bit d of
// `done` = device d; devices beyond 63 repeat the call, which is harmless)
template <typename K> static cudaError_t opt_in_smem(K kern, std::atomic<unsigned long long> &done, int *dev_out = nullptr, int *sms_out = nullptr) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev_out) *dev_out = dev;
    const unsigned long long bit = dev < 64 ? 1ull << dev : 0ull;
    if (!(done.load(std::memory_order_acquire) & bit) || sms_out) {
        int optin = 0, sms = 0;
        if ((e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev)) != cudaSuccess) return e;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if (sms_out) *sms_out = sms;
        if (!(done.load(std::memory_order_acquire) & bit)) {
            if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, optin)) != cudaSuccess) return e;
            done.fetch_or(bit, std::memory_order_release);
        }
    }
    return cudaSuccess;
}

template <typename T, int N, bool STRIDED, int PW, int SIGN>
cudaError_t launch_pass(const PassArgs &a, unsigned threads, size_t smem, cudaStream_t st) {
    auto kern = pass_kernel<T, N, STRIDED, PW, SIGN>;
    static std::atomic<unsigned long long> done{0};
    int dev = 0;
    cudaError_t e = opt_in_smem(kern, done, &dev);
    if (e != cudaSuccess) return e;
    // one wave of persistent CTAs: resident CTAs per SM for this block shape x SM count of the current device
    // (asked once per device and block shape of this instantiation; the last answer is kept)
    struct Occ { int dev; unsigned threads; size_t smem; int occ, sms; };
    static thread_local Occ last{-1, 0u, 0, 0, 0};
    if (last.dev != dev || last.threads != threads || last.smem != smem) {
        int occ = 0, sms = 0;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, (int)threads, smem)) != cudaSuccess) return e;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        last = Occ{dev, threads, smem, occ, sms};
    }
    const int occ = last.occ, num_sms = last.sms;
    if (occ < 1) return cudaErrorLaunchOutOfResources;
    long long grid = (long long)occ * num_sms;
    const long long need = ((long long)a.ntiles + a.G - 1) / a.G;
    if (grid > need) grid = need;
    kern<<<(unsigned)grid, threads, smem, st>>>(a);
    return cudaGetLastError();
}

// Programmatic dependent launch: the CTAs of a pass may start (twiddle copy, barrier setup) while the previous
// pass of the stream drains; they wait in the kernel (griddepcontrol.wait) before touching psi.
template <typename K, typename... Args>
static cudaError_t launch_pdl(K kern, unsigned grid, unsigned threads, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, args...);
}

template <typename T, int N, int MODE, int SIGN, int MAXT>
cudaError_t launch_ring(const RingArgs &a, unsigned threads, size_t smem, unsigned grid, cudaStream_t st) {
    auto kern = ring_kernel<T, N, MODE, SIGN, MAXT>;
    static std::atomic<unsigned long long> done{0};
    cudaError_t e = opt_in_smem(kern, done);
    if (e != cudaSuccess) return e;
    if (threads > (unsigned)MAXT) return cudaErrorInvalidConfiguration;
    return launch_pdl(kern, grid, threads, smem, st, a);
}

template <typename T, int N, int SMODE>
cudaError_t launch_sring(const SRingArgs &a, const void *tensor_map, unsigned threads, size_t smem, unsigned grid, cudaStream_t st) {
    auto kern = sring_kernel<T, N, SMODE>;
    static std::atomic<unsigned long long> done{0};
    cudaError_t e = opt_in_smem(kern, done);
    if (e != cudaSuccess) return e;
    if (threads > 512u) return cudaErrorInvalidConfiguration;
    return launch_pdl(kern, grid, threads, smem, st, a, *reinterpret_cast<const CUtensorMap *>(tensor_map));
}

template <typename T, int N> cudaError_t launch_line1d(const Line1dArgs &a, size_t smem, cudaStream_t st) {
    auto kern = line1d_kernel<T, N>;
    static std::atomic<unsigned long long> done{0};
    cudaError_t e = opt_in_smem(kern, done);
    if (e != cudaSuccess) return e;
    kern<<<1, N / 16, smem, st>>>(a);
    return cudaGetLastError();
}

// one cluster of CS CTAs holds the line; CS is a launch attribute (8 is the largest portable cluster size)
template <typename T, int M, int CS> cudaError_t launch_line1d_cluster(const Line1dClusterArgs &a, size_t smem, cudaStream_t st) {
    auto kern = line1d_cluster_kernel<T, M, CS>;
    static std::atomic<unsigned long long> done{0};
    cudaError_t e = opt_in_smem(kern, done);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(CS);
    cfg.blockDim = dim3(M / 16);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = CS;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    if (!a.psi) {  // query only (sso_api.cu, cluster_size_for): can the current device hold one such cluster at all?
        int nclusters = 0;
        if ((e = cudaOccupancyMaxActiveClusters(&nclusters, kern, &cfg)) != cudaSuccess) return e;
        return nclusters >= 1 ? cudaSuccess : cudaErrorLaunchOutOfResources;
    }
    return cudaLaunchKernelEx(&cfg, kern, a);
}

#define SSO_CAT3_(a, b, c) a##b##_##c
#define SSO_CAT3(a, b, c) SSO_CAT3_(a, b, c)

#define SSO_CAT4_(a, b, c) a##b##_##c
#define SSO_CAT4(a, b, c) SSO_CAT4_(a, b, c)
// lines beyond 4096 points (one 512-thread group, twiddles read from global memory for complex128) run on the
// contiguous-axis ring and the direct kernel only: no strided tile of theirs fits a ring buffer, and the 1D
// register-resident kernels hold at most 4096 points per CTA
#if defined(SSO_STUB) || SSO_N > 4096
SRingLaunchFn SSO_CAT4(sso_sring_lookup_, SSO_TNAME, SSO_N)(int) { return nullptr; }
#else
SRingLaunchFn SSO_CAT4(sso_sring_lookup_, SSO_TNAME, SSO_N)(int mode) {
    using T = SSO_T;
    constexpr int N = SSO_N;
    if (mode == SMODE_KS) return &launch_sring<T, N, SMODE_KS>;
    if (mode == SMODE_KD2) return &launch_sring<T, N, SMODE_KD2>;
    if (mode == SMODE_KD4) return &launch_sring<T, N, SMODE_KD4>;
    if (mode == SMODE_KD2F) return &launch_sring<T, N, SMODE_KD2F>;
    if (mode == SMODE_KD4F) return &launch_sring<T, N, SMODE_KD4F>;
    if (mode == SMODE_DIF) return &launch_sring<T, N, SMODE_DIF>;
    if (mode == SMODE_DIT) return &launch_sring<T, N, SMODE_DIT>;
    return nullptr;
}
#endif

#if defined(SSO_STUB) || SSO_N > 4096
Line1dLaunchFn SSO_CAT4(sso_line1d_lookup_, SSO_TNAME, SSO_N)() { return nullptr; }
#else
Line1dLaunchFn SSO_CAT4(sso_line1d_lookup_, SSO_TNAME, SSO_N)() { return &launch_line1d<SSO_T, SSO_N>; }
#endif

#if defined(SSO_STUB) || SSO_N < 512 || SSO_N > 4096
Line1dClusterLaunchFn SSO_CAT4(sso_line1d_cluster_lookup_, SSO_TNAME, SSO_N)(int) { return nullptr; }
#else
Line1dClusterLaunchFn SSO_CAT4(sso_line1d_cluster_lookup_, SSO_TNAME, SSO_N)(int cs) {
    if (cs == 4) return &launch_line1d_cluster<SSO_T, SSO_N, 4>;
    if (cs == 8) return &launch_line1d_cluster<SSO_T, SSO_N, 8>;
    return nullptr;
}
#endif

#ifdef SSO_STUB
RingLaunchFn SSO_CAT4(sso_ring_lookup_, SSO_TNAME, SSO_N)(int, int) { return nullptr; }
#else
RingLaunchFn SSO_CAT4(sso_ring_lookup_, SSO_TNAME, SSO_N)(int mode, int maxt) {
    using T = SSO_T;
    constexpr int N = SSO_N;
    if (maxt == 512) {
        if (mode == MODE_OPEN) return &launch_ring<T, N, MODE_OPEN, -1, 512>;
        if (mode == MODE_MID) return &launch_ring<T, N, MODE_MID, +1, 512>;
        if (mode == MODE_CLOSE) return &launch_ring<T, N, MODE_CLOSE, +1, 512>;
        if (mode == MODE_CLOSE_OBS) return &launch_ring<T, N, MODE_CLOSE_OBS, +1, 512>;
    }
#if SSO_N <= 4096
    else if (maxt == 384) {
        if (mode == MODE_OPEN) return &launch_ring<T, N, MODE_OPEN, -1, 384>;
        if (mode == MODE_MID) return &launch_ring<T, N, MODE_MID, +1, 384>;
        if (mode == MODE_CLOSE) return &launch_ring<T, N, MODE_CLOSE, +1, 384>;
        if (mode == MODE_CLOSE_OBS) return &launch_ring<T, N, MODE_CLOSE_OBS, +1, 384>;
    }
#endif
    return nullptr;
}
#endif

#ifdef SSO_STUB
// development builds may leave a size out (SSO_SIZES in build.py): the dispatcher then reports "unsupported"
LaunchFn SSO_CAT3(sso_lookup_, SSO_TNAME, SSO_N)(int, int, int) { return nullptr; }
#else
LaunchFn SSO_CAT3(sso_lookup_, SSO_TNAME, SSO_N)(int strided, int pw, int sign) {
    using T = SSO_T;
    constexpr int N = SSO_N;
    if (!strided) {
        if (pw == PW_KS && sign < 0) return &launch_pass<T, N, false, PW_KS, -1>;     // 1D step
        if (pw == PW_KD2 && sign < 0) return &launch_pass<T, N, false, PW_KD2, -1>;
        if (pw == PW_KD4 && sign < 0) return &launch_pass<T, N, false, PW_KD4, -1>;
    } else {
        if (pw == PW_NONE && sign < 0) return &launch_pass<T, N, true, PW_NONE, -1>;   // middle-axis DIF / DIT
        if (pw == PW_KS && sign < 0) return &launch_pass<T, N, true, PW_KS, -1>;      // kinetic sandwich
        if (pw == PW_KD2 && sign < 0) return &launch_pass<T, N, true, PW_KD2, -1>;
        if (pw == PW_KD4 && sign < 0) return &launch_pass<T, N, true, PW_KD4, -1>;
    }
    return nullptr;
}
#endif

}  // namespace sso
