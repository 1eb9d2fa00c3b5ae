// sso_line1d.cuh -- the whole 1D Schroedinger step sequence in one persistent CTA (sm_100a).
//
// A 1D line of N <= 4096 points is 64 KB at most: one CTA of N/16 threads keeps it in registers (16 points per
// thread) for all `nsteps` of a call, so psi crosses HBM once in and once out per CALL.  With so few threads every
// thread may use up to 255 registers, and the step's two pointwise tables live there too: the merged potential phase
// exp(-i V tau) of the thread's 16 points (natural order) and the kinetic phase exp(-i tau (k - q A)^2 / 2m) / N of
// its 16 slots (network order).  A step is then
//     DIF  ->  x *= K  ->  DIT  ->  x *= V        (eq. 7 merged over steps, 98 eq. 11, 107 eq. 13)
// with nothing but the stage exchanges and the twiddles touching shared memory, and no global access at all.
// (The general pass kernel re-read both 64 KB tables from L1/L2 inside the dependent chain of every step: 11.2 us per
// step for N = 4096 against 3 us of FP64 issue on one SM.)
#pragma once
#include "sso_line1d_args.h"
#include "sso_pass.cuh"

namespace sso {

template <typename T, int N>
__global__ void __launch_bounds__((N / 16 < 32 ? 32 : N / 16), 1) line1d_kernel(const Line1dArgs a) {
    using C = typename CxOf<T>::type;
    constexpr int U = N / 16;
    constexpr int LAST = Sched<N>::M - 1;
    constexpr int TWN = Sched<N>::twoff(LAST);
    constexpr int TWP = (TWN + 7) & ~7;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C *stw = reinterpret_cast<C *>(smem_raw);
    C *sl = stw + TWP;
    const int u = threadIdx.x;
    // lanes hold consecutive u: exchanges confined to 32 consecutive u need no block barrier
    const int gb = (U >= 32 || 32 % U == 0) ? GB_LANES_ARE_U : 0;
    {
        const C *__restrict__ gtw = reinterpret_cast<const C *>(a.tw);
        for (int i = threadIdx.x; i < TWN; i += blockDim.x) stw[i] = gtw[i];
    }
    C *__restrict__ gp = reinterpret_cast<C *>(a.psi);
    C x[16], hv[16], kf[16];
    auto half_phase = [&](int q) -> C {
        if (a.vrep == VREP_TABLE) return reinterpret_cast<const C *>(a.vtab)[u + q * U];
        return expi_small<T>(reinterpret_cast<const double *>(a.vtab)[u + q * U]);
    };
#pragma unroll
    for (int q = 0; q < 16; ++q) x[q] = ld_stream(&gp[u + q * U]);
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const C h = half_phase(q);
        x[q] = cmul(x[q], h);  // leading half step
        if (a.vrep == VREP_TABLE) {
            hv[q] = cmul(h, h);    // merged phase of two consecutive half steps
        } else {
            hv[q] = expi_small<T>(2.0 * reinterpret_cast<const double *>(a.vtab)[u + q * U]);
        }
        kf[q] = reinterpret_cast<const C *>(a.kph0)[q * U + u];
    }
    __syncthreads();  // twiddles are in place
    for (int rep = 0; rep < a.nsteps; ++rep) {
        DifChain<T, N, 0, -1>::run(x, u, stw, sl, gb);
#pragma unroll
        for (int q = 0; q < 16; ++q) x[q] = cmul(x[q], kf[q]);
        DitChain<T, N, LAST, +1>::run(x, u, stw, sl, gb);
        if (rep + 1 < a.nsteps) {
#pragma unroll
            for (int q = 0; q < 16; ++q) x[q] = cmul(x[q], hv[q]);
        }
    }
#pragma unroll
    for (int q = 0; q < 16; ++q) st_stream(&gp[u + q * U], cmul(x[q], half_phase(q)));  // trailing half step
}

template <typename T, int N> cudaError_t launch_line1d(const Line1dArgs &a, size_t smem, cudaStream_t st);

}  // namespace sso
