// sso_sring.cuh -- strided-axis passes of a 2D/3D lattice through the ring pipeline of sso_ring.cuh (sm_100a).
//
// Along a non-last axis the elements of a line are `inner` apart, so a tile is TL ADJACENT lines: N rows of
// TL contiguous complex numbers (TL * sizeof(complex) >= 64 bytes per row, B200 serves narrower rows at less
// than half speed).  The TMA engine moves such a tile as tensor boxes (cp.async.bulk.tensor, SASS
// UTMALDG/UTMASTG) between global memory and a ring buffer laid out [component][row][TL]; everything else is
// the ring of sso_ring.cuh.  Passes:
//
//   SMODE_KS / KD2 / KD4   forward DIF -> kinetic factor -> inverse DIT     (eq. 13; 203-232 eq. 27-33)
//   SMODE_DIF              forward DIF, result left in network order         (middle axis of a 3D lattice)
//   SMODE_DIT              inverse DIT from network order
#pragma once
#include <cuda.h>

#include "sso_ring.cuh"

namespace sso {

__device__ __forceinline__ void tma_load_3d(void *smem_dst, const CUtensorMap *map, int c0, int c1, int c2, void *bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
                 : "memory");
}

template <typename T, int N, int SMODE>
__global__ void __launch_bounds__(512, 1) sring_kernel(const SRingArgs a, const __grid_constant__ CUtensorMap tmap) {
    using C = typename CxOf<T>::type;
    constexpr int U = N / 16;
    constexpr int CC = SMODE == SMODE_KD2 ? 2 : (SMODE == SMODE_KD4 ? 4 : 1);
    constexpr int LAST = Sched<N>::M - 1;
    constexpr int TWN = Sched<N>::twoff(LAST);
    constexpr int TWP = (TWN + 7) & ~7;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C *stw = reinterpret_cast<C *>(smem_raw);
    C *bufs = stw + TWP;
    unsigned long long *full = reinterpret_cast<unsigned long long *>(bufs + (size_t)a.NB * a.bufstride);
    volatile int *ktile = reinterpret_cast<volatile int *>(full + a.NB);  // as in ring_kernel

    const int TL = a.TL, GT = a.GT, G = a.G, NB = a.NB;
    const int grp = threadIdx.x / GT;
    const int tid = threadIdx.x - grp * GT;
    // lane = u * TL + t within a component: exchanges confined to 32 / TL consecutive u stay inside a warp
    const int gb = (G > 1 ? ((grp + 1) | (GT << 8)) : 0) | ((32 % TL == 0 && (U * TL) % 32 == 0) ? (GB_LANES_ARE_U | ((31 - __clz(TL)) << GB_TL_SHIFT)) : 0);
    const int t = tid % TL;
    const int cu = tid / TL;
    const int u = cu % U;
    const int c = cu / U;
    const unsigned tile_bytes = (unsigned)(CC * TL * N * sizeof(C));
    const int nloc = a.ntiles > (int)blockIdx.x ? (a.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const int nbox = N / a.box_rows;

    auto tile_of = [&](int k) { return (int)blockIdx.x + k * (int)gridDim.x; };
    auto issue = [&](int k, int b) {
        const int tile = tile_of(k);
        const int o = tile / a.tiles_per_outer, i0 = (tile % a.tiles_per_outer) * TL;
        C *dst = bufs + (size_t)b * a.bufstride;
        mbar_expect_tx(&full[b], tile_bytes);
        for (int cc = 0; cc < CC; ++cc)
            for (int j = 0; j < nbox; ++j)
                tma_load_3d(dst + (size_t)(cc * N + j * a.box_rows) * TL, &tmap, 2 * i0, j * a.box_rows, CC > 1 ? cc : o, &full[b]);
    };

    // let the next pass of the stream start its own setup as SMs free up
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (threadIdx.x == 0) {
        ktile[NB] = NB;
        for (int b = 0; b < NB; ++b) mbar_init(&full[b], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    {
        const C *__restrict__ gtw = reinterpret_cast<const C *>(a.tw);
        for (int i = threadIdx.x; i < TWN; i += blockDim.x) stw[i] = gtw[i];
    }
    __syncthreads();
    // everything above touched only plan-owned tables; psi is valid once the previous pass has completed
    asm volatile("griddepcontrol.wait;" ::: "memory");
    // every group owns NBG = NB / G buffers: its leader fills them, its threads consume them, so a buffer's
    // mbarrier never sees a waiter that is not in step with its fills
    const int NBG = NB / G;
    auto refill = [&](int kn, int b) {
        if (kn < nloc) {
            ktile[b] = kn;
            issue(kn, b);
        } else {
            ktile[b] = -1;
            mbar_arrive(&full[b]);
        }
    };
    if (tid == 0)
        for (int j = 0; j < NBG; ++j) refill(grp * NBG + j, grp * NBG + j);

    for (int j = 0;; ++j) {
        const int b = grp * NBG + j % NBG;
        mbar_wait(&full[b], (unsigned)((j / NBG) & 1));
        const int k = ktile[b];
        if (k < 0) break;
        C *buf = bufs + (size_t)b * a.bufstride;
        C *dense = buf + (size_t)c * N * TL + t;     // TMA layout [CC][N][TL]: row r of this line at dense[r * TL]
        C *sl = buf + (c * TL + t) * a.pitch;        // exchange layout: padded lines
        const int tile = tile_of(k);
        const int line = (tile % a.tiles_per_outer) * TL + t;  // line index on the non-line axes (within a component)

        C x[16];
        if constexpr (SMODE == SMODE_DIT) {
#pragma unroll
            for (int q = 0; q < 16; ++q) x[q] = dense[(u * 16 + q) * TL];
        } else {
#pragma unroll
            for (int q = 0; q < 16; ++q) x[q] = dense[(u + q * U) * TL];
        }

        gsync(gb);  // the exchange layout overlaps the TMA layout of other warps' lines

        if constexpr (SMODE != SMODE_DIT) DifChain<T, N, 0, -1>::run(x, u, stw, sl, gb);

        if constexpr (SMODE == SMODE_KS) {
            const C *__restrict__ k0 = reinterpret_cast<const C *>(a.kph0);
            C s = mk<C>((T)1, (T)0);
            bool has_s = false;
            if (a.kph1) {
                s = reinterpret_cast<const C *>(a.kph1)[line / a.rest1];
                has_s = true;
            }
            if (a.kph2) {
                const C s2 = reinterpret_cast<const C *>(a.kph2)[line % a.rest1];
                s = has_s ? cmul(s, s2) : s2;
                has_s = true;
            }
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                C f = k0[q * U + u];
                if (has_s) f = cmul(f, s);
                x[q] = cmul(x[q], f);
            }
        } else if constexpr (SMODE == SMODE_KD2 || SMODE == SMODE_KD4) {
            double p1 = 0.0, p2 = 0.0;
            if (a.ndim == 2) p1 = a.kv2[line % a.rest1] - a.sh[1];
            if (a.ndim == 3) {
                p1 = a.kv1[line / a.rest1] - a.sh[1];
                p2 = a.kv2[line % a.rest1] - a.sh[2];
            }
            dirac_kinetic<T, CC, U>(x, u, c, sl, buf + t * a.pitch, TL * a.pitch, gb, a.kv0, a.sh[0], p1, p2, a.mass, a.clight, a.dt, a.scale);
        }

        if constexpr (SMODE != SMODE_DIF) DitChain<T, N, LAST, +1>::run(x, u, stw, sl, gb);

        fence_async_smem();  // generic-proxy accesses of the buffer before its refill through the async proxy
        gsync(gb);  // every thread of the group is done with the exchange layout
        {
            // store from registers (a warp instruction writes 32/TL rows of TL complex numbers) and refill the
            // buffer at once
            if (tid == 0) refill(atomicAdd(const_cast<int *>(&ktile[NB]), 1), b);
            const long long o = tile / a.tiles_per_outer;
            const long long i0 = (long long)(tile % a.tiles_per_outer) * TL;
            C *gout = reinterpret_cast<C *>(a.psi) + (CC > 1 ? (long long)c * a.comp_stride : o * (long long)N * a.inner) + i0 + t;
            if constexpr (SMODE == SMODE_DIF) {
#pragma unroll
                for (int q = 0; q < 16; ++q) st_stream(gout + (long long)(u * 16 + q) * a.inner, x[q]);
            } else {
#pragma unroll
                for (int q = 0; q < 16; ++q) st_stream(gout + (long long)(u + q * U) * a.inner, x[q]);
            }
        }
    }
}

template <typename T, int N, int SMODE>
cudaError_t launch_sring(const SRingArgs &a, const void *tensor_map, unsigned threads, size_t smem, unsigned grid, cudaStream_t st);

}  // namespace sso
