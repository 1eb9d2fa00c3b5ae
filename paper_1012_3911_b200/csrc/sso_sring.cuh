// sso_sring.cuh -- strided-axis passes of a 2D/3D lattice through the tile rings of sso_ring.cuh (sm_100a).
//
// Along a non-last axis the elements of a line are `inner` apart, so a tile is TL ADJACENT lines: N rows of
// TL contiguous complex numbers.  The TMA engine loads such a tile as tensor boxes (cp.async.bulk.tensor, SASS
// UTMALDG) into a ring buffer laid out [component][row][TL]; the results are stored from registers.  Passes:
//
//   SMODE_KS / KD2 / KD4   forward DIF -> kinetic factor -> inverse DIT     (eq. 13; 203-232 eq. 27-33)
//   SMODE_DIF              forward DIF, result left in network order         (middle axis of a 3D lattice)
//   SMODE_DIT              inverse DIT from network order
//
// Thread layout of a group (GT = CC * TL * N/16 threads, CC = components worked on together): with UL = 8 / TL,
//   tid = t + TL * (ulo + UL * (c + CC * uhi)),   u = ulo + UL * uhi,
// so that a quarter warp reads 128 contiguous bytes of the tile and the CC components of a k point sit in lanes
// of one warp: the Dirac kinetic factor gathers them through the exchange buffer with warp-level
// synchronisation only (a version that traded them with shuffles, 224 SHFL per thread and tile, measured slower).
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

// Thread (c, u) of a line applies the factor to the PP = 16/CC k points of slots (c PP + i) U + u, all components:
template <int CC> struct DiracScalars {
    double cs[16 / CC], sE[16 / CC];  // cos(E tau) / Ntot and sin(E tau) / (E Ntot) of those k points
};
// evaluated while x is parked in shared memory (inside the last exchange of the forward transform), so that the
// square root and the trigonometric pair run with the registers of x free.  r12 = c^2 (pi_1^2 + pi_2^2) + m^2 c^4 is
// the same for the whole line.  E^2 >= m^2 c^4 > 0, so 1/E comes from one rsqrt (E = E^2 rsqrt(E^2), a few ulp) and no
// division; FAST: |E tau| < 2^30 for every k point of the plan (checked on the host), so the quadrant reduction of
// expi_small replaces the library sincos.  Together about 40 FP64 instructions per k point against about 85.
template <int CC, int U>
__device__ __forceinline__ void dirac_scalars(DiracScalars<CC> &k, int u, int c, const double *cp0, double r12, double dt, double scale, bool fast) {
    constexpr int PP = 16 / CC;
#pragma unroll
    for (int i = 0; i < PP; ++i) {
        const double w0 = cp0[(c * PP + i) * U + u];
        const double E2 = fma(w0, w0, r12);
        const double rE = rsqrt(E2);
        const double E = E2 * rE;
        double sn, cs;
        if (fast) {
            const double2 e = expi_small<double>(E * dt);
            cs = e.x;
            sn = e.y;
        } else {
            sincos(E * dt, &sn, &cs);
        }
        k.cs[i] = cs * scale;
        k.sE[i] = sn * rE * scale;
    }
}

// Dirac kinetic factor on the DIF output (eq. 27-33, 240-242 eq. 35) in the closed form
//   U = cos(E tau) - i (sin(E tau)/E) (c alpha.pi + m c^2 beta),   E = sqrt(c^2 pi^2 + m^2 c^4),
// which follows from H^2 = E^2 by the argument of PAPER.md:168-184 (eq. 23/24).  The CC components of a k point
// are gathered into one thread through the exchange buffer, multiplied by the 2x2 / 4x4 unitary and scattered back.
// The CC threads that trade values are lanes of one warp (thread layout of the kernel), so the two hand-overs need
// a __syncwarp each and no group barrier.  `me` = this thread's 16 slots of its own line (stage layout of the last
// stage), `line0` = the same line of component 0, comp_pitch = elements between components.
//   TABLE: cs, sE come from the table `ktab` instead of `k`.
template <typename T, int CC, int U, bool TABLE>
__device__ __forceinline__ void dirac_kinetic_warp(typename CxOf<T>::type (&x)[16], int u, int c, typename CxOf<T>::type *me, typename CxOf<T>::type *line0,
                                                   int comp_pitch, const double *cp0, double w1, double w2, double mc2, const DiracScalars<CC> &k,
                                                   const double2 *__restrict__ ktab, long long ktab_stride) {
    using C = typename CxOf<T>::type;
    constexpr int PP = 16 / CC;
#pragma unroll
    for (int q = 0; q < 16; ++q) me[q] = x[q];
    __syncwarp();
    C y[CC][PP];
#pragma unroll
    for (int c2 = 0; c2 < CC; ++c2)
#pragma unroll
        for (int i = 0; i < PP; ++i) y[c2][i] = line0[c2 * comp_pitch + 17 * u + c * PP + i];
#pragma unroll
    for (int i = 0; i < PP; ++i) {
        const int slot = (c * PP + i) * U + u;
        double cs, sE;
        if constexpr (TABLE) {
            const double2 e = ld_table(ktab + (long long)slot * ktab_stride);
            cs = e.x;
            sE = e.y;
        } else {
            cs = k.cs[i];
            sE = k.sE[i];
        }
        const T fc = (T)cs;
        const T fm = (T)(sE * mc2);
        const T f0 = (T)(sE * cp0[slot]), f1 = (T)(sE * w1), f2 = (T)(sE * w2);
        // out = cs psi - i sE H psi ;  (-i)(a + i b) = b - i a
        if constexpr (CC == 2) {
            const C a0 = y[0][i], a1 = y[1][i];
            // H psi_0 = mc2 a0 + c (p0 - i p1) a1 ; H psi_1 = c (p0 + i p1) a0 - mc2 a1
            const C h0 = mk<C>(fm * a0.x + f0 * a1.x + f1 * a1.y, fm * a0.y + f0 * a1.y - f1 * a1.x);
            const C h1 = mk<C>(f0 * a0.x - f1 * a0.y - fm * a1.x, f0 * a0.y + f1 * a0.x - fm * a1.y);
            y[0][i] = mk<C>(fc * a0.x + h0.y, fc * a0.y - h0.x);
            y[1][i] = mk<C>(fc * a1.x + h1.y, fc * a1.y - h1.x);
        } else {
            const C a0 = y[0][i], a1 = y[1][i], a2 = y[2][i], a3 = y[3][i];
            // sigma.p (v0, v1) = (p2 v0 + (p0 - i p1) v1, (p0 + i p1) v0 - p2 v1)
            // H psi = (mc2 u + c sigma.p l, c sigma.p u - mc2 l)
            const C h0 = mk<C>(fm * a0.x + f2 * a2.x + f0 * a3.x + f1 * a3.y, fm * a0.y + f2 * a2.y + f0 * a3.y - f1 * a3.x);
            const C h1 = mk<C>(fm * a1.x + f0 * a2.x - f1 * a2.y - f2 * a3.x, fm * a1.y + f0 * a2.y + f1 * a2.x - f2 * a3.y);
            const C h2 = mk<C>(f2 * a0.x + f0 * a1.x + f1 * a1.y - fm * a2.x, f2 * a0.y + f0 * a1.y - f1 * a1.x - fm * a2.y);
            const C h3 = mk<C>(f0 * a0.x - f1 * a0.y - f2 * a1.x - fm * a3.x, f0 * a0.y + f1 * a0.x - f2 * a1.y - fm * a3.y);
            y[0][i] = mk<C>(fc * a0.x + h0.y, fc * a0.y - h0.x);
            y[1][i] = mk<C>(fc * a1.x + h1.y, fc * a1.y - h1.x);
            y[2][i] = mk<C>(fc * a2.x + h2.y, fc * a2.y - h2.x);
            y[3][i] = mk<C>(fc * a3.x + h3.y, fc * a3.y - h3.x);
        }
    }
#pragma unroll
    for (int c2 = 0; c2 < CC; ++c2)
#pragma unroll
        for (int i = 0; i < PP; ++i) line0[c2 * comp_pitch + 17 * u + c * PP + i] = y[c2][i];
    __syncwarp();
#pragma unroll
    for (int q = 0; q < 16; ++q) x[q] = me[q];
}

template <typename T, int N, int SMODE>
__global__ void __launch_bounds__(512, 1) sring_kernel(const SRingArgs a, const __grid_constant__ CUtensorMap tmap) {
    using C = typename CxOf<T>::type;
    constexpr int U = N / 16;
    constexpr int CC = (SMODE == SMODE_KD2 || SMODE == SMODE_KD2F) ? 2 : ((SMODE == SMODE_KD4 || SMODE == SMODE_KD4F) ? 4 : 1);
    constexpr bool KTABLE = SMODE == SMODE_KD2 || SMODE == SMODE_KD4;
    constexpr int LAST = Sched<N>::M - 1;
    constexpr int TWN = Sched<N>::twoff(LAST);
    constexpr int TWP = (TWN + 7) & ~7;
    // the pointwise table along the line (Schroedinger phase or Dirac momenta) sits in shared memory: with nearly all
    // of it given to tiles, the L1 left over is too small to keep even a 2 KB table resident
    constexpr int LTB = sring_line_table_bytes(SMODE, N, (int)sizeof(C));
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C *stw = reinterpret_cast<C *>(smem_raw);
    unsigned char *ltab = smem_raw + TWP * sizeof(C);
    C *bufs = reinterpret_cast<C *>(ltab + LTB);
    TileRing ring(bufs + (size_t)a.NB * a.bufstride, a.NB, a.G);

    const int TL = a.TL, GT = a.GT, G = a.G;
    const int grp = threadIdx.x / GT;
    const int tid = threadIdx.x - grp * GT;
    // thread layout (file header): t fastest, then UL consecutive u, then the component, then the rest of u
    const int UL = TL >= 8 ? 1 : 8 / TL;
    const int t = tid % TL;
    int r = tid / TL;
    const int ulo = r % UL;
    r /= UL;
    const int c = r % CC;
    const int u = ulo + UL * (r / CC);
    // a warp holds 32 / (TL CC) consecutive u of TL lines: exchanges confined to that many u stay inside it
    const int wl = TL * CC;
    const int gb = (G > 1 ? ((grp + 1) | (GT << 8)) : 0) | ((32 % wl == 0 && GT % 32 == 0) ? (GB_LANES_ARE_U | ((31 - __clz(wl)) << GB_TL_SHIFT)) : 0);
    const unsigned tile_bytes = (unsigned)(CC * TL * N * sizeof(C));
    const int nloc = a.ntiles > (int)blockIdx.x ? (a.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const int nbox = N / a.box_rows;

    auto tile_of = [&](int k) {
        const int tl = (int)blockIdx.x + k * (int)gridDim.x;
        return a.rev ? a.ntiles - 1 - tl : tl;  // rev: see sso_ring.cuh
    };
    auto issue = [&](int k, int b) {
        const int tile = tile_of(k);
        const int o = tile >> a.tpo_shift, i0 = (tile & (a.tiles_per_outer - 1)) * TL;  // lattice sizes are powers of two
        C *dst = bufs + (size_t)b * a.bufstride;
        mbar_expect_tx(ring.full(b), tile_bytes);
        for (int cc = 0; cc < CC; ++cc)
            for (int j = 0; j < nbox; ++j)
                tma_load_3d(dst + (size_t)(cc * N + j * a.box_rows) * TL, &tmap, 2 * i0, j * a.box_rows, CC > 1 ? cc : o, ring.full(b));
    };

    // let the next pass of the stream start its own setup as SMs free up
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    ring.init();
    {
        const C *__restrict__ gtw = reinterpret_cast<const C *>(a.tw);
        for (int i = threadIdx.x; i < TWN; i += blockDim.x) stw[i] = gtw[i];
    }
    __syncthreads();
    // everything above touched only plan-owned tables; psi is valid once the previous pass has completed
    asm volatile("griddepcontrol.wait;" ::: "memory");
    auto refill = [&](int k, int b) {
        if (k < nloc) {
            ring.publish(k, b);
            issue(k, b);
        }
    };
    if (tid == 0) {
        for (int b = grp; b < a.NB; b += G) refill(b, b);  // the first NB tiles, loaded by the groups' leaders
        ring.draw(grp);
    }
    if constexpr (LTB > 0) {
        // (the line table may have been rebuilt for this step by the kernel before this one, hence after the wait)
        double *dst = reinterpret_cast<double *>(ltab);
        if constexpr (SMODE == SMODE_KS) {
            const double *__restrict__ src = reinterpret_cast<const double *>(a.kph0);
            constexpr int ND = N * (int)sizeof(C) / 8;
            for (int i = threadIdx.x; i < ND; i += blockDim.x) dst[i] = src[i];
        } else {
            // Dirac: c pi_0 = c (k_0 - q Abar_0) per slot of the line axis (reading G16)
            for (int i = threadIdx.x; i < N; i += blockDim.x) dst[i] = a.clight * (a.kv0[i] - a.sh[0]);
        }
        __syncthreads();
    }

    gsync(gb);  // publishes the group's first ticket
    for (;;) {
        const int k = ring.drawn(grp);  // the group's next tile, in the CTA's loading order
        if (k >= nloc) break;
        const int b = ring.wait(k);
        C *buf = bufs + (size_t)b * a.bufstride;
        C *dense = buf + (size_t)c * N * TL + t;     // TMA layout [CC][N][TL]: row r of this line at dense[r * TL]
        C *sl = buf + (c * TL + t) * a.pitch;        // exchange layout: padded lines
        const int tile = tile_of(k);
        const int line = (tile & (a.tiles_per_outer - 1)) * TL + t;  // line index on the non-line axes (within a component)

        C x[16];
        if constexpr (SMODE == SMODE_DIT) {
#pragma unroll
            for (int q = 0; q < 16; ++q) x[q] = dense[(u * 16 + q) * TL];
        } else {
#pragma unroll
            for (int q = 0; q < 16; ++q) x[q] = dense[(u + q * U) * TL];
        }

        gsync(gb);  // the exchange layout overlaps the TMA layout of other warps' lines

        [[maybe_unused]] DiracScalars<(CC > 1 ? CC : 2)> dks;
        [[maybe_unused]] double w1 = 0.0, w2 = 0.0;  // c pi_1, c pi_2 of this line (pi = k - q Abar_n, reading G16)
        [[maybe_unused]] const double mc2 = a.mass * a.clight * a.clight;
        if constexpr (CC > 1) {
            if (a.ndim == 2) w1 = a.clight * (a.kv2[line & (a.rest1 - 1)] - a.sh[1]);
            if (a.ndim == 3) {
                w1 = a.clight * (a.kv1[line >> a.rest1_shift] - a.sh[1]);
                w2 = a.clight * (a.kv2[line & (a.rest1 - 1)] - a.sh[2]);
            }
        }
        // per-line factor of the Schroedinger kinetic phase (the other axes' tables), requested before the forward
        // transform so that the loads are back when it ends
        [[maybe_unused]] C s = mk<C>((T)1, (T)0);
        [[maybe_unused]] bool has_s = false;
        if constexpr (SMODE == SMODE_KS) {
            if (a.kph1) {
                s = reinterpret_cast<const C *>(a.kph1)[line >> a.rest1_shift];
                has_s = true;
            }
            if (a.kph2) {
                const C s2 = reinterpret_cast<const C *>(a.kph2)[line & (a.rest1 - 1)];
                s = has_s ? cmul(s, s2) : s2;
                has_s = true;
            }
        }
        if constexpr (SMODE == SMODE_DIT) {
        } else if constexpr (CC > 1 && !KTABLE) {
            const double r12 = w1 * w1 + w2 * w2 + mc2 * mc2;
            DifChain<T, N, 0, -1>::run(x, u, stw, sl, gb, [&]() { dirac_scalars<CC, U>(dks, u, c, reinterpret_cast<const double *>(ltab), r12, a.dt, a.scale, a.fast_trig != 0); });
        } else {
            DifChain<T, N, 0, -1>::run(x, u, stw, sl, gb);
        }

        if constexpr (SMODE == SMODE_KS) {
            const C *k0 = reinterpret_cast<const C *>(ltab);
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                C f = k0[q * U + u];
                if (has_s) f = cmul(f, s);
                x[q] = cmul(x[q], f);
            }
        } else if constexpr (CC > 1) {
            dirac_kinetic_warp<T, CC, U, KTABLE>(x, u, c, sl + 17 * u, buf + t * a.pitch, TL * a.pitch, reinterpret_cast<const double *>(ltab), w1, w2, mc2,
                                                 dks, reinterpret_cast<const double2 *>(a.ktab) + line, a.inner);
        }

        if constexpr (SMODE != SMODE_DIF) DitChain<T, N, LAST, +1>::run(x, u, stw, sl, gb);

        fence_async_smem();  // generic-proxy accesses of the buffer before its refill through the async proxy
        if (tid == 0) ring.draw(grp);  // the group's next ticket, published by the barrier
        gsync(gb);           // every thread of the group is done with the exchange layout
        // refill the buffer at once and store from registers (a warp instruction writes 32/TL rows of TL complex numbers)
        if (tid == 0) refill(ring.claim(), b);
        {
            const long long o = tile >> a.tpo_shift;
            const long long i0 = (long long)(tile & (a.tiles_per_outer - 1)) * TL;
            C *gout = reinterpret_cast<C *>(a.psi) + (CC > 1 ? (long long)c * a.comp_stride : o * (long long)N * a.inner) + i0 + t;
            // one 64-bit multiply per thread, then pointer increments
            if constexpr (SMODE == SMODE_DIF) {
                C *pq = gout + (long long)(u * 16) * a.inner;
#pragma unroll
                for (int q = 0; q < 16; ++q, pq += a.inner) st_stream(pq, x[q]);
            } else {
                C *pq = gout + (long long)u * a.inner;
                const long long rs = (long long)U * a.inner;
#pragma unroll
                for (int q = 0; q < 16; ++q, pq += rs) st_stream(pq, x[q]);
            }
        }
    }
}

template <typename T, int N, int SMODE>
cudaError_t launch_sring(const SRingArgs &a, const void *tensor_map, unsigned threads, size_t smem, unsigned grid, cudaStream_t st);

}  // namespace sso
