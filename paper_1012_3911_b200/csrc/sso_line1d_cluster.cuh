// sso_line1d_cluster.cuh -- the 1D Schroedinger step sequence on a thread-block cluster (sm_100a).
//
// A line of N = CS * M points is spread over the CS CTAs of one cluster (CS = 4 or 8 SMs, M <= 4096 points each), so
// that a 1D lattice may be longer than one SM's registers and shared memory hold (N up to 32768), and a 4096-point
// line uses the FP64 pipes of several SMs.  psi stays in registers for all `nsteps` of a call, as in sso_line1d.cuh;
// the transform of length N is split once (decimation in frequency over the cluster, the "four-step" factorisation)
//
//   X[k1 + CS k2] = sum_m  [ ( sum_c x[m + M c] w_CS^(c k1) ) w_N^(m k1) ]  w_M^(m k2),      w_n = exp(-2 pi i / n)
//
// (eq. 12 for the sign): a radix-CS butterfly over c in registers, the twiddle w_N^(m k1), an exchange
// through DISTRIBUTED SHARED MEMORY that hands row k1 to CTA k1 (remote st.shared::cluster, one cluster barrier), and
// the M-point transform of sso_pass.cuh inside each CTA.  The kinetic phase (eq. 13) meets the
// frequencies k1 + CS k2 in the order that transform leaves them; the way back is the transposed sequence, and the
// merged potential phase (eq. 11, 71 eq. 7 applied twice) is applied in position space.
//
// Ownership in position space: CTA r, thread u holds the points m + M c for c < CS and the PJ = 16/CS values
// m = r M/CS + j M/16 + u, j < PJ (register j + c PJ), so that every warp instruction of an exchange writes or reads
// consecutive elements.  Two cluster barriers per step order the two exchanges; the line buffer of a CTA is written
// by its peers only between the barrier that ends a step and the one that follows its own last read.
//
// Measured on B200 (profiles/r2_dsmem_microbenchmark.md) an all-to-all through DSMEM moves 12-22 B/clk/SM, so this is
// the one cluster variant of SURVEY 8(f) NEXT-3 that pays: an exchange moves at most 16 N bytes in total.
#pragma once
#include "sso_line1d_args.h"
#include "sso_pass.cuh"

namespace sso {

__device__ __forceinline__ unsigned cluster_ctarank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ unsigned map_to_rank(const void *p, unsigned rank) {
    unsigned a;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(a) : "r"((unsigned)__cvta_generic_to_shared(p)), "r"(rank));
    return a;
}
__device__ __forceinline__ void st_remote(unsigned addr, double2 v) {
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void st_remote(unsigned addr, float2 v) {
    asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
}

template <typename T, int M, int CS>
__global__ void __launch_bounds__((M / 16 < 32 ? 32 : M / 16), 1) line1d_cluster_kernel(const Line1dClusterArgs a) {
    using C = typename CxOf<T>::type;
    constexpr int U = M / 16;     // threads per CTA
    constexpr int PJ = 16 / CS;   // m values per thread in position space
    constexpr int MC = M / CS;    // m values owned by a CTA in position space
    constexpr int LAST = Sched<M>::M - 1;
    constexpr int TWN = Sched<M>::twoff(LAST);
    constexpr int TWP = (TWN + 7) & ~7;
    static_assert(U >= 32 && CS >= 2 && CS <= 16 && 16 % CS == 0, "cluster line: M >= 512, CS in {2, 4, 8, 16}");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C *stw = reinterpret_cast<C *>(smem_raw);   // twiddles of the M-point transform
    C *sl = stw + TWP;                          // line buffer (padded): exchange area, written by the peers
    // [CS][MC] rows coming back from the peers.  ALIAS (the largest lines, which would not fit otherwise): the same
    // memory as the line buffer, at the price of two more cluster barriers per step
    constexpr bool ALIAS = line1d_cluster_alias(M);
    C *rbuf = ALIAS ? sl : sl + (M + M / 16);
    C *tcl = sl + (M + M / 16) + (ALIAS ? 0 : M);  // [CS - 1][MC] cluster twiddles w_N^(m k1) of this CTA's m values
    const int u = threadIdx.x;
    const unsigned r = cluster_ctarank();
    const int gb = GB_LANES_ARE_U;  // lanes hold consecutive u (U >= 32)
    {
        const C *__restrict__ gtw = reinterpret_cast<const C *>(a.tw);
        for (int i = threadIdx.x; i < TWN; i += blockDim.x) stw[i] = gtw[i];
        const C *__restrict__ gcl = reinterpret_cast<const C *>(a.tcl) + (size_t)r * (CS - 1) * MC;
        for (int i = threadIdx.x; i < (CS - 1) * MC; i += blockDim.x) tcl[i] = gcl[i];
    }
    C *__restrict__ gp = reinterpret_cast<C *>(a.psi);
    C x[16], hv[16], kf[16];
    auto half_phase = [&](long long n) -> C {
        if (a.vrep == VREP_TABLE) return reinterpret_cast<const C *>(a.vtab)[n];
        return expi_small<T>(reinterpret_cast<const double *>(a.vtab)[n]);
    };
    // register j + c PJ  <->  lattice point (r MC + j U + u) + M c
    auto point = [&](int j, int c) -> long long { return (long long)r * MC + j * U + u + (long long)M * c; };
#pragma unroll
    for (int c = 0; c < CS; ++c)
#pragma unroll
        for (int j = 0; j < PJ; ++j) {
            const long long n = point(j, c);
            const C h = half_phase(n);
            x[j + c * PJ] = cmul(ld_stream(&gp[n]), h);  // leading half step
            if (a.vrep == VREP_TABLE) hv[j + c * PJ] = cmul(h, h);
            else hv[j + c * PJ] = expi_small<T>(2.0 * reinterpret_cast<const double *>(a.vtab)[n]);
        }
#pragma unroll
    for (int q = 0; q < 16; ++q) kf[q] = reinterpret_cast<const C *>(a.kph)[(size_t)r * M + q * U + u];
    // remote addresses: row k1 of the forward exchange goes to the line buffer of CTA k1, row r of the way back to
    // the receive buffer of the CTA that owns the m value
    unsigned rline[CS], rback[CS];
#pragma unroll
    for (int k = 0; k < CS; ++k) {
        rline[k] = map_to_rank(sl, (unsigned)k);
        rback[k] = map_to_rank(rbuf + (size_t)r * MC, (unsigned)k);
    }
    __syncthreads();
    cluster_barrier();  // every CTA of the cluster is resident and has its tables before anyone writes to a peer

    for (int rep = 0; rep < a.nsteps; ++rep) {
        if (ALIAS && rep > 0) cluster_barrier();  // every peer has read what came back to it in the previous step
        // ---- forward: butterfly over c, twiddle, row k1 -> CTA k1
#pragma unroll
        for (int j = 0; j < PJ; ++j) dft_reg<CS, PJ, -1>(&x[j]);
#pragma unroll
        for (int k1 = 0; k1 < CS; ++k1)
#pragma unroll
            for (int j = 0; j < PJ; ++j) {
                C v = x[j + k1 * PJ];
                if (k1 > 0) v = cmul(v, tcl[(k1 - 1) * MC + j * U + u]);
                const int m = (int)r * MC + j * U + u;
                st_remote(rline[k1] + (unsigned)(padp(m) * sizeof(C)), v);
            }
        cluster_barrier();
        // ---- row r: M-point transform, kinetic phase, transform back (stage-0 layout: position u + q U)
#pragma unroll
        for (int q = 0; q < 16; ++q) x[q] = sl[padp(u + q * U)];
        DifChain<T, M, 0, -1>::run(x, u, stw, sl, gb);
#pragma unroll
        for (int q = 0; q < 16; ++q) x[q] = cmul(x[q], kf[q]);
        DitChain<T, M, LAST, +1>::run(x, u, stw, sl, gb);
        if (ALIAS) cluster_barrier();  // every peer has finished its own transform in the buffer about to be written
        // ---- back: element m = u + q U of row r goes to the CTA that owns m (m = r' MC + j U + u, q = j + r' PJ)
#pragma unroll
        for (int q = 0; q < 16; ++q) st_remote(rback[q / PJ] + (unsigned)(((q % PJ) * U + u) * sizeof(C)), x[q]);
        cluster_barrier();
#pragma unroll
        for (int k1 = 0; k1 < CS; ++k1)
#pragma unroll
            for (int j = 0; j < PJ; ++j) {
                C v = rbuf[k1 * MC + j * U + u];
                if (k1 > 0) v = cmulc(v, tcl[(k1 - 1) * MC + j * U + u]);
                x[j + k1 * PJ] = v;
            }
#pragma unroll
        for (int j = 0; j < PJ; ++j) dft_reg<CS, PJ, +1>(&x[j]);
        if (rep + 1 < a.nsteps) {
#pragma unroll
            for (int q = 0; q < 16; ++q) x[q] = cmul(x[q], hv[q]);
        }
    }
#pragma unroll
    for (int c = 0; c < CS; ++c)
#pragma unroll
        for (int j = 0; j < PJ; ++j) {
            const long long n = point(j, c);
            st_stream(&gp[n], cmul(x[j + c * PJ], half_phase(n)));  // trailing half step
        }
    cluster_barrier();  // no CTA leaves while a peer may still write to it
}

template <typename T, int M, int CS> cudaError_t launch_line1d_cluster(const Line1dClusterArgs &a, size_t smem, cudaStream_t st);

}  // namespace sso
