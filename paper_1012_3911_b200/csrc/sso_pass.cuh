// sso_pass.cuh -- the line-pass kernel of the split-operator step (sm_100a).
//
// One CTA holds a tile of whole lattice lines on chip and applies, without
// leaving the SM,
//
//     [pre-phase]  ->  DIF FFT (sign s)  ->  [pointwise factor]  ->  DIT FFT (sign -s)  ->  [post-phase]
//
// to every line of the tile.  The pointwise factor is the potential phase of
// PAPER.md:98 (eq. 11), the Schroedinger kinetic phase of PAPER.md:107 (eq. 13)
// or the Dirac kinetic unitary of PAPER.md:203-232 (eq. 27-33) in the closed form
// U = cos(E tau) - i sin(E tau)/E (c alpha.pi + m c^2 beta), which follows from
// H^2 = E^2 by the argument of PAPER.md:168-184 (eq. 23/24).
// ("Kernels") for the data layout, the radix schedule and the byte counts.
//
// FFT structure.  A line of N = R_1 R_2 ... R_m points (R_m = 16, the other R_i
// in {2,4,8,16}) is transformed by an in-place decimation-in-frequency network
// (natural order in, mixed-radix digit-reversed order out) and transformed back
// by the transposed decimation-in-time network (digit-reversed in, natural out),
// so no reordering pass is ever needed: the pointwise tables are stored in the
// digit-reversed order instead.  Every thread holds 16 complex points in
// registers in every stage; a radix-R stage is 16/R register butterflies; between
// stages the points are exchanged through padded shared memory.  The first stage
// reads global memory directly into registers and the last stage writes it back.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sso_dispatch.h"

namespace sso {

template <typename T> struct CxOf;
template <> struct CxOf<float> { using type = float2; };
template <> struct CxOf<double> { using type = double2; };

template <typename C> __device__ __forceinline__ C mk(decltype(C::x) a, decltype(C::x) b) {
    C r;
    r.x = a;
    r.y = b;
    return r;
}
template <typename C> __device__ __forceinline__ C cadd(C a, C b) { return mk<C>(a.x + b.x, a.y + b.y); }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { return mk<C>(a.x - b.x, a.y - b.y); }
template <typename C> __device__ __forceinline__ C cmul(C a, C b) {
    return mk<C>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
template <typename C> __device__ __forceinline__ C cmulc(C a, C b) {  // a * conj(b)
    return mk<C>(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}

// psi is streamed: read once and written once per pass, so keep it out of L1 (the twiddle and phase tables
// live there) but leave the L2 policy alone (the small configs stay L2-resident between passes)
__device__ __forceinline__ double2 ld_stream(const double2 *p) {
    double2 v;
    asm volatile("ld.global.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ float2 ld_stream(const float2 *p) {
    float2 v;
    asm volatile("ld.global.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_stream(double2 *p, double2 v) {
    asm volatile("st.global.L1::no_allocate.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void st_stream(float2 *p, float2 v) {
    asm volatile("st.global.L1::no_allocate.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(v.x), "f"(v.y) : "memory");
}
// ask L2 to fetch `bytes` (multiple of 16) starting at p; used for the potential table of a tile, which is
// needed only after the first FFT
__device__ __forceinline__ void prefetch_l2_bulk(const void *p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// ------------------------------------------------------------------------------------------
// radix schedule: N = 2^LOG, last stage radix 16, the LOG-4 remaining bits in stages of <= 4 bits,
// the first stage taking the remainder.
// ------------------------------------------------------------------------------------------
__host__ __device__ constexpr int ilog2c(int n) { return n <= 1 ? 0 : 1 + ilog2c(n >> 1); }

template <int N> struct Sched {
    static constexpr int LOG = ilog2c(N);
    static_assert((1 << LOG) == N && LOG >= 4, "N must be a power of two >= 16");
    static constexpr int REM = LOG - 4;
    static constexpr int M = 1 + (REM + 3) / 4;  // number of stages
    __host__ __device__ static constexpr int lr(int i) { return i == M - 1 ? 4 : (i == 0 ? REM - 4 * (M - 2) : 4); }
    __host__ __device__ static constexpr int nprev(int i) {  // length of the sub-transform entering stage i
        int n = N;
        for (int j = 0; j < i; ++j) n >>= lr(j);
        return n;
    }
    // offset of stage i's twiddle block: stage j < M-1 stores (R_j - 1) * N_j entries, [k-1][l], l contiguous
    __host__ __device__ static constexpr int twoff(int i) {
        int o = 0;
        for (int j = 0; j < i; ++j) o += ((1 << lr(j)) - 1) * (nprev(j) >> lr(j));
        return o;
    }
};

// The twiddle blocks of a line sit in shared memory beside the line buffers -- except for the longest lines
// (8192 complex128 points: 131 KB of twiddles + 139 KB of line), whose kernels read them from global memory (L2)
template <typename C, int N> __host__ __device__ constexpr bool twiddles_in_global() {
    return (size_t)(((Sched<N>::twoff(Sched<N>::M - 1) + 7) & ~7) + N + N / 16) * sizeof(C) > (size_t)200 * 1024;
}

// cos(2 pi j/16), sin(2 pi j/16), j = 0..7
__host__ __device__ constexpr double cos16(int j) {
    return j == 0 ? 1.0
         : j == 1 ? 0.92387953251128675613
         : j == 2 ? 0.70710678118654752440
         : j == 3 ? 0.38268343236508977173
         : j == 4 ? 0.0
         : j == 5 ? -0.38268343236508977173
         : j == 6 ? -0.70710678118654752440
                  : -0.92387953251128675613;
}
__host__ __device__ constexpr double sin16(int j) {
    return j == 0 ? 0.0
         : j == 1 ? 0.38268343236508977173
         : j == 2 ? 0.70710678118654752440
         : j == 3 ? 0.92387953251128675613
         : j == 4 ? 1.0
         : j == 5 ? 0.92387953251128675613
         : j == 6 ? 0.70710678118654752440
                  : 0.38268343236508977173;
}

__host__ __device__ constexpr int brevc(int k, int bits) {
    int r = 0;
    for (int b = 0; b < bits; ++b) r |= ((k >> b) & 1) << (bits - 1 - b);
    return r;
}

// One radix-2 butterfly with the twiddle on the second input, fused into multiply-adds:
//   (a, b) <- (a + w b, a - w b),   w = exp(SIGN 2 pi i j16 / 16),
// 6 FP instructions for a general w (a + w b by four FMAs, a - w b = 2 a - (a + w b) by two more) against 8 for a
// complex multiplication followed by an addition and a subtraction; 4 when w is 1 or +-i.
template <int SIGN, typename C> __device__ __forceinline__ void bfly(C &a, C &b, int j16) {
    using T = decltype(C::x);
    if (j16 == 0) {
        const C r = cadd(a, b), d = csub(a, b);
        a = r;
        b = d;
    } else if (j16 == 4) {
        // w = SIGN i:  w b = SIGN (-b.y, b.x)
        const C wb = SIGN > 0 ? mk<C>(-b.y, b.x) : mk<C>(b.y, -b.x);
        const C r = cadd(a, wb), d = csub(a, wb);
        a = r;
        b = d;
    } else {
        const T c = (T)cos16(j16);
        const T s = (T)(SIGN > 0 ? sin16(j16) : -sin16(j16));
        C r;
        r.x = fma(-s, b.y, fma(c, b.x, a.x));
        r.y = fma(s, b.x, fma(c, b.y, a.y));
        b = mk<C>(fma((T)2, a.x, -r.x), fma((T)2, a.y, -r.y));
        a = r;
    }
}

// y[k*S] = sum_j x[j*S] exp(SIGN 2 pi i j k / R), natural order in and out, in registers: the iterative
// decimation-in-time network on the bit-reversed view A[p] = x[brev(p) S] (register renaming, no data movement),
// levels len = 2, 4, .., R with the butterflies above; A[k] = y_k at the end, copied back to natural order.
// FIRST = false skips the first level (len = 2: the pairs x[k], x[k + R/2]), for callers that fuse it with
// twiddles on the inputs.
template <int R, int S, int SIGN, int LB, typename C> __device__ __forceinline__ void dft_levels(C *x) {
    constexpr int B = ilog2c(R);
    if constexpr (LB <= B) {
        constexpr int LEN = 1 << LB, HALF = LEN / 2;
#pragma unroll
        for (int i = 0; i < R / LEN; ++i)
#pragma unroll
            for (int j = 0; j < HALF; ++j) bfly<SIGN>(x[brevc(i * LEN + j, B) * S], x[brevc(i * LEN + j + HALF, B) * S], j * (16 / LEN));
        dft_levels<R, S, SIGN, LB + 1>(x);
    }
}
template <int R, int S, int SIGN, typename C, bool FIRST = true> __device__ __forceinline__ void dft_reg(C *x) {
    if constexpr (R >= 2) {
        constexpr int B = ilog2c(R);
        dft_levels<R, S, SIGN, FIRST ? 1 : 2>(x);
        if constexpr (R > 2) {
            C t[R];
#pragma unroll
            for (int k = 0; k < R; ++k) t[k] = x[brevc(k, B) * S];
#pragma unroll
            for (int k = 0; k < R; ++k) x[k * S] = t[k];
        }
    }
}

// Layout of stage I: thread u = B' * Mi + l' holds, in register q, line position
//   pos = B' * 16 Mi + q Mi + l',   Mi = nprev(I)/16.
// In shared memory position p lives at p + (p >> 4) (one pad element per 16: every access pattern the
// stages use is then bank-conflict free at 128-byte wavefront granularity).  Because q Mi is either a
// multiple of 16 or stays inside one group of 16, the padded address splits into a per-thread base and a
// compile-time offset per register, so every LDS/STS uses [base + immediate].
__device__ __forceinline__ int padp(int p) { return p + (p >> 4); }
template <int N, int I> __device__ __forceinline__ int stage_base(int u) {
    constexpr int Mi = Sched<N>::nprev(I) / 16;
    return padp((u / Mi) * (16 * Mi) + (u % Mi));
}
template <int N, int I> __host__ __device__ constexpr int stage_delta(int q) {
    constexpr int Mi = Sched<N>::nprev(I) / 16;
    return q * Mi + ((q * Mi) >> 4);
}
__host__ __device__ constexpr int lin_delta(int q, int stride) { return q * stride + ((q * stride) >> 4); }

// one DIF stage: butterflies over the top digit of the current sub-transform, then twiddles.
// Twiddle w_NP^(l k) sits at [k-1][l] of this stage's block (shared memory copy): consecutive threads
// (consecutive l') read consecutive entries.
template <typename T, int N, int I, int SIGN> __device__ __forceinline__ void dif_stage(typename CxOf<T>::type (&x)[16], int u, const typename CxOf<T>::type *tw) {
    using C = typename CxOf<T>::type;
    constexpr int R = 1 << Sched<N>::lr(I);
    constexpr int NP = Sched<N>::nprev(I);
    constexpr int Mi = NP / 16;
    constexpr int S = 16 / R;
#pragma unroll
    for (int s = 0; s < S; ++s) dft_reg<R, S, SIGN>(&x[s]);
    if constexpr (NP > R) {
        constexpr int NI = NP / R;
        const C *tws = tw + Sched<N>::twoff(I) + (u % Mi);
#pragma unroll
        for (int s = 0; s < S; ++s) {
#pragma unroll
            for (int k = 1; k < R; ++k) {
                const C w = tws[(k - 1) * NI + s * Mi];
                x[k * S + s] = SIGN < 0 ? cmul(x[k * S + s], w) : cmulc(x[k * S + s], w);
            }
        }
    }
}

// the transposed (DIT) stage: twiddles, then butterflies
template <typename T, int N, int I, int SIGN> __device__ __forceinline__ void dit_stage(typename CxOf<T>::type (&x)[16], int u, const typename CxOf<T>::type *tw) {
    using C = typename CxOf<T>::type;
    constexpr int R = 1 << Sched<N>::lr(I);
    constexpr int NP = Sched<N>::nprev(I);
    constexpr int Mi = NP / 16;
    constexpr int S = 16 / R;
    if constexpr (NP > R) {
        // the twiddles on the inputs are fused with the first butterfly level (pairs k, k + R/2):
        //   p = x_k w_k,  r = p + x_{k+R/2} w_{k+R/2} (four FMAs),  d = 2 p - r
        constexpr int NI = NP / R, H = R / 2;
        const C *tws = tw + Sched<N>::twoff(I) + (u % Mi);
#pragma unroll
        for (int s = 0; s < S; ++s) {
#pragma unroll
            for (int k = 0; k < H; ++k) {
                C p = x[k * S + s];
                if (k > 0) {
                    const C w = tws[(k - 1) * NI + s * Mi];
                    p = SIGN < 0 ? cmul(p, w) : cmulc(p, w);
                }
                const C b = x[(k + H) * S + s];
                C w2 = tws[(k + H - 1) * NI + s * Mi];
                if (SIGN > 0) w2.y = -w2.y;  // conjugate
                C r;
                r.x = fma(-w2.y, b.y, fma(w2.x, b.x, p.x));
                r.y = fma(w2.y, b.x, fma(w2.x, b.y, p.y));
                x[(k + H) * S + s] = mk<C>(fma((T)2, p.x, -r.x), fma((T)2, p.y, -r.y));
                x[k * S + s] = r;
            }
        }
#pragma unroll
        for (int s = 0; s < S; ++s) dft_reg<R, S, SIGN, C, false>(&x[s]);
    } else {
#pragma unroll
        for (int s = 0; s < S; ++s) dft_reg<R, S, SIGN>(&x[s]);
    }
}

// barrier over one group of a CTA (groups are independent pipelines that share only the twiddle table):
// gb = 0 means the CTA holds one group (plain __syncthreads), otherwise gb = (named barrier id) | (threads << 8)
__device__ __forceinline__ void gsync(int gb) {
    if ((gb & 0x03ffffff) == 0) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(gb & 15), "r"((gb & 0x03ffffff) >> 8) : "memory");
}

// gb flag: consecutive lanes hold consecutive u of one line (contiguous-axis kernels).  The exchange between
// two stages only moves data inside blocks of max(Mi) consecutive u (Mi = sub-transform length / 16), so when
// such a block lies inside a warp the group barrier shrinks to a __syncwarp
constexpr int GB_LANES_ARE_U = 1 << 30;
// strided kernels interleave TL lines in a warp (lane = u * TL + t): bits 26..29 hold log2(TL)
constexpr int GB_TL_SHIFT = 26;

// registers (layout of stage IA) -> shared memory -> registers (layout of stage IB)
struct NoGapWork {
    __device__ __forceinline__ void operator()() const {}
};
// `gap` runs between the writes and the reads, i.e. while the registers of x are free
template <typename T, int N, int IA, int IB, typename GAP = NoGapWork>
__device__ __forceinline__ void exchange(typename CxOf<T>::type (&x)[16], int u, typename CxOf<T>::type *sl, int gb, GAP gap = GAP()) {
    using C = typename CxOf<T>::type;
    constexpr int MiA = Sched<N>::nprev(IA) / 16, MiB = Sched<N>::nprev(IB) / 16;
    constexpr int SCOPE = MiA > MiB ? MiA : MiB;
    C *wa = sl + stage_base<N, IA>(u);
    const C *rb = sl + stage_base<N, IB>(u);
    const bool warp_local = (gb & GB_LANES_ARE_U) && (SCOPE << ((gb >> GB_TL_SHIFT) & 15)) <= 32;
    if (warp_local) __syncwarp();
    else gsync(gb);
#pragma unroll
    for (int q = 0; q < 16; ++q) wa[stage_delta<N, IA>(q)] = x[q];
    if (warp_local) __syncwarp();
    else gsync(gb);
    gap();
#pragma unroll
    for (int q = 0; q < 16; ++q) x[q] = rb[stage_delta<N, IB>(q)];
}

// `gap` is work that does not touch x (e.g. the scalars of the pointwise factor): it runs inside the last exchange,
// when x sits in shared memory and its registers are free (before the only stage when the line has one stage)
template <typename T, int N, int I, int SIGN> struct DifChain {
    using C = typename CxOf<T>::type;
    template <typename GAP = NoGapWork> static __device__ __forceinline__ void run(C (&x)[16], int u, const C *tw, C *sl, int gb, GAP gap = GAP()) {
        if constexpr (Sched<N>::M == 1) gap();
        dif_stage<T, N, I, SIGN>(x, u, tw);
        if constexpr (I + 1 < Sched<N>::M) {
            if constexpr (I + 2 == Sched<N>::M) exchange<T, N, I, I + 1>(x, u, sl, gb, gap);
            else exchange<T, N, I, I + 1>(x, u, sl, gb);
            DifChain<T, N, I + 1, SIGN>::run(x, u, tw, sl, gb, gap);
        }
    }
};
template <typename T, int N, int I, int SIGN> struct DitChain {  // runs stages I, I-1, ..., 0
    using C = typename CxOf<T>::type;
    static __device__ __forceinline__ void run(C (&x)[16], int u, const C *tw, C *sl, int gb) {
        dit_stage<T, N, I, SIGN>(x, u, tw);
        if constexpr (I > 0) {
            exchange<T, N, I, I - 1>(x, u, sl, gb);
            DitChain<T, N, I - 1, SIGN>::run(x, u, tw, sl, gb);
        }
    }
};

// exp(i a) in the working precision (evaluated in double)
template <typename T> __device__ __forceinline__ typename CxOf<T>::type expi(double a) {
    double s, c;
    sincos(a, &s, &c);
    return mk<typename CxOf<T>::type>((T)c, (T)s);
}

// exp(i a) for |a| <= 4 pi, evaluated in double without the library's general argument reduction: the plan stores
// potential angles reduced to [-pi, pi] (VREP_ANGLE), so a quadrant reduction j = rint(2a/pi), r = a - j pi/2 with a
// two-term pi/2 and the Taylor polynomials of sin and cos on [-pi/4, pi/4] (truncation error r^17/17! < 5e-17,
// r^18/18! < 3e-18) are enough.  About 24 FP64 instructions against about 45 for sincos().
template <typename T> __device__ __forceinline__ typename CxOf<T>::type expi_small(double a) {
    const double magic = 6755399441055744.0;  // 1.5 * 2^52: adding it rounds to the nearest integer, kept in the low bits
    const double jm = fma(a, 0.63661977236758134308, magic);
    const int j = __double2loint(jm);
    const double jd = jm - magic;
    double r = fma(jd, -1.57079632679489655800e+00, a);   // pi/2, leading 53 bits
    r = fma(jd, -6.12323399573676603587e-17, r);          // pi/2, next bits
    const double z = r * r;
    double sp = fma(z, -1.0 / 1307674368000.0, 1.0 / 6227020800.0);
    sp = fma(z, sp, -1.0 / 39916800.0);
    sp = fma(z, sp, 1.0 / 362880.0);
    sp = fma(z, sp, -1.0 / 5040.0);
    sp = fma(z, sp, 1.0 / 120.0);
    sp = fma(z, sp, -1.0 / 6.0);
    const double sn = fma(r * z, sp, r);
    double cp = fma(z, 1.0 / 20922789888000.0, -1.0 / 87178291200.0);
    cp = fma(z, cp, 1.0 / 479001600.0);
    cp = fma(z, cp, -1.0 / 3628800.0);
    cp = fma(z, cp, 1.0 / 40320.0);
    cp = fma(z, cp, -1.0 / 720.0);
    cp = fma(z, cp, 1.0 / 24.0);
    cp = fma(z, cp, -0.5);
    const double cs = fma(z, cp, 1.0);
    // quadrant j mod 4: (cos, sin) -> (cs, sn), (-sn, cs), (-cs, -sn), (sn, -cs)
    double c = (j & 1) ? sn : cs;
    double s = (j & 1) ? cs : sn;
    if ((j + 1) & 2) c = -c;
    if (j & 2) s = -s;
    return mk<typename CxOf<T>::type>((T)c, (T)s);
}

// Dirac kinetic factor on the DIF output (eq. 27-33 in the closed form
// U = cos(E tau) - i sin(E tau)/E (c alpha.pi + m c^2 beta), see the file header): the CC components of a k point
// are gathered into one thread through the exchange buffers, multiplied by the 2x2 / 4x4 unitary and scattered
// back.  line0 = exchange line of (component 0, this thread's t); comp_pitch = elements between components.
template <typename T, int CC, int U>
__device__ __forceinline__ void dirac_kinetic(typename CxOf<T>::type (&x)[16], int u, int c, typename CxOf<T>::type *sl, typename CxOf<T>::type *line0,
                                              int comp_pitch, int gb, const double *__restrict__ kv0, double sh0, double p1, double p2, double mass,
                                              double clight, double dt, double scale) {
    using C = typename CxOf<T>::type;
    constexpr int PP = 16 / CC;
    // all components of a k point into one thread: thread (c, u) takes the PP points
    // 16 u + c PP + i of every component
    C *me = sl + 17 * u;
    gsync(gb);
#pragma unroll
    for (int q = 0; q < 16; ++q) me[q] = x[q];
    gsync(gb);
    C y[CC][PP];
#pragma unroll
    for (int c2 = 0; c2 < CC; ++c2)
#pragma unroll
        for (int i = 0; i < PP; ++i) y[c2][i] = line0[c2 * comp_pitch + 17 * u + c * PP + i];
    const double mc2 = mass * clight * clight;
#pragma unroll
    for (int i = 0; i < PP; ++i) {
        const int q2 = c * PP + i;
        const double p0 = kv0[q2 * U + u] - sh0;
        const double pp = p0 * p0 + p1 * p1 + p2 * p2;
        const double E = sqrt(clight * clight * pp + mc2 * mc2);
        double sn, cs;
        sincos(E * dt, &sn, &cs);
        double sE = E > 0.0 ? sn / E : dt;
        cs *= scale;
        sE *= scale;
        const T fc = (T)cs;
        const T fm = (T)(sE * mc2);
        const T f0 = (T)(sE * clight * p0), f1 = (T)(sE * clight * p1), f2 = (T)(sE * clight * p2);
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
    gsync(gb);
#pragma unroll
    for (int q = 0; q < 16; ++q) x[q] = me[q];
}

// step average row n, component ax (0 when there is no table)
__device__ __forceinline__ double favg(const PassArgs &a, long long n, int ax) {
    return a.step_avg ? a.step_avg[n * a.ndim + ax] : 0.0;
}

__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// ------------------------------------------------------------------------------------------
// the kernel
//   STRIDED = false: lines are contiguous in memory; a tile is TL consecutive lines.
//   STRIDED = true : consecutive line elements are `inner` apart; a tile is TL adjacent lines
//                    (TL * sizeof(complex) contiguous bytes per line element).
//   PW: pointwise factor kind.  The Dirac kinds hold all components of the tile's lines in one CTA.
//   SIGN: sign of the DIF transform (-1: forward first, the kinetic sandwich; +1: inverse first,
//         the potential sandwich).
// Persistent CTAs: the grid is one wave (resident CTAs per SM x SM count); each CTA copies the twiddle
// table to shared memory once and then pulls tiles from a global counter until none are left, asking L2
// for the next tile's data while it works on the current one.
// ------------------------------------------------------------------------------------------
template <typename T, int N, bool STRIDED, int PW, int SIGN>
__global__ void __launch_bounds__(512, (sizeof(T) == 4 ? 2 : 1)) pass_kernel(const PassArgs a) {
    using C = typename CxOf<T>::type;
    constexpr int U = N / 16;
    constexpr int CC = PW == PW_KD2 ? 2 : (PW == PW_KD4 ? 4 : 1);
    constexpr int LAST = Sched<N>::M - 1;
    constexpr int TWN = Sched<N>::twoff(LAST);
    constexpr int TWP = (TWN + 7) & ~7;  // keep the exchange buffer 128-byte aligned
    constexpr bool TWG = twiddles_in_global<C, N>();
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const C *stw = TWG ? reinterpret_cast<const C *>(a.tw) : reinterpret_cast<const C *>(smem_raw);
    C *sm = reinterpret_cast<C *>(smem_raw) + (TWG ? 0 : TWP);

    const int TL = a.TL;
    // groups: G independent pipelines of GT = CC * TL * U threads each; a group owns an exchange buffer,
    // its per-line scalars and its scheduler mailbox, and synchronises with its own named barrier
    const int GT = a.GT;
    const int grp = threadIdx.x / GT;
    const int tid = threadIdx.x - grp * GT;
    const int gb = (a.G > 1 ? ((grp + 1) | (GT << 8)) : 0) | ((!STRIDED && (U >= 32 || 32 % U == 0)) ? GB_LANES_ARE_U : 0);
    int t, c, u;
    if (STRIDED) {
        t = tid % TL;
        const int cu = tid / TL;
        u = cu % U;
        c = cu / U;
    } else {
        u = tid % U;
        const int ct = tid / U;
        t = ct % TL;
        c = ct / TL;
    }
    C *smg = sm + (size_t)grp * a.gstride;                  // this group's region
    C *sl = smg + (c * TL + t) * a.pitch;
    C *lsc = smg + CC * TL * a.pitch;                       // per-line scalars [TL] (complex)
    int *snext = reinterpret_cast<int *>(lsc + TL);         // tile scheduler mailbox [2]

    // twiddles -> shared memory, once per CTA
    if constexpr (!TWG) {
        const C *__restrict__ gtw = reinterpret_cast<const C *>(a.tw);
        C *dst = reinterpret_cast<C *>(smem_raw);
        for (int i = threadIdx.x; i < TWN; i += blockDim.x) dst[i] = gtw[i];
    }
    if (tid == 0) snext[0] = (int)atomicAdd(&a.sched[0], 1u);
    __syncthreads();
    int wtile = snext[0];
    int parity = 1;

    while (wtile < a.ntiles) {
        // fetch the next tile index early so that its data can be requested from L2 ahead of time
        if (tid == 0) snext[parity] = (int)atomicAdd(&a.sched[0], 1u);

        long long tile;
        int comp;
        if (CC == 1) {
            comp = wtile % a.ncomp;
            tile = wtile / a.ncomp;
        } else {
            comp = c;
            tile = wtile;
        }
        const long long line = tile * TL + t;  // line index within a component
        long long base, estep;
        if (STRIDED) {
            const long long o = line / a.inner, i = line % a.inner;
            base = o * (long long)N * a.inner + i;
            estep = a.inner;
        } else {
            base = line * (long long)N;
            estep = 1;
        }
        C *__restrict__ gp = reinterpret_cast<C *>(a.psi) + (long long)comp * a.comp_stride + base;

        // line coordinates on the non-line axes: line = ia * rest1 + ib
        const int ib = (int)(line % a.rest1);
        const int ia = (int)(line / a.rest1);

        // per-line kinetic scalars
        if (PW == PW_KS && (a.kph1 || a.kph2)) {
            if (u == 0 && c == 0) {
                C s = mk<C>((T)1, (T)0);
                if (a.kph1) s = reinterpret_cast<const C *>(a.kph1)[ia];
                if (a.kph2) s = a.kph1 ? cmul(s, reinterpret_cast<const C *>(a.kph2)[ib]) : reinterpret_cast<const C *>(a.kph2)[ib];
                lsc[t] = s;
            }
        }

        C x[16];
        if (a.do_dif) {
#pragma unroll
            for (int q = 0; q < 16; ++q) x[q] = ld_stream(&gp[(long long)(u + q * U) * estep]);
        } else {
#pragma unroll
            for (int q = 0; q < 16; ++q) x[q] = ld_stream(&gp[(long long)(u * 16 + q) * estep]);
        }
        // angle of the homogeneous-field phase contributed by the non-line axes of this line:
        // (tau/2) sum_ax (Ebar_na + [full] Ebar_nb)[ax] * r_ax      (eq. 11, reading G12)
        auto other_axes_angle = [&](long long n_a, long long n_b, bool full) -> double {
            double ang = 0.0;
            if (a.oaxA >= 0) {
                double e = favg(a, n_a, a.oaxA);
                if (full) e += favg(a, n_b, a.oaxA);
                ang += e * a.half_dt * ((double)ia - (double)(a.nsz[a.oaxA] / 2)) * a.dxs[a.oaxA];
            }
            if (a.oaxB >= 0) {
                double e = favg(a, n_a, a.oaxB);
                if (full) e += favg(a, n_b, a.oaxB);
                ang += e * a.half_dt * ((double)ib - (double)(a.nsz[a.oaxB] / 2)) * a.dxs[a.oaxB];
            }
            return ang;
        };

        // potential phase in natural order at the stage-0 layout (thread u holds positions u + q U);
        // mode 1: the table is in natural order (1D); mode 2: gather from the permuted table
        auto natural_v = [&](int mode, long long n_a, long long n_b, bool full) {
            if constexpr (!STRIDED) {
                const int slot_u = mode == 2 ? a.revBinv[u] : u;
                double gl = 0.0, gother = 0.0;
                if (a.field_kind == 1) {
                    double e = favg(a, n_a, a.line_axis);
                    if (full) e += favg(a, n_b, a.line_axis);
                    gl = e * a.half_dt;
                    gother = other_axes_angle(n_a, n_b, full);
                }
#pragma unroll
                for (int q = 0; q < 16; ++q) {
                    C h;
                    const long long vi = line * (long long)N + q * U + slot_u;
                    if (a.vrep == VREP_TABLE) {
                        h = reinterpret_cast<const C *>(a.vtab)[vi];
                        if (full) h = cmul(h, h);
                    } else {
                        const double ang = reinterpret_cast<const double *>(a.vtab)[vi];
                        h = expi_small<T>(full ? 2.0 * ang : ang);
                    }
                    if (a.field_kind == 1) {
                        const double r = ((double)(u + q * U) - (double)(N / 2)) * a.dxs[a.line_axis];
                        h = cmul(h, expi<T>(-(gl * r + gother)));
                    }
                    x[q] = cmul(x[q], h);
                }
            }
        };

        // every thread learns the next tile and asks L2 for its share of that tile
        gsync(gb);  // also orders the twiddle copy (first tile) and lsc before their use
        const int ntile = snext[parity];
        if (ntile < a.ntiles) {
            long long tile2 = CC == 1 ? ntile / a.ncomp : ntile;
            const int comp2 = CC == 1 ? ntile % a.ncomp : c;
            const long long line2 = tile2 * TL + t;
            long long base2;
            if (STRIDED) {
                const long long o = line2 / a.inner, i = line2 % a.inner;
                base2 = o * (long long)N * a.inner + i;
            } else {
                base2 = line2 * (long long)N;
            }
            const C *gp2 = reinterpret_cast<const C *>(a.psi) + (long long)comp2 * a.comp_stride + base2;
            // one request per 32-byte sector
            constexpr int PER = 32 / (int)sizeof(C) < 1 ? 1 : 32 / (int)sizeof(C);
            const bool mine = STRIDED ? (t % PER == 0) : (u % PER == 0);
            if (mine) {
                if (a.do_dif) {
#pragma unroll
                    for (int q = 0; q < 16; ++q) prefetch_l2(&gp2[(long long)(u + q * U) * estep]);
                } else {
#pragma unroll
                    for (int q = 0; q < 16; ++q) prefetch_l2(&gp2[(long long)(u * 16 + q) * estep]);
                }
            }
        }

        for (int rep = 0; rep < a.nrep; ++rep) {
            const long long n = a.n0 + rep;
            if (a.pre_v && rep == 0) natural_v(a.pre_v, n, n, false);

            if (a.do_dif) DifChain<T, N, 0, SIGN>::run(x, u, stw, sl, gb);

            if (a.mid_on) {
                if constexpr (PW == PW_KS) {
                    const bool has_lsc = a.kph1 || a.kph2;
                    const C *__restrict__ k0 = reinterpret_cast<const C *>(a.kph0);
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        C f = k0[q * U + u];
                        if (has_lsc) f = cmul(f, lsc[t]);
                        x[q] = cmul(x[q], f);
                    }
                } else if constexpr (PW == PW_KD2 || PW == PW_KD4) {
                    // shift of the kinetic momentum: pi = k - q Abar_n (reading G16)
                    double sh[3] = {0.0, 0.0, 0.0};
                    if (a.field_kind == 2)
                        for (int ax = 0; ax < a.ndim; ++ax) sh[ax] = a.charge * favg(a, n, ax);
                    // non-line momenta of this line: the line axis is axis 0 here
                    double p1 = 0.0, p2 = 0.0;
                    if (a.ndim == 2) p1 = a.kv2[ib] - sh[1];
                    if (a.ndim == 3) {
                        p1 = a.kv1[ia] - sh[1];
                        p2 = a.kv2[ib] - sh[2];
                    }
                    dirac_kinetic<T, CC, U>(x, u, c, sl, smg + t * a.pitch, TL * a.pitch, gb, a.kv0, sh[0], p1, p2, a.mass, a.clight, a.dt, a.scale);
                }
            }

            if (a.do_dit) DitChain<T, N, LAST, -SIGN>::run(x, u, stw, sl, gb);

            if (a.post_v) {
                if (rep + 1 < a.nrep) natural_v(a.post_v, n, n + 1, true);
                else natural_v(a.post_v, n, n, false);
            }
        }

        if (!a.do_dit && a.unpermute) {
            // registers hold frequency revB[u] + U q at position 16 u + q: scatter to natural order
            C *wa = sl + padp(a.revB[u]);
            const C *rb = sl + padp(u);
            gsync(gb);
#pragma unroll
            for (int q = 0; q < 16; ++q) wa[lin_delta(q, U)] = x[q];
            gsync(gb);
#pragma unroll
            for (int q = 0; q < 16; ++q) x[q] = rb[lin_delta(q, U)];
        }
        if (a.do_dit || a.unpermute) {
#pragma unroll
            for (int q = 0; q < 16; ++q) st_stream(&gp[(long long)(u + q * U) * estep], x[q]);
        } else {
#pragma unroll
            for (int q = 0; q < 16; ++q) st_stream(&gp[(long long)(u * 16 + q) * estep], x[q]);
        }

        wtile = ntile;
        parity ^= 1;
        gsync(gb);  // everyone is done with the exchange buffer, lsc and the mailbox slot
    }

    // the last CTA to leave resets the scheduler for the next launch on this stream
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned done = atomicAdd(&a.sched[1], 1u);
        if (done == gridDim.x - 1) {
            a.sched[0] = 0u;
            a.sched[1] = 0u;
            __threadfence();
        }
    }
}

// host-side launcher, explicitly instantiated per (T, N) in sso_inst.cu
template <typename T, int N, bool STRIDED, int PW, int SIGN>
cudaError_t launch_pass(const PassArgs &a, unsigned threads, size_t smem, cudaStream_t st);

}  // namespace sso
