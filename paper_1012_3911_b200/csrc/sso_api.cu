// sso_api.cu -- the C ABI of include/sso.h: plan builder (radix schedule, twiddles, k grids,
// phase tables), the per-step pass schedule, and the small auxiliary kernels (table builders,
// norm reduction).  The pass kernel itself is in sso_pass.cuh.
//
// Pass schedule: 1D FFTs along different axes commute and the trailing
// potential half step of step n merges with the leading one of step n+1 (eq. 7
// applied twice), so a steady-state step costs
//   1D: 0 round trips of psi through HBM (one persistent CTA keeps the line in registers),
//   2D: 2 passes   [F_1^-1 V F_1]  [F_0 K F_0^-1]
//   3D: 4 passes   [F_2^-1 V F_2]  [F_1]  [F_0 K F_0^-1]  [F_1^-1]
// plus one opening [F_last V/2] and one closing [V/2 F_last^-1] pass per sso_step call.
#include <cuda.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/sso.h"
#include "sso_debug.h"
#include "sso_dispatch.h"
#include "sso_line1d_args.h"

// cluster size the 4096-point 1D line uses by default (0: the single-CTA kernel); chosen by measurement on B200
// points of a 1D line one CTA's registers hold (sso_line1d.cuh); longer Schroedinger lines go to a cluster
#define SSO_MAX_LINE_CTA 4096
#ifndef SSO_CLUSTER_AUTO_4096
#define SSO_CLUSTER_AUTO_4096 8
#endif

namespace sso {

// ---------------------------------------------------------------------------------------------
// auxiliary kernels
// ---------------------------------------------------------------------------------------------

template <typename T> struct Cx2;
template <> struct Cx2<float> { using type = float2; };
template <> struct Cx2<double> { using type = double2; };

// potential phase table: out[line*N + slot] = exp(-i V[line*N + nat(slot)] tau/2)  (eq. 11, delta = 1/2)
// or, for the angle representation, the angle -V tau/2 reduced to [-pi, pi).
template <typename T>
__global__ void build_vtab_kernel(const double *__restrict__ V, void *__restrict__ out, long long total, int N,
                                  const int *__restrict__ slot_nat, double half_dt, int vrep) {  // half_dt: tau/2 (half step) or tau (merged)
    using C = typename Cx2<T>::type;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const long long line = i / N;
        const int slot = (int)(i % N);
        const int nat = slot_nat ? slot_nat[slot] : slot;
        const double v = V ? V[line * N + nat] : 0.0;
        const double ang = -v * half_dt;
        if (vrep == VREP_TABLE) {
            double s, c;
            sincos(ang, &s, &c);
            C h;
            h.x = (T)c;
            h.y = (T)s;
            reinterpret_cast<C *>(out)[i] = h;
        } else {
            const double twopi = 6.283185307179586476925286766559;
            reinterpret_cast<double *>(out)[i] = ang - twopi * rint(ang / twopi);
        }
    }
}

// Schroedinger kinetic phase of one axis: out[i] = scale * exp(-i tau (k[i] - shift)^2 / (2 m))   (eq. 13)
template <typename T>
__global__ void build_kphase_kernel(const double *__restrict__ kv, void *__restrict__ out, int n, double tau, double mass,
                                    const double *__restrict__ step_avg, long long row, int ndim, int axis, double charge, double scale) {
    using C = typename Cx2<T>::type;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double shift = step_avg ? charge * step_avg[row * ndim + axis] : 0.0;
    const double p = kv[i] - shift;
    const double ang = -tau * p * p / (2.0 * mass);
    double s, c;
    sincos(ang, &s, &c);
    C h;
    h.x = (T)(c * scale);
    h.y = (T)(s * scale);
    reinterpret_cast<C *>(out)[i] = h;
}

// Dirac kinetic scalars of every k point (SSO_OPT_DIRAC_TABLE = 1) in the order the pass meets them ([slot along
// axis 0][the other axes in storage order]):  out = scale * (cos(E tau), sin(E tau)/E),
// E = sqrt(c^2 |k - sh|^2 + m^2 c^4), sh = q Abar_n   (eq. 32; closed form of eq. 33, see
// sso_sring.cuh; reading G16 for the shift)
__global__ void build_ktab_kernel(double2 *__restrict__ out, const double *__restrict__ kv0, const double *__restrict__ kv1,
                                  const double *__restrict__ kv2, long long total, long long inner, int rest1, double sh0, double sh1,
                                  double sh2, double mass, double clight, double dt, double scale) {
    const long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const double mc2 = mass * clight * clight;
    for (long long i = tid; i < total; i += (long long)gridDim.x * blockDim.x) {
        const long long s = i / inner, line = i % inner;
        const double p0 = kv0[s] - sh0;
        const double p1 = kv1 ? kv1[line / rest1] - sh1 : (kv2 ? kv2[line % rest1] - sh1 : 0.0);
        const double p2 = kv1 ? kv2[line % rest1] - sh2 : 0.0;
        const double E = sqrt(clight * clight * (p0 * p0 + p1 * p1 + p2 * p2) + mc2 * mc2);
        double sn, cs;
        sincos(E * dt, &sn, &cs);
        out[i] = make_double2(cs * scale, (E > 0.0 ? sn / E : dt) * scale);
    }
}

// homogeneous E field, all passes of one sso_step call at once (2D/3D).  For every lattice axis with a field
// component, row j of out[ax] (n[ax] complex entries) is the phase exp(-i (tau/2) c_j r) with
//   j = 0        c = Ebar[n0]                      opening half step        (natural order)
//   0 < j < ns   c = Ebar[n0+j-1] + Ebar[n0+j]     merged half steps        (last axis: permuted slots)
//   j = ns       c = Ebar[n0+ns-1]                 closing half step        (natural order)
// (eq. 11 with the step averages of reading G12; merging is PAPER.md:71 eq. 7 applied twice).
struct ERowsArgs {
    void *out[3];
    int n[3];
    double dx[3];
    const int *slot_nat_last;
    const double *step_avg;
    long long n0, ns;
    int ndim;
    double half_dt;
};
template <typename T> __global__ void build_erows_kernel(const ERowsArgs e) {
    using C = typename Cx2<T>::type;
    const int ax = blockIdx.y;
    if (ax >= e.ndim || !e.out[ax]) return;
    const int n = e.n[ax];
    const long long total = (e.ns + 1) * n;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const long long j = idx / n;
        const int i = (int)(idx % n);
        double c;
        if (j == 0) c = e.step_avg[e.n0 * e.ndim + ax];
        else if (j == e.ns) c = e.step_avg[(e.n0 + e.ns - 1) * e.ndim + ax];
        else c = e.step_avg[(e.n0 + j - 1) * e.ndim + ax] + e.step_avg[(e.n0 + j) * e.ndim + ax];
        const int nat = (ax == e.ndim - 1 && j > 0 && j < e.ns) ? e.slot_nat_last[i] : i;
        const double r = ((double)nat - (double)(n / 2)) * e.dx[ax];
        double sn, cs;
        sincos(-c * e.half_dt * r, &sn, &cs);
        C h;
        h.x = (T)cs;
        h.y = (T)sn;
        reinterpret_cast<C *>(e.out[ax])[idx] = h;
    }
}

// Position-space vector-potential factor of the Dirac step (eq. 18a; 168-184 eq. 23/24; 188-198
// eq. 25/26; 236 eq. 34): at every lattice point  psi <- (cos a + i (sum_i a_i alpha_i / a) sin a) psi,
// a_i = coef * A_i(r), coef = delta tau q c, a = |a|.  With the Dirac representation (eq. 16)
// sum_i a_i alpha_i = [[0, sigma.a], [sigma.a, 0]]; the two-component forms are its {1,4} block (eq. 17, reading G7).
// One thread per point holds all components; streaming, one read and one write of psi.
template <typename T, int CC>
__global__ void apos_rotate_kernel(void *__restrict__ psi_, const double *__restrict__ A, long long npts, int ndim, double coef) {
    using C = typename Cx2<T>::type;
    C *psi = reinterpret_cast<C *>(psi_);
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < npts; j += (long long)gridDim.x * blockDim.x) {
        const double a1 = coef * A[j];
        const double a2 = ndim > 1 ? coef * A[npts + j] : 0.0;
        const double a3 = ndim > 2 ? coef * A[2 * npts + j] : 0.0;
        const double an = sqrt(a1 * a1 + a2 * a2 + a3 * a3);
        if (an == 0.0) continue;
        double sn, cs;
        sincos(an, &sn, &cs);
        const double s = sn / an;
        const T fc = (T)cs, f1 = (T)(s * a1), f2 = (T)(s * a2), f3 = (T)(s * a3);
        // i (x + i y) = -y + i x
        if (CC == 2) {
            const C p0 = psi[j], p1 = psi[npts + j];
            // (a1 - i a2) p1 and (a1 + i a2) p0
            const T h0x = f1 * p1.x + f2 * p1.y, h0y = f1 * p1.y - f2 * p1.x;
            const T h1x = f1 * p0.x - f2 * p0.y, h1y = f1 * p0.y + f2 * p0.x;
            psi[j] = C{fc * p0.x - h0y, fc * p0.y + h0x};
            psi[npts + j] = C{fc * p1.x - h1y, fc * p1.y + h1x};
        } else {
            const C u0 = psi[j], u1 = psi[npts + j], l0 = psi[2 * npts + j], l1 = psi[3 * npts + j];
            // sigma.a (v0, v1) = (a3 v0 + (a1 - i a2) v1, (a1 + i a2) v0 - a3 v1)
            const T g0x = f3 * l0.x + f1 * l1.x + f2 * l1.y, g0y = f3 * l0.y + f1 * l1.y - f2 * l1.x;  // (sigma.a l)_0
            const T g1x = f1 * l0.x - f2 * l0.y - f3 * l1.x, g1y = f1 * l0.y + f2 * l0.x - f3 * l1.y;  // (sigma.a l)_1
            const T k0x = f3 * u0.x + f1 * u1.x + f2 * u1.y, k0y = f3 * u0.y + f1 * u1.y - f2 * u1.x;  // (sigma.a u)_0
            const T k1x = f1 * u0.x - f2 * u0.y - f3 * u1.x, k1y = f1 * u0.y + f2 * u0.x - f3 * u1.y;  // (sigma.a u)_1
            psi[j] = C{fc * u0.x - g0y, fc * u0.y + g0x};
            psi[npts + j] = C{fc * u1.x - g1y, fc * u1.y + g1x};
            psi[2 * npts + j] = C{fc * l0.x - k0y, fc * l0.y + k0x};
            psi[3 * npts + j] = C{fc * l1.x - k1y, fc * l1.y + k1x};
        }
    }
}

// Dirac kinetic factor as a kernel of its own, for lines whose components do not fit one CTA together (ncomp * n_0 >
// 8192): psi is in momentum space on every axis (axis 0 in network order, as the transform-only passes leave it), one
// thread per k point holds all components and applies U = cos(E tau) - i (sin(E tau)/E) (c alpha.pi + m c^2 beta)
// (eq. 27-33 in the closed form of sso_sring.cuh; pi = k - q Abar_n, reading G16), times 1/Ntot.
template <typename T, int CC>
__global__ void dirac_pointwise_kernel(void *__restrict__ psi_, long long npts, long long inner, int rest1, const double *__restrict__ k0pos,
                                       const double *__restrict__ kv1, const double *__restrict__ kv2, double sh0, double sh1, double sh2,
                                       double mass, double clight, double dt, double scale) {
    using C = typename Cx2<T>::type;
    C *psi = reinterpret_cast<C *>(psi_);
    const double mc2 = mass * clight * clight;
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < npts; j += (long long)gridDim.x * blockDim.x) {
        const long long i0 = j / inner, line = j % inner;
        const double p0 = k0pos[i0] - sh0;
        const double p1 = kv1 ? kv1[line / rest1] - sh1 : (kv2 ? kv2[line % rest1] - sh1 : 0.0);
        const double p2 = kv1 ? kv2[line % rest1] - sh2 : 0.0;
        const double E = sqrt(clight * clight * (p0 * p0 + p1 * p1 + p2 * p2) + mc2 * mc2);
        double sn, cs;
        sincos(E * dt, &sn, &cs);
        const double sE = (E > 0.0 ? sn / E : dt) * scale;
        cs *= scale;
        const T fc = (T)cs, fm = (T)(sE * mc2), f0 = (T)(sE * clight * p0), f1 = (T)(sE * clight * p1), f2 = (T)(sE * clight * p2);
        // out = cs psi - i sE H psi ;  (-i)(a + i b) = b - i a
        if (CC == 2) {
            const C a0 = psi[j], a1 = psi[npts + j];
            // H psi_0 = mc2 a0 + c (p0 - i p1) a1 ; H psi_1 = c (p0 + i p1) a0 - mc2 a1
            const T h0x = fm * a0.x + f0 * a1.x + f1 * a1.y, h0y = fm * a0.y + f0 * a1.y - f1 * a1.x;
            const T h1x = f0 * a0.x - f1 * a0.y - fm * a1.x, h1y = f0 * a0.y + f1 * a0.x - fm * a1.y;
            psi[j] = C{fc * a0.x + h0y, fc * a0.y - h0x};
            psi[npts + j] = C{fc * a1.x + h1y, fc * a1.y - h1x};
        } else {
            const C a0 = psi[j], a1 = psi[npts + j], a2 = psi[2 * npts + j], a3 = psi[3 * npts + j];
            // sigma.p (v0, v1) = (p2 v0 + (p0 - i p1) v1, (p0 + i p1) v0 - p2 v1);  H psi = (mc2 u + c sigma.p l, c sigma.p u - mc2 l)
            const T h0x = fm * a0.x + f2 * a2.x + f0 * a3.x + f1 * a3.y, h0y = fm * a0.y + f2 * a2.y + f0 * a3.y - f1 * a3.x;
            const T h1x = fm * a1.x + f0 * a2.x - f1 * a2.y - f2 * a3.x, h1y = fm * a1.y + f0 * a2.y + f1 * a2.x - f2 * a3.y;
            const T h2x = f2 * a0.x + f0 * a1.x + f1 * a1.y - fm * a2.x, h2y = f2 * a0.y + f0 * a1.y - f1 * a1.x - fm * a2.y;
            const T h3x = f0 * a0.x - f1 * a0.y - f2 * a1.x - fm * a3.x, h3y = f0 * a0.y + f1 * a0.x - f2 * a1.y - fm * a3.y;
            psi[j] = C{fc * a0.x + h0y, fc * a0.y - h0x};
            psi[npts + j] = C{fc * a1.x + h1y, fc * a1.y - h1x};
            psi[2 * npts + j] = C{fc * a2.x + h2y, fc * a2.y - h2x};
            psi[3 * npts + j] = C{fc * a3.x + h3y, fc * a3.y - h3x};
        }
    }
}

// norm: partial sums of |psi|^2 in double, warp-shuffle tree, fixed order (deterministic)
template <typename T>
__global__ void norm_partial_kernel(const void *__restrict__ psi, long long count, double *__restrict__ partial) {
    using C = typename Cx2<T>::type;
    const C *p = reinterpret_cast<const C *>(psi);
    double acc = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
        const C v = p[i];
        acc += (double)v.x * (double)v.x + (double)v.y * (double)v.y;
    }
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    __shared__ double wsum[32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) wsum[w] = acc;
    __syncthreads();
    if (w == 0) {
        acc = lane < (int)(blockDim.x >> 5) ? wsum[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
        if (lane == 0) partial[blockIdx.x] = acc;
    }
}
__global__ void norm_final_kernel(const double *__restrict__ partial, int n, double vol, double *__restrict__ out) {
    double acc = 0.0;
    for (int i = threadIdx.x; i < n; i += 32) acc += partial[i];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if (threadIdx.x == 0) *out = acc * vol;
}


// ---- observables (section V.2) ---------------------------------------------------------------
// block-level sum of NV doubles per thread: warp-shuffle tree, then one warp over the per-warp sums; fixed order.
// On return thread 0 holds the sums in acc.
template <int NV> __device__ __forceinline__ void block_sum(double (&acc)[NV]) {
    __shared__ double wsum[NV][32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        for (int o = 16; o > 0; o >>= 1) acc[v] += __shfl_down_sync(0xffffffffu, acc[v], o);
        if (lane == 0) wsum[v][w] = acc[v];
    }
    __syncthreads();
    if (w == 0) {
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            double t = lane < (int)(blockDim.x >> 5) ? wsum[v][lane] : 0.0;
            for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
            acc[v] = t;
        }
    }
}
template <int NV> __device__ __forceinline__ void block_sum_store(double (&acc)[NV], double *__restrict__ partial) {
    block_sum<NV>(acc);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int v = 0; v < NV; ++v) partial[v * gridDim.x + blockIdx.x] = acc[v];
    }
}
// out[v] = scale * sum_b partial[v][b], one warp per value
__global__ void reduce_final_kernel(const double *__restrict__ partial, int nblocks, int nv, double scale, double *__restrict__ out) {
    const int v = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (v >= nv) return;
    double acc = 0.0;
    for (int i = lane; i < nblocks; i += 32) acc += partial[v * nblocks + i];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if (lane == 0) out[v] = acc * scale;
}

// <a|b> = sum conj(a) b: the autocorrelation function chi(t) of PAPER.md:359 eq. 40 for a = Psi(0), b = Psi(t)
template <typename T>
__global__ void overlap_partial_kernel(const void *__restrict__ a_, const void *__restrict__ b_, long long count, double *__restrict__ partial) {
    using C = typename Cx2<T>::type;
    const C *a = reinterpret_cast<const C *>(a_), *b = reinterpret_cast<const C *>(b_);
    double acc[2] = {0.0, 0.0};
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
        const C u = a[i], v = b[i];
        acc[0] += (double)u.x * (double)v.x + (double)u.y * (double)v.y;
        acc[1] += (double)u.x * (double)v.y - (double)u.y * (double)v.x;
    }
    block_sum_store<2>(acc, partial);
}

// sum over the lattice of w_a(i_a) |psi(i)|^2 for every axis a, the density summed over the components.
// Position expectation: tab = NULL, w_a(i) = (i - n_a/2) dx_a (grid of reading G14); momentum expectation: psi holds
// the transform in network order on every axis and w_a(i) = tab[a][i], the momentum at network position i.
struct AxisWeights {
    const double *tab[3];
    int n[3];
    double dx[3];
    int ndim, ncomp;
    long long npts;
};
template <typename T> __global__ void weighted_density_partial_kernel(const void *__restrict__ psi_, const AxisWeights aw, double *__restrict__ partial) {
    using C = typename Cx2<T>::type;
    const C *psi = reinterpret_cast<const C *>(psi_);
    double acc[3] = {0.0, 0.0, 0.0};
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < aw.npts; j += (long long)gridDim.x * blockDim.x) {
        double d = 0.0;
        for (int c = 0; c < aw.ncomp; ++c) {
            const C v = psi[(long long)c * aw.npts + j];
            d += (double)v.x * (double)v.x + (double)v.y * (double)v.y;
        }
        long long rem = j;
        for (int a = aw.ndim - 1; a >= 0; --a) {
            const int ia = (int)(rem % aw.n[a]);
            rem /= aw.n[a];
            const double wgt = aw.tab[a] ? aw.tab[a][ia] : ((double)ia - (double)(aw.n[a] / 2)) * aw.dx[a];
            acc[a] += wgt * d;
        }
    }
    block_sum_store<3>(acc, partial);
}

// chi~(E) = sum_n chi(t_n) (1 - cos(2 pi t_n/T)) exp(i t_n E) dts, t_n = n dts, T = nt dts (eq. 41; the
// integral as the sum over the samples, reading G30).  One block per energy.
__global__ void spectrum_kernel(const double2 *__restrict__ chi, long long nt, double dts, const double *__restrict__ E, double2 *__restrict__ out) {
    const double e = E[blockIdx.x];
    double acc[2] = {0.0, 0.0};
    for (long long n = threadIdx.x; n < nt; n += blockDim.x) {
        const double wdw = 1.0 - cospi(2.0 * (double)n / (double)nt);  // t_n / T = n / nt
        double sn, cs;
        sincos((double)n * dts * e, &sn, &cs);
        const double2 c = chi[n];
        acc[0] += wdw * (c.x * cs - c.y * sn);
        acc[1] += wdw * (c.x * sn + c.y * cs);
    }
    block_sum<2>(acc);
    if (threadIdx.x == 0) out[blockIdx.x] = make_double2(acc[0] * dts, acc[1] * dts);
}

// acc += psi (1 - cos(2 pi t/T)) exp(i E t) dts, one term of PAPER.md:367 eq. 42; acc is complex128 whatever psi is
template <typename T>
__global__ void filter_accumulate_kernel(double2 *__restrict__ acc, const void *__restrict__ psi_, long long count, double t, double Ttot, double E, double dts) {
    using C = typename Cx2<T>::type;
    const C *psi = reinterpret_cast<const C *>(psi_);
    double wi, wr;
    sincos(E * t, &wi, &wr);
    const double wdw = (1.0 - cospi(2.0 * t / Ttot)) * dts;
    wr *= wdw;
    wi *= wdw;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
        const C v = psi[i];
        double2 a = acc[i];
        a.x += wr * (double)v.x - wi * (double)v.y;
        a.y += wr * (double)v.y + wi * (double)v.x;
        acc[i] = a;
    }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------

static LaunchFn find_launch(int precision, int N, int strided, int pw, int sign) {
    switch (N) {
#define SSO_CASE(NN) \
    case NN:         \
        return precision == SSO_C64 ? sso_lookup_f32_##NN(strided, pw, sign) : sso_lookup_f64_##NN(strided, pw, sign);
        SSO_FOR_EACH_N(SSO_CASE)
#undef SSO_CASE
    }
    return nullptr;
}

static SRingLaunchFn find_sring(int precision, int N, int mode) {
    switch (N) {
#define SSO_CASE(NN) \
    case NN:         \
        return precision == SSO_C64 ? sso_sring_lookup_f32_##NN(mode) : sso_sring_lookup_f64_##NN(mode);
        SSO_FOR_EACH_N(SSO_CASE)
#undef SSO_CASE
    }
    return nullptr;
}

static Line1dLaunchFn find_line1d(int precision, int N) {
    switch (N) {
#define SSO_CASE(NN) \
    case NN:         \
        return precision == SSO_C64 ? sso_line1d_lookup_f32_##NN() : sso_line1d_lookup_f64_##NN();
        SSO_FOR_EACH_N(SSO_CASE)
#undef SSO_CASE
    }
    return nullptr;
}

static Line1dClusterLaunchFn find_line1d_cluster(int precision, int M, int cs) {
    switch (M) {
#define SSO_CASE(NN) \
    case NN:         \
        return precision == SSO_C64 ? sso_line1d_cluster_lookup_f32_##NN(cs) : sso_line1d_cluster_lookup_f64_##NN(cs);
        SSO_FOR_EACH_N(SSO_CASE)
#undef SSO_CASE
    }
    return nullptr;
}

static RingLaunchFn find_ring(int precision, int N, int mode, int maxt) {
    switch (N) {
#define SSO_CASE(NN) \
    case NN:         \
        return precision == SSO_C64 ? sso_ring_lookup_f32_##NN(mode, maxt) : sso_ring_lookup_f64_##NN(mode, maxt);
        SSO_FOR_EACH_N(SSO_CASE)
#undef SSO_CASE
    }
    return nullptr;
}

// the radix schedule of sso_pass.cuh's Sched<N>, at run time
struct HostSched {
    int m;
    int lr[8];
    explicit HostSched(int N) {
        int LOG = 0;
        while ((1 << LOG) < N) ++LOG;
        const int REM = LOG - 4;
        m = 1 + (REM + 3) / 4;
        for (int i = 0; i < m; ++i) lr[i] = (i == m - 1) ? 4 : (i == 0 ? REM - 4 * (m - 2) : 4);
    }
};

// frequency index held at network position p after the DIF stages: p = sum_i k_i N_i  ->  k_1 + R_1 k_2 + R_1 R_2 k_3 + ...
static int freq_of_pos(int N, int p) {
    HostSched s(N);
    int Ni = N, w = 1, f = 0;
    for (int i = 0; i < s.m; ++i) {
        const int R = 1 << s.lr[i];
        Ni /= R;
        const int k = (p / Ni) % R;
        f += k * w;
        w *= R;
    }
    return f;
}

// bytes of shared memory the kernels give the twiddle blocks of an n-point line: none for the longest lines, whose
// kernels read them from global memory (sso_pass.cuh, twiddles_in_global)
static int twiddle_count_padded(int N);
static size_t twiddle_smem_bytes(int n, size_t esz) {
    const size_t tw = (size_t)twiddle_count_padded(n) * esz;
    return (tw + (size_t)(n + n / 16) * esz > (size_t)200 * 1024) ? 0 : tw;
}

// entries of the twiddle blocks of all non-final stages, padded as in the kernel (TWP)
static int twiddle_count_padded(int N) {
    HostSched s(N);
    int NP = N, cnt = 0;
    for (int i = 0; i + 1 < s.m; ++i) {
        const int R = 1 << s.lr[i];
        cnt += (R - 1) * (NP / R);
        NP /= R;
    }
    return (cnt + 7) & ~7;
}

// Twiddle blocks of an n-point line, evaluated in long double and rounded once to the plan's precision.  Stage i of
// the radix schedule (sub-transform length NP, radix R, NI = NP/R) stores w_NP^(l k) = exp(-2 pi i l k / NP) at
// [k-1][l], k = 1..R-1, l < NI; the last stage needs none.
static cudaError_t upload_twiddles(int n, int precision, void **dev) {
    std::vector<long double> twr, twi;
    HostSched hs(n);
    int NP = n;
    for (int i = 0; i + 1 < hs.m; ++i) {
        const int R = 1 << hs.lr[i], NI = NP / R;
        for (int k = 1; k < R; ++k)
            for (int l = 0; l < NI; ++l) {
                const long double ang = -2.0L * 3.14159265358979323846264338327950288L * (long double)((long long)l * k % NP) / (long double)NP;
                twr.push_back(cosl(ang));
                twi.push_back(sinl(ang));
            }
        NP = NI;
    }
    if (twr.empty()) {
        twr.push_back(1.0L);
        twi.push_back(0.0L);
    }
    const size_t cnt = twr.size();
    const size_t esz = precision == SSO_C128 ? 16 : 8;
    cudaError_t e = cudaMalloc(dev, cnt * esz);
    if (e != cudaSuccess) return e;
    if (precision == SSO_C128) {
        std::vector<double2> tw(cnt);
        for (size_t t = 0; t < cnt; ++t) tw[t] = make_double2((double)twr[t], (double)twi[t]);
        return cudaMemcpy(*dev, tw.data(), cnt * esz, cudaMemcpyHostToDevice);
    }
    std::vector<float2> tw(cnt);
    for (size_t t = 0; t < cnt; ++t) tw[t] = make_float2((float)twr[t], (float)twi[t]);
    return cudaMemcpy(*dev, tw.data(), cnt * esz, cudaMemcpyHostToDevice);
}

struct Axis {
    int n = 0;
    double dx = 0.0;
    std::vector<double> k_nat;     // k_j in DFT order (Nyquist negative, reading G14)
    std::vector<int> pos_freq;     // network position -> frequency index
    std::vector<int> slot_nat;     // permuted-layout slot (q U + B') -> natural index
    void *tw = nullptr;            // device complex[n]
    int *d_revB = nullptr;         // device int[n/16]
    int *d_revBinv = nullptr;      // device int[n/16]
    int *d_slot_nat = nullptr;     // device int[n]
    double *d_kv = nullptr;        // device double[n]: k in the layout this axis uses in the kinetic pass
    void *d_kph = nullptr;         // device complex[n]: Schroedinger phase table in the same layout
    double *d_kpos = nullptr;      // device double[n]: k at network position p (sso_expect_momentum)
};

}  // namespace sso

using namespace sso;

struct sso_plan {
    int ndim = 0, ncomp = 1, precision = SSO_C128;
    Axis ax[3];
    long long npts = 1;
    double dt = 0.0;
    double mass = 1.0, clight = 137.036, charge = -1.0;
    int field_kind = SSO_FIELD_NONE;
    std::vector<double> h_avg;  // [nvals][ndim]
    long long nvals = 0;
    double *d_avg = nullptr;
    bool e_along_last = false;  // some row has a nonzero E component along the last axis
    long long tindex = 0;
    void *d_vtab = nullptr;   // exp(-i V tau/2) in natural order (1D, opening and closing passes)
    void *d_vfull = nullptr;  // exp(-i V tau) in the permuted slot order of the last axis (2D/3D steady state)
    void *d_erow[3] = {nullptr, nullptr, nullptr};  // field phase rows of the current call (build_erows_kernel)
    size_t erow_cap[3] = {0, 0, 0};
    bool e_axis_on[3] = {false, false, false};
    CUtensorMap tmap[3];             // strided-axis tile maps (sso_sring.cuh), valid for tmap_psi / tmap_tl
    const void *tmap_psi[3] = {nullptr, nullptr, nullptr};
    int tmap_tl[3] = {0, 0, 0};
    int vrep = VREP_TABLE;
    bool kph_valid = false;
    double *d_apos = nullptr; // step-averaged position-dependent A(r), [ndim][npts], or NULL (sso_set_vector_potential)
    void *d_ktab = nullptr;   // Dirac kinetic scalars per k point (SSO_OPT_DIRAC_TABLE = 1), else NULL
    bool ktab_valid = false;  // the table is current (plans without SSO_FIELD_A only; with it it changes every step)
    int opt_dirac_table = 0;
    int opt_tile_order = 0;   // SSO_OPT_TILE_ORDER
    int opt_cluster = 0;      // SSO_OPT_CLUSTER_1D
    mutable int cl_fits[2] = {-1, -1};  // can this device co-schedule a cluster of 4 / 8 CTAs of the 1D kernel: -1 not asked yet
    struct ClusterLine {      // tables of the cluster version of the 1D kernel, built on first use for (cs, M = N / cs)
        int cs = 0, M = 0;
        void *tw = nullptr;       // twiddle blocks of the M-point transform
        void *tcl = nullptr;      // cluster twiddles [cs][cs-1][M/cs]
        double *kv = nullptr;     // k of the frequencies k1 + cs k2, [cs][M], rows in slot order
        void *kph = nullptr;      // kinetic phases of those frequencies
        bool kph_valid = false;
    } cl;
    int opt_tl_middle = 0;    // SSO_OPT_LINES_PER_TILE_MIDDLE
    int opt_tl_contig = 0, opt_tl_strided = 0, opt_groups = 0, opt_ring = 0, opt_maxt = 0, opt_sring = 0;
    int device = 0, num_sms = 0;  // the device the plan was created on, its SM count
    size_t smem_optin = 0;        // largest dynamic shared memory a CTA may opt in to on that device
    struct ProfEvent {
        int kind;
        cudaEvent_t a, b;
    };
    std::vector<ProfEvent> *prof = nullptr;  // non-NULL while sso_profile_step brackets every launch with events
    bool v_valid = true;          // false between a change of the potential representation and the next sso_set_potential
    double *d_partial = nullptr, *d_norm = nullptr;  // reductions: [4][NORM_BLOCKS] partial sums, [4] results
    void *d_scratch = nullptr;    // psi-sized work buffer of sso_expect_momentum (allocated on first use)
    unsigned *d_sched = nullptr;  // tile scheduler of the pass kernel (zero between launches)
    void *d_hostbuf = nullptr;
    std::string err;
    size_t esize() const { return precision == SSO_C64 ? 8 : 16; }
};

static thread_local std::string g_create_err;
static const int NORM_BLOCKS = 592;

static int fail(sso_plan *p, int code, const std::string &msg) {
    if (p) p->err = msg;
    else g_create_err = msg;
    return code;
}
static int cuda_fail(sso_plan *p, cudaError_t e, const char *what) {
    return fail(p, SSO_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CK(call)                                                  \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return cuda_fail(plan, e_, #call); \
    } while (0)

template <typename V> static cudaError_t upload(void **dst, const std::vector<V> &src) {
    cudaError_t e = cudaMalloc(dst, src.size() * sizeof(V));
    if (e != cudaSuccess) return e;
    return cudaMemcpy(*dst, src.data(), src.size() * sizeof(V), cudaMemcpyHostToDevice);
}

static int pass_status(sso_plan *plan, const char *what, cudaError_t e) {
    if (e != cudaSuccess) return cuda_fail(plan, e, what);
    return SSO_OK;
}

// brackets the launches of one pass with CUDA events while the plan is being profiled (sso_profile_step)
struct PassTimer {
    sso_plan *p;
    cudaStream_t st;
    long idx = -1;
    PassTimer(sso_plan *plan, int kind, cudaStream_t stream) : p(plan), st(stream) {
        if (!p->prof) return;
        sso_plan::ProfEvent e{kind, nullptr, nullptr};
        if (cudaEventCreate(&e.a) != cudaSuccess || cudaEventCreate(&e.b) != cudaSuccess) return;
        cudaEventRecord(e.a, st);
        p->prof->push_back(e);
        idx = (long)p->prof->size() - 1;
    }
    ~PassTimer() {
        if (idx >= 0) cudaEventRecord((*p->prof)[(size_t)idx].b, st);
    }
};

static bool is_pow2(long long v) { return v > 0 && (v & (v - 1)) == 0; }
static int ilog2ll(long long v) {
    int l = 0;
    while ((1LL << (l + 1)) <= v) ++l;
    return l;
}

// which layout the kinetic tables of axis a use: axis 0 is the kinetic-sandwich axis (permuted slots),
// the middle axis of a 3D lattice is stored in network order, the last axis of a >=2D lattice is natural
static void kinetic_layout(const sso_plan *p, int a, std::vector<double> &kv) {
    const Axis &A = p->ax[a];
    kv.resize(A.n);
    if (a == 0) {
        for (int s = 0; s < A.n; ++s) kv[s] = A.k_nat[A.slot_nat[s]];
    } else if (a == 1 && p->ndim == 3) {
        for (int q = 0; q < A.n; ++q) kv[q] = A.k_nat[A.pos_freq[q]];
    } else {
        kv = A.k_nat;
    }
}

// Device tables whose shape depends on the plan's configuration (the twiddle/frequency tables of the 1D cluster kernel,
// the Dirac kinetic table of SSO_OPT_DIRAC_TABLE = 1).  Every call that changes the configuration -- sso_plan_create,
// sso_set_option, sso_set_field, sso_set_vector_potential -- (re)allocates them here, so that sso_step itself only
// enqueues kernels and can be captured into a CUDA graph on its very first call.
namespace {
int prepare_config_tables(sso_plan *plan);
}

extern "C" {

const char *sso_version(void) { return "sso 0.1 (sm_100a)"; }

int sso_debug_layout(int n, int *pos_freq, int *slot_nat) {
    if (!pos_freq || !slot_nat || !is_pow2(n) || n < SSO_MIN_AXIS || n > SSO_MAX_AXIS) return SSO_ERR_INVALID;
    const int U = n / 16;
    for (int p = 0; p < n; ++p) {
        const int f = freq_of_pos(n, p);
        pos_freq[p] = f;
        slot_nat[(p % 16) * U + p / 16] = f;
    }
    return SSO_OK;
}

const char *sso_last_error(const sso_plan *plan) { return plan ? plan->err.c_str() : g_create_err.c_str(); }

int sso_plan_create(sso_plan **out, int ndim, const int64_t *sizes, const double *dx, double dt, int ncomp, int precision) {
    sso_plan *plan = nullptr;  // for CK / fail before the plan exists
    if (!out) return fail(nullptr, SSO_ERR_INVALID, "out is NULL");
    *out = nullptr;
    if (!sizes || !dx) return fail(nullptr, SSO_ERR_INVALID, "sizes or dx is NULL");
    if (ndim < 1 || ndim > 3) return fail(nullptr, SSO_ERR_INVALID, "ndim must be 1, 2 or 3");
    if (precision != SSO_C64 && precision != SSO_C128) return fail(nullptr, SSO_ERR_INVALID, "precision must be SSO_C64 or SSO_C128");
    if (ncomp != 1 && ncomp != 2 && ncomp != 4) return fail(nullptr, SSO_ERR_INVALID, "ncomp must be 1, 2 or 4");
    if (ncomp == 2 && ndim == 3) return fail(nullptr, SSO_ERR_INVALID, "a 2-component Dirac spinor exists in 1 and 2 dimensions only");
    if (!isfinite(dt)) return fail(nullptr, SSO_ERR_INVALID, "dt must be finite");
    for (int a = 0; a < ndim; ++a) {
        if (!(dx[a] > 0.0) || !isfinite(dx[a])) return fail(nullptr, SSO_ERR_INVALID, "dx must be positive and finite");
        if (!is_pow2(sizes[a])) return fail(nullptr, SSO_ERR_INVALID, "sizes must be powers of two");
        // a 1D Schroedinger line may be spread over a thread-block cluster (sso_line1d_cluster.cuh)
        const int64_t nmax = (ndim == 1 && ncomp == 1) ? SSO_MAX_AXIS_1D : SSO_MAX_AXIS;
        if (sizes[a] < SSO_MIN_AXIS || sizes[a] > nmax)
            return fail(nullptr, SSO_ERR_UNSUPPORTED, "axis length outside [16, 8192] (1D Schroedinger lattices: [16, 32768])");
    }
    if (ndim == 1 && ncomp > 1 && (long long)ncomp * (sizes[0] / 16) > 512)
        return fail(nullptr, SSO_ERR_UNSUPPORTED, "1D Dirac plans need ncomp * sizes[0] <= 8192 (all components of the line share one CTA)");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, SSO_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    }
    int dev = 0, num_sms = 0, optin = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess || num_sms < 1) {
        cudaGetLastError();
        return fail(nullptr, SSO_ERR_CUDA, "cannot query the current CUDA device");
    }
    plan = new (std::nothrow) sso_plan();
    if (!plan) return fail(nullptr, SSO_ERR_ALLOC, "out of host memory");
    plan->device = dev;
    plan->num_sms = num_sms;
    plan->smem_optin = (size_t)optin;
    plan->ndim = ndim;
    plan->ncomp = ncomp;
    plan->precision = precision;
    plan->dt = dt;
    const double PI = 3.14159265358979323846264338327950288;
    for (int a = 0; a < ndim; ++a) {
        Axis &A = plan->ax[a];
        A.n = (int)sizes[a];
        A.dx = dx[a];
        plan->npts *= A.n;
        const int n = A.n, U = n / 16;
        A.k_nat.resize(n);
        for (int j = 0; j < n; ++j) {
            const int jj = j < n / 2 ? j : j - n;
            A.k_nat[j] = 2.0 * PI * (double)jj / ((double)n * A.dx);
        }
        A.pos_freq.resize(n);
        A.slot_nat.resize(n);
        std::vector<int> revB(U), revBinv(U);
        for (int p = 0; p < n; ++p) {
            const int f = freq_of_pos(n, p);
            A.pos_freq[p] = f;
            A.slot_nat[(p % 16) * U + p / 16] = f;
            if (p % 16 == 0) {
                revB[p / 16] = f;
                revBinv[f] = p / 16;
            }
        }
        cudaError_t e = upload_twiddles(n, precision, &A.tw);
        if (e == cudaSuccess) e = upload((void **)&A.d_revB, revB);
        if (e == cudaSuccess) e = upload((void **)&A.d_revBinv, revBinv);
        if (e == cudaSuccess) e = upload((void **)&A.d_slot_nat, A.slot_nat);
        std::vector<double> kv;
        kinetic_layout(plan, a, kv);
        if (e == cudaSuccess) e = upload((void **)&A.d_kv, kv);
        if (e == cudaSuccess) e = cudaMalloc(&A.d_kph, (size_t)n * plan->esize());
        {
            std::vector<double> kpos(n);
            for (int q = 0; q < n; ++q) kpos[q] = A.k_nat[A.pos_freq[q]];
            if (e == cudaSuccess) e = upload((void **)&A.d_kpos, kpos);
        }
        if (e != cudaSuccess) {
            int rc = cuda_fail(nullptr, e, "plan tables");
            sso_destroy(plan);
            return rc;
        }
    }
    cudaError_t e = cudaMalloc((void **)&plan->d_partial, sizeof(double) * 4 * NORM_BLOCKS);
    if (e == cudaSuccess) e = cudaMalloc((void **)&plan->d_norm, sizeof(double) * 8);
    if (e == cudaSuccess) e = cudaMalloc((void **)&plan->d_sched, 2 * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMemset(plan->d_sched, 0, 2 * sizeof(unsigned));
    if (e != cudaSuccess) {
        int rc = cuda_fail(nullptr, e, "plan buffers");
        sso_destroy(plan);
        return rc;
    }
    int rc = sso_set_potential(plan, nullptr, 0, nullptr);
    if (rc == SSO_OK) rc = prepare_config_tables(plan);
    if (rc != SSO_OK) {
        g_create_err = plan->err;
        sso_destroy(plan);
        return rc;
    }
    *out = plan;
    return SSO_OK;
}

int sso_destroy(sso_plan *plan) {
    if (!plan) return SSO_OK;
    for (int a = 0; a < 3; ++a) {
        Axis &A = plan->ax[a];
        cudaFree(A.tw);
        cudaFree(A.d_revB);
        cudaFree(A.d_revBinv);
        cudaFree(A.d_slot_nat);
        cudaFree(A.d_kv);
        cudaFree(A.d_kph);
        cudaFree(A.d_kpos);
    }
    cudaFree(plan->d_avg);
    cudaFree(plan->d_vtab);
    cudaFree(plan->d_vfull);
    cudaFree(plan->d_ktab);
    cudaFree(plan->d_apos);
    for (int a = 0; a < 3; ++a) cudaFree(plan->d_erow[a]);
    cudaFree(plan->d_partial);
    cudaFree(plan->d_norm);
    cudaFree(plan->d_sched);
    cudaFree(plan->d_hostbuf);
    cudaFree(plan->d_scratch);
    cudaFree(plan->cl.tw);
    cudaFree(plan->cl.tcl);
    cudaFree(plan->cl.kv);
    cudaFree(plan->cl.kph);
    delete plan;
    return SSO_OK;
}

int sso_set_constants(sso_plan *plan, double mass, double c, double charge) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (!(mass > 0.0) || !(c > 0.0) || !isfinite(mass) || !isfinite(c) || !isfinite(charge))
        return fail(plan, SSO_ERR_INVALID, "mass and c must be positive, all constants finite");
    plan->mass = mass;
    plan->clight = c;
    plan->charge = charge;
    plan->kph_valid = false;
    plan->cl.kph_valid = false;
    plan->ktab_valid = false;
    return SSO_OK;
}

int sso_set_potential(sso_plan *plan, const double *V, int on_device, void *stream) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    const long long total = plan->npts;
    const double *dV = nullptr;
    double *tmp = nullptr;
    if (V && !on_device) {
        CK(cudaMalloc((void **)&tmp, sizeof(double) * total));
        cudaError_t e = cudaMemcpyAsync(tmp, V, sizeof(double) * total, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) {
            cudaFree(tmp);
            return cuda_fail(plan, e, "upload of V");
        }
        dV = tmp;
    } else {
        dV = V;
    }
    const size_t entry = plan->vrep == VREP_TABLE ? plan->esize() : sizeof(double);
    cudaFree(plan->d_vtab);
    cudaFree(plan->d_vfull);
    plan->d_vtab = plan->d_vfull = nullptr;
    plan->v_valid = false;
    cudaError_t e = cudaMalloc(&plan->d_vtab, entry * total);
    if (e == cudaSuccess && plan->ndim >= 2) e = cudaMalloc(&plan->d_vfull, entry * total);
    if (e != cudaSuccess) {
        cudaFree(tmp);
        return fail(plan, SSO_ERR_ALLOC, std::string("potential table: ") + cudaGetErrorString(e));
    }
    const Axis &L = plan->ax[plan->ndim - 1];
    const int blocks = (int)((total + 255) / 256 < 4096 ? (total + 255) / 256 : 4096);
    if (plan->precision == SSO_C128) {
        build_vtab_kernel<double><<<blocks, 256, 0, st>>>(dV, plan->d_vtab, total, L.n, nullptr, 0.5 * plan->dt, plan->vrep);
        if (plan->d_vfull) build_vtab_kernel<double><<<blocks, 256, 0, st>>>(dV, plan->d_vfull, total, L.n, L.d_slot_nat, plan->dt, plan->vrep);
    } else {
        build_vtab_kernel<float><<<blocks, 256, 0, st>>>(dV, plan->d_vtab, total, L.n, nullptr, 0.5 * plan->dt, plan->vrep);
        if (plan->d_vfull) build_vtab_kernel<float><<<blocks, 256, 0, st>>>(dV, plan->d_vfull, total, L.n, L.d_slot_nat, plan->dt, plan->vrep);
    }
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(tmp);
    if (e != cudaSuccess) return cuda_fail(plan, e, "potential table kernel");
    plan->v_valid = true;
    return SSO_OK;
}

int sso_set_vector_potential(sso_plan *plan, const double *A, int on_device, void *stream) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (plan->ncomp == 1)
        return fail(plan, SSO_ERR_UNSUPPORTED, "the position-space vector potential is the Dirac interaction factor (ncomp 2 or 4)");
    cudaStream_t st = (cudaStream_t)stream;
    if (!A) {
        cudaFree(plan->d_apos);
        plan->d_apos = nullptr;
        return prepare_config_tables(plan);
    }
    const size_t bytes = sizeof(double) * (size_t)plan->npts * plan->ndim;
    // a host array is checked like the rows of sso_set_field; a device array is the caller's responsibility (sso.h)
    if (!on_device)
        for (size_t i = 0, cnt = (size_t)plan->npts * plan->ndim; i < cnt; ++i)
            if (!isfinite(A[i])) return fail(plan, SSO_ERR_INVALID, "A holds a non-finite value");
    if (!plan->d_apos) {
        cudaError_t e = cudaMalloc((void **)&plan->d_apos, bytes);
        if (e != cudaSuccess) return fail(plan, SSO_ERR_ALLOC, std::string("vector potential: ") + cudaGetErrorString(e));
    }
    CK(cudaMemcpyAsync(plan->d_apos, A, bytes, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));
    return prepare_config_tables(plan);
}

int sso_set_field(sso_plan *plan, int kind, const double *step_avg, int64_t nvals) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (kind != SSO_FIELD_NONE && kind != SSO_FIELD_E && kind != SSO_FIELD_A) return fail(plan, SSO_ERR_INVALID, "unknown field kind");
    if (kind == SSO_FIELD_NONE) {
        plan->field_kind = kind;
        plan->h_avg.clear();
        plan->nvals = 0;
        cudaFree(plan->d_avg);
        plan->d_avg = nullptr;
        plan->e_along_last = false;
        for (int a = 0; a < 3; ++a) plan->e_axis_on[a] = false;
        plan->kph_valid = false;
        plan->cl.kph_valid = false;
        plan->ktab_valid = false;
        return prepare_config_tables(plan);
    }
    if (!step_avg || nvals <= 0) return fail(plan, SSO_ERR_INVALID, "step_avg is NULL or nvals <= 0");
    const size_t cnt = (size_t)nvals * plan->ndim;
    for (size_t i = 0; i < cnt; ++i)
        if (!isfinite(step_avg[i])) return fail(plan, SSO_ERR_INVALID, "step_avg holds a non-finite value");
    double *d = nullptr;
    CK(cudaMalloc((void **)&d, sizeof(double) * cnt));
    cudaError_t e = cudaMemcpy(d, step_avg, sizeof(double) * cnt, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        cudaFree(d);
        return cuda_fail(plan, e, "upload of step_avg");
    }
    cudaFree(plan->d_avg);
    plan->d_avg = d;
    plan->h_avg.assign(step_avg, step_avg + cnt);
    plan->nvals = nvals;
    plan->field_kind = kind;
    plan->e_along_last = false;
    for (int a = 0; a < 3; ++a) plan->e_axis_on[a] = false;
    if (kind == SSO_FIELD_E)
        for (int64_t n = 0; n < nvals; ++n)
            for (int a = 0; a < plan->ndim; ++a)
                if (step_avg[n * plan->ndim + a] != 0.0) plan->e_axis_on[a] = true;
    plan->e_along_last = plan->e_axis_on[plan->ndim - 1];
    // phase rows of one call (2D/3D): allocated here so that sso_step only enqueues kernels
    if (kind == SSO_FIELD_E && plan->ndim >= 2) {
        int nmax = 16;
        for (int a = 0; a < plan->ndim; ++a)
            if (plan->e_axis_on[a] && plan->ax[a].n > nmax) nmax = plan->ax[a].n;
        long long chunk = (64LL << 20) / ((long long)nmax * (long long)plan->esize()) - 1;
        if (chunk < 1) chunk = 1;
        const long long rows = (nvals < chunk ? nvals : chunk) + 1;
        for (int a = 0; a < plan->ndim; ++a) {
            cudaFree(plan->d_erow[a]);
            plan->d_erow[a] = nullptr;
            plan->erow_cap[a] = 0;
            if (!plan->e_axis_on[a]) continue;
            const size_t need = (size_t)rows * plan->ax[a].n * plan->esize();
            cudaError_t ce = cudaMalloc(&plan->d_erow[a], need);
            if (ce != cudaSuccess) return fail(plan, SSO_ERR_ALLOC, std::string("field phase rows: ") + cudaGetErrorString(ce));
            plan->erow_cap[a] = need;
        }
    }
    plan->kph_valid = false;
    plan->cl.kph_valid = false;
    plan->ktab_valid = false;
    return prepare_config_tables(plan);
}

int sso_set_time_index(sso_plan *plan, int64_t n) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (n < 0) return fail(plan, SSO_ERR_INVALID, "time index must be >= 0");
    plan->tindex = n;
    return SSO_OK;
}

int sso_get_time_index(const sso_plan *plan, int64_t *n) {
    if (!plan || !n) return SSO_ERR_INVALID;
    *n = plan->tindex;
    return SSO_OK;
}

int sso_set_option(sso_plan *plan, int option, int64_t value) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    switch (option) {
        case SSO_OPT_LINES_PER_TILE_CONTIG:
        case SSO_OPT_LINES_PER_TILE_STRIDED:
        case SSO_OPT_LINES_PER_TILE_MIDDLE:
            if (value < 0 || value > 512 || (value > 0 && !is_pow2(value))) return fail(plan, SSO_ERR_INVALID, "lines per tile must be 0 or a power of two <= 512");
            (option == SSO_OPT_LINES_PER_TILE_CONTIG ? plan->opt_tl_contig : (option == SSO_OPT_LINES_PER_TILE_STRIDED ? plan->opt_tl_strided : plan->opt_tl_middle)) = (int)value;
            return SSO_OK;
        case SSO_OPT_RING_BUFFERS:
            if (value < 0 || value > 16) return fail(plan, SSO_ERR_INVALID, "ring buffers must be in [0, 16]");
            plan->opt_ring = (int)value;
            return SSO_OK;
        case SSO_OPT_THREADS_PER_CTA:
            if (value != 0 && value != 384 && value != 512) return fail(plan, SSO_ERR_INVALID, "threads per CTA must be 0, 384 or 512");
            plan->opt_maxt = (int)value;
            return SSO_OK;
        case SSO_OPT_STRIDED_RING:
            if (value < 0 || value > 2) return fail(plan, SSO_ERR_INVALID, "strided ring mode must be 0 (auto), 1 (force) or 2 (off)");
            plan->opt_sring = (int)value;
            return SSO_OK;
        case SSO_OPT_GROUPS_PER_CTA:
            if (value < 0 || value > 15) return fail(plan, SSO_ERR_INVALID, "groups per CTA must be in [0, 15]");
            plan->opt_groups = (int)value;
            return SSO_OK;
        case SSO_OPT_DIRAC_TABLE:
            if (value != 0 && value != 1) return fail(plan, SSO_ERR_INVALID, "Dirac table mode must be 0 or 1");
            plan->opt_dirac_table = (int)value;
            if (!value) {
                cudaFree(plan->d_ktab);
                plan->d_ktab = nullptr;
            }
            plan->ktab_valid = false;
            return prepare_config_tables(plan);
        case SSO_OPT_CLUSTER_1D:
            if (value != 0 && value != 1 && value != 4 && value != 8) return fail(plan, SSO_ERR_INVALID, "cluster mode must be 0 (auto), 1 (off), 4 or 8 (CTAs per cluster)");
            plan->opt_cluster = (int)value;
            return prepare_config_tables(plan);
        case SSO_OPT_TILE_ORDER:
            if (value < 0 || value > 16) return fail(plan, SSO_ERR_INVALID, "tile order must be in [0, 16]");
            plan->opt_tile_order = (int)value;
            return SSO_OK;
        case SSO_OPT_POTENTIAL_PHASE:
            if (value != VREP_TABLE && value != VREP_ANGLE) return fail(plan, SSO_ERR_INVALID, "potential phase mode must be 0 or 1");
            if ((int)value != plan->vrep) {
                plan->vrep = (int)value;
                // the plan does not keep V itself: the tables are re-made empty in the new representation and
                // sso_step refuses to run until sso_set_potential has been called again
                const int rc = sso_set_potential(plan, nullptr, 0, nullptr);
                plan->v_valid = false;
                return rc;
            }
            return SSO_OK;
    }
    return fail(plan, SSO_ERR_INVALID, "unknown option");
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// pass construction
// ---------------------------------------------------------------------------------------------
namespace {

struct Geometry {
    int axis;          // lattice axis of the lines
    bool strided;
    long long inner;   // element stride along the line
    long long lines;   // lines per component
    int rest1;
    int oaxA, oaxB;
};

Geometry geometry(const sso_plan *p, int axis) {
    Geometry g{};
    g.axis = axis;
    const int nd = p->ndim;
    g.inner = 1;
    for (int a = axis + 1; a < nd; ++a) g.inner *= p->ax[a].n;
    g.strided = g.inner > 1;
    g.lines = p->npts / p->ax[axis].n;
    g.oaxA = g.oaxB = -1;
    g.rest1 = 1;
    int others[2], no = 0;
    for (int a = 0; a < nd; ++a)
        if (a != axis) others[no++] = a;
    if (no == 1) {
        g.oaxB = others[0];
        g.rest1 = p->ax[others[0]].n;
    } else if (no == 2) {
        g.oaxA = others[0];
        g.oaxB = others[1];
        g.rest1 = p->ax[others[1]].n;
    }
    return g;
}

// Which passes walk their tiles from the highest address down (bit 0: contiguous-axis passes, 1: middle-axis
// forward, 2: middle-axis inverse, 3: kinetic).  A pass that starts where the previous one ended finds that part of
// psi still in L2 (and its dirty lines are overwritten there instead of going to HBM twice): with the contiguous-axis
// passes descending and the middle-axis passes ascending, every plane-ordered hand-over of a 3D step meets that way.
int tile_order_mask(const sso_plan *p) {
    if (p->opt_tile_order > 0) return p->opt_tile_order - 1;
    return p->ndim == 3 ? 1 : 0;
}

// Every ring pass reserves 512 bytes of shared memory behind its buffers: the pool state of sso_ring.cuh (TileRing::bytes:
// 16 NB + 8 + 4 G <= 260 for NB <= 12, G <= 15) and, from byte 448, the observable sums of the closing pass.

// lines per component per CTA
int choose_tl(const sso_plan *p, const Geometry &g, int cc) {
    const int U = p->ax[g.axis].n / 16;
    const int esz = (int)p->esize();
    long long tl;
    if (!g.strided) {
        tl = p->opt_tl_contig > 0 ? p->opt_tl_contig : (U >= 256 ? 512 : 256) / (cc * U);
        if (tl < 1) tl = 1;
        if (tl > g.lines) tl = g.lines;
    } else {
        int tlmin = 64 / esz;  // 64-byte rows: narrower rows are served at less than half speed
        while (tlmin > 1 && cc * tlmin * U > 512) tlmin /= 2;
        tl = p->opt_tl_strided > 0 ? p->opt_tl_strided : 256 / (cc * U);
        if (p->opt_tl_strided == 0 && tl < tlmin) tl = tlmin;
        if (tl > g.inner) tl = g.inner;
    }
    while (tl > 1 && (long long)cc * tl * U > 512) tl /= 2;
    return (int)tl;
}

struct PassSpec {
    int axis;
    int pw;        // PW_*
    int sign;      // sign of the DIF transform
    int do_dif, do_dit, unpermute, mid_on, pre_v, post_v;
    int nrep;
    long long n;   // step index
};

int launch(sso_plan *plan, void *psi, const PassSpec &s, cudaStream_t st) {
    PassTimer timer(plan, plan->ndim == 1 ? SSO_PASS_LINE_1D : (s.axis == 0 ? SSO_PASS_KINETIC : (s.do_dif ? SSO_PASS_MIDDLE_FORWARD : SSO_PASS_MIDDLE_INVERSE)), st);
    const Geometry g = geometry(plan, s.axis);
    const Axis &A = plan->ax[s.axis];
    const int cc = s.pw == PW_KD2 ? 2 : (s.pw == PW_KD4 ? 4 : 1);
    const int U = A.n / 16;
    const int TL = choose_tl(plan, g, cc);
    const int esz = (int)plan->esize();
    PassArgs a{};
    a.psi = psi;
    a.tw = A.tw;
    a.revB = A.d_revB;
    a.revBinv = A.d_revBinv;
    a.comp_stride = plan->npts;
    a.inner = g.inner;
    a.ncomp = plan->ncomp;
    a.TL = TL;
    int pitch = A.n + A.n / 16;
    if (g.strided) {
        const int G = 128 / esz;
        pitch += (G / TL > 1 ? G / TL : 1);
    }
    a.pitch = pitch;
    a.rest1 = g.rest1;
    a.oaxA = g.oaxA;
    a.oaxB = g.oaxB;
    a.do_dif = s.do_dif;
    a.do_dit = s.do_dit;
    a.unpermute = s.unpermute;
    a.mid_on = s.mid_on;
    a.pre_v = s.pre_v;
    a.post_v = s.post_v;
    a.nrep = s.nrep;
    a.vtab = plan->d_vtab;
    a.vrep = plan->vrep;
    a.step_avg = plan->d_avg;
    a.field_kind = plan->field_kind;
    a.ndim = plan->ndim;
    a.line_axis = s.axis;
    a.n0 = s.n;
    a.half_dt = 0.5 * plan->dt;
    a.dt = plan->dt;
    for (int i = 0; i < 3; ++i) {
        a.nsz[i] = i < plan->ndim ? plan->ax[i].n : 1;
        a.dxs[i] = i < plan->ndim ? plan->ax[i].dx : 1.0;
    }
    a.mass = plan->mass;
    a.clight = plan->clight;
    a.charge = plan->charge;
    a.scale = 1.0 / (double)plan->npts;
    if (s.pw == PW_KS) {
        a.kph0 = A.d_kph;
        a.kph1 = g.oaxA >= 0 ? plan->ax[g.oaxA].d_kph : nullptr;
        a.kph2 = g.oaxB >= 0 ? plan->ax[g.oaxB].d_kph : nullptr;
    } else if (s.pw == PW_KD2 || s.pw == PW_KD4) {
        a.kv0 = A.d_kv;
        a.kv1 = g.oaxA >= 0 ? plan->ax[g.oaxA].d_kv : nullptr;
        a.kv2 = g.oaxB >= 0 ? plan->ax[g.oaxB].d_kv : nullptr;
    }
    LaunchFn fn = find_launch(plan->precision, A.n, g.strided ? 1 : 0, s.pw, s.sign);
    if (!fn) return fail(plan, SSO_ERR_UNSUPPORTED, "no kernel built for this pass");
    const long long tiles = g.lines / TL;
    const long long work = cc == 1 ? tiles * plan->ncomp : tiles;
    if (work > 0x7fffffffLL) return fail(plan, SSO_ERR_UNSUPPORTED, "too many tiles");
    a.ntiles = (int)work;
    a.sched = plan->d_sched;
    // groups per CTA: independent pipelines (own exchange buffer and barrier) that share one twiddle copy.
    // As many as fit in 512 threads (complex128: 128 registers/thread) or 1024 (complex64) and in shared memory.
    const int GT = cc * TL * U;
    size_t greg = (size_t)cc * TL * pitch * esz + (size_t)TL * esz + 2 * sizeof(int);
    greg = (greg + 127) & ~(size_t)127;
    const size_t twbytes = twiddle_smem_bytes(A.n, (size_t)esz);
    int G = 1;
    if (GT % 32 == 0) {
        const int maxthreads = 512;
        G = plan->opt_groups > 0 ? plan->opt_groups : maxthreads / GT;
        while (G > 1 && ((size_t)G * greg + twbytes > (size_t)plan->smem_optin - 1024 || G * GT > maxthreads)) --G;
        if (G > 15) G = 15;
        if (G < 1) G = 1;
        const long long tiles_per_sm = (work + plan->num_sms - 1) / plan->num_sms;
        if (G > tiles_per_sm) G = (int)(tiles_per_sm > 0 ? tiles_per_sm : 1);
    }
    a.G = G;
    a.GT = GT;
    a.gstride = (int)(greg / esz);
    const unsigned threads = (unsigned)(G * GT);
    size_t smem = twbytes + (size_t)G * greg;
    cudaError_t e = fn(a, threads, smem, st);
    return pass_status(plan, g.strided ? "direct strided pass" : "direct contiguous pass", e);
}


// groups per CTA and tile buffers of a contiguous-axis ring pass: GT threads per group, room for bmax buffers,
// tiles_per_cta tiles to share.  As many groups as threads and buffers allow (measured: four groups beat three with
// more buffers each); SSO_OPT_RING_BUFFERS adds spare buffers to the pool (sso_ring.cuh, TileRing).
void choose_groups(const sso_plan *plan, int GT, int bmax, long long tiles_per_cta, int *G, int *NB) {
    int g = 1;
    if (GT % 32 == 0) {
        const int cap = plan->opt_maxt ? plan->opt_maxt : 512;
        const int gthr = cap / GT > 15 ? 15 : cap / GT;
        g = gthr < bmax ? gthr : bmax;
        if (plan->opt_groups > 0 && plan->opt_groups < g) g = plan->opt_groups;
        if (g > tiles_per_cta) g = (int)(tiles_per_cta > 0 ? tiles_per_cta : 1);
        if (g < 1) g = 1;
    }
    // measured (configs 2a, 3, 4, 5): the contiguous-axis passes are fastest without spare buffers
    int nb = g;
    if (plan->opt_ring > 0) nb = plan->opt_ring < bmax ? plan->opt_ring : bmax;
    if (nb < g) nb = g;
    if (nb > 12) nb = 12;
    *G = g;
    *NB = nb;
}

// observables asked of the closing pass of a call (sso_step_observe)
struct ObsRequest {
    const void *ref;
    void *facc;
    double t, T, E, dts;
    int grid;  // CTAs of the closing pass that wrote partial sums (set by launch_ring_pass)
};

// contiguous-axis pass of a 2D/3D lattice through the ring pipeline (sso_ring.cuh).  `row` selects the field
// phase row of this call (build_erows_kernel): 0 opening, j merged after step j-1, nsteps closing.
int launch_ring_pass(sso_plan *plan, void *psi, int mode, long long row, cudaStream_t st, ObsRequest *obs = nullptr) {
    PassTimer timer(plan, mode == MODE_OPEN ? SSO_PASS_OPENING : (mode == MODE_MID ? SSO_PASS_POTENTIAL : SSO_PASS_CLOSING), st);
    const int last = plan->ndim - 1;
    const Axis &A = plan->ax[last];
    const int U = A.n / 16;
    const int esz = (int)plan->esize();
    const long long lines = plan->npts / A.n;       // per component
    // group tile: 128 threads = 2048 points (fewer when the lattice has fewer lines)
    // group tile: 64 threads = 1024 points when a line is that short (measured on configs 3 and 5: 8 groups of 64
    // threads beat 4 of 128: potential pass 476 -> 427 us on config 5), else one line
    int TL = plan->opt_tl_contig > 0 ? plan->opt_tl_contig : (U >= 64 ? 1 : 64 / U);
    while (TL > 1 && (lines % TL != 0 || TL * U > 512)) TL /= 2;
    const int GT = TL * U;
    const int pitch = A.n + A.n / 16;
    size_t bufbytes = (size_t)TL * pitch * esz;
    bufbytes = (bufbytes + 127) & ~(size_t)127;
    const size_t twbytes = twiddle_smem_bytes(A.n, (size_t)esz);
    const long long ntiles = lines * plan->ncomp / TL;
    if (ntiles > 0x7fffffffLL) return fail(plan, SSO_ERR_UNSUPPORTED, "too many tiles");
    // G groups, each with its own NBG buffers (NBG = 2: the next tile loads while the current one is worked on)
    const size_t avail = (size_t)plan->smem_optin - 512 - twbytes;
    const int bmax = (int)(avail / bufbytes);
    if (bmax < 1) return fail(plan, SSO_ERR_UNSUPPORTED, "line too long for the ring pipeline");
    int G = 1, NB = 1;
    choose_groups(plan, GT, bmax, (ntiles + plan->num_sms - 1) / plan->num_sms, &G, &NB);
    // the 384-thread build (168 registers) only when the groups fit it; a knob that does not fit falls back
    const int maxt = (plan->opt_maxt && G * GT <= plan->opt_maxt) ? plan->opt_maxt : (G * GT <= 384 && A.n <= 4096 ? 384 : 512);
    RingArgs a{};
    a.psi = psi;
    a.tw = A.tw;
    a.revB = A.d_revB;
    a.ntiles = (int)ntiles;
    a.TL = TL;
    a.pitch = pitch;
    a.G = G;
    a.GT = GT;
    a.NB = NB;
    a.bufstride = (int)(bufbytes / esz);
    a.lines_per_comp = (int)lines;
    a.ncomp = plan->ncomp;
    const Geometry g = geometry(plan, last);
    a.rest1 = g.rest1;
    a.rest1_shift = ilog2ll(g.rest1);
    a.ncomp_shift = ilog2ll(plan->ncomp);
    a.vtab = mode == MODE_MID ? plan->d_vfull : plan->d_vtab;
    a.vrep = plan->vrep;
    a.rev = tile_order_mask(plan) & 1;
    if (plan->field_kind == SSO_FIELD_E) {
        if (plan->e_axis_on[last]) a.eline = (const char *)plan->d_erow[last] + (size_t)row * A.n * esz;
        if (g.oaxA >= 0 && plan->e_axis_on[g.oaxA]) a.eoA = (const char *)plan->d_erow[g.oaxA] + (size_t)row * plan->ax[g.oaxA].n * esz;
        if (g.oaxB >= 0 && plan->e_axis_on[g.oaxB]) a.eoB = (const char *)plan->d_erow[g.oaxB] + (size_t)row * plan->ax[g.oaxB].n * esz;
    }
    const unsigned grid = (unsigned)(ntiles < plan->num_sms ? ntiles : plan->num_sms);
    if (obs) {
        mode = MODE_CLOSE_OBS;
        a.ref = obs->ref;
        a.facc = obs->facc;
        a.fw_t = obs->t;
        a.fw_T = obs->T;
        a.fw_E = obs->E;
        a.fw_dts = obs->dts;
        a.obs_partial = plan->d_partial;
        a.obs_axA = g.oaxA;
        a.obs_axB = g.oaxB;
        a.obs_axL = last;
        const int axs[3] = {g.oaxA, g.oaxB, last};
        for (int i = 0; i < 3; ++i) {
            a.obs_dx[i] = axs[i] >= 0 ? plan->ax[axs[i]].dx : 0.0;
            a.obs_half[i] = axs[i] >= 0 ? plan->ax[axs[i]].n / 2 : 0;
        }
        obs->grid = (int)grid;
    }
    RingLaunchFn fn = find_ring(plan->precision, A.n, mode, maxt);
    if (!fn) return fail(plan, SSO_ERR_UNSUPPORTED, "no ring kernel built for this line length");
    const size_t smem = twbytes + (size_t)NB * bufbytes + 512;  // pool state (ring_state_bytes <= 400) + observable scratch
    cudaError_t e = fn(a, (unsigned)(G * GT), smem, grid, st);
    return pass_status(plan, mode == MODE_OPEN ? "ring opening pass" : (mode == MODE_MID ? "ring potential pass" : "ring closing pass"), e);
}


// ---- strided-axis passes through the TMA ring (sso_sring.cuh) -------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
    // a driver entry point is process-wide; the initialiser of a function-local static runs once, thread-safely
    static const EncodeTiledFn fn = [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            return (EncodeTiledFn)p;
        cudaGetLastError();
        return (EncodeTiledFn) nullptr;
    }();
    return fn;
}

struct SRingShape {
    bool ok;
    int TL, GT, G, NB, pitch, box_rows;
    size_t bufbytes, twbytes;
};

// tile shape of a strided pass, or ok = false when the pool does not fit (the direct kernel takes over).
// `light` marks the transform-only passes of the middle axis, which need fewer compute groups per byte moved.
SRingShape sring_shape(const sso_plan *plan, int axis, int cc, bool light) {
    const int smode = light ? SMODE_DIF : (cc == 1 ? SMODE_KS : SMODE_KD4);
    SRingShape r{};
    if (plan->opt_sring == 2 || !encode_tiled_fn()) return r;
    const Axis &A = plan->ax[axis];
    const Geometry g = geometry(plan, axis);
    const int U = A.n / 16, esz = (int)plan->esize();
    const int Gn = 128 / esz;  // complex numbers per 128 bytes
    // twiddles + the pass's line table come first in shared memory; 512 bytes hold the pool's barriers, slots and mailboxes
    const size_t tw = (size_t)twiddle_count_padded(A.n) * esz + (size_t)sring_line_table_bytes(smode, A.n, esz);
    if (tw + 512 >= plan->smem_optin) return r;
    const size_t room = plan->smem_optin - 512 - tw;
    auto pitch_of = [&](int TL) { return A.n + A.n / 16 + (Gn / TL > 1 ? Gn / TL : 1); };
    auto bufbytes_of = [&](int TL) { return ((size_t)cc * TL * pitch_of(TL) * esz + 127) & ~(size_t)127; };
    // a tile shape is usable when whole warps make a group, a row is at least 16 bytes, and the cc components of a
    // k point fall into one warp (thread layout of sso_sring.cuh)
    auto fits = [&](int TL, int *bmax_out) {
        if (TL < 1 || TL > g.inner || g.inner % TL != 0 || TL * esz < 16) return false;
        const int GT = cc * TL * U;
        if (GT > 512 || GT % 32 != 0) return false;
        const int UL = TL >= 8 ? 1 : (8 / TL < U ? 8 / TL : U);
        if (cc * TL * UL > 32 || U % UL != 0) return false;
        const size_t bb = bufbytes_of(TL);
        if (bb > room) return false;
        *bmax_out = (int)(room / bb);
        return true;
    };
    int TL = 0, bm = 0;
    const int want_tl = light ? plan->opt_tl_middle : plan->opt_tl_strided;
    if (want_tl > 0) {
        if (fits(want_tl, &bm)) TL = want_tl;
    } else {
        // the widest rows (up to 128 bytes; 256 bytes for the transform-only passes, measured 393 -> 336 us per pass
        // on config 5) that leave room for two buffers or more
        // (16-byte rows only when nothing wider fits at all: the 4-component 1024-point Dirac tile measured 80.7 us per
        // pass with two buffers of 16-byte rows, 76.2 with one buffer of 32-byte rows)
        for (int want = 2; want >= 1 && !TL; --want)
            for (int cand = light ? 2 * Gn : Gn; cand >= 1 && !TL; cand /= 2)
                if (fits(cand, &bm) && bm >= want && (want == 1 || cand * esz >= 32)) TL = cand;
    }
    if (!TL) return r;
    r.TL = TL;
    r.GT = cc * TL * U;
    r.pitch = pitch_of(TL);
    r.bufbytes = bufbytes_of(TL);
    r.twbytes = tw;
    int bmax = (int)(room / r.bufbytes);
    if (bmax > 12) bmax = 12;
    const long long outer = plan->npts / (A.n * g.inner);
    const long long ntiles = (cc == 1 ? outer * plan->ncomp : 1) * (g.inner / TL);
    const long long per_cta = (ntiles + plan->num_sms - 1) / plan->num_sms;
    // as many groups as threads and buffers allow; the buffers left over go round the groups (a group with two
    // buffers loads its next tile while it works).  The transform-only passes run at HBM speed single-buffered and
    // measured slightly slower with more loads in flight, so they get one buffer per group.
    int G = 512 / r.GT;
    if (plan->opt_groups > 0 && plan->opt_groups < G) G = plan->opt_groups;
    if (G > bmax) G = bmax;
    if (G > per_cta) G = (int)per_cta;
    if (G > 15) G = 15;
    if (G < 1) G = 1;
    int NB = light ? G : bmax;
    if (NB > 2 * G) NB = 2 * G;
    if (plan->opt_ring > 0) NB = plan->opt_ring < bmax ? plan->opt_ring : bmax;
    if (NB < G) NB = G;
    r.G = G;
    r.NB = NB;
    r.box_rows = A.n < 256 ? A.n : 256;
    r.ok = true;
    return r;
}

int launch_sring_pass(sso_plan *plan, void *psi, int axis, int smode, long long n, const SRingShape &sh, cudaStream_t st) {
    PassTimer timer(plan, axis == 0 ? SSO_PASS_KINETIC : (smode == SMODE_DIF ? SSO_PASS_MIDDLE_FORWARD : SSO_PASS_MIDDLE_INVERSE), st);
    const Axis &A = plan->ax[axis];
    const Geometry g = geometry(plan, axis);
    const int esz = (int)plan->esize();
    const int cc = smode == SMODE_KD2 ? 2 : (smode == SMODE_KD4 ? 4 : 1);
    if (plan->tmap_psi[axis] != psi || plan->tmap_tl[axis] != sh.TL) {
        const long long outer_c = plan->npts / (A.n * g.inner) * plan->ncomp;
        cuuint64_t gdim[3] = {(cuuint64_t)(2 * g.inner), (cuuint64_t)A.n, (cuuint64_t)outer_c};
        cuuint64_t gstr[2] = {(cuuint64_t)(g.inner * esz), (cuuint64_t)((long long)A.n * g.inner * esz)};
        cuuint32_t box[3] = {(cuuint32_t)(2 * sh.TL), (cuuint32_t)sh.box_rows, 1u};
        cuuint32_t estr[3] = {1u, 1u, 1u};
        CUresult cr = encode_tiled_fn()(&plan->tmap[axis], plan->precision == SSO_C128 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, psi,
                                        gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                        sh.TL * esz >= 128 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B : CU_TENSOR_MAP_L2_PROMOTION_L2_64B,
                                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (cr != CUDA_SUCCESS) return fail(plan, SSO_ERR_CUDA, "cuTensorMapEncodeTiled failed");
        plan->tmap_psi[axis] = psi;
        plan->tmap_tl[axis] = sh.TL;
    }
    SRingArgs a{};
    a.psi = psi;
    a.inner = g.inner;
    a.comp_stride = plan->npts;
    a.tw = A.tw;
    a.TL = sh.TL;
    a.pitch = sh.pitch;
    a.G = sh.G;
    a.GT = sh.GT;
    a.NB = sh.NB;
    a.bufstride = (int)(sh.bufbytes / esz);
    a.tiles_per_outer = (int)(g.inner / sh.TL);
    a.box_rows = sh.box_rows;
    a.rest1 = g.rest1;
    a.rest1_shift = ilog2ll(g.rest1);
    a.tpo_shift = ilog2ll(a.tiles_per_outer);
    const long long outer = plan->npts / (A.n * g.inner);
    const long long ntiles = (cc == 1 ? outer * plan->ncomp : 1) * a.tiles_per_outer;
    if (ntiles > 0x7fffffffLL) return fail(plan, SSO_ERR_UNSUPPORTED, "too many tiles");
    a.ntiles = (int)ntiles;
    a.ndim = plan->ndim;
    a.rev = (tile_order_mask(plan) >> (smode == SMODE_DIF ? 1 : (smode == SMODE_DIT ? 2 : 3))) & 1;
    a.mass = plan->mass;
    a.clight = plan->clight;
    a.dt = plan->dt;
    a.scale = 1.0 / (double)plan->npts;
    if (smode == SMODE_KS) {
        a.kph0 = A.d_kph;
        a.kph1 = g.oaxA >= 0 ? plan->ax[g.oaxA].d_kph : nullptr;
        a.kph2 = g.oaxB >= 0 ? plan->ax[g.oaxB].d_kph : nullptr;
    } else if (cc > 1) {
        a.kv0 = A.d_kv;
        a.kv1 = g.oaxA >= 0 ? plan->ax[g.oaxA].d_kv : nullptr;
        a.kv2 = g.oaxB >= 0 ? plan->ax[g.oaxB].d_kv : nullptr;
        if (plan->field_kind == SSO_FIELD_A)
            for (int ax = 0; ax < plan->ndim; ++ax) a.sh[ax] = plan->charge * plan->h_avg[(size_t)n * plan->ndim + ax];
        {   // largest |E tau| of the plan: below 2^30 the kernel's own quadrant reduction is exact enough
            double p2max = 0.0;
            for (int ax = 0; ax < plan->ndim; ++ax) {
                const double km = 3.14159265358979323846 / plan->ax[ax].dx + fabs(a.sh[ax]);
                p2max += km * km;
            }
            const double mc2 = plan->mass * plan->clight * plan->clight;
            const double emax = sqrt(plan->clight * plan->clight * p2max + mc2 * mc2);
            a.fast_trig = emax * fabs(plan->dt) < 1073741824.0 ? 1 : 0;
        }
        a.ktab = plan->d_ktab;
        if (!plan->opt_dirac_table) smode = smode == SMODE_KD2 ? SMODE_KD2F : SMODE_KD4F;
    }
    SRingLaunchFn fn = find_sring(plan->precision, A.n, smode);
    if (!fn) return fail(plan, SSO_ERR_UNSUPPORTED, "no strided ring kernel built for this line length");
    const size_t smem = sh.twbytes + (size_t)sh.NB * sh.bufbytes + 512;
    const unsigned grid = (unsigned)(ntiles < plan->num_sms ? ntiles : plan->num_sms);
    cudaError_t e = fn(a, &plan->tmap[axis], (unsigned)(a.G * sh.GT), smem, grid, st);
    return pass_status(plan, smode == SMODE_DIF ? "strided ring DIF pass" : (smode == SMODE_DIT ? "strided ring DIT pass" : "strided ring kinetic pass"), e);
}

// field phase rows for steps [n0, n0 + ns) of a 2D/3D call
int build_erows(sso_plan *plan, long long n0, long long ns, cudaStream_t st) {
    if (plan->field_kind != SSO_FIELD_E) return SSO_OK;
    ERowsArgs e{};
    bool any = false;
    for (int a = 0; a < plan->ndim; ++a) {
        e.n[a] = plan->ax[a].n;
        e.dx[a] = plan->ax[a].dx;
        if (!plan->e_axis_on[a]) continue;
        const size_t need = (size_t)(ns + 1) * plan->ax[a].n * plan->esize();
        if (need > plan->erow_cap[a]) return fail(plan, SSO_ERR_STATE, "field phase rows not allocated (sso_set_field allocates them)");
        e.out[a] = plan->d_erow[a];
        any = true;
    }
    if (!any) return SSO_OK;
    PassTimer timer(plan, SSO_PASS_TABLES, st);
    e.slot_nat_last = plan->ax[plan->ndim - 1].d_slot_nat;
    e.step_avg = plan->d_avg;
    e.n0 = n0;
    e.ns = ns;
    e.ndim = plan->ndim;
    e.half_dt = 0.5 * plan->dt;
    dim3 grid(64, plan->ndim);
    if (plan->precision == SSO_C128) build_erows_kernel<double><<<grid, 256, 0, st>>>(e);
    else build_erows_kernel<float><<<grid, 256, 0, st>>>(e);
    cudaError_t ce = cudaGetLastError();
    if (ce != cudaSuccess) return cuda_fail(plan, ce, "field phase rows kernel");
    return SSO_OK;
}

// steps of one 2D/3D call small enough for one set of field phase rows
long long erow_chunk(const sso_plan *p) {
    if (p->field_kind != SSO_FIELD_E) return 0x7fffffffffffLL;
    int nmax = 16;
    for (int a = 0; a < p->ndim; ++a)
        if (p->e_axis_on[a] && p->ax[a].n > nmax) nmax = p->ax[a].n;
    const long long c = (64LL << 20) / ((long long)nmax * (long long)p->esize()) - 1;
    return c < 1 ? 1 : c;
}

// position-space vector-potential factor over `delta` of a step (1/2: half step, 1: two merged half steps)
int launch_rotation(sso_plan *plan, void *psi, double delta, cudaStream_t st) {
    if (!plan->d_apos) return SSO_OK;
    PassTimer timer(plan, SSO_PASS_ROTATION, st);
    const double coef = delta * plan->dt * plan->charge * plan->clight;
    const int blocks = plan->num_sms * 8;
    if (plan->precision == SSO_C128) {
        if (plan->ncomp == 2) apos_rotate_kernel<double, 2><<<blocks, 256, 0, st>>>(psi, plan->d_apos, plan->npts, plan->ndim, coef);
        else apos_rotate_kernel<double, 4><<<blocks, 256, 0, st>>>(psi, plan->d_apos, plan->npts, plan->ndim, coef);
    } else {
        if (plan->ncomp == 2) apos_rotate_kernel<float, 2><<<blocks, 256, 0, st>>>(psi, plan->d_apos, plan->npts, plan->ndim, coef);
        else apos_rotate_kernel<float, 4><<<blocks, 256, 0, st>>>(psi, plan->d_apos, plan->npts, plan->ndim, coef);
    }
    return pass_status(plan, "vector-potential rotation kernel", cudaGetLastError());
}

// (re)build the Schroedinger kinetic phase tables; with SSO_FIELD_A they depend on the step
int build_kphase(sso_plan *plan, long long n, cudaStream_t st) {
    const bool shifted = plan->field_kind == SSO_FIELD_A;
    if (plan->kph_valid && !shifted) return SSO_OK;
    PassTimer timer(plan, SSO_PASS_TABLES, st);
    for (int a = 0; a < plan->ndim; ++a) {
        Axis &A = plan->ax[a];
        const double scale = a == 0 ? 1.0 / (double)plan->npts : 1.0;
        const int blocks = (A.n + 127) / 128;
        if (plan->precision == SSO_C128)
            build_kphase_kernel<double><<<blocks, 128, 0, st>>>(A.d_kv, A.d_kph, A.n, plan->dt, plan->mass, shifted ? plan->d_avg : nullptr, n, plan->ndim, a, plan->charge, scale);
        else
            build_kphase_kernel<float><<<blocks, 128, 0, st>>>(A.d_kv, A.d_kph, A.n, plan->dt, plan->mass, shifted ? plan->d_avg : nullptr, n, plan->ndim, a, plan->charge, scale);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(plan, e, "kinetic phase kernel");
    }
    plan->kph_valid = !shifted;
    return SSO_OK;
}

// table of the Dirac kinetic scalars (SSO_OPT_DIRAC_TABLE = 1): built once for a plan without SSO_FIELD_A, every step with it
bool dirac_table_per_step(const sso_plan *p) { return p->opt_dirac_table && p->ncomp > 1 && p->ndim >= 2 && p->field_kind == SSO_FIELD_A; }
int build_ktab(sso_plan *plan, long long n, cudaStream_t st) {
    if (plan->ncomp == 1 || plan->ndim < 2 || !plan->opt_dirac_table) return SSO_OK;
    const bool shifted = plan->field_kind == SSO_FIELD_A;
    if (plan->ktab_valid && !shifted) return SSO_OK;
    if (!plan->d_ktab) return fail(plan, SSO_ERR_STATE, "Dirac kinetic table missing (its allocation failed when the option was set)");
    double sh[3] = {0.0, 0.0, 0.0};
    if (shifted)
        for (int ax = 0; ax < plan->ndim; ++ax) sh[ax] = plan->charge * plan->h_avg[(size_t)n * plan->ndim + ax];
    PassTimer timer(plan, SSO_PASS_TABLES, st);
    const Geometry g = geometry(plan, 0);
    build_ktab_kernel<<<plan->num_sms * 8, 256, 0, st>>>(reinterpret_cast<double2 *>(plan->d_ktab), plan->ax[0].d_kv,
                                                        g.oaxA >= 0 ? plan->ax[g.oaxA].d_kv : nullptr, g.oaxB >= 0 ? plan->ax[g.oaxB].d_kv : nullptr,
                                                        plan->npts, g.inner, g.rest1, sh[0], sh[1], sh[2], plan->mass, plan->clight, plan->dt,
                                                        1.0 / (double)plan->npts);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(plan, e, "Dirac kinetic table kernel");
    plan->ktab_valid = !shifted;
    return SSO_OK;
}

// ---- 1D line on a thread-block cluster (sso_line1d_cluster.cuh) ---------------------------------------------
// cluster size for this plan's 1D steps, 0 = the single-CTA kernels
int cluster_size_for(const sso_plan *p) {
    if (p->ndim != 1 || p->ncomp != 1 || p->field_kind == SSO_FIELD_E || p->d_apos || p->opt_cluster == 1) return 0;
    const int n = p->ax[0].n;
    // built, and the current device can co-schedule cs CTAs with this much shared memory each (not a given on a MIG
    // slice or a GPC with few SMs): asked once per plan and cluster size, cudaOccupancyMaxActiveClusters in the launcher
    auto usable = [&](int cs) {
        if (n / cs < 512 || n / cs > SSO_MAX_LINE_CTA) return false;
        Line1dClusterLaunchFn lc = find_line1d_cluster(p->precision, n / cs, cs);
        if (!lc) return false;
        int &fits = p->cl_fits[cs == 8 ? 1 : 0];
        if (fits < 0) {
            const int M = n / cs;
            const size_t smem = ((size_t)twiddle_count_padded(M) + (M + M / 16) + (line1d_cluster_alias(M) ? 0 : M) + (size_t)(cs - 1) * (M / cs)) * p->esize();
            Line1dClusterArgs probe{};  // psi == NULL: occupancy query only, nothing is launched
            fits = lc(probe, smem, nullptr) == cudaSuccess ? 1 : 0;
            if (!fits) cudaGetLastError();
        }
        return fits == 1;
    };
    if (p->opt_cluster > 1) return usable(p->opt_cluster) ? p->opt_cluster : 0;
    if (n > SSO_MAX_LINE_CTA) return usable(8) ? 8 : (usable(4) ? 4 : 0);
    return (n == SSO_MAX_LINE_CTA && usable(SSO_CLUSTER_AUTO_4096)) ? SSO_CLUSTER_AUTO_4096 : 0;
}

int build_cluster_tables(sso_plan *plan, int cs) {
    sso_plan::ClusterLine &cl = plan->cl;
    const int N = plan->ax[0].n, M = N / cs, MC = M / cs, U = M / 16;
    if (cl.cs == cs && cl.M == M) return SSO_OK;
    cudaFree(cl.tw);
    cudaFree(cl.tcl);
    cudaFree(cl.kv);
    cudaFree(cl.kph);
    cl = sso_plan::ClusterLine();
    cudaError_t e = upload_twiddles(M, plan->precision, &cl.tw);
    // w_N^(m k1) for m = r MC + mm, stored [r][k1 - 1][mm] (eq. 12 sign), long double, rounded once
    std::vector<double2> t64((size_t)cs * (cs - 1) * MC);
    for (int r = 0; r < cs; ++r)
        for (int k1 = 1; k1 < cs; ++k1)
            for (int mm = 0; mm < MC; ++mm) {
                const long long m = (long long)r * MC + mm;
                const long double ang = -2.0L * 3.14159265358979323846264338327950288L * (long double)((m * k1) % N) / (long double)N;
                t64[((size_t)r * (cs - 1) + (k1 - 1)) * MC + mm] = make_double2((double)cosl(ang), (double)sinl(ang));
            }
    if (e == cudaSuccess) {
        if (plan->precision == SSO_C128) e = upload(&cl.tcl, t64);
        else {
            std::vector<float2> t32(t64.size());
            for (size_t i = 0; i < t64.size(); ++i) t32[i] = make_float2((float)t64[i].x, (float)t64[i].y);
            e = upload(&cl.tcl, t32);
        }
    }
    // frequency held by CTA k1 at slot s of its M-point transform: k1 + cs k2, k2 = slot_nat_M[s]
    std::vector<double> kv((size_t)N);
    for (int p = 0; p < M; ++p) {
        const int k2 = freq_of_pos(M, p), s = (p % 16) * U + p / 16;
        for (int k1 = 0; k1 < cs; ++k1) kv[(size_t)k1 * M + s] = plan->ax[0].k_nat[k1 + cs * k2];
    }
    if (e == cudaSuccess) e = upload((void **)&cl.kv, kv);
    if (e == cudaSuccess) e = cudaMalloc(&cl.kph, (size_t)N * plan->esize());
    if (e != cudaSuccess) {
        cudaFree(cl.tw);
        cudaFree(cl.tcl);
        cudaFree(cl.kv);
        cudaFree(cl.kph);
        cl = sso_plan::ClusterLine();
        return fail(plan, SSO_ERR_ALLOC, std::string("cluster line tables: ") + cudaGetErrorString(e));
    }
    cl.cs = cs;
    cl.M = M;
    return SSO_OK;
}

int prepare_config_tables(sso_plan *plan) {
    if (plan->ndim == 1) {
        const int cs = cluster_size_for(plan);
        return cs ? build_cluster_tables(plan, cs) : SSO_OK;  // a rebuilt ClusterLine starts with kph_valid = false
    }
    if (plan->opt_dirac_table && plan->ncomp > 1 && !plan->d_ktab) {
        cudaError_t e = cudaMalloc(&plan->d_ktab, sizeof(double2) * (size_t)plan->npts);
        if (e != cudaSuccess) return fail(plan, SSO_ERR_ALLOC, std::string("Dirac kinetic table: ") + cudaGetErrorString(e));
        plan->ktab_valid = false;
    }
    return SSO_OK;
}

// kinetic phases of the cluster layout (eq. 13), rebuilt every step with SSO_FIELD_A
int build_kphase_cluster(sso_plan *plan, long long n, cudaStream_t st) {
    const bool shifted = plan->field_kind == SSO_FIELD_A;
    if (plan->cl.kph_valid && !shifted) return SSO_OK;
    PassTimer timer(plan, SSO_PASS_TABLES, st);
    const int N = plan->ax[0].n;
    const int blocks = (N + 127) / 128;
    if (plan->precision == SSO_C128)
        build_kphase_kernel<double><<<blocks, 128, 0, st>>>(plan->cl.kv, plan->cl.kph, N, plan->dt, plan->mass, shifted ? plan->d_avg : nullptr, n, 1, 0, plan->charge, 1.0 / (double)N);
    else
        build_kphase_kernel<float><<<blocks, 128, 0, st>>>(plan->cl.kv, plan->cl.kph, N, plan->dt, plan->mass, shifted ? plan->d_avg : nullptr, n, 1, 0, plan->charge, 1.0 / (double)N);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(plan, e, "kinetic phase kernel (cluster layout)");
    plan->cl.kph_valid = !shifted;
    return SSO_OK;
}

// Dirac lines whose components do not fit one CTA together: the kinetic sandwich is split into a transform-only pass
// per direction and the pointwise kernel (two more round trips of psi per step)
bool dirac_split_kinetic(const sso_plan *p) { return p->ncomp > 1 && p->ndim >= 2 && (long long)p->ncomp * (p->ax[0].n / 16) > 512; }

int launch_dirac_pointwise(sso_plan *plan, void *psi, long long n, cudaStream_t st) {
    PassTimer timer(plan, SSO_PASS_KINETIC, st);
    const Geometry g = geometry(plan, 0);
    double sh[3] = {0.0, 0.0, 0.0};
    if (plan->field_kind == SSO_FIELD_A)
        for (int ax = 0; ax < plan->ndim; ++ax) sh[ax] = plan->charge * plan->h_avg[(size_t)n * plan->ndim + ax];
    const double *kv1 = g.oaxA >= 0 ? plan->ax[g.oaxA].d_kv : nullptr, *kv2 = g.oaxB >= 0 ? plan->ax[g.oaxB].d_kv : nullptr;
    const int blocks = plan->num_sms * 8;
    const double scale = 1.0 / (double)plan->npts;
#define SSO_DPW(TT, CCN)                                                                                                                      \
    dirac_pointwise_kernel<TT, CCN><<<blocks, 256, 0, st>>>(psi, plan->npts, g.inner, g.rest1, plan->ax[0].d_kpos, kv1, kv2, sh[0], sh[1], sh[2], \
                                                            plan->mass, plan->clight, plan->dt, scale)
    if (plan->precision == SSO_C128) {
        if (plan->ncomp == 2) SSO_DPW(double, 2);
        else SSO_DPW(double, 4);
    } else {
        if (plan->ncomp == 2) SSO_DPW(float, 2);
        else SSO_DPW(float, 4);
    }
#undef SSO_DPW
    return pass_status(plan, "Dirac pointwise kinetic kernel", cudaGetLastError());
}

int kinetic_pw(const sso_plan *p) { return p->ncomp == 1 ? PW_KS : (p->ncomp == 2 ? PW_KD2 : PW_KD4); }

long long launches_for(const sso_plan *p, long long nsteps) {
    if (nsteps <= 0) return 0;
    long long cnt = 0;
    const bool kshift = p->ncomp == 1 && p->field_kind == SSO_FIELD_A;
    const bool kbuild = p->ncomp == 1 && (kshift || !p->kph_valid);
    if (p->ndim == 1) {
        if (p->d_apos) return 2 * nsteps + 1;  // rotation, then one step and one rotation per step
        if (cluster_size_for(p)) return kshift ? 2 * nsteps : 1 + (p->cl.kph_valid ? 0 : 1);
        if (kshift) return nsteps * (1 + p->ndim);
        return 1 + (kbuild ? p->ndim : 0);
    }
    const long long chunk = p->d_apos ? 1 : erow_chunk(p);
    const long long nchunks = (nsteps + chunk - 1) / chunk;
    if (p->ncomp > 1 && p->opt_dirac_table && !dirac_split_kinetic(p) && sring_shape(p, 0, p->ncomp, false).ok) cnt += dirac_table_per_step(p) ? nsteps : (p->ktab_valid ? 0 : 1);  // Dirac kinetic table
    bool eph = false;
    for (int a = 0; a < p->ndim; ++a) eph = eph || (p->field_kind == SSO_FIELD_E && p->e_axis_on[a]);
    cnt += nchunks * (eph ? 2 : 1);              // opening pass (+ field phase rows)
    cnt += nsteps * (p->ndim == 3 ? 3 : 1);      // kinetic sandwich (+ middle-axis DIF and DIT)
    if (dirac_split_kinetic(p)) cnt += 2 * nsteps;  // transform, pointwise factor, transform instead of one sandwich
    cnt += nsteps;                               // potential sandwiches and the closing pass
    if (p->d_apos) cnt += nchunks + 1;           // position-space rotations: before the first opening pass, between chunks, after the last closing pass
    if (kshift) cnt += nsteps * p->ndim;
    else if (kbuild) cnt += p->ndim;
    return cnt;
}

}  // namespace

extern "C" {

int sso_launch_count(const sso_plan *plan, int64_t nsteps, int64_t *count) {
    if (!plan || !count) return SSO_ERR_INVALID;
    *count = launches_for(plan, nsteps);
    return SSO_OK;
}

// the steps of sso_step; obs != NULL: the closing pass of the call also accumulates the observables (2D/3D lattices
// without the position-space vector potential; *fused tells the caller whether it did)
static int step_impl(sso_plan *plan, void *psi, int64_t nsteps, void *stream, ObsRequest *obs, bool *fused) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (!psi) return fail(plan, SSO_ERR_INVALID, "psi is NULL");
    if (((uintptr_t)psi & 15u) != 0) return fail(plan, SSO_ERR_INVALID, "psi must be 16-byte aligned");
    if (nsteps < 0) return fail(plan, SSO_ERR_INVALID, "nsteps must be >= 0");
    if (nsteps == 0) return SSO_OK;
    if (plan->field_kind != SSO_FIELD_NONE && plan->tindex + nsteps > plan->nvals)
        return fail(plan, SSO_ERR_STATE, "field table shorter than the steps requested");
    if (!plan->v_valid || !plan->d_vtab || (plan->ndim >= 2 && !plan->d_vfull))
        return fail(plan, SSO_ERR_STATE, "no potential table: call sso_set_potential (again) before sso_step");
    cudaStream_t st = (cudaStream_t)stream;
    const int nd = plan->ndim;
    const int kpw = kinetic_pw(plan);
    const long long n0 = plan->tindex;
    int rc;
    if (nd == 1) {
        // one persistent CTA: V/2, then nsteps x [F K F^-1, V (merged) or V/2 (last)]
        const bool kshift = plan->ncomp == 1 && plan->field_kind == SSO_FIELD_A;
        // step-dependent kinetic tables, or the position-space rotation between the steps, force one launch per step
        const long long chunk = (kshift || plan->d_apos) ? 1 : nsteps;
        const int cs = cluster_size_for(plan);
        if (!cs && plan->ax[0].n > SSO_MAX_AXIS)
            return fail(plan, SSO_ERR_UNSUPPORTED, "1D lattices beyond 8192 points run on a thread-block cluster: Schroedinger without a length-gauge field only");
        // the tables of the cluster kernel were made when the configuration was set (prepare_config_tables): nothing is
        // allocated or copied here
        if (cs && (plan->cl.cs != cs || plan->cl.M != plan->ax[0].n / cs))
            return fail(plan, SSO_ERR_STATE, "cluster line tables missing (their allocation failed when the configuration was set)");
        for (long long s = 0; s < nsteps; s += chunk) {
            if (chunk > 0x7fffffffLL) return fail(plan, SSO_ERR_INVALID, "nsteps too large");
            if (cs) {
                // the line spread over a cluster of cs CTAs, psi in registers for all steps of the launch
                if ((rc = build_kphase_cluster(plan, n0 + s, st)) != SSO_OK) return rc;
                PassTimer timer(plan, SSO_PASS_LINE_1D, st);
                const int M = plan->cl.M;
                Line1dClusterArgs la{};
                la.psi = psi;
                la.tw = plan->cl.tw;
                la.tcl = plan->cl.tcl;
                la.vtab = plan->d_vtab;
                la.vrep = plan->vrep;
                la.kph = plan->cl.kph;
                la.nsteps = (int)chunk;
                const size_t smem = ((size_t)twiddle_count_padded(M) + (M + M / 16) + (line1d_cluster_alias(M) ? 0 : M) + (size_t)(cs - 1) * (M / cs)) * plan->esize();
                Line1dClusterLaunchFn lc = find_line1d_cluster(plan->precision, M, cs);
                if ((rc = pass_status(plan, "1D cluster line kernel", lc(la, smem, st))) != SSO_OK) return rc;
                continue;
            }
            // position-space factor: half a step before the first step of the call, a whole one between two steps (the
            // closing half of one and the opening half of the next use the same A), half a step after the last
            if (s == 0 && (rc = launch_rotation(plan, psi, 0.5, st)) != SSO_OK) return rc;
            if (plan->ncomp == 1 && (rc = build_kphase(plan, n0 + s, st)) != SSO_OK) return rc;
            Line1dLaunchFn l1 = (plan->ncomp == 1 && plan->field_kind != SSO_FIELD_E) ? find_line1d(plan->precision, plan->ax[0].n) : nullptr;
            if (l1) {
                // Schroedinger without a length-gauge field: both pointwise tables are constant over the launch and
                // live in registers (sso_line1d.cuh)
                PassTimer timer(plan, SSO_PASS_LINE_1D, st);
                Line1dArgs la{};
                la.psi = psi;
                la.tw = plan->ax[0].tw;
                la.vtab = plan->d_vtab;
                la.vrep = plan->vrep;
                la.kph0 = plan->ax[0].d_kph;
                la.nsteps = (int)chunk;
                const int n = plan->ax[0].n;
                const size_t smem = ((size_t)twiddle_count_padded(n) + n + n / 16) * plan->esize();
                if ((rc = pass_status(plan, "1D line kernel", l1(la, smem, st))) != SSO_OK) return rc;
                continue;
            }
            PassSpec ps{0, kpw, -1, 1, 1, 0, 1, 1, 1, (int)chunk, n0 + s};
            if ((rc = launch(plan, psi, ps, st)) != SSO_OK) return rc;
            if ((rc = launch_rotation(plan, psi, s + chunk < nsteps ? 1.0 : 0.5, st)) != SSO_OK) return rc;
        }
    } else {
        // chunks that share one set of field phase rows; each chunk opens and closes with a half step
        // Between the passes of a chunk psi is in momentum space along the last axis, so the position-space
        // rotation can only run before an opening and after a closing pass: with it every step is its own chunk.
        const long long chunk = plan->d_apos ? 1 : erow_chunk(plan);
        SRingShape shk = sring_shape(plan, 0, plan->ncomp == 1 ? 1 : plan->ncomp, false);
        SRingShape shm = nd == 3 ? sring_shape(plan, 1, 1, true) : SRingShape{};
        SRingShape sh0 = dirac_split_kinetic(plan) ? sring_shape(plan, 0, 1, true) : SRingShape{};
        for (long long c0 = 0; c0 < nsteps; c0 += chunk) {
            const long long ns = nsteps - c0 < chunk ? nsteps - c0 : chunk;
            const long long nb = n0 + c0;
            if ((rc = build_erows(plan, nb, ns, st)) != SSO_OK) return rc;
            // opening: V/2 in natural order, forward transform along the last axis, natural frequency order out
            // (position-space factor: half a step before the first chunk, a whole one between chunks, half after the last)
            if (c0 == 0 && (rc = launch_rotation(plan, psi, 0.5, st)) != SSO_OK) return rc;
            if ((rc = launch_ring_pass(plan, psi, MODE_OPEN, 0, st)) != SSO_OK) return rc;
            for (long long s = 0; s < ns; ++s) {
                const long long n = nb + s;
                if (plan->ncomp == 1 && (rc = build_kphase(plan, n, st)) != SSO_OK) return rc;
                if (nd == 3) {  // F_1, stored in network order
                    if (shm.ok) rc = launch_sring_pass(plan, psi, 1, SMODE_DIF, n, shm, st);
                    else {
                        PassSpec mid{1, PW_NONE, -1, 1, 0, 0, 0, 0, 0, 1, n};
                        rc = launch(plan, psi, mid, st);
                    }
                    if (rc != SSO_OK) return rc;
                }
                if (dirac_split_kinetic(plan)) {
                    // F_0 (components one by one), the Dirac factor as a kernel of its own, F_0^-1
                    for (int dir = 0; dir < 2; ++dir) {
                        if (sh0.ok) rc = launch_sring_pass(plan, psi, 0, dir == 0 ? SMODE_DIF : SMODE_DIT, n, sh0, st);
                        else {
                            PassSpec tr{0, PW_NONE, -1, dir == 0, dir == 1, 0, 0, 0, 0, 1, n};
                            rc = launch(plan, psi, tr, st);
                        }
                        if (rc != SSO_OK) return rc;
                        if (dir == 0 && (rc = launch_dirac_pointwise(plan, psi, n, st)) != SSO_OK) return rc;
                    }
                } else {
                    if (shk.ok && (rc = build_ktab(plan, n, st)) != SSO_OK) return rc;
                    if (shk.ok) rc = launch_sring_pass(plan, psi, 0, kpw == PW_KS ? SMODE_KS : (kpw == PW_KD2 ? SMODE_KD2 : SMODE_KD4), n, shk, st);
                    else {
                        PassSpec kin{0, kpw, -1, 1, 1, 0, 1, 0, 0, 1, n};  // F_0 K F_0^-1
                        rc = launch(plan, psi, kin, st);
                    }
                    if (rc != SSO_OK) return rc;
                }
                if (nd == 3) {  // F_1^-1 from network order
                    if (shm.ok) rc = launch_sring_pass(plan, psi, 1, SMODE_DIT, n, shm, st);
                    else {
                        PassSpec mid{1, PW_NONE, -1, 0, 1, 0, 0, 0, 0, 1, n};
                        rc = launch(plan, psi, mid, st);
                    }
                    if (rc != SSO_OK) return rc;
                }
                // F_last^-1 V(n, n+1) F_last, or the closing F_last^-1, V/2
                const bool last_of_call = s + 1 == ns && c0 + ns == nsteps;
                ObsRequest *ob = (obs && last_of_call && !plan->d_apos) ? obs : nullptr;
                if (ob && fused) *fused = true;
                if ((rc = launch_ring_pass(plan, psi, s + 1 < ns ? MODE_MID : MODE_CLOSE, s + 1, st, ob)) != SSO_OK) return rc;
            }
            if ((rc = launch_rotation(plan, psi, c0 + ns < nsteps ? 1.0 : 0.5, st)) != SSO_OK) return rc;
        }
    }
    plan->tindex += nsteps;
    return SSO_OK;
}

int sso_step(sso_plan *plan, void *psi, int64_t nsteps, void *stream) { return step_impl(plan, psi, nsteps, stream, nullptr, nullptr); }

int sso_profile_step(sso_plan *plan, void *psi, int64_t nsteps, void *stream, int64_t *count, double *mean_us) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (!count || !mean_us) return fail(plan, SSO_ERR_INVALID, "count or mean_us is NULL");
    for (int k = 0; k < SSO_PASS_KINDS; ++k) {
        count[k] = 0;
        mean_us[k] = 0.0;
    }
    std::vector<sso_plan::ProfEvent> ev;
    plan->prof = &ev;
    int rc = sso_step(plan, psi, nsteps, stream);
    plan->prof = nullptr;
    cudaError_t e = cudaStreamSynchronize((cudaStream_t)stream);
    for (auto &p : ev) {
        float ms = 0.f;
        if (rc == SSO_OK && e == cudaSuccess && cudaEventElapsedTime(&ms, p.a, p.b) == cudaSuccess && p.kind >= 0 && p.kind < SSO_PASS_KINDS) {
            count[p.kind] += 1;
            mean_us[p.kind] += (double)ms * 1e3;
        }
        cudaEventDestroy(p.a);
        cudaEventDestroy(p.b);
    }
    for (int k = 0; k < SSO_PASS_KINDS; ++k)
        if (count[k] > 0) mean_us[k] /= (double)count[k];
    if (rc != SSO_OK) return rc;
    if (e != cudaSuccess) return cuda_fail(plan, e, "sso_profile_step");
    return SSO_OK;
}

const char *sso_pass_name(int kind) {
    switch (kind) {
        case SSO_PASS_OPENING: return "opening [V/2 . F_last]";
        case SSO_PASS_POTENTIAL: return "potential [F_last^-1 . V . F_last]";
        case SSO_PASS_CLOSING: return "closing [F_last^-1 . V/2]";
        case SSO_PASS_KINETIC: return "kinetic [F_0 . K . F_0^-1]";
        case SSO_PASS_MIDDLE_FORWARD: return "middle axis [F_1]";
        case SSO_PASS_MIDDLE_INVERSE: return "middle axis [F_1^-1]";
        case SSO_PASS_LINE_1D: return "1D line, all steps in one launch";
        case SSO_PASS_TABLES: return "per-step tables";
        case SSO_PASS_ROTATION: return "position-space vector-potential rotation";
    }
    return "";
}

int sso_step_host(sso_plan *plan, void *psi_host, int64_t nsteps) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (!psi_host) return fail(plan, SSO_ERR_INVALID, "psi_host is NULL");
    if (nsteps < 0) return fail(plan, SSO_ERR_INVALID, "nsteps must be >= 0");
    const size_t bytes = (size_t)plan->npts * plan->ncomp * plan->esize();
    if (!plan->d_hostbuf) {
        cudaError_t e = cudaMalloc(&plan->d_hostbuf, bytes);
        if (e != cudaSuccess) return fail(plan, SSO_ERR_ALLOC, std::string("device buffer: ") + cudaGetErrorString(e));
    }
    CK(cudaMemcpy(plan->d_hostbuf, psi_host, bytes, cudaMemcpyHostToDevice));
    int rc = sso_step(plan, plan->d_hostbuf, nsteps, nullptr);
    if (rc != SSO_OK) return rc;
    CK(cudaMemcpy(psi_host, plan->d_hostbuf, bytes, cudaMemcpyDeviceToHost));
    return SSO_OK;
}

int sso_norm(sso_plan *plan, const void *psi, double *out_host, void *stream) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (!psi || !out_host) return fail(plan, SSO_ERR_INVALID, "psi or out_host is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    const long long count = plan->npts * plan->ncomp;
    double vol = 1.0;
    for (int a = 0; a < plan->ndim; ++a) vol *= plan->ax[a].dx;
    if (plan->precision == SSO_C128)
        norm_partial_kernel<double><<<NORM_BLOCKS, 256, 0, st>>>(psi, count, plan->d_partial);
    else
        norm_partial_kernel<float><<<NORM_BLOCKS, 256, 0, st>>>(psi, count, plan->d_partial);
    norm_final_kernel<<<1, 32, 0, st>>>(plan->d_partial, NORM_BLOCKS, vol, plan->d_norm);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(out_host, plan->d_norm, sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return SSO_OK;
}

// ---- observables -------------------------------------------------------------------------------

int sso_overlap(sso_plan *plan, const void *psi_a, const void *psi_b, double *out_host, void *stream) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (!psi_a || !psi_b || !out_host) return fail(plan, SSO_ERR_INVALID, "psi_a, psi_b or out_host is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    const long long count = plan->npts * plan->ncomp;
    double vol = 1.0;
    for (int a = 0; a < plan->ndim; ++a) vol *= plan->ax[a].dx;
    if (plan->precision == SSO_C128) overlap_partial_kernel<double><<<NORM_BLOCKS, 256, 0, st>>>(psi_a, psi_b, count, plan->d_partial);
    else overlap_partial_kernel<float><<<NORM_BLOCKS, 256, 0, st>>>(psi_a, psi_b, count, plan->d_partial);
    reduce_final_kernel<<<1, 64, 0, st>>>(plan->d_partial, NORM_BLOCKS, 2, vol, plan->d_norm);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(out_host, plan->d_norm, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return SSO_OK;
}

static int weighted_density(sso_plan *plan, const void *psi, bool momentum, double scale, double *out_host, cudaStream_t st) {
    AxisWeights aw{};
    for (int a = 0; a < 3; ++a) {
        aw.tab[a] = (momentum && a < plan->ndim) ? plan->ax[a].d_kpos : nullptr;
        aw.n[a] = a < plan->ndim ? plan->ax[a].n : 1;
        aw.dx[a] = a < plan->ndim ? plan->ax[a].dx : 1.0;
    }
    aw.ndim = plan->ndim;
    aw.ncomp = plan->ncomp;
    aw.npts = plan->npts;
    if (plan->precision == SSO_C128) weighted_density_partial_kernel<double><<<NORM_BLOCKS, 256, 0, st>>>(psi, aw, plan->d_partial);
    else weighted_density_partial_kernel<float><<<NORM_BLOCKS, 256, 0, st>>>(psi, aw, plan->d_partial);
    reduce_final_kernel<<<1, 96, 0, st>>>(plan->d_partial, NORM_BLOCKS, 3, scale, plan->d_norm);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(out_host, plan->d_norm, (size_t)plan->ndim * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return SSO_OK;
}

int sso_expect_position(sso_plan *plan, const void *psi, double *out_host, void *stream) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (!psi || !out_host) return fail(plan, SSO_ERR_INVALID, "psi or out_host is NULL");
    double vol = 1.0;
    for (int a = 0; a < plan->ndim; ++a) vol *= plan->ax[a].dx;
    return weighted_density(plan, psi, false, vol, out_host, (cudaStream_t)stream);
}

int sso_expect_momentum(sso_plan *plan, const void *psi, double *out_host, void *stream) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (!psi || !out_host) return fail(plan, SSO_ERR_INVALID, "psi or out_host is NULL");
    if (((uintptr_t)psi & 15u) != 0) return fail(plan, SSO_ERR_INVALID, "psi must be 16-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    for (int a = 0; a < plan->ndim; ++a)
        if (plan->ax[a].n > SSO_MAX_AXIS)
            return fail(plan, SSO_ERR_UNSUPPORTED, "sso_expect_momentum: axes of at most 8192 points (longer 1D lattices exist only inside the cluster step kernel)");
    const size_t bytes = (size_t)plan->npts * plan->ncomp * plan->esize();
    if (!plan->d_scratch) {
        cudaError_t e = cudaMalloc(&plan->d_scratch, bytes);
        if (e != cudaSuccess) return fail(plan, SSO_ERR_ALLOC, std::string("work buffer: ") + cudaGetErrorString(e));
    }
    CK(cudaMemcpyAsync(plan->d_scratch, psi, bytes, cudaMemcpyDeviceToDevice, st));
    // forward transform of the copy along every axis, left in network order (the momentum table is stored that way)
    for (int a = 0; a < plan->ndim; ++a) {
        const bool contiguous = a == plan->ndim - 1;
        PassSpec ps{a, contiguous ? PW_KS : PW_NONE, -1, 1, 0, 0, 0, 0, 0, 1, 0};
        const int rc = launch(plan, plan->d_scratch, ps, st);
        if (rc != SSO_OK) return rc;
    }
    double vol = 1.0;
    for (int a = 0; a < plan->ndim; ++a) vol *= plan->ax[a].dx;
    return weighted_density(plan, plan->d_scratch, true, vol / (double)plan->npts, out_host, st);
}

int sso_spectrum(sso_plan *plan, const double *chi_host, int64_t nt, double dts, const double *E_host, int64_t nE, double *out_host, void *stream) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (!chi_host || !E_host || !out_host) return fail(plan, SSO_ERR_INVALID, "chi_host, E_host or out_host is NULL");
    if (nt <= 0 || nE <= 0 || nE > 0x7fffffffLL || !isfinite(dts)) return fail(plan, SSO_ERR_INVALID, "nt and nE must be positive, dts finite");
    cudaStream_t st = (cudaStream_t)stream;
    double2 *d_chi = nullptr, *d_out = nullptr;
    double *d_E = nullptr;
    cudaError_t e = cudaMalloc((void **)&d_chi, sizeof(double2) * (size_t)nt);
    if (e == cudaSuccess) e = cudaMalloc((void **)&d_E, sizeof(double) * (size_t)nE);
    if (e == cudaSuccess) e = cudaMalloc((void **)&d_out, sizeof(double2) * (size_t)nE);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_chi, chi_host, sizeof(double2) * (size_t)nt, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_E, E_host, sizeof(double) * (size_t)nE, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) {
        spectrum_kernel<<<(unsigned)nE, 256, 0, st>>>(d_chi, nt, dts, d_E, d_out);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(out_host, d_out, sizeof(double2) * (size_t)nE, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d_chi);
    cudaFree(d_E);
    cudaFree(d_out);
    if (e != cudaSuccess) return cuda_fail(plan, e, "sso_spectrum");
    return SSO_OK;
}

int sso_filter_accumulate(sso_plan *plan, void *acc, const void *psi, double t, double T, double E, double dts, void *stream) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (!acc || !psi) return fail(plan, SSO_ERR_INVALID, "acc or psi is NULL");
    if (!(T > 0.0) || !isfinite(t) || !isfinite(T) || !isfinite(E) || !isfinite(dts)) return fail(plan, SSO_ERR_INVALID, "T must be positive, all arguments finite");
    cudaStream_t st = (cudaStream_t)stream;
    const long long count = plan->npts * plan->ncomp;
    const int blocks = plan->num_sms * 8;
    if (plan->precision == SSO_C128) filter_accumulate_kernel<double><<<blocks, 256, 0, st>>>(reinterpret_cast<double2 *>(acc), psi, count, t, T, E, dts);
    else filter_accumulate_kernel<float><<<blocks, 256, 0, st>>>(reinterpret_cast<double2 *>(acc), psi, count, t, T, E, dts);
    CK(cudaGetLastError());
    return SSO_OK;
}

int sso_step_observe(sso_plan *plan, void *psi, int64_t nsteps, const void *psi_ref, void *filter_acc, double filter_t, double filter_T,
                     double filter_E, double filter_dts, double *out_host, void *stream) {
    if (!plan) return fail(nullptr, SSO_ERR_INVALID, "plan is NULL");
    if (!out_host) return fail(plan, SSO_ERR_INVALID, "out_host is NULL");
    if (nsteps < 1) return fail(plan, SSO_ERR_INVALID, "sso_step_observe needs nsteps >= 1");
    if (filter_acc && (!(filter_T > 0.0) || !isfinite(filter_t) || !isfinite(filter_T) || !isfinite(filter_E) || !isfinite(filter_dts)))
        return fail(plan, SSO_ERR_INVALID, "filter: T must be positive, all arguments finite");
    cudaStream_t st = (cudaStream_t)stream;
    ObsRequest ob{psi_ref, filter_acc, filter_t, filter_T, filter_E, filter_dts, 0};
    bool fused = false;
    int rc = step_impl(plan, psi, nsteps, stream, &ob, &fused);
    if (rc != SSO_OK) return rc;
    for (int i = 0; i < 6; ++i) out_host[i] = 0.0;
    if (fused) {
        double vol = 1.0;
        for (int a = 0; a < plan->ndim; ++a) vol *= plan->ax[a].dx;
        reduce_final_kernel<<<1, 192, 0, st>>>(plan->d_partial, ob.grid, 6, vol, plan->d_norm);
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(out_host, plan->d_norm, 6 * sizeof(double), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        return SSO_OK;
    }
    // 1D lattices (psi never leaves the SM during a call) and plans with the position-space vector potential (its
    // rotation follows the closing pass): the same quantities by the kernels of their own
    if ((rc = sso_norm(plan, psi, &out_host[0], stream)) != SSO_OK) return rc;
    if (psi_ref && (rc = sso_overlap(plan, psi_ref, psi, &out_host[1], stream)) != SSO_OK) return rc;
    if ((rc = sso_expect_position(plan, psi, &out_host[3], stream)) != SSO_OK) return rc;
    if (filter_acc) {
        if ((rc = sso_filter_accumulate(plan, filter_acc, psi, filter_t, filter_T, filter_E, filter_dts, stream)) != SSO_OK) return rc;
        CK(cudaStreamSynchronize(st));  // the call returns with the stream drained on every path (sso.h)
    }
    return SSO_OK;
}

}  // extern "C"

// ---- sso_norm_static: the norm for callers that cannot allocate device memory ---------------------------------------
//
// sso_norm keeps its per-CTA partial sums in a buffer that sso_plan_create obtained with cudaMalloc.  Some callers
// cannot get that far: the application (or the framework it runs in) has handed the whole of HBM to an arena of its
// own, so a cudaMalloc from this library would fail; or the caller sits in a time loop that must not stall, and
// cudaMalloc / cudaFree wait for all work on the device; or it only holds a pointer to a wavefunction another
// component propagates and has no plan (every plan allocates tables).  For them the partial sums live in the array
// below.  It is part of the library image: every GPU that loads libsso.so holds these 256 KiB until the process
// exits, whether or not this entry point is ever called.
//
// In host code `g_norm_static_partial` is only a handle for the runtime, not a device address; the address on the
// current device comes from cudaGetSymbolAddress (norm_static_scratch below), once per device.
static __device__ __align__(256) double g_norm_static_partial[SSO_NORM_STATIC_MAX_COUNT / SSO_NORM_STATIC_CHUNK];

namespace {

constexpr int NORM_STATIC_THREADS = 256;
constexpr int NORM_STATIC_MAX_DEVICES = 64;

// CTA b sums |psi|^2 over elements [b * CHUNK, min(count, (b+1) * CHUNK)) in double, in a fixed order, and writes
// partial[b].  One partial per chunk of the input (not per resident CTA as in norm_partial_kernel): the sum does not
// depend on the SM count of the device.
template <typename T>
__global__ void __launch_bounds__(NORM_STATIC_THREADS) norm_static_partial_kernel(const void *__restrict__ psi, long long count, double *__restrict__ partial) {
    using C = typename Cx2<T>::type;
    const C *p = reinterpret_cast<const C *>(psi);
    const long long lo = (long long)blockIdx.x * SSO_NORM_STATIC_CHUNK;
    const long long hi = lo + SSO_NORM_STATIC_CHUNK < count ? lo + SSO_NORM_STATIC_CHUNK : count;
    double acc = 0.0;
#pragma unroll 8
    for (long long i = lo + threadIdx.x; i < hi; i += NORM_STATIC_THREADS) {
        const C v = p[i];
        acc += (double)v.x * (double)v.x + (double)v.y * (double)v.y;
    }
    double a[1] = {acc};
    block_sum<1>(a);
    if (threadIdx.x == 0) partial[blockIdx.x] = a[0];
}

// *out = vol * sum_{b < n} partial[b]; one CTA, fixed order.  Reads only the n slots the launch before it wrote.
__global__ void __launch_bounds__(1024) norm_static_final_kernel(const double *__restrict__ partial, int n, double vol, double *__restrict__ out) {
    double a[1] = {0.0};
    for (int i = threadIdx.x; i < n; i += blockDim.x) a[0] += partial[i];
    block_sum<1>(a);
    if (threadIdx.x == 0) *out = a[0] * vol;
}

// Device address of g_norm_static_partial on the CURRENT device; looked up on the first call per device, then cached.
// The look-up may make the runtime load the library's device code onto that device; it allocates nothing of ours.
static cudaError_t norm_static_scratch(double **ptr, int *device) {
    static double *cached[NORM_STATIC_MAX_DEVICES] = {};
    static std::mutex mu;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    *device = dev;
    if (dev < 0 || dev >= NORM_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!cached[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_norm_static_partial);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        cached[dev] = p;
    }
    *ptr = cached[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int sso_norm_static(const void *psi, int precision, int64_t count, double vol, double *out_dev, void *stream) {
    sso_plan *plan = nullptr;  // errors are reported like those of sso_plan_create: sso_last_error(NULL)
    if (precision != SSO_C64 && precision != SSO_C128) return fail(nullptr, SSO_ERR_INVALID, "sso_norm_static: precision must be SSO_C64 or SSO_C128");
    if (count < 0) return fail(nullptr, SSO_ERR_INVALID, "sso_norm_static: count must be >= 0");
    if (count > SSO_NORM_STATIC_MAX_COUNT)
        return fail(nullptr, SSO_ERR_INVALID,
                    "sso_norm_static: count " + std::to_string((long long)count) + " exceeds SSO_NORM_STATIC_MAX_COUNT = " +
                        std::to_string((long long)SSO_NORM_STATIC_MAX_COUNT) +
                        " complex numbers (the built-in scratch array holds one partial sum per " + std::to_string(SSO_NORM_STATIC_CHUNK) +
                        " of them); use sso_norm with a plan, or call once per piece and add the results");
    if (!out_dev) return fail(nullptr, SSO_ERR_INVALID, "sso_norm_static: out_dev is NULL");
    if (!psi && count > 0) return fail(nullptr, SSO_ERR_INVALID, "sso_norm_static: psi is NULL");
    if (!isfinite(vol)) return fail(nullptr, SSO_ERR_INVALID, "sso_norm_static: vol must be finite");
    const uintptr_t align = precision == SSO_C128 ? 16 : 8;
    if (((uintptr_t)psi % align) != 0 || ((uintptr_t)out_dev % 8) != 0) return fail(nullptr, SSO_ERR_INVALID, "sso_norm_static: psi must be aligned to one complex number, out_dev to 8 bytes");
    double *scratch = nullptr;
    int dev = -1;
    cudaError_t e = norm_static_scratch(&scratch, &dev);
    if (e != cudaSuccess) return fail(nullptr, SSO_ERR_CUDA, "sso_norm_static: address of the scratch array on device " + std::to_string(dev) + ": " + cudaGetErrorString(e));
    cudaStream_t st = (cudaStream_t)stream;
    const int nchunks = (int)((count + SSO_NORM_STATIC_CHUNK - 1) / SSO_NORM_STATIC_CHUNK);
    // nothing in the scratch array has to start at zero: this call writes slots [0, nchunks) and reads only those
    if (nchunks > 0) {
        if (precision == SSO_C128) norm_static_partial_kernel<double><<<nchunks, NORM_STATIC_THREADS, 0, st>>>(psi, count, scratch);
        else norm_static_partial_kernel<float><<<nchunks, NORM_STATIC_THREADS, 0, st>>>(psi, count, scratch);
    }
    norm_static_final_kernel<<<1, 1024, 0, st>>>(scratch, nchunks, vol, out_dev);
    CK(cudaGetLastError());
    return SSO_OK;
}
