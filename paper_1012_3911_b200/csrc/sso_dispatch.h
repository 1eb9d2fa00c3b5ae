// sso_dispatch.h -- pass descriptor shared by the kernels (sso_pass.cuh), their per-size
// instantiations (sso_inst.cu) and the host-side plan (sso_api.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sso {

enum : int { PW_NONE = 0, PW_KS = 2, PW_KD2 = 3, PW_KD4 = 4 };

// V-phase representation
enum : int { VREP_TABLE = 0, VREP_ANGLE = 1 };

struct PassArgs {
    void *psi;               // device, [ncomp][...] complex
    const void *tw;          // complex twiddle blocks, one per non-final stage: [k-1][l] = exp(-2 pi i l k / NP)
    unsigned *sched;         // device uint[2]: next tile, CTAs done (both zero between launches)
    int ntiles;              // work items of this launch (tiles x components when components are independent)
    const int *revB;         // int[N/16]: digit reversal of the last-stage thread index
    const int *revBinv;      // int[N/16]: its inverse
    long long comp_stride;   // complex elements between components
    long long inner;         // element stride along the line (1 = contiguous axis)
    int ncomp;               // components in psi
    int TL;                  // lines per component per CTA
    int pitch;               // shared-memory line pitch in complex elements
    int G, GT;               // groups per CTA (independent pipelines sharing the twiddle table), threads per group
    int gstride;             // complex elements between the shared-memory regions of consecutive groups
    int rest1;               // size of the faster non-line axis: line index = ia * rest1 + ib, >= 1
    int oaxA, oaxB;          // lattice axes that ia and ib run along (-1: absent)
    // structure of the pass
    int do_dif, do_dit, unpermute;
    int mid_on;              // apply the pointwise factor between DIF and DIT
    int pre_v, post_v;       // 0 none; 1 natural-order table (1D); 2 gather from the permuted table (opening pass)
    int nrep;                // repetitions inside the kernel (1D persistent stepping), >= 1
    // potential phase
    const void *vtab;        // 1D: complex h = exp(-i V tau/2) (VREP_TABLE) or real angle -V tau/2 (VREP_ANGLE), natural order
    int vrep;
    // field table
    const double *step_avg;  // device [nvals][ndim] or NULL
    int field_kind;          // SSO_FIELD_*
    int ndim;
    int line_axis;           // which lattice axis the lines run along
    long long n0;            // step index of the first repetition
    double half_dt;          // tau/2
    double dt;               // tau
    int nsz[3];              // lattice sizes
    double dxs[3];           // lattice spacings
    // kinetic factor
    const void *kph0;        // Schroedinger: complex[N] line-axis phase table incl. 1/Ntot, permuted layout
    const void *kph1;        // complex[rest0] storage-order table of the slower non-line axis or NULL
    const void *kph2;        // complex[rest1] table of the faster non-line axis or NULL
    const double *kv0;       // Dirac: k values along the line (permuted layout)
    const double *kv1;       // k values, slower non-line axis (storage order) or NULL
    const double *kv2;       // k values, faster non-line axis or NULL
    double mass, clight, charge;
    double scale;            // 1/Ntot (Dirac; Schroedinger folds it into kph0)
};

// launches one wave of persistent CTAs (resident CTAs per SM x SMs, at most ntiles)
using LaunchFn = cudaError_t (*)(const PassArgs &, unsigned threads, size_t smem, cudaStream_t st);

// one lookup function per compiled (precision, line length); returns NULL for a variant that is not built
#define SSO_FOR_EACH_N(X) X(16) X(32) X(64) X(128) X(256) X(512) X(1024) X(2048) X(4096) X(8192)
#define SSO_DECL_LOOKUP(N)                                         \
    LaunchFn sso_lookup_f32_##N(int strided, int pw, int sign);    \
    LaunchFn sso_lookup_f64_##N(int strided, int pw, int sign);
SSO_FOR_EACH_N(SSO_DECL_LOOKUP)
#undef SSO_DECL_LOOKUP

// the ring pipeline of sso_ring.cuh (contiguous-axis passes of 2D/3D lattices)
enum : int { MODE_OPEN = 0, MODE_MID = 1, MODE_CLOSE = 2, MODE_CLOSE_OBS = 3 };  // CLOSE_OBS: closing pass + observables

struct RingArgs {
    void *psi;                // device, all components: ntiles * TL lines of N points, contiguous
    const void *tw;           // twiddle blocks of this axis (as in PassArgs)
    const int *revB;          // int[N/16]
    int ntiles;               // tiles of TL lines over all components
    int TL;                   // lines per tile
    int pitch;                // padded line pitch (complex elements) of the exchange layout
    int G, GT;                // groups per CTA, threads per group (= TL * N/16)
    int NB;                   // ring buffers
    int bufstride;            // complex elements between ring buffers
    int lines_per_comp;       // lines of one component (the potential table repeats per component)
    int ncomp;                // components; tile index = line block * ncomp + component, so that the tiles that share
                              // a potential-table block run at the same time and the block is fetched from HBM once
    int rest1;                // table line = ia * rest1 + ib
    int rest1_shift, ncomp_shift;  // log2 of rest1 and ncomp (lattice sizes are powers of two)
    const void *vtab;         // MODE_MID: merged phase exp(-i V tau), permuted slots; else exp(-i V tau/2), natural
    int vrep;                 // VREP_TABLE (complex phases) or VREP_ANGLE (real angles, sincos in the kernel)
    const void *eline;        // complex[N] field phase along the line for this pass (same order as vtab) or NULL
    const void *eoA, *eoB;    // complex field phase rows of the other axes, indexed by ia / ib, or NULL
    int rev;                  // tiles in descending address order
    // MODE_CLOSE_OBS: observables of the final psi accumulated in the closing pass
    const void *ref;          // psi(0) for the autocorrelation function (eq. 40), laid out like psi, or NULL
    double *obs_partial;      // [6][gridDim.x]: sum |psi|^2, Re and Im of sum conj(ref) psi, sum r_a |psi|^2 for axis a = 0, 1, 2
    void *facc;               // complex128 accumulator of the eigenfunction filter (eq. 42), laid out like psi, or NULL
    double fw_t, fw_T, fw_E, fw_dts;  // its term: acc += psi (1 - cos(2 pi t/T)) exp(i E t) dts
    int obs_axA, obs_axB, obs_axL;    // lattice axes of ia, ib (-1: absent) and of the line
    double obs_dx[3];         // dx of those three
    int obs_half[3];          // n/2 of those three (grid of reading G14)
};

using RingLaunchFn = cudaError_t (*)(const RingArgs &, unsigned threads, size_t smem, unsigned grid, cudaStream_t st);

// strided-axis passes through the same ring, tiles moved as TMA tensor boxes (sso_sring.cuh)
// KD2 / KD4 read the Dirac kinetic scalars from a table, KD2F / KD4F evaluate them in the pass ("on the fly")
enum : int { SMODE_KS = 0, SMODE_KD2 = 1, SMODE_KD4 = 2, SMODE_DIF = 3, SMODE_DIT = 4, SMODE_KD2F = 5, SMODE_KD4F = 6 };
struct SRingArgs {
    void *psi;                // device base of psi (stores from registers; loads go through the tensor map)
    long long inner;          // element stride along the line
    long long comp_stride;    // elements between components
    const void *tw;           // twiddle blocks of the line axis
    int ntiles;               // tiles of TL adjacent lines (x all components when they are independent)
    int TL;                   // adjacent lines per tile: one row of a tile is TL complex numbers, contiguous in memory
    int pitch;                // padded line pitch of the exchange layout (complex elements)
    int G, GT, NB, bufstride; // groups, threads per group (CC * TL * N/16), pool buffers (any number >= 1), elements between buffers
    int tiles_per_outer;      // inner / TL
    int box_rows;             // rows per TMA box (<= 256); a tile is CC * N / box_rows boxes
    int rest1;                // line = ia * rest1 + ib on the non-line axes
    int rest1_shift, tpo_shift;  // log2 of rest1 and tiles_per_outer (lattice sizes are powers of two)
    // kinetic factor (step-dependent shifts are resolved on the host)
    const void *kph0, *kph1, *kph2;  // Schroedinger phase tables (PassArgs)
    const double *kv0, *kv1, *kv2;   // Dirac k grids (PassArgs)
    double sh[3];                    // q Abar_n per axis (SSO_FIELD_A), else 0
    const void *ktab;                // Dirac table modes: double2 (cos(E tau), sin(E tau)/E) / Ntot per k point, [slot of axis 0][inner]
    double mass, clight, dt, scale;
    int ndim;
    int rev;                         // tiles in descending order
    int fast_trig;                   // Dirac: |E tau| < 2^30 for every k point, the kernel may use its own quadrant reduction
};
// bytes of the line table a strided pass keeps in shared memory (multiple of 128): the Schroedinger kinetic phases
// of the line axis (complex[N]) or the Dirac momenta c (k_0 - q Abar_0) (double[N])
__host__ __device__ constexpr int sring_line_table_bytes(int smode, int N, int esz) {
    return smode == SMODE_KS ? (N * esz + 127) / 128 * 128 : ((smode == SMODE_DIF || smode == SMODE_DIT) ? 0 : (N * 8 + 127) / 128 * 128);
}
using SRingLaunchFn = cudaError_t (*)(const SRingArgs &, const void *tensor_map, unsigned threads, size_t smem, unsigned grid, cudaStream_t st);
#define SSO_DECL_SRING(N)                            \
    SRingLaunchFn sso_sring_lookup_f32_##N(int mode); \
    SRingLaunchFn sso_sring_lookup_f64_##N(int mode);
SSO_FOR_EACH_N(SSO_DECL_SRING)
#undef SSO_DECL_SRING
#define SSO_DECL_RING(N)                                  \
    RingLaunchFn sso_ring_lookup_f32_##N(int mode, int maxt); \
    RingLaunchFn sso_ring_lookup_f64_##N(int mode, int maxt);
SSO_FOR_EACH_N(SSO_DECL_RING)
#undef SSO_DECL_RING

// the persistent 1D Schroedinger kernel of sso_line1d.cuh
struct Line1dArgs;
using Line1dLaunchFn = cudaError_t (*)(const Line1dArgs &, size_t smem, cudaStream_t st);
#define SSO_DECL_LINE1D(N)                      \
    Line1dLaunchFn sso_line1d_lookup_f32_##N(); \
    Line1dLaunchFn sso_line1d_lookup_f64_##N();
SSO_FOR_EACH_N(SSO_DECL_LINE1D)
#undef SSO_DECL_LINE1D

// the cluster version (sso_line1d_cluster.cuh): lookup by the per-CTA length M = N / CS and the cluster size CS
struct Line1dClusterArgs;
using Line1dClusterLaunchFn = cudaError_t (*)(const Line1dClusterArgs &, size_t smem, cudaStream_t st);
#define SSO_DECL_LINE1D_CL(N)                                  \
    Line1dClusterLaunchFn sso_line1d_cluster_lookup_f32_##N(int cs); \
    Line1dClusterLaunchFn sso_line1d_cluster_lookup_f64_##N(int cs);
SSO_FOR_EACH_N(SSO_DECL_LINE1D_CL)
#undef SSO_DECL_LINE1D_CL

}  // namespace sso
