// sso_line1d_args.h -- launch descriptor of the persistent 1D Schroedinger kernel (sso_line1d.cuh)
#pragma once

namespace sso {

struct Line1dArgs {
    void *psi;          // device complex[N]
    const void *tw;     // twiddle blocks (PassArgs)
    const void *vtab;   // natural order: complex exp(-i V tau/2) (VREP_TABLE) or real angle -V tau/2 (VREP_ANGLE)
    int vrep;
    const void *kph0;   // complex[N] kinetic phases incl. 1/N, slot order
    int nsteps;         // >= 1
};

// the receive buffer of the cluster kernel shares the line buffer for M = 4096 (shared memory would not suffice)
#if defined(__CUDACC__)
__host__ __device__
#endif
constexpr bool line1d_cluster_alias(int M) { return M >= 4096; }

// the same steps with the line spread over a thread-block cluster (sso_line1d_cluster.cuh): N = CS * M
struct Line1dClusterArgs {
    void *psi;          // device complex[N]
    const void *tw;     // twiddle blocks of the M-point transform (PassArgs)
    const void *tcl;    // complex [CS][CS - 1][M / CS]: w_N^(m k1) for the m values r M/CS + mm of CTA r, k1 = 1 .. CS-1
    const void *vtab;   // natural order: complex exp(-i V tau/2) (VREP_TABLE) or real angle -V tau/2 (VREP_ANGLE)
    int vrep;
    const void *kph;    // complex [CS][M]: kinetic phases incl. 1/N of the frequencies k1 + CS k2, row k1 in the slot
                        // order of the M-point transform
    int nsteps;         // >= 1
};

}  // namespace sso
