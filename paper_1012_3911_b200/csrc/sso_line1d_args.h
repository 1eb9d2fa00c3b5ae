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

}  // namespace sso
