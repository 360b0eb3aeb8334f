// adsc_resident.cuh — declarations shared by the resident kernels (adsc_resident*.cu).
#pragma once
#include "adsc_internal.cuh"

namespace adsc {

// Scalars derived from (h, dt, ko_eps, thr) on the host once per launch.  They sit in the kernel
// parameter (constant) bank, so fp64 instructions take them as c[][] operands and no register
// holds them (generation 3; generations 1 and 2 derive them in the kernel).
struct ResConsts {
    double d4c;             // 1/(12 h)                      D4 weight
    double kw[4];           // eps_KO/(64 h) * {-20, 15, -6, 1}   KO weights by distance
    double hh;              // h/2            } telescoped delta rule for f' = -2 f
    double c25, c12, c1;    // 25h/48, h/4, h/48
    double inv12h2;         // 1/(12 h^2)     boundary flux limit (R5)
    double c_org;           // 1/(2 h)        origin l'Hopital (R4)
    double a_next[4];       // dt/2, dt/2, dt, 0      stage-state weights
    double b_w[4];          // dt/6, dt/3, dt/3, dt/6 accumulator weights
    double thr;
};

struct ResParams {
    Problem pb;
    Tables tb;
    double *U[3];
    MemberRec *rec;
    long long nsteps;
    int check_last;   // 0: the caller re-solves A after the last step and tests collapse itself
    int CL;
    ResConsts k;
};

// One compiled (points per thread, threads per CTA) configuration of a resident kernel.
// fn[j] is the kernel for a cluster of 2^j CTAs per member (nullptr: not available); if any_cl,
// fn[1] takes the cluster size at run time and serves every size 2..8.
struct ResConfig {
    const char *name;
    int P, threads, seg;
    bool acc_reg;
    size_t smem;
    bool any_cl;
    const void *fn[4];
    const void *fnf[4];    // the same for the fixed background A = 1, delta = 0 (nullptr: not compiled)
    const void *fn3[4];    // Runge-Kutta order 3 (Heun), dynamical metric
    const void *fn2[4];    // Runge-Kutta order 2 (explicit midpoint), dynamical metric
};

// generation-3 table (adsc_resident3.cu); the generation-1 table is local to adsc_resident.cu
extern const ResConfig g_cfgs3[];
extern const int n_cfgs3;

}  // namespace adsc
