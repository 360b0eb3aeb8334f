// adsc_resident.cuh — declarations shared by the resident kernels (adsc_resident*.cu).
#pragma once
#include "adsc_internal.cuh"

namespace adsc {

struct ResParams {
    Problem pb;
    Tables tb;
    double *U[3];
    MemberRec *rec;
    long long nsteps;
    int check_last;   // 0: the caller re-solves A after the last step and tests collapse itself
    int CL;
};

// One compiled (points per thread, threads per CTA) configuration of a resident kernel.
struct ResConfig {
    const char *name;
    int P, threads, seg;
    bool acc_reg;
    size_t smem;
    const void *fn_single, *fn_multi;
};

// generation-2 table (adsc_resident2.cu)
extern const ResConfig g_cfgs2[];
extern const int n_cfgs2;

}  // namespace adsc
