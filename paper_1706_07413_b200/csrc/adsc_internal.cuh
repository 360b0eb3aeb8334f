// adsc_internal.cuh — shared declarations of libadsc (CUDA path only; nothing here is
// used by, or taken from, oracle/).  Notation follows include/adsc.h and DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <cstddef>
#include <cstdint>
#include <string>

#include "../../include/adsc.h"

namespace adsc {

constexpr int HAL = 4;            // table halo on each side (3 used by the widest stencil)
constexpr int GEN_TILE = 1024;    // points per CTA tile of the streaming kernels
constexpr int GEN_THREADS = 256;  // 4 points per thread
constexpr int SP_MAX_CTAS = 1024; // persistent streaming kernel: at most this many CTAs (groups * G) have a mailbox in the workspace
constexpr int SA_MBOX = 40;       // ... doubles per chunk mailbox: 17 slots {value, stamp} + padding (adsc_stream_async.cu)

// Per-member record kept on the device (copied to the host by adsc_diagnostics).
struct MemberRec {
    long long steps_done;
    double t_collapse;
    double min_A;
    double mass;
    double resid;
    int argmin_A;
    int collapsed;
    int bad;        // streaming path: set by stage 4 / re-solve when !(A_i >= thr) for some i
    int pad;
};

// Coefficient tables, each of length NP + 2*HAL, pointer already offset so that
// index i in [-HAL, N-1+HAL] is valid; ghosts hold the mirrored values.
struct Tables {
    const double *sc;    // sin x cos x          parity (-,-), sc[0]=sc[N-1]=0
    const double *T;     // tan^2 x              parity (+,+), T[N-1]=0 (never used as a value)
    const double *C;     // cot^2 x              parity (+,+), C[0]=C[N-1]=0 (never used)
    const double *c3s;   // cos^3 x / sin x      c3s[0]=c3s[N-1]=0 (never used)
    const double *w;     // Simpson weights, 0 outside [0,N-1]
};

struct Problem {
    int N, NP, B;
    int fixed_bg;        // PAPER.md:177 (Table II): A and delta held fixed at 1 and 0 -- no scan, no exp, A not evolved
    double h, dt, ko_eps, thr;
};

// Device pointers into the caller's workspace.
struct Workspace {
    double *U[3];        // state Phi, Pi, A          [B][NP]
    double *Ua[3];       // generic streaming: stage state ping; persistent streaming: u^n in the permuted layout
    double *Ub[3];       // streaming: stage state pong
    double *ACC[3];      // streaming: u^n + dt/6 * partial sum
    double *dl;          // streaming: tile-local suffix sums of I; also delta scratch
    double *Ac;          // scratch: A from eq (5) (diagnostics)
    double *tot;         // streaming: [B][ntiles] tile totals
    double *carry;       // streaming: [B][ntiles] exclusive suffix of tot
    double *tot2, *carry2;   // tiled constraint solve: tile totals / exclusive prefix of the A integrand
    double *part;        // tiled constraint solve: [B][ntiles][6] diagnostics partials
    double *stage[2];    // host staging [B][N]
    double *sp_mbox;     // persistent streaming: [groups][2][G][SA_MBOX] chunk mailboxes (room for SP_MAX_CTAS chunks)
    double *tab;         // 5 tables
    double *tabp;        // persistent streaming: -2 sc, tan^2, cot^2/(12h) permuted per 256-point slice [NP/256][3][256]
    MemberRec *rec;      // [B]
};

struct Layout {
    size_t off_U[3], off_Ua[3], off_Ub[3], off_ACC[3], off_dl, off_Ac, off_tot, off_carry, off_tot2, off_carry2, off_part,
        off_stage[2], off_tab, off_tabp, off_rec, off_mbox, total;
    int ntiles;
};

}  // namespace adsc

struct adsc_ctx {
    adsc::Problem pb;
    double courant;
    int K_A;                 // A re-solve period (0 = never)
    int path_opt;            // ADSC_OPT_PATH
    long long steps_per_launch;
    int path;                // resolved: 1 streaming (persistent), 2 resident, 3 streaming (one kernel per phase)
    int cluster;             // CTAs per member (resident)
    int res_cfg;             // index into the resident configuration table
    bool bound, have_state;
    cudaStream_t stream;
    void *ws_base;
    adsc::Layout lay;
    adsc::Workspace ws;
    adsc::Tables tb;
    long long launches;
    long long global_step;   // steps since set_initial (lock-step over active members)
    int dev_sms;
    int dev_smem_optin;
    bool sp_ok;              // persistent streaming kernel usable (decided at adsc_bind)
    int sp_G, sp_groups, sp_SQ;   // chunks per member, concurrent members, 256-point slices per chunk
    int sms_hint;            // SM count assumed for the layout (the device's if one was visible at adsc_create, else 148)
    int spread;              // ADSC_OPT_SPREAD: narrower segments for ensembles that do not fill the device
    int spread_cap;          // ... largest cluster the spread choice may use (8; lowered at adsc_bind when the device holds fewer clusters than members)
    int rk_order;            // 4 (classical RK4, default), 3 (Heun's third-order rule) or 2 (explicit midpoint): R12, R25
    std::string err;
};

namespace adsc {

// Runge-Kutta rules in the form every kernel uses: u_{s+1} = u^n + a_next[s] k_s, u^{n+1} = u^n + sum_s b_w[s] k_s
// (weights already multiplied by dt).  PAPER.md:57; R12 (classical RK4), R25 (Heun 3, explicit midpoint).
inline void rk_tableau(int order, double dt, double a_next[4], double b_w[4])
{
    for (int s = 0; s < 4; ++s) { a_next[s] = 0.0; b_w[s] = 0.0; }
    if (order == 2) { a_next[0] = 0.5 * dt; b_w[1] = dt; }
    else if (order == 3) { a_next[0] = dt / 3.0; a_next[1] = 2.0 * dt / 3.0; b_w[0] = 0.25 * dt; b_w[2] = 0.75 * dt; }
    else {
        a_next[0] = 0.5 * dt; a_next[1] = 0.5 * dt; a_next[2] = dt;
        b_w[0] = dt / 6.0; b_w[1] = dt / 3.0; b_w[2] = dt / 3.0; b_w[3] = dt / 6.0;
    }
}

void set_thread_error(const std::string &msg);               // adsc_api.cu: message for adsc_last_error(NULL) on this thread

// ---- launchers implemented in the .cu files (all asynchronous on ctx->stream) -----------
cudaError_t launch_tables(adsc_ctx *c);
cudaError_t launch_pack(adsc_ctx *c, const double *src, int field, bool init_rec);
cudaError_t launch_unpack(adsc_ctx *c, const double *src_internal, double *dst);
cudaError_t launch_fill(adsc_ctx *c, double *dst_internal, double value);   // whole [B][NP] array
// mode bits for launch_solve
enum { SOLVE_WRITE_A = 1, SOLVE_DIAG = 2, SOLVE_ACTIVE_ONLY = 4 };
cudaError_t launch_solve(adsc_ctx *c, int mode);              // one CTA per member, or the tiled kernels for long members
cudaError_t launch_solve_tiled(adsc_ctx *c, int mode);        // adsc_solve_tiled.cu (streaming layouts only)
constexpr int SOLVE_TILED_MIN_N = 32768;                      // members at least this long use the tiled solve
cudaError_t launch_finalize(adsc_ctx *c, int inc_steps);
// adsc_modes.cu; d_out [B][J]; scratch for the slice partials (at least 2 B J doubles)
cudaError_t launch_mode_energies(adsc_ctx *c, int J, double *d_out, double *scratch, size_t scratch_doubles);
cudaError_t launch_stream_step(adsc_ctx *c);                 // one RK4 step, generic streaming kernels
// persistent streaming kernel (adsc_stream_async.cu): chunks per member, slices per chunk, concurrent members
bool stream_async_select(int N, int B, int sms, int *G, int *SQ, int *groups);
cudaError_t launch_tabp(adsc_ctx *c);                        // permuted coefficient tables for its bulk copies
cudaError_t launch_stream_async(adsc_ctx *c, long long nsteps, int check_last);
cudaError_t launch_resident(adsc_ctx *c, long long nsteps, int check_last);  // resident path
bool resident_select(adsc_ctx *c);                           // fills c->cluster, c->res_cfg
cudaError_t resident_check(adsc_ctx *c, int *clusters);      // at adsc_bind: clusters of the selected kernel the device holds at once
const char *resident_cfg_name(int cfg);

// ---- device helpers ----------------------------------------------------------------------
#ifdef __CUDACC__

// Mirror a (possibly ghost) index into [0, N-1] and return the parity sign to apply:
// u_{-k} = p0 u_k, u_{N-1+k} = ppi u_{N-1-k}  (readings R2, R3).
__device__ __forceinline__ int mirror(int j, int N, int p0, int ppi, double &sgn)
{
    sgn = 1.0;
    if (j < 0) { j = -j; sgn = (double)p0; }
    else if (j > N - 1) { j = 2 * (N - 1) - j; sgn = (double)ppi; }
    return j;
}

__device__ __forceinline__ double ld_ghost(const double *__restrict__ u, int j, int N, int p0, int ppi)
{
    double s;
    int k = mirror(j, N, p0, ppi, s);
    return s * u[k];
}

// Inclusive suffix sum over the lanes of a warp: lane l gets sum_{m>=l} v_m.
__device__ __forceinline__ double warp_suffix_incl(double v)
{
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        double o = __shfl_down_sync(0xffffffffu, v, d);
        if (lane + d < 32) v += o;
    }
    return v;
}

// Inclusive prefix sum over the lanes of a warp: lane l gets sum_{m<=l} v_m.
__device__ __forceinline__ double warp_prefix_incl(double v)
{
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        double o = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += o;
    }
    return v;
}

#endif  // __CUDACC__

}  // namespace adsc
