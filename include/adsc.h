/*
 * adsc.h — C ABI of libadsc: batched RK4 time step of the spherically symmetric
 * Einstein-Klein-Gordon system in AdS4 (Liebling & Khanna, arXiv:1706.07413,
 * Sec. II; cited below as PAPER.md:<line>), on one NVIDIA B200 (sm_100a).
 *
 * State per ensemble member: Phi = phi', Pi = e^{delta} phi_t / A and the metric
 * function A on the uniform grid x_i = i*h, h = (pi/2)/(N-1), i = 0..N-1
 * (PAPER.md:39-41).  delta is not stored: it is re-integrated from Phi, Pi
 * (eq (6)) at every Runge-Kutta stage by an on-device prefix scan,
 * which replaces the paper's per-step host round trip.
 *
 * Conventions for every entry point
 *   - "device pointer": memory of the CUDA device that was current when
 *     adsc_bind was called; "host pointer": ordinary host memory.
 *   - External field layout: row-major [batch][N] doubles, member b at
 *     ptr + b*N; rows need only 8-byte alignment.
 *   - The caller owns every buffer it passes (workspace, fields, host_out).
 *     The library owns only the handle; it never frees caller memory and keeps
 *     no field pointer after a call returns (the workspace pointer is kept
 *     until adsc_destroy or the next adsc_bind).
 *   - All work is enqueued on the stream given to adsc_bind.  Calls return
 *     without synchronising unless stated.
 *   - int-returning functions give ADSC_OK (0) or a negative ADSC_E* code; the
 *     message is available from adsc_last_error.  Nothing throws or exits.
 *   - Collapse of a member is not an error; it is reported per member.
 *   - There is no CPU fallback: without a CUDA device every compute call
 *     returns ADSC_ECUDA.
 */
#ifndef ADSC_H
#define ADSC_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ADSC_OK       0
#define ADSC_EINVAL  -1   /* bad argument                                        */
#define ADSC_ESTATE  -2   /* call order (e.g. step before bind / set_initial)    */
#define ADSC_ENOMEM  -3   /* workspace too small / host allocation failed        */
#define ADSC_ECUDA   -4   /* CUDA runtime error; text in adsc_last_error         */

/* adsc_set_option keys */
#define ADSC_OPT_COLLAPSE_THRESHOLD 1  /* thr: member collapses when !(min_i A_i >= thr)
                                          (PAPER.md:85).  Default 2^-7; paper uses 0.01. */
#define ADSC_OPT_A_RESOLVE_PERIOD   2  /* K_A: every K_A steps A is replaced by the
                                          integral of eq (5) ("periodically integrating
                                          A").  Default 0 = never.          */
#define ADSC_OPT_PATH               3  /* 0 auto (default: resident if a member fits on
                                          chip, else streaming); 1 force the streaming path
                                          (persistent kernel: stage state in shared memory,
                                          coefficient tables staged by bulk asynchronous
                                          copies, u^n and accumulator in global memory; it
                                          needs N-1 to be a multiple of 8 and all CTAs of a
                                          member co-resident, and falls back to 3 otherwise;
                                          its layout depends on the SM count of the device that
                                          is current at adsc_create: adsc_bind on a device with
                                          another SM count returns ESTATE when 1 was forced);
                                          2 force the resident (shared-memory/register)
                                          kernel, EINVAL if it cannot hold N; 3 force the
                                          generic streaming kernels (one launch per phase,
                                          any N).                                        */
#define ADSC_OPT_STEPS_PER_LAUNCH   4  /* resident path: RK4 steps per kernel launch
                                          (default 0 = all steps of a call in one launch) */

#define ADSC_OPT_FIXED_BACKGROUND    7  /* 1: evolve on the fixed background A = 1, delta = 0 (the
                                          paper's second workload, Table II): the
                                          delta integration, the exponential and the A update are
                                          compiled out of the stage kernels; adsc_set_initial sets
                                          A = 1 without solving eq (5); K_A is ignored; no member
                                          ever collapses; adsc_get_fields returns delta = 0; the
                                          diagnostics use A = 1 (mass = linear energy, residual =
                                          max |1 - A^c|).  Set it before adsc_bind (ESTATE
                                          afterwards).  Default 0.                              */

#define ADSC_OPT_RK_ORDER            8  /* 4 (default): classical RK4; 3: Heun's third-order rule; 2:
                                          explicit midpoint ("second, third, and fourth order accurate
                                          Runge-Kutta"; tableaux are readings R12, R25).
                                          All three step paths implement them.  Together with
                                          ADSC_OPT_FIXED_BACKGROUND (the paper's Table II runs:
                                          PAPER.md:57 + :177) orders 3 and 2 are supported on the two
                                          streaming paths only: the resident kernel has no build of
                                          that combination, auto then picks a streaming path and
                                          ADSC_OPT_PATH = 2 returns EINVAL.  Set it before adsc_bind. */

#define ADSC_OPT_SPREAD              9  /* 1: latency mode for ensembles that do not fill the device: the resident path cuts
                                          every member into more, shorter CTAs (clusters of up to 8 CTAs of at least 256
                                          points) as long as all clusters of the ensemble are still co-resident, so that
                                          more SMs work on each member (one member of N = 1025: 4 CTAs, 3.8 instead of
                                          4.5 microseconds per RK4 step).  Same arithmetic, same results up to the order
                                          of the scan sums.  Default 0 (widest segment: best throughput for ensembles
                                          that fill the device).  Set it before adsc_bind; adsc_bind asks the device
                                          how many clusters it really holds at once and steps back to wider segments
                                          until all members' clusters are co-resident (adsc_path tells the outcome). */

typedef struct adsc_ctx *adsc_handle;

/* One record per member, filled by adsc_diagnostics (host memory). */
typedef struct {
    double    t;                    /* steps_done*dt (= t_collapse once collapsed)          */
    long long steps_done;           /* RK4 steps taken by this member                       */
    double    min_A;                /* min_i A_i of the current state (NaNs ignored)        */
    int       argmin_A;             /* smallest i attaining min_A                           */
    int       collapsed;            /* 1 once !(min_i A_i >= thr) was seen after a step     */
    double    mass;                 /* M = int_0^{pi/2} tan^2 x A (Phi^2+Pi^2) dx,
                                       composite Simpson                      */
    double    constraint_residual;  /* max_i |A_i - A^c_i|, A^c = integral of eq (5)
                                                                           */
    double    t_collapse;           /* time of the step that tripped thr; NaN if none       */
} adsc_diag;

/* Create a solver for `batch` members on N grid points.
 *   N        >= 9 and odd (Simpson needs N-1 even)
 *   batch    1..65535 members (independent evolutions); N*batch <= 4e9
 *   courant  dt = courant*h, 0 < courant <= 1 (method-of-lines RK4)
 *   ko_eps   >= 0: Kreiss-Oliger coefficient of the 7-point dissipation added to the
 *            right-hand sides of Phi and Pi (BASELINE.json configs[0]; not in the paper)
 * Host-only: launches nothing and allocates nothing on a device (it only asks the CUDA runtime for the SM count
 * of the current device, if there is one, to size the streaming layout).  Returns NULL on bad arguments or host
 * OOM; the message is kept per calling thread for adsc_last_error(NULL). */
adsc_handle adsc_create(int N, int batch, double courant, double ko_eps);

/* Release the handle (not the workspace).  NULL is allowed. */
int adsc_destroy(adsc_handle h);

/* Bytes of device workspace adsc_bind needs (state, stage buffers, tables,
 * per-member records).  0 if h is NULL. */
size_t adsc_workspace_bytes(adsc_handle h);

/* Attach device workspace (256-byte aligned, >= adsc_workspace_bytes) and the
 * CUDA stream (a cudaStream_t cast to void*; NULL = legacy default stream) all
 * later calls run on.  Builds the coefficient tables on the device.
 * Invalidates any state previously set. */
int adsc_bind(adsc_handle h, void *d_workspace, size_t bytes, void *cuda_stream);

/* Set an option (keys above).  Allowed any time after adsc_create. */
int adsc_set_option(adsc_handle h, int key, double value);

/* Initial data: copies Phi(x,0), Pi(x,0) from device pointers
 * [batch][N], forces Phi_0 = Phi_{N-1} = Pi_{N-1} = 0 (eqs (7),(9),(10)), integrates
 * eq (6) for delta with delta(pi/2)=0 (eq (12)) and eq (5) for A with A(0)=A(pi/2)=1
 * (eqs (8),(11)); resets step counters and collapse flags.  Asynchronous. */
int adsc_set_initial(adsc_handle h, const double *d_Phi, const double *d_Pi);

/* Exact resume: like adsc_set_initial but A is taken from d_A instead of being
 * integrated (A is evolved by eq (4)).  Counters reset. */
int adsc_set_state(adsc_handle h, const double *d_Phi, const double *d_Pi, const double *d_A);

/* Advance every non-collapsed member by nsteps classical RK4 steps of
 * eqs (2)-(4): 4th-order centred differences in flux form with parity
 * ghosts at x=0 and x=pi/2, KO dissipation, delta re-integrated at every stage, A evolved
 * pointwise; after each step the collapse test of PAPER.md:85.  A member that collapses
 * is frozen at the state that tripped the threshold.  nsteps >= 0.  Asynchronous. */
int adsc_step(adsc_handle h, long long nsteps);

/* Reduce per-member diagnostics on the device, synchronise the stream and copy
 * batch records to host_out[batch] (host pointer). */
int adsc_diagnostics(adsc_handle h, adsc_diag *host_out);

/* Copy the current fields to device pointers [batch][N]; any pointer may be NULL.
 * d_delta is integrated from the current Phi, Pi.  Asynchronous. */
int adsc_get_fields(adsc_handle h, double *d_Phi, double *d_Pi, double *d_A, double *d_delta);

/* Convenience for host buffers (used by the end-to-end benchmark): the same as
 * adsc_set_initial / adsc_get_fields but with HOST pointers; the library stages
 * them through its workspace with cudaMemcpyAsync on the bound stream and, for
 * the getter, synchronises before returning. */
int adsc_set_initial_host(adsc_handle h, const double *h_Phi, const double *h_Pi);
int adsc_get_fields_host(adsc_handle h, double *h_Phi, double *h_Pi, double *h_A, double *h_delta);
/* The same without the final synchronisation: the copies are only ENQUEUED on the bound stream; the caller
 * synchronises that stream (or calls adsc_diagnostics, which does) before reading the host buffers, which should
 * be pinned for the copies to overlap other streams' work.  Lets sub-batches on different handles / streams
 * pipeline their transfers against each other's kernels. */
int adsc_get_fields_host_async(adsc_handle h, double *h_Phi, double *h_Pi, double *h_A, double *h_delta);

/* Normal-mode spectrum of the current state ("the current numerical solution can be
 * decomposed into a spectrum of normal modes").  For the AdS4 modes e_j (R19),
 * j < J <= 32: Pi_j = int Pi e_j tan^2 x dx, Phi_j = int Phi e_j' tan^2 x dx (composite Simpson, integrand 0
 * at x = pi/2), E_j = Pi_j^2 + Phi_j^2 / omega_j^2, omega_j = 3 + 2j (R24).  host_out: HOST array
 * [batch][J], row-major, owned by the caller.  Two kernel launches (slice partials over several CTAs per member,
 * then a fixed-order sum) plus one small D2H copy; synchronises the stream.  EINVAL for J outside 1..32, J > N/4
 * or a NULL pointer, ESTATE before adsc_set_initial. */
int adsc_mode_energies(adsc_handle h, int J, double *host_out);

/* The same spectrum for callers that are not allowed to allocate GPU memory, and have none to spare for a workspace.
 * Who that is: a program that gave the whole GPU to its own memory pool when it started (a training or serving
 * process with a caching allocator, a client running under a fixed per-process memory limit), so that a cudaMalloc
 * made behind its back fails or breaks its accounting; and code on a latency-critical path, where cudaMalloc and
 * cudaFree are ruled out because they stall the whole device while they run.  Such a caller can still pass its own
 * arrays, so this entry point takes the fields and the result as plain device pointers, needs no handle and no
 * workspace, and keeps the one thing the computation needs beyond them, the per-slice partial sums of the two
 * kernels, in an array of ADSC_STATIC_SCRATCH_BYTES that is built into the library.  It calls no cudaMalloc, no
 * cudaFree and no library routine that allocates.
 *   d_Phi, d_Pi  DEVICE pointers, [batch][N] doubles row-major, 8-byte aligned, read only.  Phi_{N-1}, Pi_{N-1} and
 *                Phi_0 do not enter (the integrands vanish there), so the result equals adsc_mode_energies of a
 *                handle whose state was set from the same two arrays.
 *   d_E          DEVICE pointer, [batch][J] doubles, written.
 *   cuda_stream  a cudaStream_t cast to void* (NULL = legacy default stream) on the device that is current at the
 *                call; the pointers must belong to that device.  Two kernels are enqueued; the call does not wait.
 * Limits: N odd and >= 9, 1 <= J <= 32, J <= N/4, and batch * J <= ADSC_STATIC_SCRATCH_BYTES / 16 (= 131072; e.g.
 * 4096 members at J = 32).  Beyond that the call returns ADSC_EINVAL and says so in adsc_last_error(NULL); cut the
 * batch into pieces or use adsc_mode_energies.  The price of the built-in array: every GPU on which the library's
 * code gets loaded holds those 2 MiB until the process ends, whether or not this function is ever called.
 * First call on each device: it looks up where the built-in array lives on that device (cudaGetSymbolAddress, which
 * may also be the moment the CUDA runtime loads the library's code there) and remembers it.  Make that first call
 * during start-up, before any stream capture is begun; later calls only launch the two kernels.
 * Sharing: there is ONE such array per device and every call on that device uses it, whatever the stream or thread.
 * Each call overwrites all the slots it later reads, so nothing has to be cleared and stale contents of the previous
 * call are harmless; but two calls whose kernels can run at the same time on one device (different streams, no
 * event between them) write the same slots and corrupt each other.  Keep the calls of one device on one stream, or
 * order them with events.
 * Errors: ADSC_EINVAL (arguments, limit), ADSC_ECUDA (no device, launch failure); text from adsc_last_error(NULL) on
 * the calling thread.  (R19, R24.) */
#define ADSC_STATIC_SCRATCH_BYTES (2u << 20)
int adsc_mode_energies_static(int N, int batch, int J, const double *d_Phi, const double *d_Pi, double *d_E,
                              void *cuda_stream);

/* Roofline denominators measured on the current CUDA device ("a DFMA issue-rate probe and a
 * shared-memory bandwidth probe"; none of the method's arithmetic).  kind ADSC_PROBE_FP64_FMA: *result = flop/s of
 * independent FP64 fused multiply-adds on every SM (2 flop each); ADSC_PROBE_SHARED_LOAD: *result = bytes/s of
 * conflict-free 128-bit shared-memory loads on every SM.  Runs its own kernel for about target_ms milliseconds on a
 * private stream and synchronises; needs no handle.  result is a HOST pointer.  EINVAL on bad arguments, ECUDA
 * without a device. */
#define ADSC_PROBE_FP64_FMA    0
#define ADSC_PROBE_SHARED_LOAD 1
int adsc_probe(int kind, double target_ms, double *result);

/* Self-test of the one transcendental on the hot path (e^{-delta} of eqs (2), (3)): evaluates the
 * kernels' own exponential routine on ngroups groups of 8 arguments (h_x[8*g .. 8*g+7], the 8 points one thread
 * owns; the last one is the group's reference point) and returns the results h_E[8*ngroups] and, per group, which
 * evaluation the routine chose: h_tier[g] = 0, 1, 2 for the relative polynomial with 2, 3, 5 terms (largest
 * |x_p - x_7| <= 2^-14, 2^-10, 2^-6), 3 for one full evaluation per point.  HOST pointers, owned by the caller;
 * synchronous; allocates and frees its own device scratch.  EINVAL on bad arguments, ECUDA without a device. */
int adsc_selftest_exp(int ngroups, const double *h_x, double *h_E, int *h_tier);

/* Number of kernels this handle has launched since adsc_bind (for gpu_launches). */
long long adsc_launch_count(adsc_handle h);

/* Which kernel family adsc_step uses for this handle (final after adsc_bind): 1 persistent
 * streaming, 2 resident, 3 generic streaming; *cluster (may be NULL) receives the CTAs
 * per member (cluster size of the resident path, chunks of the persistent streaming path). */
int adsc_path(adsc_handle h, int *cluster);

/* Text of the last error on this handle (or of the last failed adsc_create if
 * h is NULL).  Never NULL; valid until the next call on the handle. */
const char *adsc_last_error(adsc_handle h);

#ifdef __cplusplus
}
#endif
#endif /* ADSC_H */
