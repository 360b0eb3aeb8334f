// adsc_api.cu — the C ABI of include/adsc.h: argument checks, workspace carving, and the
// order in which kernels are enqueued.  No field arithmetic happens on the host.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "adsc_internal.cuh"

using namespace adsc;

static thread_local std::string g_create_error = "";   // per calling thread: adsc_create has no handle to hang it on

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// For entry points that take no handle: the text adsc_last_error(NULL) returns on this thread.
void adsc::set_thread_error(const std::string &msg) { g_create_error = msg; }

static void compute_layout(adsc_ctx *c)
{
    Layout &L = c->lay;
    const size_t field = align_up((size_t)c->pb.B * c->pb.NP * sizeof(double), 256);
    const size_t ext = align_up((size_t)c->pb.B * c->pb.N * sizeof(double), 256);
    L.ntiles = (c->pb.N + GEN_TILE - 1) / GEN_TILE;
    const size_t tiles = align_up((size_t)c->pb.B * L.ntiles * sizeof(double), 256);
    const bool stream = (c->path != 2);
    size_t off = 0;
    for (int v = 0; v < 3; ++v) { L.off_U[v] = off; off += field; }
    for (int v = 0; v < 3; ++v) { L.off_Ua[v] = off; off += stream ? field : 0; }
    for (int v = 0; v < 3; ++v) { L.off_Ub[v] = off; off += stream ? field : 0; }
    for (int v = 0; v < 3; ++v) { L.off_ACC[v] = off; off += stream ? field : 0; }
    L.off_dl = off; off += field;
    L.off_Ac = off; off += field;
    L.off_tot = off; off += stream ? tiles : 0;
    L.off_carry = off; off += stream ? tiles : 0;
    L.off_tot2 = off; off += stream ? tiles : 0;
    L.off_carry2 = off; off += stream ? tiles : 0;
    L.off_part = off; off += stream ? 6 * tiles : 0;
    for (int k = 0; k < 2; ++k) { L.off_stage[k] = off; off += ext; }
    L.off_tab = off; off += align_up((size_t)5 * (c->pb.NP + 2 * HAL) * sizeof(double), 256);
    L.off_tabp = off; off += (c->path == 1) ? align_up((size_t)3 * c->pb.NP * sizeof(double), 256) : 0;
    L.off_rec = off; off += align_up((size_t)c->pb.B * sizeof(MemberRec), 256);
    L.off_mbox = off; off += align_up((size_t)SP_MAX_CTAS * 2 * SA_MBOX * sizeof(double), 256);   // [groups][2][G][SA_MBOX], groups * G <= SP_MAX_CTAS
    L.total = off;
}

// Row pitch of the persistent streaming layout: G chunks of SQ 256-point slices hold the points 0..N-2; the row must
// also hold the point N-1, so one more slice is added when the chunks end exactly there.
static int sa_row_pitch(int N, int G, int SQ)
{
    const int np = G * SQ * 256;
    return np >= N ? np : np + 256;
}

// Which kernel family steps this handle, and the internal row pitch NP that goes with it: rows are padded to a
// multiple of 4 points, except on the persistent streaming path, whose rows are G chunks of SQ 256-point slices.
static void resolve_path(adsc_ctx *c)
{
    const bool can_res = resident_select(c);
    const bool can_sa = stream_async_select(c->pb.N, c->pb.B, c->sms_hint, &c->sp_G, &c->sp_SQ, &c->sp_groups);
    c->sp_ok = can_sa;
    if (c->path_opt == 3) c->path = 3;
    else if (c->path_opt == 1) c->path = can_sa ? 1 : 3;
    else if (c->path_opt == 2) c->path = can_res ? 2 : 0;
    else c->path = can_res ? 2 : (can_sa ? 1 : 3);
    if (c->path != 2) c->cluster = 1;
    c->pb.NP = (c->path == 1) ? sa_row_pitch(c->pb.N, c->sp_G, c->sp_SQ) : (c->pb.N + 3) / 4 * 4;
    compute_layout(c);
}

static int fail(adsc_ctx *c, int code, const std::string &msg)
{
    if (c) c->err = msg; else g_create_error = msg;
    return code;
}

static int cuda_fail(adsc_ctx *c, cudaError_t e, const char *where)
{
    return fail(c, ADSC_ECUDA, std::string(where) + ": " + cudaGetErrorString(e));
}

#define ADSC_CUDA(call, where)                                         \
    do {                                                               \
        cudaError_t e__ = (call);                                      \
        if (e__ != cudaSuccess) return cuda_fail(h, e__, where);       \
    } while (0)

extern "C" {

adsc_handle adsc_create(int N, int batch, double courant, double ko_eps)
{
    if (N < 9 || (N - 1) % 2 != 0) { g_create_error = "N must be >= 9 and odd"; return nullptr; }
    if (batch < 1 || batch > 65535) { g_create_error = "batch must be in 1..65535 (grid.y of the pack/solve kernels)"; return nullptr; }
    if (!(courant > 0.0 && courant <= 1.0)) { g_create_error = "courant must be in (0,1]"; return nullptr; }
    if (!(ko_eps >= 0.0)) { g_create_error = "ko_eps must be >= 0"; return nullptr; }
    if ((double)N * (double)batch > 4.0e9) { g_create_error = "N*batch too large"; return nullptr; }
    adsc_ctx *c = new (std::nothrow) adsc_ctx();
    if (!c) { g_create_error = "host allocation failed"; return nullptr; }
    c->pb.N = N; c->pb.NP = (N + 3) / 4 * 4; c->pb.B = batch;   // (NP is final after resolve_path)
    c->pb.h = 1.5707963267948966192313216916398 / (double)(N - 1);
    c->courant = courant;
    c->pb.dt = courant * c->pb.h;
    c->pb.ko_eps = ko_eps;
    c->pb.thr = 0.0078125;   // 2^-7 (BASELINE.json configs[1])
    c->pb.fixed_bg = 0;
    c->rk_order = 4;
    c->spread = 0; c->spread_cap = 8;
    c->K_A = 0; c->path_opt = 0; c->steps_per_launch = 0;
    c->bound = false; c->have_state = false; c->stream = nullptr; c->ws_base = nullptr;
    c->launches = 0; c->global_step = 0; c->dev_sms = 0; c->dev_smem_optin = 0;
    c->cluster = 1; c->res_cfg = -1;
    c->sp_ok = false; c->sp_G = 0; c->sp_groups = 0; c->sp_SQ = 0;
    // The row pitch of the persistent streaming path depends on the SM count.  adsc_create touches no device state;
    // it only asks the runtime how many SMs the current device has, and assumes a B200 (148) if there is none to ask.
    c->sms_hint = 148;
    {
        int ndev = 0, dev = 0, sms = 0;
        if (cudaGetDeviceCount(&ndev) == cudaSuccess && ndev > 0 && cudaGetDevice(&dev) == cudaSuccess
            && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
            c->sms_hint = sms;
        else (void)cudaGetLastError();
    }
    resolve_path(c);
    return c;
}

int adsc_destroy(adsc_handle h)
{
    delete h;
    return ADSC_OK;
}

size_t adsc_workspace_bytes(adsc_handle h)
{
    if (!h) return 0;
    return h->lay.total;
}

int adsc_set_option(adsc_handle h, int key, double value)
{
    if (!h) return fail(nullptr, ADSC_EINVAL, "null handle");
    switch (key) {
    case ADSC_OPT_COLLAPSE_THRESHOLD:
        if (value != value) return fail(h, ADSC_EINVAL, "threshold is NaN");
        h->pb.thr = value;
        return ADSC_OK;
    case ADSC_OPT_A_RESOLVE_PERIOD:
        if (!(value >= 0.0) || value > 2.0e9 || value != std::floor(value))
            return fail(h, ADSC_EINVAL, "A re-solve period must be a non-negative integer");
        h->K_A = (int)value;
        return ADSC_OK;
    case ADSC_OPT_PATH: {
        if (!(value == 0.0 || value == 1.0 || value == 2.0 || value == 3.0)) return fail(h, ADSC_EINVAL, "path must be 0, 1, 2 or 3");
        if (h->bound) return fail(h, ADSC_ESTATE, "set ADSC_OPT_PATH before adsc_bind");
        const int old = h->path_opt;
        h->path_opt = (int)value;
        resolve_path(h);
        if (h->path == 0) {
            h->path_opt = old; resolve_path(h);
            return fail(h, ADSC_EINVAL, "the resident path cannot hold this N");
        }
        return ADSC_OK;
    }
    case ADSC_OPT_STEPS_PER_LAUNCH:
        if (!(value >= 0.0) || value != std::floor(value)) return fail(h, ADSC_EINVAL, "steps per launch must be a non-negative integer");
        h->steps_per_launch = (long long)value;
        return ADSC_OK;
    case ADSC_OPT_FIXED_BACKGROUND:
        if (!(value == 0.0 || value == 1.0)) return fail(h, ADSC_EINVAL, "fixed background: 0 or 1");
        if (h->bound) return fail(h, ADSC_ESTATE, "set ADSC_OPT_FIXED_BACKGROUND before adsc_bind");
        h->pb.fixed_bg = (int)value;
        resolve_path(h);                 // not every resident configuration has a fixed-background kernel
        if (h->path == 0) { h->path_opt = 0; resolve_path(h); }
        return ADSC_OK;
    case ADSC_OPT_RK_ORDER:
        if (!(value == 2.0 || value == 3.0 || value == 4.0)) return fail(h, ADSC_EINVAL, "Runge-Kutta order: 2, 3 or 4");
        if (h->bound) return fail(h, ADSC_ESTATE, "set ADSC_OPT_RK_ORDER before adsc_bind");
        h->rk_order = (int)value;
        resolve_path(h);                 // (the fixed-background build of the resident kernel is RK4 only)
        if (h->path == 0) { h->path_opt = 0; resolve_path(h); }
        return ADSC_OK;
    case ADSC_OPT_SPREAD:
        if (!(value == 0.0 || value == 1.0)) return fail(h, ADSC_EINVAL, "spread: 0 or 1");
        if (h->bound) return fail(h, ADSC_ESTATE, "set ADSC_OPT_SPREAD before adsc_bind");
        h->spread = (int)value;
        resolve_path(h);
        return ADSC_OK;
    default:
        return fail(h, ADSC_EINVAL, "unknown option key");
    }
}

int adsc_bind(adsc_handle h, void *d_workspace, size_t bytes, void *cuda_stream)
{
    if (!h) return fail(nullptr, ADSC_EINVAL, "null handle");
    if (!d_workspace) return fail(h, ADSC_EINVAL, "null workspace");
    if (((uintptr_t)d_workspace & 255u) != 0) return fail(h, ADSC_EINVAL, "workspace must be 256-byte aligned");
    if (bytes < h->lay.total) return fail(h, ADSC_ENOMEM, "workspace smaller than adsc_workspace_bytes");
    int dev = 0;
    ADSC_CUDA(cudaGetDevice(&dev), "cudaGetDevice");
    ADSC_CUDA(cudaDeviceGetAttribute(&h->dev_sms, cudaDevAttrMultiProcessorCount, dev), "device attribute");
    ADSC_CUDA(cudaDeviceGetAttribute(&h->dev_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev), "device attribute");
    int cc_major = 0;
    ADSC_CUDA(cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev), "device attribute");
    if (cc_major != 10) return fail(h, ADSC_ECUDA, "libadsc is built for sm_100a only; no fallback");
    h->stream = (cudaStream_t)cuda_stream;
    h->ws_base = d_workspace;
    char *base = (char *)d_workspace;
    const Layout &L = h->lay;
    for (int v = 0; v < 3; ++v) {
        h->ws.U[v] = (double *)(base + L.off_U[v]);
        h->ws.Ua[v] = (double *)(base + L.off_Ua[v]);
        h->ws.Ub[v] = (double *)(base + L.off_Ub[v]);
        h->ws.ACC[v] = (double *)(base + L.off_ACC[v]);
    }
    h->ws.dl = (double *)(base + L.off_dl);
    h->ws.Ac = (double *)(base + L.off_Ac);
    h->ws.tot = (double *)(base + L.off_tot);
    h->ws.carry = (double *)(base + L.off_carry);
    h->ws.tot2 = (double *)(base + L.off_tot2);
    h->ws.carry2 = (double *)(base + L.off_carry2);
    h->ws.part = (double *)(base + L.off_part);
    h->ws.stage[0] = (double *)(base + L.off_stage[0]);
    h->ws.stage[1] = (double *)(base + L.off_stage[1]);
    h->ws.tab = (double *)(base + L.off_tab);
    h->ws.rec = (MemberRec *)(base + L.off_rec);
    h->ws.sp_mbox = (double *)(base + L.off_mbox);
    h->ws.tabp = (double *)(base + L.off_tabp);
    // the persistent streaming kernel needs every CTA of a member co-resident on THIS device and the row pitch the
    // layout was made for; otherwise one kernel per phase (which takes any pitch)
    if (h->path == 1) {
        int G = 0, SQ = 0, groups = 0;
        if (!stream_async_select(h->pb.N, h->pb.B, h->dev_sms, &G, &SQ, &groups) || sa_row_pitch(h->pb.N, G, SQ) != h->pb.NP) {
            // The layout (and adsc_workspace_bytes) was made for the SM count seen at adsc_create.  Asked for by name,
            // the persistent kernel is not quietly replaced by the three-launches-per-stage kernels: say what to do.
            if (h->path_opt == 1)
                return fail(h, ADSC_ESTATE, "ADSC_OPT_PATH = 1 was chosen for a device with " + std::to_string(h->sms_hint)
                            + " SMs but adsc_bind runs on one with " + std::to_string(h->dev_sms)
                            + ": call adsc_create with the device that will be bound current (cudaSetDevice first)");
            h->path = 3; h->sp_ok = false;
        }
        else { h->sp_G = G; h->sp_SQ = SQ; h->sp_groups = groups; }
    }
    // the resident configuration was chosen at adsc_create without a device: make sure THIS device can hold one
    // cluster of it (shared-memory opt-in, cluster size)
    if (h->path == 2) {
        if (h->spread && h->spread_cap != 8) { h->spread_cap = 8; (void)resident_select(h); }   // (a re-bind: start over)
        int clusters = 0;
        const cudaError_t e = resident_check(h, &clusters);
        if (e != cudaSuccess || clusters < 1) {
            (void)cudaGetLastError();
            return fail(h, ADSC_ECUDA, std::string("the resident kernel (") + resident_cfg_name(h->res_cfg) + ", "
                        + std::to_string(h->cluster) + " CTAs per member) cannot run on this device"
                        + (e != cudaSuccess ? std::string(": ") + cudaGetErrorString(e) : std::string())
                        + "; set ADSC_OPT_PATH to 1 (streaming) before adsc_bind");
        }
        // ADSC_OPT_SPREAD promises that all clusters of the ensemble are co-resident.  B * cluster <= SMs (the test
        // resident_select applies without a device) does not guarantee it: a cluster must sit inside one GPC, so the
        // device may hold fewer.  Step back to the next wider segment until the occupancy query agrees (the widest one,
        // the default, ends the loop at the latest).  The layout does not depend on the segment.
        while (h->spread && clusters < h->pb.B) {
            const int before = h->cluster;
            h->spread_cap = before - 1;
            if (h->spread_cap < 1 || !resident_select(h) || h->cluster == before) break;
            const cudaError_t e2 = resident_check(h, &clusters);
            if (e2 != cudaSuccess || clusters < 1) {
                (void)cudaGetLastError();
                return fail(h, ADSC_ECUDA, std::string("the resident kernel (") + resident_cfg_name(h->res_cfg) + ") cannot run on this device");
            }
        }
    }
    const size_t NT = (size_t)h->pb.NP + 2 * HAL;
    h->tb.sc = h->ws.tab + 0 * NT + HAL;
    h->tb.T = h->ws.tab + 1 * NT + HAL;
    h->tb.C = h->ws.tab + 2 * NT + HAL;
    h->tb.c3s = h->ws.tab + 3 * NT + HAL;
    h->tb.w = h->ws.tab + 4 * NT + HAL;
    h->launches = 0;
    h->have_state = false;
    h->bound = true;
    ADSC_CUDA(launch_tables(h), "tables kernel");
    if (h->path == 1) ADSC_CUDA(launch_tabp(h), "permuted tables kernel");
    return ADSC_OK;
}

static int set_common(adsc_handle h, const double *d_Phi, const double *d_Pi, const double *d_A)
{
    ADSC_CUDA(launch_pack(h, d_Phi, 0, true), "pack Phi");
    ADSC_CUDA(launch_pack(h, d_Pi, 1, false), "pack Pi");
    if (d_A) ADSC_CUDA(launch_pack(h, d_A, 2, false), "pack A");
    else if (h->pb.fixed_bg) ADSC_CUDA(launch_fill(h, h->ws.U[2], 1.0), "A = 1");
    else ADSC_CUDA(launch_solve(h, SOLVE_WRITE_A), "constraint solve");
    h->have_state = true;
    h->global_step = 0;
    return ADSC_OK;
}

int adsc_set_initial(adsc_handle h, const double *d_Phi, const double *d_Pi)
{
    if (!h) return fail(nullptr, ADSC_EINVAL, "null handle");
    if (!h->bound) return fail(h, ADSC_ESTATE, "adsc_bind first");
    if (!d_Phi || !d_Pi) return fail(h, ADSC_EINVAL, "null field pointer");
    if (((uintptr_t)d_Phi & 7u) || ((uintptr_t)d_Pi & 7u)) return fail(h, ADSC_EINVAL, "field pointers must be 8-byte aligned");
    return set_common(h, d_Phi, d_Pi, nullptr);
}

int adsc_set_state(adsc_handle h, const double *d_Phi, const double *d_Pi, const double *d_A)
{
    if (!h) return fail(nullptr, ADSC_EINVAL, "null handle");
    if (!h->bound) return fail(h, ADSC_ESTATE, "adsc_bind first");
    if (!d_Phi || !d_Pi || !d_A) return fail(h, ADSC_EINVAL, "null field pointer");
    if (((uintptr_t)d_Phi & 7u) || ((uintptr_t)d_Pi & 7u) || ((uintptr_t)d_A & 7u))
        return fail(h, ADSC_EINVAL, "field pointers must be 8-byte aligned");
    return set_common(h, d_Phi, d_Pi, d_A);
}

int adsc_set_initial_host(adsc_handle h, const double *h_Phi, const double *h_Pi)
{
    if (!h) return fail(nullptr, ADSC_EINVAL, "null handle");
    if (!h->bound) return fail(h, ADSC_ESTATE, "adsc_bind first");
    if (!h_Phi || !h_Pi) return fail(h, ADSC_EINVAL, "null field pointer");
    const size_t n = (size_t)h->pb.B * h->pb.N * sizeof(double);
    ADSC_CUDA(cudaMemcpyAsync(h->ws.stage[0], h_Phi, n, cudaMemcpyHostToDevice, h->stream), "H2D Phi");
    ADSC_CUDA(cudaMemcpyAsync(h->ws.stage[1], h_Pi, n, cudaMemcpyHostToDevice, h->stream), "H2D Pi");
    return set_common(h, h->ws.stage[0], h->ws.stage[1], nullptr);
}

int adsc_step(adsc_handle h, long long nsteps)
{
    if (!h) return fail(nullptr, ADSC_EINVAL, "null handle");
    if (!h->bound || !h->have_state) return fail(h, ADSC_ESTATE, "adsc_bind and adsc_set_initial first");
    if (nsteps < 0) return fail(h, ADSC_EINVAL, "nsteps must be >= 0");
    const int K = h->pb.fixed_bg ? 0 : h->K_A;
    if (h->path == 2 || h->path == 1) {
        long long left = nsteps;
        while (left > 0) {
            long long n = left;
            if (K > 0) { const long long to_b = K - (h->global_step % K); if (n > to_b) n = to_b; }
            if (h->steps_per_launch > 0 && n > h->steps_per_launch) n = h->steps_per_launch;
            if (n > (1LL << 30)) n = 1LL << 30;              // (the kernels count the steps of a launch in 32 bits)
            const bool hit = K > 0 && ((h->global_step + n) % K == 0);
            if (h->path == 2) ADSC_CUDA(launch_resident(h, n, hit ? 0 : 1), "resident kernel");
            else ADSC_CUDA(launch_stream_async(h, n, hit ? 0 : 1), "persistent streaming kernel");
            if (hit) {
                ADSC_CUDA(launch_solve(h, SOLVE_WRITE_A | SOLVE_ACTIVE_ONLY), "A re-solve");
                ADSC_CUDA(launch_finalize(h, 0), "finalize");
            }
            h->global_step += n; left -= n;
        }
    } else {
        for (long long n = 0; n < nsteps; ++n) {
            ADSC_CUDA(launch_stream_step(h), "streaming step");
            h->global_step += 1;
            if (K > 0 && h->global_step % K == 0)
                ADSC_CUDA(launch_solve(h, SOLVE_WRITE_A | SOLVE_ACTIVE_ONLY), "A re-solve");
            ADSC_CUDA(launch_finalize(h, 1), "finalize");
        }
    }
    return ADSC_OK;
}

int adsc_diagnostics(adsc_handle h, adsc_diag *host_out)
{
    if (!h) return fail(nullptr, ADSC_EINVAL, "null handle");
    if (!h->bound || !h->have_state) return fail(h, ADSC_ESTATE, "adsc_bind and adsc_set_initial first");
    if (!host_out) return fail(h, ADSC_EINVAL, "null output");
    ADSC_CUDA(launch_solve(h, SOLVE_DIAG), "diagnostics kernel");
    std::vector<MemberRec> tmp;
    try { tmp.resize((size_t)h->pb.B); } catch (...) { return fail(h, ADSC_ENOMEM, "host allocation failed"); }
    ADSC_CUDA(cudaMemcpyAsync(tmp.data(), h->ws.rec, tmp.size() * sizeof(MemberRec), cudaMemcpyDeviceToHost, h->stream), "D2H records");
    ADSC_CUDA(cudaStreamSynchronize(h->stream), "stream synchronize");
    for (int b = 0; b < h->pb.B; ++b) {
        const MemberRec &r = tmp[b];
        adsc_diag &d = host_out[b];
        d.steps_done = r.steps_done;
        d.t = (double)r.steps_done * h->pb.dt;
        d.min_A = r.min_A; d.argmin_A = r.argmin_A; d.collapsed = r.collapsed;
        d.mass = r.mass; d.constraint_residual = r.resid; d.t_collapse = r.t_collapse;
    }
    return ADSC_OK;
}

int adsc_get_fields(adsc_handle h, double *d_Phi, double *d_Pi, double *d_A, double *d_delta)
{
    if (!h) return fail(nullptr, ADSC_EINVAL, "null handle");
    if (!h->bound || !h->have_state) return fail(h, ADSC_ESTATE, "adsc_bind and adsc_set_initial first");
    double *dst[3] = { d_Phi, d_Pi, d_A };
    for (int v = 0; v < 3; ++v) {
        if (!dst[v]) continue;
        if ((uintptr_t)dst[v] & 7u) return fail(h, ADSC_EINVAL, "field pointers must be 8-byte aligned");
        ADSC_CUDA(launch_unpack(h, h->ws.U[v], dst[v]), "unpack");
    }
    if (d_delta) {
        if ((uintptr_t)d_delta & 7u) return fail(h, ADSC_EINVAL, "field pointers must be 8-byte aligned");
        if (h->pb.fixed_bg) ADSC_CUDA(launch_fill(h, h->ws.dl, 0.0), "delta = 0");
        else ADSC_CUDA(launch_solve(h, 0), "delta solve");
        ADSC_CUDA(launch_unpack(h, h->ws.dl, d_delta), "unpack delta");
    }
    return ADSC_OK;
}

static int get_fields_host_impl(adsc_handle h, double *h_Phi, double *h_Pi, double *h_A, double *h_delta, bool sync)
{
    if (!h) return fail(nullptr, ADSC_EINVAL, "null handle");
    if (!h->bound || !h->have_state) return fail(h, ADSC_ESTATE, "adsc_bind and adsc_set_initial first");
    const size_t n = (size_t)h->pb.B * h->pb.N * sizeof(double);
    double *dst[4] = { h_Phi, h_Pi, h_A, h_delta };
    for (int v = 0; v < 4; ++v) {
        if (!dst[v]) continue;
        double *stage = h->ws.stage[v & 1];
        if (v < 3) ADSC_CUDA(launch_unpack(h, h->ws.U[v], stage), "unpack");
        else {
            if (h->pb.fixed_bg) ADSC_CUDA(launch_fill(h, h->ws.dl, 0.0), "delta = 0");
            else ADSC_CUDA(launch_solve(h, 0), "delta solve");
            ADSC_CUDA(launch_unpack(h, h->ws.dl, stage), "unpack delta");
        }
        ADSC_CUDA(cudaMemcpyAsync(dst[v], stage, n, cudaMemcpyDeviceToHost, h->stream), "D2H field");
    }
    if (sync) ADSC_CUDA(cudaStreamSynchronize(h->stream), "stream synchronize");
    return ADSC_OK;
}

int adsc_get_fields_host(adsc_handle h, double *h_Phi, double *h_Pi, double *h_A, double *h_delta)
{
    return get_fields_host_impl(h, h_Phi, h_Pi, h_A, h_delta, true);
}

int adsc_get_fields_host_async(adsc_handle h, double *h_Phi, double *h_Pi, double *h_A, double *h_delta)
{
    return get_fields_host_impl(h, h_Phi, h_Pi, h_A, h_delta, false);
}

int adsc_mode_energies(adsc_handle h, int J, double *host_out)
{
    if (!h) return fail(nullptr, ADSC_EINVAL, "null handle");
    if (!h->bound || !h->have_state) return fail(h, ADSC_ESTATE, "adsc_bind and adsc_set_initial first");
    if (!host_out) return fail(h, ADSC_EINVAL, "null output");
    if (J < 1 || J > 32 || 4 * J > h->pb.NP) return fail(h, ADSC_EINVAL, "J must be in 1..32 (and <= N/4)");
    double *d_out = h->ws.Ac;                    // scratch: [B][NP] doubles: [B][J] results, then the slice partials
    // One slice per member needs 2 B J doubles behind the B J results: 3 B J <= B NP follows from 4 J <= NP above, so
    // the partials always fit in the field (the check below guards the subtraction should that condition ever change).
    const size_t total = (size_t)h->pb.B * h->pb.NP, used = (size_t)h->pb.B * J;
    if (total < used + 2 * used) return fail(h, ADSC_EINVAL, "J too large for the scratch field of this N");
    ADSC_CUDA(launch_mode_energies(h, J, d_out, d_out + used, total - used), "mode projection kernels");
    ADSC_CUDA(cudaMemcpyAsync(host_out, d_out, (size_t)h->pb.B * J * sizeof(double), cudaMemcpyDeviceToHost, h->stream),
              "D2H mode energies");
    ADSC_CUDA(cudaStreamSynchronize(h->stream), "stream synchronize");
    return ADSC_OK;
}

long long adsc_launch_count(adsc_handle h) { return h ? h->launches : 0; }

int adsc_path(adsc_handle h, int *cluster)
{
    if (!h) return ADSC_EINVAL;
    if (cluster) *cluster = (h->path == 1 && h->sp_ok) ? h->sp_G : h->cluster;
    return h->path;
}

const char *adsc_last_error(adsc_handle h)
{
    return h ? h->err.c_str() : g_create_error.c_str();
}

}  // extern "C"
