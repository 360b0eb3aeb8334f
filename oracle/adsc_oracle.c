/*
 * adsc_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU implementation (fp64, long-double scan
 * accumulators) of the hot path of Liebling & Khanna, "Scalar collapse in AdS
 * with an OpenCL open source code" (arXiv:1706.07413): the method-of-lines RK4
 * step of the spherically symmetric Einstein-Klein-Gordon system in AdS4 in the
 * variables Phi, Pi, A, delta on x in [0, pi/2] (Sec. II).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load this file.  It shares no code, header, table or
 * constant generator with the CUDA path (paper_1706_07413_b200/csrc) and
 * neither includes the other.  Compile with -O2 -ffp-contract=off so that no
 * FMA contraction changes the arithmetic written here.
 *
 * The paper fixes the continuum system (eqs 1-12), "Runge-Kutta method of
 * lines ... fourth order accurate finite differences", the
 * evolve-A / integrate-delta split, the mass integral
 * and the collapse criterion.  Every discrete
 * choice it leaves open is a reading listed in DESIGN.md ("Readings R1-R22",
 * taken from SURVEY.md 8(c)); each function below names the reading it uses.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 pure AdS bit-exact,
 * P2 delta closed form a^2 cos^8 x/8, P3 small-amplitude closed form of 1-A,
 * P4 independent adaptive ODE solve of eqs (5),(6), P5 FD residual of eq (5),
 * P6 eigen-check of the flux-form operator on AdS4 modes e_j (omega_j=3+2j),
 * P7 linear periodicity at t=pi, 2pi, P8 self-convergence, P9 mass
 * conservation, P10 linear energy, P11 BC invariants, P12 collapse sanity.
 * No function here is "parity unpinned".
 *
 * Notation: N grid points, h=(pi/2)/(N-1), x_i=i*h, dt=courant*h.
 * Layout: every field is a contiguous row of N doubles; batches are [B][N].
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------ tables */

typedef struct {
    int N;
    double h;
    double *sc;   /* sin x_i cos x_i                (eqs 4,5,6)              */
    double *T;    /* tan^2 x_i, i<N-1; T[N-1]=0 is never used as a value     */
    double *C;    /* cot^2 x_i, 1<=i<=N-2; C[0]=C[N-1]=0 never used          */
    double *c3s;  /* cos^3 x_i / sin x_i, 1<=i<=N-2 (R11)                    */
    double *w;    /* composite Simpson weights (R15)                         */
} tables;

static const long double PI_2L = 1.57079632679489661923132169163975144L;

static int tables_init(tables *tb, int N)
{
    tb->N = N;
    tb->h = (double)(PI_2L / (long double)(N - 1));
    tb->sc = calloc(N, sizeof(double));
    tb->T = calloc(N, sizeof(double));
    tb->C = calloc(N, sizeof(double));
    tb->c3s = calloc(N, sizeof(double));
    tb->w = calloc(N, sizeof(double));
    if (!tb->sc || !tb->T || !tb->C || !tb->c3s || !tb->w) return -1;
    for (int i = 0; i < N; ++i) {
        long double x = PI_2L * (long double)i / (long double)(N - 1);
        long double s = sinl(x), c = cosl(x);
        if (i == N - 1) { c = 0.0L; s = 1.0L; }   /* c_{N-1} := 0 exactly */
        if (i == 0) { s = 0.0L; c = 1.0L; }
        tb->sc[i] = (double)(s * c);
        if (i < N - 1) tb->T[i] = (double)((s / c) * (s / c));
        if (i >= 1 && i <= N - 2) {
            tb->C[i] = (double)((c / s) * (c / s));
            tb->c3s[i] = (double)(c * c * c / s);
        }
        /* Simpson 1,4,2,...,4,1 times h/3; needs N-1 even */
        double m = (i == 0 || i == N - 1) ? 1.0 : ((i & 1) ? 4.0 : 2.0);
        tb->w[i] = m * tb->h / 3.0;
    }
    return 0;
}

static void tables_free(tables *tb)
{
    free(tb->sc); free(tb->T); free(tb->C); free(tb->c3s); free(tb->w);
}

/* ------------------------------------------------------- ghosts, operators */

/* Ghost rule (readings R2, R3): u_{-k} = p0 u_k, u_{N-1+k} = ppi u_{N-1-k}.
 * Parities (p0, ppi): Phi(-,+) Pi(+,-) G(-,+) H(+,-) F(-,+) f(-,-) p(+,+). */
static double gh(const double *u, int N, int j, int p0, int ppi)
{
    if (j < 0) return (double)p0 * u[-j];
    if (j > N - 1) return (double)ppi * u[2 * (N - 1) - j];
    return u[j];
}

/* D4 u_i = (u_{i-2} - 8u_{i-1} + 8u_{i+1} - u_{i+2})/(12h): the centred
 * fourth-order first derivative ("fourth order accurate finite differences",
 * PAPER.md:57). */
static double D4(const double *u, int N, double h, int i, int p0, int ppi)
{
    return (gh(u, N, i - 2, p0, ppi) - 8.0 * gh(u, N, i - 1, p0, ppi)
            + 8.0 * gh(u, N, i + 1, p0, ppi) - gh(u, N, i + 2, p0, ppi)) / (12.0 * h);
}

/* Kreiss-Oliger dissipation (reading R6; not in the paper, required by
 * BASELINE.json): Q u_i = (eps/(64h)) (u_{i-3} - 6u_{i-2} + 15u_{i-1} - 20u_i
 * + 15u_{i+1} - 6u_{i+2} + u_{i+3}). */
static double KO(const double *u, int N, double h, double eps, int i, int p0, int ppi)
{
    return (eps / (64.0 * h)) *
           (gh(u, N, i - 3, p0, ppi) - 6.0 * gh(u, N, i - 2, p0, ppi)
            + 15.0 * gh(u, N, i - 1, p0, ppi) - 20.0 * u[i]
            + 15.0 * gh(u, N, i + 1, p0, ppi) - 6.0 * gh(u, N, i + 2, p0, ppi)
            + gh(u, N, i + 3, p0, ppi));
}

/* Cumulative 4-point rule (reading R7): the integral of g over [x_i, x_{i+1}]
 * is (h/24)[13(g_i+g_{i+1}) - (g_{i-1}+g_{i+2})], i=0..N-2 (exact for cubics). */
static double cumrule(const double *g, int N, double h, int i, int p0, int ppi)
{
    return (h / 24.0) * (13.0 * (g[i] + g[i + 1])
                         - (gh(g, N, i - 1, p0, ppi) + gh(g, N, i + 2, p0, ppi)));
}

/* ------------------------------------------------------- constraint solves */

/* delta-solve, eq (6) PAPER.md:53 with the gauge eq (12) PAPER.md:75:
 * delta' = -sin x cos x (Phi^2+Pi^2), delta(pi/2)=0, so
 * delta_i = int_{x_i}^{pi/2} sc (Phi^2+Pi^2) dx = sum_{k>=i} I_k (readings R7, R8). */
static void delta_solve(const tables *tb, const double *Phi, const double *Pi,
                        double *delta, double *f /* scratch [N] */)
{
    const int N = tb->N;
    for (int i = 0; i < N; ++i)
        f[i] = tb->sc[i] * (Phi[i] * Phi[i] + Pi[i] * Pi[i]);
    long double acc = 0.0L;
    delta[N - 1] = 0.0;
    for (int i = N - 2; i >= 0; --i) {
        acc += (long double)cumrule(f, N, tb->h, i, -1, -1);
        delta[i] = (double)acc;
    }
}

/* A-solve, eq (5) PAPER.md:51 in integrated form (reading R11):
 * (A e^{-delta} sin x/cos^3 x)' = e^{-delta} (sin x/cos^3 x)'  =>
 * 1 - A = e^{delta} (cos^3 x/sin x) int_0^x tan^2 y (Phi^2+Pi^2) e^{-delta(y)} dy,
 * with A_0 = A_{N-1} = 1 (eqs 8, 11). */
static void A_solve(const tables *tb, const double *Phi, const double *Pi,
                    const double *delta, double *A, double *p /* scratch [N] */)
{
    const int N = tb->N;
    for (int i = 0; i < N - 1; ++i)
        p[i] = tb->T[i] * (Phi[i] * Phi[i] + Pi[i] * Pi[i]) * exp(-delta[i]);
    p[N - 1] = 0.0;
    long double P = 0.0L;            /* P_0 = 0 */
    A[0] = 1.0;
    for (int i = 1; i <= N - 2; ++i) {
        P += (long double)cumrule(p, N, tb->h, i - 1, +1, +1);   /* P_i = P_{i-1}+J_{i-1} */
        A[i] = 1.0 - exp(delta[i]) * tb->c3s[i] * (double)P;
    }
    A[N - 1] = 1.0;
}

/* ------------------------------------------------------------------- rhs */

/* Right-hand sides of eqs (2),(3),(4) PAPER.md:43-47, with delta integrated
 * from the stage's Phi, Pi (reading R9), eq (3) differenced in flux form as
 * printed (R1), l'Hopital at the origin (R4), the boundary flux limit (R5),
 * KO dissipation on Phi, Pi (R6), and the Dirichlet points of eqs (7)-(11)
 * held by zero rhs. */
typedef struct { double *delta, *f, *G, *H, *F; } rhs_ws;

/* fixed_bg != 0 is the paper's second workload (Table II: "both A and delta are not
 * dynamical i.e. held fixed at 1 and 0 respectively"): delta = 0 is not integrated, the A passed in
 * (A = 1 from set_initial) is used as it is and not evolved (kA = 0).  (SURVEY.md 8(f) f1.) */
static void rhs(const tables *tb, double ko_eps, int fixed_bg, const double *Phi, const double *Pi,
                const double *A, double *kPhi, double *kPi, double *kA, rhs_ws *ws)
{
    const int N = tb->N;
    const double h = tb->h;
    double *delta = ws->delta, *G = ws->G, *H = ws->H, *F = ws->F;
    if (fixed_bg) { for (int i = 0; i < N; ++i) delta[i] = 0.0; }
    else delta_solve(tb, Phi, Pi, delta, ws->f);
    for (int i = 0; i < N; ++i) {
        double E = exp(-delta[i]);
        double AE = A[i] * E;
        G[i] = AE * Phi[i];
        H[i] = AE * Pi[i];
    }
    for (int i = 0; i < N - 1; ++i) F[i] = tb->T[i] * G[i];
    F[N - 1] = (16.0 * G[N - 2] - G[N - 3]) / (12.0 * h * h);
    for (int i = 0; i < N; ++i) {
        kPhi[i] = D4(H, N, h, i, +1, -1) + KO(Phi, N, h, ko_eps, i, -1, +1);
        if (i == 0)
            kPi[i] = 3.0 * D4(G, N, h, 0, -1, +1) + KO(Pi, N, h, ko_eps, 0, +1, -1);
        else if (i <= N - 2)
            kPi[i] = tb->C[i] * D4(F, N, h, i, -1, +1) + KO(Pi, N, h, ko_eps, i, +1, -1);
        else
            kPi[i] = 0.0;
        kA[i] = fixed_bg ? 0.0 : -2.0 * tb->sc[i] * A[i] * G[i] * Pi[i];
    }
    kPhi[0] = 0.0; kPhi[N - 1] = 0.0; kPi[N - 1] = 0.0; kA[0] = 0.0; kA[N - 1] = 0.0;
}

/* ------------------------------------------------------------- integrator */

typedef struct {
    tables tb;
    double ko_eps, dt;
    int fixed_bg;      /* A = 1, delta = 0 held fixed */
    int rk_order;      /* 4 (classical RK4, R12), 3 (Heun's third-order rule) or 2 (explicit midpoint): R25 */
    rhs_ws ws;
    double *k[3];      /* current stage slope of (Phi, Pi, A)   */
    double *us[3];     /* stage state u*                         */
    double *acc[3];    /* running sum k1 + 2k2 + 2k3 + k4        */
    double *scratch;   /* [N] */
} stepper;

static int stepper_init(stepper *st, int N, double courant, double ko_eps)
{
    memset(st, 0, sizeof(*st));
    if (tables_init(&st->tb, N)) return -1;
    st->ko_eps = ko_eps;
    st->rk_order = 4;
    st->dt = courant * st->tb.h;
    double **all[] = { &st->ws.delta, &st->ws.f, &st->ws.G, &st->ws.H, &st->ws.F,
                       &st->k[0], &st->k[1], &st->k[2], &st->us[0], &st->us[1], &st->us[2],
                       &st->acc[0], &st->acc[1], &st->acc[2], &st->scratch };
    for (unsigned a = 0; a < sizeof(all) / sizeof(all[0]); ++a) {
        *all[a] = calloc(N, sizeof(double));
        if (!*all[a]) return -1;
    }
    return 0;
}

static void stepper_free(stepper *st)
{
    tables_free(&st->tb);
    free(st->ws.delta); free(st->ws.f); free(st->ws.G); free(st->ws.H); free(st->ws.F);
    for (int v = 0; v < 3; ++v) { free(st->k[v]); free(st->us[v]); free(st->acc[v]); }
    free(st->scratch);
}

/* One Runge-Kutta step of u=(Phi,Pi,A).  "second, third, and fourth order accurate Runge-Kutta"
 * (PAPER.md:57); the tableaux are not printed.  Reading R12: classical RK4, u2=u+dt/2 k1, u3=u+dt/2 k2,
 * u4=u+dt k3, u^{n+1} = u + dt/6 (k1+2k2+2k3+k4).  Reading R25: third order =
 * Heun's rule, u2=u+dt/3 k1, u3=u+2dt/3 k2, u^{n+1} = u + dt/4 (k1 + 3 k3); second order = explicit
 * midpoint, u2=u+dt/2 k1, u^{n+1} = u + dt k2.  In all three every stage state is u^n plus a multiple of
 * the PREVIOUS slope only, which is the form written out below. */
static void rk4_step(stepper *st, double *Phi, double *Pi, double *A)
{
    const int N = st->tb.N;
    const double dt = st->dt;
    double *u[3] = { Phi, Pi, A };
    static const double a4[4] = { 0.5, 0.5, 1.0, 0.0 }, b4[4] = { 1.0, 2.0, 2.0, 1.0 };     /* x dt/6 */
    static const double a3[3] = { 1.0 / 3.0, 2.0 / 3.0, 0.0 }, b3[3] = { 0.25, 0.0, 0.75 };
    static const double a2[2] = { 0.5, 0.0 }, b2[2] = { 0.0, 1.0 };
    const int ns = st->rk_order;
    const double *a_next = (ns == 4) ? a4 : (ns == 3) ? a3 : a2;
    const double *b_w = (ns == 4) ? b4 : (ns == 3) ? b3 : b2;
    const double fin = (ns == 4) ? dt / 6.0 : dt;      /* the RK4 arithmetic is unchanged: u + (dt/6)(k1+2k2+2k3+k4) */
    for (int v = 0; v < 3; ++v) {
        memcpy(st->us[v], u[v], N * sizeof(double));
        memset(st->acc[v], 0, N * sizeof(double));
    }
    for (int s = 0; s < ns; ++s) {
        rhs(&st->tb, st->ko_eps, st->fixed_bg, st->us[0], st->us[1], st->us[2],
            st->k[0], st->k[1], st->k[2], &st->ws);
        for (int v = 0; v < 3; ++v)
            for (int i = 0; i < N; ++i) {
                st->acc[v][i] += b_w[s] * st->k[v][i];
                if (s < ns - 1) st->us[v][i] = u[v][i] + a_next[s] * dt * st->k[v][i];
            }
    }
    for (int v = 0; v < 3; ++v)
        for (int i = 0; i < N; ++i)
            u[v][i] = u[v][i] + fin * st->acc[v][i];
}

/* min A and its first index; NaN-ignoring like fmin.  The collapse predicate
 * (reading R14) is evaluated separately so that NaN counts as collapsed. */
static void min_A(const double *A, int N, double *m, int *arg)
{
    double best = INFINITY; int bi = 0;
    for (int i = 0; i < N; ++i)
        if (A[i] < best) { best = A[i]; bi = i; }
    *m = best; *arg = bi;
}

static int any_below(const double *A, int N, double thr)
{
    for (int i = 0; i < N; ++i)
        if (!(A[i] >= thr)) return 1;
    return 0;
}

/* ============================================================ exported ABI */

/* Tables, for tests that want x_i-dependent closed forms on the same grid. */
int oracle_tables(int N, double *sc, double *T, double *C, double *w)
{
    tables tb;
    if (tables_init(&tb, N)) return -1;
    memcpy(sc, tb.sc, N * sizeof(double)); memcpy(T, tb.T, N * sizeof(double));
    memcpy(C, tb.C, N * sizeof(double)); memcpy(w, tb.w, N * sizeof(double));
    tables_free(&tb);
    return 0;
}

/* Operators on one row with explicit parities (p0, ppi in {-1,+1}). */
int oracle_D4(int N, const double *u, int p0, int ppi, double *out)
{
    double h = (double)(PI_2L / (long double)(N - 1));
    for (int i = 0; i < N; ++i) out[i] = D4(u, N, h, i, p0, ppi);
    return 0;
}

int oracle_KO(int N, double eps, const double *u, int p0, int ppi, double *out)
{
    double h = (double)(PI_2L / (long double)(N - 1));
    for (int i = 0; i < N; ++i) out[i] = KO(u, N, h, eps, i, p0, ppi);
    return 0;
}

int oracle_cumrule(int N, const double *g, int p0, int ppi, double *out /* [N-1] */)
{
    double h = (double)(PI_2L / (long double)(N - 1));
    for (int i = 0; i < N - 1; ++i) out[i] = cumrule(g, N, h, i, p0, ppi);
    return 0;
}

int oracle_delta_solve(int N, const double *Phi, const double *Pi, double *delta)
{
    tables tb; if (tables_init(&tb, N)) return -1;
    double *f = malloc(N * sizeof(double));
    delta_solve(&tb, Phi, Pi, delta, f);
    free(f); tables_free(&tb);
    return 0;
}

int oracle_A_solve(int N, const double *Phi, const double *Pi, const double *delta, double *A)
{
    tables tb; if (tables_init(&tb, N)) return -1;
    double *p = malloc(N * sizeof(double));
    A_solve(&tb, Phi, Pi, delta, A, p);
    free(p); tables_free(&tb);
    return 0;
}

/* rhs of one stage; also returns the stage's delta. */
int oracle_rhs(int N, double ko_eps, const double *Phi, const double *Pi, const double *A,
               double *kPhi, double *kPi, double *kA, double *delta)
{
    stepper st; if (stepper_init(&st, N, 0.25, ko_eps)) return -1;
    rhs(&st.tb, ko_eps, 0, Phi, Pi, A, kPhi, kPi, kA, &st.ws);
    memcpy(delta, st.ws.delta, N * sizeof(double));
    stepper_free(&st);
    return 0;
}

/* The same on the fixed background A = 1, delta = 0 of PAPER.md:177 (A is an input: pass ones). */
int oracle_rhs_fixed(int N, double ko_eps, const double *Phi, const double *Pi, const double *A,
               double *kPhi, double *kPi, double *kA, double *delta)
{
    stepper st; if (stepper_init(&st, N, 0.25, ko_eps)) return -1;
    rhs(&st.tb, ko_eps, 1, Phi, Pi, A, kPhi, kPi, kA, &st.ws);
    memcpy(delta, st.ws.delta, N * sizeof(double));
    stepper_free(&st);
    return 0;
}

/* set_initial ("define Phi(x,0) and Pi(x,0) and solve Eq. (5) for
 * A(x,0) and Eq. (6) for delta(x,0)"): force the Dirichlet values of eqs
 * (7),(9),(10), then delta-solve, then A-solve.  In place on Phi, Pi. */
int oracle_set_initial(int N, int B, double *Phi, double *Pi, double *A, double *delta)
{
    tables tb; if (tables_init(&tb, N)) return -1;
    double *scr = malloc(N * sizeof(double));
    for (int b = 0; b < B; ++b) {
        double *ph = Phi + (size_t)b * N, *pi = Pi + (size_t)b * N;
        ph[0] = 0.0; ph[N - 1] = 0.0; pi[N - 1] = 0.0;
        delta_solve(&tb, ph, pi, delta + (size_t)b * N, scr);
        A_solve(&tb, ph, pi, delta + (size_t)b * N, A + (size_t)b * N, scr);
    }
    free(scr); tables_free(&tb);
    return 0;
}

/* Diagnostics: mass M = int tan^2 x A (Phi^2+Pi^2) dx by
 * composite Simpson with the integrand := 0 at i=N-1 (R15); constraint
 * residual R = max_i |A_i - A^c_i| with A^c from A-solve (R16); min A. */
int oracle_diagnostics(int N, int B, const double *Phi, const double *Pi, const double *A,
                       double *mass, double *resid, double *minA, int *argminA)
{
    tables tb; if (tables_init(&tb, N)) return -1;
    double *delta = malloc(N * sizeof(double)), *Ac = malloc(N * sizeof(double));
    double *scr = malloc(N * sizeof(double));
    for (int b = 0; b < B; ++b) {
        const double *ph = Phi + (size_t)b * N, *pi = Pi + (size_t)b * N, *a = A + (size_t)b * N;
        long double M = 0.0L;
        for (int i = 0; i < N - 1; ++i)
            M += (long double)(tb.w[i] * (tb.T[i] * a[i] * (ph[i] * ph[i] + pi[i] * pi[i])));
        mass[b] = (double)M;
        delta_solve(&tb, ph, pi, delta, scr);
        A_solve(&tb, ph, pi, delta, Ac, scr);
        double r = 0.0;
        for (int i = 0; i < N; ++i) { double d = fabs(a[i] - Ac[i]); if (d > r || d != d) r = d; }
        resid[b] = r;
        min_A(a, N, &minA[b], &argminA[b]);
    }
    free(delta); free(Ac); free(scr); tables_free(&tb);
    return 0;
}

/* Evolve every member of a batch by nsteps RK4 steps of dt = courant*h.
 * After each full step: if K_A>0 and steps_done % K_A == 0 the member's A is
 * replaced by A-solve ("periodically integrating A", R10); then
 * the collapse test (R14): if !(min A >= thr) the member is
 * flagged, t_c = steps_done*dt, and it is frozen at that state.
 * steps_done / collapsed / t_collapse are in-out per-member arrays (a fresh
 * run passes zeros / zeros / NaN).  nthreads>1 runs members in parallel
 * (members are independent; the scans stay serial inside a member). */
static int evolve(int N, int B, double courant, double ko_eps, double thr, int K_A, int fixed_bg, int rk_order,
                  long long nsteps, double *Phi, double *Pi, double *A,
                  long long *steps_done, int *collapsed, double *t_collapse, int nthreads)
{
    int err = 0;
    if (nthreads < 1) nthreads = 1;
#ifdef _OPENMP
#pragma omp parallel num_threads(nthreads)
#endif
    {
        stepper st;
        int ok = (stepper_init(&st, N, courant, ko_eps) == 0);
        st.fixed_bg = fixed_bg; st.rk_order = rk_order;
        if (!ok) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
            err = -1;
        }
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 1)
#endif
        for (int b = 0; b < B; ++b) {
            if (!ok) continue;
            double *ph = Phi + (size_t)b * N, *pi = Pi + (size_t)b * N, *a = A + (size_t)b * N;
            for (long long n = 0; n < nsteps && !collapsed[b]; ++n) {
                rk4_step(&st, ph, pi, a);
                steps_done[b] += 1;
                if (!fixed_bg && K_A > 0 && steps_done[b] % K_A == 0) {
                    delta_solve(&st.tb, ph, pi, st.ws.delta, st.scratch);
                    A_solve(&st.tb, ph, pi, st.ws.delta, a, st.scratch);
                }
                if (any_below(a, N, thr)) {
                    collapsed[b] = 1;
                    t_collapse[b] = (double)steps_done[b] * st.dt;
                }
            }
        }
        if (ok) stepper_free(&st);
    }
    return err;
}

int oracle_evolve(int N, int B, double courant, double ko_eps, double thr, int K_A,
                  long long nsteps, double *Phi, double *Pi, double *A,
                  long long *steps_done, int *collapsed, double *t_collapse, int nthreads)
{
    return evolve(N, B, courant, ko_eps, thr, K_A, 0, 4, nsteps, Phi, Pi, A, steps_done, collapsed, t_collapse, nthreads);
}

/* Evolution on the fixed background A = 1, delta = 0 (Table II): A is passed
 * in (ones) and comes back unchanged, so the collapse test never fires. */
int oracle_evolve_fixed(int N, int B, double courant, double ko_eps,
                        long long nsteps, double *Phi, double *Pi, double *A,
                        long long *steps_done, int *collapsed, double *t_collapse, int nthreads)
{
    return evolve(N, B, courant, ko_eps, 0.0, 0, 1, 4, nsteps, Phi, Pi, A, steps_done, collapsed, t_collapse, nthreads);
}

/* ---------------------------------------------------- normal-mode projection (f3)
 * "At any given time, the current numerical solution can be decomposed into a
 * spectrum of normal modes".  AdS4 modes (R19): e_j = d_j cos^3 x
 * 2F1(-j, 3+j; 3/2; sin^2 x), d_j = sqrt(16(j+1)(j+2)/pi), omega_j = 3+2j,
 * orthonormal under tan^2 x dx; their derivatives are orthogonal with norm
 * omega_j^2.  2F1(-j,3+j;3/2;z) = j!/(3/2)_j P_j^{(1/2,3/2)}(1-2z), evaluated by
 * the three-term Jacobi recurrence in long double.  Reading R24: with
 * Pi_j = int Pi e_j tan^2 x dx and Phi_j = int Phi e_j' tan^2 x dx (composite
 * Simpson, integrand := 0 at i = N-1 as in R15) the mode energy is
 * E_j = Pi_j^2 + Phi_j^2 / omega_j^2, so that sum_j E_j -> M in the linear limit. */
static long double jacobi(int n, long double a, long double b, long double y)
{
    if (n < 0) return 0.0L;
    long double p0 = 1.0L;
    if (n == 0) return p0;
    long double p1 = (a + 1.0L) + (a + b + 2.0L) * (y - 1.0L) / 2.0L;
    for (int m = 2; m <= n; ++m) {
        long double c = 2.0L * m + a + b;
        long double a1 = 2.0L * m * (m + a + b) * (c - 2.0L);
        long double a2 = (c - 1.0L) * (c * (c - 2.0L) * y + a * a - b * b);
        long double a3 = 2.0L * (m + a - 1.0L) * (m + b - 1.0L) * c;
        long double p2 = (a2 * p1 - a3 * p0) / a1;
        p0 = p1; p1 = p2;
    }
    return p1;
}

static void eigenmode(int j, long double x, long double *e, long double *de)
{
    const long double pi = 2.0L * PI_2L;
    long double d = sqrtl(16.0L * (j + 1) * (j + 2) / pi);
    long double nrm = 1.0L;                      /* j! / (3/2)_j */
    for (int m = 1; m <= j; ++m) nrm *= (long double)m / ((long double)m + 0.5L);
    long double s = sinl(x), c = cosl(x), y = cosl(2.0L * x);
    long double P = jacobi(j, 0.5L, 1.5L, y);
    long double dP = 0.5L * (j + 3.0L) * jacobi(j - 1, 1.5L, 2.5L, y);      /* dP/dy */
    *e = d * nrm * c * c * c * P;
    *de = d * nrm * (-3.0L * c * c * s * P + c * c * c * dP * (-2.0L * sinl(2.0L * x)));
}

/* e_j and e_j' on the grid (for the pins). */
int oracle_eigenmode(int N, int j, double *e, double *de)
{
    for (int i = 0; i < N; ++i) {
        long double x = (i == N - 1) ? PI_2L : PI_2L * (long double)i / (long double)(N - 1);
        long double a, b;
        eigenmode(j, x, &a, &b);
        e[i] = (double)a; de[i] = (double)b;
    }
    return 0;
}

/* out[b][j] = E_j, proj[b][2j] = Pi_j, proj[b][2j+1] = Phi_j (proj may be NULL). */
int oracle_mode_energies(int N, int B, int J, const double *Phi, const double *Pi, double *out, double *proj)
{
    tables tb; if (tables_init(&tb, N)) return -1;
    for (int j = 0; j < J; ++j) {
        long double om = 3.0L + 2.0L * j;
        for (int b = 0; b < B; ++b) {
            const double *ph = Phi + (size_t)b * N, *pi = Pi + (size_t)b * N;
            long double sp = 0.0L, sf = 0.0L;
            for (int i = 0; i < N - 1; ++i) {
                long double x = PI_2L * (long double)i / (long double)(N - 1);
                long double e, de;
                eigenmode(j, x, &e, &de);
                long double wt = (long double)tb.w[i] * (long double)tb.T[i];
                sp += wt * (long double)pi[i] * e;
                sf += wt * (long double)ph[i] * de;
            }
            out[(size_t)b * J + j] = (double)(sp * sp + sf * sf / (om * om));
            if (proj) { proj[((size_t)b * J + j) * 2] = (double)sp; proj[((size_t)b * J + j) * 2 + 1] = (double)sf; }
        }
    }
    tables_free(&tb);
    return 0;
}

/* The same evolution with the second- or third-order Runge-Kutta rule of reading R25 (rk_order 2, 3; 4 = RK4). */
int oracle_evolve_rk(int N, int B, double courant, double ko_eps, double thr, int K_A, int rk_order,
                     long long nsteps, double *Phi, double *Pi, double *A,
                     long long *steps_done, int *collapsed, double *t_collapse, int nthreads)
{
    if (rk_order < 2 || rk_order > 4) return -1;
    return evolve(N, B, courant, ko_eps, thr, K_A, 0, rk_order, nsteps, Phi, Pi, A, steps_done, collapsed, t_collapse, nthreads);
}

/* Fixed background (Table II) with the second- or third-order rule: the paper's production runs use the
 * third-order option, so its Table II timings are fixed-background RK3 evolutions.  Same evolve(), same
 * rhs(): only the two switches are set together. */
int oracle_evolve_fixed_rk(int N, int B, double courant, double ko_eps, int rk_order,
                           long long nsteps, double *Phi, double *Pi, double *A,
                           long long *steps_done, int *collapsed, double *t_collapse, int nthreads)
{
    if (rk_order < 2 || rk_order > 4) return -1;
    return evolve(N, B, courant, ko_eps, 0.0, 0, 1, rk_order, nsteps, Phi, Pi, A, steps_done, collapsed, t_collapse, nthreads);
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
