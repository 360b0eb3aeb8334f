"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin names the passage of
PAPER.md (or the DESIGN.md reading) it checks; see SURVEY.md 8(c) P1-P12.
"""
import os

import numpy as np
import pytest

import oracle
from paper_1706_07413_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _golden(name):
    out = {}
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()
            out[k] = float(v)
    return out


# ----------------------------------------------------------------- operators

def test_D4_exact_on_quartics_and_parity_ghosts():
    # "fourth order accurate finite differences": the 5-point
    # centred first derivative is exact for polynomials up to degree 4.
    N = 65
    x = inputs.grid(N)
    for deg in range(5):
        d = oracle.D4(x ** deg, +1, +1)
        np.testing.assert_allclose(d[2:-2], deg * x[2:-2] ** max(deg - 1, 0) if deg else 0 * x[2:-2],
                                   rtol=0, atol=2e-12)
    # parity ghosts (R2, R3): sin(2x) is odd about 0 and about pi/2; cos(2x) is even about both;
    # with the right parities the derivative is 4th-order accurate up to the end points.
    e1 = np.abs(oracle.D4(np.sin(2 * x), -1, -1) - 2 * np.cos(2 * x)).max()
    e2 = np.abs(oracle.D4(np.cos(2 * x), +1, +1) + 2 * np.sin(2 * x)).max()
    x2 = inputs.grid(2 * N - 1)
    e1f = np.abs(oracle.D4(np.sin(2 * x2), -1, -1) - 2 * np.cos(2 * x2)).max()
    assert 14 < e1 / e1f < 18 and e2 < 1e-5
    # wrong parity must show up as an O(1/h) error at the ends
    bad = np.abs(oracle.D4(np.cos(2 * x), -1, -1) + 2 * np.sin(2 * x)).max()
    assert bad > 1.0


def test_KO_annihilates_quintics_and_damps_nyquist():
    # R6: Q is (eps/64h) times the 6th undivided difference: zero on degree<=5, and on the
    # Nyquist mode (-1)^i it gives -(eps/h) (-1)^i, i.e. dissipative sign.
    N = 33
    x = inputs.grid(N); h = x[1]
    for deg in range(6):
        q = oracle.KO(x ** deg, 0.1, +1, +1)
        assert np.abs(q[3:-3]).max() < 1e-9
    ny = (-1.0) ** np.arange(N)
    q = oracle.KO(ny, 0.1, +1, +1)   # even ghosts keep the alternation (N-1 even)
    np.testing.assert_allclose(q, -(0.1 / h) * ny, rtol=1e-12)


def test_cumrule_exact_for_cubics_and_sums_to_integral():
    # R7: (h/24)[13(g_i+g_{i+1}) - (g_{i-1}+g_{i+2})] integrates cubics exactly on [x_i,x_{i+1}].
    N = 33
    x = inputs.grid(N)
    for deg in range(4):
        I = oracle.cumrule(x ** deg, +1, +1)
        exact = (x[1:] ** (deg + 1) - x[:-1] ** (deg + 1)) / (deg + 1)
        np.testing.assert_allclose(I[1:-1], exact[1:-1], rtol=0, atol=1e-14)
    # with the right parity the sum over the grid is the integral to 4th order or better
    e = []
    for M in (33, 65, 129):
        xm = inputs.grid(M)
        e.append(abs(oracle.cumrule(np.sin(2 * xm), -1, -1).sum() - 1.0))
    assert 14 < e[0] / e[1] < 18 and 14 < e[1] / e[2] < 18, e


def test_tables_and_simpson_weights():
    N = 129
    tb = oracle.tables(N)
    x = inputs.grid(N)
    np.testing.assert_allclose(tb["sc"][:-1], np.sin(x[:-1]) * np.cos(x[:-1]), rtol=1e-14, atol=1e-17)
    assert tb["sc"][-1] == 0.0 and tb["sc"][0] == 0.0
    np.testing.assert_allclose(tb["T"][:-1], np.tan(x[:-1]) ** 2, rtol=1e-12)
    np.testing.assert_allclose(tb["C"][1:-1] * tb["T"][1:-1], 1.0, rtol=1e-14)
    assert abs(tb["w"].sum() - np.pi / 2) < 1e-14
    # Simpson is exact for cubics
    assert abs((tb["w"] * x ** 3).sum() - (np.pi / 2) ** 4 / 4) < 1e-13


# --------------------------------------------------------------- P1 pure AdS

@pytest.mark.parametrize("N", [17, 129])
def test_P1_pure_AdS_is_bit_exact(N):
    # north_star: "pure AdS (Phi=Pi=0) staying exactly A=1, delta=0".
    z = np.zeros((2, N))
    ev = oracle.Evolution(z, z, ko_eps=0.1)
    assert np.all(ev.A == 1.0) and np.all(ev.delta == 0.0)
    ev.step(1000)
    assert np.all(ev.A == 1.0) and np.all(ev.Phi == 0.0) and np.all(ev.Pi == 0.0)
    assert np.all(ev.delta == 0.0)
    d = ev.diagnostics()
    assert np.all(d["mass"] == 0.0) and np.all(d["resid"] == 0.0) and not d["collapsed"].any()


# ----------------------------------------------------- P2, P3 closed forms

def test_P2_delta_closed_form_fourth_order():
    # eq (6)+(12): Phi=0, Pi=a cos^3 x => delta = a^2 cos^8 x / 8.
    a = 0.7
    errs = []
    for N in (65, 129, 257, 513):
        x = inputs.grid(N)
        Pi = a * np.cos(x) ** 3; Pi[-1] = 0.0
        d = oracle.delta_solve(np.zeros(N), Pi)
        exact = a * a * np.cos(x) ** 8 / 8
        errs.append(np.abs(d - exact).max())
        assert d[-1] == 0.0 and np.all(d >= -1e-11)
    r = np.array(errs[:-1]) / np.array(errs[1:])
    assert np.all(r > 13) and np.all(r < 19), (errs, r)
    assert errs[-1] < 1e-10


def test_P3_A_small_amplitude_closed_form():
    # eq (5) linearised about A=1, delta=0 (R11):
    # (1-A)/a^2 -> (cos^3/sin) [x/16 + sin2x/64 - sin4x/64 - sin6x/192].
    a = 1e-4
    errs = []
    for N in (65, 129, 257):
        x = inputs.grid(N)
        Pi = a * np.cos(x) ** 3; Pi[-1] = 0.0
        s = oracle.set_initial(np.zeros(N), Pi)
        A = s["A"][0]
        xi = x[1:-1]
        cf = (np.cos(xi) ** 3 / np.sin(xi)) * (xi / 16 + np.sin(2 * xi) / 64 - np.sin(4 * xi) / 64
                                                - np.sin(6 * xi) / 192)
        errs.append(np.abs((1 - A[1:-1]) / a ** 2 - cf).max())
        assert A[0] == 1.0 and A[-1] == 1.0
    assert errs[1] < errs[0] / 10 and errs[2] < 2e-8, errs   # O(h^4) + O(a^2) + round-off/a^2
    # total mass of the linearised data: int sin^2 cos^4 = pi/32 (closed_forms.txt P3b)
    d = oracle.diagnostics(s["Phi"], s["Pi"], s["A"])
    assert abs(d["mass"][0] / a ** 2 - np.pi / 32) < 1e-7


# ------------------------------------------------ P4 independent ODE solve

def test_P4_constraints_against_adaptive_ode_solver():
    # "solve Eq. (5) for A(x,0) and Eq. (6) for delta(x,0)".  Integrate the two
    # ODEs exactly as printed with an adaptive 8th-order solver; the oracle's scans
    # (integrated form R11, cumulative rule R7) must agree to O(h^4).
    from scipy.integrate import solve_ivp

    a, b = 0.9, 0.6

    def Phi_f(x): return b * np.sin(x) * np.cos(x) ** 2 * np.sin(2 * x)   # odd at 0, ~rho^2... at pi/2
    def Pi_f(x): return a * np.cos(x) ** 3 * (1 + 0.5 * np.cos(2 * x))     # even at 0, ~rho^3 at pi/2
    def S(x): return Phi_f(x) ** 2 + Pi_f(x) ** 2

    errsA, errsd = [], []
    for N in (129, 257, 513):
        x = inputs.grid(N)
        Phi = Phi_f(x); Pi = Pi_f(x)
        Phi[0] = Phi[-1] = 0.0; Pi[-1] = 0.0
        s = oracle.set_initial(Phi, Pi)
        # delta: integrate eq (6) from pi/2 inward
        sol = solve_ivp(lambda t, y: [-np.sin(t) * np.cos(t) * S(t)], [np.pi / 2, 0.0], [0.0],
                        method="DOP853", rtol=1e-13, atol=1e-16, t_eval=x[::-1])
        d_ref = sol.y[0][::-1]
        errsd.append(np.abs(s["delta"][0] - d_ref).max())
        # A: integrate eq (5) outward from the regular series A = 1 - S(0) x^2/3 + O(x^4)
        x0 = x[1]
        # use a two-term-safe start: shoot from a much smaller x and let the solver reach x[1]
        xs = 1e-4
        te = x[1:-1]

        def f5(t, y):
            sn, cs = np.sin(t), np.cos(t)
            return [(1 + 2 * sn * sn) / (sn * cs) * (1 - y[0]) - sn * cs * y[0] * S(t)]

        sol = solve_ivp(f5, [xs, te[-1]], [1 - S(0.0) * xs * xs / 3], method="DOP853",
                        rtol=1e-13, atol=1e-16, t_eval=te)
        assert sol.success and x0 > xs
        errsA.append(np.abs(s["A"][0][1:-1] - sol.y[0]).max())
    rA = np.array(errsA[:-1]) / np.array(errsA[1:])
    rd = np.array(errsd[:-1]) / np.array(errsd[1:])
    assert np.all(rd > 12) and np.all(rA > 12), (errsA, errsd)
    assert errsA[-1] < 2e-9 and errsd[-1] < 2e-10


def test_P5_discrete_residual_of_eq5_converges():
    # eq (5) as printed, differenced with an independent numpy 4th-order stencil at fixed
    # interior x, on the oracle's A: residual -> 0 at 4th order.
    res = []
    for N in (129, 257, 513):
        Phi, Pi, _ = inputs.make("cfg1", N=N)
        Pi = Pi * 40.0                       # strong enough for a visible metric response
        s = oracle.set_initial(Phi, Pi)
        A, ph, pi = s["A"][0], s["Phi"][0], s["Pi"][0]
        x = inputs.grid(N); h = x[1]
        i = np.arange(N // 16, N - N // 16)
        dA = (A[i - 2] - 8 * A[i - 1] + 8 * A[i + 1] - A[i + 2]) / (12 * h)
        sn, cs = np.sin(x[i]), np.cos(x[i])
        r = dA - ((1 + 2 * sn ** 2) / (sn * cs) * (1 - A[i]) - sn * cs * A[i] * (ph[i] ** 2 + pi[i] ** 2))
        res.append(np.abs(r).max())
    assert res[0] / res[1] > 10 and res[1] / res[2] > 10, res


# -------------------------------------------- P6, P7 eigenmodes, omega = 3+2j

@pytest.mark.parametrize("j", [0, 1, 2, 3])
def test_P6_flux_operator_has_AdS_eigenmodes(j):
    # eqs (2),(3) linearised: Phi=eps e_j', Pi=0 => Pi_dot = -omega_j^2 eps e_j,
    # and Pi = eps e_j, Phi=0 => Phi_dot = eps e_j'.  omega_j = 3+2j (north_star; closed_forms.txt).
    om = _golden("closed_forms.txt")[f"omega_{j}"]
    eps = 1e-7
    e_or, e_end = [], []
    for N in (129, 257, 513):
        x = inputs.grid(N)
        e, de = inputs.eigenmode(j, x)
        de[0] = de[-1] = 0.0
        e[-1] = 0.0
        kP, kQ, kA, d = oracle.rhs(eps * de, np.zeros(N), np.ones(N), 0.0)
        err = np.abs(kQ / eps + om ** 2 * e)
        e_or.append(err[0]); e_end.append(err[N // 4:].max())
        kP, kQ, kA, d = oracle.rhs(np.zeros(N), eps * e, np.ones(N), 0.0)
        assert np.abs(kP / eps - de).max() < 3e-3 * (129.0 / N) ** 4 * (1 + j) ** 5
    # origin (l'Hopital, R4) and away from it: 4th order
    assert 12 < e_or[0] / e_or[1] < 20 and 12 < e_or[1] / e_or[2] < 20, e_or
    assert e_end[0] / e_end[1] > 12 and e_end[1] / e_end[2] > 12, e_end


def test_P6_orthonormality_of_input_modes():
    # R19: int e_j e_k tan^2 = delta_jk, checked with Simpson on a fine grid (input generator pin).
    N = 2049
    x = inputs.grid(N); tb = oracle.tables(N)
    es = [inputs.eigenmode(j, x)[0] for j in range(4)]
    for j in range(4):
        for k in range(4):
            v = (tb["w"][:-1] * tb["T"][:-1] * es[j][:-1] * es[k][:-1]).sum()
            assert abs(v - (1.0 if j == k else 0.0)) < 1e-9


@pytest.mark.parametrize("j,N", [(0, 129), (1, 129), (1, 257), (2, 257)])
def test_P7_linear_periodicity_and_frequency(j, N):
    # A single small-amplitude mode oscillates at omega_j = 3+2j (north_star): with Phi=eps e_j',
    # Pi=0, phi = eps e_j cos(omega t): Phi(pi) = -Phi(0) (omega odd), Phi(2pi)=Phi(0), and the
    # projection Pi_j(t) = int Pi e_j tan^2 = -eps omega sin(omega t) has 2*omega-1 zero
    # crossings inside (0, 2pi) and amplitude eps*omega.
    om = 3 + 2 * j
    eps = 1e-5
    x = inputs.grid(N); tb = oracle.tables(N)
    e, de = inputs.eigenmode(j, x)
    Phi0 = eps * de; Phi0[0] = Phi0[-1] = 0.0
    ev = oracle.Evolution(Phi0, np.zeros(N), courant=0.25, ko_eps=0.1)
    steps_pi = 8 * (N - 1)                     # t = pi exactly: dt = h/4 = pi/(8(N-1))
    chunk = (N - 1) // 16
    proj = []
    for k in range(2 * steps_pi // chunk):
        ev.step(chunk)
        proj.append((tb["w"][:-1] * tb["T"][:-1] * ev.Pi[0][:-1] * e[:-1]).sum())
        if (k + 1) * chunk == steps_pi:
            flip = np.abs(ev.Phi[0] + Phi0).max() / np.abs(Phi0).max()
    back = np.abs(ev.Phi[0] - Phi0).max() / np.abs(Phi0).max()
    tol = 4e-5 * (129.0 / N) ** 3 * (om / 5.0) ** 4 + 3e-6
    print('P7', j, N, flip, back, tol)
    assert flip < tol and back < 2 * tol, (flip, back, tol)
    proj = np.array(proj)
    crossings = np.count_nonzero(np.sign(proj[:-2]) * np.sign(proj[1:-1]) < 0)
    assert crossings == 2 * om - 1, crossings
    assert abs(np.abs(proj).max() / (eps * om) - 1.0) < 5e-3
    # BC invariants (P11) along the way
    assert ev.Phi[0][0] == 0 and ev.Phi[0][-1] == 0 and ev.Pi[0][-1] == 0
    assert ev.A[0][0] == 1 and ev.A[0][-1] == 1 and ev.delta[0][-1] == 0


# --------------------------------- P8 self-convergence, P9 mass, constraint R

def test_P8_P9_self_convergence_mass_and_residual():
    # "solutions converge to a unique solution as the resolution is increased";
    # mass conserved; constraint residual monitored.  Same physical time on 4 levels.
    levels = (129, 257, 513, 1025)
    t_steps0 = 256                            # steps on the coarsest level: t = 256*0.25*h0 = pi/4... (0.785)
    sols, dM, R = [], [], []
    for lv, N in enumerate(levels):
        Pi = inputs.gaussian_Pi(N, 2.0, 0.25)
        ev = oracle.Evolution(np.zeros((1, N)), Pi)
        M0 = ev.diagnostics()["mass"][0]
        ev.step(t_steps0 * 2 ** lv)
        d = ev.diagnostics()
        dM.append(abs(d["mass"][0] - M0) / M0); R.append(d["resid"][0])
        st = 2 ** lv
        sols.append([ev.Phi[0][::st], ev.Pi[0][::st], ev.A[0][::st], ev.delta[0][::st]])
        assert ev.Phi[0][0] == 0 and ev.Phi[0][-1] == 0 and ev.Pi[0][-1] == 0      # P11
        assert ev.A[0][0] == 1 and ev.A[0][-1] == 1
    h0 = (np.pi / 2) / 128
    for f, name in enumerate(["Phi", "Pi", "A", "delta"]):
        d = [np.sqrt(h0 * ((sols[l][f] - sols[l + 1][f]) ** 2).sum()) for l in range(3)]
        order1, order2 = np.log2(d[0] / d[1]), np.log2(d[1] / d[2])
        assert order2 > 3.5 and order1 > 3.0, (name, d, order1, order2)
    # Hamiltonian-constraint residual (A evolved by eq 4 vs A from eq 5): 4th order
    assert R[1] / R[2] > 12 and R[2] / R[3] > 12, R
    # mass drift -> 0 at least as fast as h^4, and far below the paper's 1%
    assert dM[3] < 1e-9 and dM[1] / dM[2] > 12, dM


def test_P10_linear_energy_of_two_mode_data():
    # R20 + PAPER.md:83: for small amplitude M0 -> sum omega_j^2 a_j^2.
    N = 1025
    a_tot, ratio, th = 1e-3, 0.5, 1.1
    Phi, Pi = inputs.two_mode(N, a_tot, ratio, th)
    q = (3.0 / 5.0) * np.sqrt(ratio)
    a0 = a_tot / np.sqrt(1 + q * q); a1 = q * a0
    ev = oracle.Evolution(Phi, Pi)
    M0 = ev.diagnostics()["mass"][0]
    expect = 9 * a0 ** 2 * 1.0 + 25 * a1 ** 2      # cos^2+sin^2 of theta_1 sums to 1 for mode 1
    assert abs(M0 / expect - 1) < 1e-5, (M0, expect)


# --------------------------------------------------- survey probe cross-checks

def test_survey_probe_reference_values():
    g = _golden("survey_probe_values.txt")
    Phi, Pi, _ = inputs.make("cfg1")
    ev = oracle.Evolution(Phi, Pi)
    d = ev.diagnostics()
    assert abs(d["mass"][0] / g["M0_sigma1/16_N1025_eps1"] - 1) < 1e-11
    assert abs(d["min_A"][0] - g["minA0_sigma1/16_N1025_eps1"]) < 1e-8
    assert abs(ev.delta[0][0] / g["delta0_at_0_sigma1/16_N1025_eps1"] - 1) < 1e-6
    Pi = inputs.gaussian_Pi(2049, 1.0, 0.25)
    ev = oracle.Evolution(np.zeros_like(Pi), Pi)
    assert abs(ev.diagnostics()["mass"][0] / g["M0_sigma1/4_N2049_eps1"] - 1) < 1e-11


def test_P12_collapse_sanity_against_survey_probe():
    # collapse signalled by min A -> small; thr = 2^-7 (BASELINE.json configs[1]).
    g = _golden("survey_probe_values.txt")
    N = 1025
    Pi = inputs.gaussian_Pi(N, [45.0, 60.0, 20.0, 30.0], 1.0 / 16)
    ev = oracle.Evolution(np.zeros_like(Pi), Pi, thr=2.0 ** -7, nthreads=4)
    ev.step(10431)                                   # t = 4
    d = ev.diagnostics()
    assert list(d["collapsed"]) == [1, 1, 0, 0]
    assert d["steps_done"][0] == g["collapse_step_eps45"] and d["argmin_A"][0] == g["collapse_argmin_eps45"]
    assert d["steps_done"][1] == g["collapse_step_eps60"] and d["argmin_A"][1] == g["collapse_argmin_eps60"]
    np.testing.assert_allclose(d["t_collapse"][:2], d["steps_done"][:2] * ev.dt, rtol=1e-15)
    assert np.isnan(d["t_collapse"][2:]).all() and (d["steps_done"][2:] == 10431).all()
    assert abs(d["min_A"][2] - g["minA_t4_eps20"]) < 2e-4 and abs(d["min_A"][3] - g["minA_t4_eps30"]) < 2e-4
    # frozen members do not move when stepped again
    A_before = ev.A[:2].copy()
    ev.step(5)
    assert np.array_equal(ev.A[:2], A_before) and (ev.steps_done[2:] == 10436).all()


def test_A_resolve_period_keeps_constraint_tight():
    # PAPER.md:81 "periodically integrating A(x,t) over space helps improve stability and
    # accuracy" (R10): with K_A>0 the residual right after a re-solve is round-off.
    N = 257
    Pi = inputs.gaussian_Pi(N, 10.0, 1.0 / 8)
    free = oracle.Evolution(np.zeros_like(Pi), Pi, K_A=0).step(512).diagnostics()
    tight = oracle.Evolution(np.zeros_like(Pi), Pi, K_A=16).step(512).diagnostics()
    assert tight["resid"][0] < 1e-13 and free["resid"][0] > 1e-9
    assert abs(tight["mass"][0] / free["mass"][0] - 1) < 1e-5


# ------------------------------------------------- f1: fixed background A = 1, delta = 0

@pytest.mark.parametrize("j", [0, 2])
def test_F1_fixed_background_rhs_is_the_linear_operator(j):
    # With A = 1, delta = 0 held fixed (Table II) eqs (2), (3) are exactly linear:
    # Phi_dot = Pi', Pi_dot = tan^-2 (tan^2 Phi)'.  At FINITE amplitude the AdS4 eigenmodes must come out
    # (omega_j = 3+2j, closed_forms.txt) with no O(eps^2) remainder, and superposition must hold to rounding.
    om = _golden("closed_forms.txt")[f"omega_{j}"]
    errs = []
    for N in (129, 257, 513):
        x = inputs.grid(N)
        e, de = inputs.eigenmode(j, x)
        de[0] = de[-1] = 0.0; e[-1] = 0.0
        kP, kQ, kA, d = oracle.rhs_fixed(de, np.zeros(N), 0.0)
        assert (kA == 0).all() and (d == 0).all()
        errs.append(np.abs(kQ + om ** 2 * e)[N // 4:].max())
        kP, kQ, kA, d = oracle.rhs_fixed(np.zeros(N), e, 0.0)
        assert np.abs(kP - de).max() < 3e-3 * (129.0 / N) ** 4 * (1 + j) ** 5
    assert errs[0] / errs[1] > 12 and errs[1] / errs[2] > 12, errs
    N = 257
    x = inputs.grid(N)
    rng = np.random.default_rng(5)
    u1, u2 = (np.sin(2 * x) * np.cos(x) ** 2 * rng.uniform(0.5, 2.0) for _ in range(2))
    v1, v2 = (np.cos(x) ** 3 * rng.uniform(0.5, 2.0) * np.cos(3 * x) for _ in range(2))
    for u in (u1, u2): u[0] = u[-1] = 0.0
    for v in (v1, v2): v[-1] = 0.0
    r1 = oracle.rhs_fixed(u1, v1, 0.1); r2 = oracle.rhs_fixed(u2, v2, 0.1)
    r12 = oracle.rhs_fixed(2.5 * u1 - 0.75 * u2, 2.5 * v1 - 0.75 * v2, 0.1)
    for k in (0, 1):
        lin = 2.5 * r1[k] - 0.75 * r2[k]
        assert np.abs(r12[k] - lin).max() <= 1e-12 * max(1.0, np.abs(lin).max())


def test_F2_fixed_background_evolution_periodic_linear_and_conservative():
    # Finite-amplitude single mode on the fixed background: exact periodicity of the continuum solution
    # (all omega_j odd: Phi(pi) = -Phi(0)), exact amplitude independence (linearity of every step),
    # A = 1 and delta = 0 untouched, no collapse, and the linear energy int tan^2 (Phi^2+Pi^2) conserved.
    j, N = 1, 257
    x = inputs.grid(N); tb = oracle.tables(N)
    e, de = inputs.eigenmode(j, x)
    Phi0 = de.copy(); Phi0[0] = Phi0[-1] = 0.0
    steps_pi = 8 * (N - 1)
    big = oracle.Evolution(Phi0, np.zeros(N), fixed_background=True)
    small = oracle.Evolution(1e-3 * Phi0, np.zeros(N), fixed_background=True)
    E0 = (tb["w"][:-1] * tb["T"][:-1] * (big.Phi[0][:-1] ** 2 + big.Pi[0][:-1] ** 2)).sum()
    big.step(steps_pi); small.step(steps_pi)
    flip = np.abs(big.Phi[0] + Phi0).max() / np.abs(Phi0).max()
    assert flip < 4e-5 * (129.0 / N) ** 3 * (5 / 5.0) ** 4 + 3e-6, flip
    assert np.abs(big.Phi[0] * 1e-3 - small.Phi[0]).max() <= 1e-12 * 1e-3 * np.abs(Phi0).max()
    assert np.abs(big.Pi[0] * 1e-3 - small.Pi[0]).max() <= 1e-12 * 1e-3 * 5.0 * np.abs(e).max()   # |Pi| <= omega |e|
    assert (big.A == 1).all() and (big.delta == 0).all() and not big.collapsed.any()
    E1 = (tb["w"][:-1] * tb["T"][:-1] * (big.Phi[0][:-1] ** 2 + big.Pi[0][:-1] ** 2)).sum()
    assert abs(E1 / E0 - 1.0) < 1e-6, (E0, E1)
    assert abs(E0 - 25.0) < 1e-3          # omega_1^2 a^2 = 25 for a = 1 (R19 normalisation, P10)


def test_F3_dynamical_evolution_tends_to_fixed_background_as_amplitude_vanishes():
    # The back-reaction is O(eps^2) (delta, 1-A ~ eps^2): (Phi_dyn - Phi_fixed)/eps = O(eps^2).
    N = 129
    x = inputs.grid(N)
    e, de = inputs.eigenmode(0, x)
    Phi0 = de.copy(); Phi0[0] = Phi0[-1] = 0.0
    d = []
    for eps in (1e-2, 1e-3):
        dyn = oracle.Evolution(eps * Phi0, np.zeros(N)).step(400)
        fix = oracle.Evolution(eps * Phi0, np.zeros(N), fixed_background=True).step(400)
        d.append(np.abs(dyn.Phi[0] - fix.Phi[0]).max() / eps)
    assert d[0] < 1e-2 and 50 < d[0] / d[1] < 200, d


# ------------------------------------------------- f4: the paper's data families (input generator pins)

def test_F4_qp_family_generator_has_the_prescribed_spectrum():
    # PAPER.md:93-101 eq (13): A_k = eps exp(-mu |k - k_d|), Phi(x,0) = 0; reading R23:
    # Pi(x,0) = sum_k A_k omega_k e_k.  Orthonormality of the e_k under tan^2 x dx (R19) must give the
    # spectrum back; the Jacobi form of e_j must agree with the terminating series where that one is accurate.
    N = 2049
    x = inputs.grid(N); tb = oracle.tables(N)
    for j in range(6):
        e, _ = inputs.eigenmode(j, x)
        assert np.abs(inputs.eigenmode_jacobi(j, x) - e).max() < 5e-13
    eps = np.array([0.01, 0.04])
    Phi, Pi, Ak = inputs.qp_family(N, eps, 1.75, 5)
    assert (Phi == 0).all() and (Pi[:, -1] == 0).all() and Ak.shape[0] == 2
    assert np.allclose(Ak[1] / Ak[0], 4.0) and np.argmax(Ak[0]) == 5 and abs(Ak[0][5] - 0.01) < 1e-18
    assert abs(Ak[0][7] / Ak[0][5] - np.exp(-3.5)) < 1e-15
    for k in range(12):
        proj = (tb["w"][:-1] * tb["T"][:-1] * Pi[0][:-1] * inputs.eigenmode_jacobi(k, x)[:-1]).sum()
        assert abs(proj / inputs.omega(k) - Ak[0][k]) < 1e-12 * Ak[0][5], k


# ------------------------------------------------- f3: normal-mode projection

def test_F5_mode_projection_orthonormality_parseval_and_spectrum():
    # (i) the oracle's Jacobi-recurrence modes agree with the terminating hypergeometric series of the input
    #     generator where that one is accurate (independent routes to the same e_j, e_j');
    # (ii) Pi = e_k gives E_j = delta_jk, Phi = e_k' gives E_j = omega_k^2 delta_jk (R19; Simpson, 4th order);
    # (iii) Parseval in the linear limit: two-mode data, sum_j E_j = M(A = 1) (R15, R24);
    # (iv) the family of eq (13): sqrt(E_k)/omega_k = A_k.
    N, J = 1025, 8
    x = inputs.grid(N); tb = oracle.tables(N)
    for j in (0, 2, 5):
        e, de = inputs.eigenmode(j, x)
        eo, deo = oracle.eigenmode(N, j)
        assert np.abs(e - eo).max() < 1e-12 and np.abs(de - deo).max() < 1e-11
    for k in (0, 3):
        e, de = oracle.eigenmode(N, k)
        E, _ = oracle.mode_energies(np.zeros(N), e, J)
        ref = np.zeros(J); ref[k] = 1.0
        assert np.abs(E[0] - ref).max() < 1e-8, E
        E, _ = oracle.mode_energies(de, np.zeros(N), J)
        ref[k] = (3.0 + 2 * k) ** 2
        assert np.abs(E[0] - ref).max() < 1e-6, E
    Phi, Pi = inputs.two_mode(N, [0.05], [0.6], [1.1])
    E, proj = oracle.mode_energies(Phi, Pi, J)
    M = (tb["w"][:-1] * tb["T"][:-1] * (Phi[0][:-1] ** 2 + Pi[0][:-1] ** 2)).sum()
    assert abs(E[0].sum() / M - 1.0) < 1e-8 and E[0][2:].max() < 1e-12 * M
    assert abs(E[0][1] / E[0][0] - 0.6) < 1e-8                  # the energy ratio of R20
    Phi, Pi, Ak = inputs.qp_family(N, [0.02], 1.0, 3)
    E, _ = oracle.mode_energies(Phi, Pi, J)
    om = 3.0 + 2.0 * np.arange(J)
    assert np.abs(np.sqrt(E[0]) / om - Ak[0][:J]).max() < 1e-9 * Ak[0][3]


# ------------------------------------------------- f2: second- and third-order Runge-Kutta

def test_F6_rk_orders_of_accuracy():
    # "second, third, and fourth order accurate Runge-Kutta"; reading R25: Heun's third-order
    # rule and the explicit midpoint rule.  At FIXED grid the error against a reference with a much smaller
    # time step is the time-discretisation error: halving dt must divide it by 2^order.
    N, T = 129, 0.6
    x = inputs.grid(N)
    e1, de1 = inputs.eigenmode(1, x)
    Phi0 = 0.3 * de1; Phi0[0] = Phi0[-1] = 0.0
    Pi0 = inputs.gaussian_Pi(N, 1.0, 0.25)[0]
    h = (np.pi / 2) / (N - 1)
    def run(order, lam):
        n = int(round(T / (lam * h)))
        ev = oracle.Evolution(Phi0, Pi0, courant=T / (n * h), ko_eps=0.0, rk_order=order).step(n)
        return np.concatenate([ev.Phi[0], ev.Pi[0], ev.A[0]])
    ref = run(4, 0.0125)
    for order, lo, hi in ((2, 3.5, 4.6), (3, 7.0, 9.2), (4, 14.0, 18.5)):
        errs = [np.abs(run(order, lam) - ref).max() for lam in (0.4, 0.2, 0.1)]
        r1, r2 = errs[0] / errs[1], errs[1] / errs[2]
        assert lo < r1 < hi and lo < r2 < hi, (order, errs, r1, r2)
    # the three rules are genuinely different programs: at the same dt their results differ by far more than rounding
    assert np.abs(run(3, 0.2) - run(4, 0.2)).max() > 1e-8


def test_F7_fixed_background_rk2_rk3_orders_linearity_and_dissipation_sign():
    # PAPER.md:57 ("the results presented here use the third-order accurate option") with PAPER.md:177 (Table II:
    # A = 1, delta = 0 held fixed): the fixed-background evolution under the second- and third-order rules.
    # (1) order of accuracy at fixed grid, as F6; (2) every step is linear, so scaling the data by a power of two
    # scales the result bit for bit; (3) A = 1, delta = 0 untouched and nothing collapses; (4) the rules differ from
    # RK4 and from each other by far more than rounding; (5) the amplification of an exact eigenmode of the
    # semi-discrete operator over one period is the rule's stability polynomial: for Heun-3 |R(i w dt)| < 1 while for
    # the midpoint rule |R| > 1, so the linear energy falls under RK3 and grows under RK2 (ko_eps = 0).
    N, T = 129, 0.6
    x = inputs.grid(N); tb = oracle.tables(N)
    e1, de1 = inputs.eigenmode(1, x)
    Phi0 = 0.3 * de1; Phi0[0] = Phi0[-1] = 0.0
    Pi0 = inputs.gaussian_Pi(N, 1.0, 0.25)[0]
    h = (np.pi / 2) / (N - 1)
    def run(order, lam, scale=1.0):
        n = int(round(T / (lam * h)))
        ev = oracle.Evolution(scale * Phi0, scale * Pi0, courant=T / (n * h), ko_eps=0.0, rk_order=order,
                              fixed_background=True).step(n)
        assert (ev.A == 1).all() and (ev.delta == 0).all() and not ev.collapsed.any()
        return np.concatenate([ev.Phi[0], ev.Pi[0]])
    ref = run(4, 0.00625)
    # (the linear problem reaches the asymptotic ratio of the third-order rule later than F6's nonlinear one: its
    # dt^4 term has the opposite sign, so the ratios rise towards 8 from below)
    for order, lams, lo, hi in ((2, (0.4, 0.2, 0.1), 3.5, 4.6), (3, (0.1, 0.05, 0.025), 6.8, 8.4)):
        errs = [np.abs(run(order, lam) - ref).max() for lam in lams]
        r1, r2 = errs[0] / errs[1], errs[1] / errs[2]
        assert lo < r1 < hi and lo < r2 < hi, (order, errs, r1, r2)
        assert np.array_equal(run(order, 0.2, scale=2.0 ** -9), run(order, 0.2) * 2.0 ** -9)
    assert np.abs(run(3, 0.2) - run(4, 0.2)).max() > 1e-8 and np.abs(run(3, 0.2) - run(2, 0.2)).max() > 1e-8
    # the fixed-background rule is not the dynamical one with a small back-reaction: at this amplitude they differ
    dyn = oracle.Evolution(Phi0, Pi0, courant=0.2, ko_eps=0.0, rk_order=3).step(50)
    fix = oracle.Evolution(Phi0, Pi0, courant=0.2, ko_eps=0.0, rk_order=3, fixed_background=True).step(50)
    assert np.abs(dyn.Phi[0] - fix.Phi[0]).max() > 1e-4
    def energy(ev):
        return (tb["w"][:-1] * tb["T"][:-1] * (ev.Phi[0][:-1] ** 2 + ev.Pi[0][:-1] ** 2)).sum()
    Phi1 = de1.copy(); Phi1[0] = Phi1[-1] = 0.0
    # |R(iy)|^2 - 1 per step, y = w dt, w = omega_1 = 5: Heun-3 -y^4/12, midpoint +y^4/4; over one period t = pi.
    # (The midpoint rule amplifies EVERY mode, the grid's highest by (w_max dt)^4/4 per step: at courant 1/4 rounding
    # noise gains e^3.5 over the 1024 steps, harmless; at 1/2 it would swamp the solution.)
    for order, courant, sign in ((3, 0.5, -1.0), (2, 0.25, +1.0)):
        n = int(round(2 * (N - 1) / courant))
        ev = oracle.Evolution(Phi1, np.zeros(N), courant=courant, ko_eps=0.0, rk_order=order, fixed_background=True)
        E0 = energy(ev); ev.step(n); E1 = energy(ev)
        y = 5.0 * courant * h
        expect = (-(y ** 4) / 12.0 if order == 3 else (y ** 4) / 4.0) * n
        assert sign * (E1 / E0 - 1.0) > 0 and abs((E1 / E0 - 1.0) / expect - 1.0) < 0.02, (order, E1 / E0 - 1.0, expect)
