"""Seeded synthetic initial data, shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no stencils, scans, RK
stages): it only evaluates analytic profiles Phi(x,0), Pi(x,0) on the grid
x_i = i*(pi/2)/(N-1) and draws the ensemble parameters.  It imports neither
the oracle nor the CUDA library.

Workloads (BASELINE.json configs; recipe in DESIGN.md "Input recipe"):
  cfg1  N=1025  B=1      Gaussian Pi, sigma=1/16, eps=1
  cfg2  N=4097  B=1024   Gaussian Pi, sigma=1/16, eps~U[0.5,5]
  cfg3  N=8193  B=4096   two-mode e_0,e_1 mixture (R19, R20)
  cfg4  N=2^20+1 B=1     Gaussian Pi, sigma=1/16, eps=1
  cfg5  N=2049  B=16384  Gaussian Pi, sigma~U[0.2,0.5], eps~U[0.05,0.5]
  tcollapse N=1025 B=64  Gaussian Pi, sigma=1/16, eps~U[30,60] (test only)
  paper32k N=2^15+1 B=64 eq (13) family k_d=3, mu=1, one member per amplitude (the paper's production shape)
The paper's own initial data are mode sums with Phi(x,0)=0 (PAPER.md:89-93,
111); no public dataset is involved, these seeded ensembles stand in.  qp_family()
generates the paper's families themselves (eq (13)) for the t_c(eps) driver.
"""
from __future__ import annotations

import math

import numpy as np

SEED0 = 170607413


def grid(N: int) -> np.ndarray:
    """x_i = i*h, h=(pi/2)/(N-1); the last point is pi/2 up to rounding."""
    return np.arange(N, dtype=np.float64) * ((np.pi / 2) / (N - 1))


def gaussian_Pi(N: int, eps, sigma) -> np.ndarray:
    """Pi(x,0) = (2 eps/pi) exp(-4 tan^2 x/(pi^2 sigma^2)), Pi_{N-1}=0 exactly
    (BASELINE.json configs[0]; reading R21).  eps, sigma scalars or [B]."""
    eps = np.atleast_1d(np.asarray(eps, dtype=np.float64))[:, None]
    sigma = np.atleast_1d(np.asarray(sigma, dtype=np.float64))[:, None]
    x = grid(N)[None, :-1]
    t2 = np.tan(x) ** 2
    Pi = np.zeros((max(eps.shape[0], sigma.shape[0]), N))
    Pi[:, :-1] = (2.0 * eps / np.pi) * np.exp(-4.0 * t2 / (np.pi ** 2 * sigma ** 2))
    return Pi


def _poch(a: float, m: int) -> float:
    r = 1.0
    for q in range(m):
        r *= a + q
    return r


def eigenmode(j: int, x: np.ndarray):
    """AdS4 scalar normal mode e_j and its derivative e_j' (R19):
    e_j = d_j cos^3 x 2F1(-j, 3+j; 3/2; sin^2 x), d_j = sqrt(16(j+1)(j+2)/pi),
    orthonormal under int_0^{pi/2} e_j e_k tan^2 x dx, frequency omega_j = 3+2j.
    The hypergeometric series terminates after j+1 terms."""
    d = math.sqrt(16.0 * (j + 1) * (j + 2) / math.pi)
    s, c = np.sin(x), np.cos(x)
    z = s * s
    F = np.zeros_like(x)
    dF = np.zeros_like(x)      # dF/dz
    for m in range(j + 1):
        coef = _poch(-j, m) * _poch(3 + j, m) / (_poch(1.5, m) * math.factorial(m))
        F += coef * z ** m
        if m >= 1:
            dF += coef * m * z ** (m - 1)
    e = d * c ** 3 * F
    de = d * (-3.0 * c ** 2 * s * F + c ** 3 * dF * 2.0 * s * c)
    return e, de


def eigenmode_jacobi(j: int, x: np.ndarray) -> np.ndarray:
    """e_j through the Jacobi polynomial, 2F1(-j, 3+j; 3/2; sin^2 x) = j!/(3/2)_j P_j^(1/2,3/2)(cos 2x): the
    three-term recurrence stays accurate for the high modes of the paper's mode-sum data (the terminating
    series of eigenmode() loses digits to cancellation beyond j ~ 10)."""
    from scipy.special import eval_jacobi, gammaln
    d = math.sqrt(16.0 * (j + 1) * (j + 2) / math.pi)
    norm = math.exp(gammaln(j + 1.0) + gammaln(1.5) - gammaln(j + 1.5))
    return d * np.cos(x) ** 3 * norm * eval_jacobi(j, 0.5, 1.5, np.cos(2.0 * x))


def qp_family(N: int, eps, mu: float, kd: int, kmax: int | None = None):
    """The paper's approximately quasi-periodic families (eq (13)):
    mode amplitudes A_k = eps exp(-mu |k - k_d|), initial data with Phi(x,0) = 0 (Fig. 2 caption,
    PAPER.md:111).  Reading R23: phi = sum_k A_k e_k sin(omega_k t), so Pi(x,0) = sum_k A_k omega_k e_k(x).
    eps scalar or [B] (one member per amplitude); modes k = 0..kmax, kmax defaults to where the tail is
    below 1e-17 of the peak.  Returns (Phi, Pi, A_k[B][kmax+1])."""
    eps = np.atleast_1d(np.asarray(eps, dtype=np.float64))
    if kmax is None:
        kmax = kd + int(math.ceil(39.2 / mu))
    x = grid(N)
    k = np.arange(kmax + 1)
    shape = np.exp(-mu * np.abs(k - kd))
    prof = np.zeros(N)
    for j in k:
        prof += shape[j] * omega(int(j)) * eigenmode_jacobi(int(j), x)
    Pi = eps[:, None] * prof[None, :]
    Pi[:, -1] = 0.0
    return np.zeros_like(Pi), Pi, eps[:, None] * shape[None, :]


def omega(j: int) -> float:
    return 3.0 + 2.0 * j


def two_mode(N: int, a_tot, ratio, theta1):
    """phi = sum_{j=0,1} a_j e_j cos(omega_j t + theta_j) at t=0 (R20):
    Phi = sum a_j cos(theta_j) e_j',  Pi = -sum a_j omega_j sin(theta_j) e_j,
    theta_0=0; a_tot=sqrt(a_0^2+a_1^2); ratio = E_1/E_0 with E_j=omega_j^2 a_j^2."""
    a_tot, ratio, theta1 = (np.atleast_1d(np.asarray(v, dtype=np.float64))
                            for v in (a_tot, ratio, theta1))
    x = grid(N)
    e0, de0 = eigenmode(0, x)
    e1, de1 = eigenmode(1, x)
    q = (omega(0) / omega(1)) * np.sqrt(ratio)          # a_1/a_0
    a0 = a_tot / np.sqrt(1.0 + q * q)
    a1 = q * a0
    Phi = a0[:, None] * de0[None, :] + (a1 * np.cos(theta1))[:, None] * de1[None, :]
    Pi = -(a1 * omega(1) * np.sin(theta1))[:, None] * e1[None, :]
    Phi[:, 0] = 0.0; Phi[:, -1] = 0.0; Pi[:, -1] = 0.0
    return Phi, Pi


PAPER32K_EPS = (0.02, 0.08)       # amplitude range of the paper32k ensemble (smallest, largest)

CONFIGS = {
    # name: (N, B, steps, courant, ko_eps)
    "cfg1": dict(N=1025, B=1, steps=26076, idx=1),
    "cfg2": dict(N=4097, B=1024, steps=521519, idx=2),
    "cfg3": dict(N=8193, B=4096, steps=20000, idx=3),
    "cfg4": dict(N=2 ** 20 + 1, B=1, steps=1000, idx=4),
    "cfg5": dict(N=2049, B=16384, steps=2607595, idx=5),
    "tcollapse": dict(N=1025, B=64, steps=10431, idx=6),
    # the paper's production shape: 2^15 points, RK3, one member per amplitude of the
    # k_d = 3, mu = 1 family of eq (13); the amplitudes are ours (the paper prints none), equally spaced in 1/eps^2
    "paper32k": dict(N=2 ** 15 + 1, B=64, steps=41721513, idx=7),
}


def make(name: str, B: int | None = None, N: int | None = None, lo: int = 0):
    """(Phi, Pi, params) for a named workload, members [lo, B) of the (tiled) ensemble (default all).
    seed = 170607413 + config index; same arrays feed oracle and GPU."""
    cfg = CONFIGS[name]
    N = N or cfg["N"]
    Bfull = cfg["B"]
    B = Bfull if B is None else B
    rng = np.random.default_rng(SEED0 + cfg["idx"])
    if name in ("cfg1", "cfg4"):
        eps = np.full(Bfull, 1.0); sig = np.full(Bfull, 1.0 / 16)
    elif name == "cfg2":
        eps = rng.uniform(0.5, 5.0, Bfull); sig = np.full(Bfull, 1.0 / 16)
    elif name == "cfg5":
        sig = rng.uniform(0.2, 0.5, Bfull); eps = rng.uniform(0.05, 0.5, Bfull)
    elif name == "tcollapse":
        eps = rng.uniform(30.0, 60.0, Bfull); sig = np.full(Bfull, 1.0 / 16)
    elif name == "paper32k":
        inv2 = np.linspace(1.0 / PAPER32K_EPS[1] ** 2, 1.0 / PAPER32K_EPS[0] ** 2, Bfull)
        eps = 1.0 / np.sqrt(inv2)
        reps = -(-B // Bfull)
        eps = np.tile(eps, reps)[lo:B]
        Phi, Pi, _ = qp_family(N, eps, mu=1.0, kd=3)
        return Phi, Pi, dict(eps=eps, mu=1.0, kd=3)
    elif name == "cfg3":
        a = rng.uniform(0.01, 0.1, Bfull); r = rng.uniform(0.2, 1.0, Bfull)
        th = rng.uniform(0.0, 2 * np.pi, Bfull)
        reps = -(-B // Bfull)
        a, r, th = (np.tile(v, reps)[lo:B] for v in (a, r, th))
        Phi, Pi = two_mode(N, a, r, th)
        return Phi, Pi, dict(a_tot=a, ratio=r, theta1=th)
    reps = -(-B // Bfull)
    eps, sig = np.tile(eps, reps)[lo:B], np.tile(sig, reps)[lo:B]
    Pi = gaussian_Pi(N, eps, sig)
    Phi = np.zeros_like(Pi)
    return Phi, Pi, dict(eps=eps, sigma=sig)
