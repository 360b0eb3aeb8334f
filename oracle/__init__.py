"""ctypes view of oracle/adsc_oracle.c — TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this package.  It never imports the CUDA package.
All arithmetic lives in adsc_oracle.c; this file only builds it (gcc -O2
-ffp-contract=off -fopenmp) and marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "adsc_oracle.c")
_SO = os.path.join(_HERE, "libadsc_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle shared library beside its source (idempotent)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
             "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO




def _cpu_tag() -> str:
    """-march=native code only runs on the CPU model it was built on: one library per model."""
    import hashlib
    try:
        with open("/proc/cpuinfo") as f:
            flags = next((l for l in f if l.startswith("flags")), "")
    except OSError:
        flags = ""
    return hashlib.sha1(flags.encode()).hexdigest()[:10]


_SO_FAST = os.path.join(_HERE, f"libadsc_oracle_fast_{_cpu_tag()}.so")
FAST_FLAGS = ["-O3", "-march=native", "-ffp-contract=fast"]


def build_fast(force: bool = False) -> str:
    """The SAME source with throughput flags (gcc -O3 -march=native, contraction allowed), as a second library.
    It is not the oracle: bench.py times it beside the oracle so that the CPU baseline is not only the unoptimised
    checker, and checks it against the oracle before quoting it."""
    if force or not os.path.exists(_SO_FAST) or os.path.getmtime(_SO_FAST) < os.path.getmtime(_SRC):
        tmp = _SO_FAST + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-std=c11", *FAST_FLAGS, "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO_FAST)
    return _SO_FAST


_lib = None
_libs = {}


def use_build(which: str = "oracle"):
    """Select the library the wrappers below call: "oracle" (default; the checker) or "fast" (build_fast)."""
    global _lib
    if which not in _libs:
        _libs[which] = C.CDLL(build() if which == "oracle" else build_fast())
    _lib = _libs[which]


def lib():
    if _lib is None:
        use_build("oracle")
    return _lib


_dp = C.POINTER(C.c_double)


def _p(a):
    return a.ctypes.data_as(_dp)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def tables(N: int):
    sc, T, Cc, w = (np.zeros(N) for _ in range(4))
    assert lib().oracle_tables(C.c_int(N), _p(sc), _p(T), _p(Cc), _p(w)) == 0
    return {"sc": sc, "T": T, "C": Cc, "w": w, "h": (np.pi / 2) / (N - 1)}


def D4(u, p0: int, ppi: int):
    u = _f64(u); out = np.zeros_like(u)
    lib().oracle_D4(C.c_int(u.size), _p(u), C.c_int(p0), C.c_int(ppi), _p(out))
    return out


def KO(u, eps: float, p0: int, ppi: int):
    u = _f64(u); out = np.zeros_like(u)
    lib().oracle_KO(C.c_int(u.size), C.c_double(eps), _p(u), C.c_int(p0), C.c_int(ppi), _p(out))
    return out


def cumrule(g, p0: int, ppi: int):
    g = _f64(g); out = np.zeros(g.size - 1)
    lib().oracle_cumrule(C.c_int(g.size), _p(g), C.c_int(p0), C.c_int(ppi), _p(out))
    return out


def delta_solve(Phi, Pi):
    Phi, Pi = _f64(Phi), _f64(Pi); d = np.zeros_like(Phi)
    assert lib().oracle_delta_solve(C.c_int(Phi.size), _p(Phi), _p(Pi), _p(d)) == 0
    return d


def A_solve(Phi, Pi, delta):
    Phi, Pi, delta = _f64(Phi), _f64(Pi), _f64(delta); A = np.zeros_like(Phi)
    assert lib().oracle_A_solve(C.c_int(Phi.size), _p(Phi), _p(Pi), _p(delta), _p(A)) == 0
    return A


def rhs(Phi, Pi, A, ko_eps: float):
    Phi, Pi, A = _f64(Phi), _f64(Pi), _f64(A)
    kP, kQ, kA, d = (np.zeros_like(Phi) for _ in range(4))
    assert lib().oracle_rhs(C.c_int(Phi.size), C.c_double(ko_eps), _p(Phi), _p(Pi), _p(A),
                            _p(kP), _p(kQ), _p(kA), _p(d)) == 0
    return kP, kQ, kA, d


def rhs_fixed(Phi, Pi, ko_eps: float):
    """Right-hand side on the fixed background A = 1, delta = 0."""
    Phi, Pi = _f64(Phi), _f64(Pi)
    A = np.ones_like(Phi)
    kP, kQ, kA, d = (np.zeros_like(Phi) for _ in range(4))
    assert lib().oracle_rhs_fixed(C.c_int(Phi.size), C.c_double(ko_eps), _p(Phi), _p(Pi), _p(A),
                                  _p(kP), _p(kQ), _p(kA), _p(d)) == 0
    return kP, kQ, kA, d


def set_initial(Phi, Pi):
    """[B][N] (or [N]) -> dict of Phi, Pi (Dirichlet-forced copies), A, delta."""
    Phi = np.array(np.atleast_2d(Phi), dtype=np.float64, order="C")
    Pi = np.array(np.atleast_2d(Pi), dtype=np.float64, order="C")
    B, N = Phi.shape
    A = np.zeros_like(Phi); d = np.zeros_like(Phi)
    assert lib().oracle_set_initial(C.c_int(N), C.c_int(B), _p(Phi), _p(Pi), _p(A), _p(d)) == 0
    return {"Phi": Phi, "Pi": Pi, "A": A, "delta": d}


def diagnostics(Phi, Pi, A):
    Phi, Pi, A = (_f64(np.atleast_2d(a)) for a in (Phi, Pi, A))
    B, N = Phi.shape
    mass, resid, mn = np.zeros(B), np.zeros(B), np.zeros(B)
    arg = np.zeros(B, dtype=np.int32)
    assert lib().oracle_diagnostics(C.c_int(N), C.c_int(B), _p(Phi), _p(Pi), _p(A), _p(mass),
                                    _p(resid), _p(mn),
                                    arg.ctypes.data_as(C.POINTER(C.c_int))) == 0
    return {"mass": mass, "resid": resid, "min_A": mn, "argmin_A": arg}


class Evolution:
    """A batch evolved by the oracle: state in numpy, stepped in place."""

    def __init__(self, Phi, Pi, courant: float = 0.25, ko_eps: float = 0.1,
                 thr: float = 2.0 ** -7, K_A: int = 0, nthreads: int = 1, fixed_background: bool = False,
                 rk_order: int = 4):
        s = set_initial(Phi, Pi)
        self.Phi, self.Pi, self.A = s["Phi"], s["Pi"], s["A"]
        self.fixed_background = bool(fixed_background)
        self.rk_order = int(rk_order)
        assert self.rk_order in (2, 3, 4)
        if self.fixed_background:          # A and delta held fixed at 1 and 0
            self.A = np.ones_like(self.Phi)
        self.B, self.N = self.Phi.shape
        self.courant, self.ko_eps, self.thr, self.K_A = courant, ko_eps, thr, K_A
        self.nthreads = nthreads
        self.h = (np.pi / 2) / (self.N - 1)
        self.dt = courant * self.h
        self.steps_done = np.zeros(self.B, dtype=np.int64)
        self.collapsed = np.zeros(self.B, dtype=np.int32)
        self.t_collapse = np.full(self.B, np.nan)

    def step(self, nsteps: int):
        if self.fixed_background and self.rk_order != 4:   # PAPER.md:57 + :177: Table II runs with the third-order rule
            r = lib().oracle_evolve_fixed_rk(
                C.c_int(self.N), C.c_int(self.B), C.c_double(self.courant), C.c_double(self.ko_eps),
                C.c_int(self.rk_order), C.c_longlong(nsteps), _p(self.Phi), _p(self.Pi), _p(self.A),
                self.steps_done.ctypes.data_as(C.POINTER(C.c_longlong)),
                self.collapsed.ctypes.data_as(C.POINTER(C.c_int)), _p(self.t_collapse),
                C.c_int(self.nthreads))
            assert r == 0
            return self
        if self.fixed_background:
            r = lib().oracle_evolve_fixed(
                C.c_int(self.N), C.c_int(self.B), C.c_double(self.courant), C.c_double(self.ko_eps),
                C.c_longlong(nsteps), _p(self.Phi), _p(self.Pi), _p(self.A),
                self.steps_done.ctypes.data_as(C.POINTER(C.c_longlong)),
                self.collapsed.ctypes.data_as(C.POINTER(C.c_int)), _p(self.t_collapse),
                C.c_int(self.nthreads))
            assert r == 0
            return self
        if self.rk_order != 4:
            r = lib().oracle_evolve_rk(
                C.c_int(self.N), C.c_int(self.B), C.c_double(self.courant), C.c_double(self.ko_eps),
                C.c_double(self.thr), C.c_int(self.K_A), C.c_int(self.rk_order), C.c_longlong(nsteps),
                _p(self.Phi), _p(self.Pi), _p(self.A),
                self.steps_done.ctypes.data_as(C.POINTER(C.c_longlong)),
                self.collapsed.ctypes.data_as(C.POINTER(C.c_int)), _p(self.t_collapse),
                C.c_int(self.nthreads))
            assert r == 0
            return self
        r = lib().oracle_evolve(
            C.c_int(self.N), C.c_int(self.B), C.c_double(self.courant), C.c_double(self.ko_eps),
            C.c_double(self.thr), C.c_int(self.K_A), C.c_longlong(nsteps),
            _p(self.Phi), _p(self.Pi), _p(self.A),
            self.steps_done.ctypes.data_as(C.POINTER(C.c_longlong)),
            self.collapsed.ctypes.data_as(C.POINTER(C.c_int)), _p(self.t_collapse),
            C.c_int(self.nthreads))
        assert r == 0
        return self

    @property
    def delta(self):
        if self.fixed_background:
            return np.zeros_like(self.Phi)
        return np.stack([delta_solve(self.Phi[b], self.Pi[b]) for b in range(self.B)])

    def diagnostics(self):
        d = diagnostics(self.Phi, self.Pi, self.A)
        d.update(steps_done=self.steps_done.copy(), collapsed=self.collapsed.copy(),
                 t_collapse=self.t_collapse.copy(), t=self.steps_done * self.dt)
        return d


def eigenmode(N: int, j: int):
    """AdS4 normal mode e_j and e_j' on the grid (Jacobi recurrence in long double)."""
    e, de = np.zeros(N), np.zeros(N)
    assert lib().oracle_eigenmode(C.c_int(N), C.c_int(j), _p(e), _p(de)) == 0
    return e, de


def mode_energies(Phi, Pi, J: int):
    """E_j = Pi_j^2 + Phi_j^2/omega_j^2, j < J, per member (reading R24); also the projections."""
    Phi, Pi = (_f64(np.atleast_2d(a)) for a in (Phi, Pi))
    B, N = Phi.shape
    E = np.zeros((B, J)); proj = np.zeros((B, J, 2))
    assert lib().oracle_mode_energies(C.c_int(N), C.c_int(B), C.c_int(J), _p(Phi), _p(Pi), _p(E), _p(proj)) == 0
    return E, proj


def max_threads() -> int:
    return int(lib().oracle_max_threads())
