"""ctypes binding of libadsc.so (include/adsc.h): argument marshalling only.

Every function here has the name of the C entry point it forwards to; `Ensemble`
is a convenience wrapper that owns a torch-allocated workspace and a handle.
PyTorch supplies device memory and the stream; no field arithmetic happens in Python
and there is no CPU fallback: if the library is missing, loading raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libadsc.so")

ADSC_OK, ADSC_EINVAL, ADSC_ESTATE, ADSC_ENOMEM, ADSC_ECUDA = 0, -1, -2, -3, -4
ADSC_OPT_COLLAPSE_THRESHOLD = 1
ADSC_OPT_A_RESOLVE_PERIOD = 2
ADSC_OPT_PATH = 3
ADSC_OPT_STEPS_PER_LAUNCH = 4
ADSC_OPT_FIXED_BACKGROUND = 7
ADSC_OPT_RK_ORDER = 8
ADSC_OPT_SPREAD = 9
PATH_AUTO, PATH_STREAM, PATH_RESIDENT = 0, 1, 2
ADSC_PROBE_FP64_FMA, ADSC_PROBE_SHARED_LOAD = 0, 1


class adsc_diag(C.Structure):
    """Mirror of `adsc_diag` in include/adsc.h."""
    _fields_ = [("t", C.c_double), ("steps_done", C.c_longlong), ("min_A", C.c_double),
                ("argmin_A", C.c_int), ("collapsed", C.c_int), ("mass", C.c_double),
                ("constraint_residual", C.c_double), ("t_collapse", C.c_double)]


DIAG_DTYPE = np.dtype([("t", "f8"), ("steps_done", "i8"), ("min_A", "f8"), ("argmin_A", "i4"),
                       ("collapsed", "i4"), ("mass", "f8"), ("constraint_residual", "f8"),
                       ("t_collapse", "f8")], align=True)
assert DIAG_DTYPE.itemsize == C.sizeof(adsc_diag)


class AdscError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libadsc error {code}: {msg}")
        self.code = code


_lib = None

_SIGS = {
    "adsc_create": (C.c_void_p, [C.c_int, C.c_int, C.c_double, C.c_double]),
    "adsc_destroy": (C.c_int, [C.c_void_p]),
    "adsc_workspace_bytes": (C.c_size_t, [C.c_void_p]),
    "adsc_bind": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]),
    "adsc_set_option": (C.c_int, [C.c_void_p, C.c_int, C.c_double]),
    "adsc_set_initial": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "adsc_set_state": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "adsc_step": (C.c_int, [C.c_void_p, C.c_longlong]),
    "adsc_diagnostics": (C.c_int, [C.c_void_p, C.c_void_p]),
    "adsc_get_fields": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "adsc_set_initial_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "adsc_get_fields_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "adsc_mode_energies": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "adsc_mode_energies_static": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "adsc_get_fields_host_async": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "adsc_launch_count": (C.c_longlong, [C.c_void_p]),
    "adsc_path": (C.c_int, [C.c_void_p, C.POINTER(C.c_int)]),
    "adsc_last_error": (C.c_char_p, [C.c_void_p]),
    "adsc_selftest_exp": (C.c_int, [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]),
    "adsc_probe": (C.c_int, [C.c_int, C.c_double, C.POINTER(C.c_double)]),
}


def load_library(path: str | None = None):
    """dlopen libadsc.so and declare the prototypes.  Raises if it is not built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or _LIBPATH
    if not os.path.exists(p):
        raise ImportError(
            f"{p} is missing: build it with `python -m paper_1706_07413_b200.build` "
            "(libadsc has no CPU or PyTorch fallback)")
    lib = C.CDLL(p)
    for name, (res, args) in _SIGS.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    if path is None:
        _lib = lib
    return lib


def exported_symbols():
    return sorted(_SIGS)


def _check(h, code):
    if code != ADSC_OK:
        raise AdscError(code, load_library().adsc_last_error(h).decode())


# ------------------------------------------------------------------ plain forwards
def adsc_create(N, batch, courant, ko_eps):
    lib = load_library()
    h = lib.adsc_create(int(N), int(batch), float(courant), float(ko_eps))
    if not h:
        raise AdscError(ADSC_EINVAL, lib.adsc_last_error(None).decode())
    return h


def adsc_destroy(h):
    return load_library().adsc_destroy(h)


def adsc_workspace_bytes(h):
    return int(load_library().adsc_workspace_bytes(h))


def adsc_bind(h, d_workspace, nbytes, cuda_stream):
    _check(h, load_library().adsc_bind(h, d_workspace, nbytes, cuda_stream))


def adsc_set_option(h, key, value):
    _check(h, load_library().adsc_set_option(h, int(key), float(value)))


def adsc_set_initial(h, d_Phi, d_Pi):
    _check(h, load_library().adsc_set_initial(h, d_Phi, d_Pi))


def adsc_set_state(h, d_Phi, d_Pi, d_A):
    _check(h, load_library().adsc_set_state(h, d_Phi, d_Pi, d_A))


def adsc_step(h, nsteps):
    _check(h, load_library().adsc_step(h, int(nsteps)))


def adsc_diagnostics(h, host_out_ptr):
    _check(h, load_library().adsc_diagnostics(h, host_out_ptr))


def adsc_get_fields(h, d_Phi, d_Pi, d_A, d_delta):
    _check(h, load_library().adsc_get_fields(h, d_Phi, d_Pi, d_A, d_delta))


def adsc_set_initial_host(h, h_Phi, h_Pi):
    _check(h, load_library().adsc_set_initial_host(h, h_Phi, h_Pi))


def adsc_get_fields_host(h, h_Phi, h_Pi, h_A, h_delta):
    _check(h, load_library().adsc_get_fields_host(h, h_Phi, h_Pi, h_A, h_delta))


def adsc_mode_energies(h, J, host_out_ptr):
    _check(h, load_library().adsc_mode_energies(h, int(J), host_out_ptr))


def adsc_mode_energies_static(N, batch, J, d_Phi, d_Pi, d_E, cuda_stream):
    """Forward to the entry point that allocates nothing (scratch built into the library); device pointers."""
    _check(None, load_library().adsc_mode_energies_static(int(N), int(batch), int(J), d_Phi, d_Pi, d_E, cuda_stream))


def adsc_get_fields_host_async(h, h_Phi, h_Pi, h_A, h_delta):
    _check(h, load_library().adsc_get_fields_host_async(h, h_Phi, h_Pi, h_A, h_delta))


def adsc_launch_count(h):
    return int(load_library().adsc_launch_count(h))


def adsc_path(h):
    cl = C.c_int(0)
    p = load_library().adsc_path(h, C.byref(cl))
    return p, cl.value


def adsc_selftest_exp(x):
    """x: float64 [ngroups][8].  Returns (E [ngroups][8], tier [ngroups]) from the kernels' own exponential."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    assert x.ndim == 2 and x.shape[1] == 8
    E = np.empty_like(x)
    tier = np.empty(x.shape[0], dtype=np.int32)
    code = load_library().adsc_selftest_exp(x.shape[0], x.ctypes.data, E.ctypes.data, tier.ctypes.data)
    if code != ADSC_OK:
        raise AdscError(code, "adsc_selftest_exp failed")
    return E, tier


def adsc_probe(kind, target_ms=50.0):
    """flop/s (ADSC_PROBE_FP64_FMA) or bytes/s (ADSC_PROBE_SHARED_LOAD) measured on the current CUDA device."""
    out = C.c_double(0.0)
    code = load_library().adsc_probe(int(kind), float(target_ms), C.byref(out))
    if code != ADSC_OK:
        raise AdscError(code, "adsc_probe failed (no CUDA device?)")
    return out.value


# ------------------------------------------------------------------ convenience wrapper
class Ensemble:
    """A batch of members on one GPU.  Device tensors are torch float64 CUDA tensors of
    shape [batch, N]; host arrays are numpy float64 (pinned torch tensors also work)."""

    def __init__(self, N, batch, courant=0.25, ko_eps=0.1, device="cuda:0", stream=None,
                 path=PATH_AUTO, threshold=None, a_resolve_period=None, steps_per_launch=None,
                 fixed_background=False, rk_order=None, spread=False):
        import torch
        load_library()
        if not torch.cuda.is_available():
            raise AdscError(ADSC_ECUDA, "no CUDA device: libadsc has no CPU fallback")
        self.torch = torch
        self.N, self.batch = int(N), int(batch)
        self.device = torch.device(device)
        self.h = adsc_create(N, batch, courant, ko_eps)
        try:
            if fixed_background:
                adsc_set_option(self.h, ADSC_OPT_FIXED_BACKGROUND, 1)
            if rk_order is not None:
                adsc_set_option(self.h, ADSC_OPT_RK_ORDER, rk_order)
            if spread:
                adsc_set_option(self.h, ADSC_OPT_SPREAD, 1)
            if path != PATH_AUTO:
                adsc_set_option(self.h, ADSC_OPT_PATH, path)
            if threshold is not None:
                adsc_set_option(self.h, ADSC_OPT_COLLAPSE_THRESHOLD, threshold)
            if a_resolve_period is not None:
                adsc_set_option(self.h, ADSC_OPT_A_RESOLVE_PERIOD, a_resolve_period)
            if steps_per_launch is not None:
                adsc_set_option(self.h, ADSC_OPT_STEPS_PER_LAUNCH, steps_per_launch)
            with torch.cuda.device(self.device):
                self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
                nbytes = adsc_workspace_bytes(self.h)
                self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
                base = (self.workspace.data_ptr() + 255) // 256 * 256
                adsc_bind(self.h, base, nbytes, self.stream.cuda_stream)
        except Exception:
            adsc_destroy(self.h)
            self.h = None
            raise
        self.h_step = (np.pi / 2) / (self.N - 1)
        self.dt = courant * self.h_step

    def close(self):
        if getattr(self, "h", None):
            adsc_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers
    def _dev(self, t, name):
        torch = self.torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64
                and t.is_contiguous() and tuple(t.shape) == (self.batch, self.N)):
            raise ValueError(f"{name}: need a contiguous float64 CUDA tensor of shape "
                             f"({self.batch}, {self.N})")
        return t.data_ptr()

    def _host(self, a, name):
        torch = self.torch
        if isinstance(a, torch.Tensor):
            if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or \
                    tuple(a.shape) != (self.batch, self.N):
                raise ValueError(f"{name}: need a contiguous float64 host tensor")
            return a.data_ptr()
        if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous
                and a.shape == (self.batch, self.N)):
            raise ValueError(f"{name}: need a C-contiguous float64 array of shape "
                             f"({self.batch}, {self.N})")
        return a.ctypes.data

    # -- API
    def set_initial(self, Phi, Pi):
        with self.torch.cuda.device(self.device):
            if isinstance(Phi, self.torch.Tensor) and Phi.is_cuda:
                adsc_set_initial(self.h, self._dev(Phi, "Phi"), self._dev(Pi, "Pi"))
            else:
                adsc_set_initial_host(self.h, self._host(Phi, "Phi"), self._host(Pi, "Pi"))
        return self

    def set_state(self, Phi, Pi, A):
        with self.torch.cuda.device(self.device):
            adsc_set_state(self.h, self._dev(Phi, "Phi"), self._dev(Pi, "Pi"), self._dev(A, "A"))
        return self

    def step(self, nsteps):
        with self.torch.cuda.device(self.device):
            adsc_step(self.h, nsteps)
        return self

    def diagnostics(self):
        out = np.zeros(self.batch, dtype=DIAG_DTYPE)
        with self.torch.cuda.device(self.device):
            adsc_diagnostics(self.h, out.ctypes.data)
        return out

    def mode_energies(self, J):
        """[batch][J] normal-mode energies E_j of the current state (adsc_mode_energies)."""
        out = np.zeros((self.batch, int(J)), dtype=np.float64)
        with self.torch.cuda.device(self.device):
            adsc_mode_energies(self.h, J, out.ctypes.data)
        return out

    def get_fields(self, delta=True):
        torch = self.torch
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            out = {k: torch.empty((self.batch, self.N), dtype=torch.float64, device=self.device)
                   for k in (("Phi", "Pi", "A", "delta") if delta else ("Phi", "Pi", "A"))}
            adsc_get_fields(self.h, out["Phi"].data_ptr(), out["Pi"].data_ptr(), out["A"].data_ptr(),
                            out["delta"].data_ptr() if delta else None)
        return out

    def get_fields_host(self, delta=True, out=None, sync=True):
        """sync=False only enqueues the copies (adsc_get_fields_host_async): synchronise the stream, or call
        diagnostics(), before reading `out`."""
        keys = ("Phi", "Pi", "A", "delta") if delta else ("Phi", "Pi", "A")
        if out is None:
            out = {k: np.empty((self.batch, self.N)) for k in keys}
        fn = adsc_get_fields_host if sync else adsc_get_fields_host_async
        with self.torch.cuda.device(self.device):
            fn(self.h, *(self._host(out[k], k) if k in out else None for k in ("Phi", "Pi", "A", "delta")))
        return out

    @property
    def launch_count(self):
        return adsc_launch_count(self.h)

    @property
    def path(self):
        return adsc_path(self.h)


class PipelinedEnsemble:
    """The same batch cut into `parts` contiguous sub-batches, each with its own handle, workspace and CUDA
    stream, so that one sub-batch's host<->device transfers overlap another one's kernels (members are
    independent: there is nothing to exchange).  Host-side interface only: set_initial / get_fields_host take HOST
    arrays (pinned torch tensors overlap best) of shape [batch, N]; everything is enqueued asynchronously and
    `synchronize()` / `diagnostics()` wait for it.  Argument marshalling only, like Ensemble."""

    def __init__(self, N, batch, parts=2, device="cuda:0", **kw):
        import torch
        self.torch = torch
        self.N, self.batch = int(N), int(batch)
        parts = max(1, min(int(parts), self.batch))
        edges = [self.batch * k // parts for k in range(parts + 1)]
        self.ranges = [(edges[k], edges[k + 1]) for k in range(parts)]
        self.device = torch.device(device)
        self.streams = [torch.cuda.Stream(device=self.device) for _ in self.ranges]
        self.parts = [Ensemble(N, hi - lo, device=device, stream=st, **kw)
                      for (lo, hi), st in zip(self.ranges, self.streams)]
        self.dt = self.parts[0].dt

    def set_initial(self, Phi, Pi):
        for e, (lo, hi) in zip(self.parts, self.ranges):
            e.set_initial(Phi[lo:hi], Pi[lo:hi])
        return self

    def step(self, nsteps):
        for e in self.parts:
            e.step(nsteps)
        return self

    def get_fields_host(self, out, delta=False, sync=False):
        for e, (lo, hi) in zip(self.parts, self.ranges):
            e.get_fields_host(delta=delta, out={k: v[lo:hi] for k, v in out.items()}, sync=sync)
        return out

    def synchronize(self):
        for st in self.streams:
            st.synchronize()

    def diagnostics(self):
        return np.concatenate([e.diagnostics() for e in self.parts])

    @property
    def launch_count(self):
        return sum(e.launch_count for e in self.parts)

    def close(self):
        for e in self.parts:
            e.close()
