"""adsc_mode_energies_static: the entry point for callers that cannot allocate GPU memory.

Some users of libadsc run inside a process that handed the whole GPU to its own memory pool at start-up (a
training or serving job with a caching allocator, a client under a fixed per-process memory limit), or on a
latency-critical path where cudaMalloc / cudaFree are banned because they stall the device.  For them the library
has one entry point that needs no handle and no workspace: the caller passes Phi, Pi and the output array, and the
slice partial sums, the only memory the computation needs besides those, sit in a 2 MiB array compiled into the
library (one per GPU, shared by all calls on that GPU, never cleared between calls).

What is checked here: its output against the existing path (adsc_mode_energies on a handle set from the same
fields) at the tolerance the mode-energy parity test uses, 1e-11 of the member's largest E_j, on TWO calls in a
row whose shapes differ, so that the second call runs on top of whatever the first one left in the shared array;
then the first shape again, which must reproduce its first answer bit for bit; and that a request larger than the
built-in array is refused with a message instead of being run.  The inputs live in torch tensors only because the
test has to put them somewhere; the entry point itself never sees torch and allocates nothing.

The file name sorts after the other test files on purpose: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It passes both alone in a fresh process (the first call then does the
per-device look-up of the built-in array) and after the rest of the suite.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

RTOL = 1e-11      # of max_j E_j per member: tests/test_gpu_parity.py::test_mode_energies_match_oracle


def _existing_path(binding, torch, Phi, Pi, J):
    B, N = Phi.shape
    ens = binding.Ensemble(N, B)
    ens.set_initial(torch.from_numpy(Phi).cuda(), torch.from_numpy(Pi).cuda())
    E = ens.mode_energies(J)
    ens.close()
    return E


def _static_path(binding, torch, Phi, Pi, J):
    B, N = Phi.shape
    dPhi, dPi = torch.from_numpy(Phi).cuda(), torch.from_numpy(Pi).cuda()
    dE = torch.full((B, J), float("nan"), dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream()
    binding.adsc_mode_energies_static(N, B, J, dPhi.data_ptr(), dPi.data_ptr(), dE.data_ptr(), st.cuda_stream)
    st.synchronize()
    return dE.cpu().numpy()


def test_static_scratch_entry_point_matches_existing_path_twice():
    import torch
    from paper_1706_07413_b200 import binding, inputs
    assert torch.cuda.is_available()
    binding.load_library()
    # two shapes with different slice counts and partial-sum layouts: 5 members x 16 modes on 8193 points
    # (several slices per member), then 300 members x 7 modes on 1025 points (one slice per member)
    cases = [("cfg3", 5, 8193, 16), ("cfg5", 300, 1025, 7)]
    first = None
    for name, B, N, J in cases:
        Phi, Pi, _ = inputs.make(name, B=B, N=N)
        # the caller's arrays are used as they are: values at the end points must not matter (the handle path zeroes them)
        Phi = Phi.copy(); Pi = Pi.copy()
        Phi[:, 0] = 3.0; Phi[:, -1] = -2.0; Pi[:, -1] = 5.0
        E_ref = _existing_path(binding, torch, Phi, Pi, J)
        E = _static_path(binding, torch, Phi, Pi, J)
        assert np.isfinite(E).all()
        scale = E_ref.max(axis=1, keepdims=True)
        err = np.max(np.abs(E - E_ref) / scale)
        assert err <= RTOL, (name, err)
        if first is None:
            first = (Phi, Pi, J, E)
    # the first shape again, on top of the second call's leftovers: the same bits as before
    Phi, Pi, J, E0 = first
    assert np.array_equal(_static_path(binding, torch, Phi, Pi, J), E0)


def test_static_scratch_entry_point_refuses_what_does_not_fit():
    import torch
    from paper_1706_07413_b200 import binding
    lib = binding.load_library()
    N, J = 1025, 32
    B = 131072 // J + 1                       # batch * J one member beyond ADSC_STATIC_SCRATCH_BYTES / 16
    d = torch.zeros((B, N), dtype=torch.float64, device="cuda")
    out = torch.zeros((B, J), dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    assert lib.adsc_mode_energies_static(N, B, J, d.data_ptr(), d.data_ptr(), out.data_ptr(), st) == binding.ADSC_EINVAL
    assert b"built-in scratch" in lib.adsc_last_error(None)
    assert lib.adsc_mode_energies_static(N, B - 1, J, d.data_ptr(), d.data_ptr(), out.data_ptr(), st) == binding.ADSC_OK
    torch.cuda.synchronize()
    assert (out[: B - 1] == 0).all()
    for bad in [(1024, 4, 4), (1025, 0, 4), (1025, 4, 0), (1025, 4, 33), (9, 1, 3)]:
        assert lib.adsc_mode_energies_static(*bad, d.data_ptr(), d.data_ptr(), out.data_ptr(), st) == binding.ADSC_EINVAL
    assert lib.adsc_mode_energies_static(N, 4, 4, None, d.data_ptr(), out.data_ptr(), st) == binding.ADSC_EINVAL
