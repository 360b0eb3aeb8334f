"""CPU-only checks of the boundary and the host logic (no compute calls, no GPU):
the C-ABI library builds, loads and exports every symbol include/adsc.h declares;
host-side argument checks; member sharding incl. a world_size-2 gloo run."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1706_07413_b200 import build, binding
    build.build()
    return binding.load_library()


def _declared_in_header():
    src = open(os.path.join(ROOT, "include", "adsc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(adsc_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    from paper_1706_07413_b200 import binding
    names = _declared_in_header()
    assert len(names) >= 15 and "adsc_step" in names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/adsc.h but not exported by libadsc.so"
    # the binding forwards exactly the declared entry points, under the same names
    assert binding.exported_symbols() == names
    for n in names:
        if n in ("adsc_last_error",):
            continue
        assert callable(getattr(binding, n)), n


def test_library_is_standalone_cuda_for_sm100a():
    """libadsc.so carries sm_100a SASS and does not link torch or the oracle."""
    from paper_1706_07413_b200 import binding
    out = subprocess.run(["cuobjdump", "-lelf", binding._LIBPATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out, out
    ldd = subprocess.run(["ldd", binding._LIBPATH], capture_output=True, text=True).stdout
    assert "torch" not in ldd and "oracle" not in ldd


def test_diag_struct_layout_matches_header(lib):
    from paper_1706_07413_b200 import binding
    assert C.sizeof(binding.adsc_diag) == 56 == binding.DIAG_DTYPE.itemsize
    offs = {n: getattr(binding.adsc_diag, n).offset for n, _ in binding.adsc_diag._fields_}
    assert offs == {k: binding.DIAG_DTYPE.fields[k][1] for k in offs}


def test_create_argument_checks_and_workspace_size(lib):
    for bad in ((8, 1, 0.25, 0.1), (10, 1, 0.25, 0.1), (1025, 0, 0.25, 0.1), (1025, 1, 0.0, 0.1),
                (1025, 1, 1.5, 0.1), (1025, 1, 0.25, -1.0), (1025, 1, float("nan"), 0.1), (1025, 65536, 0.25, 0.1)):
        assert not lib.adsc_create(*bad), bad
        assert lib.adsc_last_error(None)
    h = lib.adsc_create(4097, 16, 0.25, 0.1)
    assert h
    try:
        need = lib.adsc_workspace_bytes(h)
        assert need >= 3 * 16 * 4097 * 8            # at least the three state fields
        cl = C.c_int(0)
        assert lib.adsc_path(h, C.byref(cl)) == 2 and cl.value >= 1      # resident path holds N=4097
        # call-order and argument errors are reported without touching a device
        assert lib.adsc_step(h, 1) == -2
        assert lib.adsc_set_option(h, 99, 1.0) == -1
        assert lib.adsc_set_option(h, 1, float("nan")) == -1
        assert lib.adsc_set_option(h, 2, 2.5) == -1
        assert lib.adsc_set_option(h, 2, 16.0) == 0
        assert lib.adsc_bind(h, None, 0, None) == -1
        assert lib.adsc_diagnostics(h, None) == -2
        assert lib.adsc_launch_count(h) == 0
        # forcing the streaming path changes the workspace (stage buffers)
        assert lib.adsc_set_option(h, 3, 1.0) == 0
        assert lib.adsc_path(h, None) == 1
        assert lib.adsc_workspace_bytes(h) > need
    finally:
        assert lib.adsc_destroy(h) == 0
    big = lib.adsc_create(2 ** 20 + 1, 1, 0.25, 0.1)
    assert big and lib.adsc_path(big, None) == 1                      # does not fit on chip
    assert lib.adsc_set_option(big, 3, 2.0) == -1
    lib.adsc_destroy(big)
    assert lib.adsc_workspace_bytes(None) == 0 and lib.adsc_destroy(None) == 0


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1706_07413_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "adsc_oracle" not in txt, f


def test_member_range_partitions():
    from paper_1706_07413_b200 import shard
    for n, w in ((1024, 1), (1024, 8), (10, 4), (3, 8), (0, 2)):
        r = [shard.member_range(k, w, n) for k in range(w)]
        assert r[0][0] == 0 and r[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
        sizes = [b - a for a, b in r]
        assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.member_range(2, 2, 10)


_GLOO_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import numpy as np
import torch.distributed as dist
from paper_1706_07413_b200 import shard, inputs, binding
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
B = 7
lo, hi = shard.member_range(rank, world, B)
Phi, Pi, prm = inputs.make("cfg5", B=B, N=129)
# each rank would hand Phi[lo:hi], Pi[lo:hi] to its own Ensemble; here (no GPU) the records are synthetic
rec = np.zeros(hi - lo, dtype=binding.DIAG_DTYPE)
rec["steps_done"] = np.arange(lo, hi)
rec["mass"] = prm["eps"][lo:hi]
out = shard.gather_diagnostics(rec)
if rank == 0:
    assert out.shape == (B,), out.shape
    assert (out["steps_done"] == np.arange(B)).all()
    assert np.array_equal(out["mass"], prm["eps"])
    print("GLOO_OK")
else:
    assert out is None
dist.destroy_process_group()
"""


def test_sharding_world_size_2_gloo(tmp_path):
    """N>1 host path: two gloo ranks shard the members and gather the per-member records
    (the data path has no collective — members are independent)."""
    script = tmp_path / "worker.py"
    script.write_text(_GLOO_WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29571", str(script)],
                       capture_output=True, text=True, env=env, timeout=240)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "GLOO_OK" in r.stdout
