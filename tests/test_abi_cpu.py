"""No-GPU checks of the boundary: libtc.so builds, loads, and exports every symbol include/tc.h declares;
host-side argument validation; the z-sharding helper used by bench.py --gpus N (gloo, world_size 2)."""
import ctypes, os, re, subprocess, sys
import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib():
    from paper_2304_12934_b200 import build
    return ctypes.CDLL(build.build())


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "tc.h")).read()
    names = set(re.findall(r"\b(tc_[a-z0-9_]+)\s*\(", hdr))
    assert {"tc_plan_create", "tc_plan_destroy", "tc_radon", "tc_backproject", "tc_mbir", "tc_radon1",
            "tc_power_iteration", "tc_prior_eval", "tc_last_error", "tc_launch_count", "tc_last_sched_stats", "tc_fbp",
            "tc_mbir_sharded", "tc_preprocess", "tc_host_alloc", "tc_host_free", "tc_stage_fine_grid", "tc_stage_gather", "tc_stage_spread"} <= names
    lib = _lib()
    for n in names:
        assert hasattr(lib, n), n


def test_argument_validation_without_gpu():
    from paper_2304_12934_b200 import binding as tc
    ang = np.zeros(4, dtype=np.float32)
    for kw, status in ((dict(n=63, n_det=64), tc.TC_EINVAL), (dict(n=64, n_det=63), tc.TC_EINVAL),
                       (dict(n=0, n_det=64), tc.TC_EINVAL), (dict(n=48, n_det=64), tc.TC_EUNSUPPORTED),
                       (dict(n=352, n_det=64), tc.TC_EUNSUPPORTED), (dict(n=64, n_det=26), tc.TC_EUNSUPPORTED)):      # factors 11, 13
        with pytest.raises(tc.TcError) as e:
            tc.Plan(kw["n"], kw["n_det"], ang)
        assert e.value.status == status, kw
    bad = np.array([0.0, np.nan], dtype=np.float32)
    with pytest.raises(tc.TcError) as e:
        tc.Plan(64, 64, bad)
    assert e.value.status == tc.TC_EINVAL
    g = tc.tc_geom(64, 64, 2, ang.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), -1.0, 1.5, 6)
    h = ctypes.c_void_p()
    assert tc.lib.tc_plan_create(ctypes.byref(g), 0, ctypes.byref(h)) == tc.TC_EUNSUPPORTED
    assert tc.lib.tc_plan_create(None, 0, ctypes.byref(h)) == tc.TC_EINVAL
    assert tc.lib.tc_radon(None, None, 1, None, None) == tc.TC_EINVAL
    assert b"null" in tc.lib.tc_last_error()


def test_product_path_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2304_12934_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".inc", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle|oracle/.*\.(py|c)\b.*open|#include.*oracle", src, re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2304_12934_b200" not in src and "from paper_2304_12934_b200" not in src


def test_shard_slices_partition():
    from paper_2304_12934_b200.shard import shard_slices
    for S in (1, 7, 128, 2160):
        for W in (1, 2, 3, 8):
            parts = [shard_slices(S, r, W) for r in range(W)]
            assert parts[0][0] == 0 and parts[-1][1] == S
            assert all(parts[i][1] == parts[i + 1][0] for i in range(W - 1))
            assert max(b - a for a, b in parts) - min(b - a for a, b in parts) <= 8


_WORKER = r'''
import os, sys, torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_2304_12934_b200.shard import shard_slices, max_over_ranks, TorchComm
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%s" % sys.argv[2], rank=int(sys.argv[3]), world_size=2)
r = dist.get_rank()
lo, hi = shard_slices(20, r, 2)
t = max_over_ranks(1.0 + r, device="cpu")
tot = torch.tensor([float(hi - lo)]); dist.all_reduce(tot)
assert t == 2.0 and tot.item() == 20.0, (t, tot)
# the transport of tc_mbir_sharded (include/tc.h: tc_comm): halo slices to the z-neighbours, sum of the objective's terms
c = TorchComm(4, device="cpu")
assert (c.send_down is None) == (r == 0) and (c.send_up is None) == (r == 1)
if r == 0: c.send_up.fill_(10.0)
else: c.send_down.fill_(21.0)
c.exchange()
if r == 0: assert torch.all(c.recv_up == 21.0)
else: assert torch.all(c.recv_down == 10.0)
assert c.allreduce([1.0 + r, 0.5, -2.0 * r, 0.0]) == [3.0, 1.0, -2.0, 0.0]
dist.barrier(); dist.destroy_process_group()
'''


def test_gloo_world2_sharding_and_timing_reduction(tmp_path):
    w = tmp_path / "w.py"; w.write_text(_WORKER)
    port = str(29500 + os.getpid() % 2000)
    ps = [subprocess.Popen([sys.executable, str(w), ROOT, port, str(r)]) for r in range(2)]
    assert [p.wait(timeout=120) for p in ps] == [0, 0]
