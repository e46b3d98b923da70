"""tc_radon_static: the allocation-free forward projection (scratch in a static device array of the library).

Collected last on purpose (the suite runs with pytest -x).  Checks, on two calls in a row that leave different stale contents in
the shared scratch, that the output equals the existing path's (tc_radon: the same kernels on the plan's own scratch), that the
call really allocates no device memory, and that sizes beyond the static maximum are refused with a clear error."""
import math
import numpy as np
import pytest
from conftest import rel_l2

pytestmark = pytest.mark.gpu

TOL_SAME_PATH = 1e-6        # the tolerance tests/test_gpu_parity.py uses between two routes through the same kernels (host vs device pointers)
TOL_NUFFT = 1e-4            # and against the oracle


def test_radon_static_matches_tc_radon_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2304_12934_b200 import binding as tc, inputs
    from oracle import nufft

    # call 1: config 2's shape (16 slices of 256^2, 181 angles, 256 bins: two groups of 8 through the one-group scratch)
    c = inputs.CONFIGS[2]
    ang1 = inputs.angles_uniform(c["Na"])
    vol1 = torch.from_numpy(inputs.volume_cfg2()).cuda()
    plan1 = tc.Plan(c["N"], c["Nd"], ang1, c["centre"])
    out1 = torch.empty((c["S"], c["Na"], c["Nd"]), dtype=torch.float32, device="cuda")
    plan1.radon_static(vol1, out1)                                   # before any other call on this plan: its own scratch does not exist yet
    out1c = torch.empty_like(out1)
    ref_buf = torch.empty_like(out1)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]                             # after the first call, so that one-time loading of kernel code is not counted
    plan1.radon_static(vol1, out1c)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "tc_radon_static allocated device memory"
    assert torch.equal(out1c, out1)
    ref1 = plan1.radon(vol1, out=ref_buf)                            # the existing path: only now does the plan allocate its scratch
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] < free0, "the plan's own scratch existed already: the check above proved nothing"
    assert rel_l2(out1.cpu().numpy(), ref1.cpu().numpy()) <= TOL_SAME_PATH
    assert rel_l2(out1[3].cpu().numpy(), nufft.radon_nufft(vol1[3].cpu().numpy(), ang1.astype(np.float64), c["Nd"], c["centre"])) < TOL_NUFFT

    # call 2, right after: a smaller geometry with a ragged group (11 slices of 64^2, 33 angles, 96 bins), so the shared array still
    # holds call 1's fine grid, half-plane and coefficients where this call does not write
    rng = np.random.default_rng(2)
    N2, Nd2, Na2, S2 = 64, 96, 33, 11
    ang2 = np.sort(rng.uniform(0, math.pi, Na2)).astype(np.float32)
    vol2 = torch.from_numpy(rng.random((S2, N2, N2)).astype(np.float32)).cuda()
    plan2 = tc.Plan(N2, Nd2, ang2, 47.25)
    out2 = torch.empty((S2, Na2, Nd2), dtype=torch.float32, device="cuda")
    plan2.radon_static(vol2, out2)
    ref2 = plan2.radon(vol2)
    torch.cuda.synchronize()
    assert rel_l2(out2.cpu().numpy(), ref2.cpu().numpy()) <= TOL_SAME_PATH
    assert rel_l2(out2[9].cpu().numpy(), nufft.radon_nufft(vol2[9].cpu().numpy(), ang2.astype(np.float64), Nd2, 47.25)) < TOL_NUFFT

    # and call 1 again gives call 1's result again (nothing of call 2 leaks)
    out1b = torch.empty_like(out1)
    plan1.radon_static(vol1, out1b)
    torch.cuda.synchronize()
    assert torch.equal(out1b, out1)
    plan1.close(); plan2.close()


def test_radon_static_refuses_sizes_beyond_the_static_scratch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2304_12934_b200 import binding as tc
    ang = (np.arange(8) * math.pi / 8).astype(np.float32)
    for n, nd, na in ((512, 512, 8), (256, 2048, 80)):               # n too large; n_angles * n_det = 163840 > 131072
        a = (np.arange(na) * math.pi / na).astype(np.float32)
        plan = tc.Plan(n, nd, a)
        vol = torch.zeros((1, n, n), dtype=torch.float32, device="cuda")
        out = torch.empty((1, na, nd), dtype=torch.float32, device="cuda")
        with pytest.raises(tc.TcError) as e:
            plan.radon_static(vol, out)
        assert e.value.status == tc.TC_EUNSUPPORTED and "static scratch" in str(e.value)
        plan.close()
    plan = tc.Plan(64, 64, ang)
    with pytest.raises(tc.TcError) as e:                             # host arrays: device pointers only
        plan.radon_static(np.zeros((1, 64, 64), np.float32), np.empty((1, 8, 64), np.float32))
    assert e.value.status == tc.TC_EINVAL
    plan.close()
