"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the oracle on the same seeded
inputs.  Tolerances are north_star's: rel. L2 <= 1e-4 vs the oracle NUFFT, <= 1e-3 vs the direct DFT,
adjoint mismatch <= 1e-5 (inner products in fp64), MBIR iterates <= 1e-3 after 10 iterations."""
import math
import numpy as np
import pytest
from conftest import rel_l2

pytestmark = pytest.mark.gpu

TOL_NUFFT, TOL_DIRECT, TOL_ADJ, TOL_MBIR = 1e-4, 1e-3, 1e-5, 1e-3
P, SIG, C = 1.2, 1 / 0.7, 1e-4


@pytest.fixture(scope="module")
def tc():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2304_12934_b200 import binding
    return binding


def _cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _np(t):
    import torch
    torch.cuda.synchronize()
    return t.cpu().numpy()


def _pair(tc, vol, y, ang, nd, centre, **kw):
    plan = tc.Plan(vol.shape[-1], nd, ang, centre, **kw)
    s = _np(plan.radon(_cuda(vol))); b = _np(plan.backproject(_cuda(y)))
    plan.close()
    return s, b


def _adj_mismatch(vol, y, s, b):
    lhs = np.sum(s.astype(np.float64) * y); rhs = np.sum(vol.astype(np.float64) * b)
    return abs(lhs - rhs) / max(abs(lhs), abs(rhs))


def test_config1_forward_adjoint_vs_oracle_and_direct(tc):
    from paper_2304_12934_b200 import inputs
    from oracle import nufft, direct
    c = inputs.CONFIGS[1]
    ang = inputs.angles_uniform(c["Na"]); a64 = ang.astype(np.float64)
    vol = inputs.volume_cfg1()
    y = nufft.radon_nufft(vol, a64, c["Nd"], c["centre"]).astype(np.float32)
    s, b = _pair(tc, vol, y, ang, c["Nd"], c["centre"])
    assert rel_l2(s, y) < TOL_NUFFT
    assert rel_l2(b, nufft.backproject_nufft(y, a64, c["N"], c["centre"])) < TOL_NUFFT
    assert rel_l2(s, direct.radon_direct(vol, a64, c["Nd"], c["centre"])) < TOL_DIRECT
    assert rel_l2(b, direct.backproject_direct(y, a64, c["N"], c["centre"])) < TOL_DIRECT
    rng = np.random.default_rng(11)
    yr = rng.standard_normal(y.shape).astype(np.float32)
    s2, b2 = _pair(tc, vol, yr, ang, c["Nd"], c["centre"])
    assert _adj_mismatch(vol, yr, s2, b2) < TOL_ADJ


def test_config2_forward_adjoint(tc):
    from paper_2304_12934_b200 import inputs
    from oracle import nufft, direct
    c = inputs.CONFIGS[2]
    ang = inputs.angles_uniform(c["Na"]); a64 = ang.astype(np.float64)
    vol = inputs.volume_cfg2()
    rng = np.random.default_rng(12)
    y = rng.standard_normal((c["S"], c["Na"], c["Nd"])).astype(np.float32)
    s, b = _pair(tc, vol, y, ang, c["Nd"], c["centre"])
    assert rel_l2(s, nufft.radon_nufft(vol, a64, c["Nd"], c["centre"])) < TOL_NUFFT
    assert rel_l2(b, nufft.backproject_nufft(y, a64, c["N"], c["centre"])) < TOL_NUFFT
    assert rel_l2(s[3], direct.radon_direct(vol[3], a64, c["Nd"], c["centre"])) < TOL_DIRECT
    assert rel_l2(b[5], direct.backproject_direct(y[5], a64, c["N"], c["centre"])) < TOL_DIRECT
    assert _adj_mismatch(vol, y, s, b) < TOL_ADJ


@pytest.mark.parametrize("S,N,Nd,Na,centre", [
    (3, 64, 64, 7, 35.5),        # ragged group (3 of 8 slices), odd slice count
    (9, 160, 160, 33, 83.25),    # radix-5 FFT lengths (G = 320, Nd = 160), two groups with a ragged tail
    (2, 128, 256, 20, 130.0),    # n_det = 2 n  (one fine-grid cell per radial mode)
    (2, 128, 64, 20, 30.0),      # n_det = n / 2 (four cells per mode)
    (17, 32, 32, 5, 16.0),       # smallest supported image, three groups
])
def test_shapes_and_ragged_tails(tc, S, N, Nd, Na, centre):
    from oracle import nufft
    rng = np.random.default_rng(S * 1000 + N)
    ang = (np.arange(Na) * math.pi / Na).astype(np.float32)
    vol = rng.random((S, N, N)).astype(np.float32); y = rng.standard_normal((S, Na, Nd)).astype(np.float32)
    s, b = _pair(tc, vol, y, ang, Nd, centre)
    assert rel_l2(s, nufft.radon_nufft(vol, ang.astype(np.float64), Nd, centre)) < TOL_NUFFT
    assert rel_l2(b, nufft.backproject_nufft(y, ang.astype(np.float64), N, centre)) < TOL_NUFFT
    assert _adj_mismatch(vol, y, s, b) < TOL_ADJ


def test_arbitrary_angles_unsorted_negative_and_beyond_pi(tc):
    from oracle import nufft
    rng = np.random.default_rng(13)
    ang = np.concatenate([rng.uniform(-2 * math.pi, 3 * math.pi, 21), [0.0, math.pi / 2, math.pi, -math.pi / 2, math.pi / 4]]).astype(np.float32)
    vol = rng.random((2, 64, 64)).astype(np.float32); y = rng.standard_normal((2, ang.size, 64)).astype(np.float32)
    s, b = _pair(tc, vol, y, ang, 64, 31.0)
    assert rel_l2(s, nufft.radon_nufft(vol, ang.astype(np.float64), 64, 31.0)) < TOL_NUFFT
    assert rel_l2(b, nufft.backproject_nufft(y, ang.astype(np.float64), 64, 31.0)) < TOL_NUFFT


def test_degenerate_inputs(tc):
    # zero volume -> zero sinogram; one angle; default centre (< 0 -> n_det / 2); delta input (worked example shape)
    from oracle import nufft, direct
    ang = np.array([math.pi / 5], dtype=np.float32)
    plan = tc.Plan(32, 32, ang)            # centre defaults to 16
    z = _np(plan.radon(_cuda(np.zeros((1, 32, 32), np.float32))))
    assert np.all(z == 0)
    f = np.zeros((1, 32, 32), np.float32); f[0, 17, 14] = 1.0
    s = _np(plan.radon(_cuda(f)))
    assert rel_l2(s, direct.radon_direct(f, ang.astype(np.float64), 32, 16.0)) < TOL_DIRECT
    assert rel_l2(s, nufft.radon_nufft(f, ang.astype(np.float64), 32, 16.0)) < TOL_NUFFT
    plan.close()
    s1 = _np(tc.radon1(_cuda(f), ang, 32, 16.0))
    assert np.array_equal(s1, s)


def test_host_pointer_streaming_matches_in_core(tc):
    # S1: host arrays go through the slab scheduler (forced 8-slice slabs -> 5 slabs with a ragged last one)
    import torch
    rng = np.random.default_rng(14)
    S, N, Na = 35, 64, 16
    ang = (np.arange(Na) * math.pi / Na).astype(np.float32)
    vol = rng.random((S, N, N)).astype(np.float32); y = rng.standard_normal((S, Na, N)).astype(np.float32)
    s_dev, b_dev = _pair(tc, vol, y, ang, N, 33.0)
    plan = tc.Plan(N, N, ang, 33.0, max_slab_slices=8)
    s_host = plan.radon(vol); b_host = plan.backproject(y)                    # pageable numpy
    st = plan.sched_stats()
    assert st["n_slabs"] == 5 and st["h2d_bytes"] == y.nbytes and st["d2h_bytes"] == vol.nbytes
    pv = torch.from_numpy(vol).pin_memory()
    s_pin = plan.radon(pv).numpy()                                            # pinned torch
    plan.close()
    assert rel_l2(s_host, s_dev) <= 1e-6 and rel_l2(b_host, b_dev) <= 1e-6 and rel_l2(s_pin, s_dev) <= 1e-6


def test_prior_kernels_vs_oracle(tc):
    from oracle import prior
    rng = np.random.default_rng(15)
    for shape in ((1, 32, 32), (5, 64, 96)[:1] + (40, 40), (3, 33, 33)):
        v = (rng.standard_normal(shape) * rng.choice([0.01, 1.0, 30.0])).astype(np.float32)
        v[0, :4, :4] = 0.25                                                    # flat patch: h'(0) = 0 exactly
        for pp, ss, cc in ((P, SIG, C), (2.0, 1.0, 1.0)):                      # p = 2: the exponent 2 - p is 0 (u^0 at u = 0)
            val, g = tc.prior_eval(_cuda(v), tc.prior_params(pp, ss, cc))
            assert abs(val - prior.H(v, pp, ss, cc)) <= 2e-6 * prior.H(v, pp, ss, cc)
            assert rel_l2(_np(g), prior.gradH(v, pp, ss, cc)) < 1e-5
    val, g = tc.prior_eval(_cuda(np.full((2, 32, 32), 0.7, np.float32)), tc.prior_params(P, SIG, C))
    assert val == 0.0 and np.all(_np(g) == 0.0)


def _mbir_case(tc, vol_truth, ang, nd, centre, iters, noise_seed=None):
    from oracle import nufft, mbir
    a64 = ang.astype(np.float64)
    n = vol_truth.shape[-1]
    b = nufft.radon_nufft(vol_truth, a64, nd, centre)
    if noise_seed is not None:
        b = b + 0.01 * np.random.default_rng(noise_seed).standard_normal(b.shape)
    b = b.astype(np.float32)
    L, lam_hat = mbir.lipschitz(n, a64, nd, centre, P, SIG, C, 1.0)
    plan = tc.Plan(n, nd, ang, centre)
    assert abs(plan.power_iteration(10) - lam_hat) < 1e-4 * lam_hat
    x, log = plan.mbir(_cuda(b), tc.prior_params(P, SIG, C, 1.0, L), iters)
    x = _np(x); plan.close()
    xo, logo, its = mbir.mbir(b, a64, n, centre, P, SIG, C, 1.0, L, iters, keep_iterates=True)
    acc_g, acc_o = [l["accepted"] for l in log], [l["accepted"] for l in logo]
    if acc_g != acc_o:                      # decision parity: only a tie may differ; replay the oracle with the GPU's decision
        k = next(i for i in range(iters) if acc_g[i] != acc_o[i])
        assert abs(logo[k]["margin"]) < 1e-4, (k, logo[k])
        xo, logo = mbir.mbir(b, a64, n, centre, P, SIG, C, 1.0, L, iters, forced={i: acc_g[i] for i in range(iters)})
    assert rel_l2(x, xo) < TOL_MBIR
    for lg, lo in zip(log, logo):
        assert abs(lg["F"] - lo["F"]) < 1e-4 * abs(lo["F"])
    return x, log


def test_mbir_config1_iterates(tc):
    from paper_2304_12934_b200 import inputs
    c = inputs.CONFIGS[1]
    x5, log5 = _mbir_case(tc, inputs.volume_cfg1(), inputs.angles_uniform(c["Na"]), c["Nd"], c["centre"], 5)
    x10, log10 = _mbir_case(tc, inputs.volume_cfg1(), inputs.angles_uniform(c["Na"]), c["Nd"], c["centre"], 10)
    F = [l["F"] for l in log10]
    assert all(F[i + 1] <= F[i] for i in range(len(F) - 1))


def test_mbir_nonneg_constraint_vs_oracle(tc):
    # the candidate projected on f >= 0 (A z recomputed, not carried by linearity); in core and streamed
    from paper_2304_12934_b200 import inputs
    from oracle import nufft, mbir
    S, n, na = 10, 64, 24
    ang = inputs.angles_uniform(na); a64 = ang.astype(np.float64)
    vol = inputs.volume_cfg2(S=S, n=n)
    # truth with a negative background, so that the unconstrained iterates go negative and the projection acts
    b = (nufft.radon_nufft(vol - 0.25, a64, n, 32.0) + 0.05 * np.random.default_rng(34).standard_normal((S, na, n))).astype(np.float32)
    L, _ = mbir.lipschitz(n, a64, n, 32.0, P, SIG, C, 1.0)
    pr = tc.prior_params(P, SIG, C, 1.0, L, nonneg=True)
    xo, logo = mbir.mbir(b, a64, n, 32.0, P, SIG, C, 1.0, L, 8, nonneg=True)
    xu, _ = mbir.mbir(b, a64, n, 32.0, P, SIG, C, 1.0, L, 8)
    assert xu.min() < -1e-3 and xo.min() >= 0.0                                # the constraint acts on this noisy data
    for kw in ({}, {"max_slab_slices": 8}):
        plan = tc.Plan(n, n, ang, 32.0, **kw)
        x, log = plan.mbir(b if kw else _cuda(b), pr, 8)
        x = x if kw else _np(x)
        plan.close()
        assert x.min() >= 0.0 and rel_l2(x, xo) < TOL_MBIR
        assert [l["accepted"] for l in log] == [l["accepted"] for l in logo]
        for lg, lo in zip(log, logo):
            assert abs(lg["F"] - lo["F"]) < 1e-4 * abs(lo["F"])


def test_mbir_gradient_restart_vs_oracle(tc):
    # gradient restart test.  Quadratic prior (p = 2) so that restarts occur within 30 iterations; the decision
    # is the sign of <g, z - x>, compared where it is not a tie (|dot| above the float32 noise of the inner product)
    from oracle import nufft, mbir
    n, na = 32, 16
    ang = (np.arange(na) * math.pi / na).astype(np.float32); a64 = ang.astype(np.float64)
    rng = np.random.default_rng(35)
    truth = np.zeros((2, n, n)); truth[:, 10:22, 8:20] = 1.0; truth[1, 14:18, 12:26] += 0.5
    b = (nufft.radon_nufft(truth, a64, n, 16.0) + 0.01 * rng.standard_normal((2, na, n))).astype(np.float32)
    p, sig, c, lam = 2.0, 1.0, 1.0, 200.0
    L, _ = mbir.lipschitz(n, a64, n, 16.0, p, sig, c, lam)
    xo, logo = mbir.mbir(b, a64, n, 16.0, p, sig, c, lam, L, 30, grad_restart=True)
    assert sum(l["restarted"] for l in logo) >= 1
    plan = tc.Plan(n, n, ang, 16.0)
    x, log = plan.mbir(_cuda(b), tc.prior_params(p, sig, c, lam, L, grad_restart=True), 30)
    x = _np(x); plan.close()
    scale = max(abs(l["dot"]) for l in logo)
    for lg, lo in zip(log, logo):
        assert abs(lg["dot"] - lo["dot"]) <= 1e-3 * scale
        if abs(lo["dot"]) > 2e-3 * scale:
            assert lg["restarted"] == lo["restarted"] and lg["accepted"] == lo["accepted"]
    if [l["restarted"] for l in log] == [l["restarted"] for l in logo]:
        assert rel_l2(x, xo) < TOL_MBIR
        for lg, lo in zip(log, logo):
            assert abs(lg["F"] - lo["F"]) < 1e-4 * abs(lo["F"])


def test_mbir_multislice_with_noise(tc):
    # 11 slices (two groups, ragged) so the z-coupling of the 26-neighbour prior crosses a group boundary
    from paper_2304_12934_b200 import inputs
    vol = inputs.volume_cfg2(S=11, n=64)
    _mbir_case(tc, vol, inputs.angles_uniform(24), 64, 32.0, 10, noise_seed=16)


def test_mbir_host_pointers_and_default_L(tc):
    from paper_2304_12934_b200 import inputs
    from oracle import nufft
    ang = inputs.angles_uniform(24)
    vol = inputs.volume_cfg2(S=2, n=64)
    b = nufft.radon_nufft(vol, ang.astype(np.float64), 64, 32.0).astype(np.float32)
    plan = tc.Plan(64, 64, ang, 32.0)
    xh, logh = plan.mbir(b, tc.prior_params(P, SIG, C, 1.0, 0.0), 4)          # host in/out, L estimated by the library
    xd, logd = plan.mbir(_cuda(b), tc.prior_params(P, SIG, C, 1.0, 0.0), 4)
    plan.close()
    assert np.array_equal(xh, _np(xd)) and [l["F"] for l in logh] == [l["F"] for l in logd]
    with pytest.raises(tc.TcError):
        plan2 = tc.Plan(64, 64, ang, 32.0)
        plan2.mbir(_cuda(b), tc.prior_params(0.9, SIG, C), 1)                 # p outside (1, 2]


def test_full_size_config4_geometry_sampled(tc):
    # BASELINE config 4 geometry (2048^2, 1024 angles, centre 1027.5) in the launch configuration bench.py times,
    # 8 slices (one group; groups are independent CTAs).  Slice 5: full oracle NUFFT; two angles and a few pixels
    # against the direct DFT.
    from paper_2304_12934_b200 import inputs
    from oracle import nufft, direct
    c = inputs.CONFIGS[4]
    ang = inputs.angles_uniform(c["Na"]); a64 = ang.astype(np.float64)
    vol = inputs.volume_fibres(8, c["N"], c["seed"], n_fibres=600)
    plan = tc.Plan(c["N"], c["Nd"], ang, c["centre"])
    s = _np(plan.radon(_cuda(vol)))
    so = nufft.radon_nufft(vol[5], a64, c["Nd"], c["centre"])
    assert rel_l2(s[5], so) < TOL_NUFFT
    sel = [137, 700]
    assert rel_l2(s[5][sel], direct.radon_direct(vol[5], a64[sel], c["Nd"], c["centre"])) < TOL_DIRECT
    y = so.astype(np.float32)[None].repeat(8, axis=0); y[2] *= 0.5
    b = _np(plan.backproject(_cuda(y)))
    plan.close()
    bo = nufft.backproject_nufft(y[5], a64, c["N"], c["centre"])
    assert rel_l2(b[5], bo) < TOL_NUFFT and rel_l2(b[2], 0.5 * bo) < TOL_NUFFT
    rng = np.random.default_rng(17)
    yr = rng.standard_normal((8, c["Na"], c["Nd"])).astype(np.float32)
    plan = tc.Plan(c["N"], c["Nd"], ang, c["centre"])
    br = _np(plan.backproject(_cuda(yr))); plan.close()
    assert _adj_mismatch(vol, yr, s, br) < TOL_ADJ


def test_mbir_out_of_core_streaming_matches_in_core_and_oracle(tc):
    # S1 + M1-M5: host-resident sinogram and volume, slab size forced to 8 slices -> 3 slabs (8, 8, 3) with z-halos;
    # the 26-neighbour prior couples the slabs, so a wrong halo shows up in both the iterate and F
    from paper_2304_12934_b200 import inputs
    from oracle import nufft, mbir
    S, n, na = 19, 64, 24
    ang = inputs.angles_uniform(na); a64 = ang.astype(np.float64)
    vol = inputs.volume_cfg2(S=S, n=n)
    b = (nufft.radon_nufft(vol, a64, n, 32.0) + 0.01 * np.random.default_rng(18).standard_normal((S, na, n))).astype(np.float32)
    L, _ = mbir.lipschitz(n, a64, n, 32.0, P, SIG, C, 1.0)
    pr = tc.prior_params(P, SIG, C, 1.0, L)
    plan = tc.Plan(n, n, ang, 32.0)
    x_in, log_in = plan.mbir(b, pr, 6)                                        # host pointers, fits: in-core
    assert plan.sched_stats()["n_slabs"] == 0
    plan.close()
    plan = tc.Plan(n, n, ang, 32.0, max_slab_slices=8)
    x_st, log_st = plan.mbir(b, pr, 6)                                        # forced streaming
    st = plan.sched_stats()
    plan.close()
    assert st["n_slabs"] == 3 and st["h2d_bytes"] > 0 and st["d2h_bytes"] == 6 * x_st.nbytes
    # the streamed loop recomputes A y, the in-core loop carries it by linearity: equal up to float32 rounding
    assert rel_l2(x_st, x_in) <= 1e-5
    assert [l["accepted"] for l in log_st] == [l["accepted"] for l in log_in]
    for ls, li in zip(log_st, log_in):
        assert abs(ls["F"] - li["F"]) <= 1e-6 * abs(li["F"])
    xo, logo = mbir.mbir(b, a64, n, 32.0, P, SIG, C, 1.0, L, 6)
    assert rel_l2(x_st, xo) < TOL_MBIR
    F = [l["F"] for l in log_st]
    assert all(F[i + 1] <= F[i] for i in range(len(F) - 1))


def test_full_size_config3_and_config5_geometry_sampled(tc):
    # BASELINE configs 3 (1024^2, 128 angles, porous cylinder + Poisson noise) and 5 (2560^2 = 2^9 * 5, 1313 angles) in the launch
    # configuration the library uses for them (compile-time pass lists, radix-5 last pass at 2560): 8 slices, one slice against the
    # full oracle NUFFT, a few angles against the direct DFT, adjoint identity on all 8.
    from paper_2304_12934_b200 import inputs
    from oracle import nufft, direct
    for cfg, sel in ((3, [5, 77]), (5, [611])):
        c = inputs.CONFIGS[cfg]
        ang = inputs.angles_uniform(c["Na"]); a64 = ang.astype(np.float64)
        vol = inputs.volume_porous(8, c["N"], c["seed"]) if cfg == 3 else inputs.volume_fibres(8, c["N"], c["seed"], n_fibres=400)
        plan = tc.Plan(c["N"], c["Nd"], ang, c["centre"])
        s = _np(plan.radon(_cuda(vol)))
        so = nufft.radon_nufft(vol[3], a64, c["Nd"], c["centre"])
        assert rel_l2(s[3], so) < TOL_NUFFT
        assert rel_l2(s[3][sel], direct.radon_direct(vol[3], a64[sel], c["Nd"], c["centre"])) < TOL_DIRECT
        y = inputs.poisson_sinogram(s, seed=19) if cfg == 3 else np.random.default_rng(20).standard_normal(s.shape).astype(np.float32)
        b = _np(plan.backproject(_cuda(y)))
        plan.close()
        assert rel_l2(b[3], nufft.backproject_nufft(y[3], a64, c["N"], c["centre"])) < TOL_NUFFT
        assert _adj_mismatch(vol, y, s, b) < TOL_ADJ


def test_fbp_vs_oracle(tc):
    # tc_fbp = the adjoint with ramp-weighted radial modes.  Against the oracle's NUFFT form and its definition,
    # both filters, a ragged group and host pointers; and FBP(A f) ~ f on config 1's phantom.
    from paper_2304_12934_b200 import inputs
    from oracle import fbp
    rng = np.random.default_rng(32)
    S, n, nd, na, centre = 3, 64, 128, 40, 65.25
    ang = inputs.angles_uniform(na); a64 = ang.astype(np.float64)
    y = rng.standard_normal((S, na, nd)).astype(np.float32)
    plan = tc.Plan(n, nd, ang, centre)
    for w in ("ramp", "hann"):
        f = _np(plan.fbp(_cuda(y), w))
        assert rel_l2(f, fbp.fbp_nufft(y, a64, n, centre, w)) < TOL_NUFFT
        assert rel_l2(f[1], fbp.fbp_direct(y[1], a64, n, centre, w)) < TOL_DIRECT
    assert rel_l2(plan.fbp(y, "ramp"), _np(plan.fbp(_cuda(y), "ramp"))) <= 1e-6        # host pointers: slab scheduler
    with pytest.raises(tc.TcError):
        tc._check(tc.lib.tc_fbp(plan._h, tc._ptr(y), S, 7, tc._ptr(np.empty((S, n, n), np.float32)), None))
    plan.close()
    c = inputs.CONFIGS[1]
    vol = inputs.volume_cfg1()
    ang = inputs.angles_uniform(180)
    plan = tc.Plan(c["N"], 256, ang, 128.0)
    rec = _np(plan.fbp(plan.radon(_cuda(vol))))
    plan.close()
    assert rel_l2(rec, vol) < 0.15                                   # sharp-edged ellipses, band-limited reconstruction
