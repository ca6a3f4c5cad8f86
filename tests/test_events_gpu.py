"""kf_build_best_hit_events: several events built in one call ("concurrent events ... to fill the GPU")
give, per candidate, exactly what kf_build_best_hit gives for its event alone; one event is also checked against the
oracle through that equality (tests/test_score_gpu.py holds kf_build_best_hit to the oracle)."""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as O
from workloads import barrel_events as W

pytestmark = pytest.mark.gpu
NE, NP, EMAX = 40, 64, float(np.float32(1.2))


@pytest.fixture(scope="module")
def ctx():
    import paper_1705_02876_b200 as K
    c = K.KFContext(0)
    yield c
    c.close()


def _event(seed_shift, n_tracks, noise):
    """A build event with its own tracks and noise (the generator's event index moves both)."""
    cfg = W.get_config(4)
    fit = W.simulate_event(cfg, 100 + seed_shift, n_tracks)
    rng = np.random.default_rng(991 + seed_shift)
    layers = []
    for l in range(cfg.n_layers):
        r = float(cfg.radii[l])
        eta, phi = rng.uniform(-1.2, 1.2, noise), rng.uniform(-np.pi, np.pi, noise)
        npos = np.stack([r * np.cos(phi), r * np.sin(phi), r * np.sinh(eta)])
        pos = np.concatenate([fit.hpos[l].astype(np.float64), npos], axis=1).astype(np.float32)
        cov = np.concatenate([fit.hcov[l].astype(np.float64), W.hit_covariance(phi)], axis=1).astype(np.float32)
        layers.append((r, pos, cov))
    o3 = O.fit_tracks(fit.radius[:3], fit.x_over_X0[:3], fit.Bz, fit.mass, fit.par, fit.cov, fit.q, fit.hpos[:3], fit.hcov[:3], None)
    return fit, layers, o3["par"].astype(np.float32), O.pack_cov21(o3["cov"]).astype(np.float32), o3["chi2"], o3["nhits"]


@pytest.mark.parametrize("sizes", [[(700, 3000), (1, 50), (1200, 6000), (33, 0)], [(300, 1000)] * 32])
def test_events_in_one_call_equal_one_call_per_event(ctx, sizes):
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceCandidates, DeviceLayer
    evs = [_event(i, n, noise) for i, (n, noise) in enumerate(sizes)]
    fit0 = evs[0][0]
    geom = K.Geometry(fit0.radius, fit0.x_over_X0, fit0.Bz, fit0.mass)
    L0 = 3
    # per event
    want, pools = [], []
    for fit, layers, par, cov, chi2, nh in evs:
        dls = [DeviceLayer.from_numpy(p, c, NE, NP, EMAX, "cuda:0") for (_, p, c) in layers[L0:]]
        ctx.bin_layers([r for (r, _, _) in layers[L0:]], [(d.n_hits, d.pos, d.cov, d.bins) for d in dls])
        dc = DeviceCandidates.from_numpy(par, cov, fit.q, chi2, nh, "cuda:0")
        idx, c2 = dc.build(ctx, geom, L0, dls, 2, 30.0, True, None)
        torch.cuda.synchronize()
        want.append(dict(dc.results(), idx=idx.cpu().numpy()[:, :fit.n], c2=c2.cpu().numpy()[:, :fit.n]))
        pools.append(dls)
    # all events at once
    cat = lambda k, ax: np.concatenate([e[k] for e in evs], axis=ax)
    par = np.concatenate([e[2] for e in evs], axis=1); cov = np.concatenate([e[3] for e in evs], axis=1)
    q = np.concatenate([e[0].q for e in evs]); chi2 = np.concatenate([e[4] for e in evs]); nh = np.concatenate([e[5] for e in evs])
    first = np.concatenate([[0], np.cumsum([e[0].n for e in evs])])
    dc = DeviceCandidates.from_numpy(par, cov, q, chi2, nh, "cuda:0")
    m = 10 - L0
    idx = torch.full((m, dc.ld), -9, dtype=torch.int32, device="cuda:0")
    c2 = torch.zeros((m, dc.ld), dtype=torch.float32, device="cuda:0")
    ctx.build_best_hit_events(geom, L0, first, dc.n, dc.par, dc.cov, dc.q, dc.chi2, dc.nhits, dc.status,
                              [[(d.n_hits, d.pos, d.cov, d.bins) for d in dls] for dls in pools], 2, 30.0, True, idx, c2)
    torch.cuda.synchronize()
    got = dict(dc.results(), idx=idx.cpu().numpy(), c2=c2.cpu().numpy())
    for e, w in enumerate(want):
        lo, hi = int(first[e]), int(first[e + 1])
        for k in ("par", "cov", "idx", "c2"):
            assert np.array_equal(got[k][..., lo:hi], w[k], equal_nan=True), (e, k)
        for k in ("chi2", "nhits", "status"):
            assert np.array_equal(got[k][lo:hi], w[k]), (e, k)


@pytest.mark.parametrize("sizes,n_cand", [([(700, 3000), (1, 50), (1200, 6000), (33, 0)], 4), ([(200, 1000)] * 32, 3)])
def test_combinatorial_events_in_one_call_equal_one_call_per_event(ctx, sizes, n_cand):
    """kf_build_combinatorial_events: per seed exactly what kf_build_combinatorial gives for its event alone
    (tests/test_comb_gpu.py holds that call to the oracle)."""
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceCandidates, DeviceLayer
    evs = [_event(40 + i, n, noise) for i, (n, noise) in enumerate(sizes)]
    fit0 = evs[0][0]
    geom = K.Geometry(fit0.radius, fit0.x_over_X0, fit0.Bz, fit0.mass)
    L0 = 3
    want, pools = [], []
    for fit, layers, par, cov, chi2, nh in evs:
        dls = [DeviceLayer.from_numpy(p, c, NE, NP, EMAX, "cuda:0") for (_, p, c) in layers[L0:]]
        ctx.bin_layers([r for (r, _, _) in layers[L0:]], [(d.n_hits, d.pos, d.cov, d.bins) for d in dls])
        dc = DeviceCandidates.from_numpy(par, cov, fit.q, chi2, nh, "cuda:0")
        idx, nf = dc.build_combinatorial(ctx, geom, L0, dls, n_cand)
        torch.cuda.synchronize()
        want.append(dict(dc.results(), idx=idx.cpu().numpy()[:, :fit.n], nf=nf.cpu().numpy()[:fit.n]))
        pools.append(dls)
    par = np.concatenate([e[2] for e in evs], axis=1); cov = np.concatenate([e[3] for e in evs], axis=1)
    q = np.concatenate([e[0].q for e in evs]); chi2 = np.concatenate([e[4] for e in evs]); nh = np.concatenate([e[5] for e in evs])
    first = np.concatenate([[0], np.cumsum([e[0].n for e in evs])])
    dc = DeviceCandidates.from_numpy(par, cov, q, chi2, nh, "cuda:0")
    m = 10 - L0
    idx = torch.full((m, dc.ld), -9, dtype=torch.int32, device="cuda:0")
    nf = torch.zeros(dc.ld, dtype=torch.int32, device="cuda:0")
    ctx.build_combinatorial_events(geom, L0, first, dc.n, dc.par, dc.cov, dc.q, dc.chi2, dc.nhits, dc.status,
                                   [[(d.n_hits, d.pos, d.cov, d.bins) for d in dls] for dls in pools], 2, 30.0, n_cand,
                                   idx, nf)
    torch.cuda.synchronize()
    got = dict(dc.results(), idx=idx.cpu().numpy(), nf=nf.cpu().numpy())
    for e, w in enumerate(want):
        lo, hi = int(first[e]), int(first[e + 1])
        for k in ("par", "cov", "idx"):
            assert np.array_equal(got[k][..., lo:hi], w[k], equal_nan=True), (e, k)
        for k in ("chi2", "nhits", "status", "nf"):
            assert np.array_equal(got[k][lo:hi], w[k]), (e, k)
    assert (got["idx"][:, :int(first[-1])] >= 0).mean() > 0.5
    # argument errors as in the best-hit form
    with pytest.raises(K.KFError) as err:
        ctx.build_combinatorial_events(geom, L0, [0, dc.n - 1], dc.n, dc.par, dc.cov, dc.q, dc.chi2, dc.nhits, dc.status,
                                       [[(d.n_hits, d.pos, d.cov, d.bins) for d in pools[0]]], 2, 30.0, n_cand, idx, nf)
    assert err.value.code == -2


def test_events_argument_errors(ctx):
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceCandidates, DeviceLayer
    fit, layers, par, cov, chi2, nh = _event(0, 64, 100)
    geom = K.Geometry(fit.radius, fit.x_over_X0, fit.Bz, fit.mass)
    dls = [DeviceLayer.from_numpy(p, c, NE, NP, EMAX, "cuda:0") for (_, p, c) in layers[3:]]
    ctx.bin_layers([r for (r, _, _) in layers[3:]], [(d.n_hits, d.pos, d.cov, d.bins) for d in dls])
    dc = DeviceCandidates.from_numpy(par, cov, fit.q, chi2, nh, "cuda:0")
    idx = torch.zeros((7, dc.ld), dtype=torch.int32, device="cuda:0"); c2 = torch.zeros((7, dc.ld), dtype=torch.float32, device="cuda:0")
    pools = [[(d.n_hits, d.pos, d.cov, d.bins) for d in dls]]
    for first, code in (([0, 63], -2), ([1, 64], -2), ([0, 64], 0)):
        if code:
            with pytest.raises(K.KFError) as e:
                ctx.build_best_hit_events(geom, 3, first, dc.n, dc.par, dc.cov, dc.q, dc.chi2, dc.nhits, dc.status, pools, 2, 30.0, True, idx, c2)
            assert e.value.code == code
        else:
            ctx.build_best_hit_events(geom, 3, first, dc.n, dc.par, dc.cov, dc.q, dc.chi2, dc.nhits, dc.status, pools, 2, 30.0, True, idx, c2)
    with pytest.raises(K.KFError) as e:
        ctx.build_best_hit_events(geom, 3, list(range(0, 34)), 33, dc.par, dc.cov, dc.q, dc.chi2, dc.nhits, dc.status, pools * 33, 2, 30.0, True, idx, c2)
    assert e.value.code == -4
    torch.cuda.synchronize()


@pytest.mark.parametrize("n_tracks,noise,pinned", [(1000, 5000, True), (33, 100, False), (20000, 100000, True)])
def test_build_host_path_equals_device_path(ctx, n_tracks, noise, pinned):
    """kf_build_best_hit_host (host buffers in, host buffers out, pools copied layer by layer on a second stream
    while the previous layer is binned and scored) == kf_bin_layers + kf_build_best_hit on device buffers."""
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceCandidates, DeviceLayer, padded_ld
    fit, layers, par, cov, chi2, nh = _event(7, n_tracks, noise)
    geom = K.Geometry(fit.radius, fit.x_over_X0, fit.Bz, fit.mass)
    L0 = 3
    dls = [DeviceLayer.from_numpy(p, c, NE, NP, EMAX, "cuda:0") for (_, p, c) in layers[L0:]]
    ctx.bin_layers([r for (r, _, _) in layers[L0:]], [(d.n_hits, d.pos, d.cov, d.bins) for d in dls])
    dc = DeviceCandidates.from_numpy(par, cov, fit.q, chi2, nh, "cuda:0")
    idx, c2 = dc.build(ctx, geom, L0, dls, 2, 30.0, True, None)
    torch.cuda.synchronize()
    want = dict(dc.results(), idx=idx.cpu().numpy()[:, :fit.n], c2=c2.cpu().numpy()[:, :fit.n])
    hc = DeviceCandidates.from_numpy(par, cov, fit.q, chi2, nh, "cpu")
    m = 10 - L0
    mk = lambda shape, dt: torch.zeros(shape, dtype=dt, pin_memory=pinned)
    hidx, hc2 = mk((m, hc.ld), torch.int32), mk((m, hc.ld), torch.float32)
    pools = []
    for (_, p, c) in layers[L0:]:
        H = p.shape[1]; ld = padded_ld(H)
        tp, tc = mk((3, ld), torch.float32), mk((6, ld), torch.float32)
        tp[:, :H] = torch.from_numpy(p); tc[:, :H] = torch.from_numpy(c)
        pools.append((H, tp, tc))
    for rep in range(2):                       # twice: the second call reuses the staging buffers
        hc = DeviceCandidates.from_numpy(par, cov, fit.q, chi2, nh, "cpu")
        ctx.build_best_hit_host(geom, L0, hc.n, hc.par, hc.cov, hc.q, hc.chi2, hc.nhits, hc.status, pools, NE, NP, EMAX,
                                2, 30.0, True, hidx, hc2)
        got = dict(hc.results(), idx=hidx.numpy()[:, :fit.n], c2=hc2.numpy()[:, :fit.n])
        assert np.array_equal(got["idx"], want["idx"])
        assert np.array_equal(got["nhits"], want["nhits"]) and np.array_equal(got["status"], want["status"])
        # same arithmetic in differently fused kernels: equal to fp32 rounding
        np.testing.assert_allclose(got["c2"], want["c2"], rtol=1e-5, atol=1e-6)
        np.testing.assert_allclose(got["chi2"], want["chi2"], rtol=1e-5, atol=1e-5)
        np.testing.assert_allclose(got["par"], want["par"], rtol=2e-6, atol=2e-6)
        scale = np.abs(want["cov"]).max(axis=0)
        assert np.max(np.abs(got["cov"] - want["cov"]) / scale) < 2e-5
