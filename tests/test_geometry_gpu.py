"""GPU parity of the geometry options (reading A20: path-length material, finite barrels) in
kf_fit_tracks and kf_fit_tracks_refit against the oracle.  The builder and the combinatorial builder are
covered with the same options in test_score_gpu.py / test_comb_gpu.py.

A crossing within fp32 rounding of the barrel end may fall on either side in the two precisions; such tracks
(|z'| within 2e-5 relative of the half length on any layer, by the ORACLE's own crossing) are exempt, counted
and bounded; every other track must agree in its OUTSIDE bit, hits used and state."""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as O
from tests.parity import compare_fit
from workloads import barrel_events as W

pytestmark = pytest.mark.gpu
OUT = np.uint32(O.OUTSIDE)
EDGE = 2e-5


@pytest.fixture(scope="module")
def ctx():
    import paper_1705_02876_b200 as K
    c = K.KFContext(0)
    yield c
    c.close()


def _oracle(b, hl, model):
    with O.geometry_options(model, hl):
        return O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask,
                            nthreads=8, want_trace=True)


def _near_edge(o, hl):
    zp = np.abs(o["trace"][:, :, 2])                     # [n][L] oracle crossing z' (0 where not propagated)
    return ((zp > 0) & (np.abs(zp - hl[None, :]) <= EDGE * hl[None, :])).any(axis=1)


def _compare_fit_with_outside(g, o, hl, r_last, max_div=2e-3):
    edge = _near_edge(o, hl)
    assert edge.mean() < 5e-3
    keep = ~edge
    assert np.array_equal(g["status"][keep] & OUT, o["status"][keep] & OUT)
    gg = {k: (g[k][:, keep] if k in ("par", "cov") else g[k][keep]) for k in ("par", "cov", "chi2", "nhits", "status")}
    oo = dict(par=o["par"][:, keep], cov=o["cov"][keep], chi2=o["chi2"][keep], nhits=o["nhits"][keep],
              status=o["status"][keep] & ~OUT)
    gg["status"] = gg["status"] & ~OUT                   # a track cut short by the barrel end is a valid fit
    return compare_fit(gg, oo, r_last, max_diverged_frac=max_div)


@pytest.mark.parametrize("model", [0, 1])
def test_fit_hits_beyond_the_barrel_end_are_skipped(ctx, model):
    """Config 3 generated WITHOUT acceptance (hits on every layer, |eta| up to 1.5), fitted with 60 cm barrels:
    most tracks lose their outer layers."""
    from paper_1705_02876_b200.buffers import DeviceFit
    b = W.simulate_event(W.get_config(3), 1, n_tracks=30000)
    hl = np.full(b.n_layers, 60.0, dtype=np.float32)
    b.half_length, b.material_model = hl, model
    d = DeviceFit.from_batch(b, "cuda:0")
    d.fit(ctx)
    torch.cuda.synchronize()
    g, o = d.results(), _oracle(b, hl.astype(np.float64), model)
    assert 0.2 < ((o["status"] & OUT) != 0).mean() < 0.95
    res = _compare_fit_with_outside(g, o, hl.astype(np.float64), float(b.radius[-1]))
    print(f"material model {model}: {res}")


def test_fit_generated_with_the_same_geometry(ctx):
    """Generator and fitter share the options (hits only inside 30 cm barrels, scattering with t / cos psi),
    half lengths different per layer on the fitter's side (longer outside, as real barrels are)."""
    from paper_1705_02876_b200.buffers import DeviceFit
    cfg = W.get_config(1)
    cfg.material_model, cfg.half_length_cm = 1, 30.0
    b = W.simulate_event(cfg, 6, n_tracks=20000)
    hl = np.linspace(30.0, 34.5, b.n_layers).astype(np.float32)
    b.half_length = hl
    d = DeviceFit.from_batch(b, "cuda:0")
    d.fit(ctx)
    torch.cuda.synchronize()
    g, o = d.results(), _oracle(b, hl.astype(np.float64), 1)
    res = _compare_fit_with_outside(g, o, hl.astype(np.float64), float(b.radius[-1]))
    print(res)
    # and the model matters: the flat model on the same data gives a different answer at high |eta|
    b.material_model = 0
    d0 = DeviceFit.from_batch(b, "cuda:0")
    d0.fit(ctx)
    torch.cuda.synchronize()
    g0 = d0.results()
    ok = (g["status"] == 0) & (g0["status"] == 0)
    assert np.median(np.abs(g0["cov"][20, ok] / g["cov"][20, ok] - 1.0)) > 1e-3     # C_pzpz


def test_refit_with_geometry_options(ctx):
    from paper_1705_02876_b200.buffers import DeviceFit
    b = W.simulate_event(W.get_config(3), 2, n_tracks=20000)
    hl = np.full(b.n_layers, 60.0, dtype=np.float32)
    b.half_length, b.material_model = hl, 1
    d = DeviceFit.from_batch(b, "cuda:0")
    d.fit_refit(ctx)
    torch.cuda.synchronize()
    with O.geometry_options(1, hl.astype(np.float64)):
        o = O.fit_refit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask,
                                want_trace=True)
    edge = _near_edge(dict(trace=o["trace_fwd"]), hl.astype(np.float64))
    keep = ~edge & (o["nhits"] >= 3)
    assert edge.mean() < 5e-3
    g, sg = d.results(), d.refit_results()
    assert np.array_equal(g["status"][keep] & OUT, o["status"][keep] & OUT)
    assert np.array_equal(g["nhits"][keep], o["nhits"][keep])
    # the inward pass runs over layers the forward pass used: it stays inside the barrel
    assert np.array_equal(sg["status"][keep], o["rstatus"][keep])
    ndf = np.maximum(2 * o["nhits"] - 5, 1)
    excl = (o["status"] & ~OUT) | o["rstatus"] | ((o["chi2"] > ndf + 9 * np.sqrt(2.0 * ndf)).astype(np.uint32) << 5)
    so = dict(par=o["rpar"][:, keep], cov=o["rcov"][keep], chi2=o["rchi2"][keep], nhits=o["nhits"][keep], status=excl[keep])
    gs = dict(par=sg["par"][:, keep], cov=sg["cov"][:, keep], chi2=sg["chi2"][keep], nhits=o["nhits"][keep], status=excl[keep])
    res = compare_fit(gs, so, float(b.radius[-1]), max_diverged_frac=5e-3)
    print("smoothed with options:", res)


def test_unbounded_options_equal_the_plain_geometry(ctx):
    """half_length = +inf and model 0 select the kernel with the options compiled in; it must agree with the
    specialised one to rounding (same functions, different FMA contraction)."""
    from paper_1705_02876_b200.buffers import DeviceFit
    b = W.make_fit_batch(1)
    d0 = DeviceFit.from_batch(b, "cuda:0")
    d0.fit(ctx)
    b.half_length = np.full(b.n_layers, 1e30, dtype=np.float32)     # finite: takes the option kernel
    d1 = DeviceFit.from_batch(b, "cuda:0")
    d1.fit(ctx)
    torch.cuda.synchronize()
    r0, r1 = d0.results(), d1.results()
    assert np.array_equal(r0["status"], r1["status"]) and np.array_equal(r0["nhits"], r1["nhits"])
    np.testing.assert_allclose(r1["chi2"], r0["chi2"], rtol=3e-4, atol=1e-5)     # (each is within 1e-3 of the oracle)
    np.testing.assert_allclose(r1["par"], r0["par"], rtol=3e-5, atol=3e-5)       # (tolerance to the oracle: 1e-4)


def test_geometry_option_errors(ctx):
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceFit
    b = W.simulate_event(W.get_config(1), 0, n_tracks=64)
    d = DeviceFit.from_batch(b, "cuda:0")
    for bad in (dict(material_model=2), dict(material_model=-1),
                dict(half_length_cm=np.zeros(b.n_layers, np.float32)),
                dict(half_length_cm=np.full(b.n_layers, np.nan, np.float32))):
        d.geom = K.Geometry(b.radius, b.x_over_X0, b.Bz, b.mass, **bad)
        with pytest.raises(K.KFError) as e:
            d.fit(ctx)
        assert e.value.code == -4
    with pytest.raises(ValueError):
        K.Geometry(b.radius, b.x_over_X0, b.Bz, b.mass, np.ones(3, np.float32))._c()
    d.geom = K.Geometry(b.radius, b.x_over_X0, b.Bz, b.mass, np.full(b.n_layers, np.inf, np.float32), 1)
    d.fit(ctx)                                                          # +inf half lengths are allowed
    torch.cuda.synchronize()
    assert np.all(d.results()["status"] == 0)
