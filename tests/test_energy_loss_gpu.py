"""GPU parity of the energy-loss option (reading A21) in kf_fit_tracks, kf_fit_tracks_refit and
kf_fit_tracks_indexed against the oracle, alone and together with the geometry options of reading A20.  The two
builders are covered with the option in test_score_gpu.py / test_comb_gpu.py."""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as O
from tests.parity import compare_fit
from workloads import barrel_events as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    import paper_1705_02876_b200 as K
    c = K.KFContext(0)
    yield c
    c.close()


def _soft_thick(n_tracks, event):
    cfg = W.get_config(1)
    cfg.energy_loss = 1
    cfg.x_over_X0 = 0.04
    cfg.pt_min, cfg.pt_max = 0.5, 1.0
    return W.simulate_event(cfg, event, n_tracks=n_tracks)


def _oracle_fit(b, model=0, hl=None, eloss=1):
    with O.geometry_options(model, hl, energy_loss=eloss):
        return O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask, nthreads=8)


def test_fit_with_energy_loss_thick_layers(ctx):
    """Soft tracks (pT 0.5..1 GeV) through 4 % X0 layers: 1.5 MeV lost per layer, 15 MeV over the track."""
    from paper_1705_02876_b200.buffers import DeviceFit
    b = _soft_thick(20000, 3)
    assert b.energy_loss == 1
    d = DeviceFit.from_batch(b, "cuda:0")
    d.fit(ctx)
    torch.cuda.synchronize()
    g, o = d.results(), _oracle_fit(b)
    res = compare_fit(g, o, float(b.radius[-1]), max_diverged_frac=2e-3)
    print("fit with energy loss:", res)
    # the option is felt: the same kernel without it ends with visibly more momentum
    b.energy_loss = 0
    d0 = DeviceFit.from_batch(b, "cuda:0")
    d0.fit(ctx)
    torch.cuda.synchronize()
    g0 = d0.results()
    ok = (g["status"] == 0) & (g0["status"] == 0)
    dp = np.linalg.norm(g0["par"][3:6, ok], axis=0) - np.linalg.norm(g["par"][3:6, ok], axis=0)
    assert 5e-3 < np.median(dp) < 3e-2


def test_fit_config3_energy_loss_and_path_length(ctx):
    """Config 3 (20 layers, |eta| up to 1.5, pT from 0.3 GeV) with path-length material AND energy loss in
    generator and fitter: the loss grows with 1/cos(psi) like the scattering."""
    from paper_1705_02876_b200.buffers import DeviceFit
    cfg = W.get_config(3)
    cfg.material_model, cfg.energy_loss = 1, 1
    b = W.simulate_event(cfg, 5, n_tracks=30000)
    d = DeviceFit.from_batch(b, "cuda:0")
    d.fit(ctx)
    torch.cuda.synchronize()
    g, o = d.results(), _oracle_fit(b, model=1)
    assert np.array_equal(g["nhits"], o["nhits"])
    res = compare_fit(g, o, float(b.radius[-1]), max_diverged_frac=2e-3)
    print("config 3, path length + energy loss:", res)


def test_small_batches_and_ragged_sizes(ctx):
    from paper_1705_02876_b200.buffers import DeviceFit
    for n in (1, 33, 257):
        b = _soft_thick(n, 11)
        d = DeviceFit.from_batch(b, "cuda:0")
        d.fit(ctx)
        torch.cuda.synchronize()
        compare_fit(d.results(), _oracle_fit(b), float(b.radius[-1]), max_diverged_frac=0.05)


def _slow_tracks(n):
    """30 MeV pions in a weak field (0.05 T, so that they reach every layer) through very thin layers; the fitter
    is then told that layer 4 is a slab of 2 X0, where the mean loss exceeds the kinetic energy of a few MeV."""
    cfg = W.get_config(1)
    cfg.Bz, cfg.x_over_X0 = 0.05, 1e-4
    cfg.pt_min, cfg.pt_max = 0.025, 0.04
    b = W.simulate_event(cfg, 12, n_tracks=n)
    b.x_over_X0 = np.full(b.n_layers, 1e-4, dtype=np.float32)
    b.x_over_X0[4] = 2.0
    b.energy_loss = 1
    return b


def test_a_track_that_would_stop_fails_the_layer(ctx):
    from paper_1705_02876_b200.buffers import DeviceFit
    b = _slow_tracks(500)
    d = DeviceFit.from_batch(b, "cuda:0")
    d.fit(ctx)
    torch.cuda.synchronize()
    g, o = d.results(), _oracle_fit(b)
    assert np.all(o["status"] == O.PROP_FAIL) and np.all(o["nhits"] == b.n_layers - 1)
    assert np.array_equal(g["status"], o["status"]) and np.array_equal(g["nhits"], o["nhits"])
    # the other nine layers were fitted as usual
    compare_fit(dict(g, status=np.zeros_like(g["status"])), dict(o, status=np.zeros_like(o["status"])),
                float(b.radius[-1]), max_diverged_frac=0.02)


def test_refit_with_energy_loss(ctx):
    from paper_1705_02876_b200.buffers import DeviceFit
    b = _soft_thick(20000, 4)
    d = DeviceFit.from_batch(b, "cuda:0")
    d.fit_refit(ctx)
    torch.cuda.synchronize()
    with O.geometry_options(energy_loss=1):
        o = O.fit_refit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask)
    g, sg = d.results(), d.refit_results()
    fwd = compare_fit(g, o, float(b.radius[-1]), max_diverged_frac=2e-3)
    keep = o["nhits"] >= 3
    assert np.array_equal(sg["status"][keep], o["rstatus"][keep])
    ndf = np.maximum(2 * o["nhits"] - 5, 1)
    excl = o["status"] | o["rstatus"] | ((o["chi2"] > ndf + 9 * np.sqrt(2.0 * ndf)).astype(np.uint32) << 5)
    so = dict(par=o["rpar"][:, keep], cov=o["rcov"][keep], chi2=o["rchi2"][keep], nhits=o["nhits"][keep], status=excl[keep])
    gs = dict(par=sg["par"][:, keep], cov=sg["cov"][:, keep], chi2=sg["chi2"][keep], nhits=o["nhits"][keep], status=excl[keep])
    res = compare_fit(gs, so, float(b.radius[-1]), max_diverged_frac=5e-3)
    print("forward:", fwd, "smoothed with energy loss:", res)
    # the refit gives the energy back: at the innermost layer the smoothed momentum exceeds the forward one
    # (taken at the outermost layer) by about the ten layers' loss
    ok = (o["status"] == 0) & (o["rstatus"] == 0)
    dp = np.linalg.norm(sg["par"][3:6, ok], axis=0) - np.linalg.norm(g["par"][3:6, ok], axis=0)
    assert 5e-3 < np.median(dp) < 3e-2


def test_energy_loss_option_errors(ctx):
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceFit
    b = _soft_thick(8, 13)
    d = DeviceFit.from_batch(b, "cuda:0")
    for bad in (dict(energy_loss_model=2), dict(energy_loss_model=-1), dict(energy_loss_model=1, mass_gev=0.0)):
        kw = dict(radius_cm=d.geom.radius_cm, x_over_X0=d.geom.x_over_X0, Bz_tesla=d.geom.Bz_tesla,
                  mass_gev=d.geom.mass_gev)
        kw.update(bad)
        d.geom = K.Geometry(**kw)
        with pytest.raises(K.KFError):
            d.fit(ctx)
