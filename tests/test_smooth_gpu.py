"""GPU parity of kf_fit_tracks_smooth (forward fit + inward refit, reading A18) against the oracle."""
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


def _both(ctx, b, kappa=O.SMOOTH_KAPPA):
    from paper_1705_02876_b200.buffers import DeviceFit
    d = DeviceFit.from_batch(b, "cuda:0")
    d.fit_smooth(ctx, kappa)
    torch.cuda.synchronize()
    o = O.fit_smooth_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask, kappa=kappa)
    return d, o


def _compare(d, o, r_last, max_div=1e-3):
    fwd = compare_fit(d.results(), {k: o[k] for k in ("par", "cov", "chi2", "nhits", "status")}, r_last, max_div)
    sg = d.smoothed_results()
    assert np.array_equal(sg["status"], o["sstatus"])
    # Smoothed result, same metric.  Excluded (A14): tracks the FORWARD fit flagged or that diverged there, and
    # tracks the backward pass flagged -- marked through the status word compare_fit looks at.
    ndf = np.maximum(2 * o["nhits"] - 5, 1)
    fwd_div = o["chi2"] > ndf + 9 * np.sqrt(2.0 * ndf)
    excl = o["status"] | o["sstatus"] | (fwd_div.astype(np.uint32) << 4)
    so = dict(par=o["spar"], cov=o["scov"], chi2=o["schi2"], nhits=o["nhits"], status=excl)
    sm = compare_fit(dict(sg, status=excl, nhits=o["nhits"]), so, r_last, max_diverged_frac=max(max_div, 2e-3))
    return fwd, sm


@pytest.mark.parametrize("config", [0, 1, 3])
def test_smooth_parity_full_config(ctx, config):
    b = W.make_fit_batch(config)
    d, o = _both(ctx, b)
    fwd, sm = _compare(d, o, float(b.radius[-1]))
    print(f"config {config}: forward {fwd}\n          smoothed {sm}")


def test_smooth_forward_part_equals_plain_fit(ctx):
    from paper_1705_02876_b200.buffers import DeviceFit
    b = W.make_fit_batch(1)
    d1 = DeviceFit.from_batch(b, "cuda:0"); d1.fit(ctx)
    d2 = DeviceFit.from_batch(b, "cuda:0"); d2.fit_smooth(ctx)
    torch.cuda.synchronize()
    r1, r2 = d1.results(), d2.results()
    for k in r1:
        assert np.array_equal(r1[k], r2[k]), k


def test_smooth_ragged_masks_and_flags(ctx):
    b = W.simulate_event(W.get_config(1), 8, n_tracks=1003)
    rng = np.random.default_rng(3)
    b.mask = (rng.integers(0, 1 << 10, size=b.n) | 0b111).astype(np.uint32)
    b.mask[:30] = 0                       # nothing to fit: input comes back in both results
    b.q[30] = 0                           # bad charge
    d, o = _both(ctx, b)
    sel = o["nhits"] >= 5
    sel[:31] = False
    sg, so_ = d.smoothed_results(), o
    sub = lambda r, keys: {k: (r[k][..., sel] if k in ("par", "cov") else r[k][sel]) for k in keys}
    g = sub(sg, ("par", "cov", "chi2", "nhits", "status"))
    oo = dict(par=o["spar"][:, sel], cov=o["scov"][sel], chi2=o["schi2"][sel], nhits=g["nhits"], status=o["sstatus"][sel])
    compare_fit(g, oo, float(b.radius[-1]), max_diverged_frac=0.05)
    assert np.array_equal(sg["par"][:, :31], b.par[:, :31]) and np.array_equal(sg["cov"][:, :31], b.cov[:, :31])
    assert np.all(sg["chi2"][:31] == 0)
