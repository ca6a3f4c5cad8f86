"""Pins of the oracle's geometry options (reading A20: path-length material, finite barrel; CPU only)."""
import numpy as np
import pytest

from oracle import kf_oracle as O
from workloads import barrel_events as W


def test_G1_path_length_material():
    u = np.array([3.0, 4.0, 2.0, 0.9, -0.2, 1.3])            # at rho = 5
    p = np.linalg.norm(u[3:])
    cospsi = abs(u[0] * u[3] + u[1] * u[4]) / (5.0 * p)
    Q0 = O.process_noise(u, 0.13957, 0.01)
    with O.geometry_options(material_model=1):
        Q1 = O.process_noise(u, 0.13957, 0.01)
    th_flat = W.highland_theta0(np.array([p]), 0.13957, 0.01)[0]          # the generator's own Highland
    th_path = W.highland_theta0(np.array([p]), 0.13957, 0.01 / cospsi)[0]
    assert np.linalg.eigvalsh(Q0[3:, 3:])[-1] == pytest.approx(th_flat ** 2 * p * p, rel=1e-12)
    assert np.linalg.eigvalsh(Q1[3:, 3:])[-1] == pytest.approx(th_path ** 2 * p * p, rel=1e-12)
    assert th_path > th_flat
    # normal incidence: both models agree; and the option does not leak out of the context manager
    un = np.array([3.0, 4.0, 2.0, 0.6, 0.8, 0.0])
    with O.geometry_options(material_model=1):
        Qn = O.process_noise(un, 0.13957, 0.01)
    np.testing.assert_allclose(Qn, O.process_noise(un, 0.13957, 0.01), rtol=1e-12, atol=0)
    np.testing.assert_array_equal(O.process_noise(u, 0.13957, 0.01), Q0)


def test_G2_finite_barrel_equals_masking_the_missed_layers():
    cfg = W.get_config(3)                                      # |eta| up to 1.5: many crossings beyond z = 60 cm
    b = W.simulate_event(cfg, 2, n_tracks=400)
    hl = np.full(b.n_layers, 60.0)
    with O.geometry_options(half_length=hl):
        r = O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask, want_trace=True)
    out = (r["status"] & O.OUTSIDE) != 0
    assert 0.2 < out.mean() < 0.95 and np.all((r["status"] & ~np.uint32(O.OUTSIDE)) == 0)
    used = r["trace"][:, :, 121] != 0                          # [n][L]
    mask2 = (used * (1 << np.arange(b.n_layers))).sum(axis=1).astype(np.uint32)
    r2 = O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, mask2)
    np.testing.assert_array_equal(r["par"], r2["par"])
    np.testing.assert_array_equal(r["cov"], r2["cov"])
    np.testing.assert_array_equal(r["chi2"], r2["chi2"])
    assert np.array_equal(r["nhits"], r2["nhits"]) and np.all(r2["status"] == 0)
    # the fitted point of a track flagged OUTSIDE lies inside the barrel (last used layer)
    assert np.all(np.abs(r["par"][2]) <= 60.0 + 1.0)


def test_G3_pulls_with_path_length_material():
    cfg = W.get_config(1)
    cfg.material_model = 1
    cfg.half_length_cm = 30.0
    b = W.simulate_event(cfg, 4, n_tracks=12000)
    hl = np.full(b.n_layers, 30.0)
    with O.geometry_options(material_model=1, half_length=hl):
        r = O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask, nthreads=4)
    # hits are generated only inside the barrel, so the fitter's acceptance agrees with the mask except for
    # tracks whose fitted crossing falls just beyond the end
    assert ((r["status"] & O.OUTSIDE) != 0).mean() < 0.01
    ndf = 2 * r["nhits"] - 5
    good = (r["status"] == 0) & (r["nhits"] >= 6) & (r["chi2"] <= ndf + 9 * np.sqrt(2.0 * ndf))
    last = np.array([int(np.max(np.flatnonzero((m >> np.arange(10)) & 1))) for m in b.mask])
    truth = b.truth[last, :, np.arange(b.n)].T                 # truth at each track's last hit layer
    d = (r["par"] - truth)[:, good]
    C = r["cov"][good]
    for name, i in (("px", 3), ("py", 4), ("pz", 5), ("z", 2)):
        pull = d[i] / np.sqrt(C[:, i, i])
        assert abs(pull.mean()) < 0.05 and 0.93 < pull.std() < 1.12, (name, pull.mean(), pull.std())
    assert 0.95 < (r["chi2"][good] / ndf[good]).mean() < 1.12
