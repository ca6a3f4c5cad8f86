"""Pins of the oracle's energy-loss option (reading A21; CPU only).

E1 stopping power against the PDG minimum-ionisation value for silicon; E2 the step's Jacobian against finite
differences of the applied map (and the size of the term the reading neglects); E3 energy bookkeeping and
forward/backward inversion; E4 a fit with the option off is untouched by the code path; E5 when generator and fitter share the option the momentum pulls equal those of the
loss-free event fitted loss-free, and they shift by > 0.35 sigma either way when only one side has it; E6 the same
for the smoother at the innermost layer.
"""
import numpy as np
import pytest

from oracle import kf_oracle as O
from workloads import barrel_events as W

M = 0.13957


def test_E1_minimum_ionisation_in_silicon():
    # PDG "Atomic and nuclear properties of materials": silicon <-dE/dx>_min = 1.664 MeV cm^2/g, reached near
    # beta*gamma = 3.5, INCLUDING the density-effect correction delta/2 that reading A21 leaves out.  With
    # Sternheimer's parametrisation for silicon (x0 = 0.2015, x1 = 2.8716, a = 0.1492, k = 3.2546, Cbar = 4.4351)
    # delta(beta gamma = 3.5) = 2 ln10 x - Cbar + a (x1 - x)^k, x = log10(3.5).
    bg = 3.5
    p = bg * M
    t = 1.0 / 21.82                                     # 1 g/cm^2 of silicon
    dedx = O.energy_loss(p, M, t) * 1e3                 # MeV cm^2/g, no density correction
    x = np.log10(bg)
    delta = 2.0 * np.log(10.0) * x - 4.4351 + 0.1492 * (2.8716 - x) ** 3.2546
    beta2 = bg * bg / (1.0 + bg * bg)
    with_density = dedx - 0.307075 * (14.0 / 28.0855) / beta2 * 0.5 * delta
    assert with_density == pytest.approx(1.664, abs=0.004)
    # shape: a 1/beta^2 fall, a minimum between beta*gamma = 3 and 5 (no density effect moves it up a little), then
    # the logarithmic relativistic rise
    bgs = np.geomspace(0.5, 1000.0, 400)
    curve = np.array([O.energy_loss(b * M, M, t) for b in bgs])
    assert 3.0 < bgs[np.argmin(curve)] < 5.0
    assert curve[0] > 3.0 * curve.min() and 1.2 * curve.min() < curve[-1] < 2.0 * curve.min()
    # linear in the thickness, zero without material
    assert O.energy_loss(p, M, 0.02) == pytest.approx(2.0 * O.energy_loss(p, M, 0.01), rel=1e-14)
    assert O.energy_loss(p, M, 0.0) == 0.0


@pytest.mark.parametrize("direction", [+1, -1])
def test_E2_jacobian_vs_finite_differences(direction):
    rng = np.random.default_rng(21)
    u = np.array([3.0, 4.0, 2.0, 0.21, -0.12, 0.17])     # low momentum, thick layer: a sizeable step
    t = 0.08
    A = rng.standard_normal((6, 6))
    C0 = A @ A.T
    rc, un, Cn, J = O.energy_loss_step(u, C0, M, t, direction)
    assert rc == 0
    np.testing.assert_allclose(Cn, J @ C0 @ J.T, rtol=1e-12, atol=1e-14)
    np.testing.assert_array_equal(J[:3, :3], np.eye(3))
    assert np.all(J[:3, 3:] == 0) and np.all(J[3:, :3] == 0)
    # finite differences of the map actually applied
    Jfd = np.zeros((6, 6))
    for c in range(6):
        h = 1e-6
        up, um = u.copy(), u.copy()
        up[c] += h
        um[c] -= h
        Jfd[:, c] = (O.energy_loss_step(up, C0, M, t, direction)[1] - O.energy_loss_step(um, C0, M, t, direction)[1]) / (2 * h)
    # the reading holds dE fixed in the Jacobian: J = Jfd + sign * (E''/p'') dE/dp n n^T exactly
    p = np.linalg.norm(u[3:])
    n = u[3:] / p
    dEdp = (O.energy_loss(p + 1e-6, M, t) - O.energy_loss(p - 1e-6, M, t)) / 2e-6
    pn = np.linalg.norm(un[3:])
    En = np.sqrt(pn * pn + M * M)
    corr = direction * (En / pn) * dEdp * np.outer(n, n)
    np.testing.assert_allclose(J[3:, 3:], Jfd[3:, 3:] + corr, rtol=0, atol=2e-8)
    np.testing.assert_allclose(Jfd[:3, :3], np.eye(3), atol=1e-9)
    # transverse directions scale by f = p''/p, the parallel one by g
    f = pn / p
    e_perp = np.cross(n, [0.0, 0.0, 1.0])
    e_perp /= np.linalg.norm(e_perp)
    np.testing.assert_allclose(J[3:, 3:] @ e_perp, f * e_perp, atol=1e-14)
    E = np.sqrt(p * p + M * M)
    np.testing.assert_allclose(J[3:, 3:] @ n, (En / pn) * (p / E) * n, atol=1e-14)
    # at the toy detector's working point the neglected term is below the covariance tolerance
    p1 = 0.5
    small = abs((O.energy_loss(p1 + 1e-6, M, 0.01) - O.energy_loss(p1 - 1e-6, M, 0.01)) / 2e-6)
    assert small < 1e-3


def test_E3_energy_bookkeeping_and_inverse():
    u = np.array([6.0, -5.0, 3.0, 0.4, 0.3, -0.5])
    p = np.linalg.norm(u[3:])
    E = np.sqrt(p * p + M * M)
    C0 = np.diag([1e-4, 1e-4, 1e-2, 1e-3, 1e-3, 2e-3])
    dE = O.energy_loss(p, M, 0.01)
    assert 0.25e-3 < dE < 0.6e-3                        # a few tenths of an MeV per 1 % X0 of silicon
    rc, u1, C1, J1 = O.energy_loss_step(u, C0, M, 0.01, +1)
    assert rc == 0
    p1 = np.linalg.norm(u1[3:])
    assert np.sqrt(p1 * p1 + M * M) == pytest.approx(E - dE, rel=1e-14)
    np.testing.assert_allclose(u1[3:] / p1, u[3:] / p, atol=1e-15)      # direction kept
    np.testing.assert_array_equal(u1[:3], u[:3])
    # path-length option scales the thickness seen
    with O.geometry_options(material_model=1):
        rc, u1p, _, _ = O.energy_loss_step(u, C0, M, 0.01, +1)
    cospsi = abs(u[0] * u[3] + u[1] * u[4]) / (np.hypot(u[0], u[1]) * p)
    p1p = np.linalg.norm(u1p[3:])
    assert E - np.sqrt(p1p * p1p + M * M) == pytest.approx(dE / cospsi, rel=1e-10)
    # backward step regains what the forward step took, up to (dE/dp) dE
    rc, u2, C2, J2 = O.energy_loss_step(u1, C1, M, 0.01, -1)
    assert rc == 0
    assert abs(np.linalg.norm(u2[3:]) - p) < 1e-3 * dE
    np.testing.assert_allclose(J2 @ J1, np.eye(6), atol=1e-5)
    np.testing.assert_allclose(C2, C0, atol=1e-7)
    # a particle that would stop: failure, nothing written
    slow = np.array([6.0, -5.0, 3.0, 0.004, 0.003, -0.005])
    rc, us, Cs, _ = O.energy_loss_step(slow, C0, M, 0.05, +1)
    assert rc == O.PROP_FAIL
    np.testing.assert_array_equal(us, slow)
    np.testing.assert_array_equal(Cs, C0)


def _fit(b, eloss, nthreads=4):
    with O.geometry_options(energy_loss=eloss):
        return O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask,
                            nthreads=nthreads)


def test_E4_option_off_is_the_plain_fit_and_does_not_leak():
    b = W.simulate_event(W.get_config(1), 0, n_tracks=300)
    r0 = O.fit_batch(b)
    r1 = _fit(b, 1, nthreads=1)
    r2 = O.fit_batch(b)
    for k in ("par", "cov", "chi2"):
        np.testing.assert_array_equal(r0[k], r2[k])
    # ten layers of 0.36 MeV each: the fitted momentum at the last layer is lower by a few MeV in total
    dp = np.linalg.norm(r0["par"][3:6], axis=0) - np.linalg.norm(r1["par"][3:6], axis=0)
    assert 1.5e-3 < np.median(dp) < 6e-3


def _momentum_pull(b, r):
    ndf = 2 * r["nhits"] - 5
    good = (r["status"] == 0) & (r["nhits"] == b.n_layers) & (r["chi2"] <= ndf + 9 * np.sqrt(2.0 * ndf))
    truth = b.truth[-1]                                  # truth after the last layer (scatter and loss included)
    pf = r["par"][3:6][:, good]
    pt_ = truth[3:6][:, good]
    n = pf / np.linalg.norm(pf, axis=0)
    var = np.einsum("in,nij,jn->n", n, r["cov"][good][:, 3:, 3:], n)
    return (np.linalg.norm(pf, axis=0) - np.linalg.norm(pt_, axis=0)) / np.sqrt(var)


def _soft_thick(energy_loss):
    cfg = W.get_config(1)
    cfg.energy_loss = energy_loss
    cfg.x_over_X0 = 0.04                                # thick layers and soft tracks: the loss is visible
    cfg.pt_min, cfg.pt_max = 0.5, 1.0
    return cfg


def test_E5_momentum_pulls_need_the_energy_loss():
    # The |p| estimate of a short-lever-arm fit is skewed by itself (the filter is linear in 1/R, not in p):
    # the reference is therefore the pull of the SAME event simulated and fitted without any loss.
    b0 = W.simulate_event(_soft_thick(0), 7, n_tracks=12000)
    b1 = W.simulate_event(_soft_thick(1), 7, n_tracks=12000)
    assert b1.energy_loss == 1 and b0.energy_loss == 0
    base = _momentum_pull(b0, _fit(b0, 0))
    with_loss = _momentum_pull(b1, _fit(b1, 1))
    without = _momentum_pull(b1, _fit(b1, 0))
    overdone = _momentum_pull(b0, _fit(b0, 1))
    assert abs(base.mean()) < 0.2 and 0.93 < base.std() < 1.1
    assert abs(with_loss.mean() - base.mean()) < 0.03 and abs(with_loss.std() - base.std()) < 0.03, \
        (with_loss.mean(), base.mean())
    # a fitter that ignores the loss reports the momentum the track had on the way, higher than what is left;
    # one that subtracts a loss that did not happen errs the other way by as much
    assert without.mean() > base.mean() + 0.35, without.mean()
    assert overdone.mean() < base.mean() - 0.35, overdone.mean()


def _smoothed_pull(b, eloss):
    with O.geometry_options(energy_loss=eloss):
        r = O.fit_refit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask)
    ndf = 2 * r["nhits"] - 5
    good = (r["status"] == 0) & (r["rstatus"] == 0) & (r["nhits"] == b.n_layers) & \
           (r["chi2"] <= ndf + 9 * np.sqrt(2.0 * ndf))
    truth = b.truth[0]                                   # just after the innermost layer
    pf = r["rpar"][3:6][:, good]
    n = pf / np.linalg.norm(pf, axis=0)
    var = np.einsum("in,nij,jn->n", n, r["rcov"][good][:, 3:, 3:], n)
    return (np.linalg.norm(pf, axis=0) - np.linalg.norm(truth[3:6][:, good], axis=0)) / np.sqrt(var)


def test_E6_smoother_with_energy_loss():
    b0 = W.simulate_event(_soft_thick(0), 8, n_tracks=8000)
    b1 = W.simulate_event(_soft_thick(1), 8, n_tracks=8000)
    base = _smoothed_pull(b0, 0)
    with_loss = _smoothed_pull(b1, 1)
    without = _smoothed_pull(b1, 0)
    assert abs(with_loss.mean() - base.mean()) < 0.04 and abs(with_loss.std() - base.std()) < 0.04, \
        (with_loss.mean(), base.mean())
    # the refit that never gives the energy back sees a track whose curvature changes along the way with a model
    # whose curvature cannot: its momentum at the first layer is off
    assert abs(without.mean() - base.mean()) > 0.1, (without.mean(), base.mean())
