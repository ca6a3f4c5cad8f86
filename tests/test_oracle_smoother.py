"""Pins of the oracle's fixed-interval (Rauch-Tung-Striebel) smoother, reading A22 (CPU only).

PAPER.md:57 (section 2): the last stage is "a final fit with a KF and smoother".  The smoother gives, at EVERY
used layer, the estimate of the state there from ALL hits of the track.
SM1 smoothed state and covariance at every layer == the batch weighted least squares of the affine model the
    forward EKF linearised, evaluated at that layer (brute force, L <= 6; also with holes in the hit mask, and
    with the energy-loss option whose Jacobian enters the model).
SM2 exact helix (no noise, no material): the smoothed state at every layer is the truth there.
SM3 pulls against the post-scatter truth at the first, middle and last layer have mean 0, width 1.
SM4 at the outermost used layer smoothed == filtered; everywhere C_filtered - C_smoothed is positive semi-definite
    (more information never hurts); the smoothed covariance keeps the radial null direction (rank 5).
SM5 nothing fitted -> no layer marked, zeros, forward result = input.
"""
import numpy as np
import pytest

from oracle import kf_oracle as O
from workloads import barrel_events as W


def _batch_wls_all_layers(seed, C0, trace, hits, Vs, used, Q_from_pred=False):
    """Weighted least squares of the affine model the EKF linearises, over the layers in `used` (ascending).
    Unknowns: x0 (6) and two scattering variables per used layer.  Returns per used layer the solution
    evaluated there: (x_l, Cov_l)."""
    m = len(used)
    nu = 6 + 2 * m
    rows, rhs, Ws = [np.eye(nu)[:6]], [seed], [np.linalg.inv(C0)]
    rows.append(np.eye(nu)[6:]); rhs.append(np.zeros(2 * m)); Ws.append(np.eye(2 * m))
    a = np.zeros(6); B = np.zeros((6, nu)); B[:, :6] = np.eye(6)
    xhat_prev, C_prev = seed.copy(), C0
    H = np.zeros((3, 6)); H[:, :3] = np.eye(3)
    per_layer = []
    for k, l in enumerate(used):
        t = trace[l]
        x_pred, Q, x_filt, C_filt = t[0:6], t[42:78].reshape(6, 6), t[78:84], t[84:120].reshape(6, 6)
        Gj = t[158:194].reshape(6, 6)                 # Jacobian of the whole map (= F without energy loss)
        if Q_from_pred:                                # effective process noise of the whole map (energy loss: J Q J^T)
            Q = t[122:158].reshape(6, 6) - Gj @ C_prev @ Gj.T
        else:
            assert np.array_equal(Gj, t[6:42].reshape(6, 6))
        w, v = np.linalg.eigh(0.5 * (Q + Q.T))
        Gs = v[:, -2:] * np.sqrt(np.maximum(w[-2:], 0.0))
        # (derived from the predicted covariance, Q carries the rounding of C_pred - G C G^T: 1e-16 of |C|)
        assert np.allclose(Gs @ Gs.T, Q, atol=(1e-13 * np.abs(C_prev).max() if Q_from_pred else 1e-12 * np.abs(Q).max()) + 1e-18)
        E = np.zeros((2, nu)); E[:, 6 + 2 * k: 8 + 2 * k] = np.eye(2)
        a = x_pred + Gj @ (a - xhat_prev)              # x_l = a + B theta, linearised about the filter's own points
        B = Gj @ B + Gs @ E
        rows.append(H @ B); rhs.append(hits[l] - H @ a); Ws.append(np.linalg.inv(Vs[l]))
        per_layer.append((a.copy(), B.copy()))
        xhat_prev, C_prev = x_filt, C_filt
    N = sum(R.T @ Wm @ R for R, Wm in zip(rows, Ws))
    g = sum(R.T @ Wm @ y for R, Wm, y in zip(rows, Ws, rhs))
    th = np.linalg.solve(N, g)
    Ni = np.linalg.inv(N)
    return [(a_ + B_ @ th, B_ @ Ni @ B_.T) for a_, B_ in per_layer]


def _check_against_wls(b, L, mask=None, eloss=0):
    with O.geometry_options(0, None, energy_loss=eloss):
        r = O.fit_tracks(b.radius[:L], b.x_over_X0[:L], b.Bz, b.mass, b.par, b.cov, b.q, b.hpos[:L], b.hcov[:L], mask,
                         want_trace=True)
        s = O.smooth_tracks(b.radius[:L], b.x_over_X0[:L], b.Bz, b.mass, b.par, b.cov, b.q, b.hpos[:L], b.hcov[:L], mask)
    Cs = O.unpack_cov21(b.cov.astype(np.float64))
    Vs = O.unpack_cov6(b.hcov[:L])
    worst_x = worst_c = 0.0
    for i in range(b.n):
        assert r["status"][i] == 0 and s["sstatus"][i] == 0
        used = [l for l in range(L) if (s["used"][i] >> l) & 1]
        assert used == [l for l in range(L) if r["trace"][i][l][121] != 0] and len(used) == s["nhits"][i]
        hits = b.hpos[:L, :, i].astype(np.float64)
        sol = _batch_wls_all_layers(b.par[:, i].astype(np.float64), Cs[i], r["trace"][i], hits, Vs[i], used,
                                    Q_from_pred=bool(eloss))
        for (x, Cx), l in zip(sol, used):
            np.testing.assert_allclose(s["spar"][l, :, i], x, rtol=1e-9, atol=1e-9)
            blk = np.max(np.abs(Cx))
            assert np.max(np.abs(s["scov"][i, l] - Cx)) < 1e-8 * blk
            worst_x = max(worst_x, np.max(np.abs(s["spar"][l, :, i] - x)))
            worst_c = max(worst_c, np.max(np.abs(s["scov"][i, l] - Cx)) / blk)
        for l in range(L):                       # layers not used: zeros
            if l not in used:
                assert not s["spar"][l, :, i].any() and not s["scov"][i, l].any()
    return worst_x, worst_c


@pytest.mark.parametrize("config,L", [(1, 5), (1, 3), (0, 4), (1, 6), (1, 1)])
def test_SM1_smoother_equals_batch_wls_at_every_layer(config, L):
    b = W.simulate_event(W.get_config(config), 3, n_tracks=12)
    wx, wc = _check_against_wls(b, L)
    print(f"config {config}, L = {L}: worst |dx| {wx:.2e}, worst rel dC {wc:.2e}")


def test_SM1_with_holes_in_the_hit_mask():
    b = W.simulate_event(W.get_config(1), 5, n_tracks=12)
    mask = np.array([0b111111, 0b101111, 0b110111, 0b011111, 0b111011, 0b100111, 0b111101, 0b001111, 0b110011,
                     0b010111, 0b111110, 0b101011], dtype=np.uint32)
    _check_against_wls(b, 6, mask)


def test_SM1_with_energy_loss():
    cfg = W.get_config(1)
    import dataclasses
    b = W.simulate_event(dataclasses.replace(cfg, energy_loss=1), 3, n_tracks=10)
    _check_against_wls(b, 5, eloss=1)


def test_SM2_exact_helix_recovered_at_every_layer():
    b = W.simulate_event(W.get_config(0), 7, n_tracks=200, smear_hits=False, smear_seed=False, dtype=np.float64)
    s = O.smooth_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask)
    assert np.all(s["status"] == 0) and np.all(s["sstatus"] == 0) and np.all(s["used"] == 0x3ff)
    for l in range(b.n_layers):
        np.testing.assert_allclose(s["spar"][l, :3], b.truth[l][:3], rtol=0, atol=1e-8)
        np.testing.assert_allclose(s["spar"][l, 3:], b.truth[l][3:], rtol=1e-8, atol=1e-9)


def _pulls(x, Cs, truth):
    d = x - truth
    phi = np.arctan2(x[1], x[0])
    tvec = np.stack([-np.sin(phi), np.cos(phi)])
    return {"t": (d[0] * tvec[0] + d[1] * tvec[1]) / np.sqrt(np.einsum("in,nij,jn->n", tvec, Cs[:, :2, :2], tvec)),
            "z": d[2] / np.sqrt(Cs[:, 2, 2]), "px": d[3] / np.sqrt(Cs[:, 3, 3]), "py": d[4] / np.sqrt(Cs[:, 4, 4]),
            "pz": d[5] / np.sqrt(Cs[:, 5, 5])}


@pytest.fixture(scope="module")
def cfg1_smoothed():
    b = W.make_fit_batch(1)
    n = 8000
    sl = lambda a: np.ascontiguousarray(a[..., :n])
    s = O.smooth_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, sl(b.par), sl(b.cov), sl(b.q), sl(b.hpos), sl(b.hcov),
                        sl(b.mask), nthreads=4)
    f = O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, sl(b.par), sl(b.cov), sl(b.q), sl(b.hpos), sl(b.hcov),
                     sl(b.mask), nthreads=4, want_trace=True)
    return b, n, s, f


def test_SM3_smoothed_pulls_at_first_middle_last_layer(cfg1_smoothed):
    b, n, s, f = cfg1_smoothed
    ndf = 2 * s["nhits"] - 5
    good = (s["status"] == 0) & (s["sstatus"] == 0) & (s["chi2"] <= ndf + 9 * np.sqrt(2.0 * ndf))
    assert good.mean() > 0.995
    L = b.n_layers
    for l in (0, L // 2, L - 1):
        x, Cs, truth = s["spar"][l][:, good], s["scov"][good, l], b.truth[l][:, :n][:, good]
        for name, p in _pulls(x, Cs, truth).items():
            assert abs(p.mean()) < 0.04, (l, name, p.mean())
            assert 0.95 < p.std() < 1.10, (l, name, p.std())
    # all hits constrain every point: the momentum at the FIRST layer is known as well as at the last
    # (a forward filter knows it to the 30 % prior there)
    for l in (0, L - 1):
        p = s["spar"][l][3:, good]
        Cm = s["scov"][good, l][:, 3:, 3:]
        rel = np.sqrt(np.trace(Cm, axis1=1, axis2=2)) / np.linalg.norm(p, axis=0)
        assert np.median(rel) < 0.05, (l, np.median(rel))


def test_SM4_last_layer_filtered_and_information_never_hurts(cfg1_smoothed):
    b, n, s, f = cfg1_smoothed
    L = b.n_layers
    assert np.array_equal(s["par"], f["par"]) and np.array_equal(s["cov"], f["cov"]) and np.array_equal(s["chi2"], f["chi2"])
    sel = np.flatnonzero((s["status"] == 0) & (s["used"] == (1 << L) - 1))[:1500]
    # outermost layer: smoothed == filtered == the forward result
    np.testing.assert_array_equal(s["spar"][L - 1][:, sel], f["par"][:, sel])
    np.testing.assert_array_equal(s["scov"][sel, L - 1], f["cov"][sel])
    for l in range(L - 1):
        Cf = f["trace"][sel, l, 84:120].reshape(-1, 6, 6)
        D = Cf - s["scov"][sel, l]
        w = np.linalg.eigvalsh(0.5 * (D + np.swapaxes(D, 1, 2)))
        scale = np.abs(np.linalg.eigvalsh(Cf)).max(axis=1)
        assert np.all(w[:, 0] > -1e-9 * scale), (l, (w[:, 0] / scale).min())
        # rank 5, null direction = radial direction of the FILTER's predicted point (the model's), to rounding
        ws, vs = np.linalg.eigh(s["scov"][sel, l])
        assert np.all(np.abs(ws[:, 0]) < 1e-9 * ws[:, -1]) and np.all(ws[:, 1] > 0)
        xp = f["trace"][sel, l, 0:2]
        rad = xp / np.linalg.norm(xp, axis=1, keepdims=True)
        assert np.all(np.abs(np.abs(np.einsum("ni,ni->n", vs[:, :2, 0], rad)) - 1.0) < 1e-6)
        # and it is tighter than the filtered one on the momentum by a large factor on the inner layers
        if l == 0:
            assert np.median(np.trace(Cf[:, 3:, 3:], axis1=1, axis2=2) / np.trace(s["scov"][sel, l][:, 3:, 3:], axis1=1, axis2=2)) > 50


def test_SM5_nothing_fitted_and_failed_layers():
    b = W.simulate_event(W.get_config(1), 3, n_tracks=64)
    b.q[5] = 0
    b.mask[9] = 0
    b.hpos[4, 1, 20] = np.nan                 # NONFINITE on layer 4 of track 20: skipped by the filter, so not smoothed
    s = O.smooth_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask)
    assert s["status"][5] == O.BAD_CHARGE and s["used"][5] == 0 and s["used"][9] == 0 and s["nhits"][9] == 0
    for i in (5, 9):
        assert not s["spar"][:, :, i].any() and not s["scov"][i].any()
        np.testing.assert_array_equal(s["par"][:, i], b.par[:, i].astype(np.float64))
    assert s["status"][20] == O.NONFINITE and s["used"][20] == 0x3ff & ~(1 << 4) and s["sstatus"][20] == 0
    assert not s["spar"][4, :, 20].any() and s["spar"][3, :, 20].any() and s["spar"][5, :, 20].any()
    # the same track with layer 4 masked out gives the same smoothed states, bit for bit
    b2 = W.simulate_event(W.get_config(1), 3, n_tracks=64)
    b2.mask[20] &= ~np.uint32(1 << 4)
    s2 = O.smooth_tracks(b2.radius, b2.x_over_X0, b2.Bz, b2.mass, b2.par, b2.cov, b2.q, b2.hpos, b2.hcov, b2.mask)
    np.testing.assert_array_equal(s["spar"][:, :, 20], s2["spar"][:, :, 20])
    np.testing.assert_array_equal(s["scov"][20], s2["scov"][20])
