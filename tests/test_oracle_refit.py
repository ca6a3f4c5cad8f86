"""Pins of the oracle's inward propagation and backward refit / smoother (reading A18; CPU only).
R1 (S1 in round 1) inward propagation: inverse of the outward one, invariants, Jacobian vs finite differences.
S2 exact helix: the refit recovers the truth at the innermost layer with chi2 = 0.
S3 backward EKF == batch weighted least squares of the affine model it linearises.
S4 pulls at the innermost layer, chi2/ndf, and the smoothed errors are smaller than the forward-filtered ones there."""
import math

import numpy as np
import pytest

from oracle import kf_oracle as O
from workloads import barrel_events as W

BZ = 3.8


def _rand_state(rng):
    phi = rng.uniform(0, 2 * np.pi)
    rho = rng.uniform(2.0, 32.0)
    pos = np.array([rho * np.cos(phi), rho * np.sin(phi), rng.uniform(-20, 20)])
    pt = rng.uniform(0.4, 10.0)
    dphi = phi + rng.uniform(-0.5, 0.5)
    mom = np.array([pt * np.cos(dphi), pt * np.sin(dphi), pt * np.sinh(rng.uniform(-1, 1))])
    return np.concatenate([pos, mom]), rng.choice([-1.0, 1.0])


def test_S1_inward_propagation_inverts_outward_and_jacobian():
    rng = np.random.default_rng(4)
    for _ in range(150):
        # a state that came from further in, so that every radius in between lies on its helix
        u0, q = _rand_state(rng)
        rho0 = math.hypot(u0[0], u0[1])
        rc0, u, _, _, _ = O.propagate(u0, q, BZ, rho0 + rng.uniform(1.0, 8.0), want_F=False)
        assert rc0 == 0
        rho = math.hypot(u[0], u[1])
        r_in = rng.uniform(rho0 + 0.2, rho - 0.3)
        rc, v, F, s, th = O.propagate_inward(u, q, BZ, r_in)
        assert rc == 0 and s < 0 and th * q < 0
        assert math.hypot(v[0], v[1]) == pytest.approx(r_in, rel=1e-13)
        assert math.hypot(v[3], v[4]) == pytest.approx(math.hypot(u[3], u[4]), rel=1e-13) and v[5] == u[5]
        # outward propagation from there returns to the start (same helix)
        rc2, w, F2, s2, _ = O.propagate(v, q, BZ, rho)
        assert rc2 == 0 and s2 == pytest.approx(-s, rel=1e-10)
        np.testing.assert_allclose(w, u, rtol=0, atol=2e-11)
        # Jacobian vs central finite differences, radial null at arrival, |p| conserved
        Fd = np.zeros((6, 6))
        for c in range(6):
            h = 1e-5 * max(1.0, abs(u[c]))
            up = u.copy(); um = u.copy(); up[c] += h; um[c] -= h
            Fd[:, c] = (O.propagate_inward(up, q, BZ, r_in, want_F=False)[1] - O.propagate_inward(um, q, BZ, r_in, want_F=False)[1]) / (2 * h)
        assert np.max(np.abs(F - Fd) / np.maximum(1.0, np.abs(F))) < 2e-6
        np.testing.assert_allclose(np.array([v[0], v[1], 0, 0, 0, 0]) @ F, 0.0, atol=1e-10)
        np.testing.assert_allclose(v[3:] @ F[3:, :], np.concatenate([np.zeros(3), u[3:]]), atol=1e-10)
    # wrong direction requests fail
    u, q = _rand_state(rng)
    rho = math.hypot(u[0], u[1])
    assert O.propagate_inward(u, q, BZ, rho + 1.0)[0] == O.PROP_FAIL
    assert O.propagate(u, q, BZ, rho - 1.0)[0] == O.PROP_FAIL


def test_S2_exact_helix_recovered_at_innermost_layer():
    cfg = W.get_config(0)
    b = W.simulate_event(cfg, 7, n_tracks=200, smear_hits=False, smear_seed=False, dtype=np.float64)
    r = O.fit_refit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask)
    assert np.all(r["rstatus"] == 0) and np.all(r["status"] == 0)
    truth0 = b.truth[0]
    np.testing.assert_allclose(r["rpar"][:3], truth0[:3], rtol=0, atol=1e-8)
    np.testing.assert_allclose(r["rpar"][3:], truth0[3:], rtol=1e-8, atol=1e-9)
    assert np.max(r["rchi2"]) < 1e-10


def _batch_wls_backward(x0, C0, trace, hits, Vs, layers):
    """Brute-force WLS of the affine model the backward EKF linearises.  The prior covariance C0 (the
    inflated forward covariance) has rank 5 -- no variance along the radial position direction -- so the
    state at the outermost layer is x0 + U z with U spanning the range of C0; unknowns: z (5) and two
    scattering variables per propagation step."""
    nsteps = len(layers) - 1
    w0, v0 = np.linalg.eigh(C0)
    U = v0[:, 1:]                                   # drop the single null direction
    assert abs(w0[0]) < 1e-10 * w0[-1] and w0[1] > 0
    nu = 5 + 2 * nsteps
    rows, rhs, Ws = [np.eye(nu)[:5]], [np.zeros(5)], [np.linalg.inv(U.T @ C0 @ U)]
    if nsteps:
        rows.append(np.eye(nu)[5:]); rhs.append(np.zeros(2 * nsteps)); Ws.append(np.eye(2 * nsteps))
    a = x0.copy(); B = np.zeros((6, nu)); B[:, :5] = U
    H = np.zeros((3, 6)); H[:, :3] = np.eye(3)
    xhat_prev = x0.copy()
    for k, l in enumerate(layers):
        t = trace[l]
        x_pred, F, Q, x_filt = t[0:6], t[6:42].reshape(6, 6), t[42:78].reshape(6, 6), t[78:84]
        if k > 0:
            w, v = np.linalg.eigh(Q)
            G = v[:, -2:] * np.sqrt(np.maximum(w[-2:], 0.0))
            E = np.zeros((2, nu)); E[:, 5 + 2 * (k - 1): 7 + 2 * (k - 1)] = np.eye(2)
            # x_k = x_pred + F (x_{k-1} + G w - xhat_{k-1})
            a = x_pred + F @ (a - xhat_prev)
            B = F @ (B + G @ E)
        rows.append(H @ B); rhs.append(hits[l] - H @ a); Ws.append(np.linalg.inv(Vs[l]))
        xhat_prev = x_filt
    N = sum(R.T @ Wm @ R for R, Wm in zip(rows, Ws))
    g = sum(R.T @ Wm @ y for R, Wm, y in zip(rows, Ws, rhs))
    th = np.linalg.solve(N, g)
    cost = sum((y - R @ th) @ Wm @ (y - R @ th) for R, Wm, y in zip(rows, Ws, rhs))
    return a + B @ th, B @ np.linalg.inv(N) @ B.T, cost


@pytest.mark.parametrize("config,L", [(1, 5), (1, 3), (0, 4)])
def test_S3_backward_ekf_equals_batch_wls(config, L):
    cfg = W.get_config(config)
    b = W.simulate_event(cfg, 3, n_tracks=10)
    r = O.fit_refit_tracks(b.radius[:L], b.x_over_X0[:L], b.Bz, b.mass, b.par, b.cov, b.q, b.hpos[:L], b.hcov[:L],
                            None, want_trace=True)
    Vs = O.unpack_cov6(b.hcov[:L])
    for i in range(b.n):
        assert r["status"][i] == 0 and r["rstatus"][i] == 0
        hits = b.hpos[:L, :, i].astype(np.float64)
        x0, C0 = r["par"][:, i], O.REFIT_KAPPA * r["cov"][i]
        x, Cx, cost = _batch_wls_backward(x0, C0, r["trace_bwd"][i], hits, Vs[i], list(range(L - 1, -1, -1)))
        np.testing.assert_allclose(r["rpar"][:, i], x, rtol=1e-9, atol=1e-9)
        assert np.max(np.abs(r["rcov"][i] - Cx)) < 1e-8 * np.max(np.abs(Cx))
        assert r["rchi2"][i] == pytest.approx(cost, rel=1e-8, abs=1e-9)


def test_S4_smoothed_pulls_and_gain_over_forward_filter():
    b = W.make_fit_batch(1)
    n = 6000
    sl = lambda a: np.ascontiguousarray(a[..., :n])
    r = O.fit_refit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, sl(b.par), sl(b.cov), sl(b.q), sl(b.hpos), sl(b.hcov), sl(b.mask))
    ndf = 2 * r["nhits"] - 5
    good = (r["status"] == 0) & (r["rstatus"] == 0) & (r["chi2"] <= ndf + 9 * np.sqrt(2.0 * ndf))
    assert good.mean() > 0.995
    x, Cs, truth = r["rpar"][:, good], r["rcov"][good], b.truth[0][:, :n][:, good]
    d = x - truth
    phi = np.arctan2(x[1], x[0])
    tvec = np.stack([-np.sin(phi), np.cos(phi)])
    pulls = {"t": (d[0] * tvec[0] + d[1] * tvec[1]) / np.sqrt(np.einsum("in,nij,jn->n", tvec, Cs[:, :2, :2], tvec)),
             "z": d[2] / np.sqrt(Cs[:, 2, 2]), "px": d[3] / np.sqrt(Cs[:, 3, 3]), "py": d[4] / np.sqrt(Cs[:, 4, 4]),
             "pz": d[5] / np.sqrt(Cs[:, 5, 5])}
    for name, p in pulls.items():
        assert abs(p.mean()) < 0.05, (name, p.mean())
        assert 0.93 < p.std() < 1.12, (name, p.std())
    # backward chi2 has 2 n_hits degrees of freedom minus 5 fitted, plus the weak prior: ~ same as forward
    assert 0.9 < (r["rchi2"][good] / ndf[good]).mean() < 1.15
    # all hits constrain the innermost point: its momentum is known as well as at the outermost layer and far
    # better than a forward filter knows it after one hit (prior 0.3 pT)
    pabs = np.linalg.norm(x[3:], axis=0)
    rel = np.sqrt(Cs[:, 3, 3] + Cs[:, 4, 4] + Cs[:, 5, 5]) / pabs
    assert np.median(rel) < 0.05
    assert np.median(np.abs(np.linalg.norm(d[3:], axis=0)) / pabs) < 0.05


def test_S5_nothing_fitted_comes_back_untouched():
    """A track the forward fit cannot start (bad charge, empty mask) has no backward pass: both results are the
    input, chi2 0, smoothed status 0 -- independently of what memory the call happens to get for its private trace."""
    b = W.simulate_event(W.get_config(1), 3, n_tracks=64)
    b.q[5] = 0
    b.mask[9] = 0
    for _ in range(3):                       # repeated: an uninitialised read would not be stable
        r = O.fit_refit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask)
        assert r["status"][5] == O.BAD_CHARGE and r["rstatus"][5] == 0 and r["status"][9] == 0 and r["rstatus"][9] == 0
        for i in (5, 9):
            np.testing.assert_array_equal(r["rpar"][:, i], b.par[:, i].astype(np.float64))
            np.testing.assert_array_equal(O.pack_cov21(r["rcov"][i:i + 1])[:, 0], b.cov[:, i].astype(np.float64))
            assert r["rchi2"][i] == 0 and r["nhits"][i] == 0
