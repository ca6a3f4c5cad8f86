"""Pins of the fp64 oracle against what the mathematics fixes (CPU only, no CUDA).

P1 exact helix recovery, P2 propagation invariants / RK4 / worked value, P3 Jacobian,
P4 EKF == batch weighted least squares, P5 PSD rank 5, P6 pulls, P7 Highland, P10 rotation.
(P8/P9, binning and scoring, live in test_oracle_scoring.py.)  Numbering: SURVEY.md 8(c).
"""
import math
import os

import numpy as np
import pytest

from oracle import kf_oracle as O
from workloads import barrel_events as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")
C_B = 2.99792458e-3
BZ = 3.8


def _rand_state(rng, r_max=30.0):
    """A state somewhere inside the barrel, moving outward."""
    phi = rng.uniform(0, 2 * np.pi)
    rho = rng.uniform(0.0, r_max)
    pos = np.array([rho * np.cos(phi), rho * np.sin(phi), rng.uniform(-20, 20)])
    pt = rng.uniform(0.4, 10.0)
    dphi = phi + rng.uniform(-0.6, 0.6)
    mom = np.array([pt * np.cos(dphi), pt * np.sin(dphi), pt * np.sinh(rng.uniform(-1, 1))])
    return np.concatenate([pos, mom]), rng.choice([-1.0, 1.0])


# ------------------------------------------------------------------------------------ P7
def test_P7_highland_check_values():
    rows = np.loadtxt(os.path.join(GOLD, "highland_check_values.txt"))
    for p, th in rows:
        assert O.theta0(p, 0.13957, 0.01) == pytest.approx(th, rel=1e-12)
    # values printed in SURVEY.md 8(c) A5 (independent evaluation), 6 significant digits
    for p, th in [(0.5, 2.32980e-3), (1.0, 1.13288e-3), (10.0, 1.12211e-4)]:
        assert O.theta0(p, 0.13957, 0.01) == pytest.approx(th, rel=1e-5)
    assert O.theta0(1.0, 0.13957, 0.0) == 0.0
    # beta -> 1, t = 1: theta0 -> 0.0136 / p
    assert O.theta0(1000.0, 0.13957, 1.0) == pytest.approx(0.0136 / 1000.0, rel=1e-7)


def test_P7_process_noise_structure():
    u = np.array([1.0, 2.0, 3.0, 0.7, -0.4, 1.1])
    Q = O.process_noise(u, 0.13957, 0.01)
    p = u[3:]
    th0 = O.theta0(np.linalg.norm(p), 0.13957, 0.01)
    assert np.all(Q[:3, :] == 0) and np.all(Q[:, :3] == 0)
    Qm = Q[3:, 3:]
    np.testing.assert_allclose(Qm, Qm.T, atol=0)
    np.testing.assert_allclose(Qm @ p, 0.0, atol=1e-18)          # no noise along p
    w = np.linalg.eigvalsh(Qm)
    np.testing.assert_allclose(w[1:], th0 ** 2 * p @ p, rtol=1e-12)  # isotropic transverse kick
    assert abs(w[0]) < 1e-18


# ------------------------------------------------------------------------------------ P2b
def test_P2b_worked_value_circle_through_origin():
    th, s, x, y, z, px, py, pz = np.loadtxt(os.path.join(GOLD, "helix_worked_value.txt"))
    rc, u, F, s_o, th_o = O.propagate([0, 0, 0, 1, 0, 0.5], +1, BZ, 4.0)
    assert rc == 0
    np.testing.assert_allclose(u, [x, y, z, px, py, pz], rtol=0, atol=1e-12)
    assert s_o == pytest.approx(s, abs=1e-12) and th_o == pytest.approx(th, abs=1e-13)
    # digits printed in SURVEY.md 8(c) P2b
    np.testing.assert_allclose(u[:5], [3.9989616232, -0.0911369072, 2.0001730808, 0.9989617580, -0.0455566243],
                               atol=1e-9)
    # negative charge mirrors y
    rc, um, _, _, _ = O.propagate([0, 0, 0, 1, 0, 0.5], -1, BZ, 4.0)
    np.testing.assert_allclose(um, u * np.array([1, -1, 1, 1, -1, 1]), atol=1e-13)


# ------------------------------------------------------------------------------------ P2
def _rk4(u, q, s_total, n=4000):
    k = q * C_B * BZ

    def f(v):
        pt = math.hypot(v[3], v[4])
        kap = k / pt
        return np.array([v[3] / pt, v[4] / pt, v[5] / pt, kap * v[4], -kap * v[3], 0.0])
    h = s_total / n
    v = np.array(u, dtype=np.float64)
    for _ in range(n):
        k1 = f(v); k2 = f(v + 0.5 * h * k1); k3 = f(v + 0.5 * h * k2); k4 = f(v + h * k3)
        v = v + h / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
    return v


def test_P2_propagation_invariants_and_rk4():
    rng = np.random.default_rng(1)
    for it in range(200):
        u, q = _rand_state(rng)
        rho = math.hypot(u[0], u[1])
        r1 = rho + rng.uniform(0.5, 6.0)
        r2 = r1 + rng.uniform(0.5, 6.0)
        rc, v, _, s, th = O.propagate(u, q, BZ, r1, want_F=False)
        assert rc == 0
        assert math.hypot(v[0], v[1]) == pytest.approx(r1, rel=1e-13)
        assert math.hypot(v[3], v[4]) == pytest.approx(math.hypot(u[3], u[4]), rel=1e-13)
        assert v[5] == u[5]
        assert s > 0 and th * q > 0
        assert v[2] - u[2] == pytest.approx(u[5] * s / math.hypot(u[3], u[4]), rel=1e-12, abs=1e-13)
        # composition: prop(prop(u, r1), r2) == prop(u, r2)
        rc2, w, _, _, _ = O.propagate(v, q, BZ, r2, want_F=False)
        rc3, w2, _, s2, _ = O.propagate(u, q, BZ, r2, want_F=False)
        assert rc2 == 0 and rc3 == 0
        np.testing.assert_allclose(w, w2, rtol=0, atol=2e-12)
        if it < 20:                                  # textbook integrator of the equations of motion
            np.testing.assert_allclose(_rk4(u, q, s), v, rtol=0, atol=2e-11)


def test_P2_propagation_failures():
    # target radius not outside the current one
    assert O.propagate([5, 0, 0, 1, 0, 0], 1, BZ, 5.0)[0] == O.PROP_FAIL
    assert O.propagate([5, 0, 0, 1, 0, 0], 1, BZ, 4.0)[0] == O.PROP_FAIL
    # a 0.05 GeV track from the origin has diameter 2R = 8.78 cm: cannot reach r = 12
    assert O.propagate([0, 0, 0, 0.05, 0, 0], 1, BZ, 12.0)[0] == O.PROP_FAIL
    assert O.propagate([0, 0, 0, 0.05, 0, 0], 1, BZ, 8.0)[0] == 0
    # NaN state fails rather than propagating garbage
    assert O.propagate([np.nan, 0, 0, 1, 0, 0], 1, BZ, 4.0)[0] == O.PROP_FAIL


# ------------------------------------------------------------------------------------ P3
def test_P3_jacobian_finite_differences_and_invariants():
    rng = np.random.default_rng(2)
    for _ in range(100):
        u, q = _rand_state(rng)
        r = math.hypot(u[0], u[1]) + rng.uniform(1.0, 8.0)
        rc, v, F, _, _ = O.propagate(u, q, BZ, r)
        assert rc == 0
        Fd = np.zeros((6, 6))
        for c in range(6):
            h = 1e-5 * max(1.0, abs(u[c]))
            up = u.copy(); um = u.copy(); up[c] += h; um[c] -= h
            vp = O.propagate(up, q, BZ, r, want_F=False)[1]
            vm = O.propagate(um, q, BZ, r, want_F=False)[1]
            Fd[:, c] = (vp - vm) / (2 * h)
        scale = np.maximum(1.0, np.abs(F))
        assert np.max(np.abs(F - Fd) / scale) < 2e-6
        # radial null: the arrival point stays on the cylinder
        np.testing.assert_allclose(np.array([v[0], v[1], 0, 0, 0, 0]) @ F, 0.0, atol=1e-11)
        # |p| conserved: sum_i p'_i F[p_i, u] = p_u (0 for position columns)
        lhs = v[3:] @ F[3:, :]
        np.testing.assert_allclose(lhs, np.concatenate([np.zeros(3), u[3:]]), atol=1e-11)
        # z row: F[z,z] = 1, F[pz,pz] = 1, pz decoupled
        assert F[2, 2] == 1.0 and F[5, 5] == 1.0
        assert np.all(F[5, :5] == 0) and np.all(F[[0, 1, 3, 4], 2] == 0) and np.all(F[[0, 1, 3, 4], 5] == 0)


# ------------------------------------------------------------------------------------ P1
def test_P1_exact_helix_is_recovered():
    """Seed = truth, hits = exact crossings, no material => fit == truth at the last layer, chi2 = 0.
    The truth comes from the generator's two-circle/atan2 crossing, the fit from the oracle's
    half-angle crossing: two independent formulations of the same helix."""
    cfg = W.get_config(0)
    b = W.simulate_event(cfg, 7, n_tracks=300, smear_hits=False, smear_seed=False, dtype=np.float64)
    r = O.fit_batch(b)
    assert np.all(r["status"] == 0) and np.all(r["nhits"] == 10)
    truth = b.truth[-1]
    np.testing.assert_allclose(r["par"][:3], truth[:3], rtol=0, atol=1e-9)
    np.testing.assert_allclose(r["par"][3:], truth[3:], rtol=1e-9, atol=1e-10)
    assert np.max(r["chi2"]) < 1e-12


# ------------------------------------------------------------------------------------ P4
def _batch_wls(seed, C0, trace, hits, Vs):
    """Brute-force weighted least squares of the affine model the EKF linearises.
    Unknowns: x0 (6) and two scattering variables per layer (Q_l = G_l G_l^T)."""
    L = trace.shape[0]
    nu = 6 + 2 * L
    a = np.zeros(6)
    B = np.zeros((6, nu)); B[:, :6] = np.eye(6)
    xhat_prev = seed.copy()
    a = seed.copy() * 0 + 0.0
    # x_0 = theta[0:6]
    rows, rhs, Ws = [], [], []
    # prior on x0 and unit prior on every w
    rows.append(np.eye(nu)[:6]); rhs.append(seed); Ws.append(np.linalg.inv(C0))
    rows.append(np.eye(nu)[6:]); rhs.append(np.zeros(2 * L)); Ws.append(np.eye(2 * L))
    a = np.zeros(6)                     # x_l = a + B theta
    for l in range(L):
        t = trace[l]
        x_pred, F, Q = t[0:6], t[6:42].reshape(6, 6), t[42:78].reshape(6, 6)
        x_filt = t[78:84]
        w, v = np.linalg.eigh(Q)
        G = v[:, -2:] * np.sqrt(np.maximum(w[-2:], 0.0))
        assert np.allclose(G @ G.T, Q, atol=1e-18)
        E = np.zeros((2, nu)); E[:, 6 + 2 * l: 8 + 2 * l] = np.eye(2)
        a = x_pred + F @ (a - xhat_prev)
        B = F @ B + G @ E
        H = np.zeros((3, 6)); H[:, :3] = np.eye(3)
        rows.append(H @ B); rhs.append(hits[l] - H @ a); Ws.append(np.linalg.inv(Vs[l]))
        xhat_prev = x_filt
    N = sum(R.T @ Wm @ R for R, Wm in zip(rows, Ws))
    g = sum(R.T @ Wm @ y for R, Wm, y in zip(rows, Ws, rhs))
    th = np.linalg.solve(N, g)
    cost = sum((y - R @ th) @ Wm @ (y - R @ th) for R, Wm, y in zip(rows, Ws, rhs))
    return a + B @ th, B @ np.linalg.inv(N) @ B.T, cost


@pytest.mark.parametrize("config,L", [(1, 5), (1, 3), (0, 4)])
def test_P4_ekf_equals_batch_weighted_least_squares(config, L):
    cfg = W.get_config(config)
    b = W.simulate_event(cfg, 3, n_tracks=12)
    r = O.fit_tracks(b.radius[:L], b.x_over_X0[:L], b.Bz, b.mass, b.par, b.cov, b.q,
                     b.hpos[:L], b.hcov[:L], None, want_trace=True)
    Cs = O.unpack_cov21(b.cov.astype(np.float64))
    Vs = O.unpack_cov6(b.hcov[:L])                 # [n][L][3][3]
    for i in range(b.n):
        assert r["status"][i] == 0
        hits = b.hpos[:L, :, i].astype(np.float64)
        x, Cx, cost = _batch_wls(b.par[:, i].astype(np.float64), Cs[i], r["trace"][i], hits, Vs[i])
        np.testing.assert_allclose(r["par"][:, i], x, rtol=1e-9, atol=1e-9)
        scale = np.sqrt(np.outer(np.diag(Cx).clip(1e-30), np.diag(Cx).clip(1e-30)))
        blk = np.max(np.abs(Cx))
        assert np.max(np.abs(r["cov"][i] - Cx)) < 1e-8 * blk, np.max(np.abs(r["cov"][i] - Cx) / scale)
        assert r["chi2"][i] == pytest.approx(cost, rel=1e-8, abs=1e-9)


# ------------------------------------------------------------------------------------ P5 / P6
@pytest.fixture(scope="module")
def cfg1_fit():
    b = W.make_fit_batch(1)
    return b, O.fit_batch(b, nthreads=4)


def test_P5_covariance_symmetric_psd_rank5(cfg1_fit):
    b, r = cfg1_fit
    C = r["cov"][:2000]
    assert np.array_equal(C, np.swapaxes(C, 1, 2))
    w, v = np.linalg.eigh(C)
    lmax = w[:, -1]
    assert np.all(np.abs(w[:, 0]) < 1e-12 * lmax)          # exactly one (numerically) null direction
    assert np.all(w[:, 1] > 0)
    # ... and it is the radial position direction of the fitted point
    pos = r["par"][:2, :2000].T
    rad = pos / np.linalg.norm(pos, axis=1, keepdims=True)
    null = v[:, :, 0]
    assert np.all(np.abs(np.abs(np.einsum("ni,ni->n", null[:, :2], rad)) - 1.0) < 1e-6)
    assert np.all(np.abs(null[:, 2:]) < 1e-5)


def test_P6_pulls_and_chi2(cfg1_fit):
    b, r = cfg1_fit
    ndf = 2 * r["nhits"] - 5
    good = (r["status"] == 0) & (r["chi2"] <= ndf + 9 * np.sqrt(2.0 * ndf))
    assert (~good).mean() < 1e-3                             # A14: diverged tracks are rare
    x, C, truth = r["par"][:, good], r["cov"][good], b.truth[-1][:, good]
    d = x - truth
    phi = np.arctan2(x[1], x[0])
    tvec = np.stack([-np.sin(phi), np.cos(phi)])
    pulls = {
        "t": (d[0] * tvec[0] + d[1] * tvec[1]) / np.sqrt(np.einsum("in,nij,jn->n", tvec, C[:, :2, :2], tvec)),
        "z": d[2] / np.sqrt(C[:, 2, 2]),
        "px": d[3] / np.sqrt(C[:, 3, 3]), "py": d[4] / np.sqrt(C[:, 4, 4]), "pz": d[5] / np.sqrt(C[:, 5, 5]),
    }
    for name, p in pulls.items():
        assert abs(p.mean()) < 0.03, (name, p.mean())
        assert 0.95 < p.std() < 1.10, (name, p.std())
    c = r["chi2"][good] / ndf[good]
    assert 0.97 < c.mean() < 1.10
    assert 0.8 < np.var(r["chi2"][good]) / (2 * ndf[good].mean()) < 1.3


# ------------------------------------------------------------------------------------ P10
def test_P10_rotation_about_z():
    cfg = W.get_config(1)
    b = W.simulate_event(cfg, 11, n_tracks=50, dtype=np.float64)
    beta = 0.7312
    c, s = math.cos(beta), math.sin(beta)
    R3 = np.array([[c, -s, 0], [s, c, 0], [0, 0, 1.0]])
    R6 = np.zeros((6, 6)); R6[:3, :3] = R3; R6[3:, 3:] = R3
    par2 = R6 @ b.par
    cov2 = O.pack_cov21(np.einsum("ij,njk,lk->nil", R6, O.unpack_cov21(b.cov), R6))
    hpos2 = np.einsum("ij,ljn->lin", R3, b.hpos)
    V = O.unpack_cov6(b.hcov)                                 # [n][L][3][3]
    V2 = np.einsum("ij,nljk,mk->nlim", R3, V, R3)
    hcov2 = np.stack([V2[:, :, 0, 0], V2[:, :, 0, 1], V2[:, :, 0, 2], V2[:, :, 1, 1], V2[:, :, 1, 2], V2[:, :, 2, 2]])
    hcov2 = np.transpose(hcov2, (2, 0, 1))                    # [L][6][n]
    r1 = O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask)
    r2 = O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, par2, cov2, b.q, hpos2, hcov2, b.mask)
    np.testing.assert_allclose(r2["par"], R6 @ r1["par"], rtol=0, atol=1e-10)
    np.testing.assert_allclose(r2["cov"], np.einsum("ij,njk,lk->nil", R6, r1["cov"], R6), rtol=1e-8, atol=1e-13)
    np.testing.assert_allclose(r2["chi2"], r1["chi2"], rtol=1e-10)


# ------------------------------------------------------------------------------------ regression anchor
def test_oracle_fit_matches_its_stored_values():
    """tests/golden/oracle_fit_config1_8tracks.txt was written by tests/golden/make_oracle_fit_golden.py
    (oracle only).  It does not pin the oracle to the mathematics -- P1..P10 and S1..S4 do -- it makes a
    change of the oracle's arithmetic visible."""
    import importlib.util
    spec = importlib.util.spec_from_file_location("mk", os.path.join(GOLD, "make_oracle_fit_golden.py"))
    mk = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mk)
    want = np.loadtxt(os.path.join(GOLD, "oracle_fit_config1_8tracks.txt"))
    np.testing.assert_allclose(mk.compute(), want, rtol=1e-10, atol=1e-12)
