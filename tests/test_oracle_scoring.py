"""Pins of the oracle's hit binning and best-hit scoring (CPU only).
P9 bin structure, single-precision bin rule == definition away from edges, P8 window == brute force."""
import numpy as np
import pytest

from oracle import kf_oracle as O
from workloads import barrel_events as W

NE, NP, EMAX = 40, 64, 1.2


@pytest.fixture(scope="module")
def small_event():
    return W.make_build_event(4, n_tracks=400, noise_hits=2000)


def test_bin_rule_f32_equals_definition_away_from_edges():
    rng = np.random.default_rng(5)
    r = 16.0
    n = 20000
    eta = rng.uniform(-1.3, 1.3, n)
    phi = rng.uniform(-np.pi, np.pi, n)
    x, y, z = (r * np.cos(phi)).astype(np.float32), (r * np.sin(phi)).astype(np.float32), (r * np.sinh(eta)).astype(np.float32)
    n_edge = 0
    for i in range(n):
        bd = O.bin_index_def(x[i], y[i], z[i], r, NE, NP, EMAX)
        bf = O.bin_index_f32(x[i], y[i], z[i], r, NE, NP, EMAX)
        if bd != bf:      # allowed only within float rounding of an edge
            e = np.arcsinh(float(z[i]) / r); p = np.arctan2(float(y[i]), float(x[i]))
            fe = (e + EMAX) / (2 * EMAX / NE); fp = (p + np.pi) / (2 * np.pi / NP)
            assert min(abs(fe - round(fe)), abs(fp - round(fp))) < 1e-4
            n_edge += 1
    assert n_edge < 10


def test_bin_rule_on_a_disc_layer():
    """Reading A24: radius 0 = a disc layer, the bins stay projective with eta from the point's own rho.  The
    definition with radius 0 is the textbook pseudorapidity of the point, -ln tan(theta / 2); the single-precision
    rule agrees with it away from bin edges; a point's bin does not depend on which surface it is said to lie on
    when that surface is the cylinder through it."""
    rng = np.random.default_rng(6)
    n = 20000
    NEd, EMd = 50, 2.5
    zd = 45.0
    rho = rng.uniform(4.0, 26.0, n)
    phi = rng.uniform(-np.pi, np.pi, n)
    sign = rng.choice([-1.0, 1.0], n)
    x, y, z = (rho * np.cos(phi)).astype(np.float32), (rho * np.sin(phi)).astype(np.float32), (sign * zd).astype(np.float32)
    n_edge = 0
    for i in range(n):
        xd, yd, zz = float(x[i]), float(y[i]), float(z[i])
        bd = O.bin_index_def(xd, yd, zz, 0.0, NEd, NP, EMd)
        theta = np.arctan2(np.hypot(xd, yd), zz)
        eta = -np.log(np.tan(0.5 * theta))
        ie = int(np.clip(np.floor((eta + EMd) / (2 * EMd / NEd)), 0, NEd - 1))
        ip = int(np.floor((np.arctan2(yd, xd) + np.pi) / (2 * np.pi / NP))) % NP
        fe = (eta + EMd) / (2 * EMd / NEd)
        if abs(fe - round(fe)) > 1e-9:
            assert bd == ie * NP + ip
        assert bd == O.bin_index_def(xd, yd, zz, np.hypot(xd, yd), NEd, NP, EMd)
        bf = O.bin_index_f32(x[i], y[i], z[i], 0.0, NEd, NP, EMd)
        if bd != bf:
            fp = (np.arctan2(yd, xd) + np.pi) / (2 * np.pi / NP)
            assert min(abs(fe - round(fe)), abs(fp - round(fp))) < 1e-4
            n_edge += 1
    assert n_edge < 10
    # the sort itself: stable counting sort by that rule
    pos = np.stack([x, y, z])
    ob = O.bin_hits(pos, 0.0, NEd, NP, EMd)
    assert np.array_equal(np.sort(ob["sorted_to_orig"]), np.arange(n))
    b = np.array([O.bin_index_f32(x[i], y[i], z[i], 0.0, NEd, NP, EMd) for i in range(0, n, 37)])
    assert np.array_equal(ob["bin_of"][::37], b)
    assert np.all(np.diff(ob["bin_of"][ob["sorted_to_orig"]]) >= 0)
    same = np.diff(ob["bin_of"][ob["sorted_to_orig"]]) == 0
    assert np.all(np.diff(ob["sorted_to_orig"])[same] > 0)


def test_bin_rule_special_directions():
    r = 10.0
    f = lambda x, y, z=0.0: O.bin_index_f32(x, y, z, r, NE, NP, EMAX)
    d = lambda x, y, z=0.0: O.bin_index_def(x, y, z, r, NE, NP, EMAX)
    for (x, y) in [(10, 0), (0.1, 10), (-0.1, -10), (-10, 0), (-10, -0.0), (7, 6.9), (-7, 7.1), (-7.1, -7), (6.9, -7), (-10, 1e-3), (-10, -1e-3)]:
        assert f(x, y) == d(x, y), (x, y)
    assert f(10, 0) % NP == 32 and f(-10, 0) % NP == 0 and f(-10, 1e-3) % NP == 63
    # eta clamps
    assert f(10, 0, 1e6) // NP == NE - 1 and f(10, 0, -1e6) // NP == 0 and f(10, 0, 0.0) // NP == NE // 2


def test_P9_bin_structure(small_event):
    ev = small_event
    for l in (0, 5, 9):
        lay = ev.layers[l]
        H = lay.pos.shape[1]
        b = O.bin_hits(lay.pos, lay.radius, NE, NP, EMAX)
        off, s2o, bof = b["bin_offset"], b["sorted_to_orig"], b["bin_of"]
        assert off[0] == 0 and off[-1] == H and np.all(np.diff(off) >= 0)
        assert np.array_equal(np.sort(s2o), np.arange(H))                  # a permutation
        sb = bof[s2o]
        assert np.all(np.diff(sb) >= 0)                                    # sorted by bin
        for k in range(NE * NP):
            seg = s2o[off[k]:off[k + 1]]
            assert np.all(sb[off[k]:off[k + 1]] == k)
            assert np.all(np.diff(seg) > 0)                                # stable
    e = O.bin_hits(np.zeros((3, 0), dtype=np.float32), 4.0, NE, NP, EMAX)  # empty layer
    assert np.all(e["bin_offset"] == 0) and e["sorted_to_orig"].size == 0


def _seeds_from_first_three(ev):
    f = ev.fit
    r = O.fit_tracks(f.radius[:3], f.x_over_X0[:3], f.Bz, f.mass, f.par, f.cov, f.q, f.hpos[:3], f.hcov[:3], None)
    par = r["par"].astype(np.float32)
    cov = O.pack_cov21(r["cov"]).astype(np.float32)
    return par, cov, r["chi2"], r["nhits"]


def test_P8_window_scoring_equals_brute_force(small_event):
    ev = small_event
    f = ev.fit
    par, cov, chi2, nh = _seeds_from_first_three(ev)
    a = O.Candidates(par, cov, f.q, chi2, nh)
    b = O.Candidates(par, cov, f.q, chi2, nh)
    n_acc = 0
    for l in range(3, 10):
        lay = ev.layers[l]
        bins = O.bin_hits(lay.pos, lay.radius, NE, NP, EMAX)
        ra = O.score_layer(a, lay.radius, f.x_over_X0[l], f.Bz, f.mass, lay.pos, lay.cov, bins, NE, NP, EMAX)
        rb = O.score_layer(b, lay.radius, f.x_over_X0[l], f.Bz, f.mass, lay.pos, lay.cov, None, NE, NP, EMAX, all_hits=True)
        acc = rb["best_hit"] >= 0
        assert np.array_equal(ra["best_hit"], rb["best_hit"])
        assert np.array_equal(ra["best_chi2"][acc], rb["best_chi2"][acc])
        assert np.all(ra["best_chi2"][~acc] >= 30.0)
        n_acc += acc.sum()
        # with only 2400 hits per layer the true hit is nearly always the best one
        assert (ra["best_hit"] == lay.true_index).mean() > 0.9
    np.testing.assert_array_equal(a.par, b.par)
    np.testing.assert_array_equal(a.cov, b.cov)
    assert n_acc > 0.9 * 7 * f.n
    assert np.all(a.nhits[a.status == 0] <= 10)


def test_scoring_reject_and_no_update(small_event):
    ev = small_event
    f = ev.fit
    par, cov, chi2, nh = _seeds_from_first_three(ev)
    lay = ev.layers[3]
    bins = O.bin_hits(lay.pos, lay.radius, NE, NP, EMAX)
    a = O.Candidates(par, cov, f.q, chi2, nh)
    r0 = O.score_layer(a, lay.radius, f.x_over_X0[3], f.Bz, f.mass, lay.pos, lay.cov, bins, NE, NP, EMAX, chi2_cut=0.0)
    assert np.all(r0["best_hit"] == -1) and np.array_equal(a.nhits, nh) and np.array_equal(a.chi2, chi2)
    # rejected candidates carry the propagated state: they sit on the layer
    np.testing.assert_allclose(np.hypot(a.par[:, 0], a.par[:, 1]), lay.radius, rtol=1e-12)
    b = O.Candidates(par, cov, f.q, chi2, nh)
    r1 = O.score_layer(b, lay.radius, f.x_over_X0[3], f.Bz, f.mass, lay.pos, lay.cov, bins, NE, NP, EMAX, do_update=False)
    assert (r1["best_hit"] >= 0).mean() > 0.9
    np.testing.assert_array_equal(a.par, b.par)          # do_update=0 leaves the propagated state too
    np.testing.assert_array_equal(b.nhits, nh)


def test_chi2_increment_equals_its_definition_and_the_update():
    """orc_chi2_increment is what every accept / cut / ranking decision rests on (reading A8):
    chi2 = r^T (C'_pp + V)^-1 r with r = m - H u.  Pinned against (i) the definition evaluated by numpy on the
    same numbers (a dropped V, a wrong block of C or a transposed index changes it), (ii) the chi2 that orc_update
    returns for the same inputs (which pin P4 ties to the batch weighted least squares), (iii) the closed form for
    a diagonal case, and (iv) S_NOT_PD on an S that is not positive definite."""
    rng = np.random.default_rng(17)
    for it in range(1200):
        u = rng.normal(size=6) * np.array([20, 20, 20, 3, 3, 3])
        # C': symmetric PSD of rank 5 with a general null direction (as the to-radius transport leaves it),
        # with position / momentum scales far apart and full correlations
        A = rng.normal(size=(6, 5)) * np.array([3e-2, 3e-2, 1e-1, 0.3, 0.3, 0.3])[:, None]
        Cm = A @ A.T
        B = rng.normal(size=(3, 3)) * np.array([0.1, 0.01, 0.1])[:, None]
        V = B @ B.T + 1e-6 * np.eye(3)
        m = u[:3] + rng.normal(size=3) * 0.2
        rc, c = O.chi2_increment(u, Cm, m, V)
        assert rc == 0
        r = m - u[:3]
        want = r @ np.linalg.solve(Cm[:3, :3] + V, r)
        assert c == pytest.approx(want, rel=1e-10)
        rc2, _, _, c2 = O.update(u, Cm, m, V)
        assert rc2 == 0 and c2 == pytest.approx(c, rel=1e-13)
        # sensitivity: the same call with V dropped, or with the momentum block in place of the position block,
        # gives a different number (so the two checks above would catch either slip)
        if it < 50:
            assert abs(r @ np.linalg.solve(Cm[:3, :3] + 1e-9 * np.eye(3), r) - c) > 1e-6 * c
            assert abs(r @ np.linalg.solve(Cm[3:, 3:] + V, r) - c) > 1e-6 * c
    # closed form: diagonal C and V -> sum of squared pulls
    u = np.array([1.0, 2.0, 3.0, 0.5, 0.5, 0.5])
    Cd = np.diag([0.04, 0.09, 0.16, 1.0, 1.0, 1.0])
    Vd = np.diag([0.05, 0.07, 0.09])
    m = np.array([1.3, 1.6, 3.5])
    rc, c = O.chi2_increment(u, Cd, m, Vd)
    assert rc == 0 and c == pytest.approx(0.3 ** 2 / 0.09 + 0.4 ** 2 / 0.16 + 0.5 ** 2 / 0.25, rel=1e-13)
    # S not positive definite (det <= 0): refused, by the increment and by the update alike
    Vbad = np.diag([-1.0, 0.07, 0.09])
    assert O.chi2_increment(u, Cd, m, Vbad)[0] == O.S_NOT_PD
    assert O.update(u, Cd, m, Vbad)[0] == O.S_NOT_PD
    assert O.chi2_increment(u, np.zeros((6, 6)), m, np.zeros((3, 3)))[0] == O.S_NOT_PD
