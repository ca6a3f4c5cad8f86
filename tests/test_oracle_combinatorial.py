"""Pins of the oracle's combinatorial building (reading A19; CPU only).
C1 with one candidate per seed it is the best-hit builder except for the 'no hit' preference;
C2 the surviving best track is never worse than best-hit's (more hits, or equal hits and lower chi2);
C3 brute force on tiny inputs: exhaustive enumeration of all hit assignments gives the same best track;
C4 efficiency: with more candidates the true hit list is found more often."""
import itertools

import numpy as np
import pytest

from oracle import kf_oracle as O
from workloads import barrel_events as W

NE, NP = 40, 64
EMAX = float(np.float32(1.2))


def _setup(n_tracks, noise, seed_layers=3):
    ev = W.make_build_event(4, n_tracks=n_tracks, noise_hits=noise)
    f = ev.fit
    r = O.fit_tracks(f.radius[:seed_layers], f.x_over_X0[:seed_layers], f.Bz, f.mass, f.par, f.cov, f.q,
                     f.hpos[:seed_layers], f.hcov[:seed_layers], None)
    par, cov = r["par"].astype(np.float32), O.pack_cov21(r["cov"]).astype(np.float32)
    layers = []
    for l in range(seed_layers, 10):
        lay = ev.layers[l]
        layers.append((lay.pos, lay.cov, O.bin_hits(lay.pos, lay.radius, NE, NP, EMAX)))
    return ev, par, cov, r["chi2"], r["nhits"], layers


def _best_hit(ev, par, cov, chi2, nh, layers):
    f = ev.fit
    c = O.Candidates(par, cov, f.q, chi2, nh)
    hits = []
    for j, l in enumerate(range(3, 10)):
        rr = O.score_layer(c, ev.layers[l].radius, f.x_over_X0[l], f.Bz, f.mass, layers[j][0], layers[j][1], layers[j][2],
                           NE, NP, EMAX, 2, 30.0, True)
        hits.append(rr["best_hit"])
    return c, np.stack(hits)


def test_C1_C2_one_candidate_is_best_hit_and_more_is_never_worse():
    ev, par, cov, chi2, nh, layers = _setup(300, 3000)
    f = ev.fit
    bh, bh_hits = _best_hit(ev, par, cov, chi2, nh, layers)
    one = O.build_combinatorial(f.radius, f.x_over_X0, f.Bz, f.mass, par, cov, f.q, chi2, nh, 3, layers, NE, NP, EMAX, 2, 30.0, 1)
    # with n_cand = 1 the child with a hit (nhits + 1) always outranks "no hit": exactly best-hit building
    assert np.array_equal(one["hits"], bh_hits)
    np.testing.assert_allclose(one["chi2"], bh.chi2, rtol=1e-12)
    assert np.array_equal(one["nhits"], bh.nhits)
    np.testing.assert_allclose(one["par"], bh.par.T, rtol=0, atol=1e-12)
    four = O.build_combinatorial(f.radius, f.x_over_X0, f.Bz, f.mass, par, cov, f.q, chi2, nh, 3, layers, NE, NP, EMAX, 2, 30.0, 4)
    better = (four["nhits"] > one["nhits"]) | ((four["nhits"] == one["nhits"]) & (four["chi2"] <= one["chi2"] + 1e-9))
    assert np.all(better)
    assert np.all(four["n_cand"] >= 1) and np.all(four["n_cand"] <= 4) and np.all(four["margin"] >= 0)


def test_C3_brute_force_enumeration_tiny():
    """2 layers, a handful of hits: enumerate every assignment (hit or none per layer), rank by the same key."""
    ev, par, cov, chi2, nh, layers = _setup(40, 150)
    f = ev.fit
    two = layers[:2]
    res = O.build_combinatorial(f.radius, f.x_over_X0, f.Bz, f.mass, par, cov, f.q, chi2, nh, 3, two, NE, NP, EMAX, 2, 30.0, 8)
    for i in range(40):
        u0 = par[:, i].astype(np.float64)
        C0 = O.unpack_cov21(cov[:, i:i + 1].astype(np.float64))[0]
        best = None

        def options(u, Cm, j):
            """every child of (u, Cm) on build layer j: (hit or -1, state, covariance, chi2 increment, hits added)"""
            l = 3 + j
            rc, up, F, _, _ = O.propagate(u, float(f.q[i]), f.Bz, float(f.radius[l]))
            assert rc == 0
            Cp = O.transport_cov(F, Cm, O.process_noise(up, f.mass, float(f.x_over_X0[l])))
            opts = [(-1, up, Cp, 0.0, 0)]
            hp, hc, bins = two[j]
            cb = O.bin_index_def(up[0], up[1], up[2], float(f.radius[l]), NE, NP, EMAX)
            ie, ip = cb // NP, cb % NP
            Vs = O.unpack_cov6(hc)
            for de in range(-2, 3):
                e = ie + de
                if e < 0 or e >= NE:
                    continue
                for dp in range(-2, 3):
                    b = e * NP + (ip + dp) % NP
                    for s in range(bins["bin_offset"][b], bins["bin_offset"][b + 1]):
                        h = int(bins["sorted_to_orig"][s])
                        rc2, c = O.chi2_increment(up, Cp, hp[:, h].astype(np.float64), Vs[h])
                        if rc2 == 0 and c < 30.0:
                            _, un, Cn, cc = O.update(up, Cp, hp[:, h].astype(np.float64), Vs[h])
                            opts.append((h, un, Cn, cc, 1))
            return opts
        for (h0, u1, C1, c0, k0) in options(u0, C0, 0):
            for (h1, u2, C2, c1, k1) in options(u1, C1, 1):
                key = (-(nh[i] + k0 + k1), chi2[i] + c0 + c1)
                if best is None or key < best[0]:
                    best = (key, (h0, h1))
        # with n_cand = 8 and so few compatible hits nothing is truncated: the builder must find the optimum
        assert (res["hits"][0, i], res["hits"][1, i]) == best[1], i
        assert res["nhits"][i] == -best[0][0] and res["chi2"][i] == pytest.approx(best[0][1], rel=1e-12)


def test_C4_more_candidates_find_the_true_track_more_often():
    ev, par, cov, chi2, nh, layers = _setup(1500, 30000)
    f = ev.fit
    truth = np.stack([ev.layers[l].true_index for l in range(3, 10)])
    eff = []
    for nc in (1, 4):
        r = O.build_combinatorial(f.radius, f.x_over_X0, f.Bz, f.mass, par, cov, f.q, chi2, nh, 3, layers, NE, NP, EMAX, 2, 30.0, nc)
        eff.append((r["hits"] == truth).all(axis=0).mean())
    assert eff[1] >= eff[0] and eff[1] > 0.5
