"""Degenerate and extreme shapes of every hot call, against the oracle: one scored layer, one candidate, one seed,
one- and two-layer indexed fits, chunk boundaries of the host path, 32 layers binned in one call, the widest and
the narrowest candidate window.  (The smoother once hung on geometries with fewer layers than its hit ring has
stages; these cases exist so that a shape nobody benchmarks cannot do that again.)"""
import copy
import dataclasses

import numpy as np
import pytest
import torch

from oracle import kf_oracle as O
from tests import test_comb_gpu as C
from tests import test_pipeline_gpu as P
from tests import test_score_gpu as S
from tests.parity import compare_fit
from workloads import barrel_events as W

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(300)]
NE, NP, EMAX = S.NE, S.NP, S.EMAX


@pytest.fixture(scope="module")
def ctx():
    import paper_1705_02876_b200 as K
    c = K.KFContext(0)
    yield c
    c.close()


@pytest.mark.parametrize("n_tracks,noise,first", [(1, 50, 3), (33, 200, 9), (1, 0, 9), (400, 2000, 8)])
def test_best_hit_building_small_shapes(ctx, n_tracks, noise, first):
    """One candidate; one scored layer; a layer pool holding the single true hit only."""
    ev = W.make_build_event(4, n_tracks=n_tracks, noise_hits=noise)
    ev.cfg = dataclasses.replace(ev.cfg, first_scored_layer=first)
    n_dec, _ = S._build_event_fused(ctx, ev, use_order=(n_tracks > 1))
    assert n_dec >= 0.9 * n_tracks * (10 - first)


@pytest.mark.parametrize("n_tracks,noise,n_cand,first", [(1, 50, 4, 3), (33, 200, 8, 9), (33, 200, 1, 9), (1, 0, 8, 9)])
def test_combinatorial_building_small_shapes(ctx, n_tracks, noise, n_cand, first):
    ev, g, idx, nf, o = C._run(ctx, n_tracks, noise, n_cand, first=first)
    same = (idx == o["hits"]).all(axis=0)
    clear = o["margin"] >= C.MARGIN
    assert not np.any(~same & clear)
    sel = same & clear
    assert np.array_equal(g["nhits"][sel], o["nhits"][sel]) and np.array_equal(g["status"][sel], o["status"][sel])
    assert np.array_equal(nf[sel], o["n_cand"][sel])
    np.testing.assert_allclose(g["chi2"][sel], o["chi2"][sel], rtol=2e-3, atol=2e-3)


def _truncate(ev, k):
    """The first k layers of a build event (pools, geometry and per-track hits)."""
    ev = copy.copy(ev)
    ev.layers = ev.layers[:k]
    f = copy.copy(ev.fit)
    f.radius, f.x_over_X0 = f.radius[:k], f.x_over_X0[:k]
    f.hpos, f.hcov = np.ascontiguousarray(f.hpos[:k]), np.ascontiguousarray(f.hcov[:k])
    f.mask = f.mask & np.uint32((1 << k) - 1)
    ev.fit = f
    return ev


@pytest.mark.parametrize("k,n_tracks", [(1, 1), (1, 257), (2, 33), (3, 1000)])
def test_indexed_fit_short_geometries(ctx, k, n_tracks):
    ev = _truncate(W.make_build_event(4, n_tracks=n_tracks, noise_hits=5 * n_tracks), k)
    truth = np.stack([l.true_index for l in ev.layers])
    o = P._oracle_fit_with(ev, truth)
    for rec in (False, True):
        g = P._fit_indexed(ctx, ev, truth, use_records=rec)
        assert np.array_equal(g["nhits"], o["nhits"]) and np.array_equal(g["status"], o["status"])
        compare_fit(g, o, float(ev.fit.radius[-1]), max_diverged_frac=1.0)


@pytest.mark.parametrize("n,k", [(1, 1), (131_072, 2), (131_073, 10), (5, 10), (1000, 32)])
def test_host_path_chunk_boundaries(ctx, n, k):
    """kf_fit_tracks_host cuts the batch into chunks (a multiple of 1024 tracks, their number grows with the square
    root of the batch): two whole chunks of 65 536, two ragged ones (66 560 + 64 513), a single track, a one-layer
    geometry -- same results as the resident call."""
    from paper_1705_02876_b200.buffers import DeviceFit
    cfg = dataclasses.replace(W.get_config(1), n_layers=k, n_tracks=n, layer_step_cm=4.0 if k <= 10 else 1.25)
    b = W.simulate_event(cfg, 31, n_tracks=n)
    d = DeviceFit.from_batch(b, "cuda:0")
    d.fit(ctx)
    torch.cuda.synchronize()
    r = d.results()
    h = _host_fit(ctx, b)
    assert np.array_equal(h["nhits"], r["nhits"]) and np.array_equal(h["status"], r["status"])
    o = O.fit_batch(b)
    compare_fit(h, o, float(b.radius[-1]), max_diverged_frac=1.0)


def _host_fit(ctx, b):
    """The host-buffer call on pinned tensors (what bench.py's e2e arm does)."""
    from paper_1705_02876_b200.buffers import DeviceFit
    h = DeviceFit.from_batch(b, "cpu", pin=True)
    h.fit_host(ctx)
    return h.results()


@pytest.mark.parametrize("chunked", [2, 1])
def test_bin_32_layers_in_one_call(ctx, chunked):
    """KF_MAX_LAYERS pools in one kf_bin_layers call (one launch group), ragged sizes (1 to 3 chunks of the
    chunked sort per pool), one empty pool; both forms of the sort."""
    import paper_1705_02876_b200 as K
    ctx.set_option(K.OPT_BIN_FORM, chunked)       # 2 = chunked sort wherever it applies, 1 = five-launch sort
    from paper_1705_02876_b200.buffers import DeviceLayer
    rng = np.random.default_rng(41)
    pools, radii = [], []
    for l in range(32):
        H = 0 if l == 17 else int(rng.integers(1, 6000))
        r = 2.5 * (l + 1)
        phi, eta = rng.uniform(-np.pi, np.pi, H), rng.uniform(-1.3, 1.3, H)
        pos = np.stack([r * np.cos(phi), r * np.sin(phi), r * np.sinh(eta)]).astype(np.float32)
        cov = rng.uniform(1e-4, 1e-2, (6, H)).astype(np.float32)
        pools.append((pos, cov)); radii.append(r)
    dls = [DeviceLayer.from_numpy(p, c, NE, NP, EMAX, "cuda:0") for p, c in pools]
    try:
        ctx.bin_layers(radii, [(d.n_hits, d.pos, d.cov, d.bins) for d in dls])
    finally:
        ctx.set_option(K.OPT_BIN_FORM, K.BIN_FORM_AUTO)
    torch.cuda.synchronize()
    for l, (d, (pos, cov)) in enumerate(zip(dls, pools)):
        ob = O.bin_hits(pos, radii[l], NE, NP, EMAX)
        if l == 17:
            assert np.all(d.bins.bin_offset.cpu().numpy() == 0)
        else:
            S._assert_bins_equal(d, ob, pos, cov)


@pytest.mark.parametrize("window_half", [0, 31])
def test_score_narrowest_and_widest_window(ctx, window_half):
    """window_half = 0 (the candidate's own bin) and 31 (63 of the 64 phi bins, every eta row): same decisions as
    the oracle with the same window."""
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceCandidates, DeviceLayer
    ev = W.make_build_event(4, n_tracks=300, noise_hits=3000)
    f = ev.fit
    par, cov, chi2, nh = S._seeds(ev)
    geom = K.Geometry(f.radius, f.x_over_X0, f.Bz, f.mass)
    dc = DeviceCandidates.from_numpy(par, cov, f.q, chi2, nh, "cuda:0")
    oc = O.Candidates(par, cov, f.q, chi2, nh)
    lay = ev.layers[3]
    dl = DeviceLayer.from_numpy(lay.pos, lay.cov, NE, NP, EMAX, "cuda:0")
    dl.bin(ctx, lay.radius)
    dc.score(ctx, geom, 3, dl, window_half, 30.0, True)
    torch.cuda.synchronize()
    ob = O.bin_hits(lay.pos, lay.radius, NE, NP, EMAX)
    orr = O.score_layer(oc, lay.radius, f.x_over_X0[3], f.Bz, f.mass, lay.pos, lay.cov, ob, NE, NP, EMAX,
                        window_half, 30.0, True)
    g = dc.results()
    diff = g["best_hit"] != orr["best_hit"]
    b, s2 = orr["best_chi2"], orr["second_chi2"]
    with np.errstate(invalid="ignore"):
        tie = (np.abs(s2 - b) <= 1e-4 * np.abs(b)) | (np.abs(b - 30.0) <= 1e-4 * 30.0)
    if window_half == 0:
        # fp32 against fp64 may put a candidate sitting on a bin edge into the neighbouring bin, which with a
        # one-bin window IS the whole window (A16b covers windows of >= 2 bins): allow a handful
        assert int((diff & ~tie).sum()) <= 3
    else:
        assert not np.any(diff & ~tie)
    assert (g["best_hit"] >= 0).mean() > 0.5
