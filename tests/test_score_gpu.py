"""GPU parity of kf_bin_hits (bit-exact) and kf_score_candidates (indices identical except inside the
1e-4 relative chi2 tie window of north_star) against the oracle, through the C ABI."""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as O
from tests.parity import compare_fit
from workloads import barrel_events as W

pytestmark = pytest.mark.gpu
NE, NP = 40, 64
EMAX = float(np.float32(1.2))        # both sides see the same fp32-rounded eta_max (reading A17)


@pytest.fixture(scope="module")
def ctx():
    import paper_1705_02876_b200 as K
    c = K.KFContext(0)
    yield c
    c.close()


@pytest.fixture(params=["chunked", "five_launch"])
def sort_path(request, ctx):
    """Both forms of the counting sort: the chunked one (taken for calls of >= 196 608 hits) and the five-launch
    one (small calls, more than 8192 bins).  kf_set_option(KF_OPT_BIN_FORM) forces either for any size."""
    import paper_1705_02876_b200 as K
    ctx.set_option(K.OPT_BIN_FORM, K.BIN_FORM_FIVE_LAUNCH if request.param == "five_launch" else K.BIN_FORM_CHUNKED)
    yield request.param
    ctx.set_option(K.OPT_BIN_FORM, K.BIN_FORM_AUTO)


def _bin_both(ctx, pos, cov, radius, ne=NE, nph=NP, emax=EMAX):
    from paper_1705_02876_b200.buffers import DeviceLayer
    dl = DeviceLayer.from_numpy(pos, cov, ne, nph, emax, "cuda:0")
    dl.bin(ctx, radius)
    torch.cuda.synchronize()
    return dl, O.bin_hits(pos, radius, ne, nph, emax)


def _assert_bins_equal(dl, ob, pos, cov):
    H = dl.n_hits
    assert np.array_equal(dl.bins.bin_offset.cpu().numpy(), ob["bin_offset"])
    s2o = dl.bins.sorted_to_orig.cpu().numpy()[:H]
    assert np.array_equal(s2o, ob["sorted_to_orig"])
    assert np.array_equal(dl.bins.pos_sorted.cpu().numpy()[:, :H], pos[:, s2o])
    assert np.array_equal(dl.bins.cov_sorted.cpu().numpy()[:, :H], cov[:, s2o])
    rec = dl.bins.hit_rec.cpu().numpy()[:H]
    cs = cov[:, s2o].T                                      # xx xy xz yy yz zz
    assert np.array_equal(rec[:, 0:3], pos[:, s2o].T) and np.array_equal(rec[:, 3], cs[:, 5])
    assert np.array_equal(rec[:, 4:7], cs[:, [0, 1, 3]]) and np.array_equal(rec[:, 8:10], cs[:, [2, 4]])
    assert np.array_equal(rec[:, 7].copy().view(np.int32), s2o)
    o2s = dl.bins.orig_to_sorted.cpu().numpy()[:H]
    assert np.array_equal(o2s[s2o], np.arange(H))
    box = dl.bins.bin_box.cpu().numpy()
    off = ob["bin_offset"]
    for b in np.flatnonzero(np.diff(off) > 0)[::7]:               # every 7th non-empty bin
        seg = s2o[off[b]:off[b + 1]]
        want = [pos[0, seg].min(), pos[0, seg].max(), pos[1, seg].min(), pos[1, seg].max(), pos[2, seg].min(),
                pos[2, seg].max(), max(cov[5, seg].max(), 0.0), max((cov[0, seg] + cov[3, seg]).max(), 0.0)]
        assert np.array_equal(box[b], np.array(want, dtype=np.float32)), (b, box[b], want)
    empty = np.flatnonzero(np.diff(off) == 0)
    assert np.all(np.isposinf(box[empty][:, [0, 2, 4]])) and np.all(np.isneginf(box[empty][:, [1, 3, 5]]))


@pytest.mark.parametrize("n_tracks,noise", [(400, 2000), (20000, 100000)])
def test_bin_hits_bit_exact(ctx, n_tracks, noise, sort_path):
    ev = W.make_build_event(4, n_tracks=n_tracks, noise_hits=noise)
    for l in (0, 4, 9):
        lay = ev.layers[l]
        dl, ob = _bin_both(ctx, lay.pos, lay.cov, lay.radius)
        _assert_bins_equal(dl, ob, lay.pos, lay.cov)


def test_bin_hits_edge_cases(ctx, sort_path):
    rng = np.random.default_rng(11)
    r = 12.0
    cov = np.tile(np.array([1e-2, 0, 0, 1e-2, 0, 1e-2], dtype=np.float32)[:, None], (1, 5000))
    # empty layer
    dl, ob = _bin_both(ctx, np.zeros((3, 0), np.float32), np.zeros((6, 0), np.float32), r)
    assert np.all(dl.bins.bin_offset.cpu().numpy() == 0) and np.all(ob["bin_offset"] == 0)
    # every hit in one bin (the ranking step degenerates to one long segment), 1 hit, ragged counts
    for H in (1, 3, 5000):
        pos = np.stack([np.full(H, r), np.full(H, 0.01), np.full(H, 0.3)]).astype(np.float32)
        dl, ob = _bin_both(ctx, pos, cov[:, :H], r)
        _assert_bins_equal(dl, ob, pos, cov[:, :H])
    # hits exactly on bin edges and on the axes, out-of-range eta (clamped), phi = +-pi
    phi = np.concatenate([-np.pi + np.arange(64) * (2 * np.pi / 64), [np.pi, -np.pi, 0.0]])
    eta = np.concatenate([-1.2 + np.arange(41) * 0.06, [-5.0, 5.0]])
    P, E = np.meshgrid(phi, eta)
    pos = np.stack([r * np.cos(P.ravel()), r * np.sin(P.ravel()), r * np.sinh(E.ravel())]).astype(np.float32)
    H = pos.shape[1]
    c2 = np.tile(cov[:, :1], (1, H))
    dl, ob = _bin_both(ctx, pos, c2, r)
    _assert_bins_equal(dl, ob, pos, c2)
    # other bin shapes, incl. the largest table
    pos = np.stack([r * np.cos(rng.uniform(-np.pi, np.pi, 3000)), r * np.sin(rng.uniform(-np.pi, np.pi, 3000)),
                    r * np.sinh(rng.uniform(-2.5, 2.5, 3000))]).astype(np.float32)
    # (64 x 128 = 8192 bins: the largest grid the chunked sort takes; 256 x 256 always takes the five-launch form)
    for ne, nph, emax in [(1, 2, 1.0), (7, 10, 2.0), (64, 128, 2.0), (2, 4096, 2.0), (256, 256, 2.5)]:
        dl, ob = _bin_both(ctx, pos, cov[:, :3000], r, ne, nph, float(np.float32(emax)))
        _assert_bins_equal(dl, ob, pos, cov[:, :3000])


def test_bin_hits_large_layer(ctx, sort_path):
    """A layer of 700 000 hits with a full 3 x 3 covariance each (every output plane distinguishable)."""
    H = 700_000
    rng = np.random.default_rng(12)
    r = 20.0
    phi, eta = rng.uniform(-np.pi, np.pi, H), rng.uniform(-1.3, 1.3, H)
    pos = np.stack([r * np.cos(phi), r * np.sin(phi), r * np.sinh(eta)]).astype(np.float32)
    cov = rng.uniform(1e-4, 1e-2, (6, H)).astype(np.float32)
    dl, ob = _bin_both(ctx, pos, cov, r)
    _assert_bins_equal(dl, ob, pos, cov)


def test_bin_hits_against_the_double_definition(ctx, sort_path):
    """Reading A16b makes both sides decide a hit's bin by the same single-precision edge-table rule, which is
    why bin_offset / sorted_to_orig are bit-exact.  THIS test compares the product with the DEFINITION
    (PAPER.md:71 projective bins; reading A16: eta = asinh(z/r), phi = atan2(y, x), evaluated in double by
    orc_bin_index_def): the bin the library gave a hit may differ from the definition's only where the hit lies
    within rounding (1e-6 relative of a bin width ... fp32 carries 6e-8, the edge tables another 6e-8) of a bin
    edge; such hits are counted and must be rare."""
    rng = np.random.default_rng(31)
    H = 300_000
    r = 16.0
    phi, eta = rng.uniform(-np.pi, np.pi, H), rng.uniform(-1.3, 1.3, H)
    pos = np.stack([r * np.cos(phi), r * np.sin(phi), r * np.sinh(eta)]).astype(np.float32)
    # a few hundred hits placed ON edges (to within fp32 rounding), where the two rules may legitimately differ
    k = 600
    pe = -np.pi + rng.integers(0, NP, k) * (2 * np.pi / NP)
    ee = -EMAX + rng.integers(1, NE, k) * (2 * EMAX / NE)
    pos[:, :k] = np.stack([r * np.cos(pe), r * np.sin(pe), r * np.sinh(rng.uniform(-1.1, 1.1, k))]).astype(np.float32)
    pos[:, k:2 * k] = np.stack([r * np.cos(phi[k:2 * k]), r * np.sin(phi[k:2 * k]), r * np.sinh(ee)]).astype(np.float32)
    cov = np.tile(np.array([1e-2, 0, 0, 1e-2, 0, 1e-2], dtype=np.float32)[:, None], (1, H))
    dl, _ = _bin_both(ctx, pos, cov, r)
    off = dl.bins.bin_offset.cpu().numpy()
    s2o = dl.bins.sorted_to_orig.cpu().numpy()[:H]
    gpu_bin = np.empty(H, dtype=np.int64)
    gpu_bin[s2o] = np.repeat(np.arange(NE * NP), np.diff(off))
    # the definition, in double, on the same fp32 inputs (vectorised restatement of orc_bin_index_def, which is
    # called itself on every hit that differs and on a sample)
    x, y, z = (pos[i].astype(np.float64) for i in range(3))
    fe = (np.arcsinh(z / r) + EMAX) / (2 * EMAX / NE)
    fp = (np.arctan2(y, x) + np.pi) / (2 * np.pi / NP)
    def_bin = np.clip(np.floor(fe), 0, NE - 1).astype(np.int64) * NP + (np.floor(fp).astype(np.int64) % NP)
    for i in rng.integers(0, H, 2000):
        assert def_bin[i] == O.bin_index_def(x[i], y[i], z[i], r, NE, NP, EMAX)
    differ = np.flatnonzero(gpu_bin != def_bin)
    for i in differ:
        assert def_bin[i] == O.bin_index_def(x[i], y[i], z[i], r, NE, NP, EMAX)
        d_eta = abs(fe[i] - np.round(fe[i])) if 0.5 < fe[i] < NE - 0.5 else 1.0     # (the outermost edges clamp)
        d_phi = abs(fp[i] - np.round(fp[i]))
        assert min(d_eta, d_phi) < 1e-5, (i, fe[i], fp[i])       # within rounding of an edge (bin widths)
        # ... and the library's bin is the neighbour across that edge
        ge, gp = divmod(int(gpu_bin[i]), NP); de, dp = divmod(int(def_bin[i]), NP)
        assert abs(ge - de) + min((gp - dp) % NP, (dp - gp) % NP) == 1, (i, gpu_bin[i], def_bin[i])
    print(f"bins vs the double definition: {len(differ)} of {H} hits differ, all within 1e-5 bin widths of an edge")
    assert len(differ) <= 2 * k                                   # only hits placed on edges (plus a stray few)
    assert np.count_nonzero(differ >= 2 * k) <= 5


@pytest.mark.parametrize("crowd", [4, 5, 68, 69, 300])
def test_bin_hits_crowded_bins_within_a_chunk(ctx, sort_path, crowd):
    """The count step of the chunked sort ranks a hit inside its chunk from per-bin peer lists (four entries) plus an
    overflow list of 64, and falls back to bucket lists beyond that.  Chunks (2048 consecutive hits) built to sit on
    those boundaries: bins with exactly `crowd` hits in ONE chunk -- 4 (peers only), 5 (one overflow entry), 68
    (overflow list exactly full), 69 (one too many: bucket form), 300 -- next to singly occupied bins, in shuffled
    index order, several chunks, a ragged last one.  Bit-exact against the oracle's serial counting sort."""
    rng = np.random.default_rng(100 + crowd)
    r = 12.0
    H = 5 * 2048 + 777
    phi, eta = rng.uniform(-np.pi, np.pi, H), rng.uniform(-1.19, 1.19, H)
    # per chunk: some bins filled with `crowd` hits each (bin centres, tiny jitter), the rest uniform
    d_eta, d_phi = 2 * EMAX / NE, 2 * np.pi / NP
    for c in range(6):
        lo, hi = c * 2048, min((c + 1) * 2048, H)
        n_crowded = max(1, min(64 // max(crowd - 4, 1), 12)) if crowd > 4 else 20
        idx = rng.permutation(np.arange(lo, hi))
        used = 0
        for b in range(n_crowded):
            if used + crowd > hi - lo:
                break
            ie, ip = int(rng.integers(0, NE)), int(rng.integers(0, NP))
            sel = idx[used:used + crowd]
            used += crowd
            eta[sel] = -EMAX + (ie + 0.5) * d_eta + rng.uniform(-0.2, 0.2, crowd) * d_eta
            phi[sel] = -np.pi + (ip + 0.5) * d_phi + rng.uniform(-0.2, 0.2, crowd) * d_phi
    pos = np.stack([r * np.cos(phi), r * np.sin(phi), r * np.sinh(eta)]).astype(np.float32)
    cov = rng.uniform(1e-4, 1e-2, (6, H)).astype(np.float32)
    dl, ob = _bin_both(ctx, pos, cov, r)
    assert np.diff(ob["bin_offset"]).max() >= crowd
    _assert_bins_equal(dl, ob, pos, cov)


def test_bin_layers_batched_equals_per_layer(ctx, sort_path):
    """kf_bin_layers (all layers in four launches) == kf_bin_hits layer by layer == oracle."""
    from paper_1705_02876_b200.buffers import DeviceLayer
    ev = W.make_build_event(4, n_tracks=2000, noise_hits=9000)
    dls = [DeviceLayer.from_numpy(l.pos, l.cov, NE, NP, EMAX, "cuda:0") for l in ev.layers]
    dls[2] = DeviceLayer.from_numpy(np.zeros((3, 0), np.float32), np.zeros((6, 0), np.float32), NE, NP, EMAX, "cuda:0")
    ctx.bin_layers([l.radius for l in ev.layers], [(d.n_hits, d.pos, d.cov, d.bins) for d in dls])
    torch.cuda.synchronize()
    for i, (d, l) in enumerate(zip(dls, ev.layers)):
        if i == 2:
            assert np.all(d.bins.bin_offset.cpu().numpy() == 0)
            continue
        _assert_bins_equal(d, O.bin_hits(l.pos, l.radius, NE, NP, EMAX), l.pos, l.cov)


def test_order_is_a_stable_bin_sort_and_changes_no_result(ctx):
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceCandidates, DeviceLayer
    ev = W.make_build_event(4, n_tracks=3000, noise_hits=15000)
    f = ev.fit
    par, cov, chi2, nh = _seeds(ev)
    geom = K.Geometry(f.radius, f.x_over_X0, f.Bz, f.mass)
    lay = ev.layers[3]
    dl = DeviceLayer.from_numpy(lay.pos, lay.cov, NE, NP, EMAX, "cuda:0")
    dl.bin(ctx, lay.radius)
    a = DeviceCandidates.from_numpy(par, cov, f.q, chi2, nh, "cuda:0")
    b = DeviceCandidates.from_numpy(par, cov, f.q, chi2, nh, "cuda:0")
    order = b.make_order(ctx, geom, 3, NE, NP, EMAX)
    torch.cuda.synchronize()
    o = order.cpu().numpy()[:f.n]
    assert np.array_equal(np.sort(o), np.arange(f.n))                    # a permutation
    # keys: bin of the oracle-propagated position; sorted by key, ascending index inside a key
    keys = np.empty(f.n, dtype=np.int64)
    for i in range(f.n):
        rc, u, _, _, _ = O.propagate(par[:, i].astype(np.float64), float(f.q[i]), f.Bz, lay.radius, want_F=False)
        keys[i] = O.bin_index_def(u[0], u[1], u[2], lay.radius, NE, NP, EMAX)
    ko = keys[o]
    bad = np.flatnonzero(np.diff(ko) < 0)
    assert len(bad) <= 5                                                  # fp32 vs fp64 at a bin edge only
    same = np.diff(ko) == 0
    assert np.all(np.diff(o)[same] > 0) or len(bad) > 0
    a.score(ctx, geom, 3, dl)
    b.score(ctx, geom, 3, dl, order=order)
    torch.cuda.synchronize()
    ra, rb = a.results(), b.results()
    for k in ra:
        assert np.array_equal(ra[k], rb[k], equal_nan=True), k


def _seeds(ev):
    f = ev.fit
    r = O.fit_tracks(f.radius[:3], f.x_over_X0[:3], f.Bz, f.mass, f.par, f.cov, f.q, f.hpos[:3], f.hcov[:3], None)
    return r["par"].astype(np.float32), O.pack_cov21(r["cov"]).astype(np.float32), r["chi2"], r["nhits"]


def _score_event(ctx, ev, do_update=True, chi2_cut=30.0, check_state=True, keep_local=True):
    """Layers 3..9 on both sides; returns (decisions, differing decisions inside the tie window).
    keep_local: the per-layer calls carry the candidates' local-frame state (kf_score_candidates, local_state);
    the final state is then held to the FIT tolerances."""
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceCandidates, DeviceLayer
    f, cfg = ev.fit, ev.cfg
    par, cov, chi2, nh = _seeds(ev)
    geom = K.Geometry(f.radius, f.x_over_X0, f.Bz, f.mass)
    dc = DeviceCandidates.from_numpy(par, cov, f.q, chi2, nh, "cuda:0")
    oc = O.Candidates(par, cov, f.q, chi2, nh)
    alive = np.ones(f.n, dtype=bool)         # candidates whose decisions agreed so far
    n_dec = n_tie = 0
    worst_chi2 = 0.0
    for l in range(cfg.first_scored_layer, cfg.n_layers):
        lay = ev.layers[l]
        dl = DeviceLayer.from_numpy(lay.pos, lay.cov, NE, NP, EMAX, "cuda:0")
        dl.bin(ctx, lay.radius)
        dc.score(ctx, geom, l, dl, 2, chi2_cut, do_update, keep_local=keep_local)
        torch.cuda.synchronize()
        ob = O.bin_hits(lay.pos, lay.radius, NE, NP, EMAX)
        orr = O.score_layer(oc, lay.radius, f.x_over_X0[l], f.Bz, f.mass, lay.pos, lay.cov, ob, NE, NP, EMAX,
                            2, chi2_cut, do_update)
        g = dc.results()
        diff = (g["best_hit"] != orr["best_hit"]) & alive
        b, s2 = orr["best_chi2"], orr["second_chi2"]
        # allowed: best and runner-up within 1e-4 relative, or the best within 1e-4 relative of the cut
        tie = (np.abs(s2 - b) <= 1e-4 * np.abs(b)) | (np.abs(b - chi2_cut) <= 1e-4 * chi2_cut)
        assert not np.any(diff & ~tie), f"layer {l}: {int((diff & ~tie).sum())} mismatches outside the tie window"
        n_dec += int(alive.sum())
        n_tie += int(diff.sum())
        alive &= ~diff                       # such a candidate is not compared further
        acc = alive & (orr["best_hit"] >= 0)
        # chi2 of ONE hit, held to north_star's 1e-3 max(chi2, 1) like the total (fp32 positions carry one or two ulp
        # of r = 40 cm = up to 8e-4 sigma_rphi, SURVEY hard part 3; worst seen over the 140 000 decisions of
        # configs[4]: 5.5e-4)
        rel = np.abs(g["best_chi2"][acc] - b[acc]) / np.maximum(b[acc], 1.0)
        worst_chi2 = max(worst_chi2, rel.max(initial=0))
        assert rel.max(initial=0) < 1e-3, rel.max()
        assert np.array_equal(g["status"][alive], oc.status[alive])
        assert np.array_equal(g["nhits"][alive], oc.nhits[alive])
    if check_state:
        g = dc.results()
        sel = alive & (oc.status == 0)
        sub_g = {k: (g[k][..., sel] if k in ("par", "cov") else g[k][sel]) for k in ("par", "cov", "chi2", "nhits", "status")}
        sub_o = dict(par=oc.par.T[:, sel], cov=oc.cov[sel], chi2=oc.chi2[sel], nhits=oc.nhits[sel], status=oc.status[sel])
        if keep_local:
            # the candidates stayed in the local frame between the calls: the fit tolerances, unloosened
            res = compare_fit(sub_g, sub_o, float(f.radius[-1]), max_diverged_frac=1.0)
        else:
            # Without local_state every layer hands the covariance back in the GLOBAL frame in fp32 and reads it
            # again: about 2e-3 on covariance elements per round trip (SURVEY.md hard part 1; the header says so).
            # That mode promises the decisions (checked above, unchanged) -- its state is only reported.
            res = compare_fit(sub_g, sub_o, float(f.radius[-1]), max_diverged_frac=1.0,
                              loosen=dict(cov=1e9, mom=1e9, pos=1e9, chi2=1e9))
        print(f"scoring state parity (keep_local={keep_local}):", res, " worst per-layer chi2 error:", worst_chi2)
    return n_dec, n_tie


def _build_event_fused(ctx, ev, use_order, half_length=None, material_model=0, energy_loss=0):
    """kf_build_best_hit over layers 3..9 in one call vs the oracle's layer loop: decisions by north_star's
    rule, final state at the FIT tolerances (the candidates never leave the local frame)."""
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceCandidates, DeviceLayer
    f, cfg = ev.fit, ev.cfg
    par, cov, chi2, nh = _seeds(ev)
    geom = K.Geometry(f.radius, f.x_over_X0, f.Bz, f.mass, half_length, material_model, energy_loss)
    dc = DeviceCandidates.from_numpy(par, cov, f.q, chi2, nh, "cuda:0")
    L0 = cfg.first_scored_layer
    dls = [DeviceLayer.from_numpy(l.pos, l.cov, NE, NP, EMAX, "cuda:0") for l in ev.layers[L0:]]
    ctx.bin_layers([l.radius for l in ev.layers[L0:]], [(d.n_hits, d.pos, d.cov, d.bins) for d in dls])
    order = dc.make_order(ctx, geom, L0, NE, NP, EMAX) if use_order else None
    idx, c2 = dc.build(ctx, geom, L0, dls, 2, 30.0, True, order)
    torch.cuda.synchronize()
    idx, c2 = idx.cpu().numpy()[:, :f.n], c2.cpu().numpy()[:, :f.n]
    oc = O.Candidates(par, cov, f.q, chi2, nh)
    alive = np.ones(f.n, dtype=bool)
    n_dec = n_tie = 0
    for j, l in enumerate(range(L0, cfg.n_layers)):
        lay = ev.layers[l]
        ob = O.bin_hits(lay.pos, lay.radius, NE, NP, EMAX)
        with O.geometry_options(material_model, half_length, score_layer=l, energy_loss=energy_loss):
            orr = O.score_layer(oc, lay.radius, f.x_over_X0[l], f.Bz, f.mass, lay.pos, lay.cov, ob, NE, NP, EMAX, 2, 30.0, True)
        diff = (idx[j] != orr["best_hit"]) & alive
        b, s2 = orr["best_chi2"], orr["second_chi2"]
        tie = (np.abs(s2 - b) <= 1e-4 * np.abs(b)) | (np.abs(b - 30.0) <= 1e-4 * 30.0)
        assert not np.any(diff & ~tie), f"layer {l}: {int((diff & ~tie).sum())} mismatches outside the tie window"
        n_dec += int(alive.sum()); n_tie += int(diff.sum())
        alive &= ~diff
        acc = alive & (orr["best_hit"] >= 0)
        assert (np.abs(c2[j][acc] - b[acc]) / np.maximum(b[acc], 1.0)).max(initial=0) < 1e-3
    g = dc.results()
    # a candidate beyond the barrel end (reading A20) stops there with its last state: a valid result to compare
    sel = alive & ((oc.status & ~np.uint32(O.OUTSIDE)) == 0)
    assert np.array_equal(g["status"][alive], oc.status[alive]) and np.array_equal(g["nhits"][alive], oc.nhits[alive])
    sub_g = {k: (g[k][..., sel] if k in ("par", "cov") else g[k][sel]) for k in ("par", "cov", "chi2", "nhits", "status")}
    sub_o = dict(par=oc.par.T[:, sel], cov=oc.cov[sel], chi2=oc.chi2[sel], nhits=oc.nhits[sel], status=oc.status[sel])
    sub_g["status"] = sub_g["status"] & ~np.uint32(O.OUTSIDE)      # (bits already checked equal above)
    sub_o["status"] = sub_o["status"] & ~np.uint32(O.OUTSIDE)
    # north_star fixes only the hit decisions for scoring; the state is held to the fit tolerances all the same
    # (the candidates enter the local frame in double: DESIGN.md 5.3)
    res = compare_fit(sub_g, sub_o, float(f.radius[-1]), max_diverged_frac=1.0)
    print("fused building state parity:", res)
    return n_dec, n_tie


def test_build_best_hit_small_event(ctx):
    ev = W.make_build_event(4, n_tracks=400, noise_hits=2000)
    n_dec, _ = _build_event_fused(ctx, ev, use_order=False)
    assert n_dec >= 0.99 * 7 * 400


def test_build_best_hit_full_config4(ctx):
    ev = W.make_build_event(4)
    n_dec, n_tie = _build_event_fused(ctx, ev, use_order=True)
    print(f"config 4 fused: {n_dec} decisions, {n_tie} differences inside the tie window")
    assert n_dec >= 0.99 * 7 * 20000 and n_tie <= 20


def test_build_best_hit_finite_barrel_and_path_length_material(ctx):
    """Reading A20 through the builder: 25 cm barrels cut the high-|eta| candidates off on the outer layers."""
    ev = W.make_build_event(4, n_tracks=3000, noise_hits=15000)
    L = ev.fit.n_layers
    hl = np.full(L, 25.0, dtype=np.float32)
    n_dec, _ = _build_event_fused(ctx, ev, use_order=True, half_length=hl, material_model=1)
    assert n_dec >= 0.98 * 7 * 3000


def test_build_best_hit_with_energy_loss(ctx):
    """Reading A21 through the builder (with path-length material): same decisions as the oracle with the option,
    and the option is felt (the candidates end with less momentum than without it)."""
    ev = W.make_build_event(4, n_tracks=3000, noise_hits=15000)
    n_dec, _ = _build_event_fused(ctx, ev, use_order=True, material_model=1, energy_loss=1)
    assert n_dec >= 0.98 * 7 * 3000


def test_score_small_event(ctx):
    ev = W.make_build_event(4, n_tracks=400, noise_hits=2000)
    n_dec, n_tie = _score_event(ctx, ev)
    assert n_dec >= 0.99 * 7 * 400
    n_dec, n_tie = _score_event(ctx, ev, keep_local=False)      # decisions do not need the local state
    assert n_dec >= 0.99 * 7 * 400


def test_score_full_config4(ctx):
    """BASELINE.json configs[4]: 20 000 seeds, 120 000 hits per layer, 40x64 bins, +-2-bin window."""
    ev = W.make_build_event(4)
    n_dec, n_tie = _score_event(ctx, ev)
    print(f"config 4: {n_dec} decisions, {n_tie} differences inside the tie window")
    assert n_dec >= 0.99 * 7 * 20000 and n_tie <= 20


def test_score_no_update_and_reject_all(ctx):
    ev = W.make_build_event(4, n_tracks=400, noise_hits=2000)
    _score_event(ctx, ev, do_update=False)
    _score_event(ctx, ev, chi2_cut=0.0)


def test_score_empty_window_and_errors(ctx):
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceCandidates, DeviceLayer
    ev = W.make_build_event(4, n_tracks=64, noise_hits=0)
    f = ev.fit
    par, cov, chi2, nh = _seeds(ev)
    geom = K.Geometry(f.radius, f.x_over_X0, f.Bz, f.mass)
    dc = DeviceCandidates.from_numpy(par, cov, f.q, chi2, nh, "cuda:0")
    empty = DeviceLayer.from_numpy(np.zeros((3, 0), np.float32), np.zeros((6, 0), np.float32), NE, NP, EMAX, "cuda:0")
    empty.bin(ctx, float(f.radius[3]))
    dc.score(ctx, geom, 3, empty)
    torch.cuda.synchronize()
    g = dc.results()
    assert np.all(g["best_hit"] == -1) and np.all(np.isinf(g["best_chi2"])) and np.array_equal(g["nhits"], nh)
    np.testing.assert_allclose(np.hypot(g["par"][0], g["par"][1]), f.radius[3], rtol=1e-5)   # propagated state kept
    with pytest.raises(K.KFError) as e:
        dc.score(ctx, geom, 10, empty)
    assert e.value.code == -2
    with pytest.raises(K.KFError) as e:
        dc.score(ctx, geom, 4, empty, window_half=40)
    assert e.value.code == -4
