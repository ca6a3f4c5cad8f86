"""kf_fit_tracks_indexed (hits addressed by index into the layer pools) and the whole chain
bin -> build -> fit (indexed) against the oracle."""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as O
from tests.parity import compare_fit
from workloads import barrel_events as W

pytestmark = pytest.mark.gpu
NE, NP = 40, 64
EMAX = float(np.float32(1.2))


@pytest.fixture(scope="module")
def ctx():
    import paper_1705_02876_b200 as K
    c = K.KFContext(0)
    yield c
    c.close()


def _fit_indexed(ctx, ev, index_np, use_records=False, n_fit=None):
    """Fit the event's seeds (the first n_fit of them) with hits index_np[L][n] (into ev.layers pools, -1 = none)."""
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceFit, DeviceLayer, padded_ld
    f = ev.fit
    d = DeviceFit.from_batch(f, "cuda:0")
    if n_fit is not None:
        d.n = n_fit
    pools = [DeviceLayer.from_numpy(l.pos, l.cov, NE, NP, EMAX, "cuda:0") for l in ev.layers]
    idx = torch.full((len(ev.layers), padded_ld(f.n)), -1, dtype=torch.int32, device="cuda:0")
    idx[:, :f.n] = torch.from_numpy(np.ascontiguousarray(index_np, dtype=np.int32)).to("cuda:0")
    bins = None
    if use_records:
        ctx.bin_layers([l.radius for l in ev.layers], [(p.n_hits, p.pos, p.cov, p.bins) for p in pools])
        bins = [p.bins for p in pools]
    ctx.fit_tracks_indexed(d.geom, d.n, d.par, d.cov, d.q, idx, [(p.n_hits, p.pos, p.cov) for p in pools],
                           d.out_par, d.out_cov, d.out_chi2, d.out_nhits, d.out_status, bins=bins)
    torch.cuda.synchronize()
    return d.results()


def _oracle_fit_with(ev, index_np):
    f = ev.fit
    L, n = len(ev.layers), f.n
    hpos = np.zeros((L, 3, n), dtype=np.float32)
    hcov = np.zeros((L, 6, n), dtype=np.float32)
    mask = np.zeros(n, dtype=np.uint32)
    for l in range(L):
        has = index_np[l] >= 0
        hpos[l][:, has] = ev.layers[l].pos[:, index_np[l][has]]
        hcov[l][:, has] = ev.layers[l].cov[:, index_np[l][has]]
        mask |= has.astype(np.uint32) << np.uint32(l)
    return O.fit_tracks(f.radius, f.x_over_X0, f.Bz, f.mass, f.par, f.cov, f.q, hpos, hcov, mask, nthreads=8)


def test_indexed_fit_with_true_hits_equals_the_pre_gathered_fit(ctx):
    from paper_1705_02876_b200.buffers import DeviceFit
    ev = W.make_build_event(4, n_tracks=5003, noise_hits=20000)
    truth = np.stack([l.true_index for l in ev.layers])
    g = _fit_indexed(ctx, ev, truth)
    o = _oracle_fit_with(ev, truth)
    compare_fit(g, o, float(ev.fit.radius[-1]), max_diverged_frac=2e-3)
    g2 = _fit_indexed(ctx, ev, truth, use_records=True)          # same hits through the packed records
    for k in g:
        assert np.array_equal(g[k], g2[k]), k
    d = DeviceFit.from_batch(ev.fit, "cuda:0")      # the same hits pre-gathered per track
    d.fit(ctx)
    torch.cuda.synchronize()
    r = d.results()
    assert np.array_equal(r["nhits"], g["nhits"]) and np.array_equal(r["status"], g["status"])
    np.testing.assert_allclose(r["chi2"], g["chi2"], rtol=2e-4, atol=1e-4)
    np.testing.assert_allclose(r["par"], g["par"], rtol=0, atol=2e-4)


def test_indexed_fit_reads_pools_directly_or_through_packed_records(ctx):
    """Without bins the call packs the SoA pools into records of its own (context scratch) unless the pools hold more
    than eight times the hits the tracks will read: both branches, same results bit for bit -- a few tracks against
    large pools (direct reads), all tracks (packed), and again a few (the scratch of the packed call is still there
    and must not be used)."""
    ev = W.make_build_event(4, n_tracks=4001, noise_hits=20000)
    truth = np.stack([l.true_index for l in ev.layers])
    total = sum((len(l.pos[0]) + 3) // 4 * 4 for l in ev.layers)
    L = len(ev.layers)
    assert total > 8 * 300 * L and total <= 8 * 4001 * L
    few = _fit_indexed(ctx, ev, truth, n_fit=300)                 # direct reads
    full = _fit_indexed(ctx, ev, truth)                           # packed records
    few2 = _fit_indexed(ctx, ev, truth, n_fit=300)
    rec = _fit_indexed(ctx, ev, truth, use_records=True)          # kf_bin_layers' records
    for k in full:
        assert np.array_equal(few[k], full[k][..., :300], equal_nan=True), k
        assert np.array_equal(few[k], few2[k], equal_nan=True), k
        assert np.array_equal(rec[k], full[k], equal_nan=True), k
    # a pool of a single hit, an empty pool, and a ragged last warp of the packing kernel
    import copy
    ev2 = copy.deepcopy(ev)
    keep = 20037
    for j, l in enumerate(ev2.layers):
        m = 1 if j == 2 else (0 if j == 4 else keep + j)
        l.pos, l.cov = np.ascontiguousarray(l.pos[:, :m]), np.ascontiguousarray(l.cov[:, :m])
        truth[j] = np.where(truth[j] < m, truth[j], -1)
    a = _fit_indexed(ctx, ev2, truth)
    b = _fit_indexed(ctx, ev2, truth, n_fit=300)
    o = _oracle_fit_with(ev2, truth)
    assert np.array_equal(a["nhits"], o["nhits"])
    for k in a:
        assert np.array_equal(a[k][..., :300], b[k], equal_nan=True), k
    sel = o["nhits"] >= 4
    compare_fit({k: (v[..., sel] if k in ("par", "cov") else v[sel]) for k, v in a.items()},
                {k: (v[..., sel] if k == "par" else v[sel]) for k, v in o.items()}, float(ev.fit.radius[-1]),
                max_diverged_frac=0.02)


def test_indexed_fit_with_path_length_material_and_energy_loss(ctx):
    """Readings A20 / A21 ride on the indexed fit like on every call that propagates."""
    ev = W.make_build_event(4, n_tracks=3001, noise_hits=9000)
    ev.fit.material_model, ev.fit.energy_loss = 1, 1            # picked up by DeviceFit.from_batch
    truth = np.stack([l.true_index for l in ev.layers])
    g = _fit_indexed(ctx, ev, truth, use_records=True)
    with O.geometry_options(1, None, energy_loss=1):
        o = _oracle_fit_with(ev, truth)
    compare_fit(g, o, float(ev.fit.radius[-1]), max_diverged_frac=2e-3)
    o_plain = _oracle_fit_with(ev, truth)
    assert np.median(np.linalg.norm(o_plain["par"][3:6], axis=0) - np.linalg.norm(o["par"][3:6], axis=0)) > 1e-3


def test_indexed_fit_missing_hits_and_bad_charge(ctx):
    ev = W.make_build_event(4, n_tracks=600, noise_hits=3000)
    rng = np.random.default_rng(5)
    idx = np.stack([l.true_index for l in ev.layers]).astype(np.int32)
    drop = rng.random(idx.shape) < 0.15
    drop[:3] = False                                 # keep the first three layers (see test_fit_missing_layers)
    idx[drop] = -1
    idx[:, :20] = -1                                 # nothing to fit: the seed comes back
    ev.fit.q[20] = 0
    g = _fit_indexed(ctx, ev, idx)
    o = _oracle_fit_with(ev, idx)
    assert np.array_equal(g["status"], o["status"]) and np.array_equal(g["nhits"], o["nhits"])
    assert np.array_equal(g["par"][:, :21], ev.fit.par[:, :21]) and np.array_equal(g["cov"][:, :21], ev.fit.cov[:, :21])
    sel = o["nhits"] >= 5
    sub_g = {k: (v[..., sel] if k in ("par", "cov") else v[sel]) for k, v in g.items()}
    sub_o = {k: (v[..., sel] if k == "par" else v[sel]) for k, v in o.items()}
    compare_fit(sub_g, sub_o, float(ev.fit.radius[-1]), max_diverged_frac=0.05)


def test_chain_bin_build_fit(ctx):
    """Seeds from three hits -> combinatorial building on layers 3..9 -> final fit of the found hit lists
    (layers 0..9, hits by index) from the original seeds: same tracks as the oracle chain."""
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceCandidates, DeviceLayer
    ev = W.make_build_event(4, n_tracks=3000, noise_hits=15000)
    f = ev.fit
    r3 = O.fit_tracks(f.radius[:3], f.x_over_X0[:3], f.Bz, f.mass, f.par, f.cov, f.q, f.hpos[:3], f.hcov[:3], None, nthreads=8)
    par, cov = r3["par"].astype(np.float32), O.pack_cov21(r3["cov"]).astype(np.float32)
    geom = K.Geometry(f.radius, f.x_over_X0, f.Bz, f.mass)
    dls = [DeviceLayer.from_numpy(l.pos, l.cov, NE, NP, EMAX, "cuda:0") for l in ev.layers[3:]]
    ctx.bin_layers([l.radius for l in ev.layers[3:]], [(d.n_hits, d.pos, d.cov, d.bins) for d in dls])
    dc = DeviceCandidates.from_numpy(par, cov, f.q, r3["chi2"], r3["nhits"], "cuda:0")
    found, _ = dc.build_combinatorial(ctx, geom, 3, dls, 4)
    torch.cuda.synchronize()
    found = found.cpu().numpy()[:, :f.n]
    layers = [(l.pos, l.cov, O.bin_hits(l.pos, l.radius, NE, NP, EMAX)) for l in ev.layers[3:]]
    ob = O.build_combinatorial(f.radius, f.x_over_X0, f.Bz, f.mass, par, cov, f.q, r3["chi2"], r3["nhits"], 3, layers,
                               NE, NP, EMAX, 2, 30.0, 4)
    same = (found == ob["hits"]).all(axis=0)
    assert not np.any(~same & (ob["margin"] >= 2e-3)) and same.mean() > 0.97
    # final fit over all ten layers: the three seed hits (true hits) + what building found (GPU's own lists)
    full = np.concatenate([np.stack([l.true_index for l in ev.layers[:3]]), found]).astype(np.int32)
    g = _fit_indexed(ctx, ev, full)
    o = _oracle_fit_with(ev, full)
    res = compare_fit(g, o, float(f.radius[-1]), max_diverged_frac=0.2)
    print("chain final-fit parity:", res)


def test_indexed_fit_config2_full_size(ctx):
    """kf_fit_tracks_indexed at the size bench.py times it: config 2 (2 M tracks x 10 layers), every layer's hits
    shuffled into one pool of 2 M hits, read from the SoA pools and (second call) from the packed records of
    kf_bin_layers.  Both must equal, bit for bit, each other; the oracle checks every 16th event track by track."""
    from paper_1705_02876_b200.binding import Bins
    from paper_1705_02876_b200.buffers import DeviceFit
    cfg = W.get_config(2)
    b = W.make_fit_batch(2)
    n, L = b.n, b.n_layers
    assert n == 2_000_000
    d = DeviceFit.from_batch(b, "cuda:0")
    gen = torch.Generator(device="cuda:0"); gen.manual_seed(5)
    pools, index = [], torch.full((L, d.ld), -1, dtype=torch.int32, device="cuda:0")
    for l in range(L):
        perm = torch.randperm(n, device="cuda:0", generator=gen)
        pp = torch.zeros((3, d.ld), dtype=torch.float32, device="cuda:0"); pc = torch.zeros((6, d.ld), dtype=torch.float32, device="cuda:0")
        pp[:, :n] = d.hpos[l][:, :n][:, perm]; pc[:, :n] = d.hcov[l][:, :n][:, perm]
        inv = torch.empty(n, dtype=torch.int64, device="cuda:0"); inv[perm] = torch.arange(n, device="cuda:0")
        index[l, :n] = inv.to(torch.int32)
        pools.append((n, pp, pc))
    d.hpos = d.hcov = None                                   # (free 0.7 GB: the indexed call does not read them)
    ctx.fit_tracks_indexed(d.geom, n, d.par, d.cov, d.q, index, pools, d.out_par, d.out_cov, d.out_chi2, d.out_nhits, d.out_status)
    torch.cuda.synchronize()
    g = d.results()
    pbins = [Bins.allocate(n, NE, NP, EMAX, "cuda:0", soa=False) for _ in range(L)]
    ctx.bin_layers([float(r) for r in d.geom.radius_cm], [(n, pp, pc, b_) for (_, pp, pc), b_ in zip(pools, pbins)])
    ctx.fit_tracks_indexed(d.geom, n, d.par, d.cov, d.q, index, pools, d.out_par, d.out_cov, d.out_chi2, d.out_nhits, d.out_status, bins=pbins)
    torch.cuda.synchronize()
    g2 = d.results()
    for k in g:
        assert np.array_equal(g[k], g2[k], equal_nan=True), k
    for ev in range(0, cfg.n_events, 16):
        lo, hi = ev * cfg.n_tracks, (ev + 1) * cfg.n_tracks
        o = O.fit_batch(W.simulate_event(cfg, ev), nthreads=8)
        compare_fit({k: (v[..., lo:hi] if k in ("par", "cov") else v[lo:hi]) for k, v in g.items()}, o, float(b.radius[-1]))
