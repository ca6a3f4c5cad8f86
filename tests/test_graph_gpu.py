"""kf_graph_*: a recorded sequence of hot calls replays with bit-identical results (include/kf_b200.h "graphs")."""
import copy

import numpy as np
import pytest
import torch

from workloads import barrel_events as W

pytestmark = pytest.mark.gpu
NE, NP, EMAX = 40, 64, float(np.float32(1.2))


@pytest.fixture()
def ctx():
    import paper_1705_02876_b200 as K
    st = torch.cuda.Stream()
    c = K.KFContext(0, st)
    c.torch_stream = st
    yield c
    c.close()


def _seeded_build(ctx, n_tracks=3000, noise=15000):
    """Event, candidate buffers seeded by the product's own 3-layer fit, layer pools."""
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceCandidates, DeviceFit, DeviceLayer
    ev = W.make_build_event(4, n_tracks=n_tracks, noise_hits=noise)
    f = ev.fit
    f3 = copy.copy(f)
    f3.radius, f3.x_over_X0 = f.radius[:3], f.x_over_X0[:3]
    f3.hpos, f3.hcov = np.ascontiguousarray(f.hpos[:3]), np.ascontiguousarray(f.hcov[:3])
    d3 = DeviceFit.from_batch(f3, "cuda:0")
    with torch.cuda.stream(ctx.torch_stream):
        d3.fit(ctx)
    torch.cuda.synchronize()
    s = d3.results()
    geom = K.Geometry(f.radius, f.x_over_X0, f.Bz, f.mass)
    layers = [DeviceLayer.from_numpy(l.pos, l.cov, NE, NP, EMAX, "cuda:0") for l in ev.layers[3:]]
    dc = DeviceCandidates.from_numpy(s["par"], s["cov"], f.q, s["chi2"], s["nhits"], "cuda:0")
    seed = {k: getattr(dc, k).clone() for k in ("par", "cov", "chi2", "nhits", "status")}
    return ev, geom, layers, dc, seed


def _reset(dc, seed):
    for k, v in seed.items():
        getattr(dc, k).copy_(v)
    torch.cuda.synchronize()


def test_bin_and_build_graph_equals_eager(ctx):
    ev, geom, layers, dc, seed = _seeded_build(ctx)
    radii = [l.radius for l in ev.layers[3:]]
    args = [(l.n_hits, l.pos, l.cov, l.bins) for l in layers]

    def sequence():
        ctx.bin_layers(radii, args)
        return dc.build(ctx, geom, 3, layers, 2, 30.0, True, None)

    with torch.cuda.stream(ctx.torch_stream):
        idx, c2 = sequence()                      # eager: also sizes every scratch buffer
    torch.cuda.synchronize()
    want = dict(dc.results(), idx=idx.cpu().numpy().copy(), c2=c2.cpu().numpy().copy(),
                off=[l.bins.bin_offset.cpu().numpy().copy() for l in layers])
    _reset(dc, seed)
    ctx.graph_begin()
    idx_g, c2_g = sequence()                      # recorded, not executed
    g = ctx.graph_end()
    for rep in range(3):
        _reset(dc, seed)
        idx_g.fill_(-7); c2_g.fill_(-1.0)
        for l in layers:
            l.bins.bin_offset.fill_(0)
        torch.cuda.synchronize()
        g.launch()
        torch.cuda.synchronize()
        got = dict(dc.results(), idx=idx_g.cpu().numpy(), c2=c2_g.cpu().numpy())
        for k in ("par", "cov", "chi2", "nhits", "status", "idx", "c2"):
            assert np.array_equal(got[k], want[k], equal_nan=True), (rep, k)
        for l, o in zip(layers, want["off"]):
            assert np.array_equal(l.bins.bin_offset.cpu().numpy(), o)
    g.close()


def test_fit_and_smooth_graph_equals_eager(ctx):
    from paper_1705_02876_b200.buffers import DeviceFit
    b = W.simulate_event(W.get_config(1), 3, n_tracks=20000)
    d = DeviceFit.from_batch(b, "cuda:0")
    with torch.cuda.stream(ctx.torch_stream):
        d.fit_refit(ctx)
    torch.cuda.synchronize()
    want, want_s = d.results(), d.refit_results()
    ctx.graph_begin()
    d.fit_refit(ctx)
    g = ctx.graph_end()
    d.out_par.zero_(); d.out_cov.zero_(); d.out_chi2.zero_()
    for v in d.refitted.values():                 # (fit_smooth writes into the same tensors at every call)
        v.zero_()
    torch.cuda.synchronize()
    g.launch()
    g.launch()                                    # a graph may be launched any number of times
    torch.cuda.synchronize()
    got, got_s = d.results(), d.refit_results()
    for k in want:
        assert np.array_equal(got[k], want[k], equal_nan=True), k
    for k in want_s:
        assert np.array_equal(got_s[k], want_s[k], equal_nan=True), k


def test_graph_errors_leave_the_context_usable(ctx):
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceFit
    b = W.simulate_event(W.get_config(1), 4, n_tracks=500)
    d = DeviceFit.from_batch(b, "cuda:0")
    with pytest.raises(K.KFError):
        ctx.graph_end()                           # nothing is being recorded
    ctx.graph_begin()
    with pytest.raises(K.KFError):
        ctx.graph_begin()                         # already recording
    with pytest.raises(K.KFError):
        ctx.set_stream(None)
    d.fit(ctx)
    g = ctx.graph_end()
    g.launch()
    torch.cuda.synchronize()
    first = d.results()
    # the legacy default stream cannot be recorded
    c0 = K.KFContext(0)
    c0.set_stream(None)
    raw = K.load_library()
    assert raw.kf_set_stream(c0._h, None) == 0
    with pytest.raises(K.KFError):
        c0.graph_begin()
    c0.close()
    # a call that has to grow scratch while recording voids the capture; afterwards eager calls work again
    ev, geom, layers, dc, seed = _seeded_build(ctx, n_tracks=400, noise=2000)
    ctx.graph_begin()
    try:
        ctx.bin_layers([l.radius for l in ev.layers[3:]], [(l.n_hits, l.pos, l.cov, l.bins) for l in layers])
    except K.KFError:
        pass
    with pytest.raises(K.KFError):
        ctx.graph_end()
    with torch.cuda.stream(ctx.torch_stream):
        d.fit(ctx)
    torch.cuda.synchronize()
    again = d.results()
    for k in first:
        assert np.array_equal(first[k], again[k], equal_nan=True)


def test_stale_graph_is_refused(ctx):
    """A recorded graph points into its context's scratch and bin edge tables.  Once that context reallocates
    scratch (a bigger pool) or bins with another grid, or the graph is handed to another context, kf_graph_launch
    refuses it (KF_ERR_STALE = -7) instead of replaying against freed memory or the wrong edges."""
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceLayer
    rng = np.random.default_rng(8)

    def pool(H, ne=NE, nph=NP):
        phi, eta = rng.uniform(-np.pi, np.pi, H), rng.uniform(-1.1, 1.1, H)
        pos = np.stack([10 * np.cos(phi), 10 * np.sin(phi), 10 * np.sinh(eta)]).astype(np.float32)
        cov = np.tile(np.array([1e-2, 0, 0, 1e-2, 0, 1e-2], dtype=np.float32)[:, None], (1, H))
        return DeviceLayer.from_numpy(pos, cov, ne, nph, EMAX, "cuda:0")

    def record(dl):
        with torch.cuda.stream(ctx.torch_stream):
            dl.bin(ctx, 10.0)                      # eager once: sizes the scratch, writes the tables
        torch.cuda.synchronize()
        ctx.graph_begin()
        dl.bin(ctx, 10.0)
        return ctx.graph_end()

    small = pool(3000)
    g = record(small)
    g.launch()                                     # fresh: fine
    torch.cuda.synchronize()
    want = small.bins.bin_offset.cpu().numpy().copy()
    # (1) another grid rewrites the edge tables in place
    other = pool(3000, 7, 10)
    with torch.cuda.stream(ctx.torch_stream):
        other.bin(ctx, 10.0)
    torch.cuda.synchronize()
    with pytest.raises(K.KFError) as e:
        g.launch()
    assert e.value.code == -7
    g.close()
    # (2) a bigger pool reallocates the scratch
    g = record(small)
    big = pool(400_000)
    with torch.cuda.stream(ctx.torch_stream):
        big.bin(ctx, 10.0)
    torch.cuda.synchronize()
    with pytest.raises(K.KFError) as e:
        g.launch()
    assert e.value.code == -7
    g.close()
    # (3) re-recorded, it runs again and gives the same bins; another context is refused
    g = record(small)
    small.bins.bin_offset.fill_(0)
    g.launch()
    torch.cuda.synchronize()
    assert np.array_equal(small.bins.bin_offset.cpu().numpy(), want)
    c2 = K.KFContext(0, ctx.torch_stream)
    assert c2._lib.kf_graph_launch(c2._h, g._g) == -7
    c2.close()
    g.close()


def test_indexed_fit_in_a_graph_and_its_scratch(ctx):
    """kf_fit_tracks_indexed without bins packs the pools into context scratch: recorded after one eager call the
    graph replays the packing and the fit with identical results; a later call with larger pools reallocates that
    scratch and the graph is refused (KF_ERR_STALE) instead of reading freed memory."""
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceFit, DeviceLayer, padded_ld

    def setup(n_tracks, noise):
        ev = W.make_build_event(4, n_tracks=n_tracks, noise_hits=noise)
        f = ev.fit
        d = DeviceFit.from_batch(f, "cuda:0")
        pools = [DeviceLayer.from_numpy(l.pos, l.cov, NE, NP, EMAX, "cuda:0") for l in ev.layers]
        idx = torch.full((len(ev.layers), padded_ld(f.n)), -1, dtype=torch.int32, device="cuda:0")
        idx[:, :f.n] = torch.from_numpy(np.stack([l.true_index for l in ev.layers]).astype(np.int32)).to("cuda:0")

        def call():
            ctx.fit_tracks_indexed(d.geom, f.n, d.par, d.cov, d.q, idx, [(p.n_hits, p.pos, p.cov) for p in pools],
                                   d.out_par, d.out_cov, d.out_chi2, d.out_nhits, d.out_status)
        return d, call, (pools, idx)

    d, call, keep = setup(3000, 6000)
    with torch.cuda.stream(ctx.torch_stream):
        call()
    torch.cuda.synchronize()
    want = d.results()
    ctx.graph_begin()
    call()
    g = ctx.graph_end()
    d.out_par.zero_(); d.out_cov.zero_(); d.out_chi2.zero_()
    torch.cuda.synchronize()
    g.launch()
    torch.cuda.synchronize()
    got = d.results()
    for k in want:
        assert np.array_equal(got[k], want[k], equal_nan=True), k
    assert np.count_nonzero(got["chi2"]) > 2900
    d2, call2, keep2 = setup(9000, 20000)           # larger pools: the scratch grows
    with torch.cuda.stream(ctx.torch_stream):
        call2()
    torch.cuda.synchronize()
    with pytest.raises(K.KFError) as e:
        g.launch()
    assert e.value.code == -7
    g.close()
