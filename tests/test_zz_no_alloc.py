"""kf_score_candidates_static (include/kf_b200.h): the single-layer scoring call with its per-candidate scratch in a
`static __device__` array of the library instead of cudaMalloc'ed context scratch, for callers that must not allocate.

It launches the same kernels on the same inputs as kf_score_candidates, so its outputs are compared with that
existing path's and must be IDENTICAL (best hit, chi2, candidate state, status), on two calls in a row that share the
array (the second one reads the candidate state the first one left and finds the first one's scratch contents), after a
call with more candidates than the next one (stale contents beyond n), at the maximum size, and beyond it (clear error,
nothing written).  The parity of the existing path against the oracle is tests/test_score_gpu.py.

This file is collected last on purpose (pytest -x): it must pass alone in a fresh process and after
every other test.
"""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as O
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


@pytest.fixture(scope="module")
def event():
    """configs[4]-shaped building event, reduced: 3000 seeds fitted on layers 0..2 by the oracle (inputs only)."""
    ev = W.make_build_event(4, n_tracks=3000, noise_hits=15000)
    f = ev.fit
    r = O.fit_tracks(f.radius[:3], f.x_over_X0[:3], f.Bz, f.mass, f.par, f.cov, f.q, f.hpos[:3], f.hcov[:3], None)
    seeds = (r["par"].astype(np.float32), O.pack_cov21(r["cov"]).astype(np.float32), r["chi2"], r["nhits"])
    return ev, seeds


def _layers(ctx, ev, which):
    from paper_1705_02876_b200.buffers import DeviceLayer
    out = {}
    for l in which:
        lay = ev.layers[l]
        dl = DeviceLayer.from_numpy(lay.pos, lay.cov, NE, NP, EMAX, "cuda:0")
        dl.bin(ctx, lay.radius)
        out[l] = dl
    torch.cuda.synchronize()
    return out


def _candidates(seeds, q, n=None):
    """n candidates: the event's seeds, repeated cyclically when n is larger than the event."""
    from paper_1705_02876_b200.buffers import DeviceCandidates
    par, cov, chi2, nh = seeds
    m = par.shape[1]
    n = m if n is None else n
    sel = np.arange(n) % m
    return DeviceCandidates.from_numpy(np.ascontiguousarray(par[:, sel]), np.ascontiguousarray(cov[:, sel]),
                                       np.ascontiguousarray(q[sel]), np.ascontiguousarray(chi2[sel]),
                                       np.ascontiguousarray(nh[sel]), "cuda:0")


def _assert_identical(a, b, what):
    ra, rb = a.results(), b.results()
    assert set(ra) == set(rb)
    for k in ra:
        assert np.array_equal(ra[k], rb[k], equal_nan=True), (what, k)
    assert (ra["best_hit"] >= 0).sum() > 0.5 * len(ra["best_hit"]), what      # the comparison is not vacuous


def test_static_scratch_equals_the_allocating_path_on_two_calls_in_a_row(ctx, event):
    import paper_1705_02876_b200 as K
    ev, seeds = event
    f = ev.fit
    geom = K.Geometry(f.radius, f.x_over_X0, f.Bz, f.mass)
    dls = _layers(ctx, ev, (3, 4, 5))
    ref = _candidates(seeds, f.q)
    sta = _candidates(seeds, f.q)
    # call 1 and call 2 share the static array; call 2 continues from the state call 1 left (keep_local)
    for l in (3, 4):
        ref.score(ctx, geom, l, dls[l])
        sta.score(ctx, geom, l, dls[l], static_scratch=True)
        torch.cuda.synchronize()
        _assert_identical(sta, ref, f"layer {l}")
    # a third call without the local-frame state and without the update (other branches of the same kernels)
    ref.score(ctx, geom, 5, dls[5], do_update=False, keep_local=False)
    sta.score(ctx, geom, 5, dls[5], do_update=False, keep_local=False, static_scratch=True)
    torch.cuda.synchronize()
    _assert_identical(sta, ref, "layer 5, no update")


def test_static_scratch_keeps_nothing_from_a_larger_call(ctx, event):
    """A call with many candidates, then one with few (ragged: 777), then the many again: what a call left in the
    array beyond or below the next call's n changes nothing."""
    import paper_1705_02876_b200 as K
    ev, seeds = event
    f = ev.fit
    geom = K.Geometry(f.radius, f.x_over_X0, f.Bz, f.mass)
    dl = _layers(ctx, ev, (3,))[3]
    for n in (20000, 777, 20000, 1):
        ref = _candidates(seeds, f.q, n)
        sta = _candidates(seeds, f.q, n)
        ref.score(ctx, geom, 3, dl)
        sta.score(ctx, geom, 3, dl, static_scratch=True)
        torch.cuda.synchronize()
        ra, rb = sta.results(), ref.results()
        for k in ra:
            assert np.array_equal(ra[k], rb[k], equal_nan=True), (n, k)


def test_static_scratch_maximum_size_and_beyond(ctx, event):
    import paper_1705_02876_b200 as K
    ev, seeds = event
    f = ev.fit
    geom = K.Geometry(f.radius, f.x_over_X0, f.Bz, f.mass)
    dl = _layers(ctx, ev, (3,))[3]
    nmax = K.STATIC_MAX_CANDIDATES
    ref = _candidates(seeds, f.q, nmax)
    sta = _candidates(seeds, f.q, nmax)
    ref.score(ctx, geom, 3, dl)
    sta.score(ctx, geom, 3, dl, static_scratch=True)
    torch.cuda.synchronize()
    _assert_identical(sta, ref, "n = maximum")
    # one more than the maximum: a clear error, and nothing is launched or written
    big = _candidates(seeds, f.q, nmax + 1)
    before = big.results()
    big.best_hit.fill_(-7)
    with pytest.raises(K.KFError) as err:
        big.score(ctx, geom, 3, dl, static_scratch=True)
    assert err.value.code == K.ERR_TOO_LARGE and "static scratch" in str(err.value)
    torch.cuda.synchronize()
    after = big.results()
    assert np.all(after["best_hit"] == -7)
    for k in ("par", "cov", "chi2", "nhits", "status"):
        assert np.array_equal(before[k], after[k], equal_nan=True), k
    # the allocating path takes that size
    big.score(ctx, geom, 3, dl)
    torch.cuda.synchronize()
    assert (big.results()["best_hit"] >= 0).sum() > 0.5 * (nmax + 1)


def test_static_scratch_call_allocates_no_device_memory(event):
    """Free device memory (cudaMemGetInfo) does not move across static-scratch calls of growing size on a context
    that has never scored before -- the allocating path has to grow its scratch for the same sequence."""
    import paper_1705_02876_b200 as K
    ev, seeds = event
    f = ev.fit
    geom = K.Geometry(f.radius, f.x_over_X0, f.Bz, f.mass)
    fresh = K.KFContext(0)
    try:
        dl = _layers(fresh, ev, (3,))[3]
        cands = [_candidates(seeds, f.q, n) for n in (64, 3000, 50000)]
        cands[0].score(fresh, geom, 3, dl, static_scratch=True)      # set-up call: symbol address, kernels loaded
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info(0)[0]
        for c in cands[1:]:
            c.score(fresh, geom, 3, dl, keep_local=False, static_scratch=True)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info(0)[0] == free0
        assert (cands[2].results()["best_hit"] >= 0).sum() > 25000
    finally:
        fresh.close()
