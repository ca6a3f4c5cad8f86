"""GPU parity of kf_fit_tracks (through the C ABI) against the fp64 oracle, element by element.

Tolerances: BASELINE.json north_star / DESIGN.md reading A15, written in tests/parity.py."""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as O
from tests.parity import compare_fit
from workloads import barrel_events as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    import paper_1705_02876_b200 as K
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    c = K.KFContext(0)
    yield c
    c.close()


def _gpu_fit(ctx, batch, with_mask=True):
    from paper_1705_02876_b200.buffers import DeviceFit
    d = DeviceFit.from_batch(batch, "cuda:0", with_mask=with_mask)
    d.fit(ctx)
    torch.cuda.synchronize()
    return d.results()


@pytest.mark.parametrize("config", [0, 1, 3])
def test_fit_parity_full_config(ctx, config):
    b = W.make_fit_batch(config)
    g = _gpu_fit(ctx, b)
    o = O.fit_batch(b, nthreads=8)
    res = compare_fit(g, o, float(b.radius[-1]))
    print(f"config {config}: {res}")


def test_fit_parity_config2_sampled(ctx):
    """Config 2 at full size (2M tracks, one launch, the configuration bench.py times); the oracle
    checks every 16th event's tracks one by one."""
    cfg = W.get_config(2)
    b = W.make_fit_batch(2)
    assert b.n == 2_000_000
    g = _gpu_fit(ctx, b)
    for ev in range(0, cfg.n_events, 16):
        lo, hi = ev * cfg.n_tracks, (ev + 1) * cfg.n_tracks
        sub = W.simulate_event(cfg, ev)
        assert np.array_equal(sub.par, b.par[:, lo:hi])
        o = O.fit_batch(sub, nthreads=8)
        gs = {k: (v[..., lo:hi] if k in ("par", "cov") else v[lo:hi]) for k, v in g.items()}
        compare_fit(gs, o, float(b.radius[-1]))
    ndf = 2 * g["nhits"] - 5
    assert (g["status"] != 0).mean() < 1e-3
    assert 0.9 < np.median(g["chi2"] / ndf) < 1.1


@pytest.mark.parametrize("n", [1, 31, 33, 127, 129, 1001])
def test_fit_ragged_sizes(ctx, n):
    b = W.simulate_event(W.get_config(1), 5, n_tracks=n)
    g = _gpu_fit(ctx, b)
    o = O.fit_batch(b)
    compare_fit(g, o, float(b.radius[-1]), max_diverged_frac=1.0)


@pytest.mark.parametrize("n_layers,step,n", [(32, 2.5, 3000), (32, 2.5, 160_000), (1, 4.0, 700), (2, 4.0, 700)])
def test_fit_extreme_layer_counts(ctx, n_layers, step, n):
    """KF_MAX_LAYERS = 32 layers (mask bit 31 in use; 160 000 tracks take the pair kernel, 3 000 the one-track
    kernel) and the shortest geometries (one and two layers: the fit is one or two updates of the seed)."""
    import dataclasses
    cfg = dataclasses.replace(W.get_config(3), n_layers=n_layers, layer_step_cm=step, n_tracks=n)
    b = W.simulate_event(cfg, 21, n_tracks=n)
    assert b.n_layers == n_layers and (n_layers < 32 or int(b.mask.max()) >> 31 == 1)
    g = _gpu_fit(ctx, b)
    o = O.fit_batch(b)
    compare_fit(g, o, float(b.radius[-1]), max_diverged_frac=1e-3 if n_layers > 2 else 1.0)
    assert np.array_equal(g["nhits"], o["nhits"]) and np.array_equal(g["status"], o["status"])


def test_fit_empty(ctx):
    b = W.simulate_event(W.get_config(1), 5, n_tracks=4)
    from paper_1705_02876_b200.buffers import DeviceFit
    d = DeviceFit.from_batch(b, "cuda:0")
    d.n = 0
    d.out_par.fill_(7.0)
    d.fit(ctx)
    torch.cuda.synchronize()
    assert torch.all(d.out_par == 7.0)


def test_fit_mask_null_equals_all_layers(ctx):
    b = W.simulate_event(W.get_config(1), 6, n_tracks=500)
    g1 = _gpu_fit(ctx, b, with_mask=True)
    g2 = _gpu_fit(ctx, b, with_mask=False)
    for k in g1:
        assert np.array_equal(g1[k], g2[k]), k


def test_fit_missing_layers(ctx):
    """Hit masks with holes (plus: no hit at all, a missing first layer, only the first three).
    The first three layers are kept in the random part: a track whose second hit comes 16 cm after
    its first is propagated with a 30 % momentum prior, far outside the linear regime, and fp32
    then reaches only ~1e-3 on the momentum variance."""
    b = W.simulate_event(W.get_config(1), 8, n_tracks=2000)
    rng = np.random.default_rng(3)
    b.mask = (rng.integers(0, 1 << 10, size=b.n) | 0b111).astype(np.uint32)
    b.mask[:50] = 0
    b.mask[50:100] = 0b1111111110
    b.mask[100:150] = 0b0000000111
    g = _gpu_fit(ctx, b)
    o = O.fit_batch(b)
    nh = o["nhits"]
    # tracks with >= 4 hits are well constrained: full parity; the others must agree on bookkeeping
    sel = nh >= 4
    sub_g = {k: (v[..., sel] if k in ("par", "cov") else v[sel]) for k, v in g.items()}
    sub_o = {k: (v[..., sel] if k == "par" else v[sel]) for k, v in o.items()}
    compare_fit(sub_g, sub_o, float(b.radius[-1]), max_diverged_frac=0.05)
    assert np.array_equal(g["nhits"], nh)
    # nothing fitted: the seed comes back bit-exact
    z = nh == 0
    assert z.sum() >= 50
    assert np.array_equal(g["par"][:, z], b.par[:, z]) and np.array_equal(g["cov"][:, z], b.cov[:, z])
    assert np.all(g["chi2"][z] == 0)


def _zero_status(d):
    d = dict(d)
    d["status"] = np.zeros_like(d["status"])
    return d


def test_fit_status_bits(ctx):
    """Degenerate tracks: bad charge, NaN hit (NONFINITE), non-positive-definite S (S_NOT_PD).
    Same status, same hits used and same surviving state as the oracle."""
    b = W.simulate_event(W.get_config(1), 9, n_tracks=64)
    b.q[0] = 0
    b.q[1] = 3
    b.hpos[4, 1, 4] = np.nan                       # NaN hit on layer 4 of track 4
    b.hcov[2, :, 5] = 0.0                          # zero hit covariance on layer 2 of track 5 ...
    b.hcov[2, 0, 5] = -1.0                         # ... with a negative variance: det S <= 0
    g = _gpu_fit(ctx, b)
    o = O.fit_batch(b)
    assert g["status"][0] == 8 and g["status"][1] == 8
    assert np.array_equal(g["par"][:, :2], b.par[:, :2]) and np.array_equal(g["cov"][:, :2], b.cov[:, :2])
    assert np.array_equal(g["status"], o["status"]), (g["status"][:8], o["status"][:8])
    assert np.array_equal(g["nhits"], o["nhits"])
    assert o["status"][4] == 4 and o["status"][5] == 2 and o["nhits"][4] == 9 and o["nhits"][5] == 9
    sel = np.arange(b.n) >= 2
    sub_g = {k: (v[..., sel] if k in ("par", "cov") else v[sel]) for k, v in g.items()}
    sub_o = {k: (v[..., sel] if k == "par" else v[sel]) for k, v in o.items()}
    compare_fit(_zero_status(sub_g), _zero_status(sub_o), float(b.radius[-1]), max_diverged_frac=1.0)


def test_fit_propagation_failure(ctx):
    """Tracks of pT 0.17-0.18 GeV (2R about 30 cm) asked for hits at r = 36 and 40 cm: no outward
    crossing -> PROP_FAIL on both sides, state kept from the last good layer."""
    cfg = W.BarrelConfig(1, 1, 256, 10, 0.17, 0.18, 1.0, 0.01)
    b = W.simulate_event(cfg, 21)
    assert np.all((b.mask >> 8) == 0)
    b.mask = b.mask | np.uint32(0b11 << 8)
    g = _gpu_fit(ctx, b)
    o = O.fit_batch(b)
    assert np.all(o["status"] == 1)
    assert np.array_equal(g["status"], o["status"]) and np.array_equal(g["nhits"], o["nhits"])
    compare_fit(_zero_status(g), _zero_status(o), float(b.radius[-1]), max_diverged_frac=0.05)


def test_fit_pair_kernel_edge_cases(ctx):
    """Batches of >= 151 552 tracks take the two-tracks-per-thread kernel (packed fp32x2 arithmetic); a layer
    that only one track of a pair has a hit on, or on which one of the two fails, goes through its one-track
    path.  Every degenerate case of the small tests above, at a size that selects that kernel, odd tail included."""
    cfg = W.get_config(1)
    low = W.BarrelConfig(1, 1, 256, 10, 0.17, 0.18, 1.0, 0.01)          # no crossing with the two outer layers
    parts = [W.simulate_event(cfg, 30 + e) for e in range(8)] + [W.simulate_event(low, 21), W.simulate_event(cfg, 38, n_tracks=3)]
    b = W.concat_batches(parts)
    assert b.n == 160_259 and b.n % 2 == 1
    rng = np.random.default_rng(11)
    holes = rng.random(b.n) < 0.1
    holes[160_000:] = False        # (near-looping tracks with gaps leave the linear regime: DESIGN.md 'Known limits')
    b.mask = np.where(holes, (rng.integers(0, 1 << 10, size=b.n) | 0b111), b.mask).astype(np.uint32)
    b.mask[:50] = 0
    b.mask[50:100] = 0b1111111110
    b.mask[101:150:2] = 0b0000000111                                    # odd tracks only: their partners go on
    lo = 160_000
    b.mask[lo:lo + 256] |= np.uint32(0b11 << 8)                          # PROP_FAIL on layers 8 and 9
    b.q[200] = 0
    b.q[203] = 3
    b.hpos[4, 1, 300] = np.nan                                          # NONFINITE on layer 4 of track 300
    b.hcov[2, :, 303] = 0.0
    b.hcov[2, 0, 303] = -1.0                                            # S_NOT_PD on layer 2 of track 303
    b.mask[300] = b.mask[303] = b.mask[301] = b.mask[302] = 0x3ff
    g = _gpu_fit(ctx, b)
    o = O.fit_batch(b, nthreads=8)
    assert np.array_equal(g["status"], o["status"]), np.flatnonzero(g["status"] != o["status"])[:10]
    assert np.array_equal(g["nhits"], o["nhits"])
    assert o["status"][200] == 8 and o["status"][203] == 8 and o["status"][300] == 4 and o["status"][303] == 2
    assert np.all(o["status"][lo:lo + 256] == 1)
    z = o["nhits"] == 0
    assert z.sum() >= 52
    assert np.array_equal(g["par"][:, z], b.par[:, z]) and np.array_equal(g["cov"][:, z], b.cov[:, z])
    assert np.all(g["chi2"][z] == 0)
    sel = o["nhits"] >= 4
    sub_g = {k: (v[..., sel] if k in ("par", "cov") else v[sel]) for k, v in g.items()}
    sub_o = {k: (v[..., sel] if k == "par" else v[sel]) for k, v in o.items()}
    res = compare_fit(_zero_status(sub_g), _zero_status(sub_o), float(b.radius[-1]), max_diverged_frac=0.02)
    print("pair kernel, edge cases:", res)
    # in place, same kernel
    from paper_1705_02876_b200.buffers import DeviceFit
    d = DeviceFit.from_batch(b, "cuda:0")
    ctx.fit_tracks(d.geom, d.n, d.par, d.cov, d.q, d.hpos, d.hcov, d.mask, d.par, d.cov,
                   d.out_chi2, d.out_nhits, d.out_status)
    torch.cuda.synchronize()
    assert np.array_equal(d.par[:, :d.n].cpu().numpy(), g["par"]) and np.array_equal(d.cov[:, :d.n].cpu().numpy(), g["cov"])


def test_fit_in_place(ctx):
    from paper_1705_02876_b200.buffers import DeviceFit
    b = W.simulate_event(W.get_config(1), 10, n_tracks=777)
    ref = _gpu_fit(ctx, b)
    d = DeviceFit.from_batch(b, "cuda:0")
    ctx.fit_tracks(d.geom, d.n, d.par, d.cov, d.q, d.hpos, d.hcov, d.mask, d.par, d.cov,
                   d.out_chi2, d.out_nhits, d.out_status)
    torch.cuda.synchronize()
    assert np.array_equal(d.par[:, :d.n].cpu().numpy(), ref["par"])
    assert np.array_equal(d.cov[:, :d.n].cpu().numpy(), ref["cov"])


def test_fit_host_path_equals_device_path(ctx):
    from paper_1705_02876_b200.buffers import DeviceFit
    b = W.make_fit_batch(1)
    ref = _gpu_fit(ctx, b)
    h = DeviceFit.from_batch(b, "cpu", pin=True)
    h.fit_host(ctx)
    r = h.results()
    for k in ref:
        assert np.array_equal(ref[k], r[k]), k


def test_fit_host_path_equals_device_path_across_chunks(ctx):
    """A batch large enough for the two-tracks-per-thread kernels (14 events = 280 000 tracks, holes in the masks of
    some) goes through kf_fit_tracks_host in three chunks (94 208 tracks each at this size): every chunk takes the kernel the whole batch
    takes on the device path, so the two agree bit for bit, chunk boundaries and the ragged last chunk included."""
    from paper_1705_02876_b200.buffers import DeviceFit
    b = W.make_fit_batch(2, n_events=14)
    rng = np.random.default_rng(77)
    holes = rng.random(b.n) < 0.05
    b.mask = b.mask.copy()
    b.mask[holes] &= ~(np.uint32(1) << rng.integers(0, 10, holes.sum()).astype(np.uint32))
    ref = _gpu_fit(ctx, b)
    h = DeviceFit.from_batch(b, "cpu", pin=True)
    h.fit_host(ctx)
    r = h.results()
    for k in ref:
        assert np.array_equal(ref[k], r[k], equal_nan=True), k


def test_fit_host_path_with_diagonal_seed_covariance(ctx):
    """kf_fit_tracks_host_diag: six covariance planes cross the link instead of 21; the seeds of configs[0-3] are
    diagonal (reading A13), and the results are those of the full call, bit for bit, across chunk boundaries."""
    from paper_1705_02876_b200.buffers import DeviceFit
    b = W.make_fit_batch(2, n_events=8)
    off = np.setdiff1d(np.arange(21), [0, 6, 11, 15, 18, 20])
    assert np.all(b.cov[off] == 0.0)
    h = DeviceFit.from_batch(b, "cpu", pin=True)
    h.fit_host(ctx)
    full = h.results()
    h.out_par.zero_(); h.out_cov.zero_(); h.out_chi2.zero_()
    h.fit_host(ctx, cov_diagonal=True)
    diag = h.results()
    for k in full:
        assert np.array_equal(full[k], diag[k], equal_nan=True), k
    assert np.count_nonzero(diag["chi2"]) > 0.99 * b.n


def _local_hit_variances(b, rng=None):
    """[L][3][n] fp32: v_r, v_t, v_z of every hit (the workload's resolutions; with rng, scaled hit by hit so the
    three planes are not constants) and the covariance they stand for, in fp64 from the fp32 positions and variances
    as include/kf_b200.h defines it: V = Rz(phi_h) diag(v_r, v_t, v_z) Rz(phi_h)^T, (cos, sin) phi_h = (x, y) / rho."""
    L, n = b.hpos.shape[0], b.n
    var = np.empty((L, 3, n), dtype=np.float32)
    var[:, 0], var[:, 1], var[:, 2] = W.SIGMA_R ** 2, W.SIGMA_RPHI ** 2, W.SIGMA_Z ** 2
    if rng is not None:
        var *= rng.uniform(0.5, 2.0, size=var.shape).astype(np.float32)
    x, y = b.hpos[:, 0].astype(np.float64), b.hpos[:, 1].astype(np.float64)
    rho2 = x * x + y * y
    ok = rho2 > 0
    c2 = np.where(ok, x * x / np.where(ok, rho2, 1.0), 1.0)
    s2 = np.where(ok, y * y / np.where(ok, rho2, 1.0), 0.0)
    cs = np.where(ok, x * y / np.where(ok, rho2, 1.0), 0.0)
    vr, vt, vz = (var[:, k].astype(np.float64) for k in range(3))
    zero = np.zeros_like(vr)
    full = np.stack([vr * c2 + vt * s2, (vr - vt) * cs, zero, vr * s2 + vt * c2, zero, vz], axis=1)   # [L][6][n]
    return var, full


def test_fit_host_path_with_local_hit_variances(ctx):
    """kf_fit_tracks_host_compact: three variance planes per layer cross the link instead of six covariance planes,
    and the device rebuilds the covariance from the hit position.  (1) parity with the oracle given that covariance
    in fp64, every track of a batch that spans three chunks and a ragged tail, variances that differ hit by hit;
    (2) on the workload's own hits (constant resolutions) the call agrees with the full-covariance call to rounding
    (the workload rotates by the same azimuth, so both describe the same covariance)."""
    import copy
    from paper_1705_02876_b200.buffers import DeviceFit, _to_planes
    b = W.make_fit_batch(2, n_events=14)
    b = copy.copy(b)
    var, full = _local_hit_variances(b, np.random.default_rng(5))
    h = DeviceFit.from_batch(b, "cpu", pin=True)
    hv = _to_planes(var, h.ld, torch.device("cpu"), True)
    h.fit_host(ctx, cov_diagonal=True, hit_var=hv)
    g = h.results()
    sel = slice(0, b.n, 7)                                   # every 7th track through the oracle: 40 000 of them
    o = O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par[:, sel], b.cov[:, sel], b.q[sel], b.hpos[:, :, sel],
                     full[:, :, sel], b.mask[sel], nthreads=8)
    gs = {k: (v[..., sel] if k in ("par", "cov") else v[sel]) for k, v in g.items()}
    res = compare_fit(gs, o, float(b.radius[-1]))
    print("compact host call vs oracle:", res)
    # the tail of the last chunk and the chunk boundaries, one by one
    for lo in (94_208 - 3, 131_072 - 3, 188_416 - 3, 262_144 - 3, b.n - 5):     # (chunks of 94 208 tracks at this size)
        s2 = slice(lo, min(lo + 6, b.n))
        o2 = O.fit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par[:, s2], b.cov[:, s2], b.q[s2], b.hpos[:, :, s2],
                          full[:, :, s2], b.mask[s2])
        compare_fit({k: (v[..., s2] if k in ("par", "cov") else v[s2]) for k, v in g.items()}, o2, float(b.radius[-1]),
                    max_diverged_frac=1.0)
    # (2)
    var0, _ = _local_hit_variances(b)
    h.fit_host(ctx, cov_diagonal=True)
    ref = h.results()
    h.out_par.zero_(); h.out_cov.zero_(); h.out_chi2.zero_()
    h.fit_host(ctx, cov_diagonal=True, hit_var=_to_planes(var0, h.ld, torch.device("cpu"), True))
    r = h.results()
    assert np.array_equal(ref["nhits"], r["nhits"]) and np.array_equal(ref["status"], r["status"])
    ok = ref["status"] == 0
    assert np.allclose(ref["par"][:, ok], r["par"][:, ok], rtol=2e-4, atol=2e-5)
    assert np.allclose(ref["chi2"][ok], r["chi2"][ok], rtol=2e-3, atol=2e-3)
    with pytest.raises(ValueError):
        h.fit_host(ctx, cov_diagonal=False, hit_var=hv)


def test_fit_argument_errors(ctx):
    import paper_1705_02876_b200 as K
    from paper_1705_02876_b200.buffers import DeviceFit
    b = W.simulate_event(W.get_config(1), 5, n_tracks=16)
    d = DeviceFit.from_batch(b, "cuda:0")
    d.out_par.fill_(5.0)
    bad = K.Geometry(d.geom.radius_cm[::-1].copy(), d.geom.x_over_X0, 3.8, 0.13957)
    with pytest.raises(K.KFError) as e:
        ctx.fit_tracks(bad, d.n, d.par, d.cov, d.q, d.hpos, d.hcov, d.mask, d.out_par, d.out_cov,
                       d.out_chi2, d.out_nhits, d.out_status)
    assert e.value.code == -4
    zero_b = K.Geometry(d.geom.radius_cm, d.geom.x_over_X0, 0.0, 0.13957)
    with pytest.raises(K.KFError) as e:
        ctx.fit_tracks(zero_b, d.n, d.par, d.cov, d.q, d.hpos, d.hcov, d.mask, d.out_par, d.out_cov,
                       d.out_chi2, d.out_nhits, d.out_status)
    assert e.value.code == -4
    mis_par = torch.zeros(6 * 20 + 1, dtype=torch.float32, device="cuda:0")[1:].view(6, 20)
    mis_cov = torch.zeros(21, 20, dtype=torch.float32, device="cuda:0")
    with pytest.raises(K.KFError) as e:              # plane pointer off by 4 bytes
        ctx.fit_tracks(d.geom, d.n, mis_par, mis_cov, d.q, d.hpos, d.hcov, d.mask, d.out_par, d.out_cov,
                       d.out_chi2, d.out_nhits, d.out_status)
    assert e.value.code == -3
    with pytest.raises((K.KFError, ValueError)):     # wrong number of hit layers
        ctx.fit_tracks(K.Geometry(d.geom.radius_cm[:5], d.geom.x_over_X0[:5], 3.8, 0.13957), d.n, d.par, d.cov, d.q,
                       d.hpos, d.hcov, d.mask, d.out_par, d.out_cov, d.out_chi2, d.out_nhits, d.out_status)
    torch.cuda.synchronize()
    assert torch.all(d.out_par == 5.0)               # on error no output is written
