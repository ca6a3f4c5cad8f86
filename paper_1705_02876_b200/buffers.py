"""Device-buffer helpers around the binding: allocation and layout only (no arithmetic).

A `DeviceFit` holds the SoA tensors of one kf_fit_tracks call on one GPU, with the plane stride
`ld` padded to a multiple of 4 floats as the ABI requires.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
import torch

from .binding import Geometry, KFContext


def padded_ld(n: int) -> int:
    return max(4, (int(n) + 3) // 4 * 4)


def _to_planes(a: np.ndarray, ld: int, device, pin: bool = False) -> torch.Tensor:
    """[..., n] numpy -> [..., ld] torch tensor (zero padded)."""
    a = np.ascontiguousarray(a)
    n = a.shape[-1]
    t = torch.zeros(a.shape[:-1] + (ld,), dtype=torch.from_numpy(a[..., :0]).dtype,
                    device="cpu", pin_memory=pin)
    t[..., :n] = torch.from_numpy(a)
    return t if str(device) == "cpu" else t.to(device)


@dataclass
class DeviceFit:
    n: int
    ld: int
    geom: Geometry
    par: torch.Tensor
    cov: torch.Tensor
    q: torch.Tensor
    hpos: torch.Tensor
    hcov: torch.Tensor
    mask: torch.Tensor | None
    out_par: torch.Tensor
    out_cov: torch.Tensor
    out_chi2: torch.Tensor
    out_nhits: torch.Tensor
    out_status: torch.Tensor

    @staticmethod
    def from_batch(batch, device="cuda:0", with_mask: bool = True, pin: bool = False) -> "DeviceFit":
        """`batch` is a workloads.barrel_events.FitBatch-shaped object (duck-typed numpy arrays)."""
        n = int(batch.n)
        ld = padded_ld(n)
        geom = Geometry(np.asarray(batch.radius, dtype=np.float32), np.asarray(batch.x_over_X0, dtype=np.float32),
                        float(batch.Bz), float(batch.mass), getattr(batch, "half_length", None),
                        int(getattr(batch, "material_model", 0)), int(getattr(batch, "energy_loss", 0)),
                        getattr(batch, "surface_type", None), getattr(batch, "disc_z", None),
                        getattr(batch, "disc_rmin", None), getattr(batch, "disc_rmax", None))
        dev = device
        mk = lambda shape, dt: torch.zeros(shape, dtype=dt, device=dev, pin_memory=(pin and str(dev) == "cpu"))
        return DeviceFit(
            n=n, ld=ld, geom=geom,
            par=_to_planes(batch.par, ld, dev, pin), cov=_to_planes(batch.cov, ld, dev, pin),
            q=_to_planes(batch.q.astype(np.int8), ld, dev, pin),
            hpos=_to_planes(batch.hpos, ld, dev, pin), hcov=_to_planes(batch.hcov, ld, dev, pin),
            mask=_to_planes(batch.mask.astype(np.uint32).view(np.int32), ld, dev, pin) if with_mask else None,
            out_par=mk((6, ld), torch.float32), out_cov=mk((21, ld), torch.float32),
            out_chi2=mk((ld,), torch.float32), out_nhits=mk((ld,), torch.int32), out_status=mk((ld,), torch.int32))

    def fit(self, ctx: KFContext):
        # the marshalled call is kept as long as the context and the tensors are the same objects
        ts = (self.geom, self.par, self.cov, self.q, self.hpos, self.hcov, self.mask,
              self.out_par, self.out_cov, self.out_chi2, self.out_nhits, self.out_status)
        key = (id(ctx), ctx._h.value, self.n) + tuple(id(t) for t in ts)
        cached = getattr(self, "_prepared_fit", None)
        if cached is None or cached[0] != key:
            cached = (key, ctx.prepare_fit_tracks(self.geom, self.n, *ts[1:]))
            self._prepared_fit = cached
        cached[1]()

    def fit_refit(self, ctx: KFContext, kappa: float = 10.0) -> dict:
        """kf_fit_tracks_refit; the forward result lands in the usual out_* tensors, the smoothed one in
        tensors allocated at the first call, returned and kept as self.refitted (later calls write into them)."""
        dev = self.par.device
        sm = getattr(self, "refitted", None)
        if sm is None:
            mk = lambda shape, dt: torch.zeros(shape, dtype=dt, device=dev)
            sm = dict(par=mk((6, self.ld), torch.float32), cov=mk((21, self.ld), torch.float32),
                      chi2=mk((self.ld,), torch.float32), nhits=mk((self.ld,), torch.int32), status=mk((self.ld,), torch.int32))
        ctx.fit_tracks_refit(self.geom, self.n, self.par, self.cov, self.q, self.hpos, self.hcov, self.mask, kappa,
                              self.out_par, self.out_cov, self.out_chi2, self.out_nhits, self.out_status,
                              sm["par"], sm["cov"], sm["chi2"], sm["nhits"], sm["status"])
        self.refitted = sm
        return sm

    def fit_smooth(self, ctx: KFContext) -> dict:
        """kf_fit_tracks_smooth; the forward result lands in the usual out_* tensors, the per-layer smoothed states
        in tensors allocated at the first call (kept as self.smoothed; later calls write into them)."""
        dev = self.par.device
        sm = getattr(self, "smoothed", None)
        if sm is None:
            L = int(self.geom.radius_cm.shape[0])
            sm = dict(par=torch.zeros((L, 6, self.ld), dtype=torch.float32, device=dev),
                      cov=torch.zeros((L, 21, self.ld), dtype=torch.float32, device=dev),
                      used=torch.zeros((self.ld,), dtype=torch.int32, device=dev))
        ctx.fit_tracks_smooth(self.geom, self.n, self.par, self.cov, self.q, self.hpos, self.hcov, self.mask,
                              self.out_par, self.out_cov, self.out_chi2, self.out_nhits, self.out_status,
                              sm["par"], sm["cov"], sm["used"])
        self.smoothed = sm
        return sm

    def smoothed_results(self) -> dict:
        n, sm = self.n, self.smoothed
        return dict(par=sm["par"][:, :, :n].cpu().numpy(), cov=sm["cov"][:, :, :n].cpu().numpy(),
                    used=sm["used"][:n].cpu().numpy().view(np.uint32))

    def refit_results(self) -> dict:
        n, sm = self.n, self.refitted
        return dict(par=sm["par"][:, :n].cpu().numpy(), cov=sm["cov"][:, :n].cpu().numpy(),
                    chi2=sm["chi2"][:n].cpu().numpy(), nhits=sm["nhits"][:n].cpu().numpy(),
                    status=sm["status"][:n].cpu().numpy().view(np.uint32))

    def fit_host(self, ctx: KFContext, cov_diagonal: bool = False, hit_var: torch.Tensor | None = None):
        """kf_fit_tracks_host; cov_diagonal: kf_fit_tracks_host_diag with the six diagonal planes of self.cov (kept as
        self.cov_diag, pinned like the rest; the caller asserts that the seed covariance IS diagonal).  hit_var (a host
        [L][3][ld] tensor, with cov_diagonal): kf_fit_tracks_host_compact, the variances of every hit along its own
        r^, t^, z^ in place of self.hcov."""
        cov = self.cov
        if cov_diagonal:
            cov = getattr(self, "cov_diag", None)
            if cov is None:
                cov = torch.empty((6, self.ld), dtype=torch.float32, pin_memory=self.cov.is_pinned())
                cov.copy_(self.cov[[0, 6, 11, 15, 18, 20]])
                self.cov_diag = cov
        ctx.fit_tracks_host(self.geom, self.n, self.par, cov, self.q, self.hpos, self.hcov if hit_var is None else hit_var,
                            self.mask, self.out_par, self.out_cov, self.out_chi2, self.out_nhits, self.out_status,
                            cov_diagonal, hit_var is not None)

    def results(self) -> dict:
        """Copies of the outputs (also when the buffers are host tensors: a later call must not change them)."""
        n = self.n
        host = lambda t: np.array(t.cpu().numpy(), copy=True)
        return dict(par=host(self.out_par[:, :n]), cov=host(self.out_cov[:, :n]),
                    chi2=host(self.out_chi2[:n]), nhits=host(self.out_nhits[:n]),
                    status=host(self.out_status[:n]).view(np.uint32))

    @property
    def algorithmic_bytes(self) -> int:
        """HBM bytes one fit must move: 113 in + 120 out + 36 per layer, per track."""
        L = int(self.geom.radius_cm.shape[0])
        return self.n * (233 + 36 * L)


@dataclass
class DeviceLayer:
    """All hits of one layer on the GPU plus the caller-allocated outputs of kf_bin_hits."""
    n_hits: int
    ld: int
    pos: torch.Tensor      # f32 [3][ld] original order
    cov: torch.Tensor      # f32 [6][ld]
    bins: "Bins"

    @staticmethod
    def from_numpy(pos: np.ndarray, cov: np.ndarray, n_eta: int, n_phi: int, eta_max: float,
                   device="cuda:0", soa: bool = True) -> "DeviceLayer":
        """soa = False: no SoA copy of the sorted hits (kf_layer_bins.pos_sorted / cov_sorted NULL): scoring and
        building read the packed records only."""
        from .binding import Bins
        n = int(pos.shape[1])
        ld = padded_ld(n)
        return DeviceLayer(n, ld, _to_planes(pos.astype(np.float32), ld, device),
                           _to_planes(cov.astype(np.float32), ld, device),
                           Bins.allocate(n, n_eta, n_phi, eta_max, device, soa))

    def bin(self, ctx: KFContext, radius_cm: float):
        ctx.bin_hits(radius_cm, self.n_hits, self.pos, self.cov, self.bins)


@dataclass
class DeviceCandidates:
    """Track candidates advanced in place, layer by layer, by kf_score_candidates."""
    n: int
    ld: int
    par: torch.Tensor
    cov: torch.Tensor
    q: torch.Tensor
    chi2: torch.Tensor
    nhits: torch.Tensor
    status: torch.Tensor
    best_hit: torch.Tensor
    best_chi2: torch.Tensor

    @staticmethod
    def from_numpy(par, cov21, q, chi2=None, nhits=None, device="cuda:0") -> "DeviceCandidates":
        n = int(par.shape[1])
        ld = padded_ld(n)
        z = lambda dt: torch.zeros(ld, dtype=dt, device=device)
        c = DeviceCandidates(n, ld, _to_planes(np.asarray(par, dtype=np.float32), ld, device),
                             _to_planes(np.asarray(cov21, dtype=np.float32), ld, device),
                             _to_planes(np.asarray(q, dtype=np.int8), ld, device),
                             z(torch.float32), z(torch.int32), z(torch.int32), z(torch.int32), z(torch.float32))
        if chi2 is not None:
            c.chi2[:n] = torch.from_numpy(np.asarray(chi2, dtype=np.float32)).to(device)
        if nhits is not None:
            c.nhits[:n] = torch.from_numpy(np.asarray(nhits, dtype=np.int32)).to(device)
        return c

    def score(self, ctx: KFContext, geom: Geometry, layer: int, hits: DeviceLayer, window_half: int = 2,
              chi2_cut: float = 30.0, do_update: bool = True, order: torch.Tensor | None = None,
              keep_local: bool = True, static_scratch: bool = False):
        """kf_score_candidates on one layer.  keep_local: carry the candidates' local-frame state between the
        per-layer calls (allocated and zeroed at the first call; see the header).  static_scratch: the no-allocation
        entry point kf_score_candidates_static (at most STATIC_MAX_CANDIDATES candidates)."""
        ls = None
        if keep_local:
            ls = getattr(self, "local_state", None)
            if ls is None:
                ls = self.local_state = torch.zeros((30, self.ld), dtype=torch.float32, device=self.par.device)
        ctx.score_candidates(geom, layer, self.n, self.par, self.cov, self.q, self.chi2, self.nhits, self.status,
                             hits.n_hits, hits.pos, hits.cov, hits.bins, window_half, chi2_cut, do_update,
                             self.best_hit, self.best_chi2, order, ls, static_scratch)

    def build(self, ctx: KFContext, geom: Geometry, first_layer: int, layers: list, window_half: int = 2,
              chi2_cut: float = 30.0, do_update: bool = True, order: torch.Tensor | None = None):
        """kf_build_best_hit over `layers` (DeviceLayer list for first_layer, first_layer+1, ...).
        Returns (hit_index[len(layers)][ld], hit_chi2[len(layers)][ld]) device tensors."""
        m = len(layers)
        idx = torch.empty((m, self.ld), dtype=torch.int32, device=self.par.device)
        c2 = torch.empty((m, self.ld), dtype=torch.float32, device=self.par.device)
        ctx.build_best_hit(geom, first_layer, self.n, self.par, self.cov, self.q, self.chi2, self.nhits, self.status,
                           [(l.n_hits, l.pos, l.cov, l.bins) for l in layers], window_half, chi2_cut, do_update,
                           idx, c2, order)
        return idx, c2

    def build_combinatorial(self, ctx: KFContext, geom: Geometry, first_layer: int, layers: list, n_cand: int,
                            window_half: int = 2, chi2_cut: float = 30.0):
        """kf_build_combinatorial; returns (hit_index[len(layers)][ld], n_found[ld]) device tensors."""
        idx = torch.empty((len(layers), self.ld), dtype=torch.int32, device=self.par.device)
        nf = torch.zeros(self.ld, dtype=torch.int32, device=self.par.device)
        ctx.build_combinatorial(geom, first_layer, self.n, self.par, self.cov, self.q, self.chi2, self.nhits,
                                self.status, [(l.n_hits, l.pos, l.cov, l.bins) for l in layers], window_half,
                                chi2_cut, n_cand, idx, nf)
        return idx, nf

    def make_order(self, ctx: KFContext, geom: Geometry, layer: int, n_eta: int, n_phi: int, eta_max: float):
        order = torch.empty(max(self.n, 1), dtype=torch.int32, device=self.par.device)
        ctx.order_candidates(geom, layer, self.n, self.par, self.cov, self.q, self.chi2, self.nhits, self.status,
                             n_eta, n_phi, eta_max, order)
        return order

    def results(self) -> dict:
        n = self.n
        return dict(par=self.par[:, :n].cpu().numpy(), cov=self.cov[:, :n].cpu().numpy(),
                    chi2=self.chi2[:n].cpu().numpy(), nhits=self.nhits[:n].cpu().numpy(),
                    status=self.status[:n].cpu().numpy().view(np.uint32),
                    best_hit=self.best_hit[:n].cpu().numpy(), best_chi2=self.best_chi2[:n].cpu().numpy())
