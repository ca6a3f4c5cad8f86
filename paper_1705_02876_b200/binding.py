"""ctypes binding of include/kf_b200.h: argument marshalling only.

Every step of the path (propagation, covariance transport, update, chi2, binning, scoring) runs in
the CUDA kernels behind the C ABI; this module only turns torch tensors (device memory, streams)
into the plain pointers and sizes the ABI takes.  Names follow the header: KFContext.fit_tracks ->
kf_fit_tracks, .fit_tracks_host -> kf_fit_tracks_host, .bin_hits -> kf_bin_hits,
.score_candidates -> kf_score_candidates.
"""
from __future__ import annotations

import ctypes as C
import math
import os
from dataclasses import dataclass

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("KF_B200_LIB") or os.path.join(_HERE, "libkf_b200.so")   # override: kernel experiments

STATUS_PROP_FAIL, STATUS_S_NOT_PD, STATUS_NONFINITE, STATUS_BAD_CHARGE, STATUS_OUTSIDE = 1, 2, 4, 8, 16
OPT_PAIR_MIN_TRACKS, OPT_REFIT_PAIR_MASKED, OPT_BIN_FORM = 1, 2, 3          # kf_set_option
BIN_FORM_AUTO, BIN_FORM_FIVE_LAUNCH, BIN_FORM_CHUNKED = 0, 1, 2
STATIC_MAX_CANDIDATES = 65536                                               # KF_STATIC_MAX_CANDIDATES
ERR_TOO_LARGE = -8
EXPORTS = ["kf_create", "kf_destroy", "kf_set_stream", "kf_set_option", "kf_reserve", "kf_strerror", "kf_last_cuda_error",
           "kf_abi_version", "kf_hit_record_floats", "kf_measure_fp32_peak", "kf_measure_fp32_packed_rate", "kf_fit_tracks", "kf_fit_tracks_indexed", "kf_fit_tracks_refit", "kf_fit_tracks_smooth", "kf_fit_tracks_host", "kf_fit_tracks_host_diag", "kf_fit_tracks_host_compact", "kf_bin_hits", "kf_bin_layers", "kf_order_candidates",
           "kf_score_candidates", "kf_score_candidates_static", "kf_build_best_hit", "kf_build_best_hit_events", "kf_build_best_hit_host", "kf_build_combinatorial", "kf_build_combinatorial_events",
           "kf_graph_begin", "kf_graph_end", "kf_graph_launch", "kf_graph_destroy"]


class KFError(RuntimeError):
    def __init__(self, code: int, what: str, cuda: int = 0):
        super().__init__(f"{what}: {strerror(code)} (code {code}" + (f", cudaError {cuda})" if cuda else ")"))
        self.code = code
        self.cuda = cuda


class _Geometry(C.Structure):
    _fields_ = [("n_layers", C.c_int), ("radius_cm", C.POINTER(C.c_float)), ("x_over_X0", C.POINTER(C.c_float)),
                ("Bz_tesla", C.c_float), ("mass_gev", C.c_float),
                ("half_length_cm", C.POINTER(C.c_float)), ("material_model", C.c_int),
                ("energy_loss_model", C.c_int), ("surface_type", C.POINTER(C.c_int32)),
                ("disc_z_cm", C.POINTER(C.c_float)), ("disc_rmin_cm", C.POINTER(C.c_float)),
                ("disc_rmax_cm", C.POINTER(C.c_float))]


class _Tracks(C.Structure):
    _fields_ = [("n", C.c_int64), ("ld", C.c_int64), ("par", C.c_void_p), ("cov", C.c_void_p), ("q", C.c_void_p),
                ("chi2", C.c_void_p), ("nhits", C.c_void_p), ("status", C.c_void_p)]


class _TrackHits(C.Structure):
    _fields_ = [("n_layers", C.c_int), ("n", C.c_int64), ("ld", C.c_int64), ("pos", C.c_void_p), ("cov", C.c_void_p),
                ("mask", C.c_void_p)]


class _Smoothed(C.Structure):
    _fields_ = [("n_layers", C.c_int), ("n", C.c_int64), ("ld", C.c_int64), ("par", C.c_void_p), ("cov", C.c_void_p),
                ("used", C.c_void_p)]


class _LayerHits(C.Structure):
    _fields_ = [("n_hits", C.c_int64), ("ld", C.c_int64), ("pos", C.c_void_p), ("cov", C.c_void_p)]


class _LayerBins(C.Structure):
    _fields_ = [("n_eta", C.c_int), ("n_phi", C.c_int), ("eta_max", C.c_float), ("ld", C.c_int64),
                ("bin_offset", C.c_void_p), ("sorted_to_orig", C.c_void_p), ("hit_rec", C.c_void_p),
                ("bin_box", C.c_void_p), ("orig_to_sorted", C.c_void_p), ("pos_sorted", C.c_void_p), ("cov_sorted", C.c_void_p)]


_lib = None


def lib_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen libkf_b200.so (built by `python -m paper_1705_02876_b200.build`).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH) and "KF_B200_LIB" not in os.environ:
        try:                                   # safety net: compile in-tree if nvcc is around
            from . import build as _build
            _build.build()
        except Exception as exc:               # noqa: BLE001 -- any failure ends in the loud error below
            raise ImportError(f"{_LIB_PATH} is missing and could not be built ({exc}); run "
                              "`python -m paper_1705_02876_b200.build` (there is no CPU or PyTorch fallback)")
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_1705_02876_b200.build` "
                          "(there is no CPU or PyTorch fallback)")
    lib = C.CDLL(_LIB_PATH)
    vp = C.c_void_p
    lib.kf_create.restype = C.c_int
    lib.kf_create.argtypes = [C.POINTER(vp), C.c_int, vp]
    lib.kf_destroy.restype = C.c_int
    lib.kf_destroy.argtypes = [vp]
    lib.kf_set_stream.restype = C.c_int
    lib.kf_set_stream.argtypes = [vp, vp]
    lib.kf_set_option.restype = C.c_int
    lib.kf_set_option.argtypes = [vp, C.c_int, C.c_int64]
    lib.kf_reserve.restype = C.c_int
    lib.kf_reserve.argtypes = [vp, C.c_int64, C.c_int64, C.c_int]
    lib.kf_strerror.restype = C.c_char_p
    lib.kf_strerror.argtypes = [C.c_int]
    lib.kf_last_cuda_error.restype = C.c_int
    lib.kf_last_cuda_error.argtypes = [vp]
    lib.kf_measure_fp32_peak.restype = C.c_int
    lib.kf_measure_fp32_peak.argtypes = [vp, C.c_int, C.POINTER(C.c_double)]
    lib.kf_measure_fp32_packed_rate.restype = C.c_int
    lib.kf_measure_fp32_packed_rate.argtypes = [vp, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.kf_abi_version.restype = C.c_int
    lib.kf_abi_version.argtypes = []
    lib.kf_hit_record_floats.restype = C.c_int
    lib.kf_hit_record_floats.argtypes = []
    for name in ("kf_fit_tracks", "kf_fit_tracks_host", "kf_fit_tracks_host_diag", "kf_fit_tracks_host_compact"):
        f = getattr(lib, name)
        f.restype = C.c_int
        f.argtypes = [vp, C.POINTER(_Geometry), C.POINTER(_Tracks), C.POINTER(_TrackHits), C.POINTER(_Tracks)]
    lib.kf_fit_tracks_indexed.restype = C.c_int
    lib.kf_fit_tracks_indexed.argtypes = [vp, C.POINTER(_Geometry), C.POINTER(_Tracks), vp, C.c_int64,
                                          C.POINTER(_LayerHits), C.POINTER(_LayerBins), C.POINTER(_Tracks)]
    lib.kf_fit_tracks_refit.restype = C.c_int
    lib.kf_fit_tracks_refit.argtypes = [vp, C.POINTER(_Geometry), C.POINTER(_Tracks), C.POINTER(_TrackHits), C.c_float,
                                         C.POINTER(_Tracks), C.POINTER(_Tracks)]
    lib.kf_fit_tracks_smooth.restype = C.c_int
    lib.kf_fit_tracks_smooth.argtypes = [vp, C.POINTER(_Geometry), C.POINTER(_Tracks), C.POINTER(_TrackHits),
                                         C.POINTER(_Tracks), C.POINTER(_Smoothed)]
    lib.kf_bin_hits.restype = C.c_int
    lib.kf_bin_hits.argtypes = [vp, C.c_float, C.POINTER(_LayerHits), C.POINTER(_LayerBins)]
    lib.kf_bin_layers.restype = C.c_int
    lib.kf_bin_layers.argtypes = [vp, C.c_int, C.POINTER(C.c_float), C.POINTER(_LayerHits), C.POINTER(_LayerBins)]
    lib.kf_order_candidates.restype = C.c_int
    lib.kf_order_candidates.argtypes = [vp, C.POINTER(_Geometry), C.c_int, C.POINTER(_Tracks), C.c_int, C.c_int,
                                        C.c_float, vp]
    lib.kf_score_candidates.restype = C.c_int
    lib.kf_score_candidates.argtypes = [vp, C.POINTER(_Geometry), C.c_int, C.POINTER(_Tracks), C.POINTER(_LayerHits),
                                        C.POINTER(_LayerBins), C.c_int, C.c_float, C.c_int, vp, vp, vp, vp]
    lib.kf_score_candidates_static.restype = C.c_int
    lib.kf_score_candidates_static.argtypes = lib.kf_score_candidates.argtypes
    lib.kf_build_best_hit.restype = C.c_int
    lib.kf_build_best_hit.argtypes = [vp, C.POINTER(_Geometry), C.c_int, C.c_int, C.POINTER(_Tracks),
                                      C.POINTER(_LayerHits), C.POINTER(_LayerBins), C.c_int, C.c_float, C.c_int,
                                      vp, vp, vp, C.c_int64]
    lib.kf_build_best_hit_events.restype = C.c_int
    lib.kf_build_best_hit_events.argtypes = [vp, C.POINTER(_Geometry), C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int64),
                                             C.POINTER(_Tracks), C.POINTER(_LayerHits), C.POINTER(_LayerBins), C.c_int,
                                             C.c_float, C.c_int, vp, vp, C.c_int64]
    lib.kf_build_best_hit_host.restype = C.c_int
    lib.kf_build_best_hit_host.argtypes = [vp, C.POINTER(_Geometry), C.c_int, C.c_int, C.POINTER(_Tracks),
                                           C.POINTER(_LayerHits), C.c_int, C.c_int, C.c_float, C.c_int, C.c_float,
                                           C.c_int, vp, vp, C.c_int64]
    lib.kf_build_combinatorial.restype = C.c_int
    lib.kf_build_combinatorial.argtypes = [vp, C.POINTER(_Geometry), C.c_int, C.c_int, C.POINTER(_Tracks),
                                           C.POINTER(_LayerHits), C.POINTER(_LayerBins), C.c_int, C.c_float, C.c_int,
                                           vp, vp, C.c_int64]
    lib.kf_build_combinatorial_events.restype = C.c_int
    lib.kf_build_combinatorial_events.argtypes = [vp, C.POINTER(_Geometry), C.c_int, C.c_int, C.c_int,
                                                  C.POINTER(C.c_int64), C.POINTER(_Tracks), C.POINTER(_LayerHits),
                                                  C.POINTER(_LayerBins), C.c_int, C.c_float, C.c_int, vp, vp, C.c_int64]
    lib.kf_graph_begin.restype = C.c_int
    lib.kf_graph_begin.argtypes = [vp]
    lib.kf_graph_end.restype = C.c_int
    lib.kf_graph_end.argtypes = [vp, C.POINTER(vp)]
    lib.kf_graph_launch.restype = C.c_int
    lib.kf_graph_launch.argtypes = [vp, vp]
    lib.kf_graph_destroy.restype = C.c_int
    lib.kf_graph_destroy.argtypes = [vp]
    _lib = lib
    return lib


class Graph:
    """A recorded sequence of hot calls (kf_graph); launch() enqueues it on the context's stream."""

    def __init__(self, ctx: "KFContext", handle):
        self._ctx, self._g = ctx, handle

    def launch(self):
        self._ctx._check(self._ctx._lib.kf_graph_launch(self._ctx._h, self._g), "kf_graph_launch")

    def close(self):
        if self._g:
            load_library().kf_graph_destroy(self._g)
            self._g = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def strerror(code: int) -> str:
    return load_library().kf_strerror(int(code)).decode()


def abi_version() -> int:
    return int(load_library().kf_abi_version())


def hit_record_floats() -> int:
    """Floats per packed hit record (kf_layer_bins.hit_rec) of the loaded library."""
    return int(load_library().kf_hit_record_floats())


@dataclass
class Geometry:
    """Concentric cylinders in a uniform solenoid field (host-side numbers)."""
    radius_cm: np.ndarray
    x_over_X0: np.ndarray
    Bz_tesla: float
    mass_gev: float
    half_length_cm: np.ndarray | None = None   # reading A20: barrel half lengths, None = unbounded
    material_model: int = 0                    # reading A20: 1 = thickness / cos(incidence angle)
    energy_loss_model: int = 0                 # reading A21: 1 = mean Bethe loss in silicon at every crossing
    surface_type: np.ndarray | None = None     # reading A23: 0 = barrel, 1 = disc pair; None = all barrels
    disc_z_cm: np.ndarray | None = None
    disc_rmin_cm: np.ndarray | None = None
    disc_rmax_cm: np.ndarray | None = None

    def _c(self):
        r = np.ascontiguousarray(self.radius_cm, dtype=np.float32)
        t = np.ascontiguousarray(self.x_over_X0, dtype=np.float32)
        h = None if self.half_length_cm is None else np.ascontiguousarray(self.half_length_cm, dtype=np.float32)
        if h is not None and h.shape != r.shape:
            raise ValueError("half_length_cm must have one entry per layer")
        fp = lambda a: C.POINTER(C.c_float)() if a is None else a.ctypes.data_as(C.POINTER(C.c_float))
        st = None if self.surface_type is None else np.ascontiguousarray(self.surface_type, dtype=np.int32)
        dz, lo, hi = (None if a is None else np.ascontiguousarray(a, dtype=np.float32)
                      for a in (self.disc_z_cm, self.disc_rmin_cm, self.disc_rmax_cm))
        for a in (st, dz, lo, hi):
            if a is not None and a.shape != r.shape:
                raise ValueError("surface arrays must have one entry per layer")
        stp = C.POINTER(C.c_int32)() if st is None else st.ctypes.data_as(C.POINTER(C.c_int32))
        g = _Geometry(int(r.shape[0]), r.ctypes.data_as(C.POINTER(C.c_float)), t.ctypes.data_as(C.POINTER(C.c_float)),
                      float(self.Bz_tesla), float(self.mass_gev), fp(h), int(self.material_model),
                      int(self.energy_loss_model), stp, fp(dz), fp(lo), fp(hi))
        return g, (r, t, h, st, dz, lo, hi)       # keep the arrays alive while g is in use


@dataclass
class Bins:
    """Caller-allocated outputs of kf_bin_hits for one layer (all torch CUDA tensors)."""
    n_eta: int
    n_phi: int
    eta_max: float
    bin_offset: torch.Tensor      # int32 [n_eta*n_phi + 1]
    sorted_to_orig: torch.Tensor  # int32 [n_hits]
    hit_rec: torch.Tensor         # f32 [n_hits][hit_record_floats()] packed records in bin order
    bin_box: torch.Tensor         # f32 [n_bins][8] per-bin bounds
    orig_to_sorted: torch.Tensor  # int32 [n_hits] inverse of sorted_to_orig
    pos_sorted: torch.Tensor | None = None   # f32 [3][ld] optional SoA copy
    cov_sorted: torch.Tensor | None = None   # f32 [6][ld]

    @staticmethod
    def allocate(n_hits: int, n_eta: int, n_phi: int, eta_max: float, device, soa: bool = True) -> "Bins":
        ld = max(4, (n_hits + 3) // 4 * 4)
        return Bins(n_eta, n_phi, eta_max,
                    torch.empty(n_eta * n_phi + 1, dtype=torch.int32, device=device),
                    torch.empty(max(n_hits, 1), dtype=torch.int32, device=device),
                    torch.empty((max(n_hits, 1), hit_record_floats()), dtype=torch.float32, device=device),
                    torch.empty((n_eta * n_phi, 8), dtype=torch.float32, device=device),
                    torch.empty(max(n_hits, 1), dtype=torch.int32, device=device),
                    torch.empty((3, ld), dtype=torch.float32, device=device) if soa else None,
                    torch.empty((6, ld), dtype=torch.float32, device=device) if soa else None)

    def _c(self):
        ld = int(self.pos_sorted.shape[1]) if self.pos_sorted is not None else 0
        return _LayerBins(self.n_eta, self.n_phi, float(self.eta_max), ld,
                          self.bin_offset.data_ptr(), self.sorted_to_orig.data_ptr(), self.hit_rec.data_ptr(),
                          self.bin_box.data_ptr(), self.orig_to_sorted.data_ptr(),
                          self.pos_sorted.data_ptr() if self.pos_sorted is not None else None,
                          self.cov_sorted.data_ptr() if self.cov_sorted is not None else None)


def _plane_ld(t: torch.Tensor, rows: int) -> int:
    """A [rows][ld] (or [L][k][ld]) tensor whose last dimension is contiguous and planes are ld apart."""
    if t.stride(-1) != 1:
        raise ValueError("last dimension must be contiguous")
    ld = t.stride(-2) if t.dim() >= 2 else t.shape[-1]
    if t.dim() == 3 and t.stride(0) != t.shape[1] * ld:
        raise ValueError("layer planes must be densely stacked")
    flat_rows = math.prod(t.shape[:-1])
    if flat_rows != rows:
        raise ValueError(f"expected {rows} planes, got {flat_rows}")
    return int(ld)


class KFContext:
    """kf_ctx*: one per device/stream.  Methods mirror the C ABI; tensors are torch (CUDA for the
    device calls, CPU -- ideally pinned -- for fit_tracks_host)."""

    def __init__(self, device: int | torch.device = 0, stream: torch.cuda.Stream | None = None):
        self._lib = load_library()
        self._h = C.c_void_p()
        dev = torch.device(device) if not isinstance(device, int) else torch.device("cuda", device)
        self.device = dev
        idx = dev.index if dev.index is not None else 0
        sptr = C.c_void_p(stream.cuda_stream if stream is not None else
                          (torch.cuda.current_stream(dev).cuda_stream if torch.cuda.is_available() else 0))
        rc = self._lib.kf_create(C.byref(self._h), idx, sptr)
        if rc != 0:
            raise KFError(rc, "kf_create")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.kf_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int, what: str):
        if rc != 0:
            raise KFError(rc, what, self._lib.kf_last_cuda_error(self._h))

    def set_stream(self, stream: torch.cuda.Stream | None):
        s = stream.cuda_stream if stream is not None else torch.cuda.current_stream(self.device).cuda_stream
        self._check(self._lib.kf_set_stream(self._h, C.c_void_p(s)), "kf_set_stream")

    def set_option(self, option: int, value: int):
        self._check(self._lib.kf_set_option(self._h, int(option), int(value)), "kf_set_option")

    # ------------------------------------------------------------------ kf_graph_*
    def graph_begin(self):
        """Start recording the hot calls made on this context (kf_graph_begin)."""
        self._check(self._lib.kf_graph_begin(self._h), "kf_graph_begin")

    def graph_end(self) -> "Graph":
        out = C.c_void_p()
        self._check(self._lib.kf_graph_end(self._h, C.byref(out)), "kf_graph_end")
        return Graph(self, out)

    def reserve(self, max_hits: int = 0, max_host_tracks: int = 0, max_host_layers: int = 0):
        self._check(self._lib.kf_reserve(self._h, max_hits, max_host_tracks, max_host_layers), "kf_reserve")

    def measure_fp32_peak(self, repeats: int = 5) -> float:
        """TFLOP/s of the register-only FMA microbenchmark (ALU roofline denominator)."""
        out = C.c_double(0.0)
        self._check(self._lib.kf_measure_fp32_peak(self._h, int(repeats), C.byref(out)), "kf_measure_fp32_peak")
        return float(out.value)

    def measure_fp32_packed_rate(self, repeats: int = 5) -> tuple[float, float]:
        """(shared, distinct) TFLOP/s of FFMA2 with shared operands / with three distinct register pairs."""
        a, b = C.c_double(0.0), C.c_double(0.0)
        self._check(self._lib.kf_measure_fp32_packed_rate(self._h, int(repeats), C.byref(a), C.byref(b)),
                    "kf_measure_fp32_packed_rate")
        return float(a.value), float(b.value)

    # ------------------------------------------------------------------ marshalling helpers
    @staticmethod
    def _tracks(n, par, cov, q, chi2, nhits, status) -> _Tracks:
        ld = _plane_ld(par, 6)
        if _plane_ld(cov, 21) != ld:
            raise ValueError("par and cov must share the plane stride ld")
        return _Tracks(int(n), ld, par.data_ptr(), cov.data_ptr(), q.data_ptr() if q is not None else None,
                       chi2.data_ptr(), nhits.data_ptr(), status.data_ptr())

    @staticmethod
    def _track_hits(n, L, hpos, hcov, mask, cov_planes=6) -> _TrackHits:
        ld = _plane_ld(hpos, 3 * L)
        if _plane_ld(hcov, cov_planes * L) != ld:
            raise ValueError("hpos and hcov must share the plane stride ld")
        return _TrackHits(int(L), int(n), ld, hpos.data_ptr(), hcov.data_ptr(),
                          mask.data_ptr() if mask is not None else None)

    # ------------------------------------------------------------------ kf_fit_tracks
    def fit_tracks(self, geom: Geometry, n: int, par, cov, q, hpos, hcov, mask,
                   out_par, out_cov, out_chi2, out_nhits, out_status):
        """Enqueue one fit of n tracks (device tensors; SoA [6][ld], [21][ld], [L][3][ld], [L][6][ld])."""
        g, keep = geom._c()
        seeds = self._tracks(n, par, cov, q, out_chi2, out_nhits, out_status)
        out = self._tracks(n, out_par, out_cov, None, out_chi2, out_nhits, out_status)
        hits = self._track_hits(n, g.n_layers, hpos, hcov, mask)
        self._check(self._lib.kf_fit_tracks(self._h, C.byref(g), C.byref(seeds), C.byref(hits), C.byref(out)),
                    "kf_fit_tracks")
        del keep

    def prepare_fit_tracks(self, geom: Geometry, n: int, par, cov, q, hpos, hcov, mask,
                           out_par, out_cov, out_chi2, out_nhits, out_status):
        """The marshalling of fit_tracks done once: returns a callable that enqueues the same kf_fit_tracks call
        again (for event after event through the same tensors: the ctypes structures are what an eager
        event-sized call spends most of its 20 us on).  The tensors must stay alive and in place."""
        g, keep = geom._c()
        seeds = self._tracks(n, par, cov, q, out_chi2, out_nhits, out_status)
        out = self._tracks(n, out_par, out_cov, None, out_chi2, out_nhits, out_status)
        hits = self._track_hits(n, g.n_layers, hpos, hcov, mask)
        fn, h, check = self._lib.kf_fit_tracks, self._h, self._check
        rg, rs, rh, ro = C.byref(g), C.byref(seeds), C.byref(hits), C.byref(out)
        alive = (keep, g, seeds, out, hits, par, cov, q, hpos, hcov, mask, out_par, out_cov, out_chi2, out_nhits, out_status)

        def launch(_alive=alive):
            if not h.value or h.value != self._h.value:
                raise KFError(-1, "kf_fit_tracks (prepared call: its context is closed)")
            rc = fn(h, rg, rs, rh, ro)
            if rc != 0:
                check(rc, "kf_fit_tracks")
        return launch

    def fit_tracks_indexed(self, geom: Geometry, n: int, par, cov, q, index, pools,
                           out_par, out_cov, out_chi2, out_nhits, out_status, bins=None):
        """Fit with hits addressed by index: index int32 [L][ld_index] (device), pools = [(n_hits, pos, cov), ...]
        one per geometry layer."""
        g, keep = geom._c()
        seeds = self._tracks(n, par, cov, q, out_chi2, out_nhits, out_status)
        out = self._tracks(n, out_par, out_cov, None, out_chi2, out_nhits, out_status)
        m = len(pools)
        if m != g.n_layers or index.shape[0] != m:
            raise ValueError("one pool and one index row per geometry layer")
        lhs = (_LayerHits * m)(*[self._layer_hits(nh, p, c) for (nh, p, c) in pools])
        lbs = (_LayerBins * m)(*[b._c() for b in bins]) if bins is not None else None
        self._check(self._lib.kf_fit_tracks_indexed(self._h, C.byref(g), C.byref(seeds), index.data_ptr(),
                                                    int(index.stride(0)), lhs, lbs, C.byref(out)),
                    "kf_fit_tracks_indexed")
        del keep

    def fit_tracks_refit(self, geom: Geometry, n: int, par, cov, q, hpos, hcov, mask, kappa: float,
                          out_par, out_cov, out_chi2, out_nhits, out_status,
                          s_par, s_cov, s_chi2, s_nhits, s_status):
        """Forward fit + inward refit (reading A18) in one kernel; two result sets."""
        g, keep = geom._c()
        seeds = self._tracks(n, par, cov, q, out_chi2, out_nhits, out_status)
        out = self._tracks(n, out_par, out_cov, None, out_chi2, out_nhits, out_status)
        sm = self._tracks(n, s_par, s_cov, None, s_chi2, s_nhits, s_status)
        hits = self._track_hits(n, g.n_layers, hpos, hcov, mask)
        self._check(self._lib.kf_fit_tracks_refit(self._h, C.byref(g), C.byref(seeds), C.byref(hits), float(kappa),
                                                   C.byref(out), C.byref(sm)), "kf_fit_tracks_refit")
        del keep

    def fit_tracks_smooth(self, geom: Geometry, n: int, par, cov, q, hpos, hcov, mask,
                          out_par, out_cov, out_chi2, out_nhits, out_status, s_par, s_cov, s_used):
        """Forward fit + RTS smoother (kf_fit_tracks_smooth): s_par [L][6][ld], s_cov [L][21][ld] float32 and
        s_used [n] int32 device tensors receive the smoothed state of every used layer and the used-layer mask."""
        g, keep = geom._c()
        seeds = self._tracks(n, par, cov, q, out_chi2, out_nhits, out_status)
        out = self._tracks(n, out_par, out_cov, None, out_chi2, out_nhits, out_status)
        hits = self._track_hits(n, g.n_layers, hpos, hcov, mask)
        ld = _plane_ld(s_par, 6 * g.n_layers)
        if _plane_ld(s_cov, 21 * g.n_layers) != ld:
            raise ValueError("s_par and s_cov must share the plane stride ld")
        sm = _Smoothed(g.n_layers, int(n), ld, s_par.data_ptr(), s_cov.data_ptr(), s_used.data_ptr())
        self._check(self._lib.kf_fit_tracks_smooth(self._h, C.byref(g), C.byref(seeds), C.byref(hits), C.byref(out),
                                                   C.byref(sm)), "kf_fit_tracks_smooth")
        del keep

    def fit_tracks_host(self, geom: Geometry, n: int, par, cov, q, hpos, hcov, mask,
                        out_par, out_cov, out_chi2, out_nhits, out_status, cov_diagonal: bool = False,
                        hit_cov_local: bool = False):
        """Same with HOST tensors (pinned for full overlap); returns when the outputs are complete.
        cov_diagonal: `cov` is [6][ld], the diagonal of the seed covariance (kf_fit_tracks_host_diag).
        hit_cov_local (with cov_diagonal): `hcov` is [L][3][ld], the variances of each hit along its own r^, t^, z^
        (kf_fit_tracks_host_compact)."""
        if hit_cov_local and not cov_diagonal:
            raise ValueError("hit_cov_local goes with cov_diagonal (kf_fit_tracks_host_compact)")
        for t in (par, cov, q, hpos, hcov, out_par, out_cov, out_chi2, out_nhits, out_status):
            if t.is_cuda:
                raise ValueError("fit_tracks_host takes CPU tensors")
        g, keep = geom._c()
        ld = _plane_ld(par, 6)
        if _plane_ld(cov, 6 if cov_diagonal else 21) != ld:
            raise ValueError("par and cov must share the plane stride ld")
        seeds = _Tracks(int(n), ld, par.data_ptr(), cov.data_ptr(), q.data_ptr(), out_chi2.data_ptr(), out_nhits.data_ptr(),
                        out_status.data_ptr())
        out = self._tracks(n, out_par, out_cov, None, out_chi2, out_nhits, out_status)
        hits = self._track_hits(n, g.n_layers, hpos, hcov, mask, 3 if hit_cov_local else 6)
        name = ("kf_fit_tracks_host_compact" if hit_cov_local else
                "kf_fit_tracks_host_diag" if cov_diagonal else "kf_fit_tracks_host")
        self._check(getattr(self._lib, name)(self._h, C.byref(g), C.byref(seeds), C.byref(hits), C.byref(out)), name)
        del keep

    # ------------------------------------------------------------------ kf_bin_hits / kf_bin_layers
    @staticmethod
    def _layer_hits(n_hits, pos, cov) -> _LayerHits:
        lh = _LayerHits(int(n_hits), _plane_ld(pos, 3), pos.data_ptr(), cov.data_ptr())
        if _plane_ld(cov, 6) != lh.ld:
            raise ValueError("pos and cov must share the plane stride ld")
        return lh

    def bin_hits(self, radius_cm: float, n_hits: int, pos, cov, bins: Bins):
        lh = self._layer_hits(n_hits, pos, cov)
        lb = bins._c()
        self._check(self._lib.kf_bin_hits(self._h, float(radius_cm), C.byref(lh), C.byref(lb)), "kf_bin_hits")

    def bin_layers(self, radii_cm, layers):
        """layers: sequence of (n_hits, pos, cov, bins); one batched call for all of them."""
        n = len(layers)
        rad = (C.c_float * n)(*[float(r) for r in radii_cm])
        lhs = (_LayerHits * n)(*[self._layer_hits(nh, p, c) for (nh, p, c, _) in layers])
        lbs = (_LayerBins * n)(*[b._c() for (_, _, _, b) in layers])
        self._check(self._lib.kf_bin_layers(self._h, n, rad, lhs, lbs), "kf_bin_layers")

    # ------------------------------------------------------------------ kf_order_candidates
    def order_candidates(self, geom: Geometry, layer: int, n: int, par, cov, q, chi2, nhits, status,
                         n_eta: int, n_phi: int, eta_max: float, order):
        g, keep = geom._c()
        cands = self._tracks(n, par, cov, q, chi2, nhits, status)
        self._check(self._lib.kf_order_candidates(self._h, C.byref(g), int(layer), C.byref(cands), int(n_eta),
                                                  int(n_phi), float(eta_max), order.data_ptr()),
                    "kf_order_candidates")
        del keep

    # ------------------------------------------------------------------ kf_score_candidates
    def score_candidates(self, geom: Geometry, layer: int, n: int, par, cov, q, chi2, nhits, status,
                         n_hits: int, pos, cov_hits, bins: Bins, window_half: int, chi2_cut: float,
                         do_update: bool, best_hit, best_chi2, order=None, local_state=None, static_scratch=False):
        """local_state: optional float32 [30][ld] device tensor, zeroed before the first layer (see the header).
        static_scratch: call kf_score_candidates_static (no allocation; n <= STATIC_MAX_CANDIDATES)."""
        g, keep = geom._c()
        cands = self._tracks(n, par, cov, q, chi2, nhits, status)
        lh = _LayerHits(int(n_hits), _plane_ld(pos, 3), pos.data_ptr(), cov_hits.data_ptr())
        lb = bins._c()
        fn = self._lib.kf_score_candidates_static if static_scratch else self._lib.kf_score_candidates
        self._check(fn(self._h, C.byref(g), int(layer), C.byref(cands), C.byref(lh), C.byref(lb), int(window_half),
                       float(chi2_cut), 1 if do_update else 0, order.data_ptr() if order is not None else None,
                       best_hit.data_ptr(), best_chi2.data_ptr(),
                       local_state.data_ptr() if local_state is not None else None),
                    "kf_score_candidates_static" if static_scratch else "kf_score_candidates")
        del keep

    # ------------------------------------------------------------------ kf_build_best_hit
    def build_best_hit(self, geom: Geometry, first_layer: int, n: int, par, cov, q, chi2, nhits, status,
                       layers, window_half: int, chi2_cut: float, do_update: bool, hit_index, hit_chi2, order=None):
        """layers: sequence of (n_hits, pos, cov, bins) for first_layer, first_layer+1, ...;
        hit_index / hit_chi2: [len(layers)][ld_out] int32 / float32 device tensors."""
        g, keep = geom._c()
        cands = self._tracks(n, par, cov, q, chi2, nhits, status)
        m = len(layers)
        lhs = (_LayerHits * m)(*[self._layer_hits(nh, p, c) for (nh, p, c, _) in layers])
        lbs = (_LayerBins * m)(*[b._c() for (_, _, _, b) in layers])
        self._check(self._lib.kf_build_best_hit(self._h, C.byref(g), int(first_layer), m, C.byref(cands), lhs, lbs,
                                                int(window_half), float(chi2_cut), 1 if do_update else 0,
                                                order.data_ptr() if order is not None else None,
                                                hit_index.data_ptr(), hit_chi2.data_ptr(), int(hit_index.stride(0))),
                    "kf_build_best_hit")
        del keep

    def build_best_hit_events(self, geom: Geometry, first_layer: int, event_first, n: int, par, cov, q, chi2, nhits,
                              status, layers_by_event, window_half: int, chi2_cut: float, do_update: bool, hit_index,
                              hit_chi2):
        """layers_by_event: one sequence of (n_hits, pos, cov, bins) per event (all the same length);
        event_first: candidate offsets [n_events + 1]; the candidate tensors hold all events back to back."""
        g, keep = geom._c()
        cands = self._tracks(n, par, cov, q, chi2, nhits, status)
        ne, m = len(layers_by_event), len(layers_by_event[0])
        flat = [l for ev in layers_by_event for l in ev]
        lhs = (_LayerHits * (ne * m))(*[self._layer_hits(nh, p, c) for (nh, p, c, _) in flat])
        lbs = (_LayerBins * (ne * m))(*[b._c() for (_, _, _, b) in flat])
        first = (C.c_int64 * (ne + 1))(*[int(v) for v in event_first])
        self._check(self._lib.kf_build_best_hit_events(self._h, C.byref(g), int(first_layer), m, ne, first, C.byref(cands),
                                                       lhs, lbs, int(window_half), float(chi2_cut), 1 if do_update else 0,
                                                       hit_index.data_ptr(), hit_chi2.data_ptr(), int(hit_index.stride(0))),
                    "kf_build_best_hit_events")
        del keep

    def build_best_hit_host(self, geom: Geometry, first_layer: int, n: int, par, cov, q, chi2, nhits, status, layers,
                            n_eta: int, n_phi: int, eta_max: float, window_half: int, chi2_cut: float, do_update: bool,
                            hit_index, hit_chi2):
        """Everything in HOST (CPU) tensors: layers = sequence of (n_hits, pos [3][ld], cov [6][ld])."""
        for t in (par, cov, q, chi2, nhits, status, hit_index, hit_chi2):
            if t.is_cuda:
                raise ValueError("build_best_hit_host takes CPU tensors")
        g, keep = geom._c()
        cands = self._tracks(n, par, cov, q, chi2, nhits, status)
        m = len(layers)
        lhs = (_LayerHits * m)(*[self._layer_hits(nh, p, c) for (nh, p, c) in layers])
        self._check(self._lib.kf_build_best_hit_host(self._h, C.byref(g), int(first_layer), m, C.byref(cands), lhs,
                                                     int(n_eta), int(n_phi), float(eta_max), int(window_half),
                                                     float(chi2_cut), 1 if do_update else 0, hit_index.data_ptr(),
                                                     hit_chi2.data_ptr(), int(hit_index.stride(0))),
                    "kf_build_best_hit_host")
        del keep

    # ------------------------------------------------------------------ kf_build_combinatorial
    def build_combinatorial(self, geom: Geometry, first_layer: int, n: int, par, cov, q, chi2, nhits, status,
                            layers, window_half: int, chi2_cut: float, n_cand: int, hit_index, n_found=None):
        g, keep = geom._c()
        cands = self._tracks(n, par, cov, q, chi2, nhits, status)
        m = len(layers)
        lhs = (_LayerHits * m)(*[self._layer_hits(nh, p, c) for (nh, p, c, _) in layers])
        lbs = (_LayerBins * m)(*[b._c() for (_, _, _, b) in layers])
        self._check(self._lib.kf_build_combinatorial(self._h, C.byref(g), int(first_layer), m, C.byref(cands), lhs, lbs,
                                                     int(window_half), float(chi2_cut), int(n_cand),
                                                     hit_index.data_ptr(),
                                                     n_found.data_ptr() if n_found is not None else None,
                                                     int(hit_index.stride(0))), "kf_build_combinatorial")
        del keep

    def build_combinatorial_events(self, geom: Geometry, first_layer: int, event_first, n: int, par, cov, q, chi2,
                                   nhits, status, layers_by_event, window_half: int, chi2_cut: float, n_cand: int,
                                   hit_index, n_found=None):
        """Several events in one call; arguments as build_best_hit_events (event_first in seed indices)."""
        g, keep = geom._c()
        cands = self._tracks(n, par, cov, q, chi2, nhits, status)
        ne, m = len(layers_by_event), len(layers_by_event[0])
        flat = [l for ev in layers_by_event for l in ev]
        lhs = (_LayerHits * (ne * m))(*[self._layer_hits(nh, p, c) for (nh, p, c, _) in flat])
        lbs = (_LayerBins * (ne * m))(*[b._c() for (_, _, _, b) in flat])
        first = (C.c_int64 * (ne + 1))(*[int(v) for v in event_first])
        self._check(self._lib.kf_build_combinatorial_events(self._h, C.byref(g), int(first_layer), m, ne, first,
                                                            C.byref(cands), lhs, lbs, int(window_half), float(chi2_cut),
                                                            int(n_cand), hit_index.data_ptr(),
                                                            n_found.data_ptr() if n_found is not None else None,
                                                            int(hit_index.stride(0))), "kf_build_combinatorial_events")
        del keep
