"""ctypes loader for oracle/kf_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Layout conversion only (fp32 SoA inputs -> double AoS, packed 21 -> dense 6x6, packed 6 -> dense
3x3).  All arithmetic of the method lives in kf_oracle.c; see its header for the citations, the
readings it follows and the pins.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kf_oracle.c")
_LIB = os.path.join(_HERE, "libkf_oracle.so")

PROP_FAIL, S_NOT_PD, NONFINITE, BAD_CHARGE, OUTSIDE = 1, 2, 4, 8, 16
TRACE_STRIDE = 194

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no contraction: every float product is rounded once)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", _LIB, _SRC, "-lm", "-lpthread"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        _lib.orc_theta0.restype = C.c_double
        _lib.orc_theta0.argtypes = [C.c_double] * 3
        _lib.orc_propagate.restype = C.c_int
        _lib.orc_propagate.argtypes = [dp, C.c_double, C.c_double, C.c_double, dp, dp, dp, dp]
        _lib.orc_propagate_inward.restype = C.c_int
        _lib.orc_propagate_inward.argtypes = [dp, C.c_double, C.c_double, C.c_double, dp, dp, dp, dp]
        _lib.orc_fit_refit_tracks.restype = None
        _lib.orc_process_noise.restype = None
        _lib.orc_process_noise.argtypes = [dp, C.c_double, C.c_double, dp]
        _lib.orc_transport_cov.restype = None
        _lib.orc_transport_cov.argtypes = [dp, dp, dp, dp]
        _lib.orc_chi2_increment.restype = C.c_int
        _lib.orc_chi2_increment.argtypes = [dp, dp, dp, dp, dp]
        _lib.orc_update.restype = C.c_int
        _lib.orc_update.argtypes = [dp, dp, dp, dp, dp, dp, dp]
        _lib.orc_fit_tracks.restype = C.c_int
        _lib.orc_smooth_tracks.restype = C.c_int
        _lib.orc_bin_index_def.restype = C.c_int32
        _lib.orc_bin_index_def.argtypes = [C.c_double] * 4 + [C.c_int, C.c_int, C.c_double]
        _lib.orc_bin_index_f32.restype = C.c_int32
        _lib.orc_bin_index_f32.argtypes = [C.c_float] * 4 + [C.c_int, C.c_int, C.c_double]
        _lib.orc_bin_hits.restype = None
        _lib.orc_score_layer.restype = None
        _lib.orc_set_geometry_options.restype = None
        _lib.orc_set_geometry_options.argtypes = [C.c_int, C.c_int, dp]
        _lib.orc_set_score_half_length.restype = None
        _lib.orc_set_score_half_length.argtypes = [C.c_double]
        _lib.orc_set_score_surface.restype = None
        _lib.orc_set_score_surface.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double]
        _lib.orc_set_surfaces.restype = None
        _lib.orc_set_surfaces.argtypes = [C.c_int, C.POINTER(C.c_int32), dp, dp, dp]
        _lib.orc_propagate_to_z.restype = C.c_int
        _lib.orc_propagate_to_z.argtypes = [dp, C.c_double, C.c_double, C.c_double, dp, dp, dp, dp]
        _lib.orc_set_energy_loss.restype = None
        _lib.orc_set_energy_loss.argtypes = [C.c_int]
        _lib.orc_energy_loss.restype = C.c_double
        _lib.orc_energy_loss.argtypes = [C.c_double] * 3
        _lib.orc_energy_loss_step.restype = C.c_int
        _lib.orc_energy_loss_step.argtypes = [dp, dp, C.c_double, C.c_double, C.c_int, dp]
        _lib.orc_build_combinatorial.restype = None
    return _lib


class geometry_options:
    """Context manager for the oracle's process-wide geometry options (reading A20):
    material_model 0 = flat thickness (A5), 1 = thickness / cos(incidence); half_length[l] = half length of
    barrel layer l in cm (None = infinite, A12); energy_loss 1 = mean Bethe loss in silicon at every crossing
    (reading A21).  Restores the defaults on exit."""

    def __init__(self, material_model: int = 0, half_length=None, score_layer: int | None = None,
                 energy_loss: int = 0):
        self.model = int(material_model)
        self.eloss = int(energy_loss)
        self.hl = None if half_length is None else np.ascontiguousarray(half_length, dtype=np.float64)
        self.score_layer = score_layer

    def __enter__(self):
        n = 0 if self.hl is None else len(self.hl)
        lib().orc_set_geometry_options(self.model, n, _p(self.hl))
        lib().orc_set_energy_loss(self.eloss)
        if self.hl is not None and self.score_layer is not None:
            lib().orc_set_score_half_length(float(self.hl[self.score_layer]))
        return self

    def set_score_layer(self, layer: int):
        lib().orc_set_score_half_length(float(self.hl[layer]) if self.hl is not None else float("inf"))

    def __exit__(self, *a):
        lib().orc_set_geometry_options(0, 0, None)
        lib().orc_set_energy_loss(0)
        lib().orc_set_score_half_length(float("inf"))


class score_surface:
    """Context manager: the ONE layer score_layer works on is a disc pair z = +-zd with the annulus rmin <= rho <=
    rmax (readings A23 / A24; r_layer is then unused and the bins passed in must have been made with radius 0)."""

    def __init__(self, zd: float, rmin: float, rmax: float):
        self.a = (1, float(zd), float(rmin), float(rmax))

    def __enter__(self):
        lib().orc_set_score_surface(*self.a)
        return self

    def __exit__(self, *a):
        lib().orc_set_score_surface(0, 0.0, 0.0, float("inf"))


class surfaces:
    """Context manager for the oracle's process-wide surface list (reading A23): surface_type[l] 0 = barrel
    (radius[l]), 1 = pair of endcap discs at z = +-disc_z[l] sensitive for rmin[l] <= rho <= rmax[l].
    Restores "all barrels" on exit."""

    def __init__(self, surface_type, disc_z, rmin, rmax):
        self.t = np.ascontiguousarray(surface_type, dtype=np.int32)
        self.z = np.ascontiguousarray(disc_z, dtype=np.float64)
        self.lo = np.ascontiguousarray(rmin, dtype=np.float64)
        self.hi = np.ascontiguousarray(rmax, dtype=np.float64)

    def __enter__(self):
        lib().orc_set_surfaces(len(self.t), _p(self.t, C.c_int32), _p(self.z), _p(self.lo), _p(self.hi))
        return self

    def __exit__(self, *a):
        lib().orc_set_surfaces(0, None, None, None, None)


def propagate_to_z(u, q, Bz, zt, want_F=True):
    """Helix to the plane z = zt (reading A23). -> (status, u_out[6], F[6,6] or None, s, theta)"""
    u = np.ascontiguousarray(u, dtype=np.float64)
    out = np.zeros(6)
    F = np.zeros(36) if want_F else None
    s = C.c_double(0.0)
    th = C.c_double(0.0)
    rc = lib().orc_propagate_to_z(_p(u), float(q), float(Bz), float(zt), _p(out), _p(F), C.byref(s), C.byref(th))
    return rc, out, (F.reshape(6, 6) if want_F else None), s.value, th.value


def _p(a, ct=C.c_double):
    return a.ctypes.data_as(C.POINTER(ct)) if a is not None else None


# ------------------------------------------------------------------ layout helpers (no arithmetic)
_TRI = [(i, j) for i in range(6) for j in range(i, 6)]


def unpack_cov21(c21: np.ndarray) -> np.ndarray:
    """[21][n] packed upper triangle (row-major) -> [n][6][6] dense symmetric, float64."""
    n = c21.shape[1]
    out = np.empty((n, 6, 6))
    for k, (i, j) in enumerate(_TRI):
        out[:, i, j] = c21[k]
        out[:, j, i] = c21[k]
    return out


def pack_cov21(c: np.ndarray) -> np.ndarray:
    """[n][6][6] -> [21][n]."""
    return np.stack([c[:, i, j] for (i, j) in _TRI])


def unpack_cov6(v6: np.ndarray) -> np.ndarray:
    """[..., 6, n] packed xx,xy,xz,yy,yz,zz -> [n, ..., 3, 3] dense, float64."""
    v = np.moveaxis(np.asarray(v6, dtype=np.float64), -1, 0)          # [n, ..., 6]
    idx = np.array([[0, 1, 2], [1, 3, 4], [2, 4, 5]])
    return v[..., idx]


# ------------------------------------------------------------------ scalar-level entry points
def theta0(p, mass, t):
    return lib().orc_theta0(float(p), float(mass), float(t))


def energy_loss(p, mass, t):
    """Mean Bethe energy loss [GeV] in t radiation lengths of silicon (reading A21)."""
    return lib().orc_energy_loss(float(p), float(mass), float(t))


def energy_loss_step(u, Cm, mass, t, direction):
    """Reading A21 at one layer: -> (status, u_out[6], C_out[6,6], J[6,6]); direction +1 loses, -1 regains."""
    u = np.array(u, dtype=np.float64)
    Cm = np.array(Cm, dtype=np.float64).reshape(36)
    J = np.zeros(36)
    rc = lib().orc_energy_loss_step(_p(u), _p(Cm), float(mass), float(t), int(direction), _p(J))
    return rc, u, Cm.reshape(6, 6), J.reshape(6, 6)


def propagate(u, q, Bz, r, want_F=True):
    """-> (status, u_out[6], F[6,6] or None, s, theta)"""
    u = np.ascontiguousarray(u, dtype=np.float64)
    out = np.zeros(6)
    F = np.zeros(36) if want_F else None
    s = C.c_double(0.0)
    th = C.c_double(0.0)
    rc = lib().orc_propagate(_p(u), float(q), float(Bz), float(r), _p(out), _p(F), C.byref(s), C.byref(th))
    return rc, out, (F.reshape(6, 6) if want_F else None), s.value, th.value


def propagate_inward(u, q, Bz, r, want_F=True):
    """Backward along the helix to a smaller radius (reading A18). -> (status, u_out, F, s, theta)"""
    u = np.ascontiguousarray(u, dtype=np.float64)
    out = np.zeros(6)
    F = np.zeros(36) if want_F else None
    s = C.c_double(0.0)
    th = C.c_double(0.0)
    rc = lib().orc_propagate_inward(_p(u), float(q), float(Bz), float(r), _p(out), _p(F), C.byref(s), C.byref(th))
    return rc, out, (F.reshape(6, 6) if want_F else None), s.value, th.value


def process_noise(u, mass, t):
    u = np.ascontiguousarray(u, dtype=np.float64)
    Q = np.zeros(36)
    lib().orc_process_noise(_p(u), float(mass), float(t), _p(Q))
    return Q.reshape(6, 6)


def transport_cov(F, Cm, Q):
    F = np.ascontiguousarray(F, dtype=np.float64)
    Cm = np.ascontiguousarray(Cm, dtype=np.float64)
    Q = np.ascontiguousarray(Q, dtype=np.float64)
    out = np.zeros(36)
    lib().orc_transport_cov(_p(F), _p(Cm), _p(Q), _p(out))
    return out.reshape(6, 6)


def chi2_increment(u, Cm, m, V):
    u, Cm, m, V = (np.ascontiguousarray(a, dtype=np.float64) for a in (u, Cm, m, V))
    c = C.c_double(0.0)
    rc = lib().orc_chi2_increment(_p(u), _p(Cm), _p(m), _p(V), C.byref(c))
    return rc, c.value


def update(u, Cm, m, V):
    u, Cm, m, V = (np.ascontiguousarray(a, dtype=np.float64) for a in (u, Cm, m, V))
    uo, Co = np.zeros(6), np.zeros(36)
    c = C.c_double(0.0)
    rc = lib().orc_update(_p(u), _p(Cm), _p(m), _p(V), _p(uo), _p(Co), C.byref(c))
    return rc, uo, Co.reshape(6, 6), c.value


# ------------------------------------------------------------------ batched fit
def fit_tracks(radius, x_over_X0, Bz, mass, par, cov21, q, hpos, hcov, mask=None,
               nthreads: int = 1, want_trace: bool = False, timing: dict | None = None) -> dict:
    """Fit n tracks.  Inputs in the SoA fp32 layout of the C ABI (par[6][n], cov21[21][n],
    hpos[L][3][n], hcov[L][6][n]); widened to double, transposed to AoS and handed to
    orc_fit_tracks.  Returns dict(par[6][n], cov[n][6][6], chi2, nhits, status[, trace])."""
    L = int(len(radius))
    n = int(par.shape[1])
    rad = np.ascontiguousarray(radius, dtype=np.float64)
    xx0 = np.ascontiguousarray(x_over_X0, dtype=np.float64)
    par_a = np.ascontiguousarray(np.asarray(par, dtype=np.float64).T)               # [n][6]
    cov_a = np.ascontiguousarray(unpack_cov21(np.asarray(cov21, dtype=np.float64)))  # [n][6][6]
    q_a = np.ascontiguousarray(q, dtype=np.int8)
    hp_a = np.ascontiguousarray(np.transpose(np.asarray(hpos, dtype=np.float64), (2, 0, 1)))  # [n][L][3]
    hc_a = np.ascontiguousarray(np.swapaxes(unpack_cov6(hcov), 0, 0))               # [n][L][3][3]
    m_a = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint32)
    opar = np.zeros((n, 6)); ocov = np.zeros((n, 6, 6)); ochi2 = np.zeros(n)
    onh = np.zeros(n, dtype=np.int32); ost = np.zeros(n, dtype=np.uint32)
    trace = np.zeros((n, L, TRACE_STRIDE)) if want_trace else None
    import time as _time
    _t0 = _time.perf_counter()
    rc = lib().orc_fit_tracks(C.c_int64(n), C.c_int(L), _p(rad), _p(xx0), C.c_double(Bz), C.c_double(mass),
                              _p(par_a), _p(cov_a), _p(q_a, C.c_int8), _p(hp_a), _p(hc_a),
                              _p(m_a, C.c_uint32), _p(opar), _p(ocov), _p(ochi2), _p(onh, C.c_int32),
                              _p(ost, C.c_uint32), _p(trace), C.c_int(nthreads))
    if timing is not None:          # instrumentation only: seconds spent inside the C call
        timing["seconds"] = _time.perf_counter() - _t0
    if rc != 0:
        raise RuntimeError("orc_fit_tracks failed")
    out = dict(par=np.ascontiguousarray(opar.T), cov=ocov, chi2=ochi2, nhits=onh, status=ost)
    if want_trace:
        out["trace"] = trace
    return out


def smooth_tracks(radius, x_over_X0, Bz, mass, par, cov21, q, hpos, hcov, mask=None, nthreads: int = 1) -> dict:
    """Forward fit + RTS smoother (reading A22).  Same input layout as fit_tracks.  Returns the forward results
    under the usual keys plus spar[L][6][n], scov[n][L][6][6] (smoothed state / covariance at every used layer,
    zeros elsewhere), used[n] (bit mask of those layers) and sstatus[n]."""
    L = int(len(radius))
    n = int(par.shape[1])
    rad = np.ascontiguousarray(radius, dtype=np.float64)
    xx0 = np.ascontiguousarray(x_over_X0, dtype=np.float64)
    par_a = np.ascontiguousarray(np.asarray(par, dtype=np.float64).T)
    cov_a = np.ascontiguousarray(unpack_cov21(np.asarray(cov21, dtype=np.float64)))
    q_a = np.ascontiguousarray(q, dtype=np.int8)
    hp_a = np.ascontiguousarray(np.transpose(np.asarray(hpos, dtype=np.float64), (2, 0, 1)))
    hc_a = np.ascontiguousarray(unpack_cov6(hcov))
    m_a = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint32)
    opar = np.zeros((n, 6)); ocov = np.zeros((n, 6, 6)); ochi2 = np.zeros(n)
    onh = np.zeros(n, dtype=np.int32); ost = np.zeros(n, dtype=np.uint32)
    spar = np.zeros((n, L, 6)); scov = np.zeros((n, L, 6, 6))
    used = np.zeros(n, dtype=np.uint32); sst = np.zeros(n, dtype=np.uint32)
    rc = lib().orc_smooth_tracks(C.c_int64(n), C.c_int(L), _p(rad), _p(xx0), C.c_double(Bz), C.c_double(mass),
                                 _p(par_a), _p(cov_a), _p(q_a, C.c_int8), _p(hp_a), _p(hc_a), _p(m_a, C.c_uint32),
                                 _p(opar), _p(ocov), _p(ochi2), _p(onh, C.c_int32), _p(ost, C.c_uint32), _p(spar),
                                 _p(scov), _p(used, C.c_uint32), _p(sst, C.c_uint32), C.c_int(nthreads))
    if rc != 0:
        raise RuntimeError("orc_smooth_tracks failed")
    return dict(par=np.ascontiguousarray(opar.T), cov=ocov, chi2=ochi2, nhits=onh, status=ost,
                spar=np.ascontiguousarray(np.transpose(spar, (1, 2, 0))), scov=scov, used=used, sstatus=sst)


REFIT_KAPPA = 10.0    # reading A18: inflation of the forward covariance used as the backward prior


def fit_refit_tracks(radius, x_over_X0, Bz, mass, par, cov21, q, hpos, hcov, mask=None, kappa: float = REFIT_KAPPA,
                      want_trace: bool = False) -> dict:
    """Forward fit + inward refit (smoother).  Same input layout as fit_tracks.  Returns the forward
    results under the usual keys and the smoothed ones as spar[6][n], scov[n][6][6], schi2, sstatus
    [, trace_fwd, trace_bwd]."""
    L = int(len(radius))
    n = int(par.shape[1])
    rad = np.ascontiguousarray(radius, dtype=np.float64)
    xx0 = np.ascontiguousarray(x_over_X0, dtype=np.float64)
    par_a = np.ascontiguousarray(np.asarray(par, dtype=np.float64).T)
    cov_a = np.ascontiguousarray(unpack_cov21(np.asarray(cov21, dtype=np.float64)))
    q_a = np.ascontiguousarray(q, dtype=np.int8)
    hp_a = np.ascontiguousarray(np.transpose(np.asarray(hpos, dtype=np.float64), (2, 0, 1)))
    hc_a = np.ascontiguousarray(unpack_cov6(hcov))
    m_a = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint32)
    opar = np.zeros((n, 6)); ocov = np.zeros((n, 6, 6)); ochi2 = np.zeros(n)
    onh = np.zeros(n, dtype=np.int32); ost = np.zeros(n, dtype=np.uint32)
    spar = np.zeros((n, 6)); scov = np.zeros((n, 6, 6)); schi2 = np.zeros(n); sst = np.zeros(n, dtype=np.uint32)
    snh = np.zeros(n, dtype=np.int32)
    tf = np.zeros((n, L, TRACE_STRIDE)) if want_trace else None
    tb = np.zeros((n, L, TRACE_STRIDE)) if want_trace else None
    lib().orc_fit_refit_tracks(C.c_int64(n), C.c_int(L), _p(rad), _p(xx0), C.c_double(Bz), C.c_double(mass),
                                C.c_double(kappa), _p(par_a), _p(cov_a), _p(q_a, C.c_int8), _p(hp_a), _p(hc_a),
                                _p(m_a, C.c_uint32), _p(opar), _p(ocov), _p(ochi2), _p(onh, C.c_int32),
                                _p(ost, C.c_uint32), _p(spar), _p(scov), _p(schi2), _p(sst, C.c_uint32), _p(snh, C.c_int32),
                                _p(tf), _p(tb))
    out = dict(par=np.ascontiguousarray(opar.T), cov=ocov, chi2=ochi2, nhits=onh, status=ost,
               rpar=np.ascontiguousarray(spar.T), rcov=scov, rchi2=schi2, rstatus=sst, rnhits=snh)
    if want_trace:
        out["trace_fwd"], out["trace_bwd"] = tf, tb
    return out


def fit_batch(batch, nthreads: int = 1, want_trace: bool = False) -> dict:
    """Convenience: fit a workloads.barrel_events.FitBatch-shaped object (duck-typed).  A batch that carries a
    surface list (reading A23) is fitted with it, its barrel half lengths and its material model."""
    st = getattr(batch, "surface_type", None)
    if st is None:
        return fit_tracks(batch.radius, batch.x_over_X0, batch.Bz, batch.mass, batch.par, batch.cov,
                          batch.q, batch.hpos, batch.hcov, batch.mask, nthreads, want_trace)
    with surfaces(st, batch.disc_z, batch.disc_rmin, batch.disc_rmax), \
            geometry_options(int(getattr(batch, "material_model", 0)), getattr(batch, "half_length", None),
                             energy_loss=int(getattr(batch, "energy_loss", 0))):
        return fit_tracks(batch.radius, batch.x_over_X0, batch.Bz, batch.mass, batch.par, batch.cov,
                          batch.q, batch.hpos, batch.hcov, batch.mask, nthreads, want_trace)


# ------------------------------------------------------------------ binning and scoring
def bin_index_def(x, y, z, r_layer, n_eta, n_phi, eta_max):
    return lib().orc_bin_index_def(float(x), float(y), float(z), float(r_layer), n_eta, n_phi, float(eta_max))


def bin_index_f32(x, y, z, r_layer, n_eta, n_phi, eta_max):
    return lib().orc_bin_index_f32(float(x), float(y), float(z), float(r_layer), n_eta, n_phi, float(eta_max))


def bin_hits(pos, r_layer, n_eta, n_phi, eta_max) -> dict:
    """pos[3][H] fp32 -> dict(bin_offset[n_bins+1], sorted_to_orig[H], bin_of[H])."""
    pos = np.ascontiguousarray(pos, dtype=np.float32)
    H = int(pos.shape[1])
    off = np.zeros(n_eta * n_phi + 1, dtype=np.int32)
    s2o = np.zeros(max(H, 1), dtype=np.int32)
    bof = np.zeros(max(H, 1), dtype=np.int32)
    x, y, z = (np.ascontiguousarray(pos[i]) for i in range(3))
    lib().orc_bin_hits(C.c_int64(H), _p(x, C.c_float), _p(y, C.c_float), _p(z, C.c_float),
                       C.c_float(r_layer), C.c_int(n_eta), C.c_int(n_phi), C.c_double(eta_max),
                       _p(off, C.c_int32), _p(s2o, C.c_int32), _p(bof, C.c_int32))
    return dict(bin_offset=off, sorted_to_orig=s2o[:H], bin_of=bof[:H])


class Candidates:
    """Double AoS candidate set the scoring oracle advances layer by layer."""

    def __init__(self, par, cov21, q, chi2=None, nhits=None):
        n = int(par.shape[1])
        self.n = n
        self.par = np.ascontiguousarray(np.asarray(par, dtype=np.float64).T)
        self.cov = np.ascontiguousarray(unpack_cov21(np.asarray(cov21, dtype=np.float64)))
        self.q = np.ascontiguousarray(q, dtype=np.int8)
        self.chi2 = np.zeros(n) if chi2 is None else np.ascontiguousarray(chi2, dtype=np.float64).copy()
        self.nhits = np.zeros(n, dtype=np.int32) if nhits is None else np.ascontiguousarray(nhits, dtype=np.int32).copy()
        self.status = np.zeros(n, dtype=np.uint32)


def score_layer(cands: Candidates, r_layer, x_over_X0, Bz, mass, hpos, hcov, bins: dict | None,
                n_eta, n_phi, eta_max, window_half=2, chi2_cut=30.0, do_update=True,
                all_hits=False) -> dict:
    """Advance `cands` by one layer (in place).  hpos[3][H], hcov[6][H] fp32 in ORIGINAL order.
    Returns dict(best_hit[n] (original index or -1), best_chi2[n], second_chi2[n])."""
    hp = np.ascontiguousarray(np.asarray(hpos, dtype=np.float64).T)      # [H][3]
    hc = np.ascontiguousarray(unpack_cov6(hcov))                          # [H][3][3]
    H = int(hp.shape[0])
    n = cands.n
    bh = np.zeros(n, dtype=np.int32); bc = np.zeros(n); sc = np.zeros(n)
    off = s2o = None
    if not all_hits:
        off = np.ascontiguousarray(bins["bin_offset"], dtype=np.int32)
        s2o = np.ascontiguousarray(bins["sorted_to_orig"], dtype=np.int32)
    lib().orc_score_layer(C.c_int64(n), C.c_double(r_layer), C.c_double(x_over_X0), C.c_double(Bz),
                          C.c_double(mass), _p(cands.par), _p(cands.cov), _p(cands.q, C.c_int8),
                          _p(cands.chi2), _p(cands.nhits, C.c_int32), _p(cands.status, C.c_uint32),
                          C.c_int64(H), _p(hp), _p(hc), C.c_int(n_eta), C.c_int(n_phi), C.c_double(eta_max),
                          _p(off, C.c_int32), _p(s2o, C.c_int32), C.c_int(window_half),
                          C.c_double(chi2_cut), C.c_int(1 if do_update else 0), C.c_int(1 if all_hits else 0),
                          _p(bh, C.c_int32), _p(bc), _p(sc))
    return dict(best_hit=bh, best_chi2=bc, second_chi2=sc)


def build_combinatorial(radius, x_over_X0, Bz, mass, par, cov21, q, chi2, nhits, first_layer: int, layers: list,
                        n_eta: int, n_phi: int, eta_max: float, window_half: int = 2, chi2_cut: float = 30.0,
                        n_cand: int = 4) -> dict:
    """Combinatorial building (reading A19) of all seeds over `layers` = [(hpos[3][H], hcov[6][H], bins dict), ...]
    belonging to geometry layers first_layer, first_layer + 1, ...  Seeds in the SoA fp32 layout.
    Returns the best candidate per seed: par[6][n], cov[n][6][6], chi2, nhits, status, hits[n_build][n],
    n_cand[n], margin[n] (smallest relative gap of any decision fp32 rounding could flip)."""
    n = int(par.shape[1])
    m = len(layers)
    rad = np.ascontiguousarray(radius, dtype=np.float64)
    xx0 = np.ascontiguousarray(x_over_X0, dtype=np.float64)
    par_a = np.ascontiguousarray(np.asarray(par, dtype=np.float64).T)
    cov_a = np.ascontiguousarray(unpack_cov21(np.asarray(cov21, dtype=np.float64)))
    q_a = np.ascontiguousarray(q, dtype=np.int8)
    c_a = np.ascontiguousarray(chi2, dtype=np.float64)
    nh_a = np.ascontiguousarray(nhits, dtype=np.int32)
    hp = [np.ascontiguousarray(np.asarray(l[0], dtype=np.float64).T) for l in layers]
    hc = [np.ascontiguousarray(unpack_cov6(l[1])) for l in layers]
    off = [np.ascontiguousarray(l[2]["bin_offset"], dtype=np.int32) for l in layers]
    s2o = [np.ascontiguousarray(l[2]["sorted_to_orig"], dtype=np.int32) for l in layers]
    nh = (C.c_int64 * m)(*[int(h.shape[0]) for h in hp])
    dpp = C.POINTER(C.c_double)
    ipp = C.POINTER(C.c_int32)
    hp_p = (dpp * m)(*[_p(a) for a in hp])
    hc_p = (dpp * m)(*[_p(a) for a in hc])
    off_p = (ipp * m)(*[_p(a, C.c_int32) for a in off])
    s2o_p = (ipp * m)(*[_p(a, C.c_int32) for a in s2o])
    opar = np.zeros((n, 6)); ocov = np.zeros((n, 6, 6)); ochi2 = np.zeros(n)
    onh = np.zeros(n, dtype=np.int32); ost = np.zeros(n, dtype=np.uint32)
    ohits = np.zeros((m, n), dtype=np.int32); onc = np.zeros(n, dtype=np.int32); omar = np.zeros(n)
    lib().orc_build_combinatorial(C.c_int64(n), C.c_int(len(rad)), C.c_int(first_layer), C.c_int(m), _p(rad), _p(xx0),
                                  C.c_double(Bz), C.c_double(mass), _p(par_a), _p(cov_a), _p(q_a, C.c_int8), _p(c_a),
                                  _p(nh_a, C.c_int32), nh, hp_p, hc_p, C.c_int(n_eta), C.c_int(n_phi),
                                  C.c_double(eta_max), off_p, s2o_p, C.c_int(window_half), C.c_double(chi2_cut),
                                  C.c_int(n_cand), _p(opar), _p(ocov), _p(ochi2), _p(onh, C.c_int32),
                                  _p(ost, C.c_uint32), _p(ohits, C.c_int32), _p(onc, C.c_int32), _p(omar))
    return dict(par=np.ascontiguousarray(opar.T), cov=ocov, chi2=ochi2, nhits=onh, status=ost, hits=ohits,
                n_cand=onc, margin=omar)
