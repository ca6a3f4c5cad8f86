"""Seeded synthetic barrel-detector events (input generator only).

This module stands in for the paper's in-house toy simulation (section 3.2:
"equally spaced, fixed length concentric cylinders ... Gaussian smearing of the hit positions",
seeds "derived from the first three hits"), which is not available.  The five workloads are the
ones BASELINE.json:configs[0..4] describe; the recipe (distributions, sigmas, seed prior) is
written out in DESIGN.md "Input recipe".

It is shared by the tests, bench.py and __graft_entry__.smoke().  It contains NO Kalman-filter
arithmetic (no Jacobian, no gain, no chi2, no binning) and imports neither `oracle/` nor the CUDA
package: it only *simulates* truth particles (circle/cylinder intersection written as a two-circle
intersection with atan2 turning angles -- deliberately a different formulation from the
half-angle crossing the fit uses), smears hits, scatters the truth and smears a seed.

All arithmetic is float64; everything handed to the fitters is rounded ONCE to float32
(reading A17) so the oracle and the CUDA path see bit-identical inputs.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

C_B = 2.99792458e-3          # GeV / (c * Tesla * cm): p_T[GeV] = C_B * B[T] * R[cm]
M_PION = 0.13957             # GeV, mass used for beta in the scattering angle
BASE_SEED = 170502876

SIGMA_RPHI = 0.01            # cm  (BASELINE.json:configs[0])
SIGMA_Z = 0.1                # cm  (BASELINE.json:configs[0])
SIGMA_R = 0.1                # cm  (reading A6: radial error assigned to a hit)
SEED_POS_SMEAR = 0.03        # cm  (A13)
SEED_MOM_SMEAR = 0.10        # fraction of true pT (A13, "smeared 10%")
SEED_POS_SIGMA0 = 0.3        # cm, prior sigma on position (A13)
SEED_MOM_SIGMA0 = 0.3        # fraction of seed pT, prior sigma on each momentum component (A13)


@dataclass
class BarrelConfig:
    """One of BASELINE.json:configs[i] as numbers."""
    index: int
    n_events: int
    n_tracks: int                 # per event
    n_layers: int
    pt_min: float
    pt_max: float
    eta_max: float
    x_over_X0: float
    Bz: float = 3.8
    layer_step_cm: float = 4.0
    noise_hits_per_layer: int = 0  # config 4 only
    n_eta: int = 40                # config 4 only
    n_phi: int = 64
    eta_bin_max: float = 1.2
    first_scored_layer: int = 3
    material_model: int = 0        # DESIGN.md reading A20: 1 = thickness / cos(incidence)
    half_length_cm: float = float("inf")   # A20: finite barrel (same half length for every layer)
    energy_loss: int = 0           # DESIGN.md reading A21: 1 = mean energy loss in silicon after every hit

    @property
    def radii(self) -> np.ndarray:
        return self.layer_step_cm * np.arange(1, self.n_layers + 1, dtype=np.float64)


def get_config(i: int) -> BarrelConfig:
    if i == 0:
        return BarrelConfig(0, 1, 1_000, 10, 0.5, 10.0, 1.0, 0.0)
    if i == 1:
        return BarrelConfig(1, 1, 20_000, 10, 0.5, 10.0, 1.0, 0.01)
    if i == 2:
        return BarrelConfig(2, 100, 20_000, 10, 0.5, 10.0, 1.0, 0.01)
    if i == 3:
        return BarrelConfig(3, 1, 100_000, 20, 0.3, 20.0, 1.5, 0.01)
    if i == 4:
        return BarrelConfig(4, 1, 20_000, 10, 0.5, 10.0, 1.0, 0.01, noise_hits_per_layer=100_000)
    raise ValueError(f"no such config {i}")


@dataclass
class FitBatch:
    """Inputs of one kf_fit_tracks call, SoA element-major, fp32 (what both fitters read)."""
    n: int
    radius: np.ndarray        # [L]  f32
    x_over_X0: np.ndarray     # [L]  f32
    Bz: float
    mass: float
    par: np.ndarray           # [6][n]  f32  seed x,y,z,px,py,pz
    cov: np.ndarray           # [21][n] f32  seed covariance, upper triangle row-major
    q: np.ndarray             # [n]     i8
    hpos: np.ndarray          # [L][3][n] f32
    hcov: np.ndarray          # [L][6][n] f32  xx,xy,xz,yy,yz,zz
    mask: np.ndarray          # [n] u32, bit l = track has a hit on layer l
    truth: np.ndarray = field(repr=False, default=None)   # [L][6][n] f64 post-scatter truth at each layer
    truth_vertex: np.ndarray = field(repr=False, default=None)  # [6][n] f64
    material_model: int = 0                # DESIGN.md reading A20 (geometry options of the fit)
    half_length: np.ndarray = None         # [L] f32 barrel half lengths, None = unbounded
    energy_loss: int = 0                   # DESIGN.md reading A21
    # DESIGN.md reading A23 (endcap discs); None = every layer is a barrel
    surface_type: np.ndarray = None        # [L] i32: 0 barrel (radius, half_length), 1 disc pair
    disc_z: np.ndarray = None              # [L] f32: |z| of the disc pair
    disc_rmin: np.ndarray = None           # [L] f32
    disc_rmax: np.ndarray = None           # [L] f32

    @property
    def n_layers(self) -> int:
        return int(self.radius.shape[0])


def highland_theta0(p: np.ndarray, mass: float, t) -> np.ndarray:
    """Width of the simulated scattering angle (PDG Highland form, thickness t = x/X0, scalar or per track)."""
    t = np.asarray(t, dtype=np.float64)
    if np.all(t <= 0.0):
        return np.zeros_like(p)
    beta = p / np.sqrt(p * p + mass * mass)
    return 0.0136 / (beta * p) * np.sqrt(t) * (1.0 + 0.038 * np.log(t))


def silicon_mean_energy_loss(p: np.ndarray, mass: float, t) -> np.ndarray:
    """Mean energy [GeV] a unit-charge particle of momentum p loses in t radiation lengths of silicon
    (simulation side of reading A21): PDG mean stopping power without density correction,
    S = K (Z/A) / beta^2 * [ln(2 me (beta gamma)^2 / I) - ln(1 + 2 gamma me/M + (me/M)^2) / 2 - beta^2]."""
    K, me, I = 0.307075e-3, 0.51099895e-3, 173.0e-9          # GeV cm^2/mol, GeV, GeV
    bg2 = (p / mass) ** 2
    gam = np.sqrt(1.0 + bg2)
    b2 = bg2 / (1.0 + bg2)
    bracket = np.log(2.0 * me * bg2 / I) - 0.5 * np.log1p(2.0 * gam * me / mass + (me / mass) ** 2) - b2
    return K * (14.0 / 28.0855) / b2 * bracket * (np.asarray(t, dtype=np.float64) * 21.82)


def _cross_cylinder(pos, mom, q, Bz, r):
    """First forward crossing of each truth helix with the cylinder of radius r.

    Two-circle intersection (track circle: centre c, radius R; layer circle: origin, radius r),
    turning angle from atan2 differences about the centre.  Returns new (pos, mom).
    """
    x, y, z = pos
    px, py, pz = mom
    k = q * C_B * Bz
    pt = np.hypot(px, py)
    R = pt / np.abs(k)
    cx = x + py / k
    cy = y - px / k
    d = np.hypot(cx, cy)
    a = (d * d + r * r - R * R) / (2.0 * d)
    h = np.sqrt(np.maximum(r * r - a * a, 0.0))
    ux, uy = cx / d, cy / d
    psi0 = np.arctan2(y - cy, x - cx)
    best_theta = None
    best_pt = None
    for sgn in (+1.0, -1.0):
        X = a * ux - sgn * h * uy
        Y = a * uy + sgn * h * ux
        psi = np.arctan2(Y - cy, X - cx)
        # the position angle about the centre evolves as psi(theta) = psi0 - theta, theta = kappa*s
        turn = np.where(k > 0, np.mod(psi0 - psi, 2 * np.pi), -np.mod(psi - psi0, 2 * np.pi))
        if best_theta is None:
            best_theta, best_pt = turn, (X, Y)
        else:
            take = np.abs(turn) < np.abs(best_theta)
            best_theta = np.where(take, turn, best_theta)
            best_pt = (np.where(take, X, best_pt[0]), np.where(take, Y, best_pt[1]))
    theta = best_theta
    s = theta * pt / k
    c, sn = np.cos(theta), np.sin(theta)
    return (best_pt[0], best_pt[1], z + pz * s / pt), (px * c + py * sn, -px * sn + py * c, pz)


def hit_covariance(phi_h, sigma_r=SIGMA_R, sigma_rphi=SIGMA_RPHI, sigma_z=SIGMA_Z):
    """V = Rz(phi_h) diag(sr^2, srphi^2, sz^2) Rz(phi_h)^T packed xx,xy,xz,yy,yz,zz."""
    c, s = np.cos(phi_h), np.sin(phi_h)
    vr, vt, vz = sigma_r ** 2, sigma_rphi ** 2, sigma_z ** 2
    zero = np.zeros_like(c)
    return np.stack([vr * c * c + vt * s * s, (vr - vt) * c * s, zero,
                     vr * s * s + vt * c * c, zero, zero + vz])


def simulate_event(cfg: BarrelConfig, event: int, n_tracks: int | None = None,
                   smear_hits: bool = True, smear_seed: bool = True, dtype=np.float32) -> FitBatch:
    """One event of `cfg` (rng = default_rng(BASE_SEED + 1000*config + event)).

    dtype=float64 keeps the un-rounded values (oracle pins only; the fitters' contract is fp32)."""
    rng = np.random.default_rng(BASE_SEED + 1000 * cfg.index + event)
    n = cfg.n_tracks if n_tracks is None else n_tracks
    L = cfg.n_layers
    radii = cfg.radii
    q = rng.choice(np.array([-1.0, 1.0]), size=n)
    pt = rng.uniform(cfg.pt_min, cfg.pt_max, size=n)
    phi = rng.uniform(0.0, 2 * np.pi, size=n)
    eta = rng.uniform(-cfg.eta_max, cfg.eta_max, size=n)
    mom = (pt * np.cos(phi), pt * np.sin(phi), pt * np.sinh(eta))
    pos = (np.zeros(n), np.zeros(n), np.zeros(n))
    truth_vertex = np.stack(pos + mom)

    hpos = np.zeros((L, 3, n))
    hcov = np.zeros((L, 6, n))
    truth = np.full((L, 6, n), np.nan)
    mask = np.zeros(n, dtype=np.uint32)
    alive = np.ones(n, dtype=bool)
    for l in range(L):
        r = float(radii[l])
        k = q * C_B * cfg.Bz
        ptl = np.hypot(mom[0], mom[1])
        R = ptl / np.abs(k)
        centre = np.hypot(pos[0] + mom[1] / k, pos[1] - mom[0] / k)
        alive &= ~(r > 0.9 * (R + centre))          # A12: stop before a too-shallow crossing
        with np.errstate(invalid="ignore", divide="ignore"):
            npos, nmom = _cross_cylinder(pos, mom, q, cfg.Bz, r)
        pos = tuple(np.where(alive, a, b) for a, b in zip(npos, pos))
        mom = tuple(np.where(alive, a, b) for a, b in zip(nmom, mom))
        # measurement: smear azimuth by sigma_rphi / r, z by sigma_z; the hit stays on the cylinder
        g = rng.standard_normal((2, n))
        if not smear_hits:
            g = np.zeros_like(g)
        phi_h = np.arctan2(pos[1], pos[0]) + g[0] * SIGMA_RPHI / r
        hp = np.stack([r * np.cos(phi_h), r * np.sin(phi_h), pos[2] + g[1] * SIGMA_Z])
        hv = hit_covariance(phi_h)
        inside = alive & (np.abs(pos[2]) <= cfg.half_length_cm)      # A20: a crossing beyond the barrel end leaves no hit
        hpos[l] = np.where(inside, hp, 0.0)
        hcov[l] = np.where(inside, hv, 0.0)
        mask |= (inside.astype(np.uint32) << np.uint32(l))
        # multiple scattering right after the hit: two independent angles about p-hat, |p| kept
        a = rng.standard_normal((2, n))
        if cfg.x_over_X0 > 0.0:
            px, py, pz = mom
            p = np.sqrt(px * px + py * py + pz * pz)
            t_eff = cfg.x_over_X0
            if cfg.material_model == 1:                              # path length through the layer
                t_eff = cfg.x_over_X0 * (np.hypot(pos[0], pos[1]) * p) / np.abs(pos[0] * px + pos[1] * py)
            th0 = highland_theta0(p, M_PION, t_eff)
            th0 = np.where(inside, th0, 0.0)                         # no material beyond the barrel end
            ptt = np.hypot(px, py)
            e1 = (-py / ptt, px / ptt, np.zeros(n))                      # z-hat x p-hat, normalised
            ph = (px / p, py / p, pz / p)
            e2 = (ph[1] * e1[2] - ph[2] * e1[1], ph[2] * e1[0] - ph[0] * e1[2], ph[0] * e1[1] - ph[1] * e1[0])
            t1, t2 = np.tan(a[0] * th0), np.tan(a[1] * th0)
            d = tuple(ph[i] + t1 * e1[i] + t2 * e2[i] for i in range(3))
            dn = np.sqrt(d[0] ** 2 + d[1] ** 2 + d[2] ** 2)
            mom = tuple(np.where(alive, p * d[i] / dn, mom[i]) for i in range(3))
            if cfg.energy_loss == 1:                                  # A21: mean loss, direction kept
                E = np.sqrt(p * p + M_PION * M_PION)
                E2 = E - np.where(inside, silicon_mean_energy_loss(p, M_PION, t_eff), 0.0)
                stopped = E2 <= M_PION
                alive &= ~stopped
                scale = np.sqrt(np.maximum(E2 * E2 - M_PION * M_PION, 0.0)) / p
                mom = tuple(np.where(alive, mom[i] * scale, mom[i]) for i in range(3))
        truth[l] = np.where(alive, np.stack(pos + mom), np.nan)

    # seed (A13)
    g = rng.standard_normal((6, n))
    if not smear_seed:
        g = np.zeros_like(g)
    spar = truth_vertex.copy()
    spar[0:3] += SEED_POS_SMEAR * g[0:3]
    spar[3:6] += SEED_MOM_SMEAR * pt * g[3:6]
    spt = np.hypot(spar[3], spar[4])
    scov = np.zeros((21, n))
    diag_idx = [0, 6, 11, 15, 18, 20]
    for i in range(3):
        scov[diag_idx[i]] = SEED_POS_SIGMA0 ** 2
        scov[diag_idx[3 + i]] = (SEED_MOM_SIGMA0 * spt) ** 2

    f32 = dtype
    return FitBatch(
        n=n, radius=radii.astype(f32), x_over_X0=np.full(L, cfg.x_over_X0, dtype=f32),
        Bz=cfg.Bz, mass=M_PION,
        par=np.ascontiguousarray(spar, dtype=f32), cov=np.ascontiguousarray(scov, dtype=f32),
        q=q.astype(np.int8), hpos=np.ascontiguousarray(hpos, dtype=f32),
        hcov=np.ascontiguousarray(hcov, dtype=f32), mask=mask, truth=truth, truth_vertex=truth_vertex,
        material_model=cfg.material_model,
        half_length=None if math.isinf(cfg.half_length_cm) else np.full(L, cfg.half_length_cm, dtype=f32),
        energy_loss=cfg.energy_loss)


# ---- barrel + endcap toy (reading A23; "a more realistic geometry"): six barrels of half
# length 30 cm inside four pairs of discs, |eta| up to 2.5
ENDCAP_BARREL_RADII = (4.0, 8.0, 12.0, 16.0, 20.0, 24.0)
ENDCAP_BARREL_HALF_LENGTH = 30.0
ENDCAP_DISC_Z = (35.0, 45.0, 55.0, 65.0)
ENDCAP_DISC_RMIN, ENDCAP_DISC_RMAX = 4.0, 26.0


def _cross_plane(pos, mom, q, Bz, zt):
    """Crossing of each truth helix with the plane z = zt: the turning angle follows from dz, the point by
    rotating the position about the helix centre (not the fit's sine / one-minus-cosine form)."""
    x, y, z = pos
    px, py, pz = mom
    k = q * C_B * Bz
    theta = k * (zt - z) / pz
    cx, cy = x + py / k, y - px / k
    c, sn = np.cos(theta), np.sin(theta)
    X = cx + (x - cx) * c + (y - cy) * sn
    Y = cy - (x - cx) * sn + (y - cy) * c
    return (X, Y, np.broadcast_to(zt, x.shape).astype(np.float64)), (px * c + py * sn, -px * sn + py * c, pz), theta


def simulate_endcap_event(event: int, n_tracks: int = 20_000, eta_max: float = 2.5, pt_min: float = 0.5,
                          pt_max: float = 10.0, x_over_X0: float = 0.01, Bz: float = 3.8, smear_hits: bool = True,
                          smear_seed: bool = True, material_model: int = 0, dtype=np.float32,
                          seed_prior_equals_smear: bool = False, seed_mom_smear: float = SEED_MOM_SMEAR,
                          seed_pos_smear: float = SEED_POS_SMEAR) -> FitBatch:
    """One event of the barrel + endcap toy.  Surfaces in list order: the six barrels by radius, then the four
    disc pairs by |z|; every track meets them in that order (the barrels end at |z| = 30 cm, inside the first
    disc).  A surface a track does not cross inside its sensitive area leaves no hit (mask bit 0) and no
    material; the truth moves on from the last surface it did cross.  Barrel hits as in simulate_event; disc
    hits: azimuth smeared by sigma_rphi / rho, radius by sigma_r = 0.1 cm, z exactly in the plane;
    V = Rz(phi_h) diag(sigma_r^2, sigma_rphi^2, sigma_z^2) Rz^T for both (the variance along a surface's own
    normal only keeps S invertible, reading A6).  seed_prior_equals_smear: the seed's prior covariance states the
    smearing actually applied (0.03 cm, 10 % of pT) instead of reading A13's deliberately loose 0.3 cm / 30 %: for
    pull tests on forward tracks, whose five hits on a short lever arm do not overrule the prior (with a prior
    that is trusted, the smearing must also be small enough for the filter's linearisation to hold: a 10 %
    momentum smear is a 0.1 rad direction error, 2 sigma_rphi of second-order displacement at the first layer)."""
    rng = np.random.default_rng(BASE_SEED + 1000 * 7 + event)
    n = n_tracks
    nb, nd = len(ENDCAP_BARREL_RADII), len(ENDCAP_DISC_Z)
    L = nb + nd
    q = rng.choice(np.array([-1.0, 1.0]), size=n)
    pt = rng.uniform(pt_min, pt_max, size=n)
    phi = rng.uniform(0.0, 2 * np.pi, size=n)
    eta = rng.uniform(-eta_max, eta_max, size=n)
    mom = (pt * np.cos(phi), pt * np.sin(phi), pt * np.sinh(eta))
    pos = (np.zeros(n), np.zeros(n), np.zeros(n))
    truth_vertex = np.stack(pos + mom)
    hpos = np.zeros((L, 3, n)); hcov = np.zeros((L, 6, n))
    truth = np.full((L, 6, n), np.nan)
    mask = np.zeros(n, dtype=np.uint32)
    k = q * C_B * Bz
    for l in range(L):
        ptl = np.hypot(mom[0], mom[1])
        if l < nb:
            r = ENDCAP_BARREL_RADII[l]
            R = ptl / np.abs(k)
            centre = np.hypot(pos[0] + mom[1] / k, pos[1] - mom[0] / k)
            reach = ~(r > 0.9 * (R + centre)) & (r > np.hypot(pos[0], pos[1]))
            with np.errstate(invalid="ignore", divide="ignore"):
                npos, nmom = _cross_cylinder(pos, mom, q, Bz, r)
            hit = reach & (np.abs(npos[2]) <= ENDCAP_BARREL_HALF_LENGTH)
        else:
            zt = np.where(mom[2] < 0, -1.0, 1.0) * ENDCAP_DISC_Z[l - nb]
            with np.errstate(invalid="ignore", divide="ignore"):
                npos, nmom, theta = _cross_plane(pos, mom, q, Bz, zt)
                rho = np.hypot(npos[0], npos[1])
                hit = ((zt - pos[2]) * mom[2] > 0) & (np.abs(theta) < 0.5 * np.pi) & (rho >= ENDCAP_DISC_RMIN) & (rho <= ENDCAP_DISC_RMAX)
        hit = hit & np.isfinite(npos[0]) & np.isfinite(npos[1])
        pos = tuple(np.where(hit, a, b) for a, b in zip(npos, pos))
        mom = tuple(np.where(hit, a, b) for a, b in zip(nmom, mom))
        g = rng.standard_normal((2, n))
        if not smear_hits:
            g = np.zeros_like(g)
        rho = np.hypot(pos[0], pos[1])
        phi_h = np.arctan2(pos[1], pos[0]) + g[0] * SIGMA_RPHI / np.maximum(rho, 1e-9)
        if l < nb:
            hp = np.stack([r * np.cos(phi_h), r * np.sin(phi_h), pos[2] + g[1] * SIGMA_Z])
        else:
            rh = rho + g[1] * SIGMA_R
            hp = np.stack([rh * np.cos(phi_h), rh * np.sin(phi_h), pos[2]])
        hv = hit_covariance(phi_h)
        hpos[l] = np.where(hit, hp, 0.0)
        hcov[l] = np.where(hit, hv, 0.0)
        mask |= (hit.astype(np.uint32) << np.uint32(l))
        a = rng.standard_normal((2, n))
        if x_over_X0 > 0.0:
            px, py, pz = mom
            p = np.sqrt(px * px + py * py + pz * pz)
            t_eff = x_over_X0
            if material_model == 1:
                cosn = np.abs(pos[0] * px + pos[1] * py) / (np.maximum(rho, 1e-9) * p) if l < nb else np.abs(pz) / p
                t_eff = x_over_X0 / cosn
            th0 = np.where(hit, highland_theta0(p, M_PION, t_eff), 0.0)
            ptt = np.hypot(px, py)
            e1 = (-py / ptt, px / ptt, np.zeros(n))
            ph = (px / p, py / p, pz / p)
            e2 = (ph[1] * e1[2] - ph[2] * e1[1], ph[2] * e1[0] - ph[0] * e1[2], ph[0] * e1[1] - ph[1] * e1[0])
            t1, t2 = np.tan(a[0] * th0), np.tan(a[1] * th0)
            d = tuple(ph[i] + t1 * e1[i] + t2 * e2[i] for i in range(3))
            dn = np.sqrt(d[0] ** 2 + d[1] ** 2 + d[2] ** 2)
            mom = tuple(np.where(hit, p * d[i] / dn, mom[i]) for i in range(3))
        truth[l] = np.where(hit, np.stack(pos + mom), np.nan)
    g = rng.standard_normal((6, n))
    if not smear_seed:
        g = np.zeros_like(g)
    spar = truth_vertex.copy()
    spar[0:3] += seed_pos_smear * g[0:3]
    spar[3:6] += seed_mom_smear * pt * g[3:6]
    spt = np.hypot(spar[3], spar[4])
    scov = np.zeros((21, n))
    diag_idx = [0, 6, 11, 15, 18, 20]
    for i in range(3):
        scov[diag_idx[i]] = (seed_pos_smear if seed_prior_equals_smear else SEED_POS_SIGMA0) ** 2
        scov[diag_idx[3 + i]] = (seed_mom_smear * pt) ** 2 if seed_prior_equals_smear else (SEED_MOM_SIGMA0 * spt) ** 2
    f32 = dtype
    # radius[] stays strictly increasing for the ABI's check; it is not read for disc layers
    radius = np.array(list(ENDCAP_BARREL_RADII) + [ENDCAP_BARREL_RADII[-1] + 1.0 + i for i in range(nd)])
    return FitBatch(
        n=n, radius=radius.astype(f32), x_over_X0=np.full(L, x_over_X0, dtype=f32), Bz=Bz, mass=M_PION,
        par=np.ascontiguousarray(spar, dtype=f32), cov=np.ascontiguousarray(scov, dtype=f32), q=q.astype(np.int8),
        hpos=np.ascontiguousarray(hpos, dtype=f32), hcov=np.ascontiguousarray(hcov, dtype=f32), mask=mask, truth=truth,
        truth_vertex=truth_vertex, material_model=material_model,
        half_length=np.array([ENDCAP_BARREL_HALF_LENGTH] * nb + [np.inf] * nd, dtype=f32),
        surface_type=np.array([0] * nb + [1] * nd, dtype=np.int32),
        disc_z=np.array([0.0] * nb + list(ENDCAP_DISC_Z), dtype=f32),
        disc_rmin=np.full(L, ENDCAP_DISC_RMIN, dtype=f32), disc_rmax=np.full(L, ENDCAP_DISC_RMAX, dtype=f32))


def concat_batches(batches: list[FitBatch]) -> FitBatch:
    b0 = batches[0]
    cat = lambda name, ax: np.ascontiguousarray(np.concatenate([getattr(b, name) for b in batches], axis=ax))
    return FitBatch(n=sum(b.n for b in batches), radius=b0.radius, x_over_X0=b0.x_over_X0, Bz=b0.Bz,
                    mass=b0.mass, par=cat("par", 1), cov=cat("cov", 1), q=cat("q", 0),
                    hpos=cat("hpos", 2), hcov=cat("hcov", 2), mask=cat("mask", 0),
                    truth=cat("truth", 2), truth_vertex=cat("truth_vertex", 1),
                    material_model=b0.material_model, half_length=b0.half_length, energy_loss=b0.energy_loss,
                    surface_type=b0.surface_type, disc_z=b0.disc_z, disc_rmin=b0.disc_rmin, disc_rmax=b0.disc_rmax)


def make_fit_batch(config: int, n_events: int | None = None, n_tracks: int | None = None) -> FitBatch:
    """The fit workload of config 0..3 (config 2 = 100 independent events concatenated)."""
    cfg = get_config(config)
    ne = cfg.n_events if n_events is None else n_events
    evs = [simulate_event(cfg, e, n_tracks) for e in range(ne)]
    return evs[0] if ne == 1 else concat_batches(evs)


@dataclass
class LayerHits:
    """All hits of one layer of one event (true + noise, shuffled), fp32 SoA."""
    radius: float
    pos: np.ndarray        # [3][H] f32
    cov: np.ndarray        # [6][H] f32
    true_index: np.ndarray  # [n_tracks] i32: index of track i's own hit in this pool


@dataclass
class BuildEvent:
    """config 4: one config-1-style event plus per-layer hit pools with uniform noise."""
    cfg: BarrelConfig
    fit: FitBatch              # the event's tracks with their true hits (used to make seeds)
    layers: list[LayerHits]


def make_build_event(config: int = 4, n_tracks: int | None = None, noise_hits: int | None = None) -> BuildEvent:
    cfg = get_config(config)
    fit = simulate_event(cfg, 0, n_tracks)
    rng = np.random.default_rng(BASE_SEED + 1000 * cfg.index + 500)
    n_noise = cfg.noise_hits_per_layer if noise_hits is None else noise_hits
    layers = []
    for l in range(cfg.n_layers):
        r = float(cfg.radii[l])
        eta = rng.uniform(-cfg.eta_bin_max, cfg.eta_bin_max, size=n_noise)
        phi = rng.uniform(-np.pi, np.pi, size=n_noise)
        npos = np.stack([r * np.cos(phi), r * np.sin(phi), r * np.sinh(eta)])
        ncov = hit_covariance(phi)
        pos = np.concatenate([fit.hpos[l].astype(np.float64), npos], axis=1)
        cov = np.concatenate([fit.hcov[l].astype(np.float64), ncov], axis=1)
        H = pos.shape[1]
        perm = rng.permutation(H)                      # pool slot j holds original hit perm[j]
        inv = np.empty(H, dtype=np.int64)
        inv[perm] = np.arange(H)
        layers.append(LayerHits(radius=r,
                                pos=np.ascontiguousarray(pos[:, perm], dtype=np.float32),
                                cov=np.ascontiguousarray(cov[:, perm], dtype=np.float32),
                                true_index=inv[:fit.n].astype(np.int32)))
    return BuildEvent(cfg=cfg, fit=fit, layers=layers)


@dataclass
class EndcapBuildEvent:
    """The barrel + endcap toy as a building workload: the event's tracks plus, per surface, ALL its hits (the
    tracks' own hits where they left one, and uniform noise), shuffled, fp32 SoA."""
    fit: FitBatch
    layers: list[LayerHits]     # radius = 0 for a disc layer (reading A24); true_index = -1 where the track left no hit


def make_endcap_build_event(n_tracks: int = 3000, noise_hits: int = 15000, event: int = 0, **kw) -> EndcapBuildEvent:
    fit = simulate_endcap_event(event, n_tracks, **kw)
    rng = np.random.default_rng(BASE_SEED + 77000 + event)
    layers = []
    for l in range(fit.n_layers):
        has = ((fit.mask >> l) & 1) == 1
        phi = rng.uniform(-np.pi, np.pi, size=noise_hits)
        if fit.surface_type[l] == 1:
            rho = np.sqrt(rng.uniform(fit.disc_rmin[l] ** 2, fit.disc_rmax[l] ** 2, size=noise_hits))
            z = rng.choice([-1.0, 1.0], size=noise_hits) * fit.disc_z[l]
            r_bins = 0.0
        else:
            rho = np.full(noise_hits, float(fit.radius[l]))
            hl = float(fit.half_length[l]) if fit.half_length is not None else 30.0
            z = rng.uniform(-hl, hl, size=noise_hits)
            r_bins = float(fit.radius[l])
        npos = np.stack([rho * np.cos(phi), rho * np.sin(phi), z])
        pos = np.concatenate([fit.hpos[l][:, has].astype(np.float64), npos], axis=1)
        cov = np.concatenate([fit.hcov[l][:, has].astype(np.float64), hit_covariance(phi)], axis=1)
        H = pos.shape[1]
        perm = rng.permutation(H)
        inv = np.empty(H, dtype=np.int64)
        inv[perm] = np.arange(H)
        true_index = np.full(fit.n, -1, dtype=np.int32)
        true_index[has] = inv[:int(has.sum())].astype(np.int32)
        layers.append(LayerHits(radius=r_bins, pos=np.ascontiguousarray(pos[:, perm], dtype=np.float32),
                                cov=np.ascontiguousarray(cov[:, perm], dtype=np.float32), true_index=true_index))
    return EndcapBuildEvent(fit=fit, layers=layers)
