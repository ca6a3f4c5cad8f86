/*
 * kf_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision CPU statement of what the hot path computes: batched
 * Kalman-filter track fitting and best-hit candidate scoring in a cylindrical barrel
 * (arXiv:1705.02876; "seeding, building, fitting" + chi2; PAPER.md:65 6x6 track /
 * 3x3 hit matrices in global coordinates; PAPER.md:71 projective bins; PAPER.md:73 best hit =
 * lowest chi2 increment; equations: BASELINE.json:north_star).  The paper prints no formulas;
 * every formula below is a reading listed in DESIGN.md ("Readings A1..A24").
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this.  It shares no code, header, table or constant with the CUDA path
 * (paper_1705_02876_b200/csrc) and is never a fallback for it.
 *
 * Conventions: AoS per track, dense 6x6 row-major matrices, no blocking / fusion / reordering.
 * State u = (x, y, z, px, py, pz) [cm, GeV/c]; charge q = +-1; B = Bz z-hat [Tesla].
 *
 * Pins (tests/test_oracle_pins.py, tests/test_oracle_smoother.py): P1 exact helix recovery, P2 propagation invariants + RK4 +
 * worked value, P3 Jacobian vs finite differences / radial null / |p| conservation, P4 EKF ==
 * batch weighted least squares, P5 covariance PSD rank 5, P6 pulls and chi2/ndf, P7 Highland
 * check values, P8 window scoring == brute force, P9 bin structure, P10 rotation symmetry;
 * G1-G3 geometry options (tests/test_oracle_geometry.py); E1-E6 energy loss (tests/test_oracle_energy_loss.py);
 * orc_chi2_increment against its definition and against orc_update (tests/test_oracle_scoring.py);
 * SM1-SM5 the RTS smoother (tests/test_oracle_smoother.py: batch WLS at every layer, exact helix, pulls);
 * R1-R5 the inward refit (tests/test_oracle_refit.py); C1-C4 combinatorial building;
 * D1-D9 endcap discs (tests/test_oracle_endcap.py: to-plane propagation vs RK4 and vs the to-radius form,
 * Jacobian, exact helix through barrels + discs, EKF and smoother == WLS, pulls, path-length material on a disc;
 * D7-D9 scoring on a disc layer against brute force, combinatorial building with discs, the inward refit over
 * surfaces); the bin of a disc-layer hit (reading A24) against its definition (tests/test_oracle_scoring.py).
 * Parity-unpinned: none of the functions below (efficiency / fake rate of PAPER.md:85 is not
 * computed here at all).
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_C_B 2.99792458e-3 /* GeV/(c T cm), reading A1 */
#define ORC_PI 3.14159265358979323846

enum { ORC_PROP_FAIL = 1, ORC_S_NOT_PD = 2, ORC_NONFINITE = 4, ORC_BAD_CHARGE = 8, ORC_OUTSIDE = 16 };

/* ---- geometry options (reading A20; "more realistic geometry"), process-wide, set by the
 * caller before a fit / scoring call; defaults = readings A5 (flat thickness) and A12 (infinite cylinders):
 *   material_model 1: the thickness seen by the track is t / cos(psi), psi = angle between the momentum
 *                     and the cylinder normal at the crossing, cos(psi) = |x px + y py| / (rho |p|);
 *   half_length[l]:   a crossing with |z'| > half_length[l] misses layer l: ORC_OUTSIDE, layer skipped,
 *                     track untouched (same bookkeeping as ORC_PROP_FAIL).                              */
static int g_material_model = 0;
static double g_half_length[32] = {
    INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY,
    INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY,
    INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY, INFINITY};

static int g_energy_loss = 0; /* reading A21: 0 none, 1 mean Bethe loss in silicon at every layer crossing */
void orc_set_energy_loss(int model) { g_energy_loss = model; }

/* ---- surfaces (reading A23; "a more realistic geometry" with endcaps): layer l is a barrel cylinder
 * (type 0: radius[l], optional half length) or a PAIR of endcap discs (type 1) in the planes z = +-disc_z[l],
 * sensitive for disc_rmin[l] <= rho <= disc_rmax[l].  A track meets the disc on the side it is heading to
 * (sign of pz).  Default: all barrels. */
static int g_surface_type[32] = {0};
static double g_disc_z[32], g_disc_rmin[32], g_disc_rmax[32];
void orc_set_surfaces(int n_layers, const int32_t *type, const double *disc_z, const double *rmin, const double *rmax) {
    for (int l = 0; l < 32; ++l) {
        g_surface_type[l] = (type && l < n_layers) ? type[l] : 0;
        g_disc_z[l] = (disc_z && l < n_layers) ? disc_z[l] : 0.0;
        g_disc_rmin[l] = (rmin && l < n_layers) ? rmin[l] : 0.0;
        g_disc_rmax[l] = (rmax && l < n_layers) ? rmax[l] : INFINITY;
    }
}

static double g_score_half_length = INFINITY; /* the one layer orc_score_layer works on */
void orc_set_score_half_length(double h) { g_score_half_length = h; }
/* ... and its surface (readings A23 / A24): type 0 = the cylinder of radius r_layer, 1 = the disc pair z = +-zd with
 * the annulus rmin <= rho <= rmax (r_layer is then not used). */
static int g_score_type = 0;
static double g_score_zd = 0.0, g_score_rmin = 0.0, g_score_rmax = INFINITY;
void orc_set_score_surface(int type, double zd, double rmin, double rmax) {
    g_score_type = type; g_score_zd = zd; g_score_rmin = rmin; g_score_rmax = rmax;
}

void orc_set_geometry_options(int material_model, int n_layers, const double *half_length) {
    g_material_model = material_model;
    for (int l = 0; l < 32; ++l) g_half_length[l] = (half_length && l < n_layers) ? half_length[l] : INFINITY;
}

/* ---- Highland multiple-scattering width (reading A5) --------------------------------------
 * theta0 = 0.0136 GeV / (beta p) * sqrt(t) * (1 + 0.038 ln t), t = x/X0 (flat), beta = p/E. */
double orc_theta0(double p, double mass, double t) {
    if (t <= 0.0) return 0.0;
    double beta = p / sqrt(p * p + mass * mass);
    return 0.0136 / (beta * p) * sqrt(t) * (1.0 + 0.038 * log(t));
}

/* ---- helix propagation to the cylinder of radius r, with Jacobian (readings A2, A3, A4) ----
 * Equations of motion, s = transverse path length, kappa = k / pT, k = q c_B Bz:
 *   dx/ds = px/pT  dy/ds = py/pT  dz/ds = pz/pT  dpx/ds = kappa py  dpy/ds = -kappa px  dpz/ds = 0
 * Solution with theta = kappa s, S = sin theta, Cm = 1 - cos theta:
 *   x' = x + (px S + py Cm)/k   y' = y + (py S - px Cm)/k   z' = z + pz s/pT
 *   px' = px cos + py S         py' = -px S + py cos        pz' = pz
 * First outward crossing of |pos'| = r:  a S - b Cm = D with
 *   a = x px + y py,  b = (y px - x py) - pT^2/k,  D = (k/2)(r^2 - x^2 - y^2);
 *   t = tan(theta/2) = D / (a + sqrt(a^2 - D(2b + D))).
 * F = A + (df/ds) (x) (ds/du): A = d(map)/du at fixed s, ds/du from the constraint |pos'| = r.
 * Returns 0 or ORC_PROP_FAIL (then nothing is written). F may be NULL. */
static int propagate_dir(const double u[6], double q, double Bz, double r, int inward, double out[6],
                         double F[36], double *s_out, double *theta_out) {
    double x = u[0], y = u[1], z = u[2], px = u[3], py = u[4], pz = u[5];
    double k = q * ORC_C_B * Bz;
    double pt2 = px * px + py * py;
    double pt = sqrt(pt2);
    double rho2 = x * x + y * y;
    /* outward: target radius outside the current one; inward (reading A18): inside, reached by
     * following the same helix BACKWARD in path length (D < 0 gives t < 0, theta < 0, s < 0) */
    if (inward ? !(r * r < rho2) : !(r * r > rho2)) return ORC_PROP_FAIL;
    double a = x * px + y * py;
    double b = (y * px - x * py) - pt2 / k;
    double D = 0.5 * k * (r * r - rho2);
    double disc = a * a - D * (2.0 * b + D);
    if (!(disc > 0.0)) return ORC_PROP_FAIL;
    double den = a + sqrt(disc);
    if (!(den > 0.0)) return ORC_PROP_FAIL;
    double t = D / den;
    double S = 2.0 * t / (1.0 + t * t);
    double Cm = 2.0 * t * t / (1.0 + t * t);
    double co = 1.0 - Cm;
    double theta = 2.0 * atan(t);
    double s = theta * pt / k;
    double xn = x + (px * S + py * Cm) / k;
    double yn = y + (py * S - px * Cm) / k;
    double zn = z + pz * s / pt;
    double pxn = px * co + py * S;
    double pyn = -px * S + py * co;
    if (F) {
        double A[6][6];
        memset(A, 0, sizeof A);
        for (int i = 0; i < 6; ++i) A[i][i] = 1.0;
        double taux = -theta * px / pt2, tauy = -theta * py / pt2; /* d theta / d(px,py) at fixed s */
        A[0][3] = S / k + pxn * taux / k;
        A[0][4] = Cm / k + pxn * tauy / k;
        A[1][3] = -Cm / k + pyn * taux / k;
        A[1][4] = S / k + pyn * tauy / k;
        A[2][3] = -pz * s * px / (pt2 * pt);
        A[2][4] = -pz * s * py / (pt2 * pt);
        A[2][5] = s / pt;
        A[3][3] = co + pyn * taux;
        A[3][4] = S + pyn * tauy;
        A[4][3] = -S - pxn * taux;
        A[4][4] = co - pxn * tauy;
        double kap = k / pt;
        double dfds[6] = {pxn / pt, pyn / pt, pz / pt, kap * pyn, -kap * pxn, 0.0};
        double vr = (xn * pxn + yn * pyn) / pt; /* d(|pos'|^2 / 2)/ds */
        for (int c = 0; c < 6; ++c) {
            double dsdu = -(xn * A[0][c] + yn * A[1][c]) / vr;
            for (int i = 0; i < 6; ++i) F[i * 6 + c] = A[i][c] + dfds[i] * dsdu;
        }
    }
    out[0] = xn; out[1] = yn; out[2] = zn; out[3] = pxn; out[4] = pyn; out[5] = pz;
    if (s_out) *s_out = s;
    if (theta_out) *theta_out = theta;
    return 0;
}

int orc_propagate(const double u[6], double q, double Bz, double r, double out[6], double F[36],
                  double *s_out, double *theta_out) {
    return propagate_dir(u, q, Bz, r, 0, out, F, s_out, theta_out);
}

/* Same closed form followed backward along the helix to a SMALLER radius (reading A18). */
int orc_propagate_inward(const double u[6], double q, double Bz, double r, double out[6], double F[36],
                         double *s_out, double *theta_out) {
    return propagate_dir(u, q, Bz, r, 1, out, F, s_out, theta_out);
}

/* ---- helix propagation to the plane z = zt, with Jacobian (reading A23) ---------------------------------------
 * Same equations of motion and solution as above (reading A2); the path length now follows from z' = zt:
 *   s = (zt - z) pT / pz,   theta = kappa s = k (zt - z) / pz.
 * F = A + (df/ds) (x) (ds/du) with the same A (derivative at fixed s) and ds/du from the constraint z' = zt:
 *   ds/du = -A[z, u] / (pz / pT)      (so row z of F vanishes: the arrival point stays in the plane and the
 *   transported covariance has no variance along z -- the disc's counterpart of the radial null of a cylinder).
 * Fails (ORC_PROP_FAIL, nothing written) unless the plane lies ahead (s > 0) within half a turn (|theta| < pi). */
static int propagate_to_z_dir(const double u[6], double q, double Bz, double zt, int inward, double out[6],
                              double F[36], double *s_out, double *theta_out) {
    double x = u[0], y = u[1], z = u[2], px = u[3], py = u[4], pz = u[5];
    double k = q * ORC_C_B * Bz;
    double pt2 = px * px + py * py;
    double pt = sqrt(pt2);
    if (!(pt > 0.0) || pz == 0.0) return ORC_PROP_FAIL;
    double s = (zt - z) * pt / pz;
    /* inward (the refit of reading A18 on a geometry with discs): the plane lies BEHIND the state, reached by
     * following the same helix backward in path length (s < 0, theta of the opposite sign) */
    if (inward ? !(s < 0.0) : !(s > 0.0)) return ORC_PROP_FAIL;
    double theta = k * s / pt;
    if (!(fabs(theta) < ORC_PI)) return ORC_PROP_FAIL;
    double S = sin(theta), co = cos(theta);
    double sh = sin(0.5 * theta);
    double Cm = 2.0 * sh * sh; /* 1 - cos(theta) without cancellation */
    double xn = x + (px * S + py * Cm) / k;
    double yn = y + (py * S - px * Cm) / k;
    double pxn = px * co + py * S;
    double pyn = -px * S + py * co;
    if (F) {
        double A[6][6];
        memset(A, 0, sizeof A);
        for (int i = 0; i < 6; ++i) A[i][i] = 1.0;
        double taux = -theta * px / pt2, tauy = -theta * py / pt2; /* d theta / d(px,py) at fixed s */
        A[0][3] = S / k + pxn * taux / k;
        A[0][4] = Cm / k + pxn * tauy / k;
        A[1][3] = -Cm / k + pyn * taux / k;
        A[1][4] = S / k + pyn * tauy / k;
        A[2][3] = -pz * s * px / (pt2 * pt);
        A[2][4] = -pz * s * py / (pt2 * pt);
        A[2][5] = s / pt;
        A[3][3] = co + pyn * taux;
        A[3][4] = S + pyn * tauy;
        A[4][3] = -S - pxn * taux;
        A[4][4] = co - pxn * tauy;
        double kap = k / pt;
        double dfds[6] = {pxn / pt, pyn / pt, pz / pt, kap * pyn, -kap * pxn, 0.0};
        for (int c = 0; c < 6; ++c) {
            double dsdu = -A[2][c] / (pz / pt);
            for (int i = 0; i < 6; ++i) F[i * 6 + c] = A[i][c] + dfds[i] * dsdu;
        }
    }
    out[0] = xn; out[1] = yn; out[2] = zt; out[3] = pxn; out[4] = pyn; out[5] = pz;
    if (s_out) *s_out = s;
    if (theta_out) *theta_out = theta;
    return 0;
}
int orc_propagate_to_z(const double u[6], double q, double Bz, double zt, double out[6], double F[36],
                       double *s_out, double *theta_out) {
    return propagate_to_z_dir(u, q, Bz, zt, 0, out, F, s_out, theta_out);
}

/* One layer of the geometry as the filter meets it: barrel (type 0) or disc pair (type 1, the disc on the side the
 * track is heading to).  ORC_OUTSIDE: the crossing exists but lies beyond the barrel end / outside the annulus. */
static int reach_surface(int l, const double u[6], double q, double Bz, double radius, double out[6], double F[36]) {
    if (g_surface_type[l] == 0) {
        int rc = orc_propagate(u, q, Bz, radius, out, F, NULL, NULL);
        if (!rc && fabs(out[2]) > g_half_length[l]) rc = ORC_OUTSIDE;
        return rc;
    }
    int rc = orc_propagate_to_z(u, q, Bz, u[5] < 0.0 ? -g_disc_z[l] : g_disc_z[l], out, F, NULL, NULL);
    if (!rc) {
        double rho = sqrt(out[0] * out[0] + out[1] * out[1]);
        if (rho < g_disc_rmin[l] || rho > g_disc_rmax[l]) rc = ORC_OUTSIDE;
    }
    return rc;
}

/* ---- process noise (reading A5): thin scatterer at the layer, evaluated at the propagated
 * momentum p': Q_pp = theta0^2 (|p|^2 I3 - p p^T), all other blocks zero. */
static _Thread_local int g_at_surface = 0; /* type of the surface the state handed to the two functions below stands on (fit_one sets it) */
static double cos_incidence(const double u[6]) { /* |cos| of the angle between the momentum and the surface normal */
    double p = sqrt(u[3] * u[3] + u[4] * u[4] + u[5] * u[5]);
    if (g_at_surface == 1) return fabs(u[5]) / p;                                      /* disc: normal = z axis */
    return fabs(u[0] * u[3] + u[1] * u[4]) / (sqrt(u[0] * u[0] + u[1] * u[1]) * p); /* cylinder: normal = radial */
}
void orc_process_noise(const double u[6], double mass, double t, double Q[36]) {
    memset(Q, 0, 36 * sizeof(double));
    double p2 = u[3] * u[3] + u[4] * u[4] + u[5] * u[5];
    if (g_material_model == 1 && t > 0.0) t = t / cos_incidence(u); /* A20: path length through the layer */
    double th0 = orc_theta0(sqrt(p2), mass, t);
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            Q[(3 + i) * 6 + 3 + j] = th0 * th0 * ((i == j ? p2 : 0.0) - u[3 + i] * u[3 + j]);
}

/* C' = F C F^T + Q (north_star), dense triple loops. */
void orc_transport_cov(const double F[36], const double C[36], const double Q[36], double out[36]) {
    double FC[36];
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            double acc = 0.0;
            for (int m = 0; m < 6; ++m) acc += F[i * 6 + m] * C[m * 6 + j];
            FC[i * 6 + j] = acc;
        }
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            double acc = 0.0;
            for (int m = 0; m < 6; ++m) acc += FC[i * 6 + m] * F[j * 6 + m];
            out[i * 6 + j] = acc + Q[i * 6 + j];
        }
}

/* ---- mean energy loss in the layer material (reading A21; PAPER.md:168 defers "more realistic" detector
 * descriptions; SURVEY 8(f) item 4 names energy loss) -------------------------------------------------------
 * Bethe's mean stopping power for a heavy charged particle of unit charge (PDG "Passage of particles
 * through matter"), no density-effect and no shell correction:
 *   -dE/dx = K (Z/A) (1/beta^2) [ (1/2) ln( 2 me beta^2 gamma^2 Tmax / I^2 ) - beta^2 ]      [GeV cm^2 / g]
 *   Tmax   = 2 me beta^2 gamma^2 / (1 + 2 gamma me/M + (me/M)^2)
 * with K = 0.307075 MeV cm^2/mol, me = 0.51099895 MeV.  The layers are silicon: Z/A = 14/28.0855,
 * I = 173 eV, X0 = 21.82 g/cm^2, so a layer of t radiation lengths is t * 21.82 g/cm^2 thick.
 * orc_energy_loss returns the energy [GeV] lost over t radiation lengths (t already scaled by the path
 * length where that applies). */
#define ORC_BETHE_K 0.307075e-3  /* GeV cm^2 / mol */
#define ORC_ME 0.51099895e-3     /* GeV */
#define ORC_SI_Z_OVER_A (14.0 / 28.0855)
#define ORC_SI_I 173.0e-9        /* GeV */
#define ORC_SI_X0 21.82          /* g / cm^2 */
double orc_energy_loss(double p, double mass, double t) {
    if (t <= 0.0) return 0.0;
    double E = sqrt(p * p + mass * mass);
    double beta2 = p * p / (E * E);
    double gamma = E / mass;
    double bg2 = beta2 * gamma * gamma;
    double r = ORC_ME / mass;
    double Tmax = 2.0 * ORC_ME * bg2 / (1.0 + 2.0 * gamma * r + r * r);
    double dedx = ORC_BETHE_K * ORC_SI_Z_OVER_A / beta2 *
                  (0.5 * log(2.0 * ORC_ME * bg2 * Tmax / (ORC_SI_I * ORC_SI_I)) - beta2);
    return dedx * t * ORC_SI_X0;
}

/* The effective thickness a state standing on a cylinder sees (A20 path length if that option is on). */
static double cos_incidence(const double u[6]);
static double seen_thickness(const double u[6], double t) {
    if (g_material_model == 1 && t > 0.0) t = t / cos_incidence(u);
    return t;
}

/* Energy-loss step at a layer (reading A21).  direction +1 (forward filter, on arrival, after C' = F C F^T + Q):
 * E'' = E - dE(p), direction -1 (backward refit, on leaving the layer inward): E'' = E + dE(p), dE evaluated
 * at the momentum the state HAS (so the backward step inverts the forward one to first order in dE).  The
 * momentum keeps its direction: p'' = f p, f = |p''|/|p|.  Jacobian with dE held fixed (its own dependence
 * on p changes d|p''|/d|p| by about dE/p, 1e-3 or less, neglected): d|p''|/d|p| = g = (E''/|p''|)(|p|/E), so
 *   J = blockdiag(I3, f I3 + (g - f) n n^T), n = p/|p|;   C <- J C J^T.   No straggling term is added.
 * Returns ORC_PROP_FAIL (nothing written) if the particle would stop (E'' <= mass).  J36 (optional) gets J. */
int orc_energy_loss_step(double u[6], double C[36], double mass, double t, int direction, double J36[36]) {
    double p2 = u[3] * u[3] + u[4] * u[4] + u[5] * u[5];
    double p = sqrt(p2), E = sqrt(p2 + mass * mass);
    double dE = orc_energy_loss(p, mass, seen_thickness(u, t));
    double E2 = direction > 0 ? E - dE : E + dE;
    if (!(E2 > mass)) return ORC_PROP_FAIL;
    double pn = sqrt(E2 * E2 - mass * mass);
    double f = pn / p, g = (E2 / pn) * (p / E);
    double J[36], JC[36], out[36];
    memset(J, 0, sizeof J);
    for (int i = 0; i < 3; ++i) J[i * 6 + i] = 1.0;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            J[(3 + i) * 6 + 3 + j] = (i == j ? f : 0.0) + (g - f) * u[3 + i] * u[3 + j] / p2;
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            double acc = 0.0;
            for (int m = 0; m < 6; ++m) acc += J[i * 6 + m] * C[m * 6 + j];
            JC[i * 6 + j] = acc;
        }
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            double acc = 0.0;
            for (int m = 0; m < 6; ++m) acc += JC[i * 6 + m] * J[j * 6 + m];
            out[i * 6 + j] = acc;
        }
    memcpy(C, out, sizeof out);
    for (int i = 3; i < 6; ++i) u[i] *= f;
    if (J36) memcpy(J36, J, sizeof J);
    return 0;
}

/* inverse of a symmetric 3x3 by cofactors; returns det */
static double inv3(const double S[9], double Si[9]) {
    double c00 = S[4] * S[8] - S[5] * S[7];
    double c01 = S[5] * S[6] - S[3] * S[8];
    double c02 = S[3] * S[7] - S[4] * S[6];
    double det = S[0] * c00 + S[1] * c01 + S[2] * c02;
    double id = 1.0 / det;
    Si[0] = c00 * id;
    Si[1] = (S[2] * S[7] - S[1] * S[8]) * id;
    Si[2] = (S[1] * S[5] - S[2] * S[4]) * id;
    Si[3] = c01 * id;
    Si[4] = (S[0] * S[8] - S[2] * S[6]) * id;
    Si[5] = (S[2] * S[3] - S[0] * S[5]) * id;
    Si[6] = c02 * id;
    Si[7] = (S[1] * S[6] - S[0] * S[7]) * id;
    Si[8] = (S[0] * S[4] - S[1] * S[3]) * id;
    return det;
}

/* ---- chi2 increment of hit (m, V) against state (u, C) (readings A6, A8):
 * r = m - H u, H = [I3 0]; S = C_pp + V; chi2 = r^T S^-1 r.  Returns 0 / ORC_S_NOT_PD. */
int orc_chi2_increment(const double u[6], const double C[36], const double m[3], const double V[9],
                       double *chi2) {
    double S[9], Si[9], r[3];
    for (int i = 0; i < 3; ++i) {
        r[i] = m[i] - u[i];
        for (int j = 0; j < 3; ++j) S[i * 3 + j] = C[i * 6 + j] + V[i * 3 + j];
    }
    if (!(inv3(S, Si) > 0.0)) return ORC_S_NOT_PD;
    double c = 0.0;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c += r[i] * Si[i * 3 + j] * r[j];
    *chi2 = c;
    return 0;
}

/* ---- Kalman update (reading A8): K = C H^T S^-1; x = u + K r;
 * C_new = (I - K H) C (I - K H)^T + K V K^T  (Joseph form of C - K H C), symmetrised. */
int orc_update(const double u[6], const double C[36], const double m[3], const double V[9],
               double uo[6], double Co[36], double *chi2) {
    double S[9], Si[9], r[3], K[18], c = 0.0;
    for (int i = 0; i < 3; ++i) {
        r[i] = m[i] - u[i];
        for (int j = 0; j < 3; ++j) S[i * 3 + j] = C[i * 6 + j] + V[i * 3 + j];
    }
    if (!(inv3(S, Si) > 0.0)) return ORC_S_NOT_PD;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c += r[i] * Si[i * 3 + j] * r[j];
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 3; ++j) {
            double acc = 0.0;
            for (int m2 = 0; m2 < 3; ++m2) acc += C[i * 6 + m2] * Si[m2 * 3 + j];
            K[i * 3 + j] = acc;
        }
    double un[6];
    for (int i = 0; i < 6; ++i) un[i] = u[i] + K[i * 3] * r[0] + K[i * 3 + 1] * r[1] + K[i * 3 + 2] * r[2];
    double A[36], AC[36], Cn[36];
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) A[i * 6 + j] = (i == j ? 1.0 : 0.0) - (j < 3 ? K[i * 3 + j] : 0.0);
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            double acc = 0.0;
            for (int m2 = 0; m2 < 6; ++m2) acc += A[i * 6 + m2] * C[m2 * 6 + j];
            AC[i * 6 + j] = acc;
        }
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            double acc = 0.0;
            for (int m2 = 0; m2 < 6; ++m2) acc += AC[i * 6 + m2] * A[j * 6 + m2];
            for (int a2 = 0; a2 < 3; ++a2)
                for (int b2 = 0; b2 < 3; ++b2) acc += K[i * 3 + a2] * V[a2 * 3 + b2] * K[j * 3 + b2];
            Cn[i * 6 + j] = acc;
        }
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) Co[i * 6 + j] = 0.5 * (Cn[i * 6 + j] + Cn[j * 6 + i]);
    int finite = isfinite(c);
    for (int i = 0; i < 6; ++i) finite = finite && isfinite(un[i]);
    if (!finite) return ORC_NONFINITE;
    memcpy(uo, un, sizeof un);
    *chi2 = c;
    return 0;
}

/* ---- one track, all layers (readings A10, A11): layers in increasing radius; a layer whose
 * mask bit is 0 is skipped entirely; a layer that fails (propagation / S / non-finite) sets the
 * status bit and leaves state and covariance as they were before that layer.
 * trace (optional): per layer 194 doubles = x_pred[6] F[36] Q[36] x_filt[6] C_filt[36] dchi2 used
 *                   C_pred[36] G[36], where x_pred / C_pred are the predicted state and covariance the update
 *                   was given (after the energy-loss step of reading A21 when that option is on) and G is the
 *                   Jacobian of the whole map previous filtered state -> x_pred (G = F, or J F with energy loss) */
#define ORC_TRACE_STRIDE 194
static void fit_one(int L, const double *radius, const double *xX0, double Bz, double mass,
                    const double par[6], const double cov[36], int q, const double *hpos,
                    const double *hcov, uint32_t mask, double opar[6], double ocov[36],
                    double *ochi2, int32_t *onhits, uint32_t *ostatus, double *trace) {
    double u[6], C[36];
    memcpy(u, par, sizeof u);
    memcpy(C, cov, sizeof C);
    double chi2 = 0.0;
    int nh = 0;
    uint32_t st = 0;
    if (q != 1 && q != -1) {
        st = ORC_BAD_CHARGE;
    } else {
        for (int l = 0; l < L; ++l) {
            double *tr = trace ? trace + (size_t)l * ORC_TRACE_STRIDE : NULL;
            if (tr) memset(tr, 0, ORC_TRACE_STRIDE * sizeof(double));
            if (!((mask >> l) & 1u)) continue;
            double up[6], F[36], Q[36], Cp[36], un[6], Cn[36], dchi2;
            int rc = reach_surface(l, u, (double)q, Bz, radius[l], up, F); /* cylinder, or disc (reading A23) */
            if (tr && rc == ORC_OUTSIDE) memcpy(tr, up, 6 * sizeof(double)); /* diagnostic: where it missed */
            if (rc) { st |= (uint32_t)rc; continue; }
            g_at_surface = g_surface_type[l];
            orc_process_noise(up, mass, xX0[l], Q);
            orc_transport_cov(F, C, Q, Cp);
            double G[36];
            memcpy(G, F, sizeof G);
            if (g_energy_loss) { /* A21 */
                double J[36];
                rc = orc_energy_loss_step(up, Cp, mass, xX0[l], +1, J);
                for (int i = 0; i < 6; ++i)
                    for (int j = 0; j < 6; ++j) {
                        double acc = 0.0;
                        for (int m = 0; m < 6; ++m) acc += J[i * 6 + m] * F[m * 6 + j];
                        G[i * 6 + j] = acc;
                    }
            }
            if (rc) { st |= (uint32_t)rc; continue; }
            rc = orc_update(up, Cp, hpos + 3 * l, hcov + 9 * l, un, Cn, &dchi2);
            if (rc) { st |= (uint32_t)rc; continue; }
            memcpy(u, un, sizeof u);
            memcpy(C, Cn, sizeof C);
            chi2 += dchi2;
            nh += 1;
            if (tr) {
                memcpy(tr, up, 6 * sizeof(double));
                memcpy(tr + 6, F, 36 * sizeof(double));
                memcpy(tr + 42, Q, 36 * sizeof(double));
                memcpy(tr + 78, u, 6 * sizeof(double));
                memcpy(tr + 84, C, 36 * sizeof(double));
                tr[120] = dchi2;
                tr[121] = 1.0;
                memcpy(tr + 122, Cp, 36 * sizeof(double));
                memcpy(tr + 158, G, 36 * sizeof(double));
            }
        }
    }
    g_at_surface = 0;
    memcpy(opar, u, sizeof u);
    memcpy(ocov, C, sizeof C);
    *ochi2 = chi2;
    *onhits = nh;
    *ostatus = st;
}

/* ---- fixed-interval smoother (reading A22; "a final fit with a KF and smoother") ----------------
 * The Rauch-Tung-Striebel recursion over the layers the forward filter used, k_0 < k_1 < ... < k_{m-1}, on the
 * model that filter linearised (its own predictions x^-_k, C^-_k, Jacobians G_k, filtered x^+_k, C^+_k):
 *     x^s_{m-1} = x^+_{m-1},  C^s_{m-1} = C^+_{m-1};   then for j = m-2 ... 0, with n = k_{j+1}:
 *     A     = C^+_j G_n^T (C^-_n)^+
 *     x^s_j = x^+_j + A (x^s_n - x^-_n)
 *     C^s_j = C^+_j + A (C^s_n - C^-_n) A^T
 * x^s_k is the best estimate, given ALL hits of the track, of the state just after the scatter of layer k (the
 * state the forward filter's x^+_k estimates from the hits up to k).  It equals the batch weighted-least-squares
 * solution of the linearised model evaluated at every layer (pin SM1).
 * (C^-_n)^+ is the pseudo-inverse: a covariance transported to a cylinder has no variance along the radial
 * direction e = (x^-, y^-, 0; 0, 0, 0)/rho of the predicted point (reading A4, pin P5), so with that known unit
 * null vector   (C^-)^+ = (C^- + s e e^T)^-1 - e e^T / s   for any s > 0 (s = largest position variance). */
static int inv6(const double M[36], double Mi[36]) { /* Gauss-Jordan with partial pivoting on the symmetrically
                                                        scaled matrix D M D, D = diag(1/sqrt(M_ii)) */
    double a[6][12], d[6];
    for (int i = 0; i < 6; ++i) {
        if (!(M[i * 6 + i] > 0.0)) return -1;
        d[i] = 1.0 / sqrt(M[i * 6 + i]);
    }
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            a[i][j] = d[i] * M[i * 6 + j] * d[j];
            a[i][6 + j] = i == j ? 1.0 : 0.0;
        }
    for (int c = 0; c < 6; ++c) {
        int piv = c;
        for (int r = c + 1; r < 6; ++r)
            if (fabs(a[r][c]) > fabs(a[piv][c])) piv = r;
        if (!(fabs(a[piv][c]) > 0.0)) return -1;
        if (piv != c)
            for (int j = 0; j < 12; ++j) { double t = a[c][j]; a[c][j] = a[piv][j]; a[piv][j] = t; }
        double ip = 1.0 / a[c][c];
        for (int j = 0; j < 12; ++j) a[c][j] *= ip;
        for (int r = 0; r < 6; ++r) {
            if (r == c) continue;
            double f = a[r][c];
            for (int j = 0; j < 12; ++j) a[r][j] -= f * a[c][j];
        }
    }
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) Mi[i * 6 + j] = d[i] * a[i][6 + j] * d[j];
    return 0;
}

/* pseudo-inverse of a predicted covariance whose only null direction is the normal of the surface it was
 * transported to: the radial position direction of xp (cylinder) or the z axis (disc, reading A23) */
static int pinv_radial_null(const double Cp[36], const double xp[6], int surface, double out[36]) {
    double rho = sqrt(xp[0] * xp[0] + xp[1] * xp[1]);
    if (!(rho > 0.0)) return -1;
    double e[6] = {xp[0] / rho, xp[1] / rho, 0.0, 0.0, 0.0, 0.0};
    if (surface == 1) { e[0] = 0.0; e[1] = 0.0; e[2] = 1.0; }
    double s = fmax(fmax(Cp[0], Cp[7]), Cp[14]);
    if (!(s > 0.0)) return -1;
    double M[36];
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) M[i * 6 + j] = Cp[i * 6 + j] + s * e[i] * e[j];
    if (inv6(M, out)) return -1;
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) out[i * 6 + j] -= e[i] * e[j] / s;
    return 0;
}

/* Forward fit (fit_one) + RTS smoother.  Forward outputs as fit_one; spar[L][6] / scov[L][36] = smoothed state
 * and covariance at every used layer (zeros elsewhere); *used_out = bit mask of those layers.  A smoothing step
 * whose predicted covariance cannot be inverted stops the recursion there: the layers further in keep their
 * FILTERED state and *sstatus gets ORC_S_NOT_PD (never seen on the workloads; kept so that nothing is undefined). */
void orc_smooth_one(int L, const double *radius, const double *xX0, double Bz, double mass, const double par[6],
                    const double cov[36], int q, const double *hpos, const double *hcov, uint32_t mask,
                    double opar[6], double ocov[36], double *ochi2, int32_t *onhits, uint32_t *ostatus,
                    double *spar, double *scov, uint32_t *used_out, uint32_t *sstatus) {
    double *tr = (double *)calloc((size_t)L * ORC_TRACE_STRIDE, sizeof(double));
    fit_one(L, radius, xX0, Bz, mass, par, cov, q, hpos, hcov, mask, opar, ocov, ochi2, onhits, ostatus, tr);
    memset(spar, 0, (size_t)L * 6 * sizeof(double));
    memset(scov, 0, (size_t)L * 36 * sizeof(double));
    uint32_t used = 0;
    for (int l = 0; l < L; ++l)
        if (tr[(size_t)l * ORC_TRACE_STRIDE + 121] != 0.0) used |= 1u << l;
    *used_out = used;
    *sstatus = 0;
    int next = -1, broken = 0;
    for (int l = L - 1; l >= 0; --l) {
        if (!((used >> l) & 1u)) continue;
        const double *t = tr + (size_t)l * ORC_TRACE_STRIDE;
        const double *xf = t + 78, *Cf = t + 84;
        double *xs = spar + 6 * l, *Cs = scov + 36 * l;
        if (next < 0 || broken) { /* outermost used layer (or recursion stopped): smoothed = filtered */
            memcpy(xs, xf, 6 * sizeof(double));
            memcpy(Cs, Cf, 36 * sizeof(double));
            next = l;
            continue;
        }
        const double *tn = tr + (size_t)next * ORC_TRACE_STRIDE;
        const double *xpn = tn, *Cpn = tn + 122, *Gn = tn + 158;
        const double *xsn = spar + 6 * next, *Csn = scov + 36 * next;
        double Ni[36], CG[36], A[36], D[36], AD[36];
        if (pinv_radial_null(Cpn, xpn, g_surface_type[next], Ni)) {
            *sstatus |= ORC_S_NOT_PD;
            broken = 1;
            memcpy(xs, xf, 6 * sizeof(double));
            memcpy(Cs, Cf, 36 * sizeof(double));
            next = l;
            continue;
        }
        for (int i = 0; i < 6; ++i) /* C^+ G^T */
            for (int j = 0; j < 6; ++j) {
                double acc = 0.0;
                for (int m = 0; m < 6; ++m) acc += Cf[i * 6 + m] * Gn[j * 6 + m];
                CG[i * 6 + j] = acc;
            }
        for (int i = 0; i < 6; ++i) /* A = C^+ G^T (C^-)^+ */
            for (int j = 0; j < 6; ++j) {
                double acc = 0.0;
                for (int m = 0; m < 6; ++m) acc += CG[i * 6 + m] * Ni[m * 6 + j];
                A[i * 6 + j] = acc;
            }
        for (int i = 0; i < 6; ++i) {
            double acc = 0.0;
            for (int m = 0; m < 6; ++m) acc += A[i * 6 + m] * (xsn[m] - xpn[m]);
            xs[i] = xf[i] + acc;
        }
        for (int i = 0; i < 36; ++i) D[i] = Csn[i] - Cpn[i];
        for (int i = 0; i < 6; ++i)
            for (int j = 0; j < 6; ++j) {
                double acc = 0.0;
                for (int m = 0; m < 6; ++m) acc += A[i * 6 + m] * D[m * 6 + j];
                AD[i * 6 + j] = acc;
            }
        for (int i = 0; i < 6; ++i)
            for (int j = 0; j < 6; ++j) {
                double acc = 0.0;
                for (int m = 0; m < 6; ++m) acc += AD[i * 6 + m] * A[j * 6 + m];
                Cs[i * 6 + j] = Cf[i * 6 + j] + acc;
            }
        for (int i = 0; i < 6; ++i) /* symmetrise (the two triangles differ by rounding only) */
            for (int j = i + 1; j < 6; ++j) {
                double v = 0.5 * (Cs[i * 6 + j] + Cs[j * 6 + i]);
                Cs[i * 6 + j] = v;
                Cs[j * 6 + i] = v;
            }
        next = l;
    }
    free(tr);
}

typedef struct {
    int64_t lo, hi;
    int L;
    const double *radius, *xX0;
    double Bz, mass;
    const double *par, *cov;
    const int8_t *q;
    const double *hpos, *hcov;
    const uint32_t *mask;
    double *opar, *ocov, *ochi2;
    int32_t *onhits;
    uint32_t *ostatus;
    double *spar, *scov;
    uint32_t *used, *sstatus;
} smooth_job;

static void *smooth_range(void *p) {
    smooth_job *j = (smooth_job *)p;
    for (int64_t i = j->lo; i < j->hi; ++i)
        orc_smooth_one(j->L, j->radius, j->xX0, j->Bz, j->mass, j->par + 6 * i, j->cov + 36 * i, j->q[i],
                       j->hpos + (size_t)i * j->L * 3, j->hcov + (size_t)i * j->L * 9,
                       j->mask ? j->mask[i] : 0xffffffffu, j->opar + 6 * i, j->ocov + 36 * i, j->ochi2 + i,
                       j->onhits + i, j->ostatus + i, j->spar + (size_t)i * j->L * 6,
                       j->scov + (size_t)i * j->L * 36, j->used + i, j->sstatus + i);
    return NULL;
}

/* Batched fit + smoother.  AoS double inputs as orc_fit_tracks; spar[n][L][6], scov[n][L][36], used[n], sstatus[n]. */
int orc_smooth_tracks(int64_t n, int L, const double *radius, const double *xX0, double Bz, double mass,
                      const double *par, const double *cov, const int8_t *q, const double *hpos, const double *hcov,
                      const uint32_t *mask, double *opar, double *ocov, double *ochi2, int32_t *onhits,
                      uint32_t *ostatus, double *spar, double *scov, uint32_t *used, uint32_t *sstatus, int nthreads) {
    if (nthreads < 1) nthreads = 1;
    if (nthreads > 256) nthreads = 256;
    smooth_job jobs[256];
    pthread_t th[256];
    for (int t = 0; t < nthreads; ++t) {
        smooth_job j = {n * t / nthreads, n * (t + 1) / nthreads, L, radius, xX0, Bz, mass, par, cov, q, hpos, hcov,
                        mask, opar, ocov, ochi2, onhits, ostatus, spar, scov, used, sstatus};
        jobs[t] = j;
    }
    if (nthreads == 1) {
        smooth_range(&jobs[0]);
        return 0;
    }
    for (int t = 0; t < nthreads; ++t)
        if (pthread_create(&th[t], NULL, smooth_range, &jobs[t])) return -1;
    for (int t = 0; t < nthreads; ++t) pthread_join(th[t], NULL);
    return 0;
}

/* ---- backward refit (reading A18; round 1's stand-in for the smoother -- the smoother proper is orc_smooth_one
 * above; this inward refit counts the forward information 1 + 1/kappa times) ---------
 * Starts from the forward result (u, C) standing at the outermost used hit layer, with the covariance
 * inflated by kappa (the forward information is kept only as a weak prior), and runs the same filter
 * inward over the same hits:
 *   update with the outermost hit (no propagation: the state already stands on that layer);
 *   for every further used layer, outer to inner:  C += Q(previous layer, at the current momentum)
 *   [the scatterer just left behind], propagate inward (C' = F C F^T), update with the layer's hit.
 * Result: state and covariance at the INNERMOST used hit layer (outer side of its material), chi2 of the
 * backward pass.  A failing layer sets the status bit and is skipped as in the forward fit.
 * `used` = bit mask of the layers the forward fit used (mask bit set AND no failure there).
 * trace (optional): per layer 122 doubles as in fit_one (F = I, Q = 0 for the update-only first step;
 * Q is the noise added BEFORE the propagation of that step). */
static void refit_inward_one(int L, const double *radius, const double *xX0, double Bz, double mass, double kappa,
                             const double par[6], const double cov[36], int q, const double *hpos,
                             const double *hcov, uint32_t used, double opar[6], double ocov[36], double *ochi2,
                             int32_t *onhits, uint32_t *ostatus, double *trace) {
    double u[6], C[36];
    memcpy(u, par, sizeof u);
    for (int i = 0; i < 36; ++i) C[i] = kappa * cov[i];
    double chi2 = 0.0;
    int nh = 0, prev = -1;
    uint32_t st = 0;
    for (int l = L - 1; l >= 0; --l) {
        double *tr = trace ? trace + (size_t)l * ORC_TRACE_STRIDE : NULL;
        if (tr) memset(tr, 0, ORC_TRACE_STRIDE * sizeof(double));
        if (!((used >> l) & 1u)) continue;
        double up[6], F[36], Q[36], Cp[36], un[6], Cn[36], dchi2;
        int rc;
        if (prev < 0) { /* first step: update only */
            memcpy(up, u, sizeof up);
            memcpy(Cp, C, sizeof Cp);
            memset(Q, 0, sizeof Q);
            memset(F, 0, sizeof F);
            for (int i = 0; i < 6; ++i) F[i * 6 + i] = 1.0;
        } else {
            double Cq[36], Z[36], ub[6];
            memcpy(ub, u, sizeof ub);
            memcpy(Cq, C, sizeof Cq);
            /* A21: the layer just left gives back the energy it took (before its scattering noise is added) */
            g_at_surface = g_surface_type[prev]; /* the state stands on layer prev (a cylinder or a disc, A23) */
            int el_rc = g_energy_loss ? orc_energy_loss_step(ub, Cq, mass, xX0[prev], -1, NULL) : 0;
            if (!el_rc) orc_process_noise(ub, mass, xX0[prev], Q);
            g_at_surface = 0;
            if (el_rc) { st |= ORC_PROP_FAIL; continue; }
            for (int i = 0; i < 36; ++i) Cq[i] += Q[i];
            if (g_surface_type[l] == 1) { /* back to the disc on the track's side */
                rc = propagate_to_z_dir(ub, (double)q, Bz, ub[5] < 0.0 ? -g_disc_z[l] : g_disc_z[l], 1, up, F, NULL, NULL);
                if (!rc) {
                    double rho = sqrt(up[0] * up[0] + up[1] * up[1]);
                    if (rho < g_disc_rmin[l] || rho > g_disc_rmax[l]) rc = ORC_OUTSIDE;
                }
            } else {
                rc = propagate_dir(ub, (double)q, Bz, radius[l], 1, up, F, NULL, NULL);
                if (!rc && fabs(up[2]) > g_half_length[l]) rc = ORC_OUTSIDE;
            }
            if (rc) { st |= (uint32_t)rc; continue; }
            memset(Z, 0, sizeof Z);
            orc_transport_cov(F, Cq, Z, Cp);
        }
        rc = orc_update(up, Cp, hpos + 3 * l, hcov + 9 * l, un, Cn, &dchi2);
        if (rc) { st |= (uint32_t)rc; continue; }
        memcpy(u, un, sizeof u);
        memcpy(C, Cn, sizeof C);
        chi2 += dchi2;
        nh += 1;
        prev = l;
        if (tr) {
            memcpy(tr, up, 6 * sizeof(double));
            memcpy(tr + 6, F, 36 * sizeof(double));
            memcpy(tr + 42, Q, 36 * sizeof(double));
            memcpy(tr + 78, u, 6 * sizeof(double));
            memcpy(tr + 84, C, 36 * sizeof(double));
            tr[120] = dchi2;
            tr[121] = 1.0;
        }
    }
    memcpy(opar, u, sizeof u);
    memcpy(ocov, C, sizeof C);
    *ochi2 = chi2;
    *onhits = nh;
    *ostatus = st;
}

/* Forward fit followed by the inward refit.  Outputs: forward result (opar/ocov/ochi2/onhits/ostatus) and
 * refitted result at the innermost used layer (spar/scov/schi2).  sstatus = bits of the backward pass.
 * used_out (optional) = layers the forward fit used. */
void orc_fit_refit_one(int L, const double *radius, const double *xX0, double Bz, double mass, double kappa,
                        const double par[6], const double cov[36], int q, const double *hpos,
                        const double *hcov, uint32_t mask, double opar[6], double ocov[36], double *ochi2,
                        int32_t *onhits, uint32_t *ostatus, double spar[6], double scov[36], double *schi2,
                        uint32_t *sstatus, int32_t *snhits, double *trace_fwd, double *trace_bwd) {
    double *tf = trace_fwd, *own = NULL;
    if (!tf) { own = (double *)calloc((size_t)L * ORC_TRACE_STRIDE, sizeof(double)); tf = own; } /* zeroed: fit_one writes no trace for a bad charge */
    fit_one(L, radius, xX0, Bz, mass, par, cov, q, hpos, hcov, mask, opar, ocov, ochi2, onhits, ostatus, tf);
    uint32_t used = 0;
    for (int l = 0; l < L; ++l)
        if (tf[(size_t)l * ORC_TRACE_STRIDE + 121] != 0.0) used |= 1u << l;
    int32_t nb = 0;
    if (used == 0) { /* nothing fitted: the input comes back */
        memcpy(spar, opar, 6 * sizeof(double));
        memcpy(scov, ocov, 36 * sizeof(double));
        *schi2 = 0.0;
        *sstatus = 0;
    } else {
        refit_inward_one(L, radius, xX0, Bz, mass, kappa, opar, ocov, q, hpos, hcov, used, spar, scov, schi2, &nb,
                         sstatus, trace_bwd);
    }
    if (snhits) *snhits = nb; /* hits the backward pass used */
    if (own) free(own);
}

/* Batched (single thread): AoS double inputs as in orc_fit_tracks. */
void orc_fit_refit_tracks(int64_t n, int L, const double *radius, const double *xX0, double Bz, double mass,
                           double kappa, const double *par, const double *cov, const int8_t *q,
                           const double *hpos, const double *hcov, const uint32_t *mask, double *opar,
                           double *ocov, double *ochi2, int32_t *onhits, uint32_t *ostatus, double *spar,
                           double *scov, double *schi2, uint32_t *sstatus, int32_t *snhits, double *trace_fwd,
                           double *trace_bwd) {
    for (int64_t i = 0; i < n; ++i)
        orc_fit_refit_one(L, radius, xX0, Bz, mass, kappa, par + 6 * i, cov + 36 * i, q[i],
                           hpos + (size_t)i * L * 3, hcov + (size_t)i * L * 9, mask ? mask[i] : 0xffffffffu,
                           opar + 6 * i, ocov + 36 * i, ochi2 + i, onhits + i, ostatus + i, spar + 6 * i,
                           scov + 36 * i, schi2 + i, sstatus + i, snhits ? snhits + i : NULL,
                           trace_fwd ? trace_fwd + (size_t)i * L * ORC_TRACE_STRIDE : NULL,
                           trace_bwd ? trace_bwd + (size_t)i * L * ORC_TRACE_STRIDE : NULL);
}

typedef struct {
    int64_t lo, hi;
    int L;
    const double *radius, *xX0;
    double Bz, mass;
    const double *par, *cov;
    const int8_t *q;
    const double *hpos, *hcov;
    const uint32_t *mask;
    double *opar, *ocov, *ochi2;
    int32_t *onhits;
    uint32_t *ostatus;
    double *trace;
} fit_job;

static void *fit_range(void *p) {
    fit_job *j = (fit_job *)p;
    for (int64_t i = j->lo; i < j->hi; ++i)
        fit_one(j->L, j->radius, j->xX0, j->Bz, j->mass, j->par + 6 * i, j->cov + 36 * i, j->q[i],
                j->hpos + (size_t)i * j->L * 3, j->hcov + (size_t)i * j->L * 9,
                j->mask ? j->mask[i] : 0xffffffffu, j->opar + 6 * i, j->ocov + 36 * i, j->ochi2 + i,
                j->onhits + i, j->ostatus + i,
                j->trace ? j->trace + (size_t)i * j->L * ORC_TRACE_STRIDE : NULL);
    return NULL;
}

/* Batched fit.  AoS double inputs: par[n][6], cov[n][36], hpos[n][L][3], hcov[n][L][9].
 * nthreads >= 1: contiguous track ranges, one pthread each. */
int orc_fit_tracks(int64_t n, int L, const double *radius, const double *xX0, double Bz, double mass,
                   const double *par, const double *cov, const int8_t *q, const double *hpos,
                   const double *hcov, const uint32_t *mask, double *opar, double *ocov,
                   double *ochi2, int32_t *onhits, uint32_t *ostatus, double *trace, int nthreads) {
    if (nthreads < 1) nthreads = 1;
    if (nthreads > 256) nthreads = 256;
    fit_job jobs[256];
    pthread_t th[256];
    for (int t = 0; t < nthreads; ++t) {
        fit_job j = {n * t / nthreads, n * (t + 1) / nthreads, L, radius, xX0, Bz, mass, par, cov, q,
                     hpos, hcov, mask, opar, ocov, ochi2, onhits, ostatus, trace};
        jobs[t] = j;
    }
    if (nthreads == 1) {
        fit_range(&jobs[0]);
        return 0;
    }
    for (int t = 0; t < nthreads; ++t)
        if (pthread_create(&th[t], NULL, fit_range, &jobs[t])) return -1;
    for (int t = 0; t < nthreads; ++t) pthread_join(th[t], NULL);
    return 0;
}

/* ---- hit binning (reading A16, "directionally projective bins") ----------------
 * Definition: eta = asinh(z / r_layer), phi = atan2(y, x);
 *   i_eta = clamp(floor((eta + eta_max) / (2 eta_max / n_eta)), 0, n_eta-1)
 *   i_phi = floor((phi + pi) / (2 pi / n_phi)) mod n_phi;  bin = i_eta * n_phi + i_phi.        */
int32_t orc_bin_index_def(double x, double y, double z, double r_layer, int n_eta, int n_phi,
                          double eta_max) {
    /* reading A24: r_layer = 0 says "a disc layer": the bins stay projective, eta from the point's own rho */
    if (!(r_layer > 0.0)) r_layer = sqrt(x * x + y * y);
    double eta = asinh(z / r_layer), phi = atan2(y, x);
    int ie = (int)floor((eta + eta_max) / (2.0 * eta_max / n_eta));
    if (ie < 0) ie = 0;
    if (ie > n_eta - 1) ie = n_eta - 1;
    int ip = (int)floor((phi + ORC_PI) / (2.0 * ORC_PI / n_phi));
    ip = ((ip % n_phi) + n_phi) % n_phi;
    return ie * n_phi + ip;
}

/* The same bins decided in SINGLE precision without transcendental calls, so that a hit that
 * sits within rounding of a bin edge gets one well-defined bin (reading A16b: where
 * floating point decides an integer both sides decide in the kernel's precision):
 *   u = fl32(z / r);            i_eta = #{ j in 1..n_eta-1 : u >= fl32(sinh(-eta_max + j d_eta)) }
 *   upper half plane (y > 0, or y == 0 and x > 0):
 *       i_phi = n_phi/2 + #{ j in n_phi/2+1..n_phi-1 : fl32(cx_j * y) >= fl32(sy_j * x) }
 *   y == 0 and x <= 0: i_phi = 0 (phi = +-pi wraps to the first bin)
 *   lower half plane (y < 0): i_phi = #{ j in 1..n_phi/2-1 : fl32(cx_j * y) >= fl32(sy_j * x) }
 *   (cx_j, sy_j) = fl32(cos, sin)(-pi + j 2pi/n_phi): "the hit is at or counter-clockwise past
 *   edge j".  Compiled with -ffp-contract=off: every product is rounded to float once. */
int32_t orc_bin_index_f32(float x, float y, float z, float r_layer, int n_eta, int n_phi,
                          double eta_max) {
    if (!(r_layer > 0.0f)) { /* reading A24 (disc layer): rho = fl(sqrt(fl(fl(x x) + fl(y y)))), every step rounded once */
        volatile float xx = x * x, yy = y * y;
        volatile float s2 = xx + yy;
        r_layer = sqrtf(s2);
    }
    volatile float u = z / r_layer;
    int ie = 0;
    for (int j = 1; j < n_eta; ++j) {
        float edge = (float)sinh(-eta_max + j * (2.0 * eta_max / n_eta));
        ie += (u >= edge);
    }
    int half = n_phi / 2, ip;
    if (y > 0.0f || (y == 0.0f && x > 0.0f)) {
        ip = half;
        for (int j = half + 1; j < n_phi; ++j) {
            float cx = (float)cos(-ORC_PI + j * (2.0 * ORC_PI / n_phi));
            float sy = (float)sin(-ORC_PI + j * (2.0 * ORC_PI / n_phi));
            volatile float lhs = cx * y, rhs = sy * x;
            ip += (lhs >= rhs);
        }
    } else if (y == 0.0f) {
        ip = 0;
    } else {
        ip = 0;
        for (int j = 1; j < half; ++j) {
            float cx = (float)cos(-ORC_PI + j * (2.0 * ORC_PI / n_phi));
            float sy = (float)sin(-ORC_PI + j * (2.0 * ORC_PI / n_phi));
            volatile float lhs = cx * y, rhs = sy * x;
            ip += (lhs >= rhs);
        }
    }
    return ie * n_phi + ip;
}

/* Stable counting sort of one layer's hits by bin (single-precision decision rule).
 * bin_offset[n_bins+1], sorted_to_orig[n_hits]; bin_of[n_hits] (optional) receives each bin. */
void orc_bin_hits(int64_t n_hits, const float *x, const float *y, const float *z, float r_layer,
                  int n_eta, int n_phi, double eta_max, int32_t *bin_offset, int32_t *sorted_to_orig,
                  int32_t *bin_of) {
    int nb = n_eta * n_phi;
    int32_t *b = (int32_t *)malloc((size_t)(n_hits > 0 ? n_hits : 1) * sizeof(int32_t));
    for (int i = 0; i <= nb; ++i) bin_offset[i] = 0;
    for (int64_t h = 0; h < n_hits; ++h) {
        b[h] = orc_bin_index_f32(x[h], y[h], z[h], r_layer, n_eta, n_phi, eta_max);
        bin_offset[b[h] + 1] += 1;
    }
    for (int i = 0; i < nb; ++i) bin_offset[i + 1] += bin_offset[i];
    int32_t *cur = (int32_t *)malloc((size_t)(nb > 0 ? nb : 1) * sizeof(int32_t));
    for (int i = 0; i < nb; ++i) cur[i] = bin_offset[i];
    for (int64_t h = 0; h < n_hits; ++h) sorted_to_orig[cur[b[h]]++] = (int32_t)h;
    if (bin_of) memcpy(bin_of, b, (size_t)n_hits * sizeof(int32_t));
    free(cur);
    free(b);
}

/* ---- best-hit candidate scoring on one layer (reading A16) --------------------
 * Per candidate: propagate to r_layer (+Q); candidate bin from its own (eta, phi) by the
 * definition formula; window i_eta +- w clipped, i_phi +- w wrapped; chi2 of every hit in the
 * window; best = lowest chi2, exact ties -> lowest original index; accept iff chi2 < cut; accepted
 * and do_update: Kalman update, nhits += 1, chi2 += best.  Otherwise best_hit = -1 and the state
 * stays the propagated one.  best_chi2 = lowest chi2 seen (INFINITY if the window is empty).
 * Propagation failure: status bit, candidate untouched, best_hit = -1, best_chi2 = INFINITY.
 * all_hits != 0: ignore the bins and scan every hit of the layer (brute force, pin P8).
 * Hits: double AoS hpos[H][3], hcov[H][9] in ORIGINAL order. */
void orc_score_layer(int64_t n, double r_layer, double xX0, double Bz, double mass, double *par,
                     double *cov, const int8_t *q, double *chi2, int32_t *nhits, uint32_t *status,
                     int64_t n_hits, const double *hpos, const double *hcov, int n_eta, int n_phi,
                     double eta_max, const int32_t *bin_offset, const int32_t *sorted_to_orig,
                     int window_half, double chi2_cut, int do_update, int all_hits,
                     int32_t *best_hit, double *best_chi2, double *second_chi2) {
    for (int64_t i = 0; i < n; ++i) {
        double *u = par + 6 * i, *C = cov + 36 * i;
        best_hit[i] = -1;
        best_chi2[i] = INFINITY;
        if (second_chi2) second_chi2[i] = INFINITY;
        if (q[i] != 1 && q[i] != -1) { status[i] |= ORC_BAD_CHARGE; continue; }
        double up[6], F[36], Q[36], Cp[36];
        int rc;
        if (g_score_type == 1) { /* reading A23: the disc on the side the candidate is heading to */
            rc = orc_propagate_to_z(u, (double)q[i], Bz, u[5] < 0.0 ? -g_score_zd : g_score_zd, up, F, NULL, NULL);
            if (!rc) {
                double rho = sqrt(up[0] * up[0] + up[1] * up[1]);
                if (rho < g_score_rmin || rho > g_score_rmax) rc = ORC_OUTSIDE;
            }
        } else {
            rc = orc_propagate(u, (double)q[i], Bz, r_layer, up, F, NULL, NULL);
            if (!rc && fabs(up[2]) > g_score_half_length) rc = ORC_OUTSIDE;
        }
        if (rc) { status[i] |= (uint32_t)rc; continue; }
        g_at_surface = g_score_type;
        orc_process_noise(up, mass, xX0, Q);
        orc_transport_cov(F, C, Q, Cp);
        int el_rc = g_energy_loss ? orc_energy_loss_step(up, Cp, mass, xX0, +1, NULL) : 0; /* A21 */
        g_at_surface = 0;
        if (el_rc) { status[i] |= ORC_PROP_FAIL; continue; }
        const double r_bins = g_score_type == 1 ? 0.0 : r_layer; /* reading A24: on a disc, eta from the point's own rho */
        double best = INFINITY, second = INFINITY;
        int32_t bh = -1;
        if (all_hits) {
            for (int64_t h = 0; h < n_hits; ++h) {
                double c;
                if (orc_chi2_increment(up, Cp, hpos + 3 * h, hcov + 9 * h, &c)) continue;
                if (c < best || (c == best && (int32_t)h < bh)) { second = best; best = c; bh = (int32_t)h; }
                else if (c < second) second = c;
            }
        } else {
            int cb = orc_bin_index_def(up[0], up[1], up[2], r_bins, n_eta, n_phi, eta_max);
            int ie = cb / n_phi, ip = cb % n_phi;
            for (int de = -window_half; de <= window_half; ++de) {
                int e = ie + de;
                if (e < 0 || e >= n_eta) continue;
                for (int dp = -window_half; dp <= window_half; ++dp) {
                    int p = ((ip + dp) % n_phi + n_phi) % n_phi;
                    if (2 * window_half + 1 > n_phi && dp > -window_half + n_phi - 1) continue;
                    int bin = e * n_phi + p;
                    for (int32_t sidx = bin_offset[bin]; sidx < bin_offset[bin + 1]; ++sidx) {
                        int32_t h = sorted_to_orig[sidx];
                        double c;
                        if (orc_chi2_increment(up, Cp, hpos + 3 * (size_t)h, hcov + 9 * (size_t)h, &c)) continue;
                        if (c < best || (c == best && h < bh)) { second = best; best = c; bh = h; }
                        else if (c < second) second = c;
                    }
                }
            }
        }
        best_chi2[i] = best;
        if (second_chi2) second_chi2[i] = second;
        int accepted = 0;
        if (bh >= 0 && best < chi2_cut) {
            if (do_update) {
                double un[6], Cn[36], c;
                rc = orc_update(up, Cp, hpos + 3 * (size_t)bh, hcov + 9 * (size_t)bh, un, Cn, &c);
                if (rc) { status[i] |= (uint32_t)rc; }
                else {
                    memcpy(u, un, 6 * sizeof(double));
                    memcpy(C, Cn, 36 * sizeof(double));
                    chi2[i] += c;
                    nhits[i] += 1;
                    accepted = 1;
                }
            } else accepted = 2;
            best_hit[i] = bh;
        }
        if (accepted != 1) { /* state = propagated one (Q included) */
            memcpy(u, up, 6 * sizeof(double));
            memcpy(C, Cp, 36 * sizeof(double));
        }
    }
}

/* ---- combinatorial track building (reading A19; "branching occurs to explore all possible track
 * candidates up to some cutoff number of candidates per seed") ---------------------------------
 * Every seed keeps at most n_cand candidates.  On each layer every candidate is propagated (+Q); every hit of
 * its +-window_half bin window with chi2 < chi2_cut is compatible and spawns a child (Kalman update, nhits + 1,
 * chi2 + increment); one more child takes no hit (propagated state, nhits and chi2 unchanged).  A candidate
 * that cannot be propagated yields one child, itself unchanged (status bit).  The children of a seed are ranked
 * by (nhits descending, chi2 ascending, parent slot ascending, hit original index ascending with "no hit" last)
 * and the best n_cand survive, in that order.  After the last layer slot 0 is the seed's track.
 * Outputs per seed: best candidate (state, covariance, chi2, nhits, status, hit per layer or -1), the number of
 * surviving candidates, and `margin` = the smallest relative gap met in any decision that fp32 rounding could
 * flip: |chi2 - cut| / cut of a window hit, and |chi2_a - chi2_b| / max(chi2, 1) between children of equal
 * nhits that are adjacent in the ranking (including the first one dropped).                                    */
#define ORC_MAXC 8
typedef struct {
    double u[6], C[36], chi2;
    int nhits;
    uint32_t status;
    int32_t hits[32];
} orc_cand;

typedef struct {
    orc_cand c;          /* child state */
    int parent;
    int32_t hit;         /* original index or -1 */
} orc_child;

static int child_before(const orc_child *a, const orc_child *b) {
    if (a->c.nhits != b->c.nhits) return a->c.nhits > b->c.nhits;
    if (a->c.chi2 != b->c.chi2) return a->c.chi2 < b->c.chi2;
    if (a->parent != b->parent) return a->parent < b->parent;
    {
        int64_t ha = a->hit < 0 ? (int64_t)1 << 40 : a->hit, hb = b->hit < 0 ? (int64_t)1 << 40 : b->hit;
        return ha < hb;
    }
}

void orc_build_combinatorial(int64_t n_seeds, int n_layers_total, int first_layer, int n_build, const double *radius,
                             const double *xX0, double Bz, double mass, const double *par, const double *cov,
                             const int8_t *q, const double *chi2_in, const int32_t *nhits_in,
                             const int64_t *n_hits, const double *const *hpos, const double *const *hcov,
                             int n_eta, int n_phi, double eta_max, const int32_t *const *bin_offset,
                             const int32_t *const *sorted_to_orig, int window_half, double chi2_cut, int n_cand,
                             double *opar, double *ocov, double *ochi2, int32_t *onhits, uint32_t *ostatus,
                             int32_t *ohits /* [n_build][n_seeds] */, int32_t *oncand, double *omargin) {
    (void)n_layers_total; (void)n_hits;
    if (n_cand > ORC_MAXC) n_cand = ORC_MAXC;
    orc_cand *cur = (orc_cand *)malloc(sizeof(orc_cand) * ORC_MAXC);
    size_t cap = 1024;
    orc_child *ch = (orc_child *)malloc(sizeof(orc_child) * cap);
    for (int64_t sd = 0; sd < n_seeds; ++sd) {
        int nc = 1;
        double margin = INFINITY;
        memcpy(cur[0].u, par + 6 * sd, 6 * sizeof(double));
        memcpy(cur[0].C, cov + 36 * sd, 36 * sizeof(double));
        cur[0].chi2 = chi2_in ? chi2_in[sd] : 0.0;
        cur[0].nhits = nhits_in ? nhits_in[sd] : 0;
        cur[0].status = 0;
        for (int j = 0; j < 32; ++j) cur[0].hits[j] = -1;
        int qq = q[sd];
        if (qq != 1 && qq != -1) cur[0].status = ORC_BAD_CHARGE;
        for (int j = 0; j < n_build && !(cur[0].status & ORC_BAD_CHARGE); ++j) {
            int l = first_layer + j;
            size_t nch = 0;
            for (int p = 0; p < nc; ++p) {
                double up[6], F[36], Q[36], Cp[36];
                int rc = reach_surface(l, cur[p].u, (double)qq, Bz, radius[l], up, F); /* cylinder, or disc (A23) */
                if (!rc) {
                    g_at_surface = g_surface_type[l];
                    orc_process_noise(up, mass, xX0[l], Q);
                    orc_transport_cov(F, cur[p].C, Q, Cp);
                    if (g_energy_loss) rc = orc_energy_loss_step(up, Cp, mass, xX0[l], +1, NULL); /* A21 */
                    g_at_surface = 0;
                }
#define ORC_ROOM() do { if (nch + 2 > cap) { cap *= 2; ch = (orc_child *)realloc(ch, sizeof(orc_child) * cap); } } while (0)
                ORC_ROOM();
                if (rc) { /* cannot reach the layer: survives unchanged */
                    ch[nch].c = cur[p]; ch[nch].c.status |= (uint32_t)rc; ch[nch].parent = p; ch[nch].hit = -1; ++nch;
                    continue;
                }
                /* the "no hit" child */
                ch[nch].c = cur[p];
                memcpy(ch[nch].c.u, up, sizeof up); memcpy(ch[nch].c.C, Cp, sizeof Cp);
                ch[nch].parent = p; ch[nch].hit = -1; ++nch;
                int cb = orc_bin_index_def(up[0], up[1], up[2], g_surface_type[l] == 1 ? 0.0 : radius[l], n_eta, n_phi, eta_max); /* A24 */
                int ie = cb / n_phi, ip = cb % n_phi;
                for (int de = -window_half; de <= window_half; ++de) {
                    int e = ie + de;
                    if (e < 0 || e >= n_eta) continue;
                    for (int dp = -window_half; dp <= window_half; ++dp) {
                        int pb = ((ip + dp) % n_phi + n_phi) % n_phi, bin = e * n_phi + pb;
                        for (int32_t s = bin_offset[j][bin]; s < bin_offset[j][bin + 1]; ++s) {
                            int32_t h = sorted_to_orig[j][s];
                            double c;
                            if (orc_chi2_increment(up, Cp, hpos[j] + 3 * (size_t)h, hcov[j] + 9 * (size_t)h, &c)) continue;
                            double gap = fabs(c - chi2_cut) / chi2_cut;
                            if (gap < margin) margin = gap;
                            if (!(c < chi2_cut)) continue;
                            ORC_ROOM();
                            orc_child *k = &ch[nch];
                            k->c = cur[p];
                            double cc;
                            if (orc_update(up, Cp, hpos[j] + 3 * (size_t)h, hcov[j] + 9 * (size_t)h, k->c.u, k->c.C, &cc)) continue;
                            k->c.chi2 = cur[p].chi2 + cc;
                            k->c.nhits = cur[p].nhits + 1;
                            k->c.hits[j] = h;
                            k->parent = p; k->hit = h; ++nch;
                        }
                    }
                }
            }
            /* rank: selection sort of the best n_cand + 1 (the extra one only feeds the margin) */
            int keep = (int)(nch < (size_t)n_cand ? nch : (size_t)n_cand);
            for (int a = 0; a < keep + 1 && (size_t)a < nch; ++a) {
                size_t best = (size_t)a;
                for (size_t b = (size_t)a + 1; b < nch; ++b)
                    if (child_before(&ch[b], &ch[best])) best = b;
                if (best != (size_t)a) { orc_child t = ch[a]; ch[a] = ch[best]; ch[best] = t; }
                if (a > 0 && ch[a].c.nhits == ch[a - 1].c.nhits) {
                    double sc = fmax(fmax(ch[a].c.chi2, ch[a - 1].c.chi2), 1.0);
                    double gap = fabs(ch[a].c.chi2 - ch[a - 1].c.chi2) / sc;
                    if (gap < margin) margin = gap;
                }
            }
            for (int a = 0; a < keep; ++a) cur[a] = ch[a].c;
            nc = keep;
        }
        memcpy(opar + 6 * sd, cur[0].u, 6 * sizeof(double));
        memcpy(ocov + 36 * sd, cur[0].C, 36 * sizeof(double));
        ochi2[sd] = cur[0].chi2; onhits[sd] = cur[0].nhits; ostatus[sd] = cur[0].status;
        for (int j = 0; j < n_build; ++j) ohits[(size_t)j * n_seeds + sd] = cur[0].hits[j];
        oncand[sd] = nc;
        omargin[sd] = margin;
    }
    free(ch);
    free(cur);
}
