// kf_math.cuh -- per-track Kalman-filter arithmetic shared by the fit and scoring kernels.
//
// Everything here is fp32 and register-resident: one call = one track on one layer.
// What is computed is north_star's filter (C' = F C F^T + Q, S = C'_pp + V, K = C' H^T S^-1,
// x = x' + K r, C = C' - K H C', chi2 += r^T S^-1 r) with the helix / Jacobian /
// Highland readings A1..A8 of DESIGN.md.  HOW it is computed differs from the textbook 6x6 form
// (DESIGN.md "Kernel arithmetic"):
//
//  * The covariance lives in a track-local frame: position block in (radial, tangential, z) of
//    the current layer crossing, momentum block in (b1, b2, c) = (d pT, pT d phi, pT d(pz/pT)):
//    b1 along pT, b2 the in-plane normal, c = d pz - (pz/pT) b1 the dip-slope coordinate.  These
//    are two rotations about z plus one shear, i.e. a similarity C~ = J C J^T: algebraically the
//    same filter, but the nearly rank-1 momentum block (|p| loose, direction tight) has its loose
//    direction on ONE axis (b1) and no longer cancels in fp32.
//  * In that frame the to-radius Jacobian is  F~ = I + (few rank-1 terms):
//        row r' = 0                           (arrival point stays on the cylinder)
//        row t' = G_t - tan(a') G_r
//        row z' = e_z + (theta/k) e_c + (pz/pT)(theta/k e_b1 - G_r/cos(a'))
//        row b1'= e_b1                        (|pT| is conserved)
//        row b2'= e_b2 + k/cos(a') G_r
//        row c' = e_c                         (pz/pT is conserved)
//    with G_r, G_t the fixed-turning-angle displacement of the arrival point expressed along
//    (radial', tangential') and a' the angle between momentum and radius at arrival.  So the
//    transport needs three matrix-vector products instead of two 6x6 matrix products, and the
//    propagated covariance has an exactly zero radial row/column (15 live elements).
//  * The update uses the "V form": position rows of the new C are K V (no subtraction), the
//    momentum block is C'_mm - K_m C'_pm.
//
// Complex shorthand used in comments: w = x + i y, pi = px + i py, E = exp(-i theta).
// Helix (reading A2): w' = w + (i pi / k)(E - 1), pi' = pi E, z' = z + pz theta / k.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "kf_pair.cuh"

namespace kf {

constexpr float kCB = 2.99792458e-3f;  // GeV / (c T cm), reading A1

enum : int { MODEL_PATH_LENGTH = 1, MODEL_ENERGY_LOSS = 2 };
enum : uint32_t { ST_PROP_FAIL = 1u, ST_S_NOT_PD = 2u, ST_NONFINITE = 4u, ST_BAD_CHARGE = 8u, ST_OUTSIDE = 16u, ST_SMOOTH_FAIL = 32u };

// Per-layer constants, computed once on the host in double and rounded to float.
struct LayerConst {
    float r;      // radius
    float r2;     // r^2
    float inv_r;  // 1 / r
    float ms;     // Highland: 0.0136^2 t (1 + 0.038 ln t)^2, t = x/X0 (0 if t <= 0)
    // reading A20 (geometry options)
    float half_len;  // barrel half length (+inf: unbounded)
    float ms0;       // 0.0136^2 t          (0 if t <= 0)
    float ln_t;      // ln t                (0 if t <= 0)
    // reading A21 (energy loss)
    float de0;       // K (Z/A) t X0 for silicon [GeV]: Bethe prefactor of the layer (0 if t <= 0 or option off)
    // reading A23 (endcap discs)
    int type;        // 0: barrel cylinder of radius r; 1: pair of discs in the planes z = +-zd
    float zd;        // |z| of the disc pair
    float rmin2, rmax2;  // squared bounds of the sensitive annulus
};

// Reading A21: particle-dependent constants of Bethe's formula, computed on the host in double.
struct Bethe {
    float mass;  // M
    float a;     // ln(2 me / (I M^2)):   ln(2 me (beta gamma)^2 / I) = a + ln p^2
    float b;     // 2 me / M^2:           1 + 2 gamma me/M + (me/M)^2 = c + b E
    float c;     // 1 + (me/M)^2
};

struct FitParams {
    int n_layers;
    float k0;      // c_B * Bz           (k = q k0)
    float inv_k0;  // 1 / (c_B * Bz)
    float mass2;   // mass^2
    int model;           // MODEL_* flags: reading A20 path-length material, reading A21 energy loss
    int geometry_options;  // 1 if model != 0, any layer has a finite half length, or there is a disc
    int has_discs;         // 1 if any layer is a disc pair (reading A23)
    Bethe el;            // reading A21 constants (zero unless MODEL_ENERGY_LOSS)
    LayerConst layer[32];
};

// MUFU-based reciprocal / reciprocal square root (about 1 ulp / 2 ulp), no slow path.
#if defined(__CUDA_ARCH__)
__device__ __forceinline__ float rcp_fast(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt_fast(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
#else
__device__ __forceinline__ float rcp_fast(float x) { return 1.0f / x; }
__device__ __forceinline__ float rsqrt_fast(float x) { return rsqrtf(x); }
#endif

__device__ __forceinline__ f2 rcp_fast(f2 x) { return f2(rcp_fast(x.v.x), rcp_fast(x.v.y)); }
__device__ __forceinline__ f2 rsqrt_fast(f2 x) { return f2(rsqrt_fast(x.v.x), rsqrt_fast(x.v.y)); }

// Reading A20, Highland factor of one crossing: `model` 0 is the flat L.ms; model 1 scales the thickness
// by the path length through the layer, t_eff = t f with f = 1/cos(psi) = p / (pT cos a'), where cos a' =
// e_r . e_l is the in-plane cosine between the radial direction and the transverse momentum:
//     ms_eff = 0.0136^2 t f (1 + 0.038 (ln t + ln f))^2.
template <class F>
__device__ __forceinline__ F layer_ms(const LayerConst& L, int model, F cos_a, F p2, F ipt) {
    if ((model & MODEL_PATH_LENGTH) == 0) return F(L.ms);
    const F f = sqrt_(p2) * ipt * rcp_fast(abs_(cos_a));
    const F lg = 1.0f + 0.038f * (L.ln_t + log_fast(f));
    return L.ms0 * f * lg * lg;
}

// Track in registers.  Position frame unit vector (eax, eay): position-block coordinates
// (a1, a2) mean  dw = (eax + i eay)(a1 + i a2).  The momentum frame always follows the current
// momentum: d(pi) = (px + i py)/pT (b1 + i b2), d pz = c + (pz/pT) b1.
// cXY = packed upper triangle over (a1, a2, z, b1, b2, c).
template <class F>
struct TrackT {
    F x, y, z, px, py, pz;
    F eax, eay;
    F c00, c01, c02, c03, c04, c05;
    F c11, c12, c13, c14, c15;
    F c22, c23, c24, c25;
    F c33, c34, c35;
    F c44, c45;
    F c55;
};
using Track = TrackT<float>;    // one track per thread
using Track2 = TrackT<f2>;      // two tracks per thread, packed (kf_pair.cuh)

// Change the momentum frame of the covariance: rotate (b1, b2) -> (dc + i ds)(b1 + i b2), then
// shear c -> c + k1 b1 + k2 b2 (new b's), k1 = T_old dc - T_new, k2 = T_old ds, T = pz/pT.
template <bool RADIAL_NULL = false, class F>
__device__ __forceinline__ void reaim_momentum(TrackT<F>& t, arg<F> dc, arg<F> ds, arg<F> T_old,
                                               arg<F> T_new) {
    F a, b;
    if constexpr (!RADIAL_NULL) { a = t.c03; b = t.c04; t.c03 = dc * a - ds * b; t.c04 = ds * a + dc * b; }
    a = t.c13; b = t.c14; t.c13 = dc * a - ds * b; t.c14 = ds * a + dc * b;
    a = t.c23; b = t.c24; t.c23 = dc * a - ds * b; t.c24 = ds * a + dc * b;
    a = t.c35; b = t.c45;
    const F c35 = dc * a - ds * b, c45 = ds * a + dc * b;
    const F cc = dc * dc, ss = ds * ds, cs = dc * ds;
    const F ll = t.c33, ln = t.c34, nn = t.c44;
    t.c33 = cc * ll - 2.0f * cs * ln + ss * nn;
    t.c44 = ss * ll + 2.0f * cs * ln + cc * nn;
    t.c34 = cs * (ll - nn) + (cc - ss) * ln;
    const F k1 = T_old * dc - T_new, k2 = T_old * ds;
    if constexpr (!RADIAL_NULL) t.c05 = fma_(k2, t.c04, fma_(k1, t.c03, t.c05));
    t.c15 = fma_(k2, t.c14, fma_(k1, t.c13, t.c15));
    t.c25 = fma_(k2, t.c24, fma_(k1, t.c23, t.c25));
    const F n35 = c35 + k1 * t.c33 + k2 * t.c34;
    const F n45 = c45 + k1 * t.c34 + k2 * t.c44;
    t.c55 += k1 * (c35 + n35) + k2 * (c45 + n45);
    t.c35 = n35;
    t.c45 = n45;
}

// Rotate the position-block coordinates (a1, a2) -> (dc + i ds)(a1 + i a2).
template <class F>
__device__ __forceinline__ void reframe_position(TrackT<F>& t, arg<F> dc, arg<F> ds) {
    F a, b;
    a = t.c02; b = t.c12; t.c02 = dc * a - ds * b; t.c12 = ds * a + dc * b;
    a = t.c03; b = t.c13; t.c03 = dc * a - ds * b; t.c13 = ds * a + dc * b;
    a = t.c04; b = t.c14; t.c04 = dc * a - ds * b; t.c14 = ds * a + dc * b;
    a = t.c05; b = t.c15; t.c05 = dc * a - ds * b; t.c15 = ds * a + dc * b;
    const F cc = dc * dc, ss = ds * ds, cs = dc * ds;
    const F ll = t.c00, ln = t.c01, nn = t.c11;
    t.c00 = cc * ll - 2.0f * cs * ln + ss * nn;
    t.c11 = ss * ll + 2.0f * cs * ln + cc * nn;
    t.c01 = cs * (ll - nn) + (cc - ss) * ln;
}

// Global-frame covariance (as stored) -> local frame.  Position frame stays global (ea = 1);
// the momentum block goes to (b1, b2, c).
template <class F>
__device__ __forceinline__ void enter_local_frame(TrackT<F>& t) {
    t.eax = 1.0f;
    t.eay = 0.0f;
    const F pt2 = t.px * t.px + t.py * t.py;
    if (none_of(pt2 > 0.0f)) return;     // (a pair goes on if either track has pT > 0; the other never starts)
    const F ipt = rsqrt_ieee(pt2);
    // b = conj(e_l) * d(pi): rotation by -phi_p;  c = d pz - (pz/pT) b1
    reaim_momentum(t, t.px * ipt, -t.py * ipt, 0.0f, t.pz * ipt);
}

// The same entry in DOUBLE, for tracks that come out of a fit (candidates of the builders, the per-layer scoring
// call): their Cartesian momentum block is nearly singular -- |p| loose, direction tight, eigenvalue ratio 1e4 to
// 1e5 after three hits -- and the rotation + shear to (b1, b2, c) cancels that many digits: 2.5e4 x 6e-8 = 1.5e-3
// in fp32, the whole covariance tolerance (measured on configs[4]: worst candidate 1.35 x the tolerance, 3 of
// 20 000 above it; with this entry ... see DESIGN.md).  Done once per candidate, about 120 double operations.
__device__ __forceinline__ void enter_local_frame_precise(Track& t) {
    t.eax = 1.0f;
    t.eay = 0.0f;
    const double px = t.px, py = t.py, pz = t.pz;
    const double pt2 = px * px + py * py;
    if (!(pt2 > 0.0)) return;
    const double ipt = 1.0 / sqrt(pt2);
    const double dc = px * ipt, ds = -py * ipt, k1 = -pz * ipt;   // T_old = 0, T_new = pz/pT: k1 = -T_new, k2 = 0
    double a, b;
    double c03 = t.c03, c04 = t.c04, c13 = t.c13, c14 = t.c14, c23 = t.c23, c24 = t.c24;
    a = c03; b = c04; c03 = dc * a - ds * b; c04 = ds * a + dc * b;
    a = c13; b = c14; c13 = dc * a - ds * b; c14 = ds * a + dc * b;
    a = c23; b = c24; c23 = dc * a - ds * b; c24 = ds * a + dc * b;
    a = t.c35; b = t.c45;
    const double c35 = dc * a - ds * b, c45 = ds * a + dc * b;
    const double cc = dc * dc, ss = ds * ds, cs = dc * ds;
    const double ll = t.c33, ln = t.c34, nn = t.c44;
    const double c33 = cc * ll - 2.0 * cs * ln + ss * nn;
    const double c44 = ss * ll + 2.0 * cs * ln + cc * nn;
    const double c34 = cs * (ll - nn) + (cc - ss) * ln;
    const double n35 = c35 + k1 * c33;
    const double n45 = c45 + k1 * c34;
    t.c05 = (float)((double)t.c05 + k1 * c03);
    t.c15 = (float)((double)t.c15 + k1 * c13);
    t.c25 = (float)((double)t.c25 + k1 * c23);
    t.c55 = (float)((double)t.c55 + k1 * (c35 + n35));
    t.c03 = (float)c03; t.c04 = (float)c04; t.c13 = (float)c13; t.c14 = (float)c14; t.c23 = (float)c23; t.c24 = (float)c24;
    t.c33 = (float)c33; t.c34 = (float)c34; t.c44 = (float)c44; t.c35 = (float)n35; t.c45 = (float)n45;
}

// Local frame -> global frame (inverse of the above for the current frames).
template <class F>
__device__ __forceinline__ void leave_local_frame(TrackT<F>& t) {
    reframe_position(t, t.eax, t.eay);
    const F pt2 = t.px * t.px + t.py * t.py;
    if (!none_of(pt2 > 0.0f)) {
        const F ipt = rsqrt_ieee(pt2);
        reaim_momentum(t, t.px * ipt, t.py * ipt, t.pz * ipt, 0.0f);
    }
    t.eax = 1.0f;
    t.eay = 0.0f;
}

// Result of the helix crossing + local-frame Jacobian ingredients.
template <class F>
struct CrossingT {
    F xn, yn, zn, pxn, pyn;  // arrival state (pz unchanged)
    F erx, ery;              // e_r' = w'/r
    F elx, ely;              // e_l' = pi'/pT
    F g0, g1, g3, g4;        // G_r over (a1, a2, b1, b2)
    F t0, t1, t3, t4;        // row t' = G_t - tan(a') G_r
    F z0, z1, z3, z4;        // row z' over (a1, a2, b1, b2); its z entry is 1, its c entry thk
    F thk;                   // theta / k = s / pT
    F mu;                    // k / cos(a')
    F T;                     // pz / pT (conserved along the helix)
    F pt2, ipt;
};
using Crossing = CrossingT<float>;
using Crossing2 = CrossingT<f2>;

// Reading A3: first outward crossing of the helix with the cylinder of radius L.r, half-angle
// form  t = tan(theta/2) = D / (a + sqrt(a^2 - D (2b + D))).  Returns false on PROP_FAIL.
// INWARD (reading A18): the same helix followed backward in path length to a smaller radius
// (D < 0, t < 0, theta < 0); the local-frame Jacobian below holds for either sign of theta.
template <bool INWARD = false, class F>
__device__ __forceinline__ typename num_traits<F>::mask helix_to_radius(const TrackT<F>& t, arg<F> k, arg<F> ik,
                                                                        const LayerConst& L, CrossingT<F>& o) {
    const F x = t.x, y = t.y, px = t.px, py = t.py;
    const F pt2 = px * px + py * py;
    const F rho2 = x * x + y * y;
    const F a = x * px + y * py;
    const F b = (y * px - x * py) - pt2 * ik;
    const F D = 0.5f * k * (L.r2 - rho2);
    const F disc = a * a - D * (2.0f * b + D);
    const F den = a + disc * rsqrt_fast(disc);  // NaN unless disc > 0
    // one test for the three PROP_FAIL conditions (r <= rho, disc <= 0, den <= 0; NaNs fail too)
    // (a pair stops here if either track fails; the caller then takes the two one at a time)
    const typename num_traits<F>::mask ok = (INWARD ? L.r2 < rho2 : L.r2 > rho2) & (disc > 0.0f) & (den > 0.0f);
    if (!all_of(ok)) return ok;
    const F tt = D * rcp_fast(den);
    const F i1 = rcp_fast(1.0f + tt * tt);
    const F S = 2.0f * tt * i1;
    const F Cm = tt * S;
    const F co = 1.0f - Cm;
    const F theta = 2.0f * atan_(tt);
    o.thk = theta * ik;
    o.xn = x + (px * S + py * Cm) * ik;
    o.yn = y + (py * S - px * Cm) * ik;
    o.zn = t.z + t.pz * o.thk;
    o.pxn = px * co + py * S;
    o.pyn = py * co - px * S;
    const F ipt = rsqrt_fast(pt2);
    o.pt2 = pt2;
    o.ipt = ipt;
    o.erx = o.xn * L.inv_r;
    o.ery = o.yn * L.inv_r;
    o.elx = o.pxn * ipt;
    o.ely = o.pyn * ipt;
    // exp(i a') = conj(e_r') e_l'
    const F ca = o.erx * o.elx + o.ery * o.ely;
    const F sa = o.erx * o.ely - o.ery * o.elx;
    const F ic = rcp_fast(ca);
    const F T = sa * ic;
    // P = conj(e_r') e_a
    const F pc = o.erx * t.eax + o.ery * t.eay;
    const F ps = o.erx * t.eay - o.ery * t.eax;
    // N = ((S + i Cm)/k) exp(i a')
    const F nr = (S * ca - Cm * sa) * ik;
    const F nt = (S * sa + Cm * ca) * ik;
    o.g0 = pc;  o.g1 = -ps; o.g3 = nr; o.g4 = -nt;
    o.t0 = ps - T * pc;
    o.t1 = pc + T * ps;
    o.t3 = nt - T * nr;
    o.t4 = nr + T * nt;
    const F T_ = t.pz * ipt;
    const F lam = T_ * ic;
    o.T = T_;
    o.z0 = -lam * pc;
    o.z1 = lam * ps;
    o.z3 = T_ * (o.thk - ic * nr);  // small: the |p|-at-fixed-direction mode does not move z'
    o.z4 = lam * nt;
    o.mu = k * ic;
    return ok;
}

// helix_to_radius plus the acceptance of reading A20: 0, ST_PROP_FAIL, or ST_OUTSIDE when the crossing
// lies beyond the end of the barrel (|z'| > half length; the layer is then skipped like a failed one).
// BOUNDED = false compiles the acceptance test out (kernels specialised for the unbounded toy detector).
// Pair form: per-component status; if either is non-zero the caller takes the two tracks one at a time.
template <bool INWARD = false, bool BOUNDED = true, class F>
__device__ __forceinline__ typename num_traits<F>::status reach_layer(const TrackT<F>& t, arg<F> k, arg<F> ik,
                                                                      const LayerConst& L, CrossingT<F>& o) {
    const typename num_traits<F>::mask ok = helix_to_radius<INWARD>(t, k, ik, L, o);
    if (!all_of(ok)) return select_u(ok, 0u, ST_PROP_FAIL);
    if constexpr (BOUNDED) return select_u(abs_(o.zn) > L.half_len, ST_OUTSIDE, 0u);
    else return select_u(ok, 0u, 0u);
}

// Highland factor at an arrival (forward filter) / at the state standing on a layer (backward refit).
template <class F>
__device__ __forceinline__ F ms_at_crossing(const LayerConst& L, int model, const CrossingT<F>& o, arg<F> pz) {
    if ((model & MODEL_PATH_LENGTH) == 0) return F(L.ms);
    return layer_ms<F>(L, model, o.erx * o.elx + o.ery * o.ely, o.pt2 + pz * pz, o.ipt);
}

// Propagated covariance in the arrival frame (radial row is exactly zero and not stored).
template <class F>
struct PropCovT {
    F n11, n12, n13, n14, n15;
    F n22, n23, n24, n25;
    F n33, n34, n35;
    F n44, n45;
    F n55;
};
using PropCov = PropCovT<float>;
using PropCov2 = PropCovT<f2>;

// C' = F~ C F~^T + Q~ (reading A4 Jacobian, A5 process noise at the propagated momentum).
// RADIAL_NULL: the input covariance already has a zero a1 row (every layer after the first).
template <bool RADIAL_NULL, class F>
__device__ __forceinline__ void transport_cov(const TrackT<F>& t, const CrossingT<F>& o, arg<F> ms,
                                              float mass2, PropCovT<F>& n) {
    const F g0 = o.g0, g1 = o.g1, g3 = o.g3, g4 = o.g4;
    const F t0 = o.t0, t1 = o.t1, t3 = o.t3, t4 = o.t4;
    const F z0 = o.z0, z1 = o.z1, z3 = o.z3, z4 = o.z4, thk = o.thk, mu = o.mu;
    // v = C g, w = C tau, u = C zeta   (rows 1..5; row 0 and the a1 column only before the first layer)
    F v1 = t.c11 * g1 + t.c13 * g3 + t.c14 * g4;
    F v3 = t.c13 * g1 + t.c33 * g3 + t.c34 * g4;
    F v4 = t.c14 * g1 + t.c34 * g3 + t.c44 * g4;
    F v5 = t.c15 * g1 + t.c35 * g3 + t.c45 * g4;
    F w1 = t.c11 * t1 + t.c13 * t3 + t.c14 * t4;
    F w3 = t.c13 * t1 + t.c33 * t3 + t.c34 * t4;
    F w4 = t.c14 * t1 + t.c34 * t3 + t.c44 * t4;
    F w5 = t.c15 * t1 + t.c35 * t3 + t.c45 * t4;
    F u1 = t.c12 + t.c11 * z1 + t.c13 * z3 + t.c14 * z4 + t.c15 * thk;
    F u2 = t.c22 + t.c12 * z1 + t.c23 * z3 + t.c24 * z4 + t.c25 * thk;
    F u3 = t.c23 + t.c13 * z1 + t.c33 * z3 + t.c34 * z4 + t.c35 * thk;
    F u4 = t.c24 + t.c14 * z1 + t.c34 * z3 + t.c44 * z4 + t.c45 * thk;
    F u5 = t.c25 + t.c15 * z1 + t.c35 * z3 + t.c45 * z4 + t.c55 * thk;
    F gCg = g1 * v1 + g3 * v3 + g4 * v4;
    F tCg = t1 * v1 + t3 * v3 + t4 * v4;
    F zCg = g1 * u1 + g3 * u3 + g4 * u4;
    F n11 = t1 * w1 + t3 * w3 + t4 * w4;
    F n12 = t1 * u1 + t3 * u3 + t4 * u4;
    F n22 = u2 + z1 * u1 + z3 * u3 + z4 * u4 + thk * u5;
    if constexpr (!RADIAL_NULL) {
        const F v0 = t.c00 * g0 + t.c01 * g1 + t.c03 * g3 + t.c04 * g4;
        const F w0 = t.c00 * t0 + t.c01 * t1 + t.c03 * t3 + t.c04 * t4;
        const F u0 = t.c02 + t.c00 * z0 + t.c01 * z1 + t.c03 * z3 + t.c04 * z4 + t.c05 * thk;
        // a1-column contributions to rows 1..5 (added before the dot products use them)
        const F dv1 = t.c01 * g0, dv3 = t.c03 * g0, dv4 = t.c04 * g0, dv5 = t.c05 * g0;
        const F dw1 = t.c01 * t0, dw3 = t.c03 * t0, dw4 = t.c04 * t0, dw5 = t.c05 * t0;
        const F du1 = t.c01 * z0, du2 = t.c02 * z0, du3 = t.c03 * z0, du4 = t.c04 * z0, du5 = t.c05 * z0;
        gCg += g0 * v0 + g1 * dv1 + g3 * dv3 + g4 * dv4;
        tCg += t0 * v0 + t1 * dv1 + t3 * dv3 + t4 * dv4;
        zCg += g0 * u0 + g1 * du1 + g3 * du3 + g4 * du4;
        n11 += t0 * w0 + t1 * dw1 + t3 * dw3 + t4 * dw4;
        n12 += t0 * u0 + t1 * du1 + t3 * du3 + t4 * du4;
        n22 += z0 * u0 + z1 * du1 + du2 + z3 * du3 + z4 * du4 + thk * du5;
        v1 += dv1; v3 += dv3; v4 += dv4; v5 += dv5;
        w1 += dw1; w3 += dw3; w4 += dw4; w5 += dw5;
        u1 += du1; u2 += du2; u3 += du3; u4 += du4; u5 += du5;
    }
    n.n11 = n11;
    n.n12 = n12;
    n.n13 = w3;
    n.n14 = w4 + mu * tCg;
    n.n15 = w5;
    n.n22 = n22;
    n.n23 = u3;
    n.n24 = u4 + mu * zCg;
    n.n25 = u5;
    // Highland (A5): theta0^2 = ms (p^2 + m^2) / p^4;  Q = theta0^2 (p^2 I - p p^T), p = (pT, 0, pz),
    // sheared to (b1, b2, c):  Q~ = theta0^2 [[pz^2, 0, -pz p^2/pT], [0, p^2, 0], [., 0, p^4/pT^2]]
    const F pz = t.pz;
    const F p2 = o.pt2 + pz * pz;
    const F ip2 = rcp_fast(p2);
    const F th2 = ms * (p2 + mass2) * ip2 * ip2;
    const F qc = th2 * p2 * o.ipt;  // theta0^2 p^2 / pT
    n.n33 = t.c33 + th2 * pz * pz;
    n.n34 = t.c34 + mu * v3;
    n.n35 = t.c35 - qc * pz;
    n.n44 = t.c44 + mu * (2.0f * v4 + mu * gCg) + th2 * p2;
    n.n45 = t.c45 + mu * v5;
    n.n55 = t.c55 + qc * (p2 * o.ipt);
}

// Reading A18, backward refit: the scatterer just left behind adds its Highland noise to the momentum
// block BEFORE the inward propagation (same Q~ as in transport_cov, at the current momentum).
template <class F>
__device__ __forceinline__ void add_process_noise(TrackT<F>& t, const LayerConst& L, int model, float mass2) {
    const F pt2 = t.px * t.px + t.py * t.py, pz = t.pz;
    const F ipt = rsqrt_fast(pt2);
    const F p2 = pt2 + pz * pz;
    const F ms = (model & MODEL_PATH_LENGTH) == 0 ? F(L.ms) : layer_ms<F>(L, model, (t.eax * t.px + t.eay * t.py) * ipt, p2, ipt);
    const F ip2 = rcp_fast(p2);
    const F th2 = ms * (p2 + mass2) * ip2 * ip2;
    const F qc = th2 * p2 * ipt;
    t.c33 += th2 * pz * pz;
    t.c35 -= qc * pz;
    t.c44 += th2 * p2;
    t.c55 += qc * (p2 * ipt);
}

// ---- reading A21: mean energy loss in the layer ---------------------------------------------------------
// The momentum keeps its direction and shrinks (forward filter) or grows back (backward refit) by
//   f = p''/p,  p''^2 = p^2 -+ dE (2E -+ dE),  dE = L.de0 [path factor] / beta^2 *
//                       (ln(2 me (beta gamma)^2 / I) - ln(1 + 2 gamma me/M + (me/M)^2)/2 - beta^2).
// Direction-preserving scaling leaves the frames where they are; in (b1, b2, c) its Jacobian (dE held fixed) is
//   J = [[g, 0, h], [0, f, 0], [0, 0, f]],  g = (E''/p'')(p/E),  h = (g - f) pT pz / p^2
// (b1 = d pT carries all of d|p| at fixed direction; b2 and c are direction changes times pT, which scales).
struct Eloss {
    float f, g, h;
};

// cos_a: in-plane cosine between the radial direction and the transverse momentum (path-length option only).
__device__ __forceinline__ bool energy_loss_factors(const Bethe& el, const LayerConst& L, int model, float mass2,
                                                    float cos_a, float pt2, float ipt, float pz, bool regain,
                                                    Eloss& e) {
    const float p2 = pt2 + pz * pz;
    const float ip = rsqrt_fast(p2);
    const float E2 = p2 + mass2;
    const float iE = rsqrt_fast(E2);
    const float E = E2 * iE;
    float thick = L.de0;
    if (model & MODEL_PATH_LENGTH) thick *= p2 * ip * ipt * rcp_fast(fabsf(cos_a));
    const float bracket = el.a + __logf(p2) - 0.5f * __logf(fmaf(el.b, E, el.c)) - p2 * iE * iE;
    const float dE = thick * (E2 * ip * ip) * bracket;
    const float En = regain ? E + dE : E - dE;
    if (!(En > el.mass)) return false;  // the particle would stop (NaNs fail too)
    const float pn2 = regain ? fmaf(dE, 2.0f * E + dE, p2) : fmaf(-dE, 2.0f * E - dE, p2);
    const float ipn = rsqrt_fast(pn2);
    e.f = pn2 * ipn * ip;
    e.g = En * ipn * (p2 * ip) * iE;
    e.h = (e.g - e.f) * (pt2 * ipt) * pz * (ip * ip);
    return true;
}

// Forward filter: applied to the propagated state and covariance (after C' = F C F^T + Q, before the update).
__device__ __forceinline__ void apply_energy_loss(const Eloss& e, CrossingT<float>& o, PropCovT<float>& n, float& pz) {
    const float f = e.f, g = e.g, h = e.h, ff = f * f;
    o.pxn *= f; o.pyn *= f; pz *= f;
    o.pt2 *= ff;
    o.ipt *= rcp_fast(f);
    n.n13 = g * n.n13 + h * n.n15;
    n.n23 = g * n.n23 + h * n.n25;
    n.n33 = g * (g * n.n33 + 2.0f * h * n.n35) + h * h * n.n55;
    n.n34 = f * (g * n.n34 + h * n.n45);
    n.n35 = f * (g * n.n35 + h * n.n55);
    n.n14 *= f; n.n24 *= f; n.n15 *= f; n.n25 *= f;
    n.n44 *= ff; n.n45 *= ff; n.n55 *= ff;
}

// Backward refit: applied to the track standing on the layer it is about to leave.
__device__ __forceinline__ void apply_energy_loss(const Eloss& e, TrackT<float>& t) {
    const float f = e.f, g = e.g, h = e.h, ff = f * f;
    t.px *= f; t.py *= f; t.pz *= f;
    t.c03 = g * t.c03 + h * t.c05;
    t.c13 = g * t.c13 + h * t.c15;
    t.c23 = g * t.c23 + h * t.c25;
    t.c33 = g * (g * t.c33 + 2.0f * h * t.c35) + h * h * t.c55;
    t.c34 = f * (g * t.c34 + h * t.c45);
    t.c35 = f * (g * t.c35 + h * t.c55);
    t.c04 *= f; t.c14 *= f; t.c24 *= f; t.c05 *= f; t.c15 *= f; t.c25 *= f;
    t.c44 *= ff; t.c45 *= ff; t.c55 *= ff;
}

// The track as it stands, dressed as a "crossing" with zero path length, so that kalman_update can be
// applied without a propagation (first step of the backward refit: the state already stands on the
// layer; its covariance is radially null in the frame (eax, eay) it carries).
template <class F>
__device__ __forceinline__ void crossing_in_place(const TrackT<F>& t, CrossingT<F>& o, PropCovT<F>& n) {
    const F pt2 = t.px * t.px + t.py * t.py;
    const F ipt = rsqrt_fast(pt2);
    o.xn = t.x; o.yn = t.y; o.zn = t.z; o.pxn = t.px; o.pyn = t.py;
    o.erx = t.eax; o.ery = t.eay; o.elx = t.px * ipt; o.ely = t.py * ipt;
    o.T = t.pz * ipt; o.pt2 = pt2; o.ipt = ipt;
    n.n11 = t.c11; n.n12 = t.c12; n.n13 = t.c13; n.n14 = t.c14; n.n15 = t.c15;
    n.n22 = t.c22; n.n23 = t.c23; n.n24 = t.c24; n.n25 = t.c25;
    n.n33 = t.c33; n.n34 = t.c34; n.n35 = t.c35; n.n44 = t.c44; n.n45 = t.c45; n.n55 = t.c55;
}

template <class F>
__device__ __forceinline__ void scale_cov(TrackT<F>& t, float f) {
    t.c11 *= f; t.c12 *= f; t.c13 *= f; t.c14 *= f; t.c15 *= f;
    t.c22 *= f; t.c23 *= f; t.c24 *= f; t.c25 *= f;
    t.c33 *= f; t.c34 *= f; t.c35 *= f; t.c44 *= f; t.c45 *= f; t.c55 *= f;
}

// Hit in the arrival frame: residual (r, t, z) and rotated covariance.
template <class F>
struct LocalHitT {
    F rr, rt, rz;
    F vrr, vrt, vrz, vtt, vtz, vzz;
};
using LocalHit = LocalHitT<float>;
using LocalHit2 = LocalHitT<f2>;

template <class F>
__device__ __forceinline__ void hit_to_local(const CrossingT<F>& o, arg<F> mx, arg<F> my, arg<F> mz,
                                             arg<F> vxx, arg<F> vxy, arg<F> vxz, arg<F> vyy, arg<F> vyz,
                                             arg<F> vzz, LocalHitT<F>& h) {
    const F c = o.erx, s = o.ery;
    const F dx = mx - o.xn, dy = my - o.yn;
    h.rr = c * dx + s * dy;
    h.rt = c * dy - s * dx;
    h.rz = mz - o.zn;
    const F cc = c * c, ss = s * s, cs = c * s;
    h.vrr = cc * vxx + 2.0f * cs * vxy + ss * vyy;
    h.vtt = ss * vxx - 2.0f * cs * vxy + cc * vyy;
    h.vrt = cs * (vyy - vxx) + (cc - ss) * vxy;
    h.vrz = c * vxz + s * vyz;
    h.vtz = c * vyz - s * vxz;
    h.vzz = vzz;
}

// Inverse of S = C'_pp + V~ (symmetric 3x3, cofactors).  Returns det.
struct Sym3 {
    float rr, rt, rz, tt, tz, zz;
};

__device__ __forceinline__ float invert_S(const PropCov& n, const LocalHit& h, Sym3& si) {
    const float srr = h.vrr, srt = h.vrt, srz = h.vrz;
    const float stt = n.n11 + h.vtt, stz = n.n12 + h.vtz, szz = n.n22 + h.vzz;
    const float k00 = stt * szz - stz * stz;
    const float k01 = srz * stz - srt * szz;
    const float k02 = srt * stz - srz * stt;
    const float det = srr * k00 + srt * k01 + srz * k02;
    const float id = 1.0f / det;
    si.rr = k00 * id;
    si.rt = k01 * id;
    si.rz = k02 * id;
    si.tt = (srr * szz - srz * srz) * id;
    si.tz = (srt * srz - srr * stz) * id;
    si.zz = (srr * stt - srt * srt) * id;
    return det;
}

__device__ __forceinline__ float chi2_of(const Sym3& si, const LocalHit& h) {
    const float ur = si.rr * h.rr + si.rt * h.rt + si.rz * h.rz;
    const float ut = si.rt * h.rr + si.tt * h.rt + si.tz * h.rz;
    const float uz = si.rz * h.rr + si.tz * h.rt + si.zz * h.rz;
    return h.rr * ur + h.rt * ut + h.rz * uz;
}

// chi2 of one hit against the propagated candidate, same Schur elimination as kalman_update
// (one hit of the scoring window).  Returns false when det S <= 0 (the hit is skipped).
__device__ __forceinline__ bool chi2_schur(float n11, float n12, float n22, const LocalHit& h, float& chi2) {
    const float iv = rcp_fast(h.vrr);
    const float sa = h.vrt * iv, sb = h.vrz * iv;
    const float stt = n11 + (h.vtt - sa * h.vrt), stz = n12 + (h.vtz - sa * h.vrz), szz = n22 + (h.vzz - sb * h.vrz);
    const float rt = h.rt - sa * h.rr, rz = h.rz - sb * h.rr;
    const float det2 = stt * szz - stz * stz;
    const float q = szz * rt * rt - 2.0f * stz * rt * rz + stt * rz * rz;
    chi2 = h.rr * h.rr * iv + q * rcp_fast(det2);
    return h.vrr * det2 > 0.0f;
}

// Kalman update in the arrival frame, then re-aim the momentum frame at the updated momentum.
// On success writes the new track (position frame = arrival frame) and returns the chi2
// increment through *dchi2.  Returns a status bit on failure (track untouched).
// Pair form (F = f2): both tracks are updated or neither is -- if either fails, the statuses are returned
// and the pair is left untouched (the caller then takes the two tracks one at a time).
template <class F>
__device__ __forceinline__ typename num_traits<F>::status
kalman_update(TrackT<F>& t, const CrossingT<F>& o, const PropCovT<F>& n, const LocalHitT<F>& h, F* dchi2) {
    using M = typename num_traits<F>::mask;
    // The radial row of C' is zero, so eliminating the radial component of S = C'_pp + V~ first
    // (Schur complement on v_rr) leaves a 2-D measurement in (t, z):
    //   V' = V_tz,tz - s s^T / v_rr,  s = (v_rt, v_rz);   r' = r_tz - s r_r / v_rr;
    //   S' = C'_tz,tz + V';  chi2 = r_r^2 / v_rr + r'^T S'^-1 r';  K = C'[:, tz] S'^-1;
    //   det S = v_rr det S'.
    const F iv = rcp_fast(h.vrr);
    const F sa = h.vrt * iv, sb = h.vrz * iv;
    const F qtt = h.vtt - sa * h.vrt, qtz = h.vtz - sa * h.vrz, qzz = h.vzz - sb * h.vrz;
    const F stt = n.n11 + qtt, stz = n.n12 + qtz, szz = n.n22 + qzz;
    const F rt = h.rt - sa * h.rr, rz = h.rz - sb * h.rr;
    const F det2 = stt * szz - stz * stz;
    const M pd = h.vrr * det2 > 0.0f;
    if (!all_of(pd)) return select_u(!pd, ST_S_NOT_PD, 0u);
    const F id = rcp_fast(det2);
    const F itt = szz * id, itz = -stz * id, izz = stt * id;
    const F ut = itt * rt + itz * rz, uz = itz * rt + izz * rz;
    const F chi2 = h.rr * h.rr * iv + rt * ut + rz * uz;
    // state increments d = C'[:, tz] S'^-1 r'
    const F d1 = n.n11 * ut + n.n12 * uz;
    const F d2 = n.n12 * ut + n.n22 * uz;
    const F d3 = n.n13 * ut + n.n23 * uz;
    const F d4 = n.n14 * ut + n.n24 * uz;
    const F d5 = n.n15 * ut + n.n25 * uz;
    // finite(chi2) and finite(state): any non-finite term makes this sum non-finite
    const F probe = chi2 + ((d1 + d2) + (d3 + d4) + d5) * 0.0f;
    const M fin = abs_(probe) < __int_as_float(0x7f800000);
    if (!all_of(fin)) return select_u(!fin, ST_NONFINITE, 0u);
    *dchi2 = chi2;
    // gain rows (t z b1 b2 c) x columns (t, z)
#define KF_KROW(ct, cz, kt, kz)            \
    const F kt = ct * itt + cz * itz;      \
    const F kz = ct * itz + cz * izz;
    KF_KROW(n.n11, n.n12, k1t, k1z)
    KF_KROW(n.n12, n.n22, k2t, k2z)
    KF_KROW(n.n13, n.n23, k3t, k3z)
    KF_KROW(n.n14, n.n24, k4t, k4z)
    KF_KROW(n.n15, n.n25, k5t, k5z)
#undef KF_KROW
    // state
    t.x = o.xn - o.ery * d1;
    t.y = o.yn + o.erx * d1;
    t.z = o.zn + d2;
    const F pxu = o.pxn + o.elx * d3 - o.ely * d4;
    const F pyu = o.pyn + o.ely * d3 + o.elx * d4;
    t.px = pxu;
    t.py = pyu;
    const F pzu = t.pz + d5 + o.T * d3;
    t.pz = pzu;
    t.eax = o.erx;
    t.eay = o.ery;
    // position rows ("V form", no subtraction): C[i][a] = sum_b K[i][b] V'[b][a]; radial row stays 0
    t.c00 = 0.0f; t.c01 = 0.0f; t.c02 = 0.0f; t.c03 = 0.0f; t.c04 = 0.0f; t.c05 = 0.0f;
    t.c11 = k1t * qtt + k1z * qtz;
    t.c12 = k1t * qtz + k1z * qzz;
    t.c22 = k2t * qtz + k2z * qzz;
    t.c13 = k3t * qtt + k3z * qtz;
    t.c23 = k3t * qtz + k3z * qzz;
    t.c14 = k4t * qtt + k4z * qtz;
    t.c24 = k4t * qtz + k4z * qzz;
    t.c15 = k5t * qtt + k5z * qtz;
    t.c25 = k5t * qtz + k5z * qzz;
    // momentum block: C'_mm - K_m C'_pm  (C'_pm rows t, z)
    t.c33 = fma_(-k3z, n.n23, fma_(-k3t, n.n13, n.n33));
    t.c34 = fma_(-k3z, n.n24, fma_(-k3t, n.n14, n.n34));
    t.c35 = fma_(-k3z, n.n25, fma_(-k3t, n.n15, n.n35));
    t.c44 = fma_(-k4z, n.n24, fma_(-k4t, n.n14, n.n44));
    t.c45 = fma_(-k4z, n.n25, fma_(-k4t, n.n15, n.n45));
    t.c55 = fma_(-k5z, n.n25, fma_(-k5t, n.n15, n.n55));
    // re-aim the momentum frame: exp(i d) = conj(e_l,new) e_l' = ((pT + d3) - i d4) / pT,new
    const F pt = o.pt2 * o.ipt;
    const F ar = pt + d3;
    const F iptn = rsqrt_fast(ar * ar + d4 * d4);
    reaim_momentum<true>(t, ar * iptn, -d4 * iptn, o.T, pzu * iptn);
    return select_u(pd, 0u, 0u);
}

// One step of the backward refit (reading A18) for the layer with constants L: the first step updates in place,
// every later one adds the noise of the scatterer just left (Lprev), propagates inward and updates.  Returns 0
// and the chi2 increment, or the status bits of the failure with the track as it was (layer skipped).
// Pair form: both tracks take the step or neither does.
template <bool BOUNDED, class F>
__device__ __forceinline__ typename num_traits<F>::status
refit_step(TrackT<F>& t, arg<F> k, arg<F> ik, const LayerConst& L, const LayerConst& Lprev, int model, float mass2,
           const Bethe& el, bool first, arg<F> mx, arg<F> my, arg<F> mz, arg<F> vxx, arg<F> vxy, arg<F> vxz,
           arg<F> vyy, arg<F> vyz, arg<F> vzz, F* dchi2) {
    CrossingT<F> o;
    PropCovT<F> n;
    LocalHitT<F> h;
    if constexpr (std::is_same<F, float>::value) {
        if (!first && (model & MODEL_ENERGY_LOSS)) {
            // reading A21: the layer just left gives back the energy it took, before its scattering noise is
            // added; worked on a copy so that any failure leaves the track as it was
            TrackT<float> tb = t;
            const float pt2 = tb.px * tb.px + tb.py * tb.py;
            const float ipt = rsqrt_fast(pt2);
            Eloss e;
            if (!energy_loss_factors(el, Lprev, model, mass2, (tb.eax * tb.px + tb.eay * tb.py) * ipt, pt2, ipt,
                                     tb.pz, true, e))
                return ST_PROP_FAIL;
            apply_energy_loss(e, tb);
            const uint32_t reached = reach_layer<true, BOUNDED>(tb, k, ik, L, o);
            if (reached) return reached;
            add_process_noise(tb, Lprev, model, mass2);
            transport_cov<true>(tb, o, 0.0f, mass2, n);
            hit_to_local(o, mx, my, mz, vxx, vxy, vxz, vyy, vyz, vzz, h);
            const uint32_t rc = kalman_update(tb, o, n, h, dchi2);
            if (rc == 0u) t = tb;
            return rc;
        }
    }
    const F k33 = t.c33, k35 = t.c35, k44 = t.c44, k55 = t.c55;
    if (first) crossing_in_place(t, o, n);
    else {
        const auto reached = reach_layer<true, BOUNDED>(t, k, ik, L, o);
        if (!is_zero(reached)) return reached;
        add_process_noise(t, Lprev, model, mass2);      // the scatterer just left behind
        transport_cov<true>(t, o, F(0.0f), mass2, n);
    }
    hit_to_local(o, mx, my, mz, vxx, vxy, vxz, vyy, vyz, vzz, h);
    const auto rc = kalman_update(t, o, n, h, dchi2);
    if (!is_zero(rc)) { t.c33 = k33; t.c35 = k35; t.c44 = k44; t.c55 = k55; }   // layer skipped
    return rc;
}

// ---- reading A23: endcap discs -------------------------------------------------------------------------------
// Crossing of the helix with the plane z = zt (zt = +-L.zd on the side the track is heading to):
//     theta = k (zt - z) / pz,   w' = w + (i pi / k)(E - 1),   pi' = pi E,   E = exp(-i theta).
// In the local frame the Jacobian of that map is, over (a1, a2, z | b1, b2, c), with P = conj(e_r') e_a,
// N = exp(i a')(S + i Cm)/k, exp(i a') = conj(e_r') e_l', T = pz/pT:
//     row r'  = ( Re P, -Im P, -cos a'/T, Re N - cos a' theta/k, -Im N, -cos a' theta/(k T) )
//     row t'  = ( Im P,  Re P, -sin a'/T, Im N - sin a' theta/k,  Re N, -sin a' theta/(k T) )
//     row z'  = 0                      (the arrival point stays in the plane: the z row of C' is zero)
//     row b1' = e_b1,   row b2' = e_b2 + (0, 0, k/T, theta, 0, theta/T),   row c' = e_c
// (d theta = -(k/pz) dz - (theta/pz) d pz moves the arrival point along pi'/k and turns the momentum).
struct DiscCrossing {
    float xn, yn, zt, pxn, pyn;
    float erx, ery, elx, ely;
    float pc, ps, nr, nt, ca, sa;
    float thk, theta, T, iT, pt2, ipt;
};

// Propagated covariance at a disc over (r', t' | b1, b2, c); its z row is zero.
struct DiscCov {
    float rr, rt, r3, r4, r5;
    float tt, t3, t4, t5;
    float n33, n34, n35, n44, n45, n55;
};

// Returns 0, ST_PROP_FAIL (plane behind the state, |pz| = 0, half a turn or more away) or ST_OUTSIDE.
// INWARD (the refit of reading A18): the plane lies behind the state and is reached by following the helix backward
// in path length (theta of the opposite sign; the Jacobian holds for either sign).
template <bool INWARD = false>
__device__ __forceinline__ uint32_t helix_to_plane(const Track& t, float k, float ik, const LayerConst& L, DiscCrossing& o) {
    const float px = t.px, py = t.py, pz = t.pz;
    const float zt = copysignf(L.zd, pz);
    const float dz = zt - t.z;
    const float pt2 = px * px + py * py;
    const float theta = k * dz / pz;
    // (NaNs fail every comparison)
    if (!(INWARD ? dz * pz < 0.0f : dz * pz > 0.0f) || !(fabsf(theta) < 3.14159265f) || !(pt2 > 0.0f)) return ST_PROP_FAIL;
    float sh, ch;
    sincosf(0.5f * theta, &sh, &ch);
    const float S = 2.0f * sh * ch, Cm = 2.0f * sh * sh, co = 1.0f - Cm;
    o.theta = theta;
    o.thk = theta * ik;
    o.xn = t.x + (px * S + py * Cm) * ik;
    o.yn = t.y + (py * S - px * Cm) * ik;
    o.zt = zt;
    o.pxn = px * co + py * S;
    o.pyn = py * co - px * S;
    const float rho2 = o.xn * o.xn + o.yn * o.yn;
    if (!(rho2 >= L.rmin2 && rho2 <= L.rmax2)) return ST_OUTSIDE;
    const float irho = rsqrt_fast(rho2), ipt = rsqrt_fast(pt2);
    o.pt2 = pt2; o.ipt = ipt;
    o.erx = o.xn * irho; o.ery = o.yn * irho;
    o.elx = o.pxn * ipt; o.ely = o.pyn * ipt;
    o.ca = o.erx * o.elx + o.ery * o.ely;
    o.sa = o.erx * o.ely - o.ery * o.elx;
    o.pc = o.erx * t.eax + o.ery * t.eay;
    o.ps = o.erx * t.eay - o.ery * t.eax;
    o.nr = (S * o.ca - Cm * o.sa) * ik;
    o.nt = (S * o.sa + Cm * o.ca) * ik;
    o.T = pz * ipt;
    o.iT = pt2 * ipt / pz;
    return 0u;
}

// C' = F~ C F~^T + Q~ for the to-plane map; the input covariance is general (21 elements).
__device__ __forceinline__ void transport_cov_disc(const Track& t, const DiscCrossing& o, float k, float ms, float mass2,
                                                   DiscCov& n) {
    const float R[6] = {o.pc, -o.ps, -o.ca * o.iT, o.nr - o.ca * o.thk, -o.nt, -o.ca * o.thk * o.iT};
    const float Tt[6] = {o.ps, o.pc, -o.sa * o.iT, o.nt - o.sa * o.thk, o.nr, -o.sa * o.thk * o.iT};
    const float b2z = k * o.iT, b2b = o.theta, b2c = o.theta * o.iT;     // row b2' = e_b2 + (0, 0, b2z, b2b, 0, b2c)
    const float C[6][6] = {{t.c00, t.c01, t.c02, t.c03, t.c04, t.c05}, {t.c01, t.c11, t.c12, t.c13, t.c14, t.c15},
                           {t.c02, t.c12, t.c22, t.c23, t.c24, t.c25}, {t.c03, t.c13, t.c23, t.c33, t.c34, t.c35},
                           {t.c04, t.c14, t.c24, t.c34, t.c44, t.c45}, {t.c05, t.c15, t.c25, t.c35, t.c45, t.c55}};
    float u[6], v[6], w[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        u[i] = C[i][0] * R[0] + C[i][1] * R[1] + C[i][2] * R[2] + C[i][3] * R[3] + C[i][4] * R[4] + C[i][5] * R[5];
        v[i] = C[i][0] * Tt[0] + C[i][1] * Tt[1] + C[i][2] * Tt[2] + C[i][3] * Tt[3] + C[i][4] * Tt[4] + C[i][5] * Tt[5];
        w[i] = C[i][4] + C[i][2] * b2z + C[i][3] * b2b + C[i][5] * b2c;
    }
    auto dot6 = [](const float* a, const float* b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2] + a[3] * b[3] + a[4] * b[4] + a[5] * b[5]; };
    auto dotB2 = [&](const float* a) { return a[4] + a[2] * b2z + a[3] * b2b + a[5] * b2c; };
    // Highland (A5) at the propagated momentum, sheared to (b1, b2, c) as in transport_cov
    const float pz = t.pz;
    const float p2 = o.pt2 + pz * pz;
    const float ip2 = rcp_fast(p2);
    const float th2 = ms * (p2 + mass2) * ip2 * ip2;
    const float qc = th2 * p2 * o.ipt;
    n.rr = dot6(R, u); n.rt = dot6(Tt, u); n.tt = dot6(Tt, v);
    n.r3 = u[3]; n.r4 = dotB2(u); n.r5 = u[5];
    n.t3 = v[3]; n.t4 = dotB2(v); n.t5 = v[5];
    n.n33 = t.c33 + th2 * pz * pz;
    n.n34 = w[3];
    n.n35 = t.c35 - qc * pz;
    n.n44 = dotB2(w) + th2 * p2;
    n.n45 = w[5];
    n.n55 = t.c55 + qc * (p2 * o.ipt);
}

// Highland factor at a disc: flat, or (reading A20 on a disc) thickness / |cos| of the angle to the z axis = p / |pz|.
__device__ __forceinline__ float ms_at_disc(const LayerConst& L, int model, const DiscCrossing& o, float pz) {
    if ((model & MODEL_PATH_LENGTH) == 0) return L.ms;
    const float f = sqrtf(o.pt2 + pz * pz) * rcp_fast(fabsf(pz));
    const float lg = 1.0f + 0.038f * (L.ln_t + __logf(f));
    return L.ms0 * f * lg * lg;
}

// Reading A21 at a disc: the same direction-preserving momentum scaling and Jacobian J on (b1, b2, c) as
// apply_energy_loss, on the disc's propagated state and covariance (T = pz / pT does not change).
__device__ __forceinline__ void apply_energy_loss_disc(const Eloss& e, DiscCrossing& o, DiscCov& n, float& pz) {
    const float f = e.f, g = e.g, h = e.h, ff = f * f;
    o.pxn *= f; o.pyn *= f; pz *= f;
    o.pt2 *= ff;
    o.ipt *= rcp_fast(f);
    n.r3 = g * n.r3 + h * n.r5;
    n.t3 = g * n.t3 + h * n.t5;
    n.n33 = g * (g * n.n33 + 2.0f * h * n.n35) + h * h * n.n55;
    n.n34 = f * (g * n.n34 + h * n.n45);
    n.n35 = f * (g * n.n35 + h * n.n55);
    n.r4 *= f; n.t4 *= f; n.r5 *= f; n.t5 *= f;
    n.n44 *= ff; n.n45 *= ff; n.n55 *= ff;
}

// Kalman update at a disc: C' has a zero z row, so the z component of S = C'_pp + V~ is eliminated first (Schur
// complement on v_zz), leaving a 2-D measurement in (r, t) -- the disc's counterpart of kalman_update.
__device__ __forceinline__ uint32_t kalman_update_disc(Track& t, const DiscCrossing& o, const DiscCov& n, const LocalHit& h,
                                                       float* dchi2) {
    const float iv = rcp_fast(h.vzz);
    const float sa = h.vrz * iv, sb = h.vtz * iv;
    const float qrr = h.vrr - sa * h.vrz, qrt = h.vrt - sa * h.vtz, qtt = h.vtt - sb * h.vtz;
    const float srr = n.rr + qrr, srt = n.rt + qrt, stt = n.tt + qtt;
    const float rr = h.rr - sa * h.rz, rt = h.rt - sb * h.rz;
    const float det2 = srr * stt - srt * srt;
    if (!(h.vzz * det2 > 0.0f)) return ST_S_NOT_PD;
    const float id = rcp_fast(det2);
    const float irr = stt * id, irt = -srt * id, itt = srr * id;
    const float ur = irr * rr + irt * rt, ut = irt * rr + itt * rt;
    const float chi2 = h.rz * h.rz * iv + rr * ur + rt * ut;
    const float d0 = n.rr * ur + n.rt * ut;
    const float d1 = n.rt * ur + n.tt * ut;
    const float d3 = n.r3 * ur + n.t3 * ut;
    const float d4 = n.r4 * ur + n.t4 * ut;
    const float d5 = n.r5 * ur + n.t5 * ut;
    const float probe = chi2 + ((d0 + d1) + (d3 + d4) + d5) * 0.0f;
    if (!(fabsf(probe) < __int_as_float(0x7f800000))) return ST_NONFINITE;
    *dchi2 = chi2;
#define KF_KROW(cr, ct, kr, kt)          \
    const float kr = cr * irr + ct * irt; \
    const float kt = cr * irt + ct * itt;
    KF_KROW(n.rr, n.rt, k0r, k0t)
    KF_KROW(n.rt, n.tt, k1r, k1t)
    KF_KROW(n.r3, n.t3, k3r, k3t)
    KF_KROW(n.r4, n.t4, k4r, k4t)
    KF_KROW(n.r5, n.t5, k5r, k5t)
#undef KF_KROW
    t.x = o.xn + o.erx * d0 - o.ery * d1;
    t.y = o.yn + o.ery * d0 + o.erx * d1;
    t.z = o.zt;
    const float pxu = o.pxn + o.elx * d3 - o.ely * d4;
    const float pyu = o.pyn + o.ely * d3 + o.elx * d4;
    const float pzu = t.pz + d5 + o.T * d3;
    t.px = pxu; t.py = pyu; t.pz = pzu;
    t.eax = o.erx; t.eay = o.ery;
    // position rows ("V form"), z row zero
    t.c00 = k0r * qrr + k0t * qrt;
    t.c01 = k0r * qrt + k0t * qtt;
    t.c11 = k1r * qrt + k1t * qtt;
    t.c02 = 0.0f; t.c12 = 0.0f; t.c22 = 0.0f; t.c23 = 0.0f; t.c24 = 0.0f; t.c25 = 0.0f;
    t.c03 = k3r * qrr + k3t * qrt;
    t.c13 = k3r * qrt + k3t * qtt;
    t.c04 = k4r * qrr + k4t * qrt;
    t.c14 = k4r * qrt + k4t * qtt;
    t.c05 = k5r * qrr + k5t * qrt;
    t.c15 = k5r * qrt + k5t * qtt;
    // momentum block: C'_mm - K_m C'_pm
    t.c33 = fmaf(-k3t, n.t3, fmaf(-k3r, n.r3, n.n33));
    t.c34 = fmaf(-k3t, n.t4, fmaf(-k3r, n.r4, n.n34));
    t.c35 = fmaf(-k3t, n.t5, fmaf(-k3r, n.r5, n.n35));
    t.c44 = fmaf(-k4t, n.t4, fmaf(-k4r, n.r4, n.n44));
    t.c45 = fmaf(-k4t, n.t5, fmaf(-k4r, n.r5, n.n45));
    t.c55 = fmaf(-k5t, n.t5, fmaf(-k5r, n.r5, n.n55));
    const float pt = o.pt2 * o.ipt;
    const float ar = pt + d3;
    const float iptn = rsqrt_fast(ar * ar + d4 * d4);
    reaim_momentum<false>(t, ar * iptn, -d4 * iptn, o.T, pzu * iptn);
    return 0u;
}

// chi2 of one hit against a candidate propagated to a DISC (C' has no variance along z): the z component of
// S = C'_pp + V~ is eliminated first, as in kalman_update_disc; n_rr, n_rt, n_tt = the in-plane block of C'.
__device__ __forceinline__ bool chi2_schur_disc(float nrr, float nrt, float ntt, const LocalHit& h, float& chi2) {
    const float iv = rcp_fast(h.vzz);
    const float sa = h.vrz * iv, sb = h.vtz * iv;
    const float srr = nrr + (h.vrr - sa * h.vrz), srt = nrt + (h.vrt - sa * h.vtz), stt = ntt + (h.vtt - sb * h.vtz);
    const float rr = h.rr - sa * h.rz, rt = h.rt - sb * h.rz;
    const float det2 = srr * stt - srt * srt;
    const float q = stt * rr * rr - 2.0f * srt * rr * rt + srr * rt * rt;
    chi2 = h.rz * h.rz * iv + q * rcp_fast(det2);
    return h.vzz * det2 > 0.0f;
}

// Keep the state propagated to a disc (no hit used).
__device__ __forceinline__ void commit_propagated_disc(Track& t, const DiscCrossing& o, const DiscCov& n) {
    t.x = o.xn; t.y = o.yn; t.z = o.zt; t.px = o.pxn; t.py = o.pyn;
    t.eax = o.erx; t.eay = o.ery;
    t.c00 = n.rr; t.c01 = n.rt; t.c11 = n.tt;
    t.c02 = 0.0f; t.c12 = 0.0f; t.c22 = 0.0f; t.c23 = 0.0f; t.c24 = 0.0f; t.c25 = 0.0f;
    t.c03 = n.r3; t.c04 = n.r4; t.c05 = n.r5;
    t.c13 = n.t3; t.c14 = n.t4; t.c15 = n.t5;
    t.c33 = n.n33; t.c34 = n.n34; t.c35 = n.n35;
    t.c44 = n.n44; t.c45 = n.n45;
    t.c55 = n.n55;
}

// Keep the propagated state (no hit used): position frame = arrival frame, momentum frame
// already follows the propagated momentum.
__device__ __forceinline__ void commit_propagated(Track& t, const Crossing& o, const PropCov& n) {
    t.x = o.xn; t.y = o.yn; t.z = o.zn; t.px = o.pxn; t.py = o.pyn;
    t.eax = o.erx; t.eay = o.ery;
    t.c00 = 0.0f; t.c01 = 0.0f; t.c02 = 0.0f; t.c03 = 0.0f; t.c04 = 0.0f; t.c05 = 0.0f;
    t.c11 = n.n11; t.c12 = n.n12; t.c13 = n.n13; t.c14 = n.n14; t.c15 = n.n15;
    t.c22 = n.n22; t.c23 = n.n23; t.c24 = n.n24; t.c25 = n.n25;
    t.c33 = n.n33; t.c34 = n.n34; t.c35 = n.n35;
    t.c44 = n.n44; t.c45 = n.n45;
    t.c55 = n.n55;
}

// ---- SoA load / store (element-major, plane stride ld) ---------------------------------------
__device__ __forceinline__ void load_track(Track& t, const float* __restrict__ par,
                                           const float* __restrict__ cov, int64_t ld, int64_t i) {
    t.x = __ldg(par + 0 * ld + i);  t.y = __ldg(par + 1 * ld + i);  t.z = __ldg(par + 2 * ld + i);
    t.px = __ldg(par + 3 * ld + i); t.py = __ldg(par + 4 * ld + i); t.pz = __ldg(par + 5 * ld + i);
    t.c00 = __ldg(cov + 0 * ld + i);  t.c01 = __ldg(cov + 1 * ld + i);  t.c02 = __ldg(cov + 2 * ld + i);
    t.c03 = __ldg(cov + 3 * ld + i);  t.c04 = __ldg(cov + 4 * ld + i);  t.c05 = __ldg(cov + 5 * ld + i);
    t.c11 = __ldg(cov + 6 * ld + i);  t.c12 = __ldg(cov + 7 * ld + i);  t.c13 = __ldg(cov + 8 * ld + i);
    t.c14 = __ldg(cov + 9 * ld + i);  t.c15 = __ldg(cov + 10 * ld + i);
    t.c22 = __ldg(cov + 11 * ld + i); t.c23 = __ldg(cov + 12 * ld + i); t.c24 = __ldg(cov + 13 * ld + i);
    t.c25 = __ldg(cov + 14 * ld + i);
    t.c33 = __ldg(cov + 15 * ld + i); t.c34 = __ldg(cov + 16 * ld + i); t.c35 = __ldg(cov + 17 * ld + i);
    t.c44 = __ldg(cov + 18 * ld + i); t.c45 = __ldg(cov + 19 * ld + i);
    t.c55 = __ldg(cov + 20 * ld + i);
    t.eax = 1.0f;
    t.eay = 0.0f;
}

__device__ __forceinline__ void store_track(const Track& t, float* __restrict__ par,
                                            float* __restrict__ cov, int64_t ld, int64_t i) {
    par[0 * ld + i] = t.x;  par[1 * ld + i] = t.y;  par[2 * ld + i] = t.z;
    par[3 * ld + i] = t.px; par[4 * ld + i] = t.py; par[5 * ld + i] = t.pz;
    cov[0 * ld + i] = t.c00;  cov[1 * ld + i] = t.c01;  cov[2 * ld + i] = t.c02;
    cov[3 * ld + i] = t.c03;  cov[4 * ld + i] = t.c04;  cov[5 * ld + i] = t.c05;
    cov[6 * ld + i] = t.c11;  cov[7 * ld + i] = t.c12;  cov[8 * ld + i] = t.c13;
    cov[9 * ld + i] = t.c14;  cov[10 * ld + i] = t.c15;
    cov[11 * ld + i] = t.c22; cov[12 * ld + i] = t.c23; cov[13 * ld + i] = t.c24;
    cov[14 * ld + i] = t.c25;
    cov[15 * ld + i] = t.c33; cov[16 * ld + i] = t.c34; cov[17 * ld + i] = t.c35;
    cov[18 * ld + i] = t.c44; cov[19 * ld + i] = t.c45;
    cov[20 * ld + i] = t.c55;
}

}  // namespace kf
