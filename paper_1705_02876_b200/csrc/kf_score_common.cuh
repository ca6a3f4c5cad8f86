// kf_score_common.cuh -- device helpers shared by the best-hit and the combinatorial builders
// (kf_score.cu, kf_comb.cu): the SoA scratch between the per-candidate and the per-hit kernels, the
// local-frame track store, and the full chi2 of one packed hit record.
#pragma once
#include <math_constants.h>

#include "kf_internal.h"

namespace kf {
namespace {

constexpr int kScanBlock = 128;   // 4 candidates per CTA
constexpr int kCandBlock = 128;   // threads (= candidates) per CTA of the per-candidate kernels

// Scratch planes (each [ld] floats): what the scan and the update need from the propagation.
enum : int {
    SC_XN, SC_YN, SC_ZN, SC_ERX, SC_ERY, SC_N11, SC_N12, SC_N22,   // scan + update
    SC_PXN, SC_PYN, SC_PZ, SC_ELX, SC_ELY, SC_T, SC_PT2, SC_IPT,   // update
    SC_N13, SC_N14, SC_N15, SC_N23, SC_N24, SC_N25, SC_N33, SC_N34, SC_N35, SC_N44, SC_N45, SC_N55,
    SC_BIN,                                                         // window centre (i_eta << 16 | i_phi), int bits
    SC_PLANES
};
static_assert(SC_PLANES == kScorePlanes, "scratch plane count");

__device__ __forceinline__ void put_scratch(float* __restrict__ sc, int64_t ld, int64_t i, const Crossing& o,
                                            const PropCov& n, float pz) {
#define KF_PUT(k, v) sc[(int64_t)(k) * ld + i] = (v)
    KF_PUT(SC_XN, o.xn);   KF_PUT(SC_YN, o.yn);   KF_PUT(SC_ZN, o.zn);   KF_PUT(SC_ERX, o.erx); KF_PUT(SC_ERY, o.ery);
    KF_PUT(SC_N11, n.n11); KF_PUT(SC_N12, n.n12); KF_PUT(SC_N22, n.n22);
    KF_PUT(SC_PXN, o.pxn); KF_PUT(SC_PYN, o.pyn); KF_PUT(SC_PZ, pz);     KF_PUT(SC_ELX, o.elx); KF_PUT(SC_ELY, o.ely);
    KF_PUT(SC_T, o.T);     KF_PUT(SC_PT2, o.pt2); KF_PUT(SC_IPT, o.ipt);
    KF_PUT(SC_N13, n.n13); KF_PUT(SC_N14, n.n14); KF_PUT(SC_N15, n.n15);
    KF_PUT(SC_N23, n.n23); KF_PUT(SC_N24, n.n24); KF_PUT(SC_N25, n.n25);
    KF_PUT(SC_N33, n.n33); KF_PUT(SC_N34, n.n34); KF_PUT(SC_N35, n.n35);
    KF_PUT(SC_N44, n.n44); KF_PUT(SC_N45, n.n45); KF_PUT(SC_N55, n.n55);
#undef KF_PUT
}

__device__ __forceinline__ void get_scratch(const float* __restrict__ sc, int64_t ld, int64_t i, Crossing& o,
                                            PropCov& n, float& pz) {
#define KF_GET(k) sc[(int64_t)(k) * ld + i]
    o.xn = KF_GET(SC_XN);   o.yn = KF_GET(SC_YN);   o.zn = KF_GET(SC_ZN);   o.erx = KF_GET(SC_ERX); o.ery = KF_GET(SC_ERY);
    n.n11 = KF_GET(SC_N11); n.n12 = KF_GET(SC_N12); n.n22 = KF_GET(SC_N22);
    o.pxn = KF_GET(SC_PXN); o.pyn = KF_GET(SC_PYN); pz = KF_GET(SC_PZ);     o.elx = KF_GET(SC_ELX); o.ely = KF_GET(SC_ELY);
    o.T = KF_GET(SC_T);     o.pt2 = KF_GET(SC_PT2); o.ipt = KF_GET(SC_IPT);
    n.n13 = KF_GET(SC_N13); n.n14 = KF_GET(SC_N14); n.n15 = KF_GET(SC_N15);
    n.n23 = KF_GET(SC_N23); n.n24 = KF_GET(SC_N24); n.n25 = KF_GET(SC_N25);
    n.n33 = KF_GET(SC_N33); n.n34 = KF_GET(SC_N34); n.n35 = KF_GET(SC_N35);
    n.n44 = KF_GET(SC_N44); n.n45 = KF_GET(SC_N45); n.n55 = KF_GET(SC_N55);
#undef KF_GET
}

// Local-frame track <-> scratch between the layers of kf_build_best_hit (23 floats: the radial row of the
// covariance is identically zero after the first layer).
__device__ __forceinline__ void hit_from_record(const float4* __restrict__ rec, int32_t slot, const Crossing& o,
                                                LocalHit& h) {
    const float4* r0 = rec + (int64_t)slot * kRecWords;
    const float4 A = __ldg(r0), B = __ldg(r0 + 1), C = __ldg(r0 + 2);
    hit_to_local(o, A.x, A.y, A.z, B.x, B.y, C.x, B.z, C.y, A.w, h);
}

// Propagate a local-frame track to layer Lc and park the result in the scratch.  Returns 0 if it got there,
// else the status bit that says why not (ST_PROP_FAIL, ST_OUTSIDE).
template <bool RADIAL_NULL>
__device__ __forceinline__ uint32_t propagate_to_scratch(const Track& t, float k, float ik, const LayerConst& Lc,
                                                         int model, float mass2, const Bethe& el, const BinGrid& g,
                                                         float* sc, int64_t ld, int64_t i) {
    Crossing o;
    const uint32_t reached = reach_layer(t, k, ik, Lc, o);
    if (reached) return reached;
    PropCov n;
    transport_cov<RADIAL_NULL>(t, o, ms_at_crossing(Lc, model, o, t.pz), mass2, n);
    float pz = t.pz;
    if (model & MODEL_ENERGY_LOSS) {   // reading A21
        Eloss e;
        if (!energy_loss_factors(el, Lc, model, mass2, o.erx * o.elx + o.ery * o.ely, o.pt2, o.ipt, pz, false, e))
            return ST_PROP_FAIL;
        apply_energy_loss(e, o, n, pz);
    }
    put_scratch(sc, ld, i, o, n, pz);
    // the candidate's own bin (reading A16): eta = asinh(z'/r), phi = atan2(y', x') -- once per candidate
    // here, not once per lane in the scan
    const float eta = asinhf(o.zn * Lc.inv_r);
    const float phi = atan2f(o.yn, o.xn);
    int ie = (int)floorf((eta + g.eta_max) / (2.0f * g.eta_max / (float)g.n_eta));
    ie = ie < 0 ? 0 : (ie > g.n_eta - 1 ? g.n_eta - 1 : ie);
    int ip = (int)floorf((phi + CUDART_PI_F) / (2.0f * CUDART_PI_F / (float)g.n_phi));
    ip = ((ip % g.n_phi) + g.n_phi) % g.n_phi;
    sc[(int64_t)SC_BIN * ld + i] = __int_as_float((ie << 16) | ip);
    return 0u;
}

// ---- the same for a DISC layer (readings A23 / A24) --------------------------------------------------------
// The scratch planes keep their places with the disc's meaning: SC_ZN = the plane's z, SC_N11 / N12 / N22 = the
// in-plane block rr / rt / tt of C', SC_N13..N15 = r3 r4 r5, SC_N23..N25 = t3 t4 t5.
__device__ __forceinline__ void get_scratch_disc(const float* __restrict__ sc, int64_t ld, int64_t i, DiscCrossing& o,
                                                 DiscCov& n, float& pz) {
#define KF_GET(k) sc[(int64_t)(k) * ld + i]
    o.xn = KF_GET(SC_XN);   o.yn = KF_GET(SC_YN);   o.zt = KF_GET(SC_ZN);   o.erx = KF_GET(SC_ERX); o.ery = KF_GET(SC_ERY);
    n.rr = KF_GET(SC_N11);  n.rt = KF_GET(SC_N12);  n.tt = KF_GET(SC_N22);
    o.pxn = KF_GET(SC_PXN); o.pyn = KF_GET(SC_PYN); pz = KF_GET(SC_PZ);     o.elx = KF_GET(SC_ELX); o.ely = KF_GET(SC_ELY);
    o.T = KF_GET(SC_T);     o.pt2 = KF_GET(SC_PT2); o.ipt = KF_GET(SC_IPT);
    n.r3 = KF_GET(SC_N13);  n.r4 = KF_GET(SC_N14);  n.r5 = KF_GET(SC_N15);
    n.t3 = KF_GET(SC_N23);  n.t4 = KF_GET(SC_N24);  n.t5 = KF_GET(SC_N25);
    n.n33 = KF_GET(SC_N33); n.n34 = KF_GET(SC_N34); n.n35 = KF_GET(SC_N35);
    n.n44 = KF_GET(SC_N44); n.n45 = KF_GET(SC_N45); n.n55 = KF_GET(SC_N55);
#undef KF_GET
}

__device__ __forceinline__ uint32_t propagate_to_scratch_disc(const Track& t, float k, float ik, const LayerConst& Lc,
                                                              int model, float mass2, const Bethe& el, const BinGrid& g,
                                                              float* sc, int64_t ld, int64_t i) {
    DiscCrossing o;
    const uint32_t reached = helix_to_plane(t, k, ik, Lc, o);
    if (reached) return reached;
    DiscCov n;
    transport_cov_disc(t, o, k, ms_at_disc(Lc, model, o, t.pz), mass2, n);
    float pz = t.pz;
    if (model & MODEL_ENERGY_LOSS) {   // reading A21 at a disc (path factor |p| / |pz|)
        Eloss e;
        if (!energy_loss_factors(el, Lc, model, mass2, o.T, o.pt2, o.ipt, pz, false, e)) return ST_PROP_FAIL;
        apply_energy_loss_disc(e, o, n, pz);
    }
#define KF_PUT(k, v) sc[(int64_t)(k) * ld + i] = (v)
    KF_PUT(SC_XN, o.xn);   KF_PUT(SC_YN, o.yn);   KF_PUT(SC_ZN, o.zt);   KF_PUT(SC_ERX, o.erx); KF_PUT(SC_ERY, o.ery);
    KF_PUT(SC_N11, n.rr);  KF_PUT(SC_N12, n.rt);  KF_PUT(SC_N22, n.tt);
    KF_PUT(SC_PXN, o.pxn); KF_PUT(SC_PYN, o.pyn); KF_PUT(SC_PZ, pz);     KF_PUT(SC_ELX, o.elx); KF_PUT(SC_ELY, o.ely);
    KF_PUT(SC_T, o.T);     KF_PUT(SC_PT2, o.pt2); KF_PUT(SC_IPT, o.ipt);
    KF_PUT(SC_N13, n.r3);  KF_PUT(SC_N14, n.r4);  KF_PUT(SC_N15, n.r5);
    KF_PUT(SC_N23, n.t3);  KF_PUT(SC_N24, n.t4);  KF_PUT(SC_N25, n.t5);
    KF_PUT(SC_N33, n.n33); KF_PUT(SC_N34, n.n34); KF_PUT(SC_N35, n.n35);
    KF_PUT(SC_N44, n.n44); KF_PUT(SC_N45, n.n45); KF_PUT(SC_N55, n.n55);
#undef KF_PUT
    // the candidate's own bin (reading A24): eta from the arrival point's own rho
    const float eta = asinhf(o.zt * rsqrtf(o.xn * o.xn + o.yn * o.yn));
    const float phi = atan2f(o.yn, o.xn);
    int ie = (int)floorf((eta + g.eta_max) / (2.0f * g.eta_max / (float)g.n_eta));
    ie = ie < 0 ? 0 : (ie > g.n_eta - 1 ? g.n_eta - 1 : ie);
    int ip = (int)floorf((phi + CUDART_PI_F) / (2.0f * CUDART_PI_F / (float)g.n_phi));
    ip = ((ip % g.n_phi) + g.n_phi) % g.n_phi;
    sc[(int64_t)SC_BIN * ld + i] = __int_as_float((ie << 16) | ip);
    return 0u;
}

// ---- the current local-frame track between layers (kf_build_best_hit): 29 planes -------------------------
__device__ __forceinline__ void put_track(float* __restrict__ ts, int64_t ld, int64_t i, const Track& t) {
    const float v[29] = {t.x, t.y, t.z, t.px, t.py, t.pz, t.eax, t.eay, t.c00, t.c01, t.c02, t.c03, t.c04, t.c05,
                         t.c11, t.c12, t.c13, t.c14, t.c15, t.c22, t.c23, t.c24, t.c25, t.c33, t.c34, t.c35,
                         t.c44, t.c45, t.c55};
#pragma unroll
    for (int k = 0; k < 29; ++k) ts[(int64_t)k * ld + i] = v[k];
}
__device__ __forceinline__ void get_track(const float* __restrict__ ts, int64_t ld, int64_t i, Track& t) {
    float v[29];
#pragma unroll
    for (int k = 0; k < 29; ++k) v[k] = ts[(int64_t)k * ld + i];
    t.x = v[0]; t.y = v[1]; t.z = v[2]; t.px = v[3]; t.py = v[4]; t.pz = v[5]; t.eax = v[6]; t.eay = v[7];
    t.c00 = v[8]; t.c01 = v[9]; t.c02 = v[10]; t.c03 = v[11]; t.c04 = v[12]; t.c05 = v[13];
    t.c11 = v[14]; t.c12 = v[15]; t.c13 = v[16]; t.c14 = v[17]; t.c15 = v[18];
    t.c22 = v[19]; t.c23 = v[20]; t.c24 = v[21]; t.c25 = v[22];
    t.c33 = v[23]; t.c34 = v[24]; t.c35 = v[25]; t.c44 = v[26]; t.c45 = v[27]; t.c55 = v[28];
}

enum : int32_t { FLAG_IDLE = 0, FLAG_AT_LAYER = 1, FLAG_DEAD = 2 };

// Event of candidate i when a call builds several events at once (EventPools); 0 otherwise.
__device__ __forceinline__ int event_of(const EventPools& ev, int64_t i) {
    int e = 0;
    for (int k = 1; k < ev.n; ++k) e += i >= ev.first[k] ? 1 : 0;
    return e;
}

__device__ __forceinline__ bool better(float c, int32_t h, float bc, int32_t bh) {
    return c < bc || (c == bc && h < bh);
}

struct Best {
    float chi2;
    int32_t orig, slot;
};

struct ScanCand {       // what the scan needs of the propagated candidate
    float xn, yn, zn, ec, es, n11, n12, n22;
};

// Full chi2 of the hit in `slot` against the candidate (same Schur form as the update).  DISC: the candidate stands
// on a disc (n11 / n12 / n22 = rr / rt / tt of C').
template <bool DISC = false>
__device__ __forceinline__ void score_hit(const ScanCand& c, const float4* __restrict__ rec, int32_t slot, Best& best) {
    KF_CHECK(slot >= 0);
    const float4* r0 = rec + (int64_t)slot * kRecWords;
    const float4 A = __ldg(r0), B = __ldg(r0 + 1), C = __ldg(r0 + 2);
    Crossing o;
    o.xn = c.xn; o.yn = c.yn; o.zn = c.zn; o.erx = c.ec; o.ery = c.es;
    LocalHit h;
    hit_to_local(o, A.x, A.y, A.z, B.x, B.y, C.x, B.z, C.y, A.w, h);
    float chi2;
    if (DISC ? !chi2_schur_disc(c.n11, c.n12, c.n22, h, chi2) : !chi2_schur(c.n11, c.n12, c.n22, h, chi2)) return;
    const int32_t orig = __float_as_int(B.w);
    if (better(chi2, orig, best.chi2, best.orig)) { best.chi2 = chi2; best.orig = orig; best.slot = slot; }
}


}  // namespace
}  // namespace kf
