// kf_fit.cu -- fused per-layer propagate + update track-fit kernel for sm_100a.
//
// One thread owns one track for the whole layer loop ("one thread per track";
// PAPER.md:129 merged kernels, registers over shared memory): the state, the 21 (then 15) unique
// covariance elements and the Jacobian ingredients never leave registers.  Inputs and outputs
// are element-major SoA (PAPER.md:65, 119 Matriplex), so the data of 32 consecutive tracks is a
// [rows][32] tile of 128-byte lines.
//
// All bulk traffic goes through the TMA unit (cp.async.bulk.tensor, 2-D tensor maps over the
// [planes][ld] arrays), one instruction per tile, issued by one lane:
//   * per warp, a ring of kStages hit tiles [9][32] floats (3 position + 6 covariance planes of
//     one layer -- the only per-layer HBM traffic) is kept kStages layers ahead of the math, each
//     stage guarded by its own mbarrier (complete_tx byte counting);
//   * the seed tile [27][32] is loaded the same way and its shared memory is reused to stage the
//     fitted tracks, which leave through a TMA store (out-of-range columns are clipped by the
//     tensor map, so ragged tails need no special case).
// The math reads shared memory with conflict-free LDS at immediate offsets: no per-thread address
// arithmetic, no registers held for prefetch.  Warps never synchronise with each other.
//
// Algorithmic HBM bytes per track: 113 in (6 + 21 floats, charge, mask) + 120 out (27 floats,
// chi2, nhits, status) + 36 per layer = 593 B at 10 layers.
#include <cuda.h>

#include <atomic>
#include <cstdlib>

#include "kf_internal.h"
#include "kf_tma.cuh"

namespace kf {

namespace {

#ifndef KF_FIT_MIN_BLOCKS
#define KF_FIT_MIN_BLOCKS 5
#endif
#ifndef KF_FIT_STAGES
#define KF_FIT_STAGES 3
#endif

#ifndef KF_FIT_BLOCK
#define KF_FIT_BLOCK 128
#endif
// Batches of at least this many tracks take the pair kernel (two tracks per thread); smaller ones would
// leave SMs idle with 256 tracks per CTA and keep the one-track kernel.
#ifndef KF_PAIR_SMOOTH
#define KF_PAIR_SMOOTH 1
#endif
#ifndef KF_PAIR_MIN_TRACKS
#define KF_PAIR_MIN_TRACKS 151552
#endif
constexpr int kFitBlock = KF_FIT_BLOCK;
constexpr int kWarps = kFitBlock / 32;
constexpr int kStages = KF_FIT_STAGES;           // layers in flight per warp
constexpr int kHitFloats = 9 * 32;               // one hit tile
constexpr int kSeedFloats = 27 * 32;             // seed / result tile
constexpr int kWarpFloats = kStages * kHitFloats + kSeedFloats;
constexpr int kSmemBytes = kWarps * kWarpFloats * 4 + kWarps * (kStages + 1) * 8;

struct FitMaps {
    CUtensorMap hpos, hcov, par, cov, opar, ocov, spar, scov;
};

struct Hit {
    float x, y, z, vxx, vxy, vxz, vyy, vyz, vzz;
};

// One layer for one track.  Returns 0 or the status bit of the failure (track untouched).
// One DISC layer for one track (reading A23): to-plane crossing, general covariance transport, 2-D update in the
// plane.  Compiled only into the kernels specialised for geometries that have discs (GEOM = 2): as a call it
// would force the track into local memory in every kernel that can reach it (measured: the barrel-with-options
// fit went from 0.354 to 0.535 ms per 2 M tracks), inlined it costs registers where it is used only.
__device__ __forceinline__ uint32_t fit_layer_disc(Track& t, float k, float ik, const LayerConst& L, int model, float mass2,
                                                const Bethe& el, const Hit& m, float& chi2) {
    DiscCrossing o;
    const uint32_t reached = helix_to_plane(t, k, ik, L, o);
    if (reached) return reached;
    DiscCov n;
    transport_cov_disc(t, o, k, ms_at_disc(L, model, o, t.pz), mass2, n);
    const float pz_in = t.pz;
    if (model & MODEL_ENERGY_LOSS) {   // reading A21 at a disc: the path factor is 1 / |cos| to the z axis = (p / pT) / |T|
        Eloss e;
        if (!energy_loss_factors(el, L, model, mass2, o.T, o.pt2, o.ipt, pz_in, false, e)) return ST_PROP_FAIL;
        float pz = pz_in;
        apply_energy_loss_disc(e, o, n, pz);
        t.pz = pz;
    }
    Crossing c;                       // what hit_to_local reads of it
    c.xn = o.xn; c.yn = o.yn; c.zn = o.zt; c.erx = o.erx; c.ery = o.ery;
    LocalHit h;
    hit_to_local(c, m.x, m.y, m.z, m.vxx, m.vxy, m.vxz, m.vyy, m.vyz, m.vzz, h);
    float d;
    const uint32_t rc = kalman_update_disc(t, o, n, h, &d);
    if (rc == 0u) chi2 += d;
    else t.pz = pz_in;                // layer skipped: the track stays as it was
    return rc;
}

// ---- the inward refit (reading A18) between surfaces of either kind (geometries with discs, one track per thread)
// One backward step: the layer just left (Lprev, a cylinder or a disc) gives back its energy (A21) and adds its
// scattering noise, then the state goes inward to L and takes L's hit.  first: the state already stands on L
// (update only).  Worked on a copy: any failure leaves the track as it was.
__device__ __forceinline__ uint32_t refit_step_surface(Track& t, float k, float ik, const LayerConst& L, const LayerConst& Lprev,
                                                       int model, float mass2, const Bethe& el, bool first, const Hit& m,
                                                       float* dchi2) {
    Track tb = t;
    if (!first) {
        const float pt2 = tb.px * tb.px + tb.py * tb.py;
        const float ipt = rsqrt_fast(pt2);
        // |cos| that scales the thickness seen (path-length option): to the radial direction on a cylinder, to z on a disc
        const float cos_a = Lprev.type == 1 ? tb.pz * ipt : (tb.eax * tb.px + tb.eay * tb.py) * ipt;
        if (model & MODEL_ENERGY_LOSS) {
            Eloss e;
            if (!energy_loss_factors(el, Lprev, model, mass2, cos_a, pt2, ipt, tb.pz, true, e)) return ST_PROP_FAIL;
            apply_energy_loss(e, tb);
        }
        {   // Highland noise of Lprev at the current momentum (add_process_noise with the surface's own path factor)
            const float q2 = tb.px * tb.px + tb.py * tb.py, pz = tb.pz;
            const float iq = rsqrt_fast(q2);
            const float p2 = q2 + pz * pz;
            float ms = Lprev.ms;
            if (model & MODEL_PATH_LENGTH) {
                if (Lprev.type == 1) {
                    const float f = sqrtf(p2) * rcp_fast(fabsf(pz));
                    const float lg = 1.0f + 0.038f * (Lprev.ln_t + __logf(f));
                    ms = Lprev.ms0 * f * lg * lg;
                } else {
                    ms = layer_ms<float>(Lprev, model, (tb.eax * tb.px + tb.eay * tb.py) * iq, p2, iq);
                }
            }
            const float ip2 = rcp_fast(p2);
            const float th2 = ms * (p2 + mass2) * ip2 * ip2;
            const float qc = th2 * p2 * iq;
            tb.c33 += th2 * pz * pz;
            tb.c35 -= qc * pz;
            tb.c44 += th2 * p2;
            tb.c55 += qc * (p2 * iq);
        }
    }
    uint32_t rc;
    if (L.type == 1) {
        DiscCrossing o;
        DiscCov n;
        if (first) {
            const float pt2 = tb.px * tb.px + tb.py * tb.py;
            const float ipt = rsqrt_fast(pt2);
            o.xn = tb.x; o.yn = tb.y; o.zt = tb.z; o.pxn = tb.px; o.pyn = tb.py;
            o.erx = tb.eax; o.ery = tb.eay; o.elx = tb.px * ipt; o.ely = tb.py * ipt;
            o.T = tb.pz * ipt; o.pt2 = pt2; o.ipt = ipt;
            n.rr = tb.c00; n.rt = tb.c01; n.tt = tb.c11;
            n.r3 = tb.c03; n.r4 = tb.c04; n.r5 = tb.c05; n.t3 = tb.c13; n.t4 = tb.c14; n.t5 = tb.c15;
            n.n33 = tb.c33; n.n34 = tb.c34; n.n35 = tb.c35; n.n44 = tb.c44; n.n45 = tb.c45; n.n55 = tb.c55;
        } else {
            const uint32_t reached = helix_to_plane<true>(tb, k, ik, L, o);
            if (reached) return reached;
            transport_cov_disc(tb, o, k, 0.0f, mass2, n);
        }
        Crossing c;
        c.xn = o.xn; c.yn = o.yn; c.zn = o.zt; c.erx = o.erx; c.ery = o.ery;
        LocalHit h;
        hit_to_local(c, m.x, m.y, m.z, m.vxx, m.vxy, m.vxz, m.vyy, m.vyz, m.vzz, h);
        rc = kalman_update_disc(tb, o, n, h, dchi2);
    } else {
        Crossing o;
        PropCov n;
        if (first) crossing_in_place(tb, o, n);
        else {
            const uint32_t reached = reach_layer<true, true>(tb, k, ik, L, o);
            if (reached) return reached;
            transport_cov<false>(tb, o, 0.0f, mass2, n);       // (the state may come from a disc: general covariance)
        }
        LocalHit h;
        hit_to_local(o, m.x, m.y, m.z, m.vxx, m.vxy, m.vxz, m.vyy, m.vyz, m.vzz, h);
        rc = kalman_update(tb, o, n, h, dchi2);
    }
    if (rc == 0u) t = tb;
    return rc;
}

// GEOM 0: the paper's toy detector (options compiled out); 1: the options of readings A20 / A21 on barrels;
// 2: the same plus endcap discs (reading A23).
template <bool RADIAL_NULL, int GEOM = 1>
__device__ __forceinline__ uint32_t fit_layer(Track& t, float k, float ik, const LayerConst& L, int model,
                                              float mass2, const Bethe& el, const Hit& m, float& chi2) {
    if constexpr (GEOM == 2) {
        if (L.type == 1) return fit_layer_disc(t, k, ik, L, model, mass2, el, m, chi2);
    }
    Crossing o;
    const uint32_t reached = reach_layer<false, GEOM != 0>(t, k, ik, L, o);
    if (reached) return reached;
    PropCov n;
    transport_cov<RADIAL_NULL>(t, o, ms_at_crossing(L, model, o, t.pz), mass2, n);
    const float pz_in = t.pz;
    if constexpr (GEOM != 0) {
        if (model & MODEL_ENERGY_LOSS) {   // reading A21: on arrival, after C' = F C F^T + Q
            Eloss e;
            if (!energy_loss_factors(el, L, model, mass2, o.erx * o.elx + o.ery * o.ely, o.pt2, o.ipt, pz_in, false, e))
                return ST_PROP_FAIL;
            float pz = pz_in;
            apply_energy_loss(e, o, n, pz);
            t.pz = pz;
        }
    }
    LocalHit h;
    hit_to_local(o, m.x, m.y, m.z, m.vxx, m.vxy, m.vxz, m.vyy, m.vyz, m.vzz, h);
    float d;
    const uint32_t rc = kalman_update(t, o, n, h, &d);
    if (rc == 0u) chi2 += d;
    else if constexpr (GEOM != 0) t.pz = pz_in;   // layer skipped: the track stays as it was
    return rc;
}

// Seed / result tile [27][32] in shared memory <-> registers (p = &tile[0][lane]).
__device__ __forceinline__ void track_from_tile(Track& t, const float* p) {
    t.x = p[0];         t.y = p[32];        t.z = p[64];        t.px = p[96];       t.py = p[128];      t.pz = p[160];
    t.c00 = p[192];     t.c01 = p[224];     t.c02 = p[256];     t.c03 = p[288];     t.c04 = p[320];     t.c05 = p[352];
    t.c11 = p[384];     t.c12 = p[416];     t.c13 = p[448];     t.c14 = p[480];     t.c15 = p[512];
    t.c22 = p[544];     t.c23 = p[576];     t.c24 = p[608];     t.c25 = p[640];
    t.c33 = p[672];     t.c34 = p[704];     t.c35 = p[736];
    t.c44 = p[768];     t.c45 = p[800];
    t.c55 = p[832];
    t.eax = 1.0f;
    t.eay = 0.0f;
}
__device__ __forceinline__ void track_to_tile(const Track& t, float* p) {
    p[0] = t.x;         p[32] = t.y;        p[64] = t.z;        p[96] = t.px;       p[128] = t.py;      p[160] = t.pz;
    p[192] = t.c00;     p[224] = t.c01;     p[256] = t.c02;     p[288] = t.c03;     p[320] = t.c04;     p[352] = t.c05;
    p[384] = t.c11;     p[416] = t.c12;     p[448] = t.c13;     p[480] = t.c14;     p[512] = t.c15;
    p[544] = t.c22;     p[576] = t.c23;     p[608] = t.c24;     p[640] = t.c25;
    p[672] = t.c33;     p[704] = t.c34;     p[736] = t.c35;
    p[768] = t.c44;     p[800] = t.c45;
    p[832] = t.c55;
}

// MODE 2: the filtered state of layer l in the local frame -> the per-layer arrays (coalesced 4-byte stores: lane =
// track).  Planes: par 0..5 = x y z px py pz; cov 0..14 = c11 c12 c13 c14 c15 c22 c23 c24 c25 c33 c34 c35 c44 c45
// c55, 15..16 = eax eay (17..20 are written by the backward pass only).
// (type 1: the state stands on a disc, reading A23 -- its live coordinates are (r, t | b1 b2 c) and the first nine
// planes hold rr rt r3 r4 r5 | tt t3 t4 t5 instead of tt tz t3 t4 t5 | zz z3 z4 z5.)
__device__ __forceinline__ void store_layer_state(const Track& t, const FitArgs& a, int l, int64_t i, int type = 0) {
    float* p = a.lpar + (int64_t)l * 6 * a.ld_l + i;
    float* c = a.lcov + (int64_t)l * 21 * a.ld_l + i;
    const int64_t ld = a.ld_l;
    p[0] = t.x; p[ld] = t.y; p[2 * ld] = t.z; p[3 * ld] = t.px; p[4 * ld] = t.py; p[5 * ld] = t.pz;
    if (type == 1) {
        c[0] = t.c00; c[ld] = t.c01; c[2 * ld] = t.c03; c[3 * ld] = t.c04; c[4 * ld] = t.c05;
        c[5 * ld] = t.c11; c[6 * ld] = t.c13; c[7 * ld] = t.c14; c[8 * ld] = t.c15;
    } else {
        c[0] = t.c11; c[ld] = t.c12; c[2 * ld] = t.c13; c[3 * ld] = t.c14; c[4 * ld] = t.c15;
        c[5 * ld] = t.c22; c[6 * ld] = t.c23; c[7 * ld] = t.c24; c[8 * ld] = t.c25;
    }
    c[9 * ld] = t.c33; c[10 * ld] = t.c34; c[11 * ld] = t.c35;
    c[12 * ld] = t.c44; c[13 * ld] = t.c45; c[14 * ld] = t.c55;
    c[15 * ld] = t.eax; c[16 * ld] = t.eay;
}

// SMOOTH = false: forward fit (rows a1-a7).  SMOOTH = true: forward fit, then the inward refit of reading
// A18 over the same hits (streamed again through the same ring, outermost layer first); two results.
// GEOM = false: the paper's toy detector (unbounded barrels, flat material): the options of reading A20
// are compiled out, so the headline kernel carries none of their cost.
// MODE 0: forward fit.  MODE 1 (= SMOOTH below): forward fit + the inward refit of reading A18.  MODE 2: forward fit
// that also leaves the FILTERED state of every used layer, in the local frame, in the per-layer arrays of
// kf_fit_tracks_smooth (23 floats per track and layer: the input of the backward RTS pass, kf_smooth.cu).
template <int MODE, int GEOM>
__global__ void __launch_bounds__(kFitBlock, MODE == 1 || GEOM == 2 ? 4 : KF_FIT_MIN_BLOCKS)
fit_kernel(const __grid_constant__ FitParams P, const __grid_constant__ FitMaps M, const FitArgs a) {
    constexpr bool SMOOTH = MODE == 1;
    const int model = GEOM != 0 ? P.model : 0;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    const int wid = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);   // warp-uniform by construction
    const int64_t i0 = (int64_t)blockIdx.x * kFitBlock + wid * 32;  // first track of this warp
    if (i0 >= a.n) return;                                          // whole warp out of range
    const int L = P.n_layers;
    float* wbase = reinterpret_cast<float*>(smem_raw) + wid * kWarpFloats;
    float* seed_tile = wbase + kStages * kHitFloats;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + kWarps * kWarpFloats * 4) + wid * (kStages + 1);
    const uint32_t hit0 = smem_u32(wbase), seed0 = smem_u32(seed_tile), bar0 = smem_u32(bars);
    const int col = (int)i0;

    if (elect_one()) {
#pragma unroll
        for (int s = 0; s <= kStages; ++s) mbar_init(bar0 + 8u * s, 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        // seed tile first, then the first kStages layers of hits
        mbar_expect_tx(bar0 + 8u * kStages, kSeedFloats * 4);
        tma_load_2d(seed0, &M.par, col, 0, bar0 + 8u * kStages);
        tma_load_2d(seed0 + 6 * 128, &M.cov, col, 0, bar0 + 8u * kStages);
#pragma unroll
        for (int s = 0; s < kStages; ++s)
            if (s < (SMOOTH ? 2 * L : L)) {   // fewer layers than stages: the ring's first round already turns back
                const int ls = s < L ? s : 2 * L - 1 - s;
                mbar_expect_tx(bar0 + 8u * s, kHitFloats * 4);
                tma_load_2d(hit0 + s * (kHitFloats * 4), &M.hpos, col, 3 * ls, bar0 + 8u * s);
                tma_load_2d(hit0 + s * (kHitFloats * 4) + 3 * 128, &M.hcov, col, 6 * ls, bar0 + 8u * s);
            }
    }
    __syncwarp();

    const bool valid = lane < a.n - i0;
    const int64_t i = valid ? i0 + lane : a.n - 1;  // idle lanes shadow the last track, store nothing
    const int q = a.q[i];
    const uint32_t mask = a.mask ? __ldg(a.mask + i) : 0xffffffffu;
    const bool good_q = (q == 1) | (q == -1);
    const float k = (float)q * P.k0, ik = (float)q * P.inv_k0;
    Track t;
    mbar_wait(bar0 + 8u * kStages, 0u);
    track_from_tile(t, seed_tile + lane);
    if (good_q) enter_local_frame(t);
    float chi2 = 0.0f;
    int nh = 0;
    uint32_t st = 0u;
    bool started = false;  // false: general 6x6 covariance; true: its radial row is identically zero
    uint32_t phase = 0u;   // bit s = parity the next wait on stage s expects
    uint32_t used = 0u;    // layers the forward fit used
    for (int l = 0; l < L; ++l) {
        const int s = l % kStages;
        if constexpr (SMOOTH) { mbar_wait(bar0 + 8u * s, (phase >> s) & 1u); phase ^= 1u << s; }
        else mbar_wait(bar0 + 8u * s, (uint32_t)(l / kStages) & 1u);
        const float* tp = wbase + s * kHitFloats + lane;
        Hit m;
        m.x = tp[0];         m.y = tp[32];        m.z = tp[64];
        m.vxx = tp[96];      m.vxy = tp[128];     m.vxz = tp[160];
        m.vyy = tp[192];     m.vyz = tp[224];     m.vzz = tp[256];
        __syncwarp();        // every lane has issued its reads of this stage
        if (good_q && ((mask >> l) & 1u)) {
            uint32_t rc;
            if (started) rc = fit_layer<true, GEOM>(t, k, ik, P.layer[l], model, P.mass2, P.el, m, chi2);
            else rc = fit_layer<false, GEOM>(t, k, ik, P.layer[l], model, P.mass2, P.el, m, chi2);
            st |= rc;
            if (rc == 0u) {
                nh += 1; used |= 1u << l;
                started = GEOM != 2 || P.layer[l].type == 0;   // after a disc the z row is the null one, not the radial row
                if constexpr (MODE == 2) { if (valid) store_layer_state(t, a, l, i, GEOM == 2 ? P.layer[l].type : 0); }
            }
        }
        // The hit values have been consumed by the math above, so the stage can be handed back to the
        // TMA unit (write-after-read across the generic and async proxies needs no fence once the
        // reads have completed; the refill still lands kStages - 1 layers ahead of its use).
        // In SMOOTH mode the ring runs on into the backward pass: step L + j carries layer L - 1 - j.
        const int nxt = l + kStages;
        if (nxt < (SMOOTH ? 2 * L : L)) {
            const int ln = nxt < L ? nxt : 2 * L - 1 - nxt;
            __syncwarp();
            if (elect_one()) {
                mbar_expect_tx(bar0 + 8u * s, kHitFloats * 4);
                tma_load_2d(hit0 + s * (kHitFloats * 4), &M.hpos, col, 3 * ln, bar0 + 8u * s);
                tma_load_2d(hit0 + s * (kHitFloats * 4) + 3 * 128, &M.hcov, col, 6 * ln, bar0 + 8u * s);
            }
        }
    }
    if (!good_q) st = ST_BAD_CHARGE;
    if constexpr (SMOOTH) {
        // ---- forward result out (a copy goes back to the global frame; t stays local for the refit)
        if (good_q && nh > 0) {
            Track g = t;
            leave_local_frame(g);
            track_to_tile(g, seed_tile + lane);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        const bool fstorer = elect_one();
        if (fstorer) {
            tma_store_2d(&M.opar, col, 0, seed0);
            tma_store_2d(&M.ocov, col, 0, seed0 + 6 * 128);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        if (valid) { a.chi2[i] = chi2; a.nhits[i] = nh; a.status[i] = st; }
        // ---- inward refit (reading A18)
        float schi2 = 0.0f;
        int l_prev = 0;
        int nb = 0;
        uint32_t sst = 0u;
        bool first = true;
        if (used) {
            scale_cov(t, a.kappa);
            if constexpr (GEOM == 2) {      // a result standing on a disc has its radial row live (and no z row)
                t.c00 *= a.kappa; t.c01 *= a.kappa; t.c02 *= a.kappa; t.c03 *= a.kappa; t.c04 *= a.kappa; t.c05 *= a.kappa;
            }
        }
        for (int j = 0; j < L; ++j) {
            const int l = L - 1 - j, step = L + j, s = step % kStages;
            mbar_wait(bar0 + 8u * s, (phase >> s) & 1u);
            phase ^= 1u << s;
            const float* tp = wbase + s * kHitFloats + lane;
            Hit m;
            m.x = tp[0];         m.y = tp[32];        m.z = tp[64];
            m.vxx = tp[96];      m.vxy = tp[128];     m.vxz = tp[160];
            m.vyy = tp[192];     m.vyz = tp[224];     m.vzz = tp[256];
            __syncwarp();
            if ((used >> l) & 1u) {
                float d;
                uint32_t rc;
                if constexpr (GEOM == 2) rc = refit_step_surface(t, k, ik, P.layer[l], P.layer[l_prev], model, P.mass2, P.el, first, m, &d);
                else rc = refit_step<GEOM != 0>(t, k, ik, P.layer[l], P.layer[l_prev], model, P.mass2, P.el, first,
                                                     m.x, m.y, m.z, m.vxx, m.vxy, m.vxz, m.vyy, m.vyz, m.vzz, &d);
                if (rc == 0u) { schi2 += d; nb += 1; first = false; l_prev = l; }
                else sst |= rc;
            }
            const int nxt = step + kStages;
            if (nxt < 2 * L) {
                const int ln = 2 * L - 1 - nxt;
                __syncwarp();
                if (elect_one()) {
                    mbar_expect_tx(bar0 + 8u * s, kHitFloats * 4);
                    tma_load_2d(hit0 + s * (kHitFloats * 4), &M.hpos, col, 3 * ln, bar0 + 8u * s);
                    tma_load_2d(hit0 + s * (kHitFloats * 4) + 3 * 128, &M.hcov, col, 6 * ln, bar0 + 8u * s);
                }
            }
        }
        // the forward tile must have left shared memory before the smoothed one overwrites it
        if (fstorer) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        __syncwarp();
        if (good_q && used) {
            leave_local_frame(t);
            track_to_tile(t, seed_tile + lane);
        }   // else the tile still holds the forward result = the input
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        const bool sstorer = elect_one();
        if (sstorer) {
            tma_store_2d(&M.spar, col, 0, seed0);
            tma_store_2d(&M.scov, col, 0, seed0 + 6 * 128);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        if (valid) { a.schi2[i] = schi2; a.snhits[i] = nb; a.sstatus[i] = sst; }
        if (sstorer) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        return;
    }
    if (good_q && nh > 0) {
        leave_local_frame(t);
        track_to_tile(t, seed_tile + lane);
    }   // else: bad charge or nothing fitted -- the seed tile still holds the input, bit-exact
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
    const bool storer = elect_one();
    if (storer) {
        tma_store_2d(&M.opar, col, 0, seed0);
        tma_store_2d(&M.ocov, col, 0, seed0 + 6 * 128);
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    if (valid) {
        a.chi2[i] = chi2;
        a.nhits[i] = nh;
        a.status[i] = st;
        if constexpr (MODE == 2) a.used[i] = used;
    }
    if (storer) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");  // smem must outlive the store
}

// ---- pair kernel: two tracks per thread in packed fp32x2 registers (kf_pair.cuh) ---------------------------
// Same pipeline as fit_kernel<false, false> with tiles 64 tracks wide: lane j of a warp owns tracks
// 2j (component x) and 2j + 1 (component y) of the tile, reads them as one 8-byte word per row and runs the
// arithmetic of kf_math.cuh on F = f2, i.e. one FFMA2 / FMUL2 / FADD2 where the one-track kernel issues two
// instructions.  Forward fit of the toy detector only (no smoother, no geometry options).
// One warp (64 tracks) per CTA, 12 CTAs per SM: the same 12 resident warps as 3 CTAs of 4 warps (168 registers), but
// a batch is cut into units of 64 tracks instead of 256, so mid-size batches fill the SMs evenly (measured in one
// run, 2 M tracks: 0.295 ms against 0.303 for 128 x 3; register caps 160 / 152 / 144 / 136 for 13 - 15 resident
// warps: 0.306 / 0.309 / 0.322 / 0.364 -- the spills cost more than the extra warps give; 4 or 5 ring stages: 0.299).
#ifndef KF_PAIR_BLOCK
#define KF_PAIR_BLOCK 32
#endif
#ifndef KF_PAIR_MIN_BLOCKS
#define KF_PAIR_MIN_BLOCKS 12
#endif
#ifndef KF_PAIR_SMOOTH_MIN_BLOCKS
#define KF_PAIR_SMOOTH_MIN_BLOCKS 12
#endif
constexpr int kPairBlock = KF_PAIR_BLOCK;
constexpr int kPairWarps = kPairBlock / 32;
constexpr int kPairTile = 64;                      // tracks per warp
constexpr int kHit2Floats = 9 * kPairTile;
constexpr int kSeed2Floats = 27 * kPairTile;
// One parked track (29 values + chi2) per lane (ragged pairs) lives INSIDE the seed / result tile, which is idle
// between the load of the seeds and the staging of the results (30 x 32 of its 27 x 64 floats): no shared memory of
// its own, so a deeper hit ring or more resident warps fit.  Price: a track that ends with nothing fitted can no
// longer take its input back from the tile and re-reads it from global memory (restore_unfitted).
constexpr int kPark2Floats = 30 * 32;
static_assert(kPark2Floats <= kSeed2Floats, "the park area lives inside the seed tile");
__host__ __device__ constexpr int warp2_floats(bool) { return kStages * kHit2Floats + kSeed2Floats; }
constexpr int smem2_bytes(bool smooth) { return kPairWarps * warp2_floats(smooth) * 4 + kPairWarps * (kStages + 1) * 8; }

struct Hit2 {
    f2 x, y, z, vxx, vxy, vxz, vyy, vyz, vzz;
};

// One layer for a pair of tracks that both have a hit on it.  Returns true if both went through; on any
// failure the pair is untouched and the caller takes the two tracks one at a time (fit_layer_one_of_pair).
// The hit pair is read from its shared-memory stage only where the residual is formed, after the covariance
// transport, so that it does not occupy 18 registers through the most register-hungry part of the layer.
__device__ __forceinline__ void load_hit_pair(Hit2& m, const float2* tp) {
    constexpr int R = kPairTile / 2;
    m.x = f2(tp[0]);           m.y = f2(tp[R]);           m.z = f2(tp[2 * R]);
    m.vxx = f2(tp[3 * R]);     m.vxy = f2(tp[4 * R]);     m.vxz = f2(tp[5 * R]);
    m.vyy = f2(tp[6 * R]);     m.vyz = f2(tp[7 * R]);     m.vzz = f2(tp[8 * R]);
}

template <bool RADIAL_NULL>
__device__ __forceinline__ bool fit_layer_pair(Track2& t, f2 k, f2 ik, const LayerConst& L, float mass2,
                                               const float2* tp, f2& chi2) {
    Crossing2 o;
    if (!all_of(helix_to_radius(t, k, ik, L, o))) return false;
    PropCov2 n;
    transport_cov<RADIAL_NULL>(t, o, f2(L.ms), mass2, n);
    Hit2 m;
    load_hit_pair(m, tp);
    LocalHit2 h;
    hit_to_local(o, m.x, m.y, m.z, m.vxx, m.vxy, m.vxz, m.vyy, m.vyz, m.vzz, h);
    f2 d;
    const u2 rc = kalman_update(t, o, n, h, &d);
    if ((rc.x | rc.y) != 0u) return false;
    chi2 = chi2 + d;
    return true;
}

// A layer only ONE track of the pair has a hit on: the idle one's 29 values (and its chi2) are parked in shared
// memory and its half of the pair becomes a SHADOW of the active track (same state, same charge, same hit), so
// that the pair arithmetic passes exactly when the active track's does; afterwards the idle half is put back.
// (A harmless hit alone is not enough: a track that has stopped short of the layer -- the usual reason for a
// ragged pair -- cannot be propagated there, and its failure would send the pair down the one-track path on
// every remaining layer.)
#define KF_TRACK_FIELDS(X)                                                                              \
    X(x) X(y) X(z) X(px) X(py) X(pz) X(eax) X(eay) X(c00) X(c01) X(c02) X(c03) X(c04) X(c05) X(c11) X(c12) \
    X(c13) X(c14) X(c15) X(c22) X(c23) X(c24) X(c25) X(c33) X(c34) X(c35) X(c44) X(c45) X(c55)
template <int C>
__device__ __forceinline__ void park_component(const Track2& t, float* scr) {
    int r = 0;
#define KF_PARK(f) scr[32 * r++] = C ? t.f.v.y : t.f.v.x;
    KF_TRACK_FIELDS(KF_PARK)
#undef KF_PARK
}
template <int C>
__device__ __forceinline__ void shadow_component(Track2& t) {   // component C := the other one
#define KF_SHADOW(f) if (C) t.f.v.y = t.f.v.x; else t.f.v.x = t.f.v.y;
    KF_TRACK_FIELDS(KF_SHADOW)
#undef KF_SHADOW
}
// The idle track's slot of the hit stage := the active track's hit.
__device__ __forceinline__ void shadow_hit(const float2* tp, int idle) {
    float* hp = const_cast<float*>(reinterpret_cast<const float*>(tp));   // this lane's two slots
#pragma unroll
    for (int r = 0; r < 9; ++r) hp[r * kPairTile + idle] = hp[r * kPairTile + (idle ^ 1)];
    // ordered before the TMA refill of this stage (issued by another lane after a __syncwarp)
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
template <int C>
__device__ __forceinline__ void unpark_component(Track2& t, const float* scr) {
    int r = 0;
#define KF_UNPARK(f) { const float v = scr[32 * r++]; if (C) t.f.v.y = v; else t.f.v.x = v; }
    KF_TRACK_FIELDS(KF_UNPARK)
#undef KF_UNPARK
}

// Slow path (a track of the pair fails on the layer): component c alone,
// through the one-track arithmetic.  Kept out of line so that it costs the pair path no registers.
__device__ __noinline__ uint32_t fit_layer_one_of_pair(Track2& t, int c, float k, float ik, const LayerConst& L,
                                                       float mass2, const Hit2& m, f2& chi2, bool started) {
    Track ts;
    Hit mh;
    float ch = 0.0f;
#define KF_GET(f) ts.f = c ? t.f.v.y : t.f.v.x;
    KF_TRACK_FIELDS(KF_GET)
#undef KF_GET
#define KF_GETH(f) mh.f = c ? m.f.v.y : m.f.v.x;
    KF_GETH(x) KF_GETH(y) KF_GETH(z) KF_GETH(vxx) KF_GETH(vxy) KF_GETH(vxz) KF_GETH(vyy) KF_GETH(vyz) KF_GETH(vzz)
#undef KF_GETH
    const Bethe none = {0.0f, 0.0f, 0.0f, 0.0f};
    const uint32_t rc = started ? fit_layer<true, 0>(ts, k, ik, L, 0, mass2, none, mh, ch)
                                : fit_layer<false, 0>(ts, k, ik, L, 0, mass2, none, mh, ch);
    if (rc != 0u) return rc;
#define KF_PUT(f) if (c) t.f.v.y = ts.f; else t.f.v.x = ts.f;
    KF_TRACK_FIELDS(KF_PUT)
#undef KF_PUT
    if (c) chi2.v.y += ch; else chi2.v.x += ch;
    return 0u;
}

#define KF_TRACK_ROWS(X)                                                                                   \
    X(0, x) X(1, y) X(2, z) X(3, px) X(4, py) X(5, pz) X(6, c00) X(7, c01) X(8, c02) X(9, c03) X(10, c04)   \
    X(11, c05) X(12, c11) X(13, c12) X(14, c13) X(15, c14) X(16, c15) X(17, c22) X(18, c23) X(19, c24)      \
    X(20, c25) X(21, c33) X(22, c34) X(23, c35) X(24, c44) X(25, c45) X(26, c55)

// One backward step (reading A18) for component c of a pair, out of line like fit_layer_one_of_pair.
__device__ __noinline__ uint32_t refit_step_one_of_pair(Track2& t, int c, float k, float ik, const LayerConst& L,
                                                        const LayerConst& Lprev, float mass2, bool first,
                                                        const Hit2& m, f2& schi2) {
    Track ts;
    Hit mh;
    float d = 0.0f;
#define KF_GET(f) ts.f = c ? t.f.v.y : t.f.v.x;
    KF_TRACK_FIELDS(KF_GET)
#undef KF_GET
#define KF_GETH(f) mh.f = c ? m.f.v.y : m.f.v.x;
    KF_GETH(x) KF_GETH(y) KF_GETH(z) KF_GETH(vxx) KF_GETH(vxy) KF_GETH(vxz) KF_GETH(vyy) KF_GETH(vyz) KF_GETH(vzz)
#undef KF_GETH
    const Bethe none = {0.0f, 0.0f, 0.0f, 0.0f};
    const uint32_t rc = refit_step<false>(ts, k, ik, L, Lprev, 0, mass2, none, first, mh.x, mh.y, mh.z, mh.vxx, mh.vxy,
                                          mh.vxz, mh.vyy, mh.vyz, mh.vzz, &d);
    if (rc != 0u) return rc;
#define KF_PUT(f) if (c) t.f.v.y = ts.f; else t.f.v.x = ts.f;
    KF_TRACK_FIELDS(KF_PUT)
#undef KF_PUT
    if (c) schi2.v.y += d; else schi2.v.x += d;
    return 0u;
}
#undef KF_TRACK_FIELDS

// Result pair -> the warp's [27][64] tile: both tracks with one 8-byte store per row, or only the one that
// has a result (the other's columns keep what the tile holds).
__device__ __forceinline__ void pair_to_tile(const Track2& t, float* tile, int lane, mask2 done) {
    if (all_of(done)) {
        float2* p = reinterpret_cast<float2*>(tile) + lane;
#define KF_STORE_ROW(r, f) p[(r) * (kPairTile / 2)] = t.f.v;
        KF_TRACK_ROWS(KF_STORE_ROW)
#undef KF_STORE_ROW
    } else {
        float* p = tile + 2 * lane + (done.y ? 1 : 0);
#define KF_STORE_ONE(r, f) p[(r) * kPairTile] = done.y ? t.f.v.y : t.f.v.x;
        KF_TRACK_ROWS(KF_STORE_ONE)
#undef KF_STORE_ONE
    }
}

// A track with nothing fitted goes back as it came.  Its columns of the seed tile may have served as park area in
// the meantime, so the input is read again from global memory (rare: bad charge, empty mask, nothing reached).
__device__ __forceinline__ void restore_unfitted(float* tile, const FitArgs& a, int lane, int64_t ix, int64_t iy, mask2 which) {
    if (none_of(which)) return;
#pragma unroll 1
    for (int c = 0; c < 2; ++c) {
        if (!(c ? which.y : which.x)) continue;
        const int64_t i = c ? iy : ix;
        float* p = tile + 2 * lane + c;
#pragma unroll 1
        for (int r = 0; r < 27; ++r) p[r * kPairTile] = r < 6 ? a.par[r * a.ld_in + i] : a.cov[(r - 6) * a.ld_in + i];
    }
}

// MODE 2: filtered state of layer l of one or both tracks of the pair -> the per-layer arrays (see
// store_layer_state): both with one 8-byte store per plane (tracks 2j, 2j + 1 are neighbours; ld is a multiple of
// 4 and the tile starts at a multiple of 64, so the address is 8-byte aligned), one alone with 4-byte stores.
__device__ __forceinline__ void store_layer_state_pair(const Track2& t, const FitArgs& a, int l, int64_t ix, int64_t iy,
                                                       mask2 which) {
    if (none_of(which)) return;
    const int64_t ld = a.ld_l;
    float* p = a.lpar + (int64_t)l * 6 * ld;
    float* c = a.lcov + (int64_t)l * 21 * ld;
#define KF_LAYER_PLANES(X)                                                                                        \
    X(p, 0, x) X(p, 1, y) X(p, 2, z) X(p, 3, px) X(p, 4, py) X(p, 5, pz)                                          \
    X(c, 0, c11) X(c, 1, c12) X(c, 2, c13) X(c, 3, c14) X(c, 4, c15) X(c, 5, c22) X(c, 6, c23) X(c, 7, c24)      \
    X(c, 8, c25) X(c, 9, c33) X(c, 10, c34) X(c, 11, c35) X(c, 12, c44) X(c, 13, c45) X(c, 14, c55)              \
    X(c, 15, eax) X(c, 16, eay)
    if (all_of(which)) {
#define KF_ST2(base, r, f) *reinterpret_cast<float2*>(base + (r) * ld + ix) = t.f.v;
        KF_LAYER_PLANES(KF_ST2)
#undef KF_ST2
    } else if (which.x) {
#define KF_STX(base, r, f) base[(r) * ld + ix] = t.f.v.x;
        KF_LAYER_PLANES(KF_STX)
#undef KF_STX
    } else {
#define KF_STY(base, r, f) base[(r) * ld + iy] = t.f.v.y;
        KF_LAYER_PLANES(KF_STY)
#undef KF_STY
    }
#undef KF_LAYER_PLANES
}

// SMOOTH = true: the forward fit, then the inward refit of reading A18 over the same hits (ring runs on,
// outermost layer first), as in fit_kernel<1, 0>.
template <int MODE>
#ifdef KF_PAIR_MAXNREG
__global__ void __maxnreg__(KF_PAIR_MAXNREG)       // tuning variants: a register cap instead of a CTA count
#else
__global__ void __launch_bounds__(kPairBlock, MODE == 1 ? KF_PAIR_SMOOTH_MIN_BLOCKS : KF_PAIR_MIN_BLOCKS)
#endif
fit_pair_kernel(const __grid_constant__ FitParams P, const __grid_constant__ FitMaps M, const FitArgs a) {
    constexpr bool SMOOTH = MODE == 1;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    const int wid = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    const int64_t i0 = ((int64_t)blockIdx.x * kPairWarps + wid) * kPairTile;  // first track of this warp
    if (i0 >= a.n) return;
    const int L = P.n_layers;
    constexpr int kWarp2Floats = warp2_floats(SMOOTH);
    float* wbase = reinterpret_cast<float*>(smem_raw) + wid * kWarp2Floats;
    float* seed_tile = wbase + kStages * kHit2Floats;
    float* park = seed_tile + lane;        // (inside the seed tile: see kPark2Floats)
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + kPairWarps * kWarp2Floats * 4) + wid * (kStages + 1);
    const uint32_t hit0 = smem_u32(wbase), seed0 = smem_u32(seed_tile), bar0 = smem_u32(bars);
    const int col = (int)i0;
    constexpr uint32_t kRowBytes = kPairTile * 4;

    if (elect_one()) {
#pragma unroll
        for (int s = 0; s <= kStages; ++s) mbar_init(bar0 + 8u * s, 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        mbar_expect_tx(bar0 + 8u * kStages, kSeed2Floats * 4);
        tma_load_2d(seed0, &M.par, col, 0, bar0 + 8u * kStages);
        tma_load_2d(seed0 + 6 * kRowBytes, &M.cov, col, 0, bar0 + 8u * kStages);
#pragma unroll
        for (int s = 0; s < kStages; ++s)
            if (s < (SMOOTH ? 2 * L : L)) {   // fewer layers than stages: the ring's first round already turns back
                const int ls = s < L ? s : 2 * L - 1 - s;
                mbar_expect_tx(bar0 + 8u * s, kHit2Floats * 4);
                tma_load_2d(hit0 + s * (kHit2Floats * 4), &M.hpos, col, 3 * ls, bar0 + 8u * s);
                tma_load_2d(hit0 + s * (kHit2Floats * 4) + 3 * kRowBytes, &M.hcov, col, 6 * ls, bar0 + 8u * s);
            }
    }
    __syncwarp();

    // component c of this lane = track i0 + 2 lane + c; a component beyond n shadows the last track and stores nothing
    const int64_t left = a.n - i0;
    const mask2 valid = {2 * lane < left, 2 * lane + 1 < left};
    const int64_t ix = valid.x ? i0 + 2 * lane : a.n - 1, iy = valid.y ? i0 + 2 * lane + 1 : a.n - 1;
    const int qx = a.q[ix], qy = a.q[iy];
    const uint32_t mx = a.mask ? __ldg(a.mask + ix) : 0xffffffffu, my = a.mask ? __ldg(a.mask + iy) : 0xffffffffu;
    const mask2 good_q = {(qx == 1) || (qx == -1), (qy == 1) || (qy == -1)};
    const f2 k((float)qx * P.k0, (float)qy * P.k0), ik((float)qx * P.inv_k0, (float)qy * P.inv_k0);
    Track2 t;
    mbar_wait(bar0 + 8u * kStages, 0u);
    {
        const float2* p = reinterpret_cast<const float2*>(seed_tile) + lane;
#define KF_LOAD_ROW(r, f) t.f = f2(p[(r) * (kPairTile / 2)]);
        KF_TRACK_ROWS(KF_LOAD_ROW)
#undef KF_LOAD_ROW
        t.eax = f2(1.0f);
        t.eay = f2(0.0f);
    }
    // a component with nothing to fit (bad charge, beyond n) takes no part
    const mask2 live = {valid.x && good_q.x, valid.y && good_q.y};
    if (!none_of(live)) enter_local_frame(t);
    f2 chi2(0.0f);
    int nhx = 0, nhy = 0;
    u2 st = {0u, 0u};
    mask2 started = {false, false};   // false: general 6x6 covariance; true: its radial row is identically zero
    uint32_t phase = 0u;              // SMOOTH: bit s = parity the next wait on stage s expects
    uint32_t usedx = 0u, usedy = 0u;  // layers the forward fit used
    for (int l = 0; l < L; ++l) {
        const int s = l % kStages;
        if constexpr (SMOOTH) { mbar_wait(bar0 + 8u * s, (phase >> s) & 1u); phase ^= 1u << s; }
        else mbar_wait(bar0 + 8u * s, (uint32_t)(l / kStages) & 1u);
        const float2* tp = reinterpret_cast<const float2*>(wbase + s * kHit2Floats) + lane;
        const mask2 want = {live.x && ((mx >> l) & 1u), live.y && ((my >> l) & 1u)};
        bool both = false;
        // (the smoother kernel leaves ragged pairs to the one-track path: see warp2_floats; launch_fit therefore
        // takes it only for batches whose tracks all have every hit)
        if (SMOOTH ? all_of(want) : !none_of(want)) {
            const bool ragged = !SMOOTH && !all_of(want);
            const int idle = want.x ? 1 : 0;
            f2 kk = k, ikk = ik;
            if constexpr (!SMOOTH) {
                if (ragged) {
                    if (idle) { park_component<1>(t, park); shadow_component<1>(t); kk.v.y = k.v.x; ikk.v.y = ik.v.x; }
                    else { park_component<0>(t, park); shadow_component<0>(t); kk.v.x = k.v.y; ikk.v.x = ik.v.y; }
                    park[29 * 32] = idle ? chi2.v.y : chi2.v.x;
                    shadow_hit(tp, idle);
                }
            }
            // (the general transport is also right for a track whose radial row is already zero)
            if (all_of(started | !want)) both = fit_layer_pair<true>(t, kk, ikk, P.layer[l], P.mass2, tp, chi2);
            else both = fit_layer_pair<false>(t, kk, ikk, P.layer[l], P.mass2, tp, chi2);
            if constexpr (!SMOOTH) {
                if (ragged) {
                    if (idle) { unpark_component<1>(t, park); chi2.v.y = park[29 * 32]; }
                    else { unpark_component<0>(t, park); chi2.v.x = park[29 * 32]; }
                }
            }
        }
        if (both) {
            if (want.x) { nhx += 1; started.x = true; usedx |= 1u << l; }
            if (want.y) { nhy += 1; started.y = true; usedy |= 1u << l; }
            if constexpr (MODE == 2) store_layer_state_pair(t, a, l, ix, iy, {want.x && valid.x, want.y && valid.y});
        } else if (!none_of(want)) {
            // copies whose address may be taken: the pair itself stays in registers
            Track2 tc = t;
            Hit2 mc;
            load_hit_pair(mc, tp);
            f2 cc = chi2;
            mask2 stored = {false, false};
            if (want.x) {
                const uint32_t rc = fit_layer_one_of_pair(tc, 0, k.v.x, ik.v.x, P.layer[l], P.mass2, mc, cc, started.x);
                st.x |= rc;
                if (rc == 0u) { nhx += 1; started.x = true; usedx |= 1u << l; stored.x = valid.x; }
            }
            if (want.y) {
                const uint32_t rc = fit_layer_one_of_pair(tc, 1, k.v.y, ik.v.y, P.layer[l], P.mass2, mc, cc, started.y);
                st.y |= rc;
                if (rc == 0u) { nhy += 1; started.y = true; usedy |= 1u << l; stored.y = valid.y; }
            }
            t = tc;
            chi2 = cc;
            if constexpr (MODE == 2) store_layer_state_pair(t, a, l, ix, iy, stored);
        }
        // (SMOOTH: the ring runs on into the backward pass, step L + j carries layer L - 1 - j)
        const int nxt = l + kStages;
        if (nxt < (SMOOTH ? 2 * L : L)) {
            const int ln = nxt < L ? nxt : 2 * L - 1 - nxt;
            __syncwarp();
            if (elect_one()) {
                mbar_expect_tx(bar0 + 8u * s, kHit2Floats * 4);
                tma_load_2d(hit0 + s * (kHit2Floats * 4), &M.hpos, col, 3 * ln, bar0 + 8u * s);
                tma_load_2d(hit0 + s * (kHit2Floats * 4) + 3 * kRowBytes, &M.hcov, col, 6 * ln, bar0 + 8u * s);
            }
        }
    }
    if (!good_q.x) st.x = ST_BAD_CHARGE;
    if (!good_q.y) st.y = ST_BAD_CHARGE;
    // a track with nothing fitted goes back as it came: its columns of the seed tile still hold the input
    const mask2 done = {live.x && nhx > 0, live.y && nhy > 0};
    if constexpr (SMOOTH) {
        // ---- forward result out (a copy goes back to the global frame; t stays local for the refit)
        if (!none_of(done)) {
            Track2 g = t;
            leave_local_frame(g);
            pair_to_tile(g, seed_tile, lane, done);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        const bool fstorer = elect_one();
        if (fstorer) {
            tma_store_2d(&M.opar, col, 0, seed0);
            tma_store_2d(&M.ocov, col, 0, seed0 + 6 * kRowBytes);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        if (valid.x) { a.chi2[ix] = chi2.v.x; a.nhits[ix] = nhx; a.status[ix] = st.x; }
        if (valid.y) { a.chi2[iy] = chi2.v.y; a.nhits[iy] = nhy; a.status[iy] = st.y; }
        // ---- inward refit (reading A18)
        f2 schi2(0.0f);
        int lpx = 0, lpy = 0, nbx = 0, nby = 0;
        u2 sst = {0u, 0u};
        mask2 first = {true, true};
        if (!none_of(done)) scale_cov(t, a.kappa);
        for (int j = 0; j < L; ++j) {
            const int l = L - 1 - j, step = L + j, s = step % kStages;
            mbar_wait(bar0 + 8u * s, (phase >> s) & 1u);
            phase ^= 1u << s;
            const float2* tp = reinterpret_cast<const float2*>(wbase + s * kHit2Floats) + lane;
            const mask2 want = {(bool)((usedx >> l) & 1u), (bool)((usedy >> l) & 1u)};
            bool both = false;
            if (all_of(want) && first.x == first.y && (first.x || lpx == lpy)) {
                Hit2 m;
                load_hit_pair(m, tp);
                f2 d;
                const u2 rc = refit_step<false>(t, k, ik, P.layer[l], P.layer[lpx], 0, P.mass2, P.el, first.x, m.x, m.y, m.z,
                                                m.vxx, m.vxy, m.vxz, m.vyy, m.vyz, m.vzz, &d);
                if (is_zero(rc)) {
                    schi2 = schi2 + d;
                    nbx += 1; nby += 1;
                    first.x = false; first.y = false;
                    lpx = l; lpy = l;
                    both = true;
                }
            }
            if (!both && !none_of(want)) {
                Track2 tc = t;
                Hit2 mc;
                load_hit_pair(mc, tp);
                f2 cc = schi2;
                if (want.x) {
                    const uint32_t rc = refit_step_one_of_pair(tc, 0, k.v.x, ik.v.x, P.layer[l], P.layer[lpx], P.mass2, first.x, mc, cc);
                    if (rc == 0u) { nbx += 1; first.x = false; lpx = l; } else sst.x |= rc;
                }
                if (want.y) {
                    const uint32_t rc = refit_step_one_of_pair(tc, 1, k.v.y, ik.v.y, P.layer[l], P.layer[lpy], P.mass2, first.y, mc, cc);
                    if (rc == 0u) { nby += 1; first.y = false; lpy = l; } else sst.y |= rc;
                }
                t = tc;
                schi2 = cc;
            }
            const int nxt = step + kStages;
            if (nxt < 2 * L) {
                const int ln = 2 * L - 1 - nxt;
                __syncwarp();
                if (elect_one()) {
                    mbar_expect_tx(bar0 + 8u * s, kHit2Floats * 4);
                    tma_load_2d(hit0 + s * (kHit2Floats * 4), &M.hpos, col, 3 * ln, bar0 + 8u * s);
                    tma_load_2d(hit0 + s * (kHit2Floats * 4) + 3 * kRowBytes, &M.hcov, col, 6 * ln, bar0 + 8u * s);
                }
            }
        }
        // the forward tile must have left shared memory before the smoothed one overwrites it
        if (fstorer) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        __syncwarp();
        if (!none_of(done)) {
            leave_local_frame(t);
            pair_to_tile(t, seed_tile, lane, done);
        }   // else the tile still holds the forward result = the input
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        const bool sstorer = elect_one();
        if (sstorer) {
            tma_store_2d(&M.spar, col, 0, seed0);
            tma_store_2d(&M.scov, col, 0, seed0 + 6 * kRowBytes);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        if (valid.x) { a.schi2[ix] = schi2.v.x; a.snhits[ix] = nbx; a.sstatus[ix] = sst.x; }
        if (valid.y) { a.schi2[iy] = schi2.v.y; a.snhits[iy] = nby; a.sstatus[iy] = sst.y; }
        if (sstorer) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        return;
    }
    __syncwarp();      // every lane is done with the park area inside the tile
    if (!none_of(done)) {
        leave_local_frame(t);
        pair_to_tile(t, seed_tile, lane, done);
    }
    restore_unfitted(seed_tile, a, lane, ix, iy, {valid.x && !done.x, valid.y && !done.y});
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
    const bool storer = elect_one();
    if (storer) {
        tma_store_2d(&M.opar, col, 0, seed0);
        tma_store_2d(&M.ocov, col, 0, seed0 + 6 * kRowBytes);
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    if (valid.x) { a.chi2[ix] = chi2.v.x; a.nhits[ix] = nhx; a.status[ix] = st.x; }
    if (valid.y) { a.chi2[iy] = chi2.v.y; a.nhits[iy] = nhy; a.status[iy] = st.y; }
    if constexpr (MODE == 2) {
        if (valid.x) a.used[ix] = usedx;
        if (valid.y) a.used[iy] = usedy;
    }
    if (storer) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
#undef KF_TRACK_ROWS

// ---- fit with hits addressed by index into the layer pools (the hits a track uses are
// looked up, not pre-gathered).  index[l][i] = hit of track i in pool l or -1.
// Gathered loads cannot go through TMA: each thread fetches its 9 floats itself.  The look-up is a chain of
// dependent loads (index -> slot of the packed record -> record), so it runs as a three-stage pipeline ahead of
// the math: while layer l is fitted, the hit of layer l + 1 is being fetched, the slot of layer l + 2 resolved
// and the index of layer l + 3 read -- every stage has a whole layer of arithmetic to hide behind.
__device__ __forceinline__ int32_t resolve_hit(const IndexedPools& H, int l, int32_t h) {
    if (h < 0) return -1;
    return H.use_records == 1 ? __ldg(H.orig_to_sorted[l] + h) : h;
}
__device__ __forceinline__ Hit fetch_hit(const IndexedPools& H, int l, int32_t s) {
    Hit m;
    if (H.use_records) {   // one 48-byte record (2 sectors) instead of 9 scattered sectors
        const float4* r = reinterpret_cast<const float4*>(H.hit_rec[l]) + (int64_t)s * kRecWords;
        const float4 A = __ldg(r), B = __ldg(r + 1), C = __ldg(r + 2);
        m.x = A.x; m.y = A.y; m.z = A.z; m.vzz = A.w; m.vxx = B.x; m.vxy = B.y; m.vyy = B.z; m.vxz = C.x; m.vyz = C.y;
        return m;
    }
    const float* p = H.pos[l];
    const float* c = H.cov[l];
    const int64_t ld = H.ld[l];
    m.x = __ldg(p + s);            m.y = __ldg(p + ld + s);       m.z = __ldg(p + 2 * ld + s);
    m.vxx = __ldg(c + s);          m.vxy = __ldg(c + ld + s);     m.vxz = __ldg(c + 2 * ld + s);
    m.vyy = __ldg(c + 3 * ld + s); m.vyz = __ldg(c + 4 * ld + s); m.vzz = __ldg(c + 5 * ld + s);
    return m;
}

// SoA pools -> packed records in ORIGINAL order (same 12-float layout as kf_bin_layers' records: fetch_hit reads
// both).  Reads coalesced plane by plane; a warp's 32 records are staged in shared memory and leave as 96
// consecutive 16-byte words.
__global__ void __launch_bounds__(256) pack_pool_records_kernel(const __grid_constant__ PackPools A) {
    static_assert(kRecWords == 3 || kRecWords == 4, "record layout");
    __shared__ float4 stage[8][32 * kRecWords];
    const int l = blockIdx.y;
    const int64_t n = A.n[l];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t base = (int64_t)blockIdx.x * 256 + w * 32;      // first hit of this warp
    if (base >= n) return;
    const int64_t h = base + lane;
    if (h < n) {
        const float* p = A.pos[l] + h;
        const float* c = A.cov[l] + h;
        const int64_t ld = A.ld[l];
        const float x = __ldg(p), y = __ldg(p + ld), z = __ldg(p + 2 * ld);
        const float vxx = __ldg(c), vxy = __ldg(c + ld), vxz = __ldg(c + 2 * ld);
        const float vyy = __ldg(c + 3 * ld), vyz = __ldg(c + 4 * ld), vzz = __ldg(c + 5 * ld);
        float4* s = &stage[w][lane * kRecWords];
        s[0] = make_float4(x, y, z, vzz);
        s[1] = make_float4(vxx, vxy, vyy, __int_as_float((int)h));
        s[2] = make_float4(vxz, vyz, 0.0f, 0.0f);
        if constexpr (kRecWords == 4) s[3] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    }
    __syncwarp();
    const int cnt = (int)(n - base < 32 ? n - base : 32) * kRecWords;
    float4* out = reinterpret_cast<float4*>(A.rec[l]) + base * kRecWords;
    for (int j = lane; j < cnt; j += 32) out[j] = stage[w][j];
}

template <int GEOM>
__global__ void __launch_bounds__(kFitBlock, 4)
fit_indexed_kernel(const __grid_constant__ FitParams P, const __grid_constant__ IndexedPools H, const FitArgs a) {
    const int64_t i = (int64_t)blockIdx.x * kFitBlock + threadIdx.x;
    if (i >= a.n) return;
    const int L = P.n_layers;
    const int q = a.q[i];
    Track t;
    load_track(t, a.par, a.cov, a.ld_in, i);
    float chi2 = 0.0f;
    int nh = 0;
    uint32_t st = 0u;
    if (q != 1 && q != -1) {
        st = ST_BAD_CHARGE;
    } else {
        const float k = (float)q * P.k0, ik = (float)q * P.inv_k0;
        enter_local_frame_precise(t);
        bool started = false;
        // pipeline registers: raw index of layer l + 2, slot of layer l + 1, hit of layer l
        int32_t h2 = L > 2 ? __ldg(H.index + 2 * H.ld_index + i) : -1;
        int32_t s1 = L > 1 ? resolve_hit(H, 1, __ldg(H.index + H.ld_index + i)) : -1;
        int32_t s0 = resolve_hit(H, 0, __ldg(H.index + i));
        Hit m_next;
        if (s0 >= 0) m_next = fetch_hit(H, 0, s0);
        for (int l = 0; l < L; ++l) {
            const int32_t h = s0;
            const Hit m = m_next;
            s0 = s1;
            if (s0 >= 0) m_next = fetch_hit(H, l + 1, s0);
            s1 = l + 2 < L ? resolve_hit(H, l + 2, h2) : -1;
            h2 = l + 3 < L ? __ldg(H.index + (int64_t)(l + 3) * H.ld_index + i) : -1;
            if (h < 0) continue;
            uint32_t rc;
            if (started) rc = fit_layer<true, GEOM>(t, k, ik, P.layer[l], P.model, P.mass2, P.el, m, chi2);
            else rc = fit_layer<false, GEOM>(t, k, ik, P.layer[l], P.model, P.mass2, P.el, m, chi2);
            st |= rc;
            if (rc == 0u) { nh += 1; started = GEOM != 2 || P.layer[l].type == 0; }
        }
        if (nh > 0) leave_local_frame(t);
        else load_track(t, a.par, a.cov, a.ld_in, i);   // nothing fitted: the seed, bit-exact
    }
    store_track(t, a.opar, a.ocov, a.ld_out, i);
    a.chi2[i] = chi2;
    a.nhits[i] = nh;
    a.status[i] = st;
}

}  // namespace

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute: set once for every device a context
// launches on (the caller has made that device current).
cudaError_t ensure_fit_attributes() {
    static std::atomic<uint64_t> done{0};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const uint64_t bit = 1ull << (dev & 63);
    if (done.load(std::memory_order_acquire) & bit) return cudaSuccess;
    e = cudaFuncSetAttribute(fit_kernel<0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fit_kernel<0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fit_kernel<0, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fit_kernel<1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fit_kernel<1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fit_kernel<1, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fit_kernel<2, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fit_kernel<2, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fit_kernel<2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fit_pair_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem2_bytes(false));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fit_pair_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem2_bytes(true));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fit_pair_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem2_bytes(false));
    if (e == cudaSuccess) done.fetch_or(bit, std::memory_order_release);
    return e;
}

bool fit_takes_pair_form(int64_t n, int n_layers, const LaunchOptions& opt) {
    // (the pair form pays once the machine is full: at least 151 552 tracks, or 2 M track-layers -- config 3's
    // 100 000 x 20 layers: 0.0429 ms against 0.0451 for the one-track kernel)
    if (opt.pair_min_tracks > 0) return n >= opt.pair_min_tracks;
    return n >= (int64_t)KF_PAIR_MIN_TRACKS || n * (int64_t)n_layers >= 2000000;
}

cudaError_t launch_fit(const FitParams& P, const FitArgs& a, cudaStream_t stream, const LaunchOptions& opt) {
    if (a.n == 0) return cudaSuccess;
    const cudaError_t attr = ensure_fit_attributes();
    if (attr != cudaSuccess) return attr;
    const bool smooth = a.spar != nullptr;   // the refit of reading A18 (two results)
    const bool store = a.lpar != nullptr;    // per-layer filtered states for the RTS smoother
    const int L = P.n_layers;
    FitMaps M;
    // Two tracks per thread.  The pair form of the refit takes ragged pairs (a layer only one of the two tracks
    // has a hit on) through the one-track path and then loses badly (1.2 % of tracks stopping short: 0.81 ms against
    // 0.49 ms for 600 000 twenty-layer tracks), so it is taken only where the caller says that every track has
    // every hit (mask == NULL); the pair form of the fit parks and shadows the idle track and wins either way.
    // (Option refit_pair_masked lifts that condition: the tests use it to drive the pair refit's ragged-pair code,
    // which failures can reach without any mask, with masks.)
    const bool big = fit_takes_pair_form(a.n, L, opt);
    if (P.geometry_options == 0 && big &&
        (!smooth || (KF_PAIR_SMOOTH && (a.mask == nullptr || opt.refit_pair_masked != 0)))) {
        constexpr int W = kPairTile;
        if (!make_map(&M.hpos, a.hpos, a.n, a.ld_hit, (int64_t)L * 3, 3, W) ||
            !make_map(&M.hcov, a.hcov, a.n, a.ld_hit, (int64_t)L * 6, 6, W) ||
            !make_map(&M.par, a.par, a.n, a.ld_in, 6, 6, W) || !make_map(&M.cov, a.cov, a.n, a.ld_in, 21, 21, W) ||
            !make_map(&M.opar, a.opar, a.n, a.ld_out, 6, 6, W) || !make_map(&M.ocov, a.ocov, a.n, a.ld_out, 21, 21, W))
            return cudaErrorInvalidValue;
        if (smooth && (!make_map(&M.spar, a.spar, a.n, a.ld_s, 6, 6, W) || !make_map(&M.scov, a.scov, a.n, a.ld_s, 21, 21, W)))
            return cudaErrorInvalidValue;
        const int64_t per_block = (int64_t)kPairWarps * kPairTile;
        const int64_t blocks = (a.n + per_block - 1) / per_block;
        if (smooth) fit_pair_kernel<1><<<(unsigned)blocks, kPairBlock, smem2_bytes(true), stream>>>(P, M, a);
        else if (store) fit_pair_kernel<2><<<(unsigned)blocks, kPairBlock, smem2_bytes(false), stream>>>(P, M, a);
        else fit_pair_kernel<0><<<(unsigned)blocks, kPairBlock, smem2_bytes(false), stream>>>(P, M, a);
        return cudaGetLastError();
    }
    if (!make_map(&M.hpos, a.hpos, a.n, a.ld_hit, (int64_t)L * 3, 3) ||
        !make_map(&M.hcov, a.hcov, a.n, a.ld_hit, (int64_t)L * 6, 6) ||
        !make_map(&M.par, a.par, a.n, a.ld_in, 6, 6) || !make_map(&M.cov, a.cov, a.n, a.ld_in, 21, 21) ||
        !make_map(&M.opar, a.opar, a.n, a.ld_out, 6, 6) || !make_map(&M.ocov, a.ocov, a.n, a.ld_out, 21, 21))
        return cudaErrorInvalidValue;
    if (smooth && (!make_map(&M.spar, a.spar, a.n, a.ld_s, 6, 6) || !make_map(&M.scov, a.scov, a.n, a.ld_s, 21, 21)))
        return cudaErrorInvalidValue;
    const int64_t blocks = (a.n + kFitBlock - 1) / kFitBlock;
    const bool geom = P.geometry_options != 0;   // reading A20 options in use
    if (smooth && P.has_discs) fit_kernel<1, 2><<<(unsigned)blocks, kFitBlock, kSmemBytes, stream>>>(P, M, a);
    else if (smooth && geom) fit_kernel<1, 1><<<(unsigned)blocks, kFitBlock, kSmemBytes, stream>>>(P, M, a);
    else if (smooth) fit_kernel<1, 0><<<(unsigned)blocks, kFitBlock, kSmemBytes, stream>>>(P, M, a);
    else if (store && P.has_discs) fit_kernel<2, 2><<<(unsigned)blocks, kFitBlock, kSmemBytes, stream>>>(P, M, a);
    else if (store && geom) fit_kernel<2, 1><<<(unsigned)blocks, kFitBlock, kSmemBytes, stream>>>(P, M, a);
    else if (store) fit_kernel<2, 0><<<(unsigned)blocks, kFitBlock, kSmemBytes, stream>>>(P, M, a);
    else if (P.has_discs) fit_kernel<0, 2><<<(unsigned)blocks, kFitBlock, kSmemBytes, stream>>>(P, M, a);
    else if (geom) fit_kernel<0, 1><<<(unsigned)blocks, kFitBlock, kSmemBytes, stream>>>(P, M, a);
    else fit_kernel<0, 0><<<(unsigned)blocks, kFitBlock, kSmemBytes, stream>>>(P, M, a);
    return cudaGetLastError();
}

cudaError_t IndexScratch::reserve(size_t bytes, cudaStream_t stream) {
    if (bytes <= cap) return cudaSuccess;
    cudaError_t e = cudaStreamSynchronize(stream);       // the records of the previous call may still be read
    if (e != cudaSuccess) return e;
    release();
    ++gen;
    if ((e = cudaMalloc(&rec, bytes)) != cudaSuccess) { rec = nullptr; return e; }
    cap = bytes;
    return cudaSuccess;
}

void IndexScratch::release() {
    if (rec) cudaFree(rec);
    rec = nullptr;
    cap = 0;
}

cudaError_t launch_pack_pools(const PackPools& A, int n_layers, cudaStream_t stream) {
    int64_t most = 0;
    for (int l = 0; l < n_layers; ++l) most = A.n[l] > most ? A.n[l] : most;
    if (most == 0) return cudaSuccess;
    const dim3 grid((unsigned)((most + 255) / 256), (unsigned)n_layers);
    pack_pool_records_kernel<<<grid, 256, 0, stream>>>(A);
    return cudaGetLastError();
}

cudaError_t launch_fit_indexed(const FitParams& P, const IndexedPools& H, const FitArgs& a, cudaStream_t stream) {
    if (a.n == 0) return cudaSuccess;
    const int64_t blocks = (a.n + kFitBlock - 1) / kFitBlock;
    if (P.has_discs) fit_indexed_kernel<2><<<(unsigned)blocks, kFitBlock, 0, stream>>>(P, H, a);
    else fit_indexed_kernel<1><<<(unsigned)blocks, kFitBlock, 0, stream>>>(P, H, a);
    return cudaGetLastError();
}

}  // namespace kf
