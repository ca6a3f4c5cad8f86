// kf_score.cu -- best-hit candidate scoring ("the hit that produced the lowest chi2
// increment"; PAPER.md:133-141 hits looked up through the (eta, phi) bins), one layer at a time
// (kf_score_candidates) or over consecutive layers with the candidates kept in the track-local frame
// in between (kf_build_best_hit).
//
// Work is split by its natural parallelism:
//   * per-CANDIDATE arithmetic (propagation, covariance transport, Kalman update, frame changes) runs
//     one thread per candidate (`propagate_*_kernel`, `update_*_kernel`) and talks to the scan through
//     a small SoA scratch (28 floats per candidate) owned by the context;
//   * the per-HIT scan runs one warp per candidate (`scan_kernel`): the lanes stride over the hits of
//     the +-window_half bin window, which is, per eta row, one contiguous run of the bin-ordered packed
//     hit records (two runs when the phi ring wraps).
//
// Two-phase scan.  Nearly every hit of a window is many sigma away, and for any unit vector u
//     chi2 = r^T S^-1 r >= (u.r)^2 / (u^T S u)           (Cauchy-Schwarz, S positive definite),
// so with u = z-hat and u = tangent-hat (S_zz = C'_zz + v_zz, S_tt = C'_tt + v~_tt) a hit whose bound
// exceeds the threshold T = min(chi2_cut, best chi2 so far) can neither be accepted nor beat the
// current best and is dropped after ~20 instructions and two of its three 128-bit words.  The
// survivors (a few per cent) are compacted through a per-warp list in shared memory (ballot + popc)
// and evaluated densely, 32 at a time, with the same Schur-form chi2 as the update.  A 1 % margin on
// the bound covers fp32 rounding.  The same two bounds are first applied to whole BINS (bounding box of
// the bin's hits and its largest variances, made by kf_bin_layers): typically 2-4 of the 25 bins of a
// window survive, the others are never touched.  A shuffle arg-min then picks (lowest chi2, lowest
// original index).
// Warp w scans candidate order[w] when an order is given (kf_order_candidates), so neighbouring warps
// share their windows in L1/L2; the order never changes a result.
#include <mutex>

#include "kf_score_common.cuh"

namespace kf {

namespace {


// Candidate i stands at the layer (scratch filled): apply the scan's decision.  On return t is the
// candidate after this layer in the local frame.
// MULTI: the call builds several events at once (EventPools); compiled out of the single-event kernels, whose
// inner loops it would otherwise cost 9 % (measured: 0.177 -> 0.194 ms per configs[4] build).
// disc: the layer the candidate stands at is a disc (readings A23 / A24).
template <bool MULTI>
__device__ __forceinline__ void apply_decision(const ScoreArgs& a, int64_t i, Track& t, bool disc = false) {
    const int32_t slot = a.slot[i];
    if (disc) {
        DiscCrossing o;
        DiscCov n;
        float pz;
        get_scratch_disc(a.scratch, a.ld_sc, i, o, n, pz);
        t.pz = pz;
        bool updated = false;
        if (slot >= 0 && a.do_update) {
            Crossing c;                       // what hit_to_local reads of it
            c.xn = o.xn; c.yn = o.yn; c.zn = o.zt; c.erx = o.erx; c.ery = o.ery;
            LocalHit h;
            const float* recs = MULTI ? a.ev.hit_rec[event_of(a.ev, i)] : a.hit_rec;
            hit_from_record(reinterpret_cast<const float4*>(recs), slot, c, h);
            float d;
            const uint32_t rc = kalman_update_disc(t, o, n, h, &d);
            if (rc == 0u) { updated = true; a.chi2[i] += d; a.nhits[i] += 1; }
            else a.status[i] |= rc;
        }
        if (!updated) commit_propagated_disc(t, o, n);
        return;
    }
    Crossing o;
    PropCov n;
    float pz;
    get_scratch(a.scratch, a.ld_sc, i, o, n, pz);
    t.pz = pz;
    bool updated = false;
    if (slot >= 0 && a.do_update) {
        LocalHit h;
        const float* recs = MULTI ? a.ev.hit_rec[event_of(a.ev, i)] : a.hit_rec;
        hit_from_record(reinterpret_cast<const float4*>(recs), slot, o, h);
        float d;
        const uint32_t rc = kalman_update(t, o, n, h, &d);
        if (rc == 0u) { updated = true; a.chi2[i] += d; a.nhits[i] += 1; }
        else a.status[i] |= rc;
    }
    if (!updated) commit_propagated(t, o, n);
}

// First step: global-frame candidate -> local frame -> propagate to `layer`.
__global__ void __launch_bounds__(kCandBlock)
propagate_global_kernel(const __grid_constant__ FitParams P, const ScoreArgs a, int layer, int keep_track) {
    pdl_start();
    const int64_t i = (int64_t)blockIdx.x * kCandBlock + threadIdx.x;
    if (i >= a.n) return;
    const int q = a.q[i];
    if (q != 1 && q != -1) { a.status[i] |= ST_BAD_CHARGE; a.flag[i] = FLAG_DEAD; return; }
    Track t;
    // the per-layer call with a caller-kept local-frame state (kf_score_candidates, local_state): plane 29 says
    // whether planes 0..28 hold this candidate
    if (a.lstate && __float_as_int(a.lstate[29 * a.ld_ls + i]) != 0) {
        get_track(a.lstate, a.ld_ls, i, t);
    } else {
        load_track(t, a.par, a.cov, a.ld, i);
        enter_local_frame_precise(t);
    }
    if (keep_track) put_track(a.track, a.ld_sc, i, t);
    const float k = (float)q * P.k0, ik = (float)q * P.inv_k0;
    const BinGrid grid{a.n_eta, a.n_phi, a.eta_max};
    const uint32_t rc = P.layer[layer].type == 1
        ? propagate_to_scratch_disc(t, k, ik, P.layer[layer], P.model, P.mass2, P.el, grid, a.scratch, a.ld_sc, i)
        : propagate_to_scratch<false>(t, k, ik, P.layer[layer], P.model, P.mass2, P.el, grid, a.scratch, a.ld_sc, i);
    if (rc) a.status[i] |= rc;
    a.flag[i] = rc ? FLAG_IDLE : FLAG_AT_LAYER;
}

// Middle step of kf_build_best_hit: decision of the previous layer, then on to `layer`.
template <bool MULTI>
__global__ void __launch_bounds__(kCandBlock)
update_propagate_kernel(const __grid_constant__ FitParams P, const ScoreArgs a, int layer, int prev_layer) {
    pdl_start();
    const int64_t i = (int64_t)blockIdx.x * kCandBlock + threadIdx.x;
    if (i >= a.n) return;
    const int32_t f = a.flag[i];
    if (f == FLAG_DEAD) return;
    Track t;
    if (f == FLAG_AT_LAYER) { apply_decision<MULTI>(a, i, t, P.layer[prev_layer].type == 1); put_track(a.track, a.ld_sc, i, t); }
    else get_track(a.track, a.ld_sc, i, t);
    const float qf = (float)a.q[i];
    const BinGrid grid{a.n_eta, a.n_phi, a.eta_max};
    const uint32_t rc = P.layer[layer].type == 1
        ? propagate_to_scratch_disc(t, qf * P.k0, qf * P.inv_k0, P.layer[layer], P.model, P.mass2, P.el, grid, a.scratch, a.ld_sc, i)
        : propagate_to_scratch<false>(t, qf * P.k0, qf * P.inv_k0, P.layer[layer], P.model, P.mass2, P.el, grid, a.scratch,
                                                    a.ld_sc, i);
    if (rc) a.status[i] |= rc;
    a.flag[i] = rc ? FLAG_IDLE : FLAG_AT_LAYER;
}

// Last step: decision of the last layer, back to the global frame, store.
// have_track = 0 (single-layer call): a candidate that did not reach the layer is left untouched.
template <bool MULTI>
__global__ void __launch_bounds__(kCandBlock)
update_global_kernel(const ScoreArgs a, int have_track, int disc) {
    pdl_start();
    const int64_t i = (int64_t)blockIdx.x * kCandBlock + threadIdx.x;
    if (i >= a.n) return;
    const int32_t f = a.flag[i];
    if (f == FLAG_DEAD) return;
    Track t;
    if (f == FLAG_AT_LAYER) apply_decision<MULTI>(a, i, t, disc != 0);
    else if (have_track) get_track(a.track, a.ld_sc, i, t);
    else return;
    if (a.lstate) {   // the candidate as it stands now, in the local frame, for the next per-layer call
        put_track(a.lstate, a.ld_ls, i, t);
        a.lstate[29 * a.ld_ls + i] = __int_as_float(1);
    }
    leave_local_frame(t);
    store_track(t, a.par, a.cov, a.ld, i);
}

// DISC: the layer is a disc pair (readings A23 / A24): the candidate's live position coordinates are (r, t) in the
// plane instead of (t, z) on the cylinder, so the two Cauchy-Schwarz bounds are taken along r-hat and t-hat.
template <bool MULTI, bool DISC = false>
__global__ void __launch_bounds__(kScanBlock)
scan_kernel(const ScoreArgs a, float inv_r) {
    pdl_start();
    __shared__ int32_t survivors[kScanBlock / 32][96];
    const int lane = threadIdx.x & 31;
    const int64_t w = ((int64_t)blockIdx.x * kScanBlock + threadIdx.x) >> 5;
    if (w >= a.n) return;
    const int64_t i = a.order ? (int64_t)__ldg(a.order + w) : w;
    if (a.flag[i] != FLAG_AT_LAYER) {
        if (lane == 0) { a.slot[i] = -1; a.best_hit[i] = -1; a.best_chi2[i] = CUDART_INF_F; }
        return;
    }
    ScanCand c;
    c.xn = a.scratch[SC_XN * a.ld_sc + i];   c.yn = a.scratch[SC_YN * a.ld_sc + i];
    c.zn = a.scratch[SC_ZN * a.ld_sc + i];   c.ec = a.scratch[SC_ERX * a.ld_sc + i];
    c.es = a.scratch[SC_ERY * a.ld_sc + i];  c.n11 = a.scratch[SC_N11 * a.ld_sc + i];
    c.n12 = a.scratch[SC_N12 * a.ld_sc + i]; c.n22 = a.scratch[SC_N22 * a.ld_sc + i];

    const int cbin = __float_as_int(a.scratch[SC_BIN * a.ld_sc + i]);   // window centre, made by the propagate kernel
    const int ie = cbin >> 16, ip = cbin & 0xffff;

    Best best;
    best.chi2 = CUDART_INF_F; best.orig = 0x7fffffff; best.slot = -1;
    int32_t* list = survivors[threadIdx.x >> 5];
    int cnt = 0;                               // warp-uniform number of listed survivors
    float thr = 1.01f * a.chi2_cut;            // 1.01 * min(cut, best so far); NaN cut -> nothing passes
    const unsigned lt_mask = (1u << lane) - 1u;
    const float ecc = c.ec * c.ec, ess = c.es * c.es, ecs2 = 2.0f * c.ec * c.es;
    const int wh = a.window_half;
    const int ev = MULTI ? event_of(a.ev, i) : 0;          // warp-uniform
    const float4* __restrict__ rec = reinterpret_cast<const float4*>(MULTI ? a.ev.hit_rec[ev] : a.hit_rec);
    const float4* __restrict__ box = reinterpret_cast<const float4*>(MULTI ? a.ev.bin_box[ev] : a.bin_box);
    const int32_t* __restrict__ bin_offset = MULTI ? a.ev.bin_offset[ev] : a.bin_offset;
    const int side = 2 * wh + 1, n_win = side * side;
    // The window, 32 bins at a time: lane j tests bin j against the same two bounds applied to the bin's
    // bounding box (the closest any of its hits can be) and its largest variances; a bin that cannot hold
    // a hit under the threshold is skipped without touching its hits.
    for (int wb = 0; wb < n_win; wb += 32) {
        const int j = wb + lane;
        bool keep = false;
        int32_t s0 = 0, s1 = 0;
        if (j < n_win) {
            const int q = j / side;
            const int e = ie - wh + q;
            int p = ip - wh + (j - q * side);   // 0 <= ip < n_phi and side <= n_phi: one wrap either way is enough
            p += p < 0 ? a.n_phi : 0;
            p -= p >= a.n_phi ? a.n_phi : 0;
            if (e >= 0 && e < a.n_eta) {
                const int bin = e * a.n_phi + p;
                s0 = __ldg(bin_offset + bin);
                s1 = __ldg(bin_offset + bin + 1);
                KF_CHECK(s0 >= 0 && s1 >= s0 && (MULTI || s1 <= a.n_hits));
                const float4 X = __ldg(box + 2 * bin), Z = __ldg(box + 2 * bin + 1);
                const float dzm = fmaxf(0.0f, fmaxf(Z.x - c.zn, c.zn - Z.y));
                // rt(x, y) = ec (y - yn) - es (x - xn) is linear: its range over the box is at the corners
                const float ax = -c.es, ay = c.ec;
                const float x0 = X.x - c.xn, x1 = X.y - c.xn, y0 = X.z - c.yn, y1 = X.w - c.yn;
                const float lo = fminf(ax * x0, ax * x1) + fminf(ay * y0, ay * y1);
                const float hi = fmaxf(ax * x0, ax * x1) + fmaxf(ay * y0, ay * y1);
                const float rtm = lo > 0.0f ? lo : (hi < 0.0f ? -hi : 0.0f);
                if constexpr (DISC) {
                    // rr(x, y) = ec (x - xn) + es (y - yn) over the box; any in-plane variance of a hit <= vxx + vyy
                    const float lor = fminf(c.ec * x0, c.ec * x1) + fminf(c.es * y0, c.es * y1);
                    const float hir = fmaxf(c.ec * x0, c.ec * x1) + fmaxf(c.es * y0, c.es * y1);
                    const float rrm = lor > 0.0f ? lor : (hir < 0.0f ? -hir : 0.0f);
                    keep = (s1 > s0) & (rrm * rrm <= thr * (c.n11 + Z.w)) & (rtm * rtm <= thr * (c.n22 + Z.w));
                } else
                keep = (s1 > s0) & (dzm * dzm <= thr * (c.n22 + Z.z)) & (rtm * rtm <= thr * (c.n11 + Z.w));
            }
        }
        unsigned kept = __ballot_sync(0xffffffffu, keep);
        while (kept) {
            const int src = __ffs(kept) - 1;
            kept &= kept - 1;
            const int32_t b0 = __shfl_sync(0xffffffffu, s0, src), b1 = __shfl_sync(0xffffffffu, s1, src);
            // 64 hits per step: two records per lane, four independent 128-bit loads in flight
            const float4* p = rec + (int64_t)(b0 + lane) * kRecWords;
            for (int32_t sb = b0; sb < b1; sb += 64, p += 64 * kRecWords) {   // warp-uniform trip count
                const int32_t sA = sb + lane, sB = sA + 32;
                const bool vA = sA < b1, vB = sB < b1;
                float4 A0 = make_float4(0.f, 0.f, 0.f, 0.f), B0 = A0, A1 = A0, B1 = A0;
                if (vA) { A0 = __ldg(p); B0 = __ldg(p + 1); }
                if (vB) { A1 = __ldg(p + 32 * kRecWords); B1 = __ldg(p + 32 * kRecWords + 1); }
                const float dz0 = A0.z - c.zn, dz1 = A1.z - c.zn;
                const float rt0 = c.ec * (A0.y - c.yn) - c.es * (A0.x - c.xn);
                const float rt1 = c.ec * (A1.y - c.yn) - c.es * (A1.x - c.xn);
                const float vt0 = ess * B0.x - ecs2 * B0.y + ecc * B0.z;
                const float vt1 = ess * B1.x - ecs2 * B1.y + ecc * B1.z;
                bool pA, pB;
                if constexpr (DISC) {
                    const float rr0 = c.ec * (A0.x - c.xn) + c.es * (A0.y - c.yn);
                    const float rr1 = c.ec * (A1.x - c.xn) + c.es * (A1.y - c.yn);
                    const float vr0 = ecc * B0.x + ecs2 * B0.y + ess * B0.z;
                    const float vr1 = ecc * B1.x + ecs2 * B1.y + ess * B1.z;
                    pA = vA & (rr0 * rr0 <= thr * (c.n11 + vr0)) & (rt0 * rt0 <= thr * (c.n22 + vt0));
                    pB = vB & (rr1 * rr1 <= thr * (c.n11 + vr1)) & (rt1 * rt1 <= thr * (c.n22 + vt1));
                } else {
                    pA = vA & (dz0 * dz0 <= thr * (c.n22 + A0.w)) & (rt0 * rt0 <= thr * (c.n11 + vt0));
                    pB = vB & (dz1 * dz1 <= thr * (c.n22 + A1.w)) & (rt1 * rt1 <= thr * (c.n11 + vt1));
                }
                const unsigned mA = __ballot_sync(0xffffffffu, pA);
                const unsigned mB = __ballot_sync(0xffffffffu, pB);
                if (pA) list[cnt + __popc(mA & lt_mask)] = sA;
                cnt += __popc(mA);
                if (pB) list[cnt + __popc(mB & lt_mask)] = sB;
                cnt += __popc(mB);
                while (cnt >= 32) {                          // evaluate 32 survivors densely
                    __syncwarp();
                    const int32_t sl = list[lane];
                    const int32_t c1 = lane + 32 < cnt ? list[lane + 32] : 0;
                    const int32_t c2 = lane + 64 < cnt ? list[lane + 64] : 0;
                    __syncwarp();
                    if (lane + 32 < cnt) list[lane] = c1;
                    if (lane + 64 < cnt) list[lane + 32] = c2;
                    cnt -= 32;
                    score_hit<DISC>(c, rec, sl, best);
                    float bmin = best.chi2;
#pragma unroll
                    for (int d = 16; d > 0; d >>= 1) bmin = fminf(bmin, __shfl_xor_sync(0xffffffffu, bmin, d));
                    thr = fminf(thr, 1.01f * bmin);
                }
            }
        }
    }
    __syncwarp();
    if (lane < cnt) score_hit<DISC>(c, rec, list[lane], best);
    // warp arg-min on (chi2, original index)
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        const float oc = __shfl_xor_sync(0xffffffffu, best.chi2, d);
        const int32_t oo = __shfl_xor_sync(0xffffffffu, best.orig, d);
        const int32_t os = __shfl_xor_sync(0xffffffffu, best.slot, d);
        if (better(oc, oo, best.chi2, best.orig)) { best.chi2 = oc; best.orig = oo; best.slot = os; }
    }
    if (lane == 0) {
        const bool accept = best.slot >= 0 && best.chi2 < a.chi2_cut;
        a.slot[i] = accept ? best.slot : -1;
        a.best_hit[i] = accept ? best.orig : -1;
        a.best_chi2[i] = best.chi2;
    }
}

}  // namespace

cudaError_t ScoreScratch::reserve(int64_t n, cudaStream_t stream) {
    if (n <= cap) return cudaSuccess;
    cudaError_t e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return e;
    release();
    ++gen;
    const int64_t ldn = (n + 3) / 4 * 4;
    if ((e = cudaMalloc(&scratch, (size_t)kScorePlanes * ldn * 4)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&track, (size_t)29 * ldn * 4)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&flag, (size_t)ldn * 4)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&slot, (size_t)ldn * 4)) != cudaSuccess) { release(); return e; }
    cap = ldn;
    ld = ldn;
    return cudaSuccess;
}

void ScoreScratch::release() {
    void* ptrs[] = {scratch, track, flag, slot};
    for (void* p : ptrs)
        if (p) cudaFree(p);
    scratch = track = nullptr;
    flag = slot = nullptr;
    cap = ld = 0;
}

// Score `n_layers` consecutive steps.  steps[j] gives the geometry layer and the hit pool of step j.
cudaError_t launch_build(ScoreScratch& s, const FitParams& P, ScoreArgs a, int n_steps, const ScoreStep* steps,
                         cudaStream_t stream) {
    if (a.n == 0 || n_steps <= 0) return cudaSuccess;
    cudaError_t e = s.reserve(a.n, stream);
    if (e != cudaSuccess) return e;
    a.scratch = s.scratch; a.track = s.track; a.flag = s.flag; a.slot = s.slot; a.ld_sc = s.ld;
    const unsigned cblocks = (unsigned)((a.n + kCandBlock - 1) / kCandBlock);
    const unsigned sblocks = (unsigned)((a.n + kScanBlock / 32 - 1) / (kScanBlock / 32));
    const int keep = n_steps > 1 ? 1 : 0;
    const bool multi = a.ev.n > 1;
    const dim3 cgrid(cblocks), sgrid(sblocks), cblock(kCandBlock), sblock(kScanBlock);
    cudaError_t e2 = cudaSuccess;
    auto ok = [&](cudaError_t r) { if (e2 == cudaSuccess) e2 = r; };
    for (int j = 0; j < n_steps; ++j) {
        const ScoreStep& st = steps[j];
        if (j == 0) ok(launch_chained(propagate_global_kernel, cgrid, cblock, 0, stream, P, a, st.layer, keep));
        else if (multi) ok(launch_chained(update_propagate_kernel<true>, cgrid, cblock, 0, stream, P, a, st.layer, steps[j - 1].layer));   // a.hit_rec still step j-1
        else ok(launch_chained(update_propagate_kernel<false>, cgrid, cblock, 0, stream, P, a, st.layer, steps[j - 1].layer));
        a.hit_rec = st.hit_rec; a.bin_box = st.bin_box; a.bin_offset = st.bin_offset; a.n_hits = st.n_hits;
        a.best_hit = st.best_hit; a.best_chi2 = st.best_chi2;
        for (int e = 0; e < a.ev.n; ++e) {
            a.ev.hit_rec[e] = st.ev_hit_rec[e]; a.ev.bin_box[e] = st.ev_bin_box[e]; a.ev.bin_offset[e] = st.ev_bin_offset[e];
        }
        const bool disc = P.layer[st.layer].type == 1;
        if (multi) ok(disc ? launch_chained(scan_kernel<true, true>, sgrid, sblock, 0, stream, a, P.layer[st.layer].inv_r)
                           : launch_chained(scan_kernel<true, false>, sgrid, sblock, 0, stream, a, P.layer[st.layer].inv_r));
        else ok(disc ? launch_chained(scan_kernel<false, true>, sgrid, sblock, 0, stream, a, P.layer[st.layer].inv_r)
                     : launch_chained(scan_kernel<false, false>, sgrid, sblock, 0, stream, a, P.layer[st.layer].inv_r));
    }
    const int last_disc = P.layer[steps[n_steps - 1].layer].type == 1 ? 1 : 0;
    if (multi) ok(launch_chained(update_global_kernel<true>, cgrid, cblock, 0, stream, a, keep, last_disc));
    else ok(launch_chained(update_global_kernel<false>, cgrid, cblock, 0, stream, a, keep, last_disc));
    if (e2 != cudaSuccess) return e2;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------- kf_score_candidates_static
// The scratch of the single-layer call for callers that must not allocate (include/kf_b200.h): the propagated
// candidate planes, the flag and the winning slot, for at most kStaticMaxCands candidates, compiled into the
// library.  Each device that loads the module has its own copy (7.75 MiB) until the process exits.  The single-layer
// call never uses the between-layers track planes (keep = 0), so they have no static counterpart.
//
// In HOST code the name g_static_scratch is a host-side stand-in for the symbol, not a device address: the kernels
// get the address cudaGetSymbolAddress returns, resolved once per device with that device current.
}  // namespace kf

static __device__ __align__(256) float g_static_scratch[(size_t)kf::kStaticPlanes * kf::kStaticMaxCands];

namespace kf {

namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
float* g_static_addr[kStaticMaxDevices] = {};   // device address of g_static_scratch per device ordinal

cudaError_t static_scratch_address(float** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kStaticMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_static_addr[dev] = static_cast<float*>(p);
    }
    *out = g_static_addr[dev];
    return cudaSuccess;
}

}  // namespace

// Same three launches as launch_build with n_steps = 1 (propagate, scan, decision); only the scratch differs.
// Nothing in the array has to start at zero: propagate_global_kernel writes flag[i] for every i < n and the scratch
// planes of every candidate it flags FLAG_AT_LAYER, scan_kernel writes slot[i] for exactly those, and
// update_global_kernel reads nothing else.  What an earlier call left beyond that is never read.
cudaError_t launch_score_static(const FitParams& P, ScoreArgs a, const ScoreStep& st, cudaStream_t stream) {
    if (a.n == 0) return cudaSuccess;
    if (a.n > kStaticMaxCands) return cudaErrorInvalidValue;
    float* base = nullptr;
    cudaError_t e = static_scratch_address(&base);
    if (e != cudaSuccess) return e;
    const int64_t ld = (a.n + 63) / 64 * 64;                    // planes stay 256-byte aligned; ld <= kStaticMaxCands
    if (ld > kStaticMaxCands) return cudaErrorInvalidValue;      // (cannot happen: kStaticMaxCands is a multiple of 64)
    a.scratch = base;
    a.track = nullptr;                                          // keep_track = 0 below: never dereferenced
    a.flag = reinterpret_cast<int32_t*>(base + (int64_t)kScorePlanes * ld);
    a.slot = a.flag + ld;
    a.ld_sc = ld;
    a.ev.n = 0;
    const unsigned cblocks = (unsigned)((a.n + kCandBlock - 1) / kCandBlock);
    const unsigned sblocks = (unsigned)((a.n + kScanBlock / 32 - 1) / (kScanBlock / 32));
    propagate_global_kernel<<<cblocks, kCandBlock, 0, stream>>>(P, a, st.layer, 0);
    a.hit_rec = st.hit_rec; a.bin_box = st.bin_box; a.bin_offset = st.bin_offset; a.n_hits = st.n_hits;
    a.best_hit = st.best_hit; a.best_chi2 = st.best_chi2;
    const bool disc = P.layer[st.layer].type == 1;
    if (disc) scan_kernel<false, true><<<sblocks, kScanBlock, 0, stream>>>(a, P.layer[st.layer].inv_r);
    else scan_kernel<false, false><<<sblocks, kScanBlock, 0, stream>>>(a, P.layer[st.layer].inv_r);
    update_global_kernel<false><<<cblocks, kCandBlock, 0, stream>>>(a, 0, disc ? 1 : 0);
    return cudaGetLastError();
}

}  // namespace kf
