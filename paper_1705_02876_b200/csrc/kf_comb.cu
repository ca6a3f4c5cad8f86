// kf_comb.cu -- combinatorial track building ("branching occurs to explore all possible track
// candidates up to some cutoff number of candidates per seed"; PAPER.md:73, 79 clone engine
// per-candidate bookkeeping on the GPU; reading A19).
//
// Every seed owns NC candidate slots.  Per layer, four launches:
//   comb_propagate  one thread per live slot: local-frame track -> propagate (+Q) -> scratch (as best-hit);
//   comb_scan       one warp per live slot: the same bin-pruned, pre-filtered window scan as the best-hit
//                   scan, but it keeps the NC best compatible hits (chi2 < cut) instead of one;
//   comb_select     one warp per seed ("clone engine"): ranks the children of all its
//                   candidates -- each kept hit, plus "no hit" -- by (nhits desc, chi2 asc, parent slot,
//                   hit index) and writes the NC best as (parent, hit) descriptors: only descriptors are
//                   sorted, no track is copied here;
//   comb_update     one thread per surviving child: parent's propagated state + its hit -> Kalman update ->
//                   the other half of the double-buffered track store; one (parent, hit) history entry.
// The hit list of the winner is recovered at the end by walking the history backwards, so branching never
// copies hit lists either.  Instead of the paper's shared-memory heaps the top-NC selection
// is a handful of warp arg-min rounds over the few survivors of the pre-filter.
#include "kf_score_common.cuh"

namespace kf {

namespace {

constexpr int kMaxC = 8;

struct CombArgs {
    int64_t n_seeds, ld;          // seeds and plane stride of the caller's candidate arrays
    float* par; float* cov; const int8_t* q; float* chi2; int32_t* nhits; uint32_t* status;
    int nc;                       // candidates per seed (<= kMaxC)
    int64_t n_slots, ld_s;        // n_seeds * nc, padded
    // double-buffered candidate store (local frame)
    float* trk_in; float* trk_out;
    float* chi2_in; float* chi2_out; int32_t* nh_in; int32_t* nh_out; uint32_t* st_in; uint32_t* st_out;
    int32_t* ncand_in; int32_t* ncand_out;      // [n_seeds]
    // per-layer scratch
    float* scratch; int32_t* flag;
    int32_t* top_rec; float* top_chi2; int32_t* top_orig; int32_t* top_n;   // [n_slots][kMaxC], [n_slots]
    int32_t* child_parent; int32_t* child_rec; int32_t* child_orig; float* child_chi2;   // [n_slots]
    int32_t* hist_parent; int32_t* hist_hit;    // [n_build][ld_s] (this layer's row passed in)
    // hits of the layer
    const float* hit_rec; const float* bin_box; const int32_t* bin_offset;
    int n_eta, n_phi; float eta_max; int window_half; float chi2_cut;
    EventPools ev;                // kf_build_combinatorial_events (ev.n > 1): seeds of event e are first[e] .. first[e + 1] - 1
};

constexpr int32_t REC_NONE = -1;      // child takes no hit
constexpr int32_t REC_STUCK = -2;     // parent could not be propagated: child = parent unchanged

// Seeds (global frame) -> slot 0 of each seed.
__global__ void __launch_bounds__(128)
comb_init_kernel(const CombArgs a) {
    const int64_t sd = (int64_t)blockIdx.x * 128 + threadIdx.x;
    if (sd >= a.n_seeds) return;
    const int q = a.q[sd];
    if (q != 1 && q != -1) { a.status[sd] |= ST_BAD_CHARGE; a.ncand_in[sd] = 0; return; }
    Track t;
    load_track(t, a.par, a.cov, a.ld, sd);
    enter_local_frame_precise(t);
    const int64_t slot = sd * a.nc;
    put_track(a.trk_in, a.ld_s, slot, t);
    a.chi2_in[slot] = a.chi2[sd];
    a.nh_in[slot] = a.nhits[sd];
    a.st_in[slot] = a.status[sd];
    a.ncand_in[sd] = 1;
}

__global__ void __launch_bounds__(128)
comb_propagate_kernel(const __grid_constant__ FitParams P, const CombArgs a, int layer) {
    const int64_t slot = (int64_t)blockIdx.x * 128 + threadIdx.x;
    if (slot >= a.n_slots) return;
    const int64_t sd = slot / a.nc;
    if ((int)(slot - sd * a.nc) >= a.ncand_in[sd]) { a.flag[slot] = FLAG_DEAD; return; }
    Track t;
    get_track(a.trk_in, a.ld_s, slot, t);
    const float qf = (float)a.q[sd];
    const BinGrid grid{a.n_eta, a.n_phi, a.eta_max};
    const uint32_t rc = P.layer[layer].type == 1       // readings A23 / A24: a disc layer
        ? propagate_to_scratch_disc(t, qf * P.k0, qf * P.inv_k0, P.layer[layer], P.model, P.mass2, P.el, grid, a.scratch, a.ld_s, slot)
        : propagate_to_scratch<false>(t, qf * P.k0, qf * P.inv_k0, P.layer[layer], P.model, P.mass2, P.el, grid, a.scratch,
                                                    a.ld_s, slot);
    if (rc) a.st_in[slot] |= rc;   // its one child (REC_STUCK) inherits the reason
    a.flag[slot] = rc ? FLAG_IDLE : FLAG_AT_LAYER;
}

// Per-warp accumulator of accepted hits (chi2 < cut) in shared memory.
struct AccEntry {
    float chi2;
    int32_t orig, rec;
};
constexpr int kAccCap = 96;

// Keep the `keep` best entries of acc[0..n) (by chi2, then original index) at the front, in order.
// Warp-cooperative; returns the new count.  out_* (optional): write them to global memory as well.
__device__ __forceinline__ int acc_top(AccEntry* acc, int n, int keep, int lane) {
    AccEntry mine[kAccCap / 32];
#pragma unroll
    for (int r = 0; r < kAccCap / 32; ++r) {
        const int idx = lane + 32 * r;
        mine[r].chi2 = idx < n ? acc[idx].chi2 : CUDART_INF_F;
        mine[r].orig = idx < n ? acc[idx].orig : 0x7fffffff;
        mine[r].rec = idx < n ? acc[idx].rec : -1;
    }
    __syncwarp();
    const int m = n < keep ? n : keep;
    for (int kq = 0; kq < m; ++kq) {
        // this lane's best remaining entry
        float bc = CUDART_INF_F; int32_t bo = 0x7fffffff; int br = -1;
#pragma unroll
        for (int r = 0; r < kAccCap / 32; ++r)
            if (better(mine[r].chi2, mine[r].orig, bc, bo)) { bc = mine[r].chi2; bo = mine[r].orig; br = r; }
        float wc = bc; int32_t wo = bo;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            const float oc = __shfl_xor_sync(0xffffffffu, wc, d);
            const int32_t oo = __shfl_xor_sync(0xffffffffu, wo, d);
            if (better(oc, oo, wc, wo)) { wc = oc; wo = oo; }
        }
        // the lane that owns the winner (original indices are unique) publishes and retires it
        if (br >= 0 && bc == wc && bo == wo) {
            acc[kq].chi2 = wc; acc[kq].orig = wo;
#pragma unroll
            for (int r = 0; r < kAccCap / 32; ++r)
                if (r == br) { acc[kq].rec = mine[r].rec; mine[r].chi2 = CUDART_INF_F; mine[r].orig = 0x7fffffff; }
        }
        __syncwarp();
    }
    return m;
}

// MULTI: several events in one call (EventPools), compiled out of the single-event kernel as in kf_score.cu.
// DISC: the layer is a disc pair (bounds along r and t in the plane, as in scan_kernel of kf_score.cu).
template <bool MULTI, bool DISC = false>
__global__ void __launch_bounds__(kScanBlock)
comb_scan_kernel(const CombArgs a, float inv_r) {
    __shared__ int32_t survivors[kScanBlock / 32][96];
    __shared__ AccEntry accs[kScanBlock / 32][kAccCap];
    const int lane = threadIdx.x & 31;
    const int64_t slot = ((int64_t)blockIdx.x * kScanBlock + threadIdx.x) >> 5;
    if (slot >= a.n_slots) return;
    if (a.flag[slot] != FLAG_AT_LAYER) { if (lane == 0) a.top_n[slot] = 0; return; }
    ScanCand c;
    c.xn = a.scratch[SC_XN * a.ld_s + slot];   c.yn = a.scratch[SC_YN * a.ld_s + slot];
    c.zn = a.scratch[SC_ZN * a.ld_s + slot];   c.ec = a.scratch[SC_ERX * a.ld_s + slot];
    c.es = a.scratch[SC_ERY * a.ld_s + slot];  c.n11 = a.scratch[SC_N11 * a.ld_s + slot];
    c.n12 = a.scratch[SC_N12 * a.ld_s + slot]; c.n22 = a.scratch[SC_N22 * a.ld_s + slot];
    const int cbin = __float_as_int(a.scratch[SC_BIN * a.ld_s + slot]);   // window centre, made by the propagate kernel
    const int ie = cbin >> 16, ip = cbin & 0xffff;

    int32_t* list = survivors[threadIdx.x >> 5];
    AccEntry* acc = accs[threadIdx.x >> 5];
    int cnt = 0, nacc = 0;
    const float thr = 1.01f * a.chi2_cut;      // every compatible hit is wanted: the threshold stays at the cut
    const unsigned lt_mask = (1u << lane) - 1u;
    const float ecc = c.ec * c.ec, ess = c.es * c.es, ecs2 = 2.0f * c.ec * c.es;
    const int wh = a.window_half;
    const int event = MULTI ? event_of(a.ev, slot / a.nc) : 0;
    const float4* __restrict__ rec = reinterpret_cast<const float4*>(MULTI ? a.ev.hit_rec[event] : a.hit_rec);
    const float4* __restrict__ box = reinterpret_cast<const float4*>(MULTI ? a.ev.bin_box[event] : a.bin_box);
    const int32_t* __restrict__ bin_offset = MULTI ? a.ev.bin_offset[event] : a.bin_offset;
    const int side = 2 * wh + 1, n_win = side * side;

    // full chi2 of up to 32 listed survivors; the compatible ones go to the accumulator
    auto evaluate = [&](int n_take) {
        __syncwarp();
        Best b;
        b.chi2 = CUDART_INF_F; b.orig = 0x7fffffff; b.slot = -1;
        if (lane < n_take) score_hit<DISC>(c, rec, list[lane], b);
        const bool ok = b.slot >= 0 && b.chi2 < a.chi2_cut;
        const unsigned m = __ballot_sync(0xffffffffu, ok);
        if (ok) { AccEntry e; e.chi2 = b.chi2; e.orig = b.orig; e.rec = b.slot; acc[nacc + __popc(m & lt_mask)] = e; }
        nacc += __popc(m);
        __syncwarp();
        if (nacc > kAccCap - 32) nacc = acc_top(acc, nacc, a.nc, lane);
    };

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
                const float4 X = __ldg(box + 2 * bin), Z = __ldg(box + 2 * bin + 1);
                const float dzm = fmaxf(0.0f, fmaxf(Z.x - c.zn, c.zn - Z.y));
                const float ax = -c.es, ay = c.ec;
                const float x0 = X.x - c.xn, x1 = X.y - c.xn, y0 = X.z - c.yn, y1 = X.w - c.yn;
                const float lo = fminf(ax * x0, ax * x1) + fminf(ay * y0, ay * y1);
                const float hi = fmaxf(ax * x0, ax * x1) + fmaxf(ay * y0, ay * y1);
                const float rtm = lo > 0.0f ? lo : (hi < 0.0f ? -hi : 0.0f);
                if constexpr (DISC) {
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
            const float4* p = rec + (int64_t)(b0 + lane) * kRecWords;
            for (int32_t sb = b0; sb < b1; sb += 64, p += 64 * kRecWords) {
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
                while (cnt >= 32) {
                    evaluate(32);
                    const int32_t c1 = lane + 32 < cnt ? list[lane + 32] : 0;
                    const int32_t c2 = lane + 64 < cnt ? list[lane + 64] : 0;
                    __syncwarp();
                    if (lane + 32 < cnt) list[lane] = c1;
                    if (lane + 64 < cnt) list[lane + 32] = c2;
                    cnt -= 32;
                }
            }
        }
    }
    if (cnt > 0) evaluate(cnt);
    nacc = acc_top(acc, nacc, a.nc, lane);
    if (lane < nacc) {
        a.top_rec[slot * kMaxC + lane] = acc[lane].rec;
        a.top_chi2[slot * kMaxC + lane] = acc[lane].chi2;
        a.top_orig[slot * kMaxC + lane] = acc[lane].orig;
    }
    if (lane == 0) a.top_n[slot] = nacc;
}

// "Clone engine": ranks the children of a seed's candidates and writes the best nc as
// descriptors.  Key: nhits descending, chi2 ascending, parent slot ascending, hit index ascending with
// "no hit" last.  Nothing but descriptors moves here.
struct ChildKey {
    int nh;          // hits after this layer
    float chi2;
    int parent;
    int32_t orig;    // original hit index, INT_MAX for "no hit"
    int e;           // child id = parent * (kMaxC + 1) + (k + 1), -1 = none
};

__device__ __forceinline__ bool child_before(const ChildKey& x, const ChildKey& y) {
    if (y.e < 0) return x.e >= 0;
    if (x.e < 0) return false;
    if (x.nh != y.nh) return x.nh > y.nh;
    if (x.chi2 != y.chi2) return x.chi2 < y.chi2;
    if (x.parent != y.parent) return x.parent < y.parent;
    return x.orig < y.orig;
}

// One WARP per seed: the <= nc * (nc + 1) children sit three to a lane; nc rounds of warp arg-min.
__global__ void __launch_bounds__(128)
comb_select_kernel(const CombArgs a) {
    const int lane = threadIdx.x & 31;
    const int64_t sd = ((int64_t)blockIdx.x * 128 + threadIdx.x) >> 5;
    if (sd >= a.n_seeds) return;
    const int ncur = a.ncand_in[sd];
    const int64_t base = sd * a.nc;
    constexpr int kPer = (kMaxC * (kMaxC + 1) + 31) / 32;   // 3
    ChildKey mine[kPer];
    int32_t rec[kPer];
#pragma unroll
    for (int r = 0; r < kPer; ++r) {
        const int e = lane + 32 * r;
        const int p = e / (kMaxC + 1), k = e % (kMaxC + 1) - 1;
        mine[r].e = -1; mine[r].nh = 0; mine[r].chi2 = 0.0f; mine[r].parent = p; mine[r].orig = 0x7fffffff;
        rec[r] = REC_NONE;
        if (p < ncur) {
            const int64_t sp = base + p;
            const bool at = a.flag[sp] == FLAG_AT_LAYER;
            const int nk = at ? a.top_n[sp] : 0;
            if (k < nk) {
                mine[r].e = e;
                mine[r].nh = a.nh_in[sp] + (k >= 0 ? 1 : 0);
                mine[r].chi2 = a.chi2_in[sp] + (k >= 0 ? a.top_chi2[sp * kMaxC + k] : 0.0f);
                if (k >= 0) { mine[r].orig = a.top_orig[sp * kMaxC + k]; rec[r] = a.top_rec[sp * kMaxC + k]; }
                else rec[r] = at ? REC_NONE : REC_STUCK;
            }
        }
    }
    int kept = 0;
    for (int out = 0; out < a.nc; ++out) {
        ChildKey b = mine[0];
        int br = 0;
#pragma unroll
        for (int r = 1; r < kPer; ++r)
            if (child_before(mine[r], b)) { b = mine[r]; br = r; }
        ChildKey w = b;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            ChildKey o;
            o.nh = __shfl_xor_sync(0xffffffffu, w.nh, d);
            o.chi2 = __shfl_xor_sync(0xffffffffu, w.chi2, d);
            o.parent = __shfl_xor_sync(0xffffffffu, w.parent, d);
            o.orig = __shfl_xor_sync(0xffffffffu, w.orig, d);
            o.e = __shfl_xor_sync(0xffffffffu, w.e, d);
            if (child_before(o, w)) w = o;
        }
        if (w.e < 0) break;                       // warp-uniform: no child left
        if (b.e == w.e) {                         // this lane owns the winner
            const int64_t so = base + out;
            a.child_parent[so] = w.parent;
            a.child_orig[so] = w.orig == 0x7fffffff ? -1 : w.orig;
#pragma unroll
            for (int r = 0; r < kPer; ++r)
                if (r == br) { a.child_rec[so] = rec[r]; mine[r].e = -1; }
        }
        kept = out + 1;
    }
    if (lane == 0) a.ncand_out[sd] = kept;
}

// One thread per surviving child: materialise it in the other half of the candidate store.
template <bool MULTI>
__global__ void __launch_bounds__(128)
comb_update_kernel(const CombArgs a, int disc) {
    const int64_t so = (int64_t)blockIdx.x * 128 + threadIdx.x;
    if (so >= a.n_slots) return;
    const int64_t sd = so / a.nc;
    if ((int)(so - sd * a.nc) >= a.ncand_out[sd]) return;
    const int64_t sp = sd * a.nc + a.child_parent[so];
    const int32_t r = a.child_rec[so];
    Track t;
    float chi2 = a.chi2_in[sp];
    int nh = a.nh_in[sp];
    uint32_t st = a.st_in[sp];
    if (r == REC_STUCK) {
        get_track(a.trk_in, a.ld_s, sp, t);   // st already carries ST_PROP_FAIL / ST_OUTSIDE (comb_propagate_kernel)
    } else if (disc) {
        DiscCrossing o;
        DiscCov n;
        float pz;
        get_scratch_disc(a.scratch, a.ld_s, sp, o, n, pz);
        t.pz = pz;
        bool updated = false;
        if (r >= 0) {
            Crossing c;                       // what hit_to_local reads of it
            c.xn = o.xn; c.yn = o.yn; c.zn = o.zt; c.erx = o.erx; c.ery = o.ery;
            LocalHit h;
            const float* recs = MULTI ? a.ev.hit_rec[event_of(a.ev, sd)] : a.hit_rec;
            hit_from_record(reinterpret_cast<const float4*>(recs), r, c, h);
            float d;
            const uint32_t rc = kalman_update_disc(t, o, n, h, &d);
            if (rc == 0u) { updated = true; chi2 += d; nh += 1; } else st |= rc;
        }
        if (!updated) commit_propagated_disc(t, o, n);
    } else {
        Crossing o;
        PropCov n;
        float pz;
        get_scratch(a.scratch, a.ld_s, sp, o, n, pz);
        t.pz = pz;
        bool updated = false;
        if (r >= 0) {
            LocalHit h;
            const float* recs = MULTI ? a.ev.hit_rec[event_of(a.ev, sd)] : a.hit_rec;
            hit_from_record(reinterpret_cast<const float4*>(recs), r, o, h);
            float d;
            const uint32_t rc = kalman_update(t, o, n, h, &d);
            if (rc == 0u) { updated = true; chi2 += d; nh += 1; } else st |= rc;
        }
        if (!updated) commit_propagated(t, o, n);
    }
    put_track(a.trk_out, a.ld_s, so, t);
    a.chi2_out[so] = chi2;
    a.nh_out[so] = nh;
    a.st_out[so] = st;
    a.hist_parent[so] = a.child_parent[so];
    a.hist_hit[so] = a.child_orig[so];
}

// Slot 0 of every seed is its track: back to the global frame, and its hit list by walking the history.
__global__ void __launch_bounds__(128)
comb_finish_kernel(const CombArgs a, int n_build, const int32_t* __restrict__ hist_parent_all,
                   const int32_t* __restrict__ hist_hit_all, int32_t* __restrict__ hit_index, int64_t ld_out,
                   int32_t* __restrict__ n_found) {
    const int64_t sd = (int64_t)blockIdx.x * 128 + threadIdx.x;
    if (sd >= a.n_seeds) return;
    const int nc = a.ncand_in[sd];
    if (n_found) n_found[sd] = nc;
    if (nc <= 0) {                                 // bad charge: untouched, no hits
        for (int j = 0; j < n_build; ++j) hit_index[(int64_t)j * ld_out + sd] = -1;
        return;
    }
    const int64_t s0 = sd * a.nc;
    Track t;
    get_track(a.trk_in, a.ld_s, s0, t);
    leave_local_frame(t);
    store_track(t, a.par, a.cov, a.ld, sd);
    a.chi2[sd] = a.chi2_in[s0];
    a.nhits[sd] = a.nh_in[s0];
    a.status[sd] = a.st_in[s0];
    int c = 0;
    for (int j = n_build - 1; j >= 0; --j) {
        const int64_t s = (int64_t)j * a.ld_s + s0 + c;
        hit_index[(int64_t)j * ld_out + sd] = hist_hit_all[s];
        c = hist_parent_all[s];
    }
}

}  // namespace

cudaError_t CombScratch::reserve(int64_t words, cudaStream_t stream) {
    if (words <= cap_words) return cudaSuccess;
    cudaError_t e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return e;
    release();
    ++gen;
    if ((e = cudaMalloc(&buf, (size_t)words * 4)) != cudaSuccess) { buf = nullptr; return e; }
    cap_words = words;
    return cudaSuccess;
}

void CombScratch::release() {
    if (buf) cudaFree(buf);
    buf = nullptr;
    cap_words = 0;
}

cudaError_t launch_comb(CombScratch& s, const FitParams& P, const CombCall& call, int n_steps, const ScoreStep* steps,
                        cudaStream_t stream) {
    if (call.n_seeds == 0 || n_steps <= 0) return cudaSuccess;
    const int nc = call.n_cand;
    const int64_t n_slots = call.n_seeds * nc, S = (n_slots + 3) / 4 * 4, NS = (call.n_seeds + 3) / 4 * 4;
    const int64_t words = S * (2 * 29 + 6 + kScorePlanes + 1 + 3 * kMaxC + 1 + 4 + 2 * (int64_t)n_steps) + 2 * NS;
    cudaError_t e = s.reserve(words, stream);
    if (e != cudaSuccess) return e;
    int32_t* w = reinterpret_cast<int32_t*>(s.buf);
    auto take = [&](int64_t n) { int32_t* p = w; w += n; return p; };
    CombArgs a;
    a.n_seeds = call.n_seeds; a.ld = call.ld; a.par = call.par; a.cov = call.cov; a.q = call.q;
    a.chi2 = call.chi2; a.nhits = call.nhits; a.status = call.status;
    a.nc = nc; a.n_slots = n_slots; a.ld_s = S;
    float* trk[2] = {reinterpret_cast<float*>(take(29 * S)), reinterpret_cast<float*>(take(29 * S))};
    float* c2[2] = {reinterpret_cast<float*>(take(S)), reinterpret_cast<float*>(take(S))};
    int32_t* nh[2] = {take(S), take(S)};
    uint32_t* st[2] = {reinterpret_cast<uint32_t*>(take(S)), reinterpret_cast<uint32_t*>(take(S))};
    int32_t* ncd[2] = {take(NS), take(NS)};
    a.scratch = reinterpret_cast<float*>(take((int64_t)kScorePlanes * S));
    a.flag = take(S);
    a.top_rec = take(kMaxC * S); a.top_chi2 = reinterpret_cast<float*>(take(kMaxC * S)); a.top_orig = take(kMaxC * S);
    a.top_n = take(S);
    a.child_parent = take(S); a.child_rec = take(S); a.child_orig = take(S); a.child_chi2 = reinterpret_cast<float*>(take(S));
    int32_t* hist_parent = take((int64_t)n_steps * S);
    int32_t* hist_hit = take((int64_t)n_steps * S);
    a.n_eta = call.n_eta; a.n_phi = call.n_phi; a.eta_max = call.eta_max;
    a.window_half = call.window_half; a.chi2_cut = call.chi2_cut;
    const unsigned seed_blocks = (unsigned)((call.n_seeds + 127) / 128);
    const unsigned slot_blocks = (unsigned)((n_slots + 127) / 128);
    const unsigned scan_blocks = (unsigned)((n_slots + kScanBlock / 32 - 1) / (kScanBlock / 32));
    int cur = 0;
    auto bind = [&](int in) {
        a.trk_in = trk[in]; a.trk_out = trk[in ^ 1]; a.chi2_in = c2[in]; a.chi2_out = c2[in ^ 1];
        a.nh_in = nh[in]; a.nh_out = nh[in ^ 1]; a.st_in = st[in]; a.st_out = st[in ^ 1];
        a.ncand_in = ncd[in]; a.ncand_out = ncd[in ^ 1];
    };
    bind(cur);
    a.hit_rec = nullptr; a.bin_box = nullptr; a.bin_offset = nullptr; a.hist_parent = hist_parent; a.hist_hit = hist_hit;
    a.ev = call.ev;
    const bool multi = a.ev.n > 1;
    comb_init_kernel<<<seed_blocks, 128, 0, stream>>>(a);
    for (int j = 0; j < n_steps; ++j) {
        const ScoreStep& sp = steps[j];
        a.hit_rec = sp.hit_rec; a.bin_box = sp.bin_box; a.bin_offset = sp.bin_offset;
        for (int e = 0; e < a.ev.n; ++e) {
            a.ev.hit_rec[e] = sp.ev_hit_rec[e]; a.ev.bin_box[e] = sp.ev_bin_box[e]; a.ev.bin_offset[e] = sp.ev_bin_offset[e];
        }
        a.hist_parent = hist_parent + (int64_t)j * S;
        a.hist_hit = hist_hit + (int64_t)j * S;
        comb_propagate_kernel<<<slot_blocks, 128, 0, stream>>>(P, a, sp.layer);
        const bool disc = P.layer[sp.layer].type == 1;
        if (multi && disc) comb_scan_kernel<true, true><<<scan_blocks, kScanBlock, 0, stream>>>(a, P.layer[sp.layer].inv_r);
        else if (multi) comb_scan_kernel<true, false><<<scan_blocks, kScanBlock, 0, stream>>>(a, P.layer[sp.layer].inv_r);
        else if (disc) comb_scan_kernel<false, true><<<scan_blocks, kScanBlock, 0, stream>>>(a, P.layer[sp.layer].inv_r);
        else comb_scan_kernel<false, false><<<scan_blocks, kScanBlock, 0, stream>>>(a, P.layer[sp.layer].inv_r);
        comb_select_kernel<<<(unsigned)((call.n_seeds + 3) / 4), 128, 0, stream>>>(a);
        if (multi) comb_update_kernel<true><<<slot_blocks, 128, 0, stream>>>(a, disc ? 1 : 0);
        else comb_update_kernel<false><<<slot_blocks, 128, 0, stream>>>(a, disc ? 1 : 0);
        cur ^= 1;
        bind(cur);
    }
    comb_finish_kernel<<<seed_blocks, 128, 0, stream>>>(a, n_steps, hist_parent, hist_hit, call.hit_index, call.ld_out,
                                                        call.n_found);
    return cudaGetLastError();
}

}  // namespace kf
