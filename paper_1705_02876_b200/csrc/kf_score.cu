// kf_score.cu -- best-hit candidate scoring on one layer ("the hit that produced the
// lowest chi2 increment"; PAPER.md:133-141 one GPU thread group per candidate, hits looked up
// through the (eta, phi) bins).
//
// One WARP owns one candidate.  Every lane propagates the candidate redundantly (state and C' in
// registers, no shuffles needed afterwards), then the lanes stride over the hits of the
// +-window_half bin window.  The window is, per eta row, one contiguous run of the bin-ordered
// packed hit records (two runs when the phi ring wraps); a record is 12 floats, so a lane fetches a
// hit with three 128-bit loads and a warp reads 1.5 KB of consecutive memory per step.  Two hits per
// lane are in flight per iteration.  chi2 = r^T (C'_pp + V_h)^-1 r is evaluated in the candidate's
// local frame with the same Schur elimination as the update; a shuffle arg-min picks (lowest chi2,
// then lowest original index); all lanes apply the Kalman update with the winner, lane 0 stores.
// Warp w processes candidate order[w] when an order is given (kf_order_candidates): neighbouring
// warps then share their windows in L1/L2.  The order never changes a result.
#include <math_constants.h>

#include "kf_internal.h"

namespace kf {

namespace {

constexpr int kScoreBlock = 128;  // 4 candidates per CTA

__device__ __forceinline__ bool better(float c, int32_t h, float bc, int32_t bh) {
    return c < bc || (c == bc && h < bh);
}

struct Best {
    float chi2;
    int32_t orig, slot;
};

__device__ __forceinline__ void score_hit(const Crossing& o, const PropCov& n, const float4& A, const float4& B,
                                          const float4& C, int32_t slot, Best& best) {
    LocalHit h;
    hit_to_local(o, A.x, A.y, A.z, A.w, B.x, B.y, B.z, B.w, C.x, h);
    float c;
    if (!chi2_schur(n.n11, n.n12, n.n22, h, c)) return;
    const int32_t orig = __float_as_int(C.y);
    if (better(c, orig, best.chi2, best.orig)) { best.chi2 = c; best.orig = orig; best.slot = slot; }
}

__global__ void __launch_bounds__(kScoreBlock)
score_kernel(const __grid_constant__ FitParams P, const ScoreArgs a) {
    const int lane = threadIdx.x & 31;
    const int64_t w = ((int64_t)blockIdx.x * kScoreBlock + threadIdx.x) >> 5;
    if (w >= a.n) return;
    const int64_t i = a.order ? (int64_t)__ldg(a.order + w) : w;
    const LayerConst& Lc = P.layer[a.layer];
    const int q = a.q[i];
    if (q != 1 && q != -1) {
        if (lane == 0) { a.status[i] |= ST_BAD_CHARGE; a.best_hit[i] = -1; a.best_chi2[i] = CUDART_INF_F; }
        return;
    }
    Track t;
    load_track(t, a.par, a.cov, a.ld, i);
    enter_local_frame(t);
    const float k = (float)q * P.k0, ik = (float)q * P.inv_k0;
    Crossing o;
    if (!helix_to_radius(t, k, ik, Lc, o)) {
        if (lane == 0) { a.status[i] |= ST_PROP_FAIL; a.best_hit[i] = -1; a.best_chi2[i] = CUDART_INF_F; }
        return;
    }
    PropCov n;
    transport_cov<false>(t, o, Lc.ms, P.mass2, n);

    // the candidate's own bin (reading A16): eta = asinh(z'/r), phi = atan2(y', x')
    const float eta = asinhf(o.zn * Lc.inv_r);
    const float phi = atan2f(o.yn, o.xn);
    const float d_eta = 2.0f * a.eta_max / (float)a.n_eta;
    const float d_phi = 2.0f * CUDART_PI_F / (float)a.n_phi;
    int ie = (int)floorf((eta + a.eta_max) / d_eta);
    ie = ie < 0 ? 0 : (ie > a.n_eta - 1 ? a.n_eta - 1 : ie);
    int ip = (int)floorf((phi + CUDART_PI_F) / d_phi);
    ip = ((ip % a.n_phi) + a.n_phi) % a.n_phi;

    Best best;
    best.chi2 = CUDART_INF_F; best.orig = 0x7fffffff; best.slot = -1;
    const int wh = a.window_half;
    const float4* __restrict__ rec = reinterpret_cast<const float4*>(a.hit_rec);
    const int e_lo = ie - wh < 0 ? 0 : ie - wh, e_hi = ie + wh > a.n_eta - 1 ? a.n_eta - 1 : ie + wh;
    // phi bins p0 .. p0 + 2w (mod n_phi): one run of the ordered records, or two when it wraps
    const int p0 = ((ip - wh) % a.n_phi + a.n_phi) % a.n_phi;
    const int p1 = p0 + 2 * wh;  // inclusive, may exceed n_phi - 1
    const int nseg = p1 >= a.n_phi ? 2 : 1;
    for (int e = e_lo; e <= e_hi; ++e) {
        const int row = e * a.n_phi;
        for (int sgi = 0; sgi < nseg; ++sgi) {
            int32_t s0, s1;
            if (nseg == 1) { s0 = __ldg(a.bin_offset + row + p0); s1 = __ldg(a.bin_offset + row + p1 + 1); }
            else if (sgi == 0) { s0 = __ldg(a.bin_offset + row + p0); s1 = __ldg(a.bin_offset + row + a.n_phi); }
            else { s0 = __ldg(a.bin_offset + row); s1 = __ldg(a.bin_offset + row + p1 - a.n_phi + 1); }
            int32_t s = s0 + lane;
            for (; s + 32 < s1; s += 64) {   // two hits per lane in flight
                const float4* r0 = rec + (int64_t)s * 3;
                const float4* r1 = rec + (int64_t)(s + 32) * 3;
                const float4 A0 = __ldg(r0), B0 = __ldg(r0 + 1), C0 = __ldg(r0 + 2);
                const float4 A1 = __ldg(r1), B1 = __ldg(r1 + 1), C1 = __ldg(r1 + 2);
                score_hit(o, n, A0, B0, C0, s, best);
                score_hit(o, n, A1, B1, C1, s + 32, best);
            }
            if (s < s1) {
                const float4* r0 = rec + (int64_t)s * 3;
                const float4 A0 = __ldg(r0), B0 = __ldg(r0 + 1), C0 = __ldg(r0 + 2);
                score_hit(o, n, A0, B0, C0, s, best);
            }
        }
    }
    // warp arg-min on (chi2, original index)
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        const float oc = __shfl_xor_sync(0xffffffffu, best.chi2, d);
        const int32_t oo = __shfl_xor_sync(0xffffffffu, best.orig, d);
        const int32_t os = __shfl_xor_sync(0xffffffffu, best.slot, d);
        if (better(oc, oo, best.chi2, best.orig)) { best.chi2 = oc; best.orig = oo; best.slot = os; }
    }
    const bool found = best.slot >= 0;
    const bool accept = found && best.chi2 < a.chi2_cut;
    bool updated = false;
    uint32_t st_add = 0u;
    float dchi2 = 0.0f;
    if (accept && a.do_update) {
        const float4* r0 = rec + (int64_t)best.slot * 3;
        const float4 A0 = __ldg(r0), B0 = __ldg(r0 + 1), C0 = __ldg(r0 + 2);
        LocalHit h;
        hit_to_local(o, A0.x, A0.y, A0.z, A0.w, B0.x, B0.y, B0.z, B0.w, C0.x, h);
        const uint32_t rc = kalman_update(t, o, n, h, &dchi2);
        if (rc == 0u) updated = true; else st_add = rc;
    }
    if (!updated) commit_propagated(t, o, n);
    leave_local_frame(t);
    if (lane == 0) {
        store_track(t, a.par, a.cov, a.ld, i);
        a.best_hit[i] = accept ? best.orig : -1;
        a.best_chi2[i] = best.chi2;
        if (updated) { a.chi2[i] += dchi2; a.nhits[i] += 1; }
        if (st_add) a.status[i] |= st_add;
    }
}

}  // namespace

cudaError_t launch_score(const FitParams& P, const ScoreArgs& a, cudaStream_t stream) {
    if (a.n == 0) return cudaSuccess;
    const int per_block = kScoreBlock / 32;
    const unsigned blocks = (unsigned)((a.n + per_block - 1) / per_block);
    score_kernel<<<blocks, kScoreBlock, 0, stream>>>(P, a);
    return cudaGetLastError();
}

}  // namespace kf
