// kf_score.cu -- best-hit candidate scoring on one layer ("the hit that produced the
// lowest chi2 increment"; PAPER.md:133-141 one GPU thread group per candidate, hits looked up
// through the (eta, phi) bins).
//
// One WARP owns one candidate.  Every lane propagates the candidate redundantly (state and C' in
// registers, no shuffles needed afterwards), then the lanes stride over the hits of the
// +-window_half bin window -- contiguous runs of the bin-sorted SoA copy, so each load is one
// coalesced 128-byte line served from L2/L1 -- computing chi2 = r^T (C'_pp + V_h)^-1 r in the
// candidate's local frame; a shuffle arg-min picks (lowest chi2, then lowest original index);
// all lanes apply the Kalman update with the winner and lane 0 stores the candidate.
#include <math_constants.h>

#include "kf_internal.h"

namespace kf {

namespace {

constexpr int kScoreBlock = 128;  // 4 candidates per CTA

__device__ __forceinline__ bool better(float c, int32_t h, float bc, int32_t bh) {
    return c < bc || (c == bc && h < bh);
}

__global__ void __launch_bounds__(kScoreBlock)
score_kernel(const __grid_constant__ FitParams P, const ScoreArgs a) {
    const int lane = threadIdx.x & 31;
    const int64_t i = ((int64_t)blockIdx.x * kScoreBlock + threadIdx.x) >> 5;
    if (i >= a.n) return;
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

    float best = CUDART_INF_F;
    int32_t best_orig = 0x7fffffff;
    int32_t best_slot = -1;
    const int w = a.window_half;
    const float* __restrict__ hp = a.pos_sorted;
    const float* __restrict__ hc = a.cov_sorted;
    const int64_t ld = a.ld_hit;
    for (int e = (ie - w < 0 ? 0 : ie - w); e <= (ie + w > a.n_eta - 1 ? a.n_eta - 1 : ie + w); ++e) {
        // phi bins p0 .. p0 + 2w (mod n_phi): one run of the sorted array, or two when it wraps
        const int p0 = ((ip - w) % a.n_phi + a.n_phi) % a.n_phi;
        const int p1 = p0 + 2 * w;  // inclusive, may exceed n_phi - 1
        const int row = e * a.n_phi;
        const int nseg = p1 >= a.n_phi ? 2 : 1;
        for (int sgi = 0; sgi < nseg; ++sgi) {
            int32_t s0, s1;
            if (nseg == 1) { s0 = a.bin_offset[row + p0]; s1 = a.bin_offset[row + p1 + 1]; }
            else if (sgi == 0) { s0 = a.bin_offset[row + p0]; s1 = a.bin_offset[row + a.n_phi]; }
            else { s0 = a.bin_offset[row]; s1 = a.bin_offset[row + p1 - a.n_phi + 1]; }
            for (int32_t s = s0 + lane; s < s1; s += 32) {
                LocalHit h;
                hit_to_local(o, __ldg(hp + s), __ldg(hp + ld + s), __ldg(hp + 2 * ld + s), __ldg(hc + s),
                             __ldg(hc + ld + s), __ldg(hc + 2 * ld + s), __ldg(hc + 3 * ld + s),
                             __ldg(hc + 4 * ld + s), __ldg(hc + 5 * ld + s), h);
                Sym3 si;
                const float det = invert_S(n, h, si);
                if (!(det > 0.0f)) continue;
                const float c = chi2_of(si, h);
                const int32_t orig = __ldg(a.sorted_to_orig + s);
                if (better(c, orig, best, best_orig)) { best = c; best_orig = orig; best_slot = s; }
            }
        }
    }
    // warp arg-min on (chi2, original index)
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        const float oc = __shfl_xor_sync(0xffffffffu, best, d);
        const int32_t oo = __shfl_xor_sync(0xffffffffu, best_orig, d);
        const int32_t os = __shfl_xor_sync(0xffffffffu, best_slot, d);
        if (better(oc, oo, best, best_orig)) { best = oc; best_orig = oo; best_slot = os; }
    }
    const bool found = best_slot >= 0;
    const bool accept = found && best < a.chi2_cut;
    bool updated = false;
    uint32_t st_add = 0u;
    float dchi2 = 0.0f;
    if (accept && a.do_update) {
        const int32_t s = best_slot;
        LocalHit h;
        hit_to_local(o, __ldg(hp + s), __ldg(hp + ld + s), __ldg(hp + 2 * ld + s), __ldg(hc + s),
                     __ldg(hc + ld + s), __ldg(hc + 2 * ld + s), __ldg(hc + 3 * ld + s),
                     __ldg(hc + 4 * ld + s), __ldg(hc + 5 * ld + s), h);
        const uint32_t rc = kalman_update(t, o, n, h, &dchi2);
        if (rc == 0u) updated = true; else st_add = rc;
    }
    if (!updated) commit_propagated(t, o, n);
    leave_local_frame(t);
    if (lane == 0) {
        store_track(t, a.par, a.cov, a.ld, i);
        a.best_hit[i] = accept ? best_orig : -1;
        a.best_chi2[i] = best;
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
