// kf_smooth.cu -- backward pass of kf_fit_tracks_smooth: the Rauch-Tung-Striebel recursion (reading A22;
// PAPER.md:57 "a final fit with a KF and smoother") over the filtered states the forward kernel left in the
// per-layer arrays (fit_kernel<2, .> / fit_pair_kernel<2>, kf_fit.cu).
//
// One thread owns one track, outermost layer first.  Per warp, the [6 + 17][32] tile of the filtered local-frame
// states of one layer comes in through TMA into a two-stage ring (stage refilled as soon as its values are in
// registers, so a layer's tile is requested two layers before it is needed); the smoothed state and covariance go
// back to the SAME slots, in global coordinates, as 27 coalesced 4-byte stores per lane.  The arithmetic of one
// step is kf_rts.cuh.  The hits are not read again: the RTS recursion needs the filter's own states only.
//
// Algorithmic HBM bytes of the whole call per track: 113 in + 36 L hits + 120 forward
// result + 4 used mask + 108 L smoothed states.  This implementation moves 92 L more twice (the filtered states,
// written by the forward kernel and read here).
#include "kf_internal.h"
#include "kf_rts.cuh"
#include "kf_tma.cuh"

namespace kf {

namespace {

constexpr int kRtsBlock = 128;
constexpr int kRtsWarps = kRtsBlock / 32;
constexpr int kRtsStages = 2;
constexpr int kRtsRows = 23;                               // 6 state planes + 17 covariance / frame planes
constexpr int kRtsTileFloats = kRtsRows * 32;
constexpr int kRtsSmemBytes = kRtsWarps * kRtsStages * kRtsTileFloats * 4 + kRtsWarps * kRtsStages * 8;

struct RtsMaps {
    CUtensorMap par, cov;
};

__device__ __forceinline__ void filtered_from_tile(Track& t, const float* p) {
    t.x = p[0];        t.y = p[32];       t.z = p[64];       t.px = p[96];      t.py = p[128];     t.pz = p[160];
    t.c11 = p[192];    t.c12 = p[224];    t.c13 = p[256];    t.c14 = p[288];    t.c15 = p[320];
    t.c22 = p[352];    t.c23 = p[384];    t.c24 = p[416];    t.c25 = p[448];
    t.c33 = p[480];    t.c34 = p[512];    t.c35 = p[544];
    t.c44 = p[576];    t.c45 = p[608];
    t.c55 = p[640];
    t.eax = p[672];    t.eay = p[704];
    t.c00 = 0.0f; t.c01 = 0.0f; t.c02 = 0.0f; t.c03 = 0.0f; t.c04 = 0.0f; t.c05 = 0.0f;
}

// state (sx .. spz) + global covariance of g -> slot of layer l
__device__ __forceinline__ void store_smoothed(const FitArgs& a, int l, int64_t i, float sx, float sy, float sz,
                                               float spx, float spy, float spz, const Track& g) {
    // (plane stride as an unsigned 32-bit factor -- launch_rts checks that it fits: every plane address is then one
    // 32 x 32 -> 64-bit multiply-add instead of a 64-bit multiplication, 54 instead of 138 instructions for the 27
    // stores, 11 % of what this issue-bound kernel executed)
    const uint32_t ld = (uint32_t)a.ld_l;
    float* p = a.lpar + (int64_t)l * 6 * a.ld_l + i;
    float* c = a.lcov + (int64_t)l * 21 * a.ld_l + i;
    p[0] = sx; p[ld] = sy; p[2 * ld] = sz; p[3 * ld] = spx; p[4 * ld] = spy; p[5 * ld] = spz;
    c[0] = g.c00;       c[ld] = g.c01;      c[2 * ld] = g.c02;  c[3 * ld] = g.c03;  c[4 * ld] = g.c04;  c[5 * ld] = g.c05;
    c[6 * ld] = g.c11;  c[7 * ld] = g.c12;  c[8 * ld] = g.c13;  c[9 * ld] = g.c14;  c[10 * ld] = g.c15;
    c[11 * ld] = g.c22; c[12 * ld] = g.c23; c[13 * ld] = g.c24; c[14 * ld] = g.c25;
    c[15 * ld] = g.c33; c[16 * ld] = g.c34; c[17 * ld] = g.c35;
    c[18 * ld] = g.c44; c[19 * ld] = g.c45;
    c[20 * ld] = g.c55;
}

// One layer of one track: the RTS step from the smoothed state of layer l_next (or smoothed = filtered at the
// outermost used layer and after a failure), conversion to global coordinates, store, and the state carried on.
template <bool ELOSS>
__device__ __forceinline__ void smooth_one_layer(const Track& t, float k, float ik, const FitParams& P, int model,
                                                 const FitArgs& a, int l, int64_t i, SmoothedNext& nx, int& l_next,
                                                 bool& broken) {
    SmoothedStateT<float> s = {t.x, t.y, t.z, t.px, t.py, t.pz};
    Sym5 Cs;
    sym5_from_track(t, Cs);
    if (l_next >= 0 && !broken) {
        const uint32_t rc = rts_step<float, ELOSS>(t, k, ik, P.layer[l_next], model, P.mass2, P.el, nx, s, Cs);
        if (rc != 0u) {              // cannot happen on a well-posed fit; the layers further in keep the filtered state
            broken = true;
            a.status[i] |= ST_SMOOTH_FAIL;
        }
    }
    Track g;
    sym5_to_global(Cs, t, g);
    store_smoothed(a, l, i, s.x, s.y, s.z, s.px, s.py, s.pz, g);
    nx.x = s.x; nx.y = s.y; nx.z = s.z; nx.px = s.px; nx.py = s.py; nx.pz = s.pz;
    nx.fpx = t.px; nx.fpy = t.py; nx.fpz = t.pz;
    nx.Cs = Cs;
    l_next = l;
}

// The same for geometries with endcap discs (reading A23): the 15 stored covariance values are the upper triangle
// over the layer's live coordinates (barrel: t z b1 b2 c, disc: r t b1 b2 c), see store_layer_state.
__device__ __forceinline__ void filtered_from_tile_surface(Track& t, Sym5& C, const float* p) {
    t.x = p[0];        t.y = p[32];       t.z = p[64];       t.px = p[96];      t.py = p[128];     t.pz = p[160];
    int r = 6;
#pragma unroll
    for (int i = 0; i < 5; ++i)
#pragma unroll
        for (int j = i; j < 5; ++j) { const float v = p[32 * r++]; C.m[i][j] = v; C.m[j][i] = v; }
    t.eax = p[672];    t.eay = p[704];
}

template <bool ELOSS>
__device__ __forceinline__ void smooth_one_layer_surface(const Track& t, const Sym5& C, float k, float ik, const FitParams& P,
                                                         int model, const FitArgs& a, int l, int64_t i, SmoothedNext& nx,
                                                         int& l_next, bool& broken) {
    const int type = P.layer[l].type;
    SmoothedStateT<float> s = {t.x, t.y, t.z, t.px, t.py, t.pz};
    Sym5 Cs = C;
    if (l_next >= 0 && !broken) {
        const uint32_t rc = rts_step_surface<ELOSS>(t, C, type, k, ik, P.layer[l_next], model, P.mass2, P.el, nx, s, Cs);
        if (rc != 0u) {
            broken = true;
            a.status[i] |= ST_SMOOTH_FAIL;
        }
    }
    Track g = t;
    track_from_sym5_surface(Cs, type, g);
    leave_local_frame(g);
    store_smoothed(a, l, i, s.x, s.y, s.z, s.px, s.py, s.pz, g);
    nx.x = s.x; nx.y = s.y; nx.z = s.z; nx.px = s.px; nx.py = s.py; nx.pz = s.pz;
    nx.fpx = t.px; nx.fpy = t.py; nx.fpz = t.pz;
    nx.fax = t.eax; nx.fay = t.eay;
    nx.Cs = Cs;
    l_next = l;
}

#ifndef KF_RTS_MIN_BLOCKS
#define KF_RTS_MIN_BLOCKS 3
#endif
// SURFACES: the geometry has endcap discs (own instantiation: the dense step costs the barrel-only kernel nothing).
template <bool ELOSS, bool SURFACES = false>
__global__ void __launch_bounds__(kRtsBlock, KF_RTS_MIN_BLOCKS)
rts_kernel(const __grid_constant__ FitParams P, const __grid_constant__ RtsMaps M, const FitArgs a) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    const int wid = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    const int64_t i0 = (int64_t)blockIdx.x * kRtsBlock + wid * 32;
    if (i0 >= a.n) return;
    const int L = P.n_layers;
    float* wbase = reinterpret_cast<float*>(smem_raw) + wid * (kRtsStages * kRtsTileFloats);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + kRtsWarps * kRtsStages * kRtsTileFloats * 4) + wid * kRtsStages;
    const uint32_t tile0 = smem_u32(wbase), bar0 = smem_u32(bars);
    const int col = (int)i0;

    // step j carries layer L - 1 - j
    auto request = [&](int step) {
        const int s = step % kRtsStages, l = L - 1 - step;
        const uint32_t dst = tile0 + s * (kRtsTileFloats * 4), bar = bar0 + 8u * s;
        mbar_expect_tx(bar, kRtsTileFloats * 4);
        tma_load_2d(dst, &M.par, col, 6 * l, bar);
        tma_load_2d(dst + 6 * 128, &M.cov, col, 21 * l, bar);
    };
    if (elect_one()) {
#pragma unroll
        for (int s = 0; s < kRtsStages; ++s) mbar_init(bar0 + 8u * s, 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
#pragma unroll
        for (int s = 0; s < kRtsStages; ++s)
            if (s < L) request(s);
    }
    __syncwarp();

    const bool valid = lane < a.n - i0;
    const int64_t i = valid ? i0 + lane : a.n - 1;
    const uint32_t used = valid ? a.used[i] : 0u;
    const float qf = (float)a.q[i];
    const float k = qf * P.k0, ik = qf * P.inv_k0;
    const int model = P.model;

    SmoothedNext nx;
    int l_next = -1;
    bool broken = false;
    for (int step = 0; step < L; ++step) {
        const int s = step % kRtsStages, l = L - 1 - step;
        mbar_wait(bar0 + 8u * s, (uint32_t)(step / kRtsStages) & 1u);
        Track t;
        Sym5 C;
        if constexpr (SURFACES) filtered_from_tile_surface(t, C, wbase + s * kRtsTileFloats + lane);
        else filtered_from_tile(t, wbase + s * kRtsTileFloats + lane);
        __syncwarp();   // every lane holds its values: the stage can be refilled
        if (step + kRtsStages < L && elect_one()) request(step + kRtsStages);
        if (!((used >> l) & 1u)) continue;
        if constexpr (SURFACES) smooth_one_layer_surface<ELOSS>(t, C, k, ik, P, model, a, l, i, nx, l_next, broken);
        else smooth_one_layer<ELOSS>(t, k, ik, P, model, a, l, i, nx, l_next, broken);
    }
}

// (A two-tracks-per-thread form of this kernel -- rts_step is written on the number type F like the filter -- was
// built and measured in round 2: 221 registers without spills, 9 resident warps per SM, results identical, but
// 1.61 ms per 2 M tracks for fit + smoother against 1.38 ms with this one-track kernel: the LDL^T factorisation and
// the row solves are long dependent chains, and with 2.25 warps per scheduler their latency is no longer hidden.
// It was removed again; profiles/r02_counters.md has the numbers.)

// (23.6 KB of dynamic shared memory: below the 48 KB that needs no opt-in)

}  // namespace

cudaError_t launch_rts(const FitParams& P, const FitArgs& a, cudaStream_t stream) {
    if (a.n == 0) return cudaSuccess;
    if (a.ld_l > 0xffffffffLL) return cudaErrorInvalidValue;
    const int L = P.n_layers;
    RtsMaps M;
    if (!make_map(&M.par, a.lpar, a.n, a.ld_l, (int64_t)L * 6, 6) || !make_map(&M.cov, a.lcov, a.n, a.ld_l, (int64_t)L * 21, 17))
        return cudaErrorInvalidValue;
    const int64_t blocks = (a.n + kRtsBlock - 1) / kRtsBlock;
    if (P.has_discs) {
        if (P.model & MODEL_ENERGY_LOSS) rts_kernel<true, true><<<(unsigned)blocks, kRtsBlock, kRtsSmemBytes, stream>>>(P, M, a);
        else rts_kernel<false, true><<<(unsigned)blocks, kRtsBlock, kRtsSmemBytes, stream>>>(P, M, a);
    } else if (P.model & MODEL_ENERGY_LOSS) rts_kernel<true><<<(unsigned)blocks, kRtsBlock, kRtsSmemBytes, stream>>>(P, M, a);
    else rts_kernel<false><<<(unsigned)blocks, kRtsBlock, kRtsSmemBytes, stream>>>(P, M, a);
    return cudaGetLastError();
}

}  // namespace kf
