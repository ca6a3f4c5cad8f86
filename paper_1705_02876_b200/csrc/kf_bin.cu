// kf_bin.cu -- (eta, phi) binning of layer hit pools, and the same counting sort reused to give
// candidates a cache-friendly processing order ("directionally projective bins";
// PAPER.md:135 hits are regrouped on the GPU).
//
// bin = i_eta * n_phi + i_phi, eta = asinh(z / r_layer), phi = atan2(y, x) in [-pi, pi).
// The bin of a hit is an integer decided by floating point, so it is decided in single precision
// against tabulated edges with single-rounded operations only (reading A16b):
//     u = fl(z / r);          i_eta = #{ j in 1..n_eta-1 : u >= fl(sinh(-eta_max + j d_eta)) }
//     upper half plane (y > 0, or y == 0 and x > 0):
//         i_phi = n_phi/2 + #{ j in n_phi/2+1..n_phi-1 : fl(cos_j y) >= fl(sin_j x) }
//     y == 0 and x <= 0:     i_phi = 0
//     lower half plane:      i_phi = #{ j in 1..n_phi/2-1 : fl(cos_j y) >= fl(sin_j x) }
// with (cos_j, sin_j) = fl(cos, sin)(-pi + j d_phi).  No transcendental is evaluated on the GPU.
//
// Two forms of one stable counting sort with bit-identical results: the chunked form further down (large calls on
// hit pools) and this one (small calls, more than 8192 bins, ordering of candidates).
// Counting sort, stable, batched over layers (grid.y = layer, 5 launches + 1 memset for ALL layers):
// (1) key of every item + histogram; the histogram atomic's return value is the item's arrival number inside its
// bin, (2) exclusive scan -> bin_offset, (3) every item goes to slot bin_offset[bin] + arrival number -- no second
// round of atomics -- and, for hits, its nine values are read here, coalesced, and parked as a packed record in
// that slot of a scratch buffer, (4) every slot ranks its index inside its segment (indices are unique, so
// ascending index IS the stable order: the arrival order, which differs from run to run, never shows) and moves
// its record to its final place: a packed 12-float record per hit for the scoring kernel
// (x y z vzz | vxx vxy vyy index | vxz vyz 0 0: the first 128-bit word serves the z pre-filter,
// the second the tangential one, the third only full evaluations); (5) a warp per bin reads the final records and
// writes the optional SoA copies (coalesced) and the per-bin boxes.
// Every read of the inputs is coalesced; the only scattered traffic is one 48-byte record per hit in step (3).
#include <atomic>
#include <cmath>
#include <cstdlib>

#include "kf_internal.h"

namespace kf {

namespace {

constexpr int kBlock = 256;
constexpr double kPi = 3.14159265358979323846;

__device__ __forceinline__ int bin_of_hit(float x, float y, float z, float r, int n_eta, int n_phi,
                                          const float* __restrict__ eta_edge,
                                          const float* __restrict__ phi_cos,
                                          const float* __restrict__ phi_sin) {
    // reading A24: r = 0 says "a disc layer" -- eta from the hit's own rho, every operation rounded once
    if (!(r > 0.0f)) r = __fsqrt_rn(__fadd_rn(__fmul_rn(x, x), __fmul_rn(y, y)));
    const float u = __fdiv_rn(z, r);
    // edges are non-decreasing in j, so "count of edges <= u" is an upper-bound search
    int lo = 1, hi = n_eta;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (u >= eta_edge[mid]) lo = mid + 1; else hi = mid;
    }
    const int ie = lo - 1;
    // The predicate fl(cos_j y) >= fl(sin_j x) says "phi >= edge j" and is true up to the hit's own edge and false
    // beyond it within one half plane (only the edge nearest to the hit is within rounding of the decision, and
    // either answer there keeps the sequence monotone), so the count of true predicates is a bisection.
    const int half = n_phi >> 1;
    int ip = 0;
    if (y > 0.0f || (y == 0.0f && x > 0.0f)) {
        int lo = half + 1, hi = n_phi;      // first j in [half + 1, n_phi) with a false predicate
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (__fmul_rn(phi_cos[mid], y) >= __fmul_rn(phi_sin[mid], x)) lo = mid + 1; else hi = mid;
        }
        ip = lo - 1;
    } else if (y == 0.0f) {
        ip = 0;
    } else {
        int lo = 1, hi = half;              // first j in [1, half)
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (__fmul_rn(phi_cos[mid], y) >= __fmul_rn(phi_sin[mid], x)) lo = mid + 1; else hi = mid;
        }
        ip = lo - 1;
    }
    return ie * n_phi + ip;
}

__global__ void __launch_bounds__(kBlock)
bin_key_kernel(const __grid_constant__ BinBatch B, const float* __restrict__ eta_edge,
               const float* __restrict__ phi_cos, const float* __restrict__ phi_sin) {
    const BinLayerDev& L = B.layer[blockIdx.y];
    const int64_t h = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (h >= L.n) return;
    const int b = bin_of_hit(__ldg(L.pos + h), __ldg(L.pos + L.ld_in + h), __ldg(L.pos + 2 * L.ld_in + h),
                             L.radius, B.n_eta, B.n_phi, eta_edge, phi_cos, phi_sin);
    L.key[h] = b;
    L.pib[h] = atomicAdd(L.counts + b, 1);
}

// Exclusive scan of counts[0..nb) -> bin_offset[0..nb].  One block of 1024 per layer.
__global__ void __launch_bounds__(1024)
bin_scan_kernel(const __grid_constant__ BinBatch B) {
    const BinLayerDev& L = B.layer[blockIdx.y];
    const int nb = B.n_eta * B.n_phi;
    __shared__ int32_t warp_sum[32];
    __shared__ int32_t carry_s;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < nb; base += 1024) {
        const int i = base + tid;
        const int32_t c = i < nb ? L.counts[i] : 0;
        int32_t incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int32_t o = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += o;
        }
        if (lane == 31) warp_sum[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            int32_t s = warp_sum[lane];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int32_t o = __shfl_up_sync(0xffffffffu, s, d);
                if (lane >= d) s += o;
            }
            warp_sum[lane] = s;  // inclusive over warps
        }
        __syncthreads();
        const int32_t carry = carry_s;
        const int32_t excl = carry + (wid ? warp_sum[wid - 1] : 0) + incl - c;
        if (i < nb) L.bin_offset[i] = excl;
        __syncthreads();
        if (tid == 1023) carry_s = excl + c;
        __syncthreads();
    }
    if (tid == 0) L.bin_offset[nb] = carry_s;
}

__global__ void __launch_bounds__(kBlock)
bin_scatter_kernel(const __grid_constant__ BinBatch B) {
    const BinLayerDev& L = B.layer[blockIdx.y];
    const int64_t h = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (h >= L.n) return;
    const int64_t slot = (int64_t)L.bin_offset[L.key[h]] + L.pib[h];
    KF_CHECK(slot >= 0 && slot < L.n);
    L.unsorted[slot] = (int32_t)h;
    if (!L.rec_tmp) return;  // ordering only (candidates)
    float v[9];
#pragma unroll
    for (int k = 0; k < 3; ++k) v[k] = __ldg(L.pos + k * L.ld_in + h);
#pragma unroll
    for (int k = 0; k < 6; ++k) v[3 + k] = __ldg(L.cov + k * L.ld_in + h);
    float4* rec = reinterpret_cast<float4*>(L.rec_tmp + slot * 12);
    rec[0] = make_float4(v[0], v[1], v[2], v[8]);                          // x y z vzz
    rec[1] = make_float4(v[3], v[4], v[6], __int_as_float((int32_t)h));    // vxx vxy vyy, original index
    rec[2] = make_float4(v[5], v[7], 0.0f, 0.0f);                          // vxz vyz
}

// Slot p holds item `mine` of bin b; its final place is bin_offset[b] + #{indices in the segment
// smaller than mine}.  Neighbouring threads scan the same segment, so the loads broadcast.
__global__ void __launch_bounds__(kBlock)
bin_rank_gather_kernel(const __grid_constant__ BinBatch B) {
    const BinLayerDev& L = B.layer[blockIdx.y];
    const int64_t p = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (p >= L.n) return;
    const int32_t mine = L.unsorted[p];
    const int32_t b = L.key[mine];
    const int32_t s = L.bin_offset[b], e = L.bin_offset[b + 1];
    int32_t rank = 0;
    for (int32_t j = s; j < e; ++j) rank += (__ldg(L.unsorted + j) < mine) ? 1 : 0;
    const int64_t dst = (int64_t)s + rank;
    KF_CHECK(dst >= 0 && dst < L.n && rank < e - s);
    if (!L.hit_rec) L.sorted_to_orig[dst] = mine;   // else from the record's index word, coalesced (bin_finish_kernel)
    if (L.orig_to_sorted) L.orig_to_sorted[mine] = (int32_t)dst;
    if (!L.rec_tmp) return;  // ordering only (candidates)
    const float4* src = reinterpret_cast<const float4*>(L.rec_tmp + p * 12);
    const float4 A = src[0], Bw = src[1], C = src[2];
    if (L.hit_rec) {
        float4* rec = reinterpret_cast<float4*>(L.hit_rec + dst * kRecFloats);
        rec[0] = A;
        rec[1] = Bw;
        rec[2] = C;
        if (kRecWords == 4) rec[3] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    }
    if (L.hit_rec) return;   // the SoA copies are then written from the final records, coalesced (bin_finish_kernel)
    if (L.pos_sorted) {
        L.pos_sorted[dst] = A.x; L.pos_sorted[L.ld_out + dst] = A.y; L.pos_sorted[2 * L.ld_out + dst] = A.z;
    }
    if (L.cov_sorted) {   // xx xy xz yy yz zz
        L.cov_sorted[dst] = Bw.x;                 L.cov_sorted[L.ld_out + dst] = Bw.y;
        L.cov_sorted[2 * L.ld_out + dst] = C.x;   L.cov_sorted[3 * L.ld_out + dst] = Bw.z;
        L.cov_sorted[4 * L.ld_out + dst] = C.y;   L.cov_sorted[5 * L.ld_out + dst] = A.w;
    }
}

// Last step, one warp per bin over the final records: sorted_to_orig and the optional SoA copies (the scattered
// store path of an SM is what bounds the sort, so they are written here, where a warp holds CONSECUTIVE slots,
// instead of ten scattered 4-byte stores per hit in the rank step) and the per-bin bounds for the scan's bin pruning: bounding
// box of the hits of the bin and the largest v_zz and v_xx + v_yy (>= the tangential variance in any frame).
// No atomics.  NaN components are ignored (such a hit can never pass a chi2 bound either).  Empty bin: lo = +inf.
__global__ void __launch_bounds__(kBlock)
bin_finish_kernel(const __grid_constant__ BinBatch B) {
    const BinLayerDev& L = B.layer[blockIdx.y];
    if (!L.hit_rec) return;
    const int lane = threadIdx.x & 31;
    const int b = (int)((blockIdx.x * (unsigned)kBlock + threadIdx.x) >> 5);
    if (b >= B.n_eta * B.n_phi) return;
    const int32_t s0 = L.bin_offset[b], s1 = L.bin_offset[b + 1];
    const float inf = __int_as_float(0x7f800000);
    float xl = inf, xh = -inf, yl = inf, yh = -inf, zl = inf, zh = -inf, vz = 0.0f, vt = 0.0f;
    const float4* rec = reinterpret_cast<const float4*>(L.hit_rec);
    for (int32_t s = s0 + lane; s < s1; s += 32) {
        const float4 A = rec[(int64_t)s * kRecWords], Bw = rec[(int64_t)s * kRecWords + 1];
        L.sorted_to_orig[s] = __float_as_int(Bw.w);
        if (L.pos_sorted) {
            L.pos_sorted[s] = A.x; L.pos_sorted[L.ld_out + s] = A.y; L.pos_sorted[2 * L.ld_out + s] = A.z;
        }
        if (L.cov_sorted) {   // xx xy xz yy yz zz
            const float4 C = rec[(int64_t)s * kRecWords + 2];
            L.cov_sorted[s] = Bw.x;                 L.cov_sorted[L.ld_out + s] = Bw.y;
            L.cov_sorted[2 * L.ld_out + s] = C.x;   L.cov_sorted[3 * L.ld_out + s] = Bw.z;
            L.cov_sorted[4 * L.ld_out + s] = C.y;   L.cov_sorted[5 * L.ld_out + s] = A.w;
        }
        xl = fminf(xl, A.x); xh = fmaxf(xh, A.x); yl = fminf(yl, A.y); yh = fmaxf(yh, A.y);
        zl = fminf(zl, A.z); zh = fmaxf(zh, A.z); vz = fmaxf(vz, A.w); vt = fmaxf(vt, Bw.x + Bw.z);
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        xl = fminf(xl, __shfl_xor_sync(0xffffffffu, xl, d)); xh = fmaxf(xh, __shfl_xor_sync(0xffffffffu, xh, d));
        yl = fminf(yl, __shfl_xor_sync(0xffffffffu, yl, d)); yh = fmaxf(yh, __shfl_xor_sync(0xffffffffu, yh, d));
        zl = fminf(zl, __shfl_xor_sync(0xffffffffu, zl, d)); zh = fmaxf(zh, __shfl_xor_sync(0xffffffffu, zh, d));
        vz = fmaxf(vz, __shfl_xor_sync(0xffffffffu, vz, d)); vt = fmaxf(vt, __shfl_xor_sync(0xffffffffu, vt, d));
    }
    if (lane == 0 && L.bin_box) {
        float4* o = reinterpret_cast<float4*>(L.bin_box + (int64_t)b * 8);
        o[0] = make_float4(xl, xh, yl, yh);
        o[1] = make_float4(zl, zh, vz, vt);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Chunked form of the same stable counting sort for hit pools (three launches + the finish step, every record
// written ONCE): a layer is cut into chunks of kChunk consecutive hits, one CTA per chunk.
//   chunk_count   bin of every hit (first guess from a look-up table, corrected against the edge tables); shared-
//                 memory histogram of the chunk; every hit counts the smaller indices among the hits of its bin = its
//                 stable rank INSIDE the chunk (the arrival order of the shared-memory atomics never shows; peer lists
//                 of four per bin + a short overflow list, bucket lists for coarse grids); one word per hit
//                 (bin << 16 | rank) and the chunk's histogram go to global memory.  512 threads x 4 hits: the kernel
//                 is one wave of CTAs and its duration the instruction chain of a warp (~370 per hit with bisections
//                 and bucket lists), so fewer hits per thread and fewer instructions per hit = a shorter kernel
//   chunk_prefix  per bin: prefix of the chunk histograms over the chunks (chunks are consecutive index ranges, so
//                 earlier chunk = smaller index) and the bin total; four warps per column, a quarter of the chunks
//                 each, so that a whole column is in flight at once
//   chunk_place   every CTA scans the bin totals itself (-> bin_offset, handed to the caller by chunk 0); final slot
//                 = bin_offset[bin] + hits of the bin in earlier chunks + rank inside the chunk; the nine values are
//                 read coalesced, four hits in flight per thread, and the packed record goes straight to its final place
// Same results as the five-launch path, bit for bit.  Limits: n_bins <= kChunkMaxBins (shared memory).
// Measured on configs[4] (7 x 120 000 hits, graph replay, no SoA copies), warm incremental cost per kernel:
// count 17.7, prefix 3.5, place 16.2, finish 8.6 us = 46 us (round-2 start: 19.5 / 8.2 (+ scan) / 13.9 / 8.6 = 50);
// with the peer lists and the look-up-table guesses in the count step: 43.7 us.
#ifndef KF_BIN_CHUNK
#define KF_BIN_CHUNK 2048
#endif

// In-place exclusive scan of a[0 .. n) in shared memory by a block of THREADS threads (thread t owns a contiguous
// range); returns the total to every thread.  wsum: THREADS / 32 words of shared memory.  Ends with a barrier.
template <int THREADS>
__device__ __forceinline__ int32_t block_exclusive_scan(int32_t* a, int n, int32_t* wsum) {
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int per = (n + THREADS - 1) / THREADS;
    const int r0 = tid * per < n ? tid * per : n, r1 = r0 + per < n ? r0 + per : n;
    int32_t sum = 0;
    for (int i = r0; i < r1; ++i) sum += a[i];
    int32_t incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int32_t o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) wsum[wid] = incl;
    __syncthreads();
    int32_t run = incl - sum, total = 0;
#pragma unroll
    for (int w = 0; w < THREADS / 32; ++w) {
        const int32_t v = wsum[w];
        run += w < wid ? v : 0;
        total += v;
    }
    for (int i = r0; i < r1; ++i) { const int32_t c = a[i]; a[i] = run; run += c; }
    __syncthreads();
    return total;
}
constexpr int kChunk = KF_BIN_CHUNK;
constexpr int kChunkBlock = kChunk / 8;     // chunk_place_kernel: 8 hits per thread
constexpr int kChunkPer = kChunk / kChunkBlock;
#ifndef KF_BIN_COUNT_PER
#define KF_BIN_COUNT_PER 4
#endif
constexpr int kCountPer = KF_BIN_COUNT_PER;  // chunk_count_kernel: hits per thread.  The kernel is one wave of CTAs and a warp runs
constexpr int kCountBlock = kChunk / kCountPer;   // ~370 instructions per hit one after the other, so its duration is the
                                                  // length of that chain: 4 hits per thread (512 threads) instead of 8
constexpr int kChunkMaxBins = 8192;

__global__ void __launch_bounds__(kCountBlock)
chunk_count_kernel(const __grid_constant__ BinBatch B, const float* __restrict__ eta_edge_g,
                   const float* __restrict__ phi_cos_g, const float* __restrict__ phi_sin_g,
                   const int32_t* __restrict__ lut_g, float lut_u0, float lut_uscale) {
    const BinLayerDev& L = B.layer[blockIdx.y];
    const int c = blockIdx.x;
    const int64_t h0 = (int64_t)c * kChunk;
    if (h0 >= L.n) return;
    const int m = (int)(L.n - h0 < kChunk ? L.n - h0 : kChunk);
    const int nb = B.n_eta * B.n_phi;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int32_t* cnt = reinterpret_cast<int32_t*>(smem_raw);              // [nb] histogram of the chunk
    int32_t* loc = cnt + nb;                                           // [nb] start of each bin's bucket (+ [nb] spare: peer lists)
    uint32_t* ka = reinterpret_cast<uint32_t*>(loc + 2 * nb);          // [kChunk] bin << 16 | arrival number
    uint16_t* bucket = reinterpret_cast<uint16_t*>(ka + kChunk);       // [kChunk] chunk-local hit indices by bin
    float* eta_edge = reinterpret_cast<float*>(bucket + kChunk);       // [n_eta] [n_phi] [n_phi]
    float* phi_cos = eta_edge + B.n_eta;
    float* phi_sin = phi_cos + B.n_phi;
    __shared__ int32_t wsum[kCountBlock / 32];
    __shared__ uint16_t lut[3 * kLutCells];
    for (int i = tid; i < 3 * kLutCells; i += kCountBlock) lut[i] = (uint16_t)lut_g[i];
    // histogram = 0, peer lists = empty (0xffff); 16 bytes per store where the grid allows it
    const bool vec4 = (nb & 3) == 0;
    if (vec4) {
        for (int i = tid; i < nb / 4; i += kCountBlock) reinterpret_cast<int4*>(cnt)[i] = make_int4(0, 0, 0, 0);
        for (int i = tid; i < nb / 2; i += kCountBlock) reinterpret_cast<uint4*>(loc)[i] = make_uint4(~0u, ~0u, ~0u, ~0u);
    } else {
        for (int i = tid; i < nb; i += kCountBlock) { cnt[i] = 0; reinterpret_cast<uint2*>(loc)[i] = make_uint2(~0u, ~0u); }
    }
    for (int i = tid; i < B.n_eta; i += kCountBlock) eta_edge[i] = eta_edge_g[i];
    for (int i = tid; i < B.n_phi; i += kCountBlock) { phi_cos[i] = phi_cos_g[i]; phi_sin[i] = phi_sin_g[i]; }
    __syncthreads();
    // The bin rule of bin_of_hit for this thread's kCountPer hits at once: all loads first, then the two searches.
    {
        float x[kCountPer], y[kCountPer], u[kCountPer];
        int pe[kCountPer], pp[kCountPer], lim[kCountPer];
        const int half = B.n_phi >> 1;
#pragma unroll
        for (int it = 0; it < kCountPer; ++it) {
            const int li = tid + it * kCountBlock;
            const int64_t h = h0 + (li < m ? li : 0);
            x[it] = __ldg(L.pos + h); y[it] = __ldg(L.pos + L.ld_in + h);
            u[it] = __ldg(L.pos + 2 * L.ld_in + h);
        }
#pragma unroll
        for (int it = 0; it < kCountPer; ++it) {
            const float rr = L.radius > 0.0f ? L.radius      // (reading A24: radius 0 = a disc layer, the hit's own rho)
                                             : __fsqrt_rn(__fadd_rn(__fmul_rn(x[it], x[it]), __fmul_rn(y[it], y[it])));
            u[it] = __fdiv_rn(u[it], rr);
            const bool upper = y[it] > 0.0f || (y[it] == 0.0f && x[it] > 0.0f);
            pe[it] = 0;
            pp[it] = upper ? half : 0;
            lim[it] = upper ? B.n_phi - 1 : (y[it] == 0.0f ? 0 : half - 1);
        }
        // First guess from the look-up tables, then the exact rule: the largest index whose predicate holds, found
        // by stepping up while the next edge is still below the hit and down while the own edge is above it (the
        // predicates are monotone in the index, so this is the count the rule asks for -- the same answer as a
        // bisection, for ~25 instructions per hit instead of ~95; a NaN makes every predicate false: index 0 / start).
        const int ne1 = B.n_eta - 1;
#pragma unroll
        for (int it = 0; it < kCountPer; ++it) {
            int ce = __float2int_rd((u[it] - lut_u0) * lut_uscale);
            ce = ce < 0 ? 0 : (ce > kLutCells - 1 ? kLutCells - 1 : ce);
            int g = lut[ce];
            g = g > ne1 ? ne1 : g;
            // the guess is the bin or the one below it: one look at the next edge, one at the edge that then decides
            const bool up = g < ne1 && u[it] >= eta_edge[g + 1];
            g += up ? 1 : 0;
            const int pi = up ? (g < ne1 ? g + 1 : ne1) : g;
            const bool ge = u[it] >= eta_edge[pi];
            if (up ? (g < ne1 && ge) : (g > 0 && !ge)) {          // rare: further than one bin off (coarse table, NaN)
                while (g < ne1 && u[it] >= eta_edge[g + 1]) ++g;
                while (g > 0 && !(u[it] >= eta_edge[g])) --g;
            }
            pe[it] = g;
        }
#pragma unroll
        for (int it = 0; it < kCountPer; ++it) {
            const bool upper = pp[it] != 0;                    // (pp = start of the search: half in the upper half plane)
            const float t = __fdividef(x[it], fabsf(x[it]) + fabsf(y[it]));
            int cp = __float2int_rd((upper ? 1.0f - t : 1.0f + t) * (0.5f * kLutCells));
            cp = cp < 0 ? 0 : (cp > kLutCells - 1 ? kLutCells - 1 : cp);
            const int start = pp[it], hi = lim[it];
            int g = lut[(upper ? 2 * kLutCells : kLutCells) + cp];
            g = g < start ? start : (g > hi ? hi : g);
            const int n1 = g < hi ? g + 1 : hi;
            const bool up = g < hi && __fmul_rn(phi_cos[n1], y[it]) >= __fmul_rn(phi_sin[n1], x[it]);
            g += up ? 1 : 0;
            const int pi = up ? (g < hi ? g + 1 : hi) : g;
            const bool ge = __fmul_rn(phi_cos[pi], y[it]) >= __fmul_rn(phi_sin[pi], x[it]);
            if (up ? (g < hi && ge) : (g > start && !ge)) {
                while (g < hi && __fmul_rn(phi_cos[g + 1], y[it]) >= __fmul_rn(phi_sin[g + 1], x[it])) ++g;
                while (g > start && !(__fmul_rn(phi_cos[g], y[it]) >= __fmul_rn(phi_sin[g], x[it]))) --g;
            }
            pp[it] = g;
        }
#pragma unroll
        for (int it = 0; it < kCountPer; ++it) {
            const int li = tid + it * kCountBlock;
            if (li < m) {
                const int b = pe[it] * B.n_phi + pp[it];
                ka[li] = ((uint32_t)b << 16) | (uint32_t)atomicAdd(cnt + b, 1);
            }
        }
    }
    __syncthreads();
    // Stable rank inside the chunk = number of smaller indices among the hits of the same bin.
    // Fast form (taken when at most kOverflowMax hits of the chunk arrived in their bin behind kPeers others, which
    // is every chunk of a grid as fine as configs[4]'s: 0.8 hits per bin and chunk): the first kPeers arrivals of a
    // bin are kept in peer[arrival][bin], later ones in a short overflow list; a hit compares itself with the
    // (at most kPeers) peers of its bin and, if the bin has more, with the overflow entries of that bin.  No scan
    // over the bins, no bucket lists.  Otherwise (coarse grids, all hits in one bin ...) the general form below.
    {
        constexpr int kPeers = 4, kOverflowMax = 64;
        static_assert(kPeers == 4 && kChunk < 65535, "peer lists: four 16-bit indices per bin, 0xffff = empty");
        uint16_t* peer = reinterpret_cast<uint16_t*>(loc);              // [nb][kPeers], in the loc + spare area, preset to 0xffff
        __shared__ int32_t n_over_s;
        __shared__ uint32_t over[kOverflowMax];                          // bin << 16 | chunk-local index
        if (tid == 0) n_over_s = 0;
        __syncthreads();
#pragma unroll
        for (int it = 0; it < kCountPer; ++it) {
            const int li = tid + it * kCountBlock;
            if (li < m) {
                const uint32_t k = ka[li];
                const int b = (int)(k >> 16), a = (int)(k & 0xffffu);
                KF_CHECK(b >= 0 && b < nb);
                if (a < kPeers) peer[b * kPeers + a] = (uint16_t)li;
                else {
                    const int32_t j = atomicAdd(&n_over_s, 1);
                    if (j < kOverflowMax) over[j] = ((uint32_t)b << 16) | (uint32_t)li;
                }
            }
        }
        __syncthreads();
        const int n_over = n_over_s;
        if (n_over <= kOverflowMax) {
#pragma unroll
            for (int it = 0; it < kCountPer; ++it) {
                const int li = tid + it * kCountBlock;
                if (li < m) {
                    const int b = (int)(ka[li] >> 16);
                    const uint2 p = reinterpret_cast<const uint2*>(peer)[b];       // the bin's four peers (0xffff: none)
                    const uint32_t me = (uint32_t)li;
                    int rank = ((p.x & 0xffffu) < me ? 1 : 0) + ((p.x >> 16) < me ? 1 : 0) +
                               ((p.y & 0xffffu) < me ? 1 : 0) + ((p.y >> 16) < me ? 1 : 0);
                    if ((p.y >> 16) != 0xffffu && n_over > 0)                     // four or more: some may be in the overflow list
                        for (int j = 0; j < n_over; ++j) {
                            const uint32_t o = over[j];
                            rank += ((int)(o >> 16) == b && (int)(o & 0xffffu) < li) ? 1 : 0;
                        }
                    L.key[h0 + li] = (b << 16) | rank;     // one word per hit for chunk_place_kernel (rank < kChunk <= 65536, b < 8192)
                }
            }
            if (vec4) {                                                           // [chunk][bin]
                int4* row = reinterpret_cast<int4*>(L.chunk_cnt + (int64_t)c * nb);
                for (int i = tid; i < nb / 4; i += kCountBlock) row[i] = reinterpret_cast<const int4*>(cnt)[i];
            } else {
                for (int b = tid; b < nb; b += kCountBlock) L.chunk_cnt[(int64_t)c * nb + b] = cnt[b];
            }
            return;
        }
        __syncthreads();                                                 // (the general form reuses the peer area as loc)
    }
    // exclusive scan of cnt -> loc: thread t owns the bins [r0, r1)
    const int per = (nb + kCountBlock - 1) / kCountBlock;
    const int r0 = tid * per < nb ? tid * per : nb, r1 = r0 + per < nb ? r0 + per : nb;
    int32_t sum = 0;
    for (int b = r0; b < r1; ++b) { loc[b] = sum; sum += cnt[b]; }
    int32_t incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int32_t o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) wsum[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        int32_t w = lane < kCountBlock / 32 ? wsum[lane] : 0;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int32_t o = __shfl_up_sync(0xffffffffu, w, d);
            if (lane >= d) w += o;
        }
        if (lane < kCountBlock / 32) wsum[lane] = w;   // inclusive over warps
    }
    __syncthreads();
    const int32_t excl = (wid ? wsum[wid - 1] : 0) + incl - sum;
    for (int b = r0; b < r1; ++b) loc[b] += excl;
    __syncthreads();
#pragma unroll
    for (int it = 0; it < kCountPer; ++it) {
        const int li = tid + it * kCountBlock;
        if (li < m) { const uint32_t k = ka[li]; bucket[loc[k >> 16] + (int)(k & 0xffffu)] = (uint16_t)li; }
    }
    __syncthreads();
#pragma unroll
    for (int it = 0; it < kCountPer; ++it) {
        const int li = tid + it * kCountBlock;
        if (li < m) {
            const int b = (int)(ka[li] >> 16);
            const int s0 = loc[b], s1 = s0 + cnt[b];
            int rank = 0;
            for (int j = s0; j < s1; ++j) rank += bucket[j] < (uint16_t)li ? 1 : 0;
            L.key[h0 + li] = (b << 16) | rank;     // one word per hit for chunk_place_kernel (rank < kChunk <= 65536, b < 8192)
        }
    }
    for (int b = tid; b < nb; b += kCountBlock) L.chunk_cnt[(int64_t)c * nb + b] = cnt[b];   // [chunk][bin]
}

// A thread per bin: chunk_cnt[c][b] becomes the number of hits of bin b in chunks before c (sixteen independent
// loads in flight at a time); the bin total goes to counts[b].  bin_offset = the exclusive scan of the totals is
// made by every CTA of chunk_place_kernel for itself (a microsecond of a kernel that has to read the totals anyway;
// as a launch of its own, one CTA per layer, it took 5 us, and as the last-CTA-done tail of this kernel 3.5 us).
__global__ void __launch_bounds__(128)
chunk_prefix_kernel(const __grid_constant__ BinBatch B) {
    const BinLayerDev& L = B.layer[blockIdx.y];
    const int nb = B.n_eta * B.n_phi;
    const int nc = (int)((L.n + kChunk - 1) / kChunk);
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    // A CTA owns 32 bins; warp g takes the g-th quarter of the chunks (a contiguous range, so the four partial
    // prefixes chain through shared memory): the column of a bin is read by four threads at once and a whole
    // quarter of it is in flight per thread -- one round trip to L2 instead of four for configs[4]'s 59 chunks.
    const int b = blockIdx.x * 32 + lane;
    const int Q = (nc + 3) / 4;
    const int c_lo = wid * Q < nc ? wid * Q : nc, c_hi = c_lo + Q < nc ? c_lo + Q : nc;
    __shared__ int32_t part[4][32];
    int32_t tot = 0;
    if (b < nb) {
        int32_t* col = L.chunk_cnt + b;            // [chunk][bin]: neighbouring lanes, neighbouring words
        for (int c0 = c_lo; c0 < c_hi; c0 += 16) {
            int32_t v[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) v[k] = c0 + k < c_hi ? col[(int64_t)(c0 + k) * nb] : 0;
#pragma unroll
            for (int k = 0; k < 16; ++k) tot += v[k];
        }
    }
    part[wid][lane] = tot;
    __syncthreads();
    if (b < nb) {
        int32_t run = 0;
        for (int g = 0; g < wid; ++g) run += part[g][lane];
        int32_t* col = L.chunk_cnt + b;
        for (int c0 = c_lo; c0 < c_hi; c0 += 16) {   // second pass over the quarter: the words are in L1 / L2 now
            int32_t v[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) v[k] = c0 + k < c_hi ? col[(int64_t)(c0 + k) * nb] : 0;
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                if (c0 + k < c_hi) col[(int64_t)(c0 + k) * nb] = run;
                run += v[k];
            }
        }
        if (wid == 3) L.counts[b] = part[0][lane] + part[1][lane] + part[2][lane] + part[3][lane];
    }
}

__global__ void __launch_bounds__(kChunkBlock, 4)
chunk_place_kernel(const __grid_constant__ BinBatch B) {
    const BinLayerDev& L = B.layer[blockIdx.y];
    const int c = blockIdx.x;
    const int64_t h0 = (int64_t)c * kChunk;
    if (h0 >= L.n && c != 0) return;                         // (chunk 0 of an EMPTY layer still owes the caller bin_offset)
    const int m = h0 >= L.n ? 0 : (int)(L.n - h0 < kChunk ? L.n - h0 : kChunk);
    const int nb = B.n_eta * B.n_phi;
    const int tid = threadIdx.x;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int32_t* base = reinterpret_cast<int32_t*>(smem_raw);   // [nb] final slot of this chunk's first hit of a bin
    // Per warp: 32 records staged in shared memory and written out kRecWords lanes to a record, so that one store
    // instruction covers whole records (with 64-byte records: two whole sectors each) instead of 32 separate
    // 16-byte pieces.
    __shared__ __align__(16) float4 stage[kChunkBlock / 32][32 * kRecWords];
    __shared__ int32_t stage_dst[kChunkBlock / 32][32];
    const int lane = tid & 31, wid = tid >> 5;
    __shared__ int32_t wsum[kChunkBlock / 32];
    for (int b = tid; b < nb; b += kChunkBlock) base[b] = L.counts[b];      // the layer's hits per bin (chunk_prefix_kernel)
    __syncthreads();
    const int32_t total = block_exclusive_scan<kChunkBlock>(base, nb, wsum);     // = bin_offset
    if (c == 0) {                                                           // one CTA per layer hands it to the caller
        for (int b = tid; b < nb; b += kChunkBlock) L.bin_offset[b] = base[b];
        if (tid == 0) L.bin_offset[nb] = total;
    }
    if (m == 0) return;
    __syncthreads();
    for (int b = tid; b < nb; b += kChunkBlock) base[b] += L.chunk_cnt[(int64_t)c * nb + b];
    __syncthreads();
    // The loads of kPlaceBatch hits (9 values + the key word each) are issued together: the kernel is one wave of
    // CTAs, so its duration is a CTA's latency, and eight dependent round trips to memory were most of it.  Four at
    // a time keeps the kernel at 64 registers = 4 CTAs per SM = every chunk of configs[4] resident at once (all
    // eight at a time: 128 registers, two waves, slower on configs[4] although faster beyond the L2 size).
    constexpr int kPlaceBatch = 4;
    static_assert(kChunkPer % kPlaceBatch == 0, "chunk_place_kernel batches");
    for (int it0 = 0; it0 < kChunkPer; it0 += kPlaceBatch) {
        float v[kPlaceBatch][9];
        int32_t kr[kPlaceBatch];
#pragma unroll
        for (int j = 0; j < kPlaceBatch; ++j) {
            const int li = tid + (it0 + j) * kChunkBlock;        // (a warp's 32 hits are consecutive)
            const int64_t h = h0 + (li < m ? li : 0);
            kr[j] = __ldg(L.key + h);                            // bin << 16 | rank inside the chunk (chunk_count_kernel)
#pragma unroll
            for (int k = 0; k < 3; ++k) v[j][k] = __ldg(L.pos + k * L.ld_in + h);
#pragma unroll
            for (int k = 0; k < 6; ++k) v[j][3 + k] = __ldg(L.cov + k * L.ld_in + h);
        }
#pragma unroll
        for (int j = 0; j < kPlaceBatch; ++j) {
            const int li = tid + (it0 + j) * kChunkBlock;
            int32_t dst = -1;
            if (li < m) {
                const int64_t h = h0 + li;
                KF_CHECK((kr[j] >> 16) >= 0 && (kr[j] >> 16) < nb);
                dst = base[kr[j] >> 16] + (kr[j] & 0xffff);
                KF_CHECK(dst >= 0 && dst < L.n);
                if (L.orig_to_sorted) L.orig_to_sorted[h] = dst;
                stage[wid][lane * kRecWords + 0] = make_float4(v[j][0], v[j][1], v[j][2], v[j][8]);                       // x y z vzz
                stage[wid][lane * kRecWords + 1] = make_float4(v[j][3], v[j][4], v[j][6], __int_as_float((int32_t)h));    // vxx vxy vyy, index
                stage[wid][lane * kRecWords + 2] = make_float4(v[j][5], v[j][7], 0.0f, 0.0f);                             // vxz vyz
                if (kRecWords == 4) stage[wid][lane * kRecWords + 3] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            }
            stage_dst[wid][lane] = dst;
            __syncwarp();
#pragma unroll
            for (int r = 0; r < kRecWords; ++r) {
                const int w = r * 32 + lane, rec = w / kRecWords, part = w - rec * kRecWords;
                const int32_t d = stage_dst[wid][rec];
                if (d >= 0) reinterpret_cast<float4*>(L.hit_rec + (int64_t)d * kRecFloats)[part] = stage[wid][w];
            }
            __syncwarp();
        }
    }
}

// Candidate keys for kf_order_candidates: the (eta, phi) bin of the candidate's crossing with the layer
// (definition formula in fp32; the order only steers cache locality, never a result).
__global__ void __launch_bounds__(kBlock)
cand_key_kernel(const __grid_constant__ FitParams P, int layer, int64_t n, int64_t ld,
                const float* __restrict__ par, const int8_t* __restrict__ q, int n_eta, int n_phi,
                float eta_max, int32_t* __restrict__ key, int32_t* __restrict__ pib,
                int32_t* __restrict__ counts) {
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i >= n) return;
    Track t;
    t.x = __ldg(par + i);           t.y = __ldg(par + ld + i);      t.z = __ldg(par + 2 * ld + i);
    t.px = __ldg(par + 3 * ld + i); t.py = __ldg(par + 4 * ld + i); t.pz = __ldg(par + 5 * ld + i);
    t.eax = 1.0f; t.eay = 0.0f;
    const float qf = (float)q[i];
    float x = t.x, y = t.y, z = t.z;
    if (P.layer[layer].type == 1) {            // a disc layer (readings A23 / A24)
        DiscCrossing o;
        const uint32_t rc = helix_to_plane(t, qf * P.k0, qf * P.inv_k0, P.layer[layer], o);
        if (rc == 0u || rc == ST_OUTSIDE) { x = o.xn; y = o.yn; z = o.zt; }
    } else {
        Crossing o;
        if (helix_to_radius(t, qf * P.k0, qf * P.inv_k0, P.layer[layer], o)) { x = o.xn; y = o.yn; z = o.zn; }
    }
    const float rho = sqrtf(x * x + y * y);
    const float eta = asinhf(z / fmaxf(rho, 1e-20f));
    const float phi = atan2f(y, x);
    int ie = (int)floorf((eta + eta_max) / (2.0f * eta_max / (float)n_eta));
    ie = ie < 0 ? 0 : (ie > n_eta - 1 ? n_eta - 1 : ie);          // NaN -> 0 through the casts below
    int ip = (int)floorf((phi + 3.14159265358979f) / (6.28318530717959f / (float)n_phi));
    ip = ((ip % n_phi) + n_phi) % n_phi;
    int b = ie * n_phi + ip;
    if (!(b >= 0 && b < n_eta * n_phi)) b = 0;
    key[i] = b;
    pib[i] = atomicAdd(counts + b, 1);
}

}  // namespace

cudaError_t BinScratch::reserve(int64_t n_items, int64_t n_bins, cudaStream_t stream, bool records) {
    const bool grow_rec = records && n_items > cap_rec;
    if (n_items <= cap_items && n_bins <= cap_bins && !grow_rec) return cudaSuccess;
    // growing: drain the stream that may still use the old buffers, then reallocate
    cudaError_t e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return e;
    const int64_t ni = n_items > cap_items ? n_items : cap_items;
    const int64_t nb = n_bins > cap_bins ? n_bins : cap_bins;
    const bool want_rec = records || cap_rec > 0;
    release();
    ++gen;
    const size_t items_b = (size_t)(ni > 0 ? ni : 1) * sizeof(int32_t);
    const size_t bins_b = (size_t)(nb > 0 ? nb : 1) * sizeof(int32_t);
    const size_t tab_b = (size_t)(KF_MAX_BINS_INTERNAL + 1) * sizeof(float);
    if ((e = cudaMalloc(&key, items_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&unsorted, items_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&pib, items_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&counts, bins_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&eta_edge, tab_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&phi_cos, tab_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&phi_sin, tab_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&guess_lut, (size_t)3 * kLutCells * sizeof(int32_t))) != cudaSuccess) { release(); return e; }
    if (want_rec) {
        if ((e = cudaMalloc(&rec_tmp, (size_t)(ni > 0 ? ni : 1) * 12 * sizeof(float))) != cudaSuccess) { release(); return e; }
        cap_rec = ni;
    }
    cap_items = ni;
    cap_bins = nb;
    return cudaSuccess;
}

cudaError_t BinScratch::reserve_chunk_cnt(int64_t words, cudaStream_t stream) {
    if (words <= cap_chunk_cnt) return cudaSuccess;
    cudaError_t e = cudaStreamSynchronize(stream);   // the old buffer may still be in use
    if (e != cudaSuccess) return e;
    if (chunk_cnt) cudaFree(chunk_cnt);
    chunk_cnt = nullptr;
    cap_chunk_cnt = 0;
    ++gen;
    if ((e = cudaMalloc(&chunk_cnt, (size_t)words * sizeof(int32_t))) != cudaSuccess) return e;
    cap_chunk_cnt = words;
    return cudaSuccess;
}

void BinScratch::release() {
    void* ptrs[] = {key, unsorted, pib, counts, eta_edge, phi_cos, phi_sin, rec_tmp, chunk_cnt, guess_lut};
    for (void* p : ptrs)
        if (p) cudaFree(p);
    key = unsorted = pib = counts = nullptr;
    eta_edge = phi_cos = phi_sin = nullptr;
    guess_lut = nullptr;
    rec_tmp = nullptr;
    chunk_cnt = nullptr;
    cap_chunk_cnt = 0;
    cap_items = 0;
    cap_bins = 0;
    cap_rec = 0;
    tab_n_eta = tab_n_phi = 0;
    tab_eta_max = 0.0f;
}

// Edge tables, evaluated in double on the host and rounded once to float (reading A16b).
cudaError_t BinScratch::tables(int n_eta, int n_phi, float eta_max, cudaStream_t stream) {
    if (n_eta == tab_n_eta && n_phi == tab_n_phi && eta_max == tab_eta_max) return cudaSuccess;
    // the previous tables may still be in use by queued kernels, and host_tab by a queued copy
    cudaError_t e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return e;
    ++gen;   // a recorded graph that bins with the old tables is stale from here on
    host_tab.assign((size_t)n_eta + 2 * (size_t)n_phi, 0.0f);
    float* he = host_tab.data();
    float* hc = he + n_eta;
    float* hs = hc + n_phi;
    const double em = (double)eta_max;
    const double d_eta = 2.0 * em / n_eta, d_phi = 2.0 * kPi / n_phi;
    for (int j = 1; j < n_eta; ++j) he[j] = (float)std::sinh(-em + j * d_eta);
    for (int j = 0; j < n_phi; ++j) {
        hc[j] = (float)std::cos(-kPi + j * d_phi);
        hs[j] = (float)std::sin(-kPi + j * d_phi);
    }
    if ((e = cudaMemcpyAsync(eta_edge, he, (size_t)n_eta * 4, cudaMemcpyHostToDevice, stream)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(phi_cos, hc, (size_t)n_phi * 4, cudaMemcpyHostToDevice, stream)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(phi_sin, hs, (size_t)n_phi * 4, cudaMemcpyHostToDevice, stream)) != cudaSuccess) return e;
    // First guesses for chunk_count_kernel's searches (any guess is corrected there against the tables above, in both
    // directions, so these only have to be close): eta over kLutCells cells of u = z / r, phi over kLutCells cells of
    // the "diamond angle" x / (|x| + |y|) per half plane.
    {
        host_lut.assign((size_t)3 * kLutCells, 0);
        const float u0 = (float)std::sinh(-em), u1 = (float)std::sinh(em);
        lut_u0 = u0;
        lut_uscale = (float)((double)kLutCells / ((double)u1 - (double)u0));
        const int half = n_phi / 2;
        for (int c = 0; c < kLutCells; ++c) {
            const double lo = (double)u0 + (double)c / (double)lut_uscale;
            int g = 0;
            for (int j = 1; j < n_eta; ++j) g += (double)he[j] <= lo ? 1 : 0;
            host_lut[c] = g;
            const double tl = -1.0 + 2.0 * c / kLutCells, tu = 1.0 - 2.0 * c / kLutCells;
            const double pl = -std::atan2(1.0 - std::fabs(tl), tl), pu = std::atan2(1.0 - std::fabs(tu), tu);
            int gl = 0, gu = half;
            for (int j = 1; j < half; ++j) gl += (-kPi + j * d_phi) <= pl ? 1 : 0;
            for (int j = half + 1; j < n_phi; ++j) gu += (-kPi + j * d_phi) <= pu ? 1 : 0;
            host_lut[kLutCells + c] = gl;
            host_lut[2 * kLutCells + c] = gu;
        }
        if ((e = cudaMemcpyAsync(guess_lut, host_lut.data(), host_lut.size() * sizeof(int32_t), cudaMemcpyHostToDevice, stream)) != cudaSuccess) return e;
    }
    tab_n_eta = n_eta;
    tab_n_phi = n_phi;
    tab_eta_max = eta_max;
    return cudaSuccess;
}

// The chunked sort for a group of layers, when it applies (hit pools with packed records, n_bins within the
// shared-memory limit, enough hits to pay).
namespace {

size_t chunk_count_smem(int n_eta, int n_phi) {
    return (size_t)3 * n_eta * n_phi * 4 + (size_t)kChunk * 6 + ((size_t)n_eta + 2 * (size_t)n_phi) * 4;   // (+ static: lut, wsum, overflow)
}

int64_t chunk_cnt_words(int64_t chunks, int nb) { return (chunks > 0 ? chunks : 1) * (int64_t)nb; }

// Option bin_form (kf_set_option KF_OPT_BIN_FORM; the tests switch between the two forms): 1 = never,
// 2 = wherever it applies, 0 = where it pays, i.e. groups of at least kChunkedMinHits hits (7 pools, chunked
// against five-launch: 126 000 hits 36 / 32 us, 210 000 hits 37 / 38 us, 336 000 hits 41 / 48 us, 840 000 hits
// 62 / 101 us; one pool of 120 000 hits 33 / 32 us).
constexpr int64_t kChunkedMinHits = 3 << 16;   // measured crossover on 7 pools of 40 x 64 bins: 180 000 - 210 000 hits

bool chunked_wanted(int64_t total_hits, int bin_form) {
    if (bin_form == 1 || (bin_form == 0 && total_hits < kChunkedMinHits)) return false;
    return ensure_bin_attributes() == cudaSuccess;
}

// returns cudaSuccess and *done = true if the group was sorted here
cudaError_t try_chunk_sort(BinScratch& s, BinBatch& B, int m, int64_t group_max, cudaStream_t stream, int bin_form,
                           bool* done) {
    *done = false;
    const int nb = B.n_eta * B.n_phi;
    if (nb > kChunkMaxBins || nb > 65535 || group_max <= 0) return cudaSuccess;
    int64_t total = 0;
    for (int j = 0; j < m; ++j) {
        if (!B.layer[j].pos || !B.layer[j].hit_rec) return cudaSuccess;
        total += B.layer[j].n;
    }
    if (!chunked_wanted(total, bin_form)) return cudaSuccess;
    const int64_t nc = (group_max + kChunk - 1) / kChunk;
    if (nc > 65535) return cudaSuccess;
    int64_t chunks = 0;
    for (int j = 0; j < m; ++j) chunks += (B.layer[j].n + kChunk - 1) / kChunk;
    if (chunk_cnt_words(chunks, nb) > ((int64_t)1 << 28)) return cudaSuccess;   // > 1 GB of counters: not this form
    cudaError_t e = s.reserve_chunk_cnt(chunk_cnt_words(chunks, nb), stream);
    if (e != cudaSuccess) return e;
    chunks = 0;
    for (int j = 0; j < m; ++j) {
        B.layer[j].chunk_cnt = s.chunk_cnt + chunks * nb;     // [chunks of layer j][nb]
        chunks += (B.layer[j].n + kChunk - 1) / kChunk;
    }
    const dim3 grid((unsigned)nc, (unsigned)m);
    chunk_count_kernel<<<grid, kCountBlock, chunk_count_smem(B.n_eta, B.n_phi), stream>>>(B, s.eta_edge, s.phi_cos, s.phi_sin, s.guess_lut, s.lut_u0, s.lut_uscale);
    chunk_prefix_kernel<<<dim3((unsigned)((nb + 31) / 32), (unsigned)m), 128, 0, stream>>>(B);
    chunk_place_kernel<<<grid, kChunkBlock, (size_t)nb * 4, stream>>>(B);
    bin_finish_kernel<<<dim3((unsigned)((nb * 32 + kBlock - 1) / kBlock), (unsigned)m), kBlock, 0, stream>>>(B);
    *done = true;
    return cudaGetLastError();
}

}  // namespace

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute: set once for every device a context
// launches on (the caller has made that device current).
cudaError_t ensure_bin_attributes() {
    static std::atomic<uint64_t> done{0};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const uint64_t bit = 1ull << (dev & 63);
    if (done.load(std::memory_order_acquire) & bit) return cudaSuccess;
    e = cudaFuncSetAttribute(chunk_count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)chunk_count_smem(1, kChunkMaxBins));
    if (e == cudaSuccess) done.fetch_or(bit, std::memory_order_release);
    return e;
}

// Scratch of the chunked sort for calls of up to max_hits hits in up to KF_MAX_LAYERS pools with any bin grid it
// takes (kf_reserve): chunks <= max_hits / kChunk + pools.
cudaError_t reserve_chunked(BinScratch& s, int64_t max_hits, int max_layers, cudaStream_t stream) {
    const int64_t words = chunk_cnt_words(max_hits / kChunk + max_layers, kChunkMaxBins);
    return s.reserve_chunk_cnt(words < ((int64_t)1 << 28) ? words : ((int64_t)1 << 28), stream);
}

// Bin up to kBinBatchMax layers per group of launches.  All layers share (n_eta, n_phi, eta_max).
cudaError_t launch_bin(BinScratch& s, int n_layers, const BinArgs* args, cudaStream_t stream, const LaunchOptions& opt) {
    if (n_layers <= 0) return cudaSuccess;
    const int n_eta = args[0].n_eta, n_phi = args[0].n_phi;
    const int nb = n_eta * n_phi;
    int64_t total = 0, max_hits = 0;
    for (int l = 0; l < n_layers; ++l) { total += args[l].n_hits; if (args[l].n_hits > max_hits) max_hits = args[l].n_hits; }
    cudaError_t e = s.reserve(total, (int64_t)(nb + 1) * n_layers, stream, true);
    if (e != cudaSuccess) return e;
    if ((e = s.tables(n_eta, n_phi, args[0].eta_max, stream)) != cudaSuccess) return e;
    bool zeroed = false;   // the histogram of the five-launch path (the chunked sort keeps its own in shared memory)
    int64_t item_off = 0;
    for (int l0 = 0; l0 < n_layers; l0 += kBinBatchMax) {
        const int m = n_layers - l0 < kBinBatchMax ? n_layers - l0 : kBinBatchMax;
        BinBatch B;
        B.n_layers = m; B.n_eta = n_eta; B.n_phi = n_phi;
        int64_t group_max = 0;
        for (int j = 0; j < m; ++j) {
            const BinArgs& a = args[l0 + j];
            BinLayerDev& L = B.layer[j];
            L.n = a.n_hits; L.ld_in = a.ld_in; L.ld_out = a.ld_out; L.pos = a.pos; L.cov = a.cov; L.radius = a.radius;
            L.bin_offset = a.bin_offset; L.sorted_to_orig = a.sorted_to_orig;
            L.pos_sorted = a.pos_sorted; L.cov_sorted = a.cov_sorted; L.hit_rec = a.hit_rec; L.bin_box = a.bin_box; L.orig_to_sorted = a.orig_to_sorted;
            L.key = s.key + item_off; L.unsorted = s.unsorted + item_off;
            L.counts = s.counts + (int64_t)(l0 + j) * (nb + 1);
            L.pib = s.pib + item_off; L.rec_tmp = a.pos ? s.rec_tmp + item_off * 12 : nullptr;
            L.chunk_cnt = nullptr;
            item_off += a.n_hits;
            if (a.n_hits > group_max) group_max = a.n_hits;
        }
        bool done = false;
        if ((e = try_chunk_sort(s, B, m, group_max, stream, opt.bin_form, &done)) != cudaSuccess) return e;
        if (done) continue;
        if (!zeroed) {
            if ((e = cudaMemsetAsync(s.counts, 0, (size_t)(nb + 1) * n_layers * sizeof(int32_t), stream)) != cudaSuccess) return e;
            zeroed = true;
        }
        const dim3 grid((unsigned)((group_max + kBlock - 1) / kBlock), (unsigned)m);
        if (group_max > 0) bin_key_kernel<<<grid, kBlock, 0, stream>>>(B, s.eta_edge, s.phi_cos, s.phi_sin);
        bin_scan_kernel<<<dim3(1, m), 1024, 0, stream>>>(B);
        if (group_max > 0) {
            bin_scatter_kernel<<<grid, kBlock, 0, stream>>>(B);
            bin_rank_gather_kernel<<<grid, kBlock, 0, stream>>>(B);
        }
        bin_finish_kernel<<<dim3((unsigned)((nb * 32 + kBlock - 1) / kBlock), (unsigned)m), kBlock, 0, stream>>>(B);
    }
    return cudaGetLastError();
}

// Stable order of candidates by the bin they reach on `layer`.
cudaError_t launch_order(BinScratch& s, const FitParams& P, int layer, int64_t n, int64_t ld, const float* par,
                         const int8_t* q, int n_eta, int n_phi, float eta_max, int32_t* order,
                         cudaStream_t stream) {
    if (n == 0) return cudaSuccess;
    const int nb = n_eta * n_phi;
    cudaError_t e = s.reserve(n, 2 * (int64_t)(nb + 1), stream);
    if (e != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(s.counts, 0, (size_t)(nb + 1) * sizeof(int32_t), stream)) != cudaSuccess) return e;
    BinBatch B;
    B.n_layers = 1; B.n_eta = n_eta; B.n_phi = n_phi;
    BinLayerDev& L = B.layer[0];
    L.n = n; L.ld_in = 0; L.ld_out = 0; L.pos = nullptr; L.cov = nullptr; L.radius = 0.0f;
    L.bin_offset = s.counts + (nb + 1);  // second half of the counts buffer holds the offsets
    L.sorted_to_orig = order; L.pos_sorted = nullptr; L.cov_sorted = nullptr; L.hit_rec = nullptr; L.bin_box = nullptr; L.orig_to_sorted = nullptr;
    L.key = s.key; L.unsorted = s.unsorted; L.counts = s.counts; L.pib = s.pib; L.rec_tmp = nullptr; L.chunk_cnt = nullptr;
    const dim3 grid((unsigned)((n + kBlock - 1) / kBlock), 1);
    cand_key_kernel<<<grid, kBlock, 0, stream>>>(P, layer, n, ld, par, q, n_eta, n_phi, eta_max, s.key, s.pib, s.counts);
    bin_scan_kernel<<<dim3(1, 1), 1024, 0, stream>>>(B);
    bin_scatter_kernel<<<grid, kBlock, 0, stream>>>(B);
    bin_rank_gather_kernel<<<grid, kBlock, 0, stream>>>(B);
    return cudaGetLastError();
}

}  // namespace kf
