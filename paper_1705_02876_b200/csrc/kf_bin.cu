// kf_bin.cu -- (eta, phi) binning of one layer's hits ("directionally projective
// bins"; PAPER.md:135 hits are regrouped on the GPU).
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
// Counting sort, stable: (1) bin of every hit + histogram, (2) exclusive scan -> bin_offset,
// (3) scatter hit indices into their bin segment in arbitrary order (atomic cursor), (4) every
// slot ranks its index inside its segment (indices are unique, so sorting them ascending IS the
// stable order) and gathers the 9 floats of the hit into the bin-sorted SoA copy.
#include <cmath>

#include "kf_internal.h"

namespace kf {

namespace {

constexpr int kBlock = 256;
constexpr double kPi = 3.14159265358979323846;

__device__ __forceinline__ int bin_of_hit(float x, float y, float z, float r, int n_eta, int n_phi,
                                          const float* __restrict__ eta_edge,
                                          const float* __restrict__ phi_cos,
                                          const float* __restrict__ phi_sin) {
    const float u = __fdiv_rn(z, r);
    // edges are non-decreasing in j, so "count of edges <= u" is an upper-bound search
    int lo = 1, hi = n_eta;  // answer - 1 ... first j in [1, n_eta) with !(u >= edge[j]), else n_eta
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (u >= __ldg(eta_edge + mid)) lo = mid + 1; else hi = mid;
    }
    const int ie = lo - 1;
    const int half = n_phi >> 1;
    int ip = 0;
    if (y > 0.0f || (y == 0.0f && x > 0.0f)) {
        ip = half;
        for (int j = half + 1; j < n_phi; ++j)
            ip += (__fmul_rn(__ldg(phi_cos + j), y) >= __fmul_rn(__ldg(phi_sin + j), x)) ? 1 : 0;
    } else if (y == 0.0f) {
        ip = 0;
    } else {
        for (int j = 1; j < half; ++j)
            ip += (__fmul_rn(__ldg(phi_cos + j), y) >= __fmul_rn(__ldg(phi_sin + j), x)) ? 1 : 0;
    }
    return ie * n_phi + ip;
}

__global__ void __launch_bounds__(kBlock)
bin_count_kernel(int64_t n_hits, int64_t ld, const float* __restrict__ pos, float r, int n_eta,
                 int n_phi, const float* __restrict__ eta_edge, const float* __restrict__ phi_cos,
                 const float* __restrict__ phi_sin, int32_t* __restrict__ bin_of,
                 int32_t* __restrict__ counts) {
    const int64_t h = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (h >= n_hits) return;
    const int b = bin_of_hit(__ldg(pos + h), __ldg(pos + ld + h), __ldg(pos + 2 * ld + h), r, n_eta,
                             n_phi, eta_edge, phi_cos, phi_sin);
    bin_of[h] = b;
    atomicAdd(counts + b, 1);
}

// Exclusive scan of counts[0..nb) -> bin_offset[0..nb], cursor = copy.  One block of 1024.
__global__ void __launch_bounds__(1024)
bin_scan_kernel(int nb, const int32_t* __restrict__ counts, int32_t* __restrict__ bin_offset,
                int32_t* __restrict__ cursor) {
    __shared__ int32_t warp_sum[32];
    __shared__ int32_t carry_s;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < nb; base += 1024) {
        const int i = base + tid;
        const int32_t c = i < nb ? counts[i] : 0;
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
        if (i < nb) { bin_offset[i] = excl; cursor[i] = excl; }
        __syncthreads();
        if (tid == 1023) carry_s = excl + c;
        __syncthreads();
    }
    if (tid == 0) bin_offset[nb] = carry_s;
}

__global__ void __launch_bounds__(kBlock)
bin_scatter_kernel(int64_t n_hits, const int32_t* __restrict__ bin_of, int32_t* __restrict__ cursor,
                   int32_t* __restrict__ unsorted) {
    const int64_t h = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (h >= n_hits) return;
    const int32_t slot = atomicAdd(cursor + bin_of[h], 1);
    unsorted[slot] = (int32_t)h;
}

// Slot p holds hit `mine` of bin b; its final place is bin_offset[b] + #{indices in the segment
// smaller than mine}.  Neighbouring threads scan the same segment, so the loads broadcast.
__global__ void __launch_bounds__(kBlock)
bin_rank_gather_kernel(int64_t n_hits, int64_t ld_in, int64_t ld_out,
                       const float* __restrict__ pos, const float* __restrict__ cov,
                       const int32_t* __restrict__ bin_of, const int32_t* __restrict__ bin_offset,
                       const int32_t* __restrict__ unsorted, int32_t* __restrict__ sorted_to_orig,
                       float* __restrict__ pos_sorted, float* __restrict__ cov_sorted) {
    const int64_t p = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (p >= n_hits) return;
    const int32_t mine = unsorted[p];
    const int32_t b = bin_of[mine];
    const int32_t s = bin_offset[b], e = bin_offset[b + 1];
    int32_t rank = 0;
    for (int32_t j = s; j < e; ++j) rank += (__ldg(unsorted + j) < mine) ? 1 : 0;
    const int64_t dst = (int64_t)s + rank;
    sorted_to_orig[dst] = mine;
#pragma unroll
    for (int k = 0; k < 3; ++k) pos_sorted[k * ld_out + dst] = __ldg(pos + k * ld_in + mine);
#pragma unroll
    for (int k = 0; k < 6; ++k) cov_sorted[k * ld_out + dst] = __ldg(cov + k * ld_in + mine);
}

}  // namespace

cudaError_t BinScratch::reserve(int64_t n_hits, int n_bins, cudaStream_t stream) {
    if (n_hits <= cap_hits && n_bins <= cap_bins) return cudaSuccess;
    // growing: drain the stream that may still use the old buffers, then reallocate
    cudaError_t e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return e;
    const int64_t nh = n_hits > cap_hits ? n_hits : cap_hits;
    const int nb = n_bins > cap_bins ? n_bins : cap_bins;
    release();
    const size_t hits_b = (size_t)(nh > 0 ? nh : 1) * sizeof(int32_t);
    const size_t bins_b = (size_t)(nb + 1) * sizeof(int32_t);
    if ((e = cudaMalloc(&bin_of, hits_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&unsorted, hits_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&counts, bins_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&cursor, bins_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&eta_edge, bins_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&phi_cos, bins_b)) != cudaSuccess) { release(); return e; }
    if ((e = cudaMalloc(&phi_sin, bins_b)) != cudaSuccess) { release(); return e; }
    cap_hits = nh;
    cap_bins = nb;
    return cudaSuccess;
}

void BinScratch::release() {
    void* ptrs[] = {bin_of, unsorted, counts, cursor, eta_edge, phi_cos, phi_sin};
    for (void* p : ptrs)
        if (p) cudaFree(p);
    bin_of = unsorted = counts = cursor = nullptr;
    eta_edge = phi_cos = phi_sin = nullptr;
    cap_hits = 0;
    cap_bins = 0;
    tab_n_eta = tab_n_phi = 0;
    tab_eta_max = 0.0f;
}

// Edge tables, evaluated in double on the host and rounded once to float (reading A16b).
cudaError_t BinScratch::tables(int n_eta, int n_phi, float eta_max, cudaStream_t stream) {
    if (n_eta == tab_n_eta && n_phi == tab_n_phi && eta_max == tab_eta_max) return cudaSuccess;
    // the previous tables may still be in use by queued kernels, and host_tab by a queued copy
    cudaError_t e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return e;
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
    tab_n_eta = n_eta;
    tab_n_phi = n_phi;
    tab_eta_max = eta_max;
    return cudaSuccess;
}

cudaError_t launch_bin(BinScratch& s, const BinArgs& a, cudaStream_t stream) {
    const int nb = a.n_eta * a.n_phi;
    cudaError_t e = s.tables(a.n_eta, a.n_phi, a.eta_max, stream);
    if (e != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(s.counts, 0, (size_t)(nb + 1) * sizeof(int32_t), stream)) != cudaSuccess) return e;
    const unsigned blocks = (unsigned)((a.n_hits + kBlock - 1) / kBlock);
    if (a.n_hits > 0) {
        bin_count_kernel<<<blocks, kBlock, 0, stream>>>(a.n_hits, a.ld_in, a.pos, a.radius, a.n_eta, a.n_phi,
                                                        s.eta_edge, s.phi_cos, s.phi_sin, s.bin_of, s.counts);
    }
    bin_scan_kernel<<<1, 1024, 0, stream>>>(nb, s.counts, a.bin_offset, s.cursor);
    if (a.n_hits > 0) {
        bin_scatter_kernel<<<blocks, kBlock, 0, stream>>>(a.n_hits, s.bin_of, s.cursor, s.unsorted);
        bin_rank_gather_kernel<<<blocks, kBlock, 0, stream>>>(a.n_hits, a.ld_in, a.ld_out, a.pos, a.cov, s.bin_of,
                                                              a.bin_offset, s.unsorted, a.sorted_to_orig,
                                                              a.pos_sorted, a.cov_sorted);
    }
    return cudaGetLastError();
}

}  // namespace kf
