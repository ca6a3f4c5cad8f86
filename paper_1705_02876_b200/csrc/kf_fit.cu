// kf_fit.cu -- fused per-layer propagate + update track-fit kernel for sm_100a.
//
// One thread owns one track for the whole layer loop ("one thread per track";
// PAPER.md:129 merged kernels, registers over shared memory): the state, the 21 (then 15) unique
// covariance elements and the Jacobian ingredients never leave registers.  Inputs and outputs
// are element-major SoA (PAPER.md:65, 119 Matriplex), so a warp's access to one element of 32
// consecutive tracks is one 128-byte line.  Per-layer hits (9 floats per track and layer, the
// only per-layer HBM traffic) are prefetched one layer ahead into registers.
//
// Algorithmic HBM bytes per track: 113 in (6 + 21 floats, charge, mask) + 120 out (27 floats,
// chi2, nhits, status) + 36 per layer = 593 B at 10 layers.
#include "kf_internal.h"

namespace kf {

namespace {

constexpr int kFitBlock = 128;

struct Hit {
    float x, y, z, vxx, vxy, vxz, vyy, vyz, vzz;
};

__device__ __forceinline__ Hit load_hit(const float* __restrict__ hpos,
                                        const float* __restrict__ hcov, int64_t ld, int l,
                                        int64_t i) {
    const float* p = hpos + (int64_t)l * 3 * ld + i;
    const float* c = hcov + (int64_t)l * 6 * ld + i;
    Hit h;
    h.x = __ldg(p);           h.y = __ldg(p + ld);      h.z = __ldg(p + 2 * ld);
    h.vxx = __ldg(c);         h.vxy = __ldg(c + ld);    h.vxz = __ldg(c + 2 * ld);
    h.vyy = __ldg(c + 3 * ld); h.vyz = __ldg(c + 4 * ld); h.vzz = __ldg(c + 5 * ld);
    return h;
}

// One layer for one track.  Returns 0 or the status bit of the failure (track untouched).
template <bool RADIAL_NULL>
__device__ __forceinline__ uint32_t fit_layer(Track& t, float k, float ik, const LayerConst& L,
                                              float mass2, const Hit& m, float& chi2) {
    Crossing o;
    if (!helix_to_radius(t, k, ik, L, o)) return ST_PROP_FAIL;
    PropCov n;
    transport_cov<RADIAL_NULL>(t, o, L.ms, mass2, n);
    LocalHit h;
    hit_to_local(o, m.x, m.y, m.z, m.vxx, m.vxy, m.vxz, m.vyy, m.vyz, m.vzz, h);
    float d;
    const uint32_t rc = kalman_update(t, o, n, h, &d);
    if (rc == 0u) chi2 += d;
    return rc;
}

__global__ void __launch_bounds__(kFitBlock, 4)
fit_kernel(const __grid_constant__ FitParams P, const FitArgs a) {
    const int64_t i = (int64_t)blockIdx.x * kFitBlock + threadIdx.x;
    if (i >= a.n) return;
    const int q = a.q[i];
    const uint32_t mask = a.mask ? __ldg(a.mask + i) : 0xffffffffu;
    Track t;
    load_track(t, a.par, a.cov, a.ld_in, i);
    float chi2 = 0.0f;
    int nh = 0;
    uint32_t st = 0u;
    if (q != 1 && q != -1) {
        st = ST_BAD_CHARGE;  // copied through untouched
    } else {
        const int L = P.n_layers;
        const float k = (float)q * P.k0, ik = (float)q * P.inv_k0;
        enter_local_frame(t);
        Hit next = load_hit(a.hpos, a.hcov, a.ld_hit, 0, i);
        int l = 0;
        // until the first successful layer the covariance is a general 6x6 ...
        bool started = false;
        for (; l < L && !started; ++l) {
            const Hit cur = next;
            if (l + 1 < L) next = load_hit(a.hpos, a.hcov, a.ld_hit, l + 1, i);
            if (!((mask >> l) & 1u)) continue;
            const uint32_t rc = fit_layer<false>(t, k, ik, P.layer[l], P.mass2, cur, chi2);
            st |= rc;
            if (rc == 0u) { nh += 1; started = true; }
        }
        // ... afterwards its radial row is identically zero
        for (; l < L; ++l) {
            const Hit cur = next;
            if (l + 1 < L) next = load_hit(a.hpos, a.hcov, a.ld_hit, l + 1, i);
            if (!((mask >> l) & 1u)) continue;
            const uint32_t rc = fit_layer<true>(t, k, ik, P.layer[l], P.mass2, cur, chi2);
            st |= rc;
            nh += (rc == 0u);
        }
        if (nh > 0) leave_local_frame(t);
        else load_track(t, a.par, a.cov, a.ld_in, i);  // nothing fitted: hand the seed back bit-exact
    }
    store_track(t, a.opar, a.ocov, a.ld_out, i);
    a.chi2[i] = chi2;
    a.nhits[i] = nh;
    a.status[i] = st;
}

}  // namespace

cudaError_t launch_fit(const FitParams& P, const FitArgs& a, cudaStream_t stream) {
    if (a.n == 0) return cudaSuccess;
    const int64_t blocks = (a.n + kFitBlock - 1) / kFitBlock;
    fit_kernel<<<(unsigned)blocks, kFitBlock, 0, stream>>>(P, a);
    return cudaGetLastError();
}

int fit_kernel_count() { return 1; }

}  // namespace kf
