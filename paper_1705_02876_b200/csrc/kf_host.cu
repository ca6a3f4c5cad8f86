// kf_host.cu -- kf_fit_tracks_host: host buffers in, host buffers out.
//
// The tracks are cut into chunks; each chunk goes H2D (one strided 2-D copy per SoA array),
// through the same fit kernel as the device path, and D2H, on one of kSlots internal streams, so
// copies in both directions overlap the kernel of neighbouring chunks ("overlapped
// with kernels via streams"; PAPER.md:164 transfers are half of the wall time when they are not).
// With pinned host memory the copies are truly asynchronous; with pageable memory the runtime
// stages them and the pipeline degrades gracefully.
#include <cmath>
#include <cstring>

#include <cstdint>

#include "kf_internal.h"

namespace kf {

namespace {

// Tracks per chunk.  A call costs  (copies in) + k x (starting the eleven copies of a chunk: 52 us, measured as the
// slope of the call time against the number of chunks) + (kernel + copies out of the LAST chunk ~ 4.3 ms / k at 2 M
// tracks), so the best number of chunks is k = sqrt(n x 4.1e-5): nine chunks of 223 232 tracks for 2 M tracks (16.6
// ms; sixteen of 131 072: 16.9; thirty-one of 65 536: 17.7).  Chunks are multiples of 1024 tracks, so the pairs of
// the two-tracks-per-thread kernel are the same as in one launch over the whole batch.  -DKF_HOST_CHUNK=n fixes it.
inline int64_t host_chunk_for(int64_t n) {
    int64_t c;
#ifdef KF_HOST_CHUNK
    c = KF_HOST_CHUNK;
#else
    const double k = std::sqrt((double)n * 4.1e-5);
    const int64_t kk = k < 1.0 ? 1 : (int64_t)(k + 0.5);
    c = ((n + kk - 1) / kk + 1023) / 1024 * 1024;
    if (c < 32768) c = 32768;
    if (c > 524288) c = 524288;
#endif
    if (n <= c) c = n < 4 ? 4 : (n + 3) / 4 * 4;
    return c;
}

inline size_t align256(size_t b) { return (b + 255) & ~size_t(255); }

// Offsets of the SoA arrays of one chunk inside a slot buffer.
struct SlotLayout {
    size_t par, cov, q, mask, hpos, hcov, opar, ocov, chi2, nhits, status, diag, hvar, total;
    SlotLayout(int64_t chunk, int L) {
        size_t o = 0;
        auto take = [&](size_t bytes) { size_t at = o; o += align256(bytes); return at; };
        par = take(6 * chunk * 4);   cov = take(21 * chunk * 4);
        q = take(chunk);             mask = take(chunk * 4);
        hpos = take((size_t)L * 3 * chunk * 4); hcov = take((size_t)L * 6 * chunk * 4);
        opar = take(6 * chunk * 4);  ocov = take(21 * chunk * 4);
        chi2 = take(chunk * 4);      nhits = take(chunk * 4);  status = take(chunk * 4);
        diag = take(6 * chunk * 4);  // kf_fit_tracks_host_diag: the six variance planes as they arrive
        hvar = take((size_t)L * 3 * chunk * 4);  // kf_fit_tracks_host_compact: v_r v_t v_z of every hit as they arrive
        total = o;
    }
};

// kf_fit_tracks_host_compact: the hit covariance from its three variances in the hit's own cylindrical frame,
// V = R_z(phi_h) diag(v_r, v_t, v_z) R_z(phi_h)^T with (cos, sin) phi_h = (x, y) / rho of the hit position
// (include/kf_b200.h states the five lines below; four tracks per thread, planes are 16-byte aligned).
__global__ void __launch_bounds__(256) expand_hit_cov_kernel(const float* __restrict__ hpos, const float* __restrict__ hvar,
                                                             float* __restrict__ hcov, int64_t m, int64_t ld) {
    const int64_t t = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (t >= m) return;
    const int l = blockIdx.y;
    const float* p = hpos + (size_t)l * 3 * ld + t;
    const float* v = hvar + (size_t)l * 3 * ld + t;
    float* c = hcov + (size_t)l * 6 * ld + t;
    const float4 x4 = *reinterpret_cast<const float4*>(p), y4 = *reinterpret_cast<const float4*>(p + ld);
    const float4 r4 = *reinterpret_cast<const float4*>(v), t4 = *reinterpret_cast<const float4*>(v + ld);
    const float4 z4 = *reinterpret_cast<const float4*>(v + 2 * ld);
    const float x[4] = {x4.x, x4.y, x4.z, x4.w}, y[4] = {y4.x, y4.y, y4.z, y4.w};
    const float vr[4] = {r4.x, r4.y, r4.z, r4.w}, vt[4] = {t4.x, t4.y, t4.z, t4.w};
    float xx[4], xy[4], yy[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float rho2 = __fadd_rn(__fmul_rn(x[k], x[k]), __fmul_rn(y[k], y[k]));
        float c2 = 1.0f, s2 = 0.0f, cs = 0.0f;
        if (rho2 > 0.0f) {
            c2 = __fdiv_rn(__fmul_rn(x[k], x[k]), rho2);
            s2 = __fdiv_rn(__fmul_rn(y[k], y[k]), rho2);
            cs = __fdiv_rn(__fmul_rn(x[k], y[k]), rho2);
        }
        xx[k] = __fadd_rn(__fmul_rn(vr[k], c2), __fmul_rn(vt[k], s2));
        xy[k] = __fmul_rn(__fsub_rn(vr[k], vt[k]), cs);
        yy[k] = __fadd_rn(__fmul_rn(vr[k], s2), __fmul_rn(vt[k], c2));
    }
    const float4 zero = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    *reinterpret_cast<float4*>(c) = make_float4(xx[0], xx[1], xx[2], xx[3]);
    *reinterpret_cast<float4*>(c + ld) = make_float4(xy[0], xy[1], xy[2], xy[3]);
    *reinterpret_cast<float4*>(c + 2 * ld) = zero;
    *reinterpret_cast<float4*>(c + 3 * ld) = make_float4(yy[0], yy[1], yy[2], yy[3]);
    *reinterpret_cast<float4*>(c + 4 * ld) = zero;
    *reinterpret_cast<float4*>(c + 5 * ld) = z4;
}

// kf_fit_tracks_host_diag: the six variance planes as they arrived -> the 21-plane packed covariance (rows xx yy zz
// pxpx pypy pzpz of the upper triangle are 0, 6, 11, 15, 18, 20; the other 15 are zero).  Four tracks per thread.
__global__ void __launch_bounds__(256) spread_diag_kernel(const float* __restrict__ diag, float* __restrict__ cov,
                                                          int64_t m, int64_t ld) {
    const int64_t t = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (t >= m) return;
    int k = 0;
#pragma unroll
    for (int r = 0; r < 21; ++r) {
        float4 v = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (r == 0 || r == 6 || r == 11 || r == 15 || r == 18 || r == 20) {
            v = *reinterpret_cast<const float4*>(diag + (size_t)k * ld + t);
            ++k;
        }
        *reinterpret_cast<float4*>(cov + (size_t)r * ld + t) = v;
    }
}

}  // namespace

cudaError_t HostStage::reserve(int64_t max_tracks, int max_layers) {
    int64_t want = host_chunk_for(max_tracks);
    if (want <= chunk && max_layers <= layers) return cudaSuccess;
    if (want < chunk) want = chunk;
    if (max_layers < layers) max_layers = layers;
    release();
    SlotLayout lay(want, max_layers);
    cudaError_t e0 = cudaStreamCreateWithFlags(&out_stream, cudaStreamNonBlocking);
    if (e0 != cudaSuccess) { release(); return e0; }
    for (int s = 0; s < kSlots; ++s) {
        cudaError_t e = cudaStreamCreateWithFlags(&stream[s], cudaStreamNonBlocking);
        if (e != cudaSuccess) { release(); return e; }
        if ((e = cudaEventCreateWithFlags(&fitted[s], cudaEventDisableTiming)) != cudaSuccess) { release(); return e; }
        if ((e = cudaEventCreateWithFlags(&drained[s], cudaEventDisableTiming)) != cudaSuccess) { release(); return e; }
        e = cudaMalloc(&buf[s], lay.total);
        if (e != cudaSuccess) { release(); return e; }
    }
    buf_bytes = lay.total;
    chunk = want;
    layers = max_layers;
    return cudaSuccess;
}

void HostStage::release() {
    for (int s = 0; s < kSlots; ++s) {
        if (buf[s]) cudaFree(buf[s]);
        if (stream[s]) cudaStreamDestroy(stream[s]);
        if (fitted[s]) cudaEventDestroy(fitted[s]);
        if (drained[s]) cudaEventDestroy(drained[s]);
        buf[s] = nullptr;
        stream[s] = nullptr;
        fitted[s] = drained[s] = nullptr;
    }
    if (out_stream) cudaStreamDestroy(out_stream);
    out_stream = nullptr;
    chunk = 0;
    layers = 0;
    buf_bytes = 0;
}

cudaError_t HostStage::fit(const FitParams& P, const HostFitIO& io, const LaunchOptions& opt) {
    cudaError_t e = reserve(io.n, io.L);
    if (e != cudaSuccess) return e;
    const SlotLayout lay(chunk, layers);     // `chunk` = tracks a slot buffer holds = the pitch of its planes
    const int L = io.L;
    const size_t cw = (size_t)chunk * 4;  // device pitch of float planes
    const int64_t step = host_chunk_for(io.n) < chunk ? host_chunk_for(io.n) : chunk;   // tracks per chunk of THIS call
    // every chunk takes the kernel the WHOLE batch would take in kf_fit_tracks (chunks start at multiples of 64, so
    // the pairs are the same too): host path and device path agree bit for bit
    LaunchOptions chunk_opt = opt;
    chunk_opt.pair_min_tracks = fit_takes_pair_form(io.n, L, opt) ? 1 : INT64_MAX;
    int slot = 0;
    // The last chunk's kernel and copies out overlap nothing: the tail of the batch goes as a half and two quarters
    // of a chunk (2 M tracks: 0.46 ms of drain become 0.11 at the price of two more chunks).
    int64_t m = 0;
    int n_chunks = 0;
    for (int64_t t0 = 0; t0 < io.n; t0 += m, slot = (slot + 1) % kSlots, ++n_chunks) {
        const int64_t left = io.n - t0;
        m = left < step ? left : step;
        if (left <= step + step / 2 && left >= 4 * 16384) {
            const int64_t piece = (left > step ? left / 3 : left / 2 + 1023) / 1024 * 1024;   // (multiples of 1024: see above)
            m = piece < left ? piece : left;
        }
        cudaStream_t st = stream[slot];
        char* b = buf[slot];
        const size_t w = (size_t)m * 4;
#define KF_TRY(x) do { e = (x); if (e != cudaSuccess) goto fail; } while (0)
        // Order of submission (measured on 2 M tracks, each variant against this one on the same box): the spreading of
        // the diagonal right after the planes it reads, the hits last.  Queued after the chunk's last copy the
        // spreading costs 0.5 ms per call (17.5 against 17.0 ms), whether it is a kernel or a memset and six
        // device-to-device copies; hits first and seeds last costs the compact call 1.1 ms (13.8 against 12.7 ms).
        KF_TRY(cudaMemcpy2DAsync(b + lay.par, cw, io.par + t0, (size_t)io.ld_in * 4, w, 6, cudaMemcpyHostToDevice, st));
        if (io.cov_diagonal) {
            // 6 of the 21 planes travel, as ONE copy (six separate host-to-device copies of 0.5 MB each cost the link
            // more than the bytes they saved); spread_diag_kernel puts them in place
            KF_TRY(cudaMemcpy2DAsync(b + lay.diag, cw, io.cov + t0, (size_t)io.ld_in * 4, w, 6, cudaMemcpyHostToDevice, st));
            spread_diag_kernel<<<(unsigned)((m + 1023) / 1024), 256, 0, st>>>((const float*)(b + lay.diag), (float*)(b + lay.cov), m, chunk);
            KF_TRY(cudaGetLastError());
        } else {
            KF_TRY(cudaMemcpy2DAsync(b + lay.cov, cw, io.cov + t0, (size_t)io.ld_in * 4, w, 21, cudaMemcpyHostToDevice, st));
        }
        KF_TRY(cudaMemcpyAsync(b + lay.q, io.q + t0, (size_t)m, cudaMemcpyHostToDevice, st));
        if (io.mask) KF_TRY(cudaMemcpyAsync(b + lay.mask, io.mask + t0, w, cudaMemcpyHostToDevice, st));
        KF_TRY(cudaMemcpy2DAsync(b + lay.hpos, cw, io.hpos + t0, (size_t)io.ld_hit * 4, w, (size_t)L * 3, cudaMemcpyHostToDevice, st));
        if (io.hit_cov_local) {
            // 3 of the 6 planes per layer travel; the covariance is rebuilt beside the hit positions
            KF_TRY(cudaMemcpy2DAsync(b + lay.hvar, cw, io.hcov + t0, (size_t)io.ld_hit * 4, w, (size_t)L * 3, cudaMemcpyHostToDevice, st));
            const dim3 grid((unsigned)((m + 1023) / 1024), (unsigned)L);
            expand_hit_cov_kernel<<<grid, 256, 0, st>>>((const float*)(b + lay.hpos), (const float*)(b + lay.hvar),
                                                        (float*)(b + lay.hcov), m, chunk);
            KF_TRY(cudaGetLastError());
        } else {
            KF_TRY(cudaMemcpy2DAsync(b + lay.hcov, cw, io.hcov + t0, (size_t)io.ld_hit * 4, w, (size_t)L * 6, cudaMemcpyHostToDevice, st));
        }
        {
            FitArgs a;
            a.n = m;
            a.par = (const float*)(b + lay.par); a.cov = (const float*)(b + lay.cov); a.ld_in = chunk;
            a.q = (const int8_t*)(b + lay.q);
            a.hpos = (const float*)(b + lay.hpos); a.hcov = (const float*)(b + lay.hcov); a.ld_hit = chunk;
            a.mask = io.mask ? (const uint32_t*)(b + lay.mask) : nullptr;
            a.opar = (float*)(b + lay.opar); a.ocov = (float*)(b + lay.ocov); a.ld_out = chunk;
            a.chi2 = (float*)(b + lay.chi2); a.nhits = (int32_t*)(b + lay.nhits); a.status = (uint32_t*)(b + lay.status);
            // the results of the chunk that used this slot before must have left (the inputs above may land earlier:
            // they do not touch the output planes)
            if (n_chunks >= kSlots) KF_TRY(cudaStreamWaitEvent(st, drained[slot], 0));
            KF_TRY(launch_fit(P, a, st, chunk_opt));
            KF_TRY(cudaEventRecord(fitted[slot], st));
        }
        // results out on a stream of their own: the slot's stream carries host-to-device copies and kernels only
        KF_TRY(cudaStreamWaitEvent(out_stream, fitted[slot], 0));
        KF_TRY(cudaMemcpy2DAsync(io.opar + t0, (size_t)io.ld_out * 4, b + lay.opar, cw, w, 6, cudaMemcpyDeviceToHost, out_stream));
        KF_TRY(cudaMemcpy2DAsync(io.ocov + t0, (size_t)io.ld_out * 4, b + lay.ocov, cw, w, 21, cudaMemcpyDeviceToHost, out_stream));
        KF_TRY(cudaMemcpyAsync(io.chi2 + t0, b + lay.chi2, w, cudaMemcpyDeviceToHost, out_stream));
        KF_TRY(cudaMemcpyAsync(io.nhits + t0, b + lay.nhits, w, cudaMemcpyDeviceToHost, out_stream));
        KF_TRY(cudaMemcpyAsync(io.status + t0, b + lay.status, w, cudaMemcpyDeviceToHost, out_stream));
        KF_TRY(cudaEventRecord(drained[slot], out_stream));
#undef KF_TRY
    }
    for (int s = 0; s < kSlots; ++s) {
        cudaError_t es = cudaStreamSynchronize(stream[s]);
        if (es != cudaSuccess && e == cudaSuccess) e = es;
    }
    {
        cudaError_t es = cudaStreamSynchronize(out_stream);
        if (es != cudaSuccess && e == cudaSuccess) e = es;
    }
    return e;
fail:
    for (int s = 0; s < kSlots; ++s) cudaStreamSynchronize(stream[s]);
    cudaStreamSynchronize(out_stream);
    return e;
}

// ---------------------------------------------------------------------------------------------------------------
// kf_build_best_hit_host
cudaError_t BuildHostStage::reserve(size_t bytes) {
    cudaError_t e;
    if (!copy_stream) {
        if ((e = cudaStreamCreateWithFlags(&copy_stream, cudaStreamNonBlocking)) != cudaSuccess) return e;
        for (int j = 0; j < 32; ++j)
            if ((e = cudaEventCreateWithFlags(&ready[j], cudaEventDisableTiming)) != cudaSuccess) return e;
        if ((e = cudaEventCreateWithFlags(&done, cudaEventDisableTiming)) != cudaSuccess) return e;
    }
    if (bytes <= cap) return cudaSuccess;
    if (buf) cudaFree(buf);
    buf = nullptr;
    cap = 0;
    if ((e = cudaMalloc(&buf, bytes)) != cudaSuccess) return e;
    cap = bytes;
    return cudaSuccess;
}

void BuildHostStage::release() {
    if (buf) cudaFree(buf);
    buf = nullptr;
    cap = 0;
    if (copy_stream) {
        cudaStreamDestroy(copy_stream);
        for (int j = 0; j < 32; ++j)
            if (ready[j]) cudaEventDestroy(ready[j]);
        if (done) cudaEventDestroy(done);
        copy_stream = nullptr;
        done = nullptr;
        for (int j = 0; j < 32; ++j) ready[j] = nullptr;
    }
}

cudaError_t build_best_hit_host(BuildHostStage& hs, BinScratch& bs, ScoreScratch& ss, const FitParams& P, const BuildHostIO& io,
                                cudaStream_t stream, const LaunchOptions& opt) {
    const int L = io.n_layers;
    const int nb = io.n_eta * io.n_phi;
    const int64_t ldc = (io.n + 3) / 4 * 4;
    // device layout: candidates, local state, outputs, then per layer: pool (9 planes), bins
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += align256(bytes); return at; };
    const size_t o_par = take((size_t)6 * ldc * 4), o_cov = take((size_t)21 * ldc * 4), o_q = take((size_t)ldc);
    const size_t o_chi2 = take((size_t)ldc * 4), o_nh = take((size_t)ldc * 4), o_st = take((size_t)ldc * 4);
    const size_t o_ls = take((size_t)30 * ldc * 4);
    const size_t o_idx = take((size_t)L * ldc * 4), o_c2 = take((size_t)L * ldc * 4);
    size_t o_pos[32], o_hcov[32], o_off[32], o_s2o[32], o_rec[32], o_box[32];
    int64_t ldh[32];
    for (int j = 0; j < L; ++j) {
        ldh[j] = (io.n_hits[j] + 3) / 4 * 4;
        if (ldh[j] < 4) ldh[j] = 4;
        o_pos[j] = take((size_t)3 * ldh[j] * 4); o_hcov[j] = take((size_t)6 * ldh[j] * 4);
        o_off[j] = take((size_t)(nb + 1) * 4); o_s2o[j] = take((size_t)ldh[j] * 4);
        o_rec[j] = take((size_t)ldh[j] * kRecFloats * 4); o_box[j] = take((size_t)nb * 32);
    }
    cudaError_t e = cudaStreamSynchronize(stream);       // the staging buffers may still serve the previous call
    if (e != cudaSuccess) return e;
    if ((e = hs.reserve(o)) != cudaSuccess) return e;
    char* b = hs.buf;
#define KF_TRY(x) do { e = (x); if (e != cudaSuccess) goto fail; } while (0)
    // Candidates first, on the compute stream: host-to-device copies are served in the order they were submitted,
    // whatever their stream, so candidate copies queued behind the pools would hold the first layer's kernels back
    // until every pool had arrived (measured: call time = copies + kernels, no overlap at all).
    {
        const size_t w = (size_t)io.n * 4, cw = (size_t)ldc * 4;
        KF_TRY(cudaMemcpy2DAsync(b + o_par, cw, io.par, (size_t)io.ld * 4, w, 6, cudaMemcpyHostToDevice, stream));
        KF_TRY(cudaMemcpy2DAsync(b + o_cov, cw, io.cov, (size_t)io.ld * 4, w, 21, cudaMemcpyHostToDevice, stream));
        KF_TRY(cudaMemcpyAsync(b + o_q, io.q, (size_t)io.n, cudaMemcpyHostToDevice, stream));
        KF_TRY(cudaMemcpyAsync(b + o_chi2, io.chi2, w, cudaMemcpyHostToDevice, stream));
        KF_TRY(cudaMemcpyAsync(b + o_nh, io.nhits, w, cudaMemcpyHostToDevice, stream));
        KF_TRY(cudaMemcpyAsync(b + o_st, io.status, w, cudaMemcpyHostToDevice, stream));
        KF_TRY(cudaMemsetAsync(b + o_ls + (size_t)29 * ldc * 4, 0, (size_t)ldc * 4, stream));   // local-state flags
    }
    // pools: copy stream, one event per layer
    for (int j = 0; j < L; ++j) {
        const size_t w = (size_t)io.n_hits[j] * 4;
        if (io.n_hits[j] > 0) {
            KF_TRY(cudaMemcpy2DAsync(b + o_pos[j], (size_t)ldh[j] * 4, io.pos[j], (size_t)io.ld_hits[j] * 4, w, 3, cudaMemcpyHostToDevice, hs.copy_stream));
            KF_TRY(cudaMemcpy2DAsync(b + o_hcov[j], (size_t)ldh[j] * 4, io.cov_hits[j], (size_t)io.ld_hits[j] * 4, w, 6, cudaMemcpyHostToDevice, hs.copy_stream));
        }
        KF_TRY(cudaEventRecord(hs.ready[j], hs.copy_stream));
    }
    {
        // layer by layer: wait for the pool, bin it, score it
        const size_t w = (size_t)io.n * 4, cw = (size_t)ldc * 4;
        for (int j = 0; j < L; ++j) {
            KF_TRY(cudaStreamWaitEvent(stream, hs.ready[j], 0));
            BinArgs ba;
            ba.n_hits = io.n_hits[j]; ba.ld_in = ldh[j];
            ba.pos = (const float*)(b + o_pos[j]); ba.cov = (const float*)(b + o_hcov[j]);
            ba.radius = P.layer[io.first_layer + j].type == 1 ? 0.0f : P.layer[io.first_layer + j].r;   // (reading A24)
            ba.n_eta = io.n_eta; ba.n_phi = io.n_phi; ba.eta_max = io.eta_max;
            ba.ld_out = ldh[j]; ba.bin_offset = (int32_t*)(b + o_off[j]); ba.sorted_to_orig = (int32_t*)(b + o_s2o[j]);
            ba.pos_sorted = nullptr; ba.cov_sorted = nullptr; ba.hit_rec = (float*)(b + o_rec[j]);
            ba.bin_box = (float*)(b + o_box[j]); ba.orig_to_sorted = nullptr;
            KF_TRY(launch_bin(bs, 1, &ba, stream, opt));
            ScoreStep st;
            st.layer = io.first_layer + j; st.n_hits = io.n_hits[j];
            st.hit_rec = ba.hit_rec; st.bin_box = ba.bin_box; st.bin_offset = ba.bin_offset;
            st.best_hit = (int32_t*)(b + o_idx) + (int64_t)j * ldc;
            st.best_chi2 = (float*)(b + o_c2) + (int64_t)j * ldc;
            ScoreArgs a;
            memset(&a, 0, sizeof(a));
            a.n = io.n; a.ld = ldc; a.par = (float*)(b + o_par); a.cov = (float*)(b + o_cov); a.q = (const int8_t*)(b + o_q);
            a.chi2 = (float*)(b + o_chi2); a.nhits = (int32_t*)(b + o_nh); a.status = (uint32_t*)(b + o_st);
            a.n_eta = io.n_eta; a.n_phi = io.n_phi; a.eta_max = io.eta_max;
            a.window_half = io.window_half; a.chi2_cut = io.chi2_cut; a.do_update = io.do_update;
            a.lstate = (float*)(b + o_ls); a.ld_ls = ldc;
            KF_TRY(launch_build(ss, P, a, 1, &st, stream));
        }
        KF_TRY(cudaMemcpy2DAsync(io.par, (size_t)io.ld * 4, b + o_par, cw, w, 6, cudaMemcpyDeviceToHost, stream));
        KF_TRY(cudaMemcpy2DAsync(io.cov, (size_t)io.ld * 4, b + o_cov, cw, w, 21, cudaMemcpyDeviceToHost, stream));
        KF_TRY(cudaMemcpyAsync(io.chi2, b + o_chi2, w, cudaMemcpyDeviceToHost, stream));
        KF_TRY(cudaMemcpyAsync(io.nhits, b + o_nh, w, cudaMemcpyDeviceToHost, stream));
        KF_TRY(cudaMemcpyAsync(io.status, b + o_st, w, cudaMemcpyDeviceToHost, stream));
        KF_TRY(cudaMemcpy2DAsync(io.hit_index, (size_t)io.ld_out * 4, b + o_idx, cw, w, (size_t)L, cudaMemcpyDeviceToHost, stream));
        KF_TRY(cudaMemcpy2DAsync(io.hit_chi2, (size_t)io.ld_out * 4, b + o_c2, cw, w, (size_t)L, cudaMemcpyDeviceToHost, stream));
    }
#undef KF_TRY
    e = cudaStreamSynchronize(stream);
    {
        cudaError_t e2 = cudaStreamSynchronize(hs.copy_stream);
        if (e == cudaSuccess) e = e2;
    }
    return e;
fail:
    cudaStreamSynchronize(stream);
    cudaStreamSynchronize(hs.copy_stream);
    return e;
}

}  // namespace kf
