// kf_host.cu -- kf_fit_tracks_host: host buffers in, host buffers out.
//
// The tracks are cut into chunks; each chunk goes H2D (one strided 2-D copy per SoA array),
// through the same fit kernel as the device path, and D2H, on one of kSlots internal streams, so
// copies in both directions overlap the kernel of neighbouring chunks ("overlapped
// with kernels via streams"; PAPER.md:164 transfers are half of the wall time when they are not).
// With pinned host memory the copies are truly asynchronous; with pageable memory the runtime
// stages them and the pipeline degrades gracefully.
#include "kf_internal.h"

namespace kf {

namespace {

constexpr int64_t kDefaultChunk = 1 << 17;  // 131072 tracks per chunk

inline size_t align256(size_t b) { return (b + 255) & ~size_t(255); }

// Offsets of the SoA arrays of one chunk inside a slot buffer.
struct SlotLayout {
    size_t par, cov, q, mask, hpos, hcov, opar, ocov, chi2, nhits, status, total;
    SlotLayout(int64_t chunk, int L) {
        size_t o = 0;
        auto take = [&](size_t bytes) { size_t at = o; o += align256(bytes); return at; };
        par = take(6 * chunk * 4);   cov = take(21 * chunk * 4);
        q = take(chunk);             mask = take(chunk * 4);
        hpos = take((size_t)L * 3 * chunk * 4); hcov = take((size_t)L * 6 * chunk * 4);
        opar = take(6 * chunk * 4);  ocov = take(21 * chunk * 4);
        chi2 = take(chunk * 4);      nhits = take(chunk * 4);  status = take(chunk * 4);
        total = o;
    }
};

}  // namespace

cudaError_t HostStage::reserve(int64_t max_tracks, int max_layers) {
    int64_t want = max_tracks < kDefaultChunk ? ((max_tracks + 3) / 4) * 4 : kDefaultChunk;
    if (want < 4) want = 4;
    if (want <= chunk && max_layers <= layers) return cudaSuccess;
    if (want < chunk) want = chunk;
    if (max_layers < layers) max_layers = layers;
    release();
    SlotLayout lay(want, max_layers);
    for (int s = 0; s < kSlots; ++s) {
        cudaError_t e = cudaStreamCreateWithFlags(&stream[s], cudaStreamNonBlocking);
        if (e != cudaSuccess) { release(); return e; }
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
        buf[s] = nullptr;
        stream[s] = nullptr;
    }
    chunk = 0;
    layers = 0;
    buf_bytes = 0;
}

cudaError_t HostStage::fit(const FitParams& P, const HostFitIO& io, const LaunchOptions& opt) {
    cudaError_t e = reserve(io.n, io.L);
    if (e != cudaSuccess) return e;
    const SlotLayout lay(chunk, layers);
    const int L = io.L;
    const size_t cw = (size_t)chunk * 4;  // device pitch of float planes
    int slot = 0;
    for (int64_t t0 = 0; t0 < io.n; t0 += chunk, slot = (slot + 1) % kSlots) {
        const int64_t m = io.n - t0 < chunk ? io.n - t0 : chunk;
        cudaStream_t st = stream[slot];
        char* b = buf[slot];
        const size_t w = (size_t)m * 4;
#define KF_TRY(x) do { e = (x); if (e != cudaSuccess) goto fail; } while (0)
        KF_TRY(cudaMemcpy2DAsync(b + lay.par, cw, io.par + t0, (size_t)io.ld_in * 4, w, 6, cudaMemcpyHostToDevice, st));
        KF_TRY(cudaMemcpy2DAsync(b + lay.cov, cw, io.cov + t0, (size_t)io.ld_in * 4, w, 21, cudaMemcpyHostToDevice, st));
        KF_TRY(cudaMemcpyAsync(b + lay.q, io.q + t0, (size_t)m, cudaMemcpyHostToDevice, st));
        if (io.mask) KF_TRY(cudaMemcpyAsync(b + lay.mask, io.mask + t0, w, cudaMemcpyHostToDevice, st));
        KF_TRY(cudaMemcpy2DAsync(b + lay.hpos, cw, io.hpos + t0, (size_t)io.ld_hit * 4, w, (size_t)L * 3, cudaMemcpyHostToDevice, st));
        KF_TRY(cudaMemcpy2DAsync(b + lay.hcov, cw, io.hcov + t0, (size_t)io.ld_hit * 4, w, (size_t)L * 6, cudaMemcpyHostToDevice, st));
        {
            FitArgs a;
            a.n = m;
            a.par = (const float*)(b + lay.par); a.cov = (const float*)(b + lay.cov); a.ld_in = chunk;
            a.q = (const int8_t*)(b + lay.q);
            a.hpos = (const float*)(b + lay.hpos); a.hcov = (const float*)(b + lay.hcov); a.ld_hit = chunk;
            a.mask = io.mask ? (const uint32_t*)(b + lay.mask) : nullptr;
            a.opar = (float*)(b + lay.opar); a.ocov = (float*)(b + lay.ocov); a.ld_out = chunk;
            a.chi2 = (float*)(b + lay.chi2); a.nhits = (int32_t*)(b + lay.nhits); a.status = (uint32_t*)(b + lay.status);
            KF_TRY(launch_fit(P, a, st, opt));
        }
        KF_TRY(cudaMemcpy2DAsync(io.opar + t0, (size_t)io.ld_out * 4, b + lay.opar, cw, w, 6, cudaMemcpyDeviceToHost, st));
        KF_TRY(cudaMemcpy2DAsync(io.ocov + t0, (size_t)io.ld_out * 4, b + lay.ocov, cw, w, 21, cudaMemcpyDeviceToHost, st));
        KF_TRY(cudaMemcpyAsync(io.chi2 + t0, b + lay.chi2, w, cudaMemcpyDeviceToHost, st));
        KF_TRY(cudaMemcpyAsync(io.nhits + t0, b + lay.nhits, w, cudaMemcpyDeviceToHost, st));
        KF_TRY(cudaMemcpyAsync(io.status + t0, b + lay.status, w, cudaMemcpyDeviceToHost, st));
#undef KF_TRY
    }
    for (int s = 0; s < kSlots; ++s) {
        cudaError_t es = cudaStreamSynchronize(stream[s]);
        if (es != cudaSuccess && e == cudaSuccess) e = es;
    }
    return e;
fail:
    for (int s = 0; s < kSlots; ++s) cudaStreamSynchronize(stream[s]);
    return e;
}

}  // namespace kf
