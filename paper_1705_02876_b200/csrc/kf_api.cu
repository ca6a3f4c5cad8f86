// kf_api.cu -- the C ABI of include/kf_b200.h: argument checks, host-side per-layer constants,
// context scratch, kernel launches.  No arithmetic of the method lives here except the per-layer
// constants (radius^2, 1/radius, Highland prefactor) that the kernels read.
#include <atomic>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "../../include/kf_b200.h"
#include "kf_internal.h"

using namespace kf;

struct kf_graph {
    cudaGraphExec_t exec = nullptr;
    int device = 0;
    uint64_t ctx_id = 0;      // the context whose scratch the recorded kernels point into
    uint64_t scratch_gen = 0; // that context's scratch generation when the recording ended
};

struct kf_ctx {
    uint64_t id = 0;          // process-wide serial number (a graph remembers which context recorded it)
    LaunchOptions opt;
    int device = 0;
    bool capturing = false;
    cudaStream_t stream = nullptr;
    int last_cuda = 0;
    // kf_bin_hits scratch
    BinScratch bin;
    // kf_score_candidates / kf_build_best_hit scratch
    ScoreScratch score;
    CombScratch comb;
    // kf_fit_tracks_indexed: the pools as packed records
    IndexScratch index;
    // *_host staging
    HostStage host;
    BuildHostStage build_host;
    // every reallocation of scratch and every rewrite of the bin edge tables moves this on
    uint64_t scratch_gen() const { return bin.gen + score.gen + comb.gen + index.gen; }
};

namespace {

constexpr int kAbiVersion = 14;
static_assert(kRecFloats == KF_HIT_RECORD_FLOATS || kRecWords == 4, "kf_internal.h and kf_b200.h disagree on the hit record");

// Makes the context's device current for the duration of an ABI call and puts the caller's device back on
// return (the library links its own cudart next to torch's: both see the same current device).
struct DeviceGuard {
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int device) {
        err = cudaGetDevice(&prev);
        if (err != cudaSuccess) { prev = -1; return; }
        if (prev != device) err = cudaSetDevice(device);
    }
    ~DeviceGuard() {
        if (prev >= 0) {
            int now = -1;
            if (cudaGetDevice(&now) == cudaSuccess && now != prev) cudaSetDevice(prev);
        }
    }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};
#define KF_ON_DEVICE(c)                                    \
    DeviceGuard kf_guard_((c)->device);                    \
    if (kf_guard_.err != cudaSuccess) return cuda_fail((c), kf_guard_.err)

int cuda_fail(kf_ctx* c, cudaError_t e) {
    if (c) c->last_cuda = (int)e;
    return KF_ERR_CUDA;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// Geometry -> kernel constants.  Returns KF_OK or an error code.  allow_discs: the call knows disc layers
// (reading A23: kf_fit_tracks, kf_fit_tracks_indexed, kf_fit_tracks_host); every other call refuses them.
int make_params(const kf_geometry* g, FitParams* P, bool allow_discs = false) {
    if (!g || !g->radius_cm || !g->x_over_X0) return KF_ERR_NULL;
    if (g->n_layers < 1) return KF_ERR_SHAPE;
    if (g->n_layers > KF_MAX_LAYERS) return KF_ERR_UNSUPPORTED;
    if (!(std::fabs((double)g->Bz_tesla) >= 1e-6)) return KF_ERR_UNSUPPORTED;
    std::memset(P, 0, sizeof(*P));
    P->n_layers = g->n_layers;
    const double k0 = 2.99792458e-3 * (double)g->Bz_tesla;  // reading A1
    P->k0 = (float)k0;
    P->inv_k0 = (float)(1.0 / k0);
    P->mass2 = (float)((double)g->mass_gev * (double)g->mass_gev);
    double prev = 0.0;
    bool discs = false;
    for (int l = 0; l < g->n_layers; ++l) {
        const double r = g->radius_cm[l];
        if (!(r > prev)) return KF_ERR_UNSUPPORTED;  // strictly increasing, > 0 (also rejects NaN)
        prev = r;
        P->layer[l].type = 0;
        P->layer[l].rmax2 = INFINITY;
        if (g->surface_type && g->surface_type[l] != 0) {   // reading A23: a pair of endcap discs
            if (g->surface_type[l] != 1 || !allow_discs) return KF_ERR_UNSUPPORTED;
            if (!g->disc_z_cm || !g->disc_rmin_cm || !g->disc_rmax_cm) return KF_ERR_NULL;
            const double zd = g->disc_z_cm[l], lo = g->disc_rmin_cm[l], hi = g->disc_rmax_cm[l];
            if (!(zd > 0.0) || !(lo >= 0.0) || !(hi > lo)) return KF_ERR_UNSUPPORTED;
            P->layer[l].type = 1;
            P->layer[l].zd = (float)zd;
            P->layer[l].rmin2 = (float)(lo * lo);
            P->layer[l].rmax2 = (float)(hi * hi);
            discs = true;
        }
        const double t = g->x_over_X0[l];
        double ms = 0.0;
        if (t > 0.0) {  // reading A5: theta0 = 0.0136/(beta p) sqrt(t) (1 + 0.038 ln t)
            const double f = 1.0 + 0.038 * std::log(t);
            ms = 0.0136 * 0.0136 * t * f * f;
        }
        P->layer[l].r = (float)r;
        P->layer[l].r2 = (float)(r * r);
        P->layer[l].inv_r = (float)(1.0 / r);
        P->layer[l].ms = (float)ms;
        // reading A20
        P->layer[l].ms0 = t > 0.0 ? (float)(0.0136 * 0.0136 * t) : 0.0f;
        P->layer[l].ln_t = t > 0.0 ? (float)std::log(t) : 0.0f;
        float hl = INFINITY;
        if (g->half_length_cm) {
            hl = g->half_length_cm[l];
            if (!(hl > 0.0f)) return KF_ERR_UNSUPPORTED;   // also rejects NaN; +inf = unbounded
        }
        P->layer[l].half_len = hl;
    }
    if (g->material_model != 0 && g->material_model != 1) return KF_ERR_UNSUPPORTED;
    if (g->energy_loss_model != 0 && g->energy_loss_model != 1) return KF_ERR_UNSUPPORTED;
    P->model = (g->material_model ? (int)MODEL_PATH_LENGTH : 0) | (g->energy_loss_model ? (int)MODEL_ENERGY_LOSS : 0);
    if (g->energy_loss_model) {  // reading A21: Bethe, silicon
        const double m = (double)g->mass_gev, me = 0.51099895e-3, I = 173.0e-9;
        if (!(m > 0.0)) return KF_ERR_UNSUPPORTED;
        P->el.a = (float)std::log(2.0 * me / (I * m * m));    // ln(2 me (beta gamma)^2 / I) = a + ln p^2
        P->el.b = (float)(2.0 * me / (m * m));                // 1 + 2 gamma me/M + (me/M)^2 = c + b E
        P->el.c = (float)(1.0 + (me / m) * (me / m));
        P->el.mass = (float)m;
        for (int l = 0; l < g->n_layers; ++l) {
            const double t = g->x_over_X0[l];
            P->layer[l].de0 = t > 0.0 ? (float)(0.307075e-3 * (14.0 / 28.0855) * t * 21.82) : 0.0f;
        }
    }
    P->geometry_options = (P->model != 0 || discs) ? 1 : 0;
    P->has_discs = discs ? 1 : 0;
    for (int l = 0; l < g->n_layers; ++l) P->geometry_options |= std::isfinite(P->layer[l].half_len) ? 1 : 0;
    return KF_OK;
}

int check_tracks(const kf_tracks* t, bool need_q, bool device) {
    if (!t) return KF_ERR_NULL;
    if (t->n < 0 || t->ld < t->n) return KF_ERR_SHAPE;
    if (t->n == 0) return KF_OK;
    if (!t->par || !t->cov || !t->chi2 || !t->nhits || !t->status) return KF_ERR_NULL;
    if (need_q && !t->q) return KF_ERR_NULL;
    if (device) {
        if (t->ld % 4 != 0) return KF_ERR_ALIGN;
        if (!aligned16(t->par) || !aligned16(t->cov)) return KF_ERR_ALIGN;
    }
    return KF_OK;
}

int check_track_hits(const kf_track_hits* h, const kf_geometry* g, int64_t n, bool device) {
    if (!h) return KF_ERR_NULL;
    if (h->n_layers != g->n_layers || h->n != n || h->ld < h->n) return KF_ERR_SHAPE;
    if (n == 0) return KF_OK;
    if (!h->pos || !h->cov) return KF_ERR_NULL;
    if (device) {
        if (h->ld % 4 != 0) return KF_ERR_ALIGN;
        if (!aligned16(h->pos) || !aligned16(h->cov)) return KF_ERR_ALIGN;
    }
    return KF_OK;
}

}  // namespace

extern "C" {

int kf_abi_version(void) { return kAbiVersion; }

int kf_hit_record_floats(void) { return kRecFloats; }

const char* kf_strerror(int code) {
    switch (code) {
        case KF_OK: return "ok";
        case KF_ERR_NULL: return "a required pointer is NULL";
        case KF_ERR_SHAPE: return "inconsistent sizes (n, ld, n_layers or layer index)";
        case KF_ERR_ALIGN: return "device pointer not 16-byte aligned or ld not a multiple of 4";
        case KF_ERR_UNSUPPORTED: return "unsupported configuration (layers > 32, |Bz| < 1e-6 T, radii not increasing, bins)";
        case KF_ERR_CUDA: return "a CUDA runtime call failed (see kf_last_cuda_error)";
        case KF_ERR_NOMEM: return "scratch allocation failed";
        case KF_ERR_STALE: return "stale graph: its context is gone or has reallocated scratch / changed the bin grid since the recording";
        case KF_ERR_TOO_LARGE: return "more candidates than the static scratch holds (KF_STATIC_MAX_CANDIDATES = 65536)";
        default: return "unknown error code";
    }
}

int kf_create(kf_ctx** out, int device, void* cuda_stream) {
    if (!out) return KF_ERR_NULL;
    *out = nullptr;
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess || device < 0 || device >= count) return KF_ERR_CUDA;  // no CPU fallback
    {
        DeviceGuard g(device);   // creates the primary context of `device` if need be, leaves the caller's device current
        if (g.err != cudaSuccess) return KF_ERR_CUDA;
        if ((e = cudaFree(nullptr)) != cudaSuccess) return KF_ERR_CUDA;
    }
    kf_ctx* c = new (std::nothrow) kf_ctx();
    if (!c) return KF_ERR_NOMEM;
    static std::atomic<uint64_t> serial{0};
    c->id = ++serial;
    c->device = device;
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    *out = c;
    return KF_OK;
}

int kf_destroy(kf_ctx* c) {
    if (!c) return KF_ERR_NULL;
    DeviceGuard g(c->device);
    c->bin.release();
    c->score.release();
    c->comb.release();
    c->index.release();
    c->host.release();
    c->build_host.release();
    delete c;
    return KF_OK;
}

int kf_set_stream(kf_ctx* c, void* cuda_stream) {
    if (!c) return KF_ERR_NULL;
    if (c->capturing) return KF_ERR_UNSUPPORTED;
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    return KF_OK;
}

int kf_set_option(kf_ctx* c, int option, int64_t value) {
    if (!c) return KF_ERR_NULL;
    switch (option) {
        case KF_OPT_PAIR_MIN_TRACKS:
            if (value < 0) return KF_ERR_SHAPE;
            c->opt.pair_min_tracks = value;
            return KF_OK;
        case KF_OPT_REFIT_PAIR_MASKED:
            c->opt.refit_pair_masked = value != 0;
            return KF_OK;
        case KF_OPT_BIN_FORM:
            if (value < 0 || value > 2) return KF_ERR_SHAPE;
            c->opt.bin_form = (int)value;
            return KF_OK;
        default:
            return KF_ERR_UNSUPPORTED;
    }
}

int kf_last_cuda_error(const kf_ctx* c) { return c ? c->last_cuda : 0; }

// ---- CUDA-graph capture of a sequence of hot calls (include/kf_b200.h "graphs") ----------------------------
int kf_graph_begin(kf_ctx* c) {
    if (!c) return KF_ERR_NULL;
    if (c->capturing || c->stream == nullptr) return KF_ERR_UNSUPPORTED;  // the legacy default stream cannot be captured
    KF_ON_DEVICE(c);
    cudaError_t e;
    // relaxed: other host threads (torch's allocator, NCCL watchdogs) may keep calling the runtime meanwhile
    if ((e = cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeRelaxed)) != cudaSuccess) return cuda_fail(c, e);
    c->capturing = true;
    return KF_OK;
}

int kf_graph_end(kf_ctx* c, kf_graph** out) {
    if (!c || !out) return KF_ERR_NULL;
    *out = nullptr;
    if (!c->capturing) return KF_ERR_UNSUPPORTED;
    KF_ON_DEVICE(c);
    c->capturing = false;
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->stream, &g);
    if (e != cudaSuccess || !g) {   // a captured call synchronised or allocated (scratch not reserved): capture void
        if (g) cudaGraphDestroy(g);
        cudaGetLastError();
        return cuda_fail(c, e != cudaSuccess ? e : cudaErrorStreamCaptureInvalidated);
    }
    kf_graph* kg = new (std::nothrow) kf_graph();
    if (!kg) { cudaGraphDestroy(g); return KF_ERR_NOMEM; }
    kg->device = c->device;
    kg->ctx_id = c->id;
    kg->scratch_gen = c->scratch_gen();
    e = cudaGraphInstantiate(&kg->exec, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { delete kg; return cuda_fail(c, e); }
    *out = kg;
    return KF_OK;
}

int kf_graph_launch(kf_ctx* c, kf_graph* g) {
    if (!c || !g || !g->exec) return KF_ERR_NULL;
    if (c->capturing || g->device != c->device) return KF_ERR_UNSUPPORTED;
    // The recorded kernels point into the recording context's scratch and bin edge tables: a graph is stale
    // (and is refused) once that context is gone or has reallocated scratch / rewritten the tables since.
    if (g->ctx_id != c->id || g->scratch_gen != c->scratch_gen()) return KF_ERR_STALE;
    KF_ON_DEVICE(c);
    cudaError_t e;
    if ((e = cudaGraphLaunch(g->exec, c->stream)) != cudaSuccess) return cuda_fail(c, e);
    return KF_OK;
}

int kf_graph_destroy(kf_graph* g) {
    if (!g) return KF_ERR_NULL;
    if (g->exec) cudaGraphExecDestroy(g->exec);
    delete g;
    return KF_OK;
}

int kf_reserve(kf_ctx* c, int64_t max_hits, int64_t max_host_tracks, int max_host_layers) {
    if (!c) return KF_ERR_NULL;
    if (max_hits < 0 || max_host_tracks < 0 || max_host_layers < 0 || max_host_layers > KF_MAX_LAYERS)
        return KF_ERR_SHAPE;
    KF_ON_DEVICE(c);
    cudaError_t e;
    if (max_hits > 0) {
        e = c->bin.reserve(max_hits, 2 * (KF_MAX_BINS + 1), c->stream, true);
        if (e == cudaSuccess) e = reserve_chunked(c->bin, max_hits, KF_MAX_LAYERS, c->stream);
        if (e == cudaSuccess) e = c->index.reserve((size_t)(max_hits + 4 * KF_MAX_LAYERS) * kRecFloats * 4, c->stream);
        if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? KF_ERR_NOMEM : cuda_fail(c, e);
    }
    if (max_host_tracks > 0 && max_host_layers > 0) {
        e = c->host.reserve(max_host_tracks, max_host_layers);
        if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? KF_ERR_NOMEM : cuda_fail(c, e);
    }
    return KF_OK;
}

int kf_measure_fp32_packed_rate(kf_ctx* c, int repeats, double* shared_tflops, double* distinct_tflops) {
    if (!c || !shared_tflops || !distinct_tflops) return KF_ERR_NULL;
    if (repeats < 1) return KF_ERR_SHAPE;
    if (c->capturing) return KF_ERR_UNSUPPORTED;
    KF_ON_DEVICE(c);
    cudaError_t e;
    constexpr int kWords = 32 * 3 * 8 * 2 + 4;
    float* scratch = nullptr;
    if ((e = cudaMalloc(&scratch, kWords * 4)) != cudaSuccess) return cuda_fail(c, e);
    static float init[kWords];
    for (int i = 0; i < kWords; ++i) init[i] = 0.999f + 1e-5f * (float)(i % 7);
    e = cudaMemcpyAsync(scratch, init, kWords * 4, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e == cudaSuccess) e = measure_fp32_packed_rate(c->stream, repeats, scratch, shared_tflops, distinct_tflops);
    cudaFree(scratch);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return KF_OK;
}

int kf_measure_fp32_peak(kf_ctx* c, int repeats, double* tflops_out) {
    if (!c || !tflops_out) return KF_ERR_NULL;
    if (repeats < 1) return KF_ERR_SHAPE;
    KF_ON_DEVICE(c);
    cudaError_t e;
    float* sink = nullptr;
    if ((e = cudaMalloc(&sink, 16)) != cudaSuccess) return cuda_fail(c, e);
    const double t = measure_fp32_peak(c->stream, repeats, sink);
    cudaFree(sink);
    if (t < 0.0) return cuda_fail(c, (cudaError_t)(int)(-t));
    *tflops_out = t;
    return KF_OK;
}

int kf_fit_tracks(kf_ctx* c, const kf_geometry* geom, const kf_tracks* seeds,
                  const kf_track_hits* hits, kf_tracks* out) {
    if (!c || !geom || !seeds || !hits || !out) return KF_ERR_NULL;
    FitParams P;
    int rc = make_params(geom, &P, true);
    if (rc) return rc;
    if ((rc = check_tracks(seeds, true, true))) return rc;
    if ((rc = check_tracks(out, false, true))) return rc;
    if (out->n != seeds->n) return KF_ERR_SHAPE;
    if ((rc = check_track_hits(hits, geom, seeds->n, true))) return rc;
    if (seeds->n == 0) return KF_OK;
    if (seeds->n > 0x7fffffffLL) return KF_ERR_UNSUPPORTED;  // TMA tile coordinates are int32
    FitArgs a;
    a.n = seeds->n;
    a.par = seeds->par; a.cov = seeds->cov; a.ld_in = seeds->ld; a.q = seeds->q;
    a.hpos = hits->pos; a.hcov = hits->cov; a.ld_hit = hits->ld; a.mask = hits->mask;
    a.opar = out->par; a.ocov = out->cov; a.ld_out = out->ld;
    a.chi2 = out->chi2; a.nhits = out->nhits; a.status = out->status;
    KF_ON_DEVICE(c);
    cudaError_t e = launch_fit(P, a, c->stream, c->opt);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return KF_OK;
}

int kf_fit_tracks_indexed(kf_ctx* c, const kf_geometry* geom, const kf_tracks* seeds, const int32_t* index,
                          int64_t ld_index, const kf_layer_hits* pools, const kf_layer_bins* bins, kf_tracks* out) {
    if (!c || !geom || !seeds || !pools || !out) return KF_ERR_NULL;
    FitParams P;
    int rc = make_params(geom, &P, true);
    if (rc) return rc;
    if ((rc = check_tracks(seeds, true, true))) return rc;
    if ((rc = check_tracks(out, false, true))) return rc;
    if (out->n != seeds->n || ld_index < seeds->n) return KF_ERR_SHAPE;
    if (seeds->n == 0) return KF_OK;
    if (!index) return KF_ERR_NULL;
    IndexedPools H;
    std::memset(&H, 0, sizeof(H));
    for (int l = 0; l < geom->n_layers; ++l) {
        if (pools[l].n_hits < 0 || pools[l].ld < pools[l].n_hits) return KF_ERR_SHAPE;
        if (pools[l].n_hits > 0 && (!pools[l].pos || !pools[l].cov)) return KF_ERR_NULL;
        H.pos[l] = pools[l].pos; H.cov[l] = pools[l].cov; H.ld[l] = pools[l].ld;
        if (bins) {
            if (pools[l].n_hits > 0 && (!bins[l].hit_rec || !bins[l].orig_to_sorted)) return KF_ERR_NULL;
            if (!aligned16(bins[l].hit_rec)) return KF_ERR_ALIGN;
            H.hit_rec[l] = bins[l].hit_rec; H.orig_to_sorted[l] = bins[l].orig_to_sorted;
        }
    }
    H.use_records = bins ? 1 : 0;
    H.index = index; H.ld_index = ld_index;
    FitArgs a;
    a.n = seeds->n;
    a.par = seeds->par; a.cov = seeds->cov; a.ld_in = seeds->ld; a.q = seeds->q;
    a.hpos = nullptr; a.hcov = nullptr; a.ld_hit = 0; a.mask = nullptr;
    a.opar = out->par; a.ocov = out->cov; a.ld_out = out->ld;
    a.chi2 = out->chi2; a.nhits = out->nhits; a.status = out->status;
    KF_ON_DEVICE(c);
    cudaError_t e;
    if (!bins) {
        // SoA pools: nine scattered 4-byte loads per hit cost nine memory sectors.  Unless the pools are far larger
        // than what the tracks will read of them, pack them once into 48-byte records (original order, context
        // scratch) and gather those: two sectors per hit.
        PackPools A;
        std::memset(&A, 0, sizeof(A));
        int64_t total = 0;
        for (int l = 0; l < geom->n_layers; ++l) total += (pools[l].n_hits + 3) / 4 * 4;
        if (total > 0 && total <= 8 * seeds->n * (int64_t)geom->n_layers) {
            e = c->index.reserve((size_t)total * kRecFloats * 4, c->stream);
            if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? KF_ERR_NOMEM : cuda_fail(c, e);
            int64_t at = 0;
            for (int l = 0; l < geom->n_layers; ++l) {
                A.pos[l] = pools[l].pos; A.cov[l] = pools[l].cov; A.ld[l] = pools[l].ld; A.n[l] = pools[l].n_hits;
                A.rec[l] = c->index.rec + at * kRecFloats;
                H.hit_rec[l] = A.rec[l];
                at += (pools[l].n_hits + 3) / 4 * 4;
            }
            e = launch_pack_pools(A, geom->n_layers, c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e);
            H.use_records = 2;
        }
    }
    e = launch_fit_indexed(P, H, a, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return KF_OK;
}

int kf_fit_tracks_refit(kf_ctx* c, const kf_geometry* geom, const kf_tracks* seeds, const kf_track_hits* hits,
                         float kappa, kf_tracks* out, kf_tracks* smoothed) {
    if (!c || !geom || !seeds || !hits || !out || !smoothed) return KF_ERR_NULL;
    FitParams P;
    int rc = make_params(geom, &P, true);
    if (rc) return rc;
    if (!(kappa >= 1.0f)) return KF_ERR_UNSUPPORTED;
    if ((rc = check_tracks(seeds, true, true))) return rc;
    if ((rc = check_tracks(out, false, true))) return rc;
    if ((rc = check_tracks(smoothed, false, true))) return rc;
    if (out->n != seeds->n || smoothed->n != seeds->n) return KF_ERR_SHAPE;
    if ((rc = check_track_hits(hits, geom, seeds->n, true))) return rc;
    if (seeds->n == 0) return KF_OK;
    if (seeds->n > 0x7fffffffLL) return KF_ERR_UNSUPPORTED;
    if (smoothed->par == seeds->par || smoothed->par == out->par || smoothed->cov == seeds->cov ||
        smoothed->cov == out->cov)
        return KF_ERR_UNSUPPORTED;
    FitArgs a;
    a.n = seeds->n;
    a.par = seeds->par; a.cov = seeds->cov; a.ld_in = seeds->ld; a.q = seeds->q;
    a.hpos = hits->pos; a.hcov = hits->cov; a.ld_hit = hits->ld; a.mask = hits->mask;
    a.opar = out->par; a.ocov = out->cov; a.ld_out = out->ld;
    a.chi2 = out->chi2; a.nhits = out->nhits; a.status = out->status;
    a.spar = smoothed->par; a.scov = smoothed->cov; a.ld_s = smoothed->ld;
    a.schi2 = smoothed->chi2; a.snhits = smoothed->nhits; a.sstatus = smoothed->status;
    a.kappa = kappa;
    KF_ON_DEVICE(c);
    cudaError_t e = launch_fit(P, a, c->stream, c->opt);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return KF_OK;
}

int kf_fit_tracks_smooth(kf_ctx* c, const kf_geometry* geom, const kf_tracks* seeds, const kf_track_hits* hits,
                         kf_tracks* out, kf_smoothed* sm) {
    if (!c || !geom || !seeds || !hits || !out || !sm) return KF_ERR_NULL;
    FitParams P;
    int rc = make_params(geom, &P, true);   // (discs: reading A23, the forward kernel and the backward step both know them)
    if (rc) return rc;
    if ((rc = check_tracks(seeds, true, true))) return rc;
    if ((rc = check_tracks(out, false, true))) return rc;
    if (out->n != seeds->n || sm->n != seeds->n || sm->n_layers != geom->n_layers || sm->ld < sm->n) return KF_ERR_SHAPE;
    if ((rc = check_track_hits(hits, geom, seeds->n, true))) return rc;
    if (seeds->n == 0) return KF_OK;
    if (seeds->n > 0x7fffffffLL) return KF_ERR_UNSUPPORTED;
    if (!sm->par || !sm->cov || !sm->used) return KF_ERR_NULL;
    if (sm->ld % 4 != 0 || !aligned16(sm->par) || !aligned16(sm->cov)) return KF_ERR_ALIGN;
    FitArgs a;
    a.n = seeds->n;
    a.par = seeds->par; a.cov = seeds->cov; a.ld_in = seeds->ld; a.q = seeds->q;
    a.hpos = hits->pos; a.hcov = hits->cov; a.ld_hit = hits->ld; a.mask = hits->mask;
    a.opar = out->par; a.ocov = out->cov; a.ld_out = out->ld;
    a.chi2 = out->chi2; a.nhits = out->nhits; a.status = out->status;
    a.lpar = sm->par; a.lcov = sm->cov; a.ld_l = sm->ld; a.used = sm->used;
    KF_ON_DEVICE(c);
    cudaError_t e = launch_fit(P, a, c->stream, c->opt);
    if (e == cudaSuccess) e = launch_rts(P, a, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return KF_OK;
}

namespace {
int fit_tracks_host(kf_ctx* c, const kf_geometry* geom, const kf_tracks* seeds, const kf_track_hits* hits, kf_tracks* out,
                    bool cov_diagonal, bool hit_cov_local = false);
}
int kf_fit_tracks_host(kf_ctx* c, const kf_geometry* geom, const kf_tracks* seeds,
                       const kf_track_hits* hits, kf_tracks* out) {
    return fit_tracks_host(c, geom, seeds, hits, out, false);
}
int kf_fit_tracks_host_diag(kf_ctx* c, const kf_geometry* geom, const kf_tracks* seeds,
                            const kf_track_hits* hits, kf_tracks* out) {
    return fit_tracks_host(c, geom, seeds, hits, out, true);
}
int kf_fit_tracks_host_compact(kf_ctx* c, const kf_geometry* geom, const kf_tracks* seeds,
                               const kf_track_hits* hits, kf_tracks* out) {
    return fit_tracks_host(c, geom, seeds, hits, out, true, true);
}
}  // extern "C"
namespace {
int fit_tracks_host(kf_ctx* c, const kf_geometry* geom, const kf_tracks* seeds, const kf_track_hits* hits, kf_tracks* out,
                    bool cov_diagonal, bool hit_cov_local) {
    if (!c || !geom || !seeds || !hits || !out) return KF_ERR_NULL;
    FitParams P;
    int rc = make_params(geom, &P, true);
    if (rc) return rc;
    if ((rc = check_tracks(seeds, true, false))) return rc;
    if ((rc = check_tracks(out, false, false))) return rc;
    if (out->n != seeds->n) return KF_ERR_SHAPE;
    if ((rc = check_track_hits(hits, geom, seeds->n, false))) return rc;
    if (seeds->n == 0) return KF_OK;
    KF_ON_DEVICE(c);
    cudaError_t e;
    HostFitIO io;
    io.n = seeds->n; io.L = geom->n_layers;
    io.par = seeds->par; io.cov = seeds->cov; io.ld_in = seeds->ld; io.q = seeds->q;
    io.hpos = hits->pos; io.hcov = hits->cov; io.ld_hit = hits->ld; io.mask = hits->mask;
    io.opar = out->par; io.ocov = out->cov; io.ld_out = out->ld;
    io.chi2 = out->chi2; io.nhits = out->nhits; io.status = out->status;
    io.cov_diagonal = cov_diagonal;
    io.hit_cov_local = hit_cov_local;
    e = c->host.fit(P, io, c->opt);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? KF_ERR_NOMEM : cuda_fail(c, e);
    return KF_OK;
}
}  // namespace
extern "C" {

namespace {

int check_bin_args(const kf_layer_hits* hits, const kf_layer_bins* out, float radius_cm) {
    if (!hits || !out) return KF_ERR_NULL;
    if (hits->n_hits < 0 || hits->ld < hits->n_hits) return KF_ERR_SHAPE;
    if (out->n_eta < 1 || out->n_phi < 2) return KF_ERR_SHAPE;
    if (out->n_phi % 2 != 0 || (int64_t)out->n_eta * out->n_phi > KF_MAX_BINS) return KF_ERR_UNSUPPORTED;
    if (!(radius_cm >= 0.0f) || !(out->eta_max > 0.0f)) return KF_ERR_UNSUPPORTED;   // (0: a disc layer, reading A24)
    if (hits->n_hits > 0x7fffffffLL) return KF_ERR_UNSUPPORTED;
    if (!out->bin_offset || !out->bin_box) return KF_ERR_NULL;
    if (!aligned16(out->bin_box)) return KF_ERR_ALIGN;
    if (hits->n_hits > 0) {
        if (!hits->pos || !hits->cov || !out->sorted_to_orig || !out->hit_rec) return KF_ERR_NULL;
        if (hits->ld % 4 != 0 || !aligned16(hits->pos) || !aligned16(hits->cov) || !aligned16(out->hit_rec))
            return KF_ERR_ALIGN;
        if (out->pos_sorted || out->cov_sorted) {
            if (out->ld < hits->n_hits) return KF_ERR_SHAPE;
            if (out->ld % 4 != 0 || !aligned16(out->pos_sorted) || !aligned16(out->cov_sorted)) return KF_ERR_ALIGN;
        }
    }
    return KF_OK;
}

BinArgs to_bin_args(float radius_cm, const kf_layer_hits* hits, const kf_layer_bins* out) {
    BinArgs a;
    a.n_hits = hits->n_hits; a.ld_in = hits->ld; a.pos = hits->pos; a.cov = hits->cov;
    a.radius = radius_cm; a.n_eta = out->n_eta; a.n_phi = out->n_phi; a.eta_max = out->eta_max;
    a.ld_out = out->ld; a.bin_offset = out->bin_offset; a.sorted_to_orig = out->sorted_to_orig;
    a.pos_sorted = out->pos_sorted; a.cov_sorted = out->cov_sorted; a.hit_rec = out->hit_rec; a.bin_box = out->bin_box;
    a.orig_to_sorted = out->orig_to_sorted;
    return a;
}

}  // namespace

int kf_bin_layers(kf_ctx* c, int n_layers, const float* radius_cm, const kf_layer_hits* hits, kf_layer_bins* out) {
    if (!c || !radius_cm || !hits || !out) return KF_ERR_NULL;
    if (n_layers < 0 || n_layers > KF_MAX_LAYERS) return KF_ERR_SHAPE;
    if (n_layers == 0) return KF_OK;
    BinArgs args[KF_MAX_LAYERS];
    for (int l = 0; l < n_layers; ++l) {
        const int rc = check_bin_args(hits + l, out + l, radius_cm[l]);
        if (rc) return rc;
        if (out[l].n_eta != out[0].n_eta || out[l].n_phi != out[0].n_phi || out[l].eta_max != out[0].eta_max)
            return KF_ERR_UNSUPPORTED;
        args[l] = to_bin_args(radius_cm[l], hits + l, out + l);
    }
    KF_ON_DEVICE(c);
    cudaError_t e = launch_bin(c->bin, n_layers, args, c->stream, c->opt);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? KF_ERR_NOMEM : cuda_fail(c, e);
    return KF_OK;
}

int kf_bin_hits(kf_ctx* c, float radius_cm, const kf_layer_hits* hits, kf_layer_bins* out) {
    return kf_bin_layers(c, 1, &radius_cm, hits, out);
}

int kf_order_candidates(kf_ctx* c, const kf_geometry* geom, int layer, const kf_tracks* cands, int n_eta,
                        int n_phi, float eta_max, int32_t* order) {
    if (!c || !geom || !cands) return KF_ERR_NULL;
    FitParams P;
    int rc = make_params(geom, &P, true);
    if (rc) return rc;
    if (layer < 0 || layer >= geom->n_layers) return KF_ERR_SHAPE;
    if (cands->n < 0 || cands->ld < cands->n || n_eta < 1 || n_phi < 2) return KF_ERR_SHAPE;
    if ((int64_t)n_eta * n_phi > KF_MAX_BINS || !(eta_max > 0.0f) || cands->n > 0x7fffffffLL) return KF_ERR_UNSUPPORTED;
    if (cands->n == 0) return KF_OK;
    if (!cands->par || !cands->q || !order) return KF_ERR_NULL;
    KF_ON_DEVICE(c);
    cudaError_t e = launch_order(c->bin, P, layer, cands->n, cands->ld, cands->par, cands->q, n_eta, n_phi, eta_max, order,
                     c->stream);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? KF_ERR_NOMEM : cuda_fail(c, e);
    return KF_OK;
}

namespace {

int check_score_bins(const kf_layer_hits* hits, const kf_layer_bins* bins, int window_half) {
    if (!hits || !bins) return KF_ERR_NULL;
    if (hits->n_hits < 0) return KF_ERR_SHAPE;
    if (bins->n_eta < 1 || bins->n_phi < 2 || window_half < 0) return KF_ERR_SHAPE;
    if (bins->n_phi % 2 != 0 || (int64_t)bins->n_eta * bins->n_phi > KF_MAX_BINS) return KF_ERR_UNSUPPORTED;
    if (2 * window_half + 1 > bins->n_phi) return KF_ERR_UNSUPPORTED;
    if (!(bins->eta_max > 0.0f)) return KF_ERR_UNSUPPORTED;
    if (!bins->bin_offset || !bins->bin_box) return KF_ERR_NULL;
    if (!aligned16(bins->bin_box)) return KF_ERR_ALIGN;
    if (hits->n_hits > 0) {
        if (!bins->hit_rec) return KF_ERR_NULL;
        if (!aligned16(bins->hit_rec)) return KF_ERR_ALIGN;
    }
    return KF_OK;
}

}  // namespace

namespace {
int build_best_hit(kf_ctx* c, const kf_geometry* geom, int first_layer, int n_build_layers, kf_tracks* cands,
                   const kf_layer_hits* hits, const kf_layer_bins* bins, int window_half, float chi2_cut,
                   int do_update, const int32_t* order, int32_t* hit_index, float* hit_chi2, int64_t ld_out,
                   float* local_state) {
    if (!c || !geom || !cands || !hits || !bins) return KF_ERR_NULL;
    FitParams P;
    int rc = make_params(geom, &P, true);   // (discs: readings A23 / A24)
    if (rc) return rc;
    if (n_build_layers < 0 || first_layer < 0 || first_layer + n_build_layers > geom->n_layers) return KF_ERR_SHAPE;
    if ((rc = check_tracks(cands, true, true))) return rc;
    if (n_build_layers == 0 || cands->n == 0) return KF_OK;
    if (!hit_index || !hit_chi2) return KF_ERR_NULL;
    if (ld_out < cands->n) return KF_ERR_SHAPE;
    ScoreStep steps[KF_MAX_LAYERS];
    for (int j = 0; j < n_build_layers; ++j) {
        if ((rc = check_score_bins(hits + j, bins + j, window_half))) return rc;
        if (bins[j].n_eta != bins[0].n_eta || bins[j].n_phi != bins[0].n_phi || bins[j].eta_max != bins[0].eta_max)
            return KF_ERR_UNSUPPORTED;
        steps[j].layer = first_layer + j;
        steps[j].n_hits = hits[j].n_hits;
        steps[j].hit_rec = bins[j].hit_rec;
        steps[j].bin_box = bins[j].bin_box;
        steps[j].bin_offset = bins[j].bin_offset;
        steps[j].best_hit = hit_index + (int64_t)j * ld_out;
        steps[j].best_chi2 = hit_chi2 + (int64_t)j * ld_out;
    }
    ScoreArgs a;
    std::memset(&a, 0, sizeof(a));
    a.n = cands->n; a.ld = cands->ld; a.par = cands->par; a.cov = cands->cov; a.q = cands->q;
    a.chi2 = cands->chi2; a.nhits = cands->nhits; a.status = cands->status;
    a.order = order;
    a.n_eta = bins[0].n_eta; a.n_phi = bins[0].n_phi; a.eta_max = bins[0].eta_max;
    a.window_half = window_half; a.chi2_cut = chi2_cut; a.do_update = do_update ? 1 : 0;
    if (local_state && !aligned16(local_state)) return KF_ERR_ALIGN;
    a.lstate = local_state; a.ld_ls = cands->ld;
    KF_ON_DEVICE(c);
    cudaError_t e = launch_build(c->score, P, a, n_build_layers, steps, c->stream);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? KF_ERR_NOMEM : cuda_fail(c, e);
    return KF_OK;
}
}  // namespace

int kf_build_best_hit(kf_ctx* c, const kf_geometry* geom, int first_layer, int n_build_layers, kf_tracks* cands,
                      const kf_layer_hits* hits, const kf_layer_bins* bins, int window_half, float chi2_cut,
                      int do_update, const int32_t* order, int32_t* hit_index, float* hit_chi2, int64_t ld_out) {
    return build_best_hit(c, geom, first_layer, n_build_layers, cands, hits, bins, window_half, chi2_cut, do_update,
                          order, hit_index, hit_chi2, ld_out, nullptr);
}

int kf_build_best_hit_events(kf_ctx* c, const kf_geometry* geom, int first_layer, int n_build_layers, int n_events,
                             const int64_t* event_first, kf_tracks* cands, const kf_layer_hits* hits,
                             const kf_layer_bins* bins, int window_half, float chi2_cut, int do_update,
                             int32_t* hit_index, float* hit_chi2, int64_t ld_out) {
    if (!c || !geom || !cands || !hits || !bins || !event_first) return KF_ERR_NULL;
    FitParams P;
    int rc = make_params(geom, &P, true);
    if (rc) return rc;
    if (n_build_layers < 0 || first_layer < 0 || first_layer + n_build_layers > geom->n_layers) return KF_ERR_SHAPE;
    if (n_events < 1) return KF_ERR_SHAPE;
    if (n_events > kMaxBuildEvents) return KF_ERR_UNSUPPORTED;
    if ((rc = check_tracks(cands, true, true))) return rc;
    if (event_first[0] != 0 || event_first[n_events] != cands->n) return KF_ERR_SHAPE;
    for (int e = 0; e < n_events; ++e)
        if (event_first[e + 1] < event_first[e]) return KF_ERR_SHAPE;
    if (n_build_layers == 0 || cands->n == 0) return KF_OK;
    if (!hit_index || !hit_chi2) return KF_ERR_NULL;
    if (ld_out < cands->n) return KF_ERR_SHAPE;
    ScoreStep steps[KF_MAX_LAYERS];
    for (int j = 0; j < n_build_layers; ++j) {
        for (int e = 0; e < n_events; ++e) {
            const kf_layer_hits* h = hits + (int64_t)e * n_build_layers + j;
            const kf_layer_bins* b = bins + (int64_t)e * n_build_layers + j;
            if ((rc = check_score_bins(h, b, window_half))) return rc;
            if (b->n_eta != bins[0].n_eta || b->n_phi != bins[0].n_phi || b->eta_max != bins[0].eta_max)
                return KF_ERR_UNSUPPORTED;
            steps[j].ev_hit_rec[e] = b->hit_rec;
            steps[j].ev_bin_box[e] = b->bin_box;
            steps[j].ev_bin_offset[e] = b->bin_offset;
        }
        steps[j].layer = first_layer + j;
        steps[j].n_hits = hits[j].n_hits;
        steps[j].hit_rec = bins[j].hit_rec;
        steps[j].bin_box = bins[j].bin_box;
        steps[j].bin_offset = bins[j].bin_offset;
        steps[j].best_hit = hit_index + (int64_t)j * ld_out;
        steps[j].best_chi2 = hit_chi2 + (int64_t)j * ld_out;
    }
    ScoreArgs a;
    std::memset(&a, 0, sizeof(a));
    a.n = cands->n; a.ld = cands->ld; a.par = cands->par; a.cov = cands->cov; a.q = cands->q;
    a.chi2 = cands->chi2; a.nhits = cands->nhits; a.status = cands->status;
    a.n_eta = bins[0].n_eta; a.n_phi = bins[0].n_phi; a.eta_max = bins[0].eta_max;
    a.window_half = window_half; a.chi2_cut = chi2_cut; a.do_update = do_update ? 1 : 0;
    a.ev.n = n_events;
    for (int e = 0; e <= n_events; ++e) a.ev.first[e] = event_first[e];
    KF_ON_DEVICE(c);
    cudaError_t e = launch_build(c->score, P, a, n_build_layers, steps, c->stream);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? KF_ERR_NOMEM : cuda_fail(c, e);
    return KF_OK;
}

int kf_build_best_hit_host(kf_ctx* c, const kf_geometry* geom, int first_layer, int n_build_layers, kf_tracks* cands,
                           const kf_layer_hits* hits, int n_eta, int n_phi, float eta_max, int window_half,
                           float chi2_cut, int do_update, int32_t* hit_index, float* hit_chi2, int64_t ld_out) {
    if (!c || !geom || !cands || !hits) return KF_ERR_NULL;
    if (c->capturing) return KF_ERR_UNSUPPORTED;
    FitParams P;
    int rc = make_params(geom, &P, true);
    if (rc) return rc;
    if (n_build_layers < 0 || first_layer < 0 || first_layer + n_build_layers > geom->n_layers) return KF_ERR_SHAPE;
    if ((rc = check_tracks(cands, true, false))) return rc;
    if (n_eta < 1 || n_phi < 2 || window_half < 0) return KF_ERR_SHAPE;
    if (n_phi % 2 != 0 || (int64_t)n_eta * n_phi > KF_MAX_BINS || 2 * window_half + 1 > n_phi || !(eta_max > 0.0f))
        return KF_ERR_UNSUPPORTED;
    if (n_build_layers == 0 || cands->n == 0) return KF_OK;
    if (!hit_index || !hit_chi2) return KF_ERR_NULL;
    if (ld_out < cands->n || cands->n > 0x7fffffffLL) return KF_ERR_SHAPE;
    int64_t nh[KF_MAX_LAYERS], ldh[KF_MAX_LAYERS];
    const float* pos[KF_MAX_LAYERS];
    const float* cov[KF_MAX_LAYERS];
    for (int j = 0; j < n_build_layers; ++j) {
        if (hits[j].n_hits < 0 || hits[j].ld < hits[j].n_hits || hits[j].n_hits > 0x7fffffffLL) return KF_ERR_SHAPE;
        if (hits[j].n_hits > 0 && (!hits[j].pos || !hits[j].cov)) return KF_ERR_NULL;
        nh[j] = hits[j].n_hits; ldh[j] = hits[j].ld; pos[j] = hits[j].pos; cov[j] = hits[j].cov;
    }
    BuildHostIO io;
    io.n = cands->n; io.ld = cands->ld; io.par = cands->par; io.cov = cands->cov; io.q = cands->q;
    io.chi2 = cands->chi2; io.nhits = cands->nhits; io.status = cands->status;
    io.first_layer = first_layer; io.n_layers = n_build_layers;
    io.n_hits = nh; io.ld_hits = ldh; io.pos = pos; io.cov_hits = cov;
    io.n_eta = n_eta; io.n_phi = n_phi; io.eta_max = eta_max; io.window_half = window_half; io.chi2_cut = chi2_cut;
    io.do_update = do_update ? 1 : 0;
    io.hit_index = hit_index; io.hit_chi2 = hit_chi2; io.ld_out = ld_out;
    KF_ON_DEVICE(c);
    cudaError_t e = build_best_hit_host(c->build_host, c->bin, c->score, P, io, c->stream, c->opt);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? KF_ERR_NOMEM : cuda_fail(c, e);
    return KF_OK;
}

int kf_build_combinatorial(kf_ctx* c, const kf_geometry* geom, int first_layer, int n_build_layers, kf_tracks* cands,
                           const kf_layer_hits* hits, const kf_layer_bins* bins, int window_half, float chi2_cut,
                           int n_cand, int32_t* hit_index, int32_t* n_found, int64_t ld_out) {
    if (!c || !geom || !cands || !hits || !bins) return KF_ERR_NULL;
    FitParams P;
    int rc = make_params(geom, &P, true);
    if (rc) return rc;
    if (n_build_layers < 0 || first_layer < 0 || first_layer + n_build_layers > geom->n_layers) return KF_ERR_SHAPE;
    if (n_cand < 1 || n_cand > 8) return KF_ERR_UNSUPPORTED;
    if ((rc = check_tracks(cands, true, true))) return rc;
    if (n_build_layers == 0 || cands->n == 0) return KF_OK;
    if (!hit_index) return KF_ERR_NULL;
    if (ld_out < cands->n) return KF_ERR_SHAPE;
    if (cands->n * (int64_t)n_cand > 0x7fffffffLL) return KF_ERR_UNSUPPORTED;
    ScoreStep steps[KF_MAX_LAYERS];
    for (int j = 0; j < n_build_layers; ++j) {
        if ((rc = check_score_bins(hits + j, bins + j, window_half))) return rc;
        if (bins[j].n_eta != bins[0].n_eta || bins[j].n_phi != bins[0].n_phi || bins[j].eta_max != bins[0].eta_max)
            return KF_ERR_UNSUPPORTED;
        steps[j].layer = first_layer + j;
        steps[j].n_hits = hits[j].n_hits;
        steps[j].hit_rec = bins[j].hit_rec;
        steps[j].bin_box = bins[j].bin_box;
        steps[j].bin_offset = bins[j].bin_offset;
        steps[j].best_hit = nullptr;
        steps[j].best_chi2 = nullptr;
    }
    CombCall call;
    call.n_seeds = cands->n; call.ld = cands->ld; call.par = cands->par; call.cov = cands->cov; call.q = cands->q;
    call.chi2 = cands->chi2; call.nhits = cands->nhits; call.status = cands->status;
    call.n_cand = n_cand;
    call.n_eta = bins[0].n_eta; call.n_phi = bins[0].n_phi; call.eta_max = bins[0].eta_max;
    call.window_half = window_half; call.chi2_cut = chi2_cut;
    call.hit_index = hit_index; call.ld_out = ld_out; call.n_found = n_found;
    KF_ON_DEVICE(c);
    cudaError_t e = launch_comb(c->comb, P, call, n_build_layers, steps, c->stream);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? KF_ERR_NOMEM : cuda_fail(c, e);
    return KF_OK;
}

int kf_build_combinatorial_events(kf_ctx* c, const kf_geometry* geom, int first_layer, int n_build_layers, int n_events,
                                  const int64_t* event_first, kf_tracks* cands, const kf_layer_hits* hits,
                                  const kf_layer_bins* bins, int window_half, float chi2_cut, int n_cand,
                                  int32_t* hit_index, int32_t* n_found, int64_t ld_out) {
    if (!c || !geom || !cands || !hits || !bins || !event_first) return KF_ERR_NULL;
    FitParams P;
    int rc = make_params(geom, &P, true);
    if (rc) return rc;
    if (n_build_layers < 0 || first_layer < 0 || first_layer + n_build_layers > geom->n_layers) return KF_ERR_SHAPE;
    if (n_cand < 1 || n_cand > 8) return KF_ERR_UNSUPPORTED;
    if (n_events < 1) return KF_ERR_SHAPE;
    if (n_events > kMaxBuildEvents) return KF_ERR_UNSUPPORTED;
    if ((rc = check_tracks(cands, true, true))) return rc;
    if (event_first[0] != 0 || event_first[n_events] != cands->n) return KF_ERR_SHAPE;
    for (int e = 0; e < n_events; ++e)
        if (event_first[e + 1] < event_first[e]) return KF_ERR_SHAPE;
    if (n_build_layers == 0 || cands->n == 0) return KF_OK;
    if (!hit_index) return KF_ERR_NULL;
    if (ld_out < cands->n) return KF_ERR_SHAPE;
    if (cands->n * (int64_t)n_cand > 0x7fffffffLL) return KF_ERR_UNSUPPORTED;
    ScoreStep steps[KF_MAX_LAYERS];
    for (int j = 0; j < n_build_layers; ++j) {
        for (int e = 0; e < n_events; ++e) {
            const kf_layer_hits* h = hits + (int64_t)e * n_build_layers + j;
            const kf_layer_bins* b = bins + (int64_t)e * n_build_layers + j;
            if ((rc = check_score_bins(h, b, window_half))) return rc;
            if (b->n_eta != bins[0].n_eta || b->n_phi != bins[0].n_phi || b->eta_max != bins[0].eta_max)
                return KF_ERR_UNSUPPORTED;
            steps[j].ev_hit_rec[e] = b->hit_rec;
            steps[j].ev_bin_box[e] = b->bin_box;
            steps[j].ev_bin_offset[e] = b->bin_offset;
        }
        steps[j].layer = first_layer + j;
        steps[j].n_hits = hits[j].n_hits;
        steps[j].hit_rec = bins[j].hit_rec;
        steps[j].bin_box = bins[j].bin_box;
        steps[j].bin_offset = bins[j].bin_offset;
        steps[j].best_hit = nullptr;
        steps[j].best_chi2 = nullptr;
    }
    CombCall call;
    call.n_seeds = cands->n; call.ld = cands->ld; call.par = cands->par; call.cov = cands->cov; call.q = cands->q;
    call.chi2 = cands->chi2; call.nhits = cands->nhits; call.status = cands->status;
    call.n_cand = n_cand;
    call.n_eta = bins[0].n_eta; call.n_phi = bins[0].n_phi; call.eta_max = bins[0].eta_max;
    call.window_half = window_half; call.chi2_cut = chi2_cut;
    call.hit_index = hit_index; call.ld_out = ld_out; call.n_found = n_found;
    call.ev.n = n_events;
    for (int e = 0; e <= n_events; ++e) call.ev.first[e] = event_first[e];
    KF_ON_DEVICE(c);
    cudaError_t e = launch_comb(c->comb, P, call, n_build_layers, steps, c->stream);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? KF_ERR_NOMEM : cuda_fail(c, e);
    return KF_OK;
}

int kf_score_candidates(kf_ctx* c, const kf_geometry* geom, int layer, kf_tracks* cands,
                        const kf_layer_hits* hits, const kf_layer_bins* bins, int window_half,
                        float chi2_cut, int do_update, const int32_t* order, int32_t* best_hit,
                        float* best_chi2, float* local_state) {
    if (!c || !geom || !cands) return KF_ERR_NULL;
    if (cands->n > 0 && (!best_hit || !best_chi2)) return KF_ERR_NULL;
    return build_best_hit(c, geom, layer, 1, cands, hits, bins, window_half, chi2_cut, do_update, order,
                          best_hit, best_chi2, cands->n > 0 ? cands->ld : 0, local_state);
}

static_assert(kStaticMaxCands == KF_STATIC_MAX_CANDIDATES, "kf_internal.h and kf_b200.h disagree on the static scratch size");

// The single-layer call on the static scratch of kf_score.cu: the argument checks of build_best_hit for one layer,
// then launch_score_static.  No allocation on any path; the context's scratch is neither read nor resized.
int kf_score_candidates_static(kf_ctx* c, const kf_geometry* geom, int layer, kf_tracks* cands,
                               const kf_layer_hits* hits, const kf_layer_bins* bins, int window_half,
                               float chi2_cut, int do_update, const int32_t* order, int32_t* best_hit,
                               float* best_chi2, float* local_state) {
    if (!c || !geom || !cands || !hits || !bins) return KF_ERR_NULL;
    FitParams P;
    int rc = make_params(geom, &P, true);
    if (rc) return rc;
    if (layer < 0 || layer >= geom->n_layers) return KF_ERR_SHAPE;
    if ((rc = check_tracks(cands, true, true))) return rc;
    if (cands->n > KF_STATIC_MAX_CANDIDATES) return KF_ERR_TOO_LARGE;
    if (cands->n == 0) return KF_OK;
    if (!best_hit || !best_chi2) return KF_ERR_NULL;
    if ((rc = check_score_bins(hits, bins, window_half))) return rc;
    if (local_state && !aligned16(local_state)) return KF_ERR_ALIGN;
    ScoreStep st;
    std::memset(&st, 0, sizeof(st));
    st.layer = layer;
    st.n_hits = hits->n_hits;
    st.hit_rec = bins->hit_rec; st.bin_box = bins->bin_box; st.bin_offset = bins->bin_offset;
    st.best_hit = best_hit; st.best_chi2 = best_chi2;
    ScoreArgs a;
    std::memset(&a, 0, sizeof(a));
    a.n = cands->n; a.ld = cands->ld; a.par = cands->par; a.cov = cands->cov; a.q = cands->q;
    a.chi2 = cands->chi2; a.nhits = cands->nhits; a.status = cands->status;
    a.order = order;
    a.n_eta = bins->n_eta; a.n_phi = bins->n_phi; a.eta_max = bins->eta_max;
    a.window_half = window_half; a.chi2_cut = chi2_cut; a.do_update = do_update ? 1 : 0;
    a.lstate = local_state; a.ld_ls = cands->ld;
    KF_ON_DEVICE(c);
    const cudaError_t e = launch_score_static(P, a, st, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return KF_OK;
}

}  // extern "C"
