// kf_internal.h -- declarations shared by the translation units of libkf_b200 (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "kf_math.cuh"

namespace kf {

// Per-context launch options (kf_set_option): read at kf_create / set by the caller, never from the
// environment on the launch path.
struct LaunchOptions {
    int64_t pair_min_tracks = 0;   // 0: the built-in rule (tracks x layers); > 0: batches of at least this many tracks take the pair kernels
    int refit_pair_masked = 0;     // 1: the pair form of the refit also for batches with a hit mask (tests)
    int bin_form = 0;              // 0: by size; 1: always the five-launch sort; 2: the chunked sort wherever it applies
};

// One-time per-device kernel attributes (dynamic shared memory above 48 KB is a per-device function attribute).
cudaError_t ensure_fit_attributes();
cudaError_t ensure_bin_attributes();

// ---------------------------------------------------------------------------------- fit
struct FitArgs {
    int64_t n;
    // inputs
    const float* par; const float* cov; int64_t ld_in;
    const int8_t* q;
    const float* hpos; const float* hcov; int64_t ld_hit;
    const uint32_t* mask;  // may be null
    // outputs
    float* opar; float* ocov; int64_t ld_out;
    float* chi2; int32_t* nhits; uint32_t* status;
    // smoother outputs (spar == nullptr: forward fit only)
    float* spar = nullptr; float* scov = nullptr; int64_t ld_s = 0;
    float* schi2 = nullptr; int32_t* snhits = nullptr; uint32_t* sstatus = nullptr;
    float kappa = 10.0f;
    // kf_fit_tracks_smooth (RTS): per-layer arrays [L][6][ld_l] / [L][21][ld_l] and the used-layer mask
    // (lpar == nullptr: not wanted).  The forward kernel leaves the filtered local-frame state of every used layer
    // there; the backward kernel (kf_smooth.cu) turns it into the smoothed state in global coordinates.
    float* lpar = nullptr; float* lcov = nullptr; int64_t ld_l = 0; uint32_t* used = nullptr;
};

struct IndexedPools {           // per-layer hit pools + the per-track hit indices into them
    const float* pos[32];
    const float* cov[32];
    int64_t ld[32];
    const int32_t* index;       // [n_layers][ld_index], -1 = no hit
    int64_t ld_index;
    // optional fast path: the packed bin-ordered records of kf_bin_layers and the map into them
    const float* hit_rec[32];
    const int32_t* orig_to_sorted[32];
    int use_records;            // 0: SoA pools; 1: bin-ordered records through orig_to_sorted; 2: records in ORIGINAL order
};

// kf_fit_tracks_indexed without bins: the SoA pools are packed once into 48-byte records in original order (context
// scratch), so that the gather costs 2 memory sectors per hit instead of 9.
struct PackPools {
    const float* pos[32];
    const float* cov[32];
    int64_t ld[32];
    int64_t n[32];
    float* rec[32];
};
struct IndexScratch {
    uint64_t gen = 0;
    size_t cap = 0;
    float* rec = nullptr;
    cudaError_t reserve(size_t bytes, cudaStream_t stream);
    void release();
};
cudaError_t launch_pack_pools(const PackPools& A, int n_layers, cudaStream_t stream);

// kf_fit.cu
cudaError_t launch_fit_indexed(const FitParams& P, const IndexedPools& H, const FitArgs& a, cudaStream_t stream);
cudaError_t launch_fit(const FitParams& P, const FitArgs& a, cudaStream_t stream, const LaunchOptions& opt = LaunchOptions());
// The size rule of launch_fit: does a batch of n tracks x n_layers take the two-tracks-per-thread kernels?
// (kf_fit_tracks_host decides it on the WHOLE batch and launches every chunk accordingly, so that the host path gives,
// bit for bit, what kf_fit_tracks gives on the same tracks.)
bool fit_takes_pair_form(int64_t n, int n_layers, const LaunchOptions& opt);

// kf_smooth.cu: backward RTS pass over the per-layer arrays the forward kernel filled
cudaError_t launch_rts(const FitParams& P, const FitArgs& a, cudaStream_t stream);

// ---------------------------------------------------------------------------------- host path
struct HostFitIO {
    int64_t n; int L;
    const float* par; const float* cov; int64_t ld_in; const int8_t* q;
    const float* hpos; const float* hcov; int64_t ld_hit; const uint32_t* mask;
    float* opar; float* ocov; int64_t ld_out; float* chi2; int32_t* nhits; uint32_t* status;
    bool cov_diagonal = false;   // kf_fit_tracks_host_diag: cov is [6][ld_in], the diagonal of the seed covariance
    bool hit_cov_local = false;  // kf_fit_tracks_host_compact: hcov is [L][3][ld_hit], the variances along r^ t^ z^ of the hit
};

// Device staging for kf_fit_tracks_host: kSlots chunk buffers, each with its own stream, so the
// H2D copy of chunk c+1, the kernel of chunk c and the D2H copy of chunk c-1 overlap.
struct HostStage {
    static constexpr int kSlots = 3;
    int64_t chunk = 0;  // tracks per chunk (multiple of 4)
    int layers = 0;
    cudaStream_t stream[kSlots] = {nullptr, nullptr, nullptr};
    cudaStream_t out_stream = nullptr;                          // every device-to-host copy
    cudaEvent_t fitted[kSlots] = {nullptr, nullptr, nullptr};   // chunk's kernel done (out_stream waits for it)
    cudaEvent_t drained[kSlots] = {nullptr, nullptr, nullptr};  // chunk's results are in host memory (the slot's next kernel waits)
    char* buf[kSlots] = {nullptr, nullptr, nullptr};
    size_t buf_bytes = 0;
    cudaError_t reserve(int64_t max_tracks, int max_layers);
    cudaError_t fit(const FitParams& P, const HostFitIO& io, const LaunchOptions& opt);
    void release();
};

// ---------------------------------------------------------------------------------- binning
constexpr int KF_MAX_BINS_INTERNAL = 65536;
constexpr int kLutCells = 256;
constexpr int kBinBatchMax = 32;  // layers per group of launches (the descriptors travel as one 4.4 KB kernel parameter)

struct BinArgs {
    int64_t n_hits, ld_in;
    const float* pos; const float* cov;
    float radius; int n_eta, n_phi; float eta_max;
    int64_t ld_out;
    int32_t* bin_offset; int32_t* sorted_to_orig;
    float* pos_sorted; float* cov_sorted;  // optional SoA copies (may be null)
    float* hit_rec;                        // [n_hits][12] packed records (may be null)
    float* bin_box;                        // [n_bins][8] per-bin bounds (may be null)
    int32_t* orig_to_sorted;               // [n_hits] inverse of sorted_to_orig (may be null)
};

// One layer (or one candidate set) as the batched sort kernels see it.
struct BinLayerDev {
    int64_t n, ld_in, ld_out;
    const float* pos; const float* cov;    // null: order items only, gather nothing
    float radius;
    int32_t* bin_offset; int32_t* sorted_to_orig;
    float* pos_sorted; float* cov_sorted; float* hit_rec; float* bin_box; int32_t* orig_to_sorted;
    int32_t* key;       // [n] bin of each item
    int32_t* unsorted;  // [n] item indices grouped by bin, arbitrary order inside
    int32_t* counts;    // [n_bins + 1]
    int32_t* pib;       // [n] arrival number of each item inside its bin (value returned by the histogram atomic)
    float* rec_tmp;     // [n][12] hit records grouped by bin in arrival order (null when nothing is gathered)
    int32_t* chunk_cnt; // [chunks][n_bins] chunked sort: hits of a bin per chunk, then their prefix over chunks
};

struct BinBatch {
    int n_layers, n_eta, n_phi;
    BinLayerDev layer[kBinBatchMax];
};

struct BinScratch {
    uint64_t gen = 0;            // bumped whenever a buffer is reallocated or the edge tables are rewritten (kf_graph staleness)
    int64_t cap_items = 0, cap_bins = 0;
    int32_t* key = nullptr;
    int32_t* unsorted = nullptr;
    int32_t* counts = nullptr;
    int32_t* pib = nullptr;
    float* rec_tmp = nullptr;    // [cap_items][12], allocated on the first call that gathers hits
    int64_t cap_rec = 0;
    int32_t* chunk_cnt = nullptr; // chunked sort: [layers][n_bins][chunks] counters
    int64_t cap_chunk_cnt = 0;
    cudaError_t reserve_chunk_cnt(int64_t words, cudaStream_t stream);
    // edge tables (device) for the (n_eta, n_phi, eta_max) last used
    float* eta_edge = nullptr;   // fl32(sinh(-eta_max + j d_eta)), j = 1..n_eta-1 at [j]
    float* phi_cos = nullptr;    // fl32(cos(-pi + j d_phi))
    float* phi_sin = nullptr;
    int tab_n_eta = 0, tab_n_phi = 0;
    float tab_eta_max = 0.0f;
    std::vector<float> host_tab; // persistent host copy of the three tables (source of the async copy)
    // first guesses for the edge searches of chunk_count_kernel: [3][kLutCells] = eta, phi lower / upper half plane
    int32_t* guess_lut = nullptr;
    std::vector<int32_t> host_lut;
    float lut_u0 = 0.0f, lut_uscale = 0.0f;   // eta cell of u = z / r: floor((u - u0) * uscale)
    cudaError_t reserve(int64_t n_items, int64_t n_bins, cudaStream_t stream, bool records = false);
    cudaError_t tables(int n_eta, int n_phi, float eta_max, cudaStream_t stream);
    void release();
};

// kf_bin.cu
cudaError_t launch_bin(BinScratch& s, int n_layers, const BinArgs* args, cudaStream_t stream, const LaunchOptions& opt = LaunchOptions());
cudaError_t reserve_chunked(BinScratch& s, int64_t max_hits, int max_layers, cudaStream_t stream);
cudaError_t launch_order(BinScratch& s, const FitParams& P, int layer, int64_t n, int64_t ld, const float* par,
                         const int8_t* q, int n_eta, int n_phi, float eta_max, int32_t* order,
                         cudaStream_t stream);

// ---------------------------------------------------------------------------------- bounds checks of a debug build
// compute-sanitizer is not available on the pool this was developed on; `-DKF_DEBUG_BOUNDS` (python -m
// paper_1705_02876_b200.build -DKF_DEBUG_BOUNDS --out=...) turns the index computations that SCATTER or GATHER
// (final slots of the counting sort, hit records read by the scans, peer and overflow lists, the static scratch)
// into traps when they leave their arrays; the GPU test suite is run against that build before a release.
#ifdef KF_DEBUG_BOUNDS
#define KF_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define KF_CHECK(cond) do { } while (0)
#endif

// ---------------------------------------------------------------------------------- dependent launches
// The building and binning calls are chains of 4 - 30 short kernels, each reading what the one before wrote; at
// event size a kernel boundary (drain, launch, ramp) costs 2 - 3 us of a 5 - 15 us kernel.  With programmatic
// dependent launch the next kernel of the chain is scheduled while the current one is still running: every kernel
// of a chain starts with pdl_start() -- `launch_dependents` lets the NEXT grid's CTAs take free slots as soon as all
// CTAs of this grid have started, `wait` holds this grid until the PREVIOUS grid has completed and its writes are
// visible -- and is launched with launch_chained().  Nothing is read or written before pdl_start(), so the order
// of all memory effects is that of plain stream order.  A kernel launched the plain way runs both instructions as
// no-ops.  Recorded in a graph (kf_graph_begin) the launches become programmatic edges.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_start() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}
#endif

template <class... KArgs, class... Args>
inline cudaError_t launch_chained(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                                  Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ---------------------------------------------------------------------------------- scoring
constexpr int kScorePlanes = 29;

// Packed hit record of kf_bin_hits (kf_layer_bins.hit_rec): kRecWords 16-byte words per hit,
//   x y z vzz | vxx vxy vyy index | vxz vyz 0 0 [ | 0 0 0 0 ].
// Three words = 48 bytes is what the library ships.  Four words (a 64-byte record = two whole, aligned sectors,
// written once by four lanes, the pre-filters' two words in its first sector) is a build option
// (-DKF_REC_WORDS=4) kept for measurements: on configs[4] (everything L2-resident) it LOST everywhere -- binning
// 49.8 -> 58.8 us, best-hit building 177 -> 203 us, combinatorial 824 -> 899 us (a third more bytes through L2 per
// hit scanned) -- and only won once the pools no longer fit in L2 (binning 28 x 120 000 hits: 241 -> 212 us).
#ifndef KF_REC_WORDS
#define KF_REC_WORDS 3
#endif
constexpr int kRecWords = KF_REC_WORDS;
constexpr int kRecFloats = 4 * kRecWords;

struct BinGrid { int n_eta, n_phi; float eta_max; };

constexpr int kMaxBuildEvents = 32;

// Several events in one building call ("concurrent events should be adapted to track building because
// this will help to fill the GPU"): candidates of event e are first[e] .. first[e + 1] - 1 of the one candidate
// array; every event has its own hit pools and bins.  n <= 1: the single-event pointers of ScoreArgs are used.
struct EventPools {
    int n;
    int64_t first[kMaxBuildEvents + 1];
    const float* hit_rec[kMaxBuildEvents];
    const float* bin_box[kMaxBuildEvents];
    const int32_t* bin_offset[kMaxBuildEvents];
};

struct ScoreArgs {
    int64_t n, ld;
    float* par; float* cov; const int8_t* q; float* chi2; int32_t* nhits; uint32_t* status;
    // current step
    int64_t n_hits;
    const float* hit_rec;
    const float* bin_box;
    const int32_t* bin_offset;
    int32_t* best_hit; float* best_chi2;
    // common
    const int32_t* order;  // may be null
    int n_eta, n_phi; float eta_max;
    int window_half; float chi2_cut; int do_update;
    // context scratch (filled by launch_build)
    float* scratch; float* track; int32_t* flag; int32_t* slot; int64_t ld_sc;
    // kf_score_candidates: the caller's local-frame candidate state [30][ld_ls] (null: none)
    float* lstate; int64_t ld_ls;
    EventPools ev;           // kf_build_best_hit_events (ev.n > 1), set per step
};

struct ScoreStep {
    int layer;               // geometry layer
    int64_t n_hits;
    const float* hit_rec;
    const float* bin_box;
    const int32_t* bin_offset;
    int32_t* best_hit;       // [n]
    float* best_chi2;        // [n]
    // several events (n_events > 1): per-event pools of this step, in the order of EventPools::first
    const float* ev_hit_rec[kMaxBuildEvents];
    const float* ev_bin_box[kMaxBuildEvents];
    const int32_t* ev_bin_offset[kMaxBuildEvents];
};

struct ScoreScratch {
    uint64_t gen = 0;
    int64_t cap = 0, ld = 0;
    float* scratch = nullptr;  // [kScorePlanes][ld] propagated candidate (scan + update inputs)
    float* track = nullptr;    // [29][ld] local-frame track between layers
    int32_t* flag = nullptr;   // [ld]
    int32_t* slot = nullptr;   // [ld] winning sorted slot or -1
    cudaError_t reserve(int64_t n, cudaStream_t stream);
    void release();
};

// kf_score.cu
cudaError_t launch_build(ScoreScratch& s, const FitParams& P, ScoreArgs a, int n_steps, const ScoreStep* steps,
                         cudaStream_t stream);

// kf_score_candidates_static: one layer with the per-candidate scratch in a `static __device__` array of kf_score.cu
// (no allocation of any kind).  n <= kStaticMaxCands is the caller's check; cudaErrorInvalidValue beyond it.
constexpr int64_t kStaticMaxCands = 65536;            // = KF_STATIC_MAX_CANDIDATES (checked in kf_api.cu)
constexpr int kStaticPlanes = kScorePlanes + 2;       // propagated candidate + flag + slot
cudaError_t launch_score_static(const FitParams& P, ScoreArgs a, const ScoreStep& step, cudaStream_t stream);

// ---------------------------------------------------------------------------------- combinatorial building
struct CombCall {
    int64_t n_seeds, ld;
    float* par; float* cov; const int8_t* q; float* chi2; int32_t* nhits; uint32_t* status;
    int n_cand;
    int n_eta, n_phi; float eta_max; int window_half; float chi2_cut;
    int32_t* hit_index; int64_t ld_out; int32_t* n_found;
    EventPools ev = {};      // kf_build_combinatorial_events: ev.n > 1, ev.first in SEED indices; pools per step in ScoreStep::ev_*
};

struct CombScratch {
    uint64_t gen = 0;
    int64_t cap_words = 0;
    void* buf = nullptr;
    cudaError_t reserve(int64_t words, cudaStream_t stream);
    void release();
};

// kf_comb.cu
cudaError_t launch_comb(CombScratch& s, const FitParams& P, const CombCall& call, int n_steps, const ScoreStep* steps,
                        cudaStream_t stream);

// ---------------------------------------------------------------------------------- host path of building
// kf_build_best_hit_host: one event with every buffer in host memory.  Layer j's pool is copied on a second stream
// while layer j - 1 is binned and scored (transfers are about half of the building wall time when they
// are not overlapped).
struct BuildHostIO {
    int64_t n, ld;                         // candidates (HOST SoA, in/out)
    float* par; float* cov; const int8_t* q; float* chi2; int32_t* nhits; uint32_t* status;
    int first_layer, n_layers;
    const int64_t* n_hits; const int64_t* ld_hits;             // [n_layers]
    const float* const* pos; const float* const* cov_hits;     // [n_layers] HOST [3][ld], [6][ld]
    int n_eta, n_phi; float eta_max; int window_half; float chi2_cut; int do_update;
    int32_t* hit_index; float* hit_chi2; int64_t ld_out;       // HOST [n_layers][ld_out]
};

struct BuildHostStage {
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ready[32] = {};            // layer j's pool is on the device
    cudaEvent_t done = nullptr;            // compute finished with the staging buffers of the previous call
    char* buf = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t bytes);
    void release();
};

cudaError_t build_best_hit_host(BuildHostStage& hs, BinScratch& bs, ScoreScratch& ss, const FitParams& P, const BuildHostIO& io,
                                cudaStream_t stream, const LaunchOptions& opt);

// kf_peak.cu
double measure_fp32_peak(cudaStream_t stream, int repeats, float* sink);
cudaError_t measure_fp32_packed_rate(cudaStream_t stream, int repeats, float* scratch, double* shared_tflops,
                                     double* distinct_tflops);

}  // namespace kf
