/*
 * kf_b200.h -- C ABI of the B200-native batched Kalman-filter track fitter.
 *
 * What it computes (arXiv:1705.02876):
 *   - track fitting = the Kalman filter applied layer after layer, without branching, to the fixed
 *     hit list of each track, giving the parameters and a chi2 (section 2 "a final
 *     fit with a KF ... to compute a measure of the track quality in terms of a chi2";
 *     PAPER.md:61 "track fitting can repeatedly apply the KF algorithm without branching");
 *   - track state = 6 parameters in global coordinates with a 6x6 covariance, hit = 3-D point
 *     with a 3x3 covariance (section 2.1);
 *   - many small matrices stored matrix-major: "elements with the same index but from different
 *     matrices are stored consecutively" (PAPER.md:65 Matriplex; section 4.1) --
 *     here: structure of arrays, element-major across tracks, plane stride `ld`;
 *   - hits of a layer placed in "directionally projective bins" (eta, phi) for fast look-up
 *     (section 3);
 *   - best-hit building: per candidate and layer "the hit that produced the lowest chi2 increment"
 *     (section 3), one GPU thread group per candidate (section 4.3).
 * The paper prints no formulas.  The equations are BASELINE.json:north_star's
 *     C' = F C F^T + Q,  S = H C' H^T + V,  K = C' H^T S^-1,  x = x' + K r,  C = C' - K H C',
 *     chi2 += r^T S^-1 r,      H = [I3 0],  r = m - H x'
 * with the helix, Jacobian, Highland process noise and bin definitions written out in DESIGN.md
 * ("Readings A1..A17").
 *
 * Units: cm, GeV/c, Tesla.  State order (x, y, z, px, py, pz).  Symmetric 6x6 packed as the upper
 * triangle, row-major, 21 values: index(i<=j) = i*6 - i*(i-1)/2 + (j-i).  Symmetric 3x3 packed
 * xx, xy, xz, yy, yz, zz.  Every array is element-major: element e of track t is at
 * base[e*ld + t].
 *
 * Conventions for every call
 *   Ownership: all buffers are caller-owned; the library keeps no pointer after a call returns.
 *              The context owns only its scratch (kf_reserve / grown on demand by kf_bin_hits and
 *              the *_host calls; growing synchronises the stream, steady state never allocates).
 *   Memory:    "DEV" = device pointer on the context's device, "HOST" = host pointer.  Device
 *              pointers must be 16-byte aligned and ld % 4 == 0 (so every plane is 16-byte aligned).
 *   Async:     device-pointer calls enqueue on the context's stream and return without
 *              synchronising.  *_host calls return after the results are in the host buffers.
 *   Errors:    0 = KF_OK; negative = argument or launch error, and then no output is written.
 *              No exception crosses this boundary.  Per-track trouble is data, not an error: it is
 *              reported in `status` bits and the track keeps its last good state.
 *   No CPU fallback exists: without a CUDA device kf_create fails with KF_ERR_CUDA.
 */
#ifndef KF_B200_H
#define KF_B200_H

#include <stdint.h>

#if defined(__GNUC__)
#define KF_API __attribute__((visibility("default")))
#else
#define KF_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

/* ---- return codes -------------------------------------------------------------------------- */
enum {
    KF_OK = 0,
    KF_ERR_NULL = -1,        /* a required pointer is NULL                                        */
    KF_ERR_SHAPE = -2,       /* n < 0, ld < n, n_layers mismatch, layer index out of range ...    */
    KF_ERR_ALIGN = -3,       /* device pointer not 16-byte aligned or ld % 4 != 0                 */
    KF_ERR_UNSUPPORTED = -4, /* n_layers > 32, |Bz| < 1e-6 T, radii not strictly increasing,
                                bins > KF_MAX_BINS, window wider than the phi ring                */
    KF_ERR_CUDA = -5,        /* a CUDA runtime call failed (kf_last_cuda_error has the code)      */
    KF_ERR_NOMEM = -6,       /* scratch allocation failed                                         */
    KF_ERR_STALE = -7,       /* kf_graph_launch: the graph's context is gone, or has reallocated scratch or
                                changed the bin grid since the recording (record it again)          */
    KF_ERR_TOO_LARGE = -8    /* kf_score_candidates_static: more than KF_STATIC_MAX_CANDIDATES candidates */
};

/* ---- per-track status bits (outputs) ---------------------------------------------------------- */
enum {
    KF_STATUS_PROP_FAIL = 1,  /* helix has no outward crossing with the layer (disc <= 0, r <= rho) */
    KF_STATUS_S_NOT_PD = 2,   /* det S <= 0                                                         */
    KF_STATUS_NONFINITE = 4,  /* update produced a non-finite state or chi2                         */
    KF_STATUS_BAD_CHARGE = 8, /* q not in {+1, -1}: track is copied through untouched               */
    KF_STATUS_OUTSIDE = 16,   /* a crossing fell beyond the end of the barrel (|z'| > half_length_cm):
                                 that layer was skipped (reading A20)                      */
    KF_STATUS_SMOOTH_FAIL = 32 /* kf_fit_tracks_smooth only: a backward step could not be taken (predicted
                                 covariance not positive definite / non-finite); that layer and the layers
                                 further in carry the FILTERED state                                  */
};

#define KF_MAX_LAYERS 32
#define KF_MAX_BINS 65536

typedef struct kf_ctx kf_ctx; /* opaque: device, borrowed stream, scratch */

/* Create a context on `device`.  `cuda_stream` is a borrowed cudaStream_t (e.g. the raw handle of a
 * torch stream); NULL = the legacy default stream.  Fails with KF_ERR_CUDA if there is no device. */
KF_API int kf_create(kf_ctx** out, int device, void* cuda_stream);
KF_API int kf_destroy(kf_ctx* ctx);
/* Change the borrowed stream used by later calls. */
KF_API int kf_set_stream(kf_ctx* ctx, void* cuda_stream);
/* Every call makes the context's device current for its own duration and restores the caller's current device
 * before it returns, so contexts on several devices can be driven from one thread. */

/* Launch options of a context (kernel selection only: no option changes a result beyond fp32 rounding).  They
 * exist for tests and measurements; the defaults are the measured best. */
enum {
    KF_OPT_PAIR_MIN_TRACKS = 1,   /* > 0: batches of at least this many tracks take the two-tracks-per-thread
                                     kernels; 0 (default) = the built-in size rule                          */
    KF_OPT_REFIT_PAIR_MASKED = 2, /* 1: kf_fit_tracks_refit takes its two-tracks-per-thread form for batches WITH
                                     a hit mask too (default 0: only without a mask)                        */
    KF_OPT_BIN_FORM = 3           /* kf_bin_layers: 0 (default) = by size, 1 = always the five-launch counting
                                     sort, 2 = the chunked sort wherever it applies                         */
};
KF_API int kf_set_option(kf_ctx* ctx, int option, int64_t value);
/* Pre-size scratch so that no later call allocates: `max_hits` hits in total over the layers of one kf_bin_layers call
 * (or over the pools of one kf_fit_tracks_indexed call without bins, which packs them into 48-byte records),
 * `max_host_tracks` x `max_host_layers` for the *_host staging buffers (0 = leave as is). */
KF_API int kf_reserve(kf_ctx* ctx, int64_t max_hits, int64_t max_host_tracks, int max_host_layers);
/* Static, never NULL. */
KF_API const char* kf_strerror(int code);
/* cudaError_t of the last KF_ERR_CUDA on this context (0 if none). */
KF_API int kf_last_cuda_error(const kf_ctx* ctx);
/* ---- graphs: record a fixed sequence of hot calls once, replay it with one launch ---------------------------
 * Event-sized work (10 000 - 20 000 tracks per event) is bound by kernel-launch and host-call
 * overhead, not by the device: one kf_bin_layers + kf_build_best_hit over 7 layers is 20 launches of 5 - 25 us.
 * Between kf_graph_begin and kf_graph_end every device-pointer hot call on this context (kf_fit_tracks[_indexed /
 * _smooth], kf_bin_hits / kf_bin_layers, kf_order_candidates, kf_score_candidates, kf_build_best_hit,
 * kf_build_combinatorial) is RECORDED into a CUDA graph instead of executed; kf_graph_launch then enqueues the
 * whole sequence on the context's stream with the pointers, sizes and geometry it was recorded with (the caller
 * refills the same buffers between launches).  Requirements: a non-NULL stream; scratch already sized, i.e. the
 * same sequence has run once before (or kf_reserve), because a call that has to grow scratch synchronises and
 * voids the capture (kf_graph_end then returns KF_ERR_CUDA and no graph).  kf_fit_tracks_host, kf_reserve,
 * kf_measure_fp32_peak and kf_set_stream must not be called while recording.  Results are bit-identical to
 * the eager calls.  A graph belongs to the context that recorded it: the recorded kernels point into that
 * context's scratch and bin edge tables, so kf_graph_launch refuses it with KF_ERR_STALE once the context has
 * reallocated scratch (a later call needed more) or binned with another (n_eta, n_phi, eta_max) grid, and
 * with KF_ERR_STALE as well when handed another context.  Never launch a graph whose context has been destroyed
 * unless through a live context (which is then refused the same way).  Destroy it with kf_graph_destroy. */
typedef struct kf_graph kf_graph;
KF_API int kf_graph_begin(kf_ctx* ctx);
KF_API int kf_graph_end(kf_ctx* ctx, kf_graph** out);
KF_API int kf_graph_launch(kf_ctx* ctx, kf_graph* graph);
KF_API int kf_graph_destroy(kf_graph* graph);
/* Measurement utility (not on the hot path): sustained FP32 FMA throughput of the device in TFLOP/s
 * from a register-only FMA microbenchmark (8 independent chains per thread, 2048 threads per SM, best
 * of `repeats` launches).  Synchronises the stream.  This is the denominator of the ALU roofline. */
KF_API int kf_measure_fp32_peak(kf_ctx* ctx, int repeats, double* tflops_out);
/* The same for the packed instruction the two-tracks-per-thread kernels are made of (FFMA2, one fp32x2 FMA per lane:
 * 4 flop): `shared_tflops` with two of the three operands shared by every chain (the FMA pipe's own rate),
 * `distinct_tflops` with three distinct register pairs per instruction, which is what arithmetic on per-track
 * matrices issues and what the register file can feed (about 2/3 of the former on B200).  Synchronises the stream;
 * not to be called while recording a graph. */
KF_API int kf_measure_fp32_packed_rate(kf_ctx* ctx, int repeats, double* shared_tflops, double* distinct_tflops);
/* ABI version, bumped when a struct or signature changes. */
KF_API int kf_abi_version(void);
/* Floats per packed hit record of kf_layer_bins.hit_rec as this build writes it (= KF_HIT_RECORD_FLOATS). */
#define KF_HIT_RECORD_FLOATS 12
KF_API int kf_hit_record_floats(void);

/* ---- geometry: concentric cylinders in a uniform solenoid field (PAPER.md:83 toy detector) ---- */
typedef struct {
    int n_layers;             /* 1..KF_MAX_LAYERS                                                  */
    const float* radius_cm;   /* HOST [n_layers], strictly increasing, > 0                         */
    const float* x_over_X0;   /* HOST [n_layers], thickness in radiation lengths, 0 = no material  */
    float Bz_tesla;           /* |Bz| >= 1e-6                                                      */
    float mass_gev;           /* mass entering beta of the Highland formula (reading A5)           */
    /* Geometry options ("more realistic" geometry is the stated direction; DESIGN.md
     * reading A20).  Zero-initialised = the toy detector of the paper: infinite barrels, flat material. */
    const float* half_length_cm; /* HOST [n_layers] barrel half lengths (> 0, +inf allowed), or NULL =
                                    unbounded.  A propagated crossing with |z'| > half length misses the
                                    layer: it is skipped and KF_STATUS_OUTSIDE is set.               */
    int material_model;       /* 0: thickness x_over_X0 as given.  1: path length through the layer,
                                 x_over_X0 / cos(psi), psi = angle between the propagated momentum and
                                 the cylinder normal at the crossing (in Highland's sqrt AND log term) */
    int energy_loss_model;    /* DESIGN.md reading A21.  0: none.  1: at every layer crossing the track loses
                                 the mean Bethe energy loss of a unit-charge particle of mass_gev in
                                 x_over_X0 radiation lengths of SILICON (Z/A = 14/28.0855, I = 173 eV,
                                 X0 = 21.82 g/cm^2; no density correction, no straggling), over the path
                                 length if material_model = 1; the momentum keeps its direction, the
                                 covariance is transported with dE held fixed; the backward refit gives
                                 the energy back.  A track that would stop fails that layer
                                 (KF_STATUS_PROP_FAIL).  Needs mass_gev > 0.                            */
    /* Endcap discs ("a more realistic geometry"; reading A23).  NULL surface_type = every
     * layer is a barrel.  A layer with surface_type[l] = 1 is a PAIR of discs in the planes z = +-disc_z_cm[l],
     * sensitive for disc_rmin_cm[l] <= rho <= disc_rmax_cm[l]; a track meets the disc on the side it is heading to
     * (sign of pz).  Layers are met in list order (barrels that end inside the first disc, then the discs by |z|).
     * The state is propagated to the plane (theta = k (zt - z) / pz); the transported covariance then has no
     * variance along z instead of along the radius; a crossing outside the annulus sets KF_STATUS_OUTSIDE and the
     * layer is skipped; a plane that lies behind the state or half a turn or more away is KF_STATUS_PROP_FAIL.
     * radius_cm[l] of a disc layer is not used but must keep the list increasing.  Discs are known to every call
     * (the pool of a disc layer is binned with radius 0: kf_bin_hits).  material_model and energy_loss_model apply
     * at a disc with the path factor 1 / |cos| of the angle to the z axis = |p| / |pz|. */
    const int32_t* surface_type;  /* HOST [n_layers] 0 = barrel, 1 = disc pair; or NULL                        */
    const float* disc_z_cm;       /* HOST [n_layers] |z| of the disc pair (> 0), read where surface_type = 1   */
    const float* disc_rmin_cm;    /* HOST [n_layers] inner radius of the annulus (>= 0)                         */
    const float* disc_rmax_cm;    /* HOST [n_layers] outer radius (> inner)                                     */
} kf_geometry;

/* ---- tracks (seeds in, fitted tracks out; candidates in/out) ------------------------------------ */
typedef struct {
    int64_t n, ld;            /* n tracks; plane stride ld >= n, ld % 4 == 0                        */
    float* par;               /* [6][ld]  x y z px py pz                                           */
    float* cov;               /* [21][ld] packed upper triangle                                    */
    int8_t* q;                /* [n] charge +1 / -1                                                */
    float* chi2;              /* [n]   fit: output total; scoring: in/out running total            */
    int32_t* nhits;           /* [n]   fit: output hits used; scoring: in/out                      */
    uint32_t* status;         /* [n]   fit: output; scoring: in/out (bits are OR-ed in)            */
} kf_tracks;

/* ---- per-track hit lists for fitting (the hit collection is fixed after building) -- */
typedef struct {
    int n_layers;             /* must equal geometry n_layers                                      */
    int64_t n, ld;
    const float* pos;         /* [n_layers][3][ld] hit of track t on layer l: x y z                */
    const float* cov;         /* [n_layers][6][ld] its covariance xx xy xz yy yz zz                */
    const uint32_t* mask;     /* [n] bit l set = track has a hit on layer l; NULL = all layers     */
} kf_track_hits;

/* Fit n tracks: for each layer in increasing radius whose mask bit is set, propagate state and
 * covariance along the helix to the layer radius (C' = F C F^T + Q), then Kalman-update with the
 * track's hit on that layer and add the chi2 increment (north_star).
 * A layer that fails (status bit) is skipped and the track keeps its previous state.
 * `out` may alias `seeds` (in-place); otherwise out->par/cov/chi2/nhits/status are written and
 * out->q is ignored.  out->n/ld may differ from seeds->ld but out->n must equal seeds->n.
 * All pointers DEV.  Enqueues one kernel on the context stream. */
KF_API int kf_fit_tracks(kf_ctx* ctx, const kf_geometry* geom, const kf_tracks* seeds,
                  const kf_track_hits* hits, kf_tracks* out);

/* Fit and REFIT inward (reading A18; kept from round 1 -- it is NOT the smoother of PAPER.md:57,
 * see kf_fit_tracks_smooth below): the forward fit of kf_fit_tracks, then the same filter run INWARD over the
 * same hits, starting from the forward result with its covariance inflated by `kappa` (10 is the documented
 * choice): update with the outermost used hit, then for each further used layer, outer to inner, add the process
 * noise of the layer just left, propagate backward along the helix to the smaller radius, update.  The forward
 * information is therefore counted 1 + 1/kappa times: the refitted covariance is too small by about that factor
 * and its chi2 is not chi2-distributed exactly.  What it is good for: a state at the INNERMOST used layer that
 * was linearised a second time around a better trajectory, at the cost of one more pass over the hits and no
 * per-layer storage.  `out` receives the forward result exactly as kf_fit_tracks writes it (state at the
 * outermost used layer); `refitted` receives the state and covariance at the innermost used layer (outer side
 * of its material), chi2 = chi2 of the backward pass, nhits = hits it used, status = its failure bits.  A track
 * the forward fit could not start comes back as its input in both.  All pointers DEV; `out` may alias `seeds`,
 * `refitted` may not alias either.  One kernel.  Performance note: hits->mask == NULL states that every track has
 * a hit on every layer; large batches then run two tracks per thread (7 % faster).  With a mask the one-track
 * kernel runs, whose speed does not depend on how ragged the tracks are.  Results agree within the tolerances. */
KF_API int kf_fit_tracks_refit(kf_ctx* ctx, const kf_geometry* geom, const kf_tracks* seeds,
                               const kf_track_hits* hits, float kappa, kf_tracks* out, kf_tracks* refitted);

/* ---- fit + smoother (section 2: "a final fit with a KF and smoother"; reading A22) -------
 * The forward fit of kf_fit_tracks followed by the fixed-interval (Rauch-Tung-Striebel) smoother over the layers
 * the fit used, k_0 < ... < k_{m-1}: x^s = x^+ at the outermost one, then, outer to inner,
 *     A = C^+_k G^T (C^-_n)^+,   x^s_k = x^+_k + A (x^s_n - x^-_n),   C^s_k = C^+_k + A (C^s_n - C^-_n) A^T
 * with x^+_k, C^+_k the filtered state of layer k, x^-_n, C^-_n the filter's prediction for the next used layer n
 * and G the Jacobian between them: at EVERY used layer the estimate, from ALL hits of the track, of the state just
 * after that layer's scatter.  It equals the weighted least squares of the linearised track model evaluated at
 * that layer (the oracle's pin SM1).  Layout: layer-major, element-major inside a layer. */
typedef struct {
    int n_layers;             /* must equal geometry n_layers                                      */
    int64_t n, ld;            /* n tracks; plane stride ld >= n, ld % 4 == 0                       */
    float* par;               /* DEV [n_layers][6][ld]  smoothed x y z px py pz at layer l          */
    float* cov;               /* DEV [n_layers][21][ld] its covariance, packed upper triangle       */
    uint32_t* used;           /* DEV [n] bit l set = layer l was used by the fit and has a smoothed
                                 state; the slots of other layers are not written                   */
} kf_smoothed;

/* `out` receives the forward result exactly as kf_fit_tracks writes it (it equals the smoothed state at the
 * outermost used layer); `out` may alias `seeds`.  While the call runs, sm->par / sm->cov also hold its
 * intermediate per-layer states (no other scratch is used).  A backward step that fails sets
 * KF_STATUS_SMOOTH_FAIL in out->status (see there).  Path-length material, finite barrels and the energy-loss
 * option are honoured (with energy loss the map between two layers is J F, reading A21: its Jacobian and its
 * process noise J Q J^T enter the recursion), and so are endcap discs (the smoothed covariance of a layer that
 * is a disc has no variance along z).  All pointers DEV.  Two kernels. */
KF_API int kf_fit_tracks_smooth(kf_ctx* ctx, const kf_geometry* geom, const kf_tracks* seeds,
                                const kf_track_hits* hits, kf_tracks* out, kf_smoothed* sm);

/* Same call with every pointer HOST (pageable or pinned): copies in, fits, copies out, in chunks
 * pipelined over internal streams, and returns when `out` is complete.  This is the end-to-end
 * path (transfers overlapped with kernels).  Alignment rules do not apply.  The results are
 * those of kf_fit_tracks on the same tracks, bit for bit (every chunk runs the kernel the whole batch would). */
KF_API int kf_fit_tracks_host(kf_ctx* ctx, const kf_geometry* geom, const kf_tracks* seeds,
                       const kf_track_hits* hits, kf_tracks* out);

/* kf_fit_tracks_host for seeds whose covariance is DIAGONAL (what a seeding step hands over: reading A13; the seeds
 * of configs[0-3]): seeds->cov is HOST [6][ld], the variances xx yy zz pxpx pypy pzpz, and only those six planes
 * cross the link (24 instead of 84 bytes per track; the end-to-end path is bound by the host-to-device link, and 84
 * of a track's 473 input bytes at ten layers were that covariance).  The other 15 elements are zero on the device.
 * Results are those of kf_fit_tracks_host given the same covariance in full, bit for bit.  `out->cov` is the full
 * [21][ld] as always (and must not alias seeds->cov). */
KF_API int kf_fit_tracks_host_diag(kf_ctx* ctx, const kf_geometry* geom, const kf_tracks* seeds,
                                   const kf_track_hits* hits, kf_tracks* out);

/* kf_fit_tracks_host_diag for hits whose covariance is diagonal in the hit's OWN cylindrical frame (what a strip or
 * pixel sensor measures, and how the hits of every config here are made: a resolution along the radius, one along
 * r-phi, one along z; PAPER.md:168 names the host-device transfers as the bottleneck to address next, and 240 of the
 * 413 input bytes per ten-layer track of the _diag call are hit covariances).  hits->cov is HOST [n_layers][3][ld]:
 * the variances v_r, v_t, v_z of the hit of track t on layer l along r^ = (x, y, 0)/rho, t^ = (-y, x, 0)/rho and z^,
 * (x, y) the hit's own position; only those three planes per layer cross the link (12 instead of 24 bytes per hit).
 * The device rebuilds, in fp32,
 *     c2 = x x / rho2, s2 = y y / rho2, cs = x y / rho2, rho2 = x x + y y   (rho2 = 0: c2 = 1, s2 = cs = 0)
 *     xx = v_r c2 + v_t s2,  xy = (v_r - v_t) cs,  yy = v_r s2 + v_t c2,  xz = yz = 0,  zz = v_z
 * and fits as kf_fit_tracks does.  Results are those of kf_fit_tracks_host_diag given that covariance in full, up to
 * the rounding of the five lines above (not bit for bit when the caller rebuilt it in another order or precision).
 * seeds->cov is HOST [6][ld] as in kf_fit_tracks_host_diag. */
KF_API int kf_fit_tracks_host_compact(kf_ctx* ctx, const kf_geometry* geom, const kf_tracks* seeds,
                                      const kf_track_hits* hits, kf_tracks* out);

/* ---- hits of one layer and their (eta, phi) bins ------------------------------------ */
typedef struct {
    int64_t n_hits, ld;       /* ld >= n_hits, ld % 4 == 0                                         */
    const float* pos;         /* DEV [3][ld]                                                       */
    const float* cov;         /* DEV [6][ld]                                                       */
} kf_layer_hits;

typedef struct {
    int n_eta, n_phi;         /* n_eta*n_phi <= KF_MAX_BINS, n_phi even                            */
    float eta_max;            /* eta bins cover [-eta_max, eta_max), out-of-range hits clamp       */
    int64_t ld;               /* plane stride of pos_sorted / cov_sorted, >= n_hits, % 4 == 0      */
    int32_t* bin_offset;      /* DEV [n_eta*n_phi + 1] first sorted slot of each bin               */
    int32_t* sorted_to_orig;  /* DEV [n_hits] original index of the hit in each sorted slot        */
    float* hit_rec;           /* DEV [n_hits][KF_HIT_RECORD_FLOATS] hits in bin order, packed for scoring:
                                 x y z vzz | vxx vxy vyy index(int32 bits) | vxz vyz 0 0           */
    float* bin_box;           /* DEV [n_eta*n_phi][8] per-bin bounds for the scan's bin pruning:
                                 x_lo x_hi y_lo y_hi | z_lo z_hi max(vzz) max(vxx+vyy)              */
    int32_t* orig_to_sorted;  /* DEV [n_hits] inverse of sorted_to_orig; optional (NULL = not written) */
    float* pos_sorted;        /* DEV [3][ld] hits in bin order, SoA; optional (NULL = not written)  */
    float* cov_sorted;        /* DEV [6][ld] optional (NULL = not written)                          */
} kf_layer_bins;

/* Fit with the hits addressed by index (what a builder hands to the fitter): the hit of
 * track t on layer l is hit index[l*ld_index + t] of pools[l] (HOST array of n_layers descriptors, DEV
 * buffers inside), -1 = no hit on that layer.  Otherwise exactly kf_fit_tracks (same arithmetic, same
 * status semantics, `out` may alias `seeds`).  index: DEV int32 [n_layers][ld_index], ld_index >= n.
 * `bins` = NULL, or a HOST array of n_layers kf_layer_bins made from the same pools by kf_bin_layers with
 * hit_rec and orig_to_sorted filled: the hits are then read from those packed records (2 memory sectors per
 * hit instead of 9), same values, same results.  With bins = NULL the call packs the pools into records of its own
 * first (context scratch of 48 bytes per pool hit, grown on demand like the other scratch: a call that has to grow
 * it synchronises the stream and cannot be recorded into a graph), unless the pools hold more than eight times the
 * hits the tracks can read, in which case the SoA planes are read directly.  Same results either way, bit for bit. */
KF_API int kf_fit_tracks_indexed(kf_ctx* ctx, const kf_geometry* geom, const kf_tracks* seeds,
                                 const int32_t* index, int64_t ld_index, const kf_layer_hits* pools,
                                 const kf_layer_bins* bins, kf_tracks* out);

/* Bin one layer's hits: bin = i_eta*n_phi + i_phi with eta = asinh(z/radius), phi = atan2(y,x) over
 * [-pi, pi); stable counting sort (within a bin, original order).  The bin of a hit is decided in
 * single precision against tabulated edges (reading A16b).  radius_cm = 0 says that the pool belongs to a
 * DISC layer (reading A24): the bins stay projective, eta = asinh(z / rho) with each hit's own rho = sqrt(x^2 + y^2)
 * (in the single-precision rule rho = fl(sqrt(fl(fl(x x) + fl(y y))))).  `out` arrays are
 * caller-allocated.  n_hits == 0 is valid (all offsets 0). */
KF_API int kf_bin_hits(kf_ctx* ctx, float radius_cm, const kf_layer_hits* hits, kf_layer_bins* out);

/* The same for n_layers layers at once (HOST arrays of descriptors, DEV buffers inside): four or five kernel
 * launches in total instead of four per layer.  All layers must share n_eta, n_phi and eta_max. */
KF_API int kf_bin_layers(kf_ctx* ctx, int n_layers, const float* radius_cm, const kf_layer_hits* hits,
                         kf_layer_bins* out);

/* Optional: a processing order for kf_score_candidates that puts candidates reaching the same
 * (eta, phi) bin of `layer` next to each other (stable counting sort of the candidates by that bin),
 * so that neighbouring warps share their hit windows in cache.  order[n] DEV, a permutation of 0..n-1.
 * Purely a scheduling hint: results do not depend on it. */
KF_API int kf_order_candidates(kf_ctx* ctx, const kf_geometry* geom, int layer, const kf_tracks* cands,
                               int n_eta, int n_phi, float eta_max, int32_t* order);

/* Best-hit scoring of n candidates on ONE layer (`layer` indexes the geometry): propagate (+Q),
 * take the candidate's own (eta, phi) bin, score chi2 = r^T (C'_pp + V_h)^-1 r for every hit in
 * the window i_eta +- window_half (clipped), i_phi +- window_half (wrapped); best = lowest chi2,
 * exact ties -> lowest original index; accepted iff chi2 < chi2_cut.
 * Accepted and do_update: Kalman update, nhits += 1, chi2 += best.  Otherwise the candidate keeps
 * the propagated state (Q included).  best_hit[n] = ORIGINAL hit index or -1; best_chi2[n] = the
 * lowest chi2 in the window when it is below chi2_cut, otherwise some value >= chi2_cut (hits that
 * provably cannot beat the cut are not evaluated; +inf if none was).  Propagation failure: status bit, candidate untouched,
 * best_hit = -1, best_chi2 = +inf.  Reads bins->bin_offset, bins->hit_rec and bins->bin_box.  `order` = NULL or the
 * output of kf_order_candidates.  All pointers DEV.  The caller loops over layers.
 * `local_state` (optional, DEV [30][cands->ld] floats, 16-byte aligned, caller-allocated and ZEROED before the
 * first layer): the candidates in the kernels' track-local frame, kept between the per-layer calls.  A Cartesian
 * 6 x 6 covariance in fp32 cannot carry a fitted track to the tolerances of this library (|p| loose, direction
 * tight: the momentum block is nearly singular); handed back in `cands` after every layer and read again, it
 * costs about 2e-3 on covariance elements per round trip.  With `local_state` the call reads a candidate whose
 * flag (plane 29) is set from there instead of from cands->par / cov, and leaves the updated candidate there
 * (flag set) as well as in `cands`, so a chain of per-layer calls meets the same tolerances as
 * kf_build_best_hit and kf_fit_tracks.  Opaque otherwise; zero plane 29 (or all of it) whenever `cands` is
 * changed by anything but this call.  NULL: the candidate is read from `cands` (converted in double). */
KF_API int kf_score_candidates(kf_ctx* ctx, const kf_geometry* geom, int layer, kf_tracks* cands,
                               const kf_layer_hits* hits, const kf_layer_bins* bins, int window_half,
                               float chi2_cut, int do_update, const int32_t* order, int32_t* best_hit,
                               float* best_chi2, float* local_state);

/* kf_score_candidates for callers that must not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same arguments, same kernels, same results, but the per-candidate scratch
 * (the propagated candidate the scan reads, 31 floats per candidate) lives in ONE array compiled into the library,
 * `static __device__` in kf_score.cu, instead of the context's cudaMalloc'ed scratch.  The call makes no
 * cudaMalloc / cudaFree and calls no allocating routine, at any size, first call included; it never touches the
 * context's scratch (kf_graph_launch staleness is unaffected).
 *   Limit:  cands->n <= KF_STATIC_MAX_CANDIDATES, else KF_ERR_TOO_LARGE and nothing is launched.  The array is
 *           31 * KF_STATIC_MAX_CANDIDATES * 4 bytes = 7.75 MiB; every GPU that loads the library holds it until
 *           the process exits, whether or not this call is used.
 *   Shared: every call on a device, from every context and stream, uses the same array, and the array keeps the
 *           last call's contents.  Nothing in it has to start at zero (every slot below cands->n is written before
 *           it is read), so nothing is cleared.  Two calls that overlap on the GPU (different streams, or graph
 *           branches) RACE on it: keep calls of this entry point on one device ordered.
 *   Set-up: the first call on each device resolves the array's device address (cudaGetSymbolAddress, with that
 *           device current; no stream work) and keeps it. */
#define KF_STATIC_MAX_CANDIDATES 65536
KF_API int kf_score_candidates_static(kf_ctx* ctx, const kf_geometry* geom, int layer, kf_tracks* cands,
                                      const kf_layer_hits* hits, const kf_layer_bins* bins, int window_half,
                                      float chi2_cut, int do_update, const int32_t* order, int32_t* best_hit,
                                      float* best_chi2, float* local_state);

/* Best-hit building over n_build_layers consecutive layers first_layer, first_layer+1, ... in one call
 * (PAPER.md:73, 133): per layer exactly what kf_score_candidates does, but the candidates stay in the
 * kernel's track-local frame between layers, so the fitted state meets the same tolerances as
 * kf_fit_tracks (the per-layer call has to hand the covariance back in the global frame in fp32 after
 * every layer).  hits[j] / bins[j] (HOST arrays, DEV buffers inside) belong to layer first_layer + j.
 * hit_index[j*ld_out + i] = ORIGINAL index of the hit taken by candidate i on that layer or -1,
 * hit_chi2[j*ld_out + i] = its chi2 (see kf_score_candidates for rejected candidates); both DEV,
 * [n_build_layers][ld_out], ld_out >= n.  A candidate that reaches no layer at all comes back through
 * the local frame (equal to its input within fp32 rounding); a bad charge leaves it untouched. */
KF_API int kf_build_best_hit(kf_ctx* ctx, const kf_geometry* geom, int first_layer, int n_build_layers,
                             kf_tracks* cands, const kf_layer_hits* hits, const kf_layer_bins* bins,
                             int window_half, float chi2_cut, int do_update, const int32_t* order,
                             int32_t* hit_index, float* hit_chi2, int64_t ld_out);

/* Best-hit building of SEVERAL EVENTS in one call (section 4.3: "concurrent events should be adapted
 * to track building because this will help to fill the GPU's stream multiprocessors"; the fit gains
 * a factor 3 from several events at once).  One event of 20 000 candidates is 157 CTAs of per-candidate work and
 * about two waves of scanning warps on 148 SMs; n_events of them in one call fill the device with the same
 * 2 n_build_layers + 1 launches.  `cands` holds the candidates of all events back to back: event e owns
 * event_first[e] .. event_first[e + 1] - 1 (HOST int64 [n_events + 1], event_first[0] = 0, last = cands->n).
 * hits / bins: HOST arrays [n_events][n_build_layers] (event-major), every event with its own pools, all bins
 * with one (n_eta, n_phi, eta_max).  n_events <= 32.  Per candidate the result is exactly what kf_build_best_hit
 * gives for its event alone (bit for bit); outputs as there. */
KF_API int kf_build_best_hit_events(kf_ctx* ctx, const kf_geometry* geom, int first_layer, int n_build_layers,
                                    int n_events, const int64_t* event_first, kf_tracks* cands,
                                    const kf_layer_hits* hits, const kf_layer_bins* bins, int window_half,
                                    float chi2_cut, int do_update, int32_t* hit_index, float* hit_chi2,
                                    int64_t ld_out);

/* Best-hit building of one event with every buffer in HOST memory (pageable or pinned; pinned for overlap):
 * the end-to-end path of building (section 4.3: on the K40 "almost half" of the building wall
 * time went into transfers).  The candidates and, layer by layer on a second stream, the hit pools go to the
 * device; layer j is binned (n_eta x n_phi bins over [-eta_max, eta_max) x [-pi, pi)) and scored while layer j + 1
 * is still on its way; the candidates stay in the local frame between the layers; candidates, hit_index and
 * hit_chi2 (HOST [n_build_layers][ld_out]) come back and the call returns when they are complete.  hits: HOST
 * array of n_build_layers descriptors with HOST buffers inside.  Results are those of kf_bin_layers +
 * kf_build_best_hit on the same data (the bins themselves stay on the device and are not returned).  Alignment
 * rules do not apply.  Not recordable in a graph. */
KF_API int kf_build_best_hit_host(kf_ctx* ctx, const kf_geometry* geom, int first_layer, int n_build_layers,
                                  kf_tracks* cands, const kf_layer_hits* hits, int n_eta, int n_phi, float eta_max,
                                  int window_half, float chi2_cut, int do_update, int32_t* hit_index,
                                  float* hit_chi2, int64_t ld_out);

/* Combinatorial building (reading A19) over n_build_layers consecutive
 * layers.  Every seed keeps at most n_cand (1..8) candidates.  On each layer every candidate is propagated
 * (+Q); every hit of its window with chi2 < chi2_cut spawns a child (Kalman update, nhits + 1, chi2 +
 * increment; only a candidate's n_cand best hits can survive, so only those are kept), one more child takes
 * no hit; a candidate that cannot reach the layer yields itself unchanged (PROP_FAIL bit).  The children of a
 * seed are ranked by (nhits descending, chi2 ascending, parent slot, hit original index with "no hit" last)
 * and the best n_cand survive.  On return `cands` holds the best candidate of every seed (state, covariance,
 * chi2, nhits, status); hit_index[j*ld_out + i] = original index of its hit on layer first_layer + j or -1;
 * n_found[i] (optional, DEV [n]) = candidates alive at the end.  With n_cand = 1 this is kf_build_best_hit.
 * hits[j] / bins[j]: HOST arrays as in kf_build_best_hit.  A bad charge leaves the seed untouched. */
KF_API int kf_build_combinatorial(kf_ctx* ctx, const kf_geometry* geom, int first_layer, int n_build_layers,
                                  kf_tracks* cands, const kf_layer_hits* hits, const kf_layer_bins* bins,
                                  int window_half, float chi2_cut, int n_cand, int32_t* hit_index,
                                  int32_t* n_found, int64_t ld_out);

/* Combinatorial building of SEVERAL EVENTS in one call (as kf_build_best_hit_events): `cands` holds
 * the seeds of all events back to back, event e owns event_first[e] .. event_first[e + 1] - 1 (HOST int64
 * [n_events + 1], event_first[0] = 0, last = cands->n); hits / bins: HOST arrays [n_events][n_build_layers]
 * (event-major), every event with its own pools, all bins with one (n_eta, n_phi, eta_max); n_events <= 32.  The
 * same 4 n_build_layers + 2 launches as one event.  Per seed the result is exactly what kf_build_combinatorial gives
 * for its event alone (bit for bit); outputs as there. */
KF_API int kf_build_combinatorial_events(kf_ctx* ctx, const kf_geometry* geom, int first_layer, int n_build_layers,
                                         int n_events, const int64_t* event_first, kf_tracks* cands,
                                         const kf_layer_hits* hits, const kf_layer_bins* bins, int window_half,
                                         float chi2_cut, int n_cand, int32_t* hit_index, int32_t* n_found,
                                         int64_t ld_out);

#ifdef __cplusplus
}
#endif
#endif /* KF_B200_H */
