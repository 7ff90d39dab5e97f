/*
 * hough.h -- C ABI of the B200-native Hough-transform track finder (libhough_b200.so).
 *
 * The operation is the data-parallel hot path of the fast tracking algorithm of
 * arXiv:1305.4855: "each hit maps to a curve in the track-parameter space, the curves of
 * all hits are accumulated, local maxima of the accumulator are the track candidates"
 * (section 7; Fig. 3; section 8 for the curved
 * 2-parameter case; "accumulator and peak detection reside in GPU memory").
 * BASELINE.json north_star fixes its concrete form (restated as SURVEY.md section 8(c)
 * A1..A7, which DESIGN.md section 2 adopts):
 *
 *   - parameters (phi0, d0, kappa); for every hit (x, y, layer), every phi0 bin centre i
 *     and every d0 bin centre j:  s = -x sin(phi0_i) + y cos(phi0_i),
 *       kappa = 2 (s - d0_j) / (r^2 - 2 d0_j s + d0_j^2),      r^2 = x^2 + y^2;
 *     if kappa_min <= kappa < kappa_max the hit's layer bit is OR-ed into the uint32
 *     mask of bin (i, j, k), k = the kappa bin;
 *   - a bin is a peak iff popcount(mask) >= L_min and it beats all (up to 26)
 *     neighbours, ties going to the lower linear index; phi0 may wrap;
 *   - every peak is emitted, in ascending linear index, with its mask and the ascending
 *     list of the hits that voted into exactly that bin.
 *   All arithmetic is IEEE-754 binary32, round-to-nearest-even, unfused, in a fixed
 *   order, so results are bit-identical to the CPU oracle.
 *
 * Conventions
 *   - Pointers marked [device] are CUDA device pointers on the handle's device; [host]
 *     are ordinary host pointers (pinned memory makes the async copies truly async).
 *   - The library never allocates device memory: the caller hands in one workspace
 *     (e.g. a torch tensor) and the output arrays, and keeps them alive.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *     Calls that take a stream only ENQUEUE work and return without synchronising,
 *     unless stated otherwise.  One handle is used from one stream at a time.  The handle owns one
 *     auxiliary stream of its own (created by hough_create): hough_vote builds the per-event hit index
 *     of the hit lists there, beside the vote kernel, and hough_peaks makes `cuda_stream` wait for it
 *     through events -- invisible to the caller, whose stream order is all that matters.
 *   - Every int-returning call returns HOUGH_OK (0) or a negative HOUGH_E* code; nothing
 *     throws across the boundary.  All configuration is the hough_config struct: the library
 *     reads no environment variable.  Its only process-wide state is a mutex-guarded record
 *     of the dynamic shared-memory limit it has set per (kernel, device) -- a CUDA attribute
 *     that is itself process-wide; handles share nothing else and may live on different threads.
 *   - There is no CPU fallback: without a CUDA device every compute call returns
 *     HOUGH_ECUDA.
 *   - Accumulator layout: bin (i, j, k) at linear index lin = (i*n_d0 + j)*n_kappa + k
 *     (kappa fastest).
 */
#ifndef HOUGH_B200_H
#define HOUGH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HOUGH_OK 0
#define HOUGH_EINVAL (-1) /* bad argument / configuration */
#define HOUGH_ENOMEM (-2) /* workspace or capacity too small */
#define HOUGH_ECUDA (-3)  /* a CUDA runtime call failed (or no device) */
#define HOUGH_ESTATE (-4) /* call order violated (e.g. hough_peaks before hough_vote) */

/* hough_counts.flags */
#define HOUGH_TRUNCATED_PEAKS 1u /* n_peaks > cap_peaks: only the first cap_peaks (in lin order) were written */
#define HOUGH_TRUNCATED_HITS 2u  /* n_hit_entries > cap_hits: hit_index holds the first cap_hits entries */
#define HOUGH_INDEX16 4u         /* hit_index16 was written as well (the event has <= 65536 hits) */
#define HOUGH_LIST_MISMATCH 8u   /* set by the list check (HOUGH_OPT_CHECK_LISTS / hough_check_lists): some peak's hit
                                    list is not ascending or the OR of its hits' layer bits is not the peak's mask */

/* hough_config.options */
#define HOUGH_OPT_NO_CULL 1u      /* evaluate every (hit, cell): the unpruned sweep (for measurements/tests) */
#define HOUGH_OPT_STAGE_TIMING 2u /* record a CUDA event after every kernel (see hough_stage_times) */
#define HOUGH_OPT_EXACT_ONLY 8u   /* evaluate every bin with the exact recipe (no fixed-point fast path with
                                     exact fallback near bin edges; results are identical either way) */
#define HOUGH_OPT_LIST_SWEEP 16u  /* hit lists by a second sweep of all hits over all cells (the round-1 path)
                                     instead of the peak-driven lists; results are identical either way */
#define HOUGH_OPT_LINE 32u        /* f3, straight-line transform (Fig. 3; recipe E1):
                                     the phi axis is the line's direction theta, n_d0 must be 1 and the kappa axis
                                     is rho [cm]; a hit votes rho = -x sin(theta_i) + y cos(theta_i) */
#define HOUGH_OPT_INTERVAL 64u    /* f3, interval voting (recipe E2): a hit sets every kappa bin
                                     between its closed-form values at the two EDGES of phi0 bin i (d0 centre j);
                                     n_votes counts the bins set.  Not together with HOUGH_OPT_LINE */
#define HOUGH_OPT_FUSED_PEAKS 128u /* a5, fused variant (north_star: "peak finding is fused on the tile"): hough_vote's
                                     tile kernel decides the peak flags of the cells that are not on the edge of its
                                     tile from shared memory, hough_peaks only visits the tile-edge cells
                                     (k_peak_cells) instead of sweeping the whole accumulator.  Needs n_layers <= 16
                                     and not HOUGH_OPT_UNPACKED.  Results are identical either way */
#define HOUGH_OPT_CELL_PEAKS 256u /* peak flags of EVERY cell by the cell-wise kernel (k_peak_cells) instead of the
                                     streaming sweep: cross-check and measurement of that kernel */
#define HOUGH_OPT_CHECK_LISTS 512u /* run hough_check_lists at the end of every hough_peaks (a safety net for the
                                     peak-driven lists, whose candidate windows are supersets by derivation: a hit
                                     missing from a list shows up as HOUGH_LIST_MISMATCH instead of silently) */
#define HOUGH_OPT_UNPACKED 4u     /* one mask per 32-bit word of the vote tile even with <= 16 layers (test hook
                                     for the tile layout used with 17..32 layers) */

typedef struct hough_handle hough_handle; /* opaque */

/*
 * Grid and detector description (BASELINE.json north_star: "hough_create(layer radii,
 * grid ranges/bins, L_min)").  Bin centres: phi0_i = phi_min + (i + 0.5)(phi_max - phi_min)/n_phi,
 * d0_j likewise; kappa bins are the n_kappa equal half-open intervals of
 * [kappa_min, kappa_max).  n_d0 = 1 with d0_min = d0_max = 0 is the 2-parameter transform
 * through the interaction point.
 */
typedef struct hough_config {
    int32_t n_layers;              /* 1..32; hit layer l sets mask bit l */
    const double *layer_radius_cm; /* [host] n_layers radii, > 0; metadata only: the vote uses the hit's own x^2+y^2 */
    double phi_min, phi_max;       /* phi_max > phi_min */
    double d0_min, d0_max;         /* d0_max >= d0_min (equal only if n_d0 == 1); |d0| <= 1e15 */
    double kappa_min, kappa_max;   /* kappa_max > kappa_min; |kappa| <= 1e15 */
    int32_t n_phi, n_d0, n_kappa;  /* >= 1; n_kappa a multiple of 32, <= 16384; n_phi*n_d0*n_kappa < 2^32 */
    int32_t L_min;                 /* 1..n_layers */
    int32_t phi_wrap;              /* 1: phi0 is periodic in the peak test (needs n_phi >= 3); 0: not */
    uint32_t max_hits;             /* largest n accepted by hough_vote / hough_process_host (<= 1 044 480) */
    uint32_t cap_peaks;            /* capacity of the caller's peak arrays (>= 1) */
    uint64_t cap_hits;             /* capacity of the caller's hit_index array (>= 1) */
    int32_t tile_phi, tile_d0;     /* accumulator tile owned by one CTA, in cells; 0 = choose automatically */
    uint32_t options;              /* HOUGH_OPT_* */
    int32_t device;                /* CUDA device ordinal */
} hough_config;

/* Counters of one event, 48 bytes, same layout on host and device. */
typedef struct hough_counts {
    uint64_t n_votes;       /* votes cast (in-range solutions over all hit x cell pairs) */
    uint64_t n_hit_entries; /* TRUE total length of the hit lists of the reported peaks */
    uint64_t n_evals;       /* closed-form evaluations the vote kernel executed after its conservative
                               cull (<= n * n_phi * n_d0; equal to it with HOUGH_OPT_NO_CULL) */
    uint64_t n_list_evals;  /* evaluations the hit-list stage executed (0 after hough_peaks_only) */
    uint32_t n_peaks;       /* TRUE number of peaks (may exceed cap_peaks) */
    uint32_t n_bad_hits;    /* hits with layer outside [0, n_layers): cast no vote */
    uint32_t flags;         /* HOUGH_TRUNCATED_* */
    uint32_t reserved;
} hough_counts;

/*
 * Output arrays of hough_peaks, all [device], caller-owned.  Peaks are in ascending lin.
 * Peak p (p < min(n_peaks, cap_peaks)): bin[p] = lin, mask[p] = its layer mask, and its
 * hits are hit_index[hit_offset[p] .. hit_offset[p+1]) in ascending hit index.
 * hit_offset[min(n_peaks, cap_peaks)] = n_hit_entries.  Entries at positions >= cap_hits
 * are not written (lists are complete while they fit).
 */
typedef struct hough_peaks_out {
    uint32_t *bin;        /* [device] cap_peaks */
    uint32_t *mask;       /* [device] cap_peaks */
    uint64_t *hit_offset; /* [device] cap_peaks + 1 */
    uint32_t *hit_index;  /* [device] cap_hits */
    hough_counts *counts; /* [device] 1 */
    uint16_t *hit_index16; /* [device] cap_hits, OPTIONAL (NULL: not wanted): the same entries as 16-bit values,
                              written beside hit_index when the event has <= 65536 hits and the lists come from
                              the default (peak-driven) path or the vote variants; counts->flags then carries
                              HOUGH_INDEX16.  Halves the bytes a host has to read back (see hough_host_out) */
} hough_peaks_out;

/* Host mirror of hough_peaks_out for hough_process_host ([host] pointers, same capacities). */
typedef struct hough_host_out {
    uint32_t *bin;
    uint32_t *mask;
    uint64_t *hit_offset;
    uint32_t *hit_index; /* may be NULL: hit lists are then computed but not copied back */
    hough_counts *counts;
    uint16_t *hit_index16; /* OPTIONAL (NULL: not wanted), cap_hits entries: when the event's counts carry
                              HOUGH_INDEX16 the lists are copied back in this form INSTEAD of hit_index (halves the
                              bytes of the lists: a config-3 event returns 19.7 MB instead of 31.8 MB in all);
                              otherwise hit_index is used as above */
} hough_host_out;

/* Bytes of device workspace hough_create needs for cfg (0 if cfg is invalid). */
size_t hough_workspace_bytes(const hough_config *cfg);

/*
 * Validate cfg, build the bin-centre tables on the host in fp64 and round them once to
 * fp32 (sin/cos of phi0_i, d0_j, 2 d0_j, d0_j^2, kappa_min, kappa_max, n_kappa/(kappa_max-kappa_min)),
 * upload them and carve the accumulator and scratch out of `workspace` ([device], 256-byte
 * aligned, >= hough_workspace_bytes(cfg)).  Synchronises the device once.  The library
 * owns *out (free with hough_destroy); the caller owns the workspace.
 * Errors: HOUGH_EINVAL (bad cfg / NULL), HOUGH_ENOMEM (workspace too small), HOUGH_ECUDA.
 */
int hough_create(const hough_config *cfg, void *workspace, size_t workspace_bytes, hough_handle **out);

/* Free the handle and its table memory.  NULL is a no-op.  Never frees caller memory. */
void hough_destroy(hough_handle *h);

/*
 * Process ONE event's hits (BASELINE.json north_star: "hough_vote(hits, n, stream)"):
 * x, y [device] fp32[n] transverse coordinates in cm, layer [device] int32[n].  The
 * accumulator is defined from scratch by this call (no accumulation across calls):
 * hit preparation (r^2, layer bit), per-tile hit staging, shared-memory tile voting,
 * tile write-out and the vote count are enqueued on the stream.  n = 0 is legal (all-zero
 * accumulator).  Hits with a layer outside [0, n_layers) or non-finite coordinates cast no vote.
 * The hit arrays must stay valid until the stream has passed this call's work (the first kernel
 * copies them into the workspace; everything after it, hit lists and hough_fit included, reads that copy).
 * Errors: HOUGH_EINVAL (NULL handle, n > max_hits, NULL arrays with n > 0), HOUGH_ECUDA.
 */
int hough_vote(hough_handle *h, const float *x, const float *y, const int32_t *layer, uint32_t n,
               void *cuda_stream);

/*
 * Peak finding, compaction and hit lists of the event last given to hough_vote
 * (north_star: "hough_peaks(out)"), enqueued on the stream; results go to the caller's
 * device arrays, including out->counts, so that many events can be processed
 * back-to-back without a host synchronisation.
 * Errors: HOUGH_EINVAL, HOUGH_ESTATE (no hough_vote before), HOUGH_ECUDA.
 */
int hough_peaks(hough_handle *h, const hough_peaks_out *out, void *cuda_stream);

/* [device] pointer to the n_phi*n_d0*n_kappa uint32 masks (lin order), valid after
 * hough_vote's work has completed and until the next hough_vote.  NULL for a NULL handle. */
const uint32_t *hough_accumulator(const hough_handle *h);

/*
 * Whole path for one event with HOST buffers: copies x, y, layer host->device (async on
 * the stream), runs hough_vote + hough_peaks into `dev` (device arrays as for
 * hough_peaks), copies counts, the peak arrays and (if host->hit_index != NULL) the hit
 * lists back to `host`, and SYNCHRONISES the stream before returning.  Only the filled
 * prefixes are copied back (a second small synchronisation on counts is used for that).
 * It stages the hits where slot 0 of the pipeline below stages its own, so it is refused with
 * HOUGH_ESTATE while an event submitted in slot 0 has not been collected.
 */
int hough_process_host(hough_handle *h, const float *x, const float *y, const int32_t *layer,
                       uint32_t n, const hough_peaks_out *dev, const hough_host_out *host,
                       void *cuda_stream);

/*
 * The same as a pipeline, so that three things run at once (the paper's production model,
 * "simultaneously ... processing one event, transferring data ... for the next event
 * ... and returning the results ... for the previously processed event"; steady-state throughput).
 * `slot` (0 .. HOUGH_MAX_SLOTS-1) names one in-flight event; each slot in use needs its own `dev`
 * arrays and `host` buffers.
 *   hough_submit_host    copies x, y, layer host->device on a stream of the LIBRARY's own (created at the
 *                        first call, destroyed with the handle) into the slot's own staging arrays, so the
 *                        inputs of event e+1 land while event e computes; makes `cuda_stream` wait for
 *                        them; enqueues hough_vote + hough_peaks into `dev` and a 48-byte copy of the
 *                        counters to pinned memory of the library; returns at once.
 *   hough_collect_begin  waits ON THE HOST until the slot's computation is complete, writes host->counts,
 *                        enqueues the copies of the filled prefixes of the peak arrays and hit lists to
 *                        `host` on `copy_stream` and returns (no device round trip for the sizes).
 *   hough_collect_end    waits on the host until those copies have landed; the slot is free again.
 *   hough_collect_host   = hough_collect_begin + hough_collect_end.
 * Patterns:  two slots:   submit(e, e&1);  if (e > 0) collect_host(e-1);  ...
 *            three slots: submit(e, e%3);  if (e > 0) collect_begin(e-1);  if (e > 1) collect_end(e-2);  ...
 *            (the device->host copy engine never waits for the host).
 * The pipeline's stream, events and pinned counters are created by the first hough_submit_host, all or nothing:
 * if that fails (HOUGH_ECUDA) nothing is kept and the next call starts over.
 * A slot must be collected (end) before it is submitted again.  The host arrays must be pinned for the
 * copies to overlap.  Errors as hough_process_host; HOUGH_ESTATE if the slot is not in the state the call
 * needs.  One handle computes one event at a time: `cuda_stream` should be the same stream for all slots.
 */
#define HOUGH_MAX_SLOTS 4
int hough_submit_host(hough_handle *h, const float *x, const float *y, const int32_t *layer,
                      uint32_t n, const hough_peaks_out *dev, int32_t slot, void *cuda_stream);
int hough_collect_begin(hough_handle *h, const hough_peaks_out *dev, const hough_host_out *host,
                        int32_t slot, void *copy_stream);
int hough_collect_end(hough_handle *h, int32_t slot);
int hough_collect_host(hough_handle *h, const hough_peaks_out *dev, const hough_host_out *host,
                       int32_t slot, void *copy_stream);

/*
 * Stand-alone accumulator kernels, used for the
 * HBM-roofline measurements and as cross-checks:
 *   hough_clear       zero the global accumulator (pure HBM write);
 *   hough_peak_sweep  run only the peak-flag sweep over the current accumulator (reads
 *                     4 B/bin once, writes 1 bit/bin) and leave the result in the workspace.
 */
int hough_clear(hough_handle *h, void *cuda_stream);
int hough_peak_sweep(hough_handle *h, void *cuda_stream);

/*
 * Device-side invariant of the hit lists in `out` (as hough_peaks of the event last voted on this handle
 * left them): every complete list (one that ends within cap_hits) is strictly ascending, holds valid hit
 * indices, and the OR of its hits' layer bits equals the peak's mask -- which is what "each peak is emitted
 * with its sorted hit list" (north_star) implies, since the mask IS the OR of the votes of exactly those
 * hits.  A violation ORs HOUGH_LIST_MISMATCH into out->counts->flags (on the device, after hough_peaks has
 * written the counters).  One kernel, one warp per peak; costs about as much as reading the lists once.
 * Errors: HOUGH_EINVAL, HOUGH_ESTATE (no hough_vote before), HOUGH_ECUDA.
 */
int hough_check_lists(hough_handle *h, const hough_peaks_out *out, void *cuda_stream);

/* Overwrite the accumulator from a [device] array of n_bins masks (test hook for the peak
 * rule: lets a test run hough_peak_sweep / hough_peaks_only on a hand-made accumulator). */
int hough_set_accumulator(hough_handle *h, const uint32_t *acc_dev, void *cuda_stream);
/* Peak flags + compaction only (no hit lists: hit_offset/hit_index untouched, n_hit_entries = 0). */
int hough_peaks_only(hough_handle *h, const hough_peaks_out *out, void *cuda_stream);

/*
 * Shared-memory atomic micro-benchmark that defines the "shared-atomic roofline" on the
 * box: every SM runs `ctas_per_sm` CTAs of `threads` threads,
 * each thread issues `iters` no-return 32-bit OR operations into the CTA's shared-memory table.
 * mode 0: atomicOr, conflict-free (32 lanes -> 32 banks, distinct addresses);
 * mode 1: atomicOr, pseudo-random addresses (bank conflicts as they fall);
 * mode 2: plain load/OR/store on the same conflict-free addresses (no atomic), for comparison.
 * Enqueues on the stream; *lane_ops (host) receives the number of lane-operations one
 * launch performs.  sink_dev: [device] 4 bytes of caller-owned scratch (keeps the compiler from
 * dropping the loop; the library allocates nothing).  Time it with CUDA events around the call.
 */
int hough_microbench_smem(int device, int mode, int threads, int ctas_per_sm, int iters,
                          uint32_t *sink_dev, void *cuda_stream, uint64_t *lane_ops);

/*
 * ---- f1: the second Hough transform, over the peaks of the first (section 9:
 * "the crossings all lie along a single sinusoidal curve in the parameter space ... that one
 * sinusoidal curve corresponds to a point in the original x-y space ... the vertex of the
 * displaced jet ... use the Hough transform a second time, this time applying it not to the hits
 * in the x-y space but the crossings in the parameter space").  Recipe E3 of DESIGN.md section 8:
 * a reported peak (i, j, k) is the point (phi0_i, d0_j) of the parameter space; the sinusoid of a
 * vertex (xv, yv) is d0 = -xv sin(phi0) + yv cos(phi0), so the peak votes along the line it
 * defines in the (xv, yv) plane, once per bin centre of the axis the line is less steep against
 * (|cos phi0_i| >= |sin phi0_i|: every x centre a, yv = (d0_j + xc[a] sin)/cos; otherwise every y
 * centre b, xv = (yc[b] cos - d0_j)/sin; binary32 round-to-nearest, unfused, in that order), adding 1
 * to the uint32 count of bin (a, b), lin = a*n_y + b.  A bin is a vertex iff its count >= V_min
 * and it beats its (up to 8) neighbours, ties to the lower lin (no wrap).  Every vertex is emitted
 * in ascending lin with its count and the ascending list of the positions p (in the peak arrays)
 * of the peaks whose own vote at the vertex's column (row for steep lines) lands in its bin.
 */
typedef struct hough_vertex_config {
    double x_min, x_max;   /* x_max > x_min [cm] */
    double y_min, y_max;   /* y_max > y_min */
    int32_t n_x, n_y;      /* 1..2048 each */
    int32_t V_min;         /* >= 1 */
    uint32_t cap_vertices; /* capacity of the caller's vertex arrays (>= 1, <= 65536) */
    uint64_t cap_members;  /* capacity of the caller's member_index array (>= 1) */
} hough_vertex_config;

typedef struct hough_vertex_counts { /* 32 bytes, same layout on host and device */
    uint64_t n_vertex_votes;   /* votes cast into the (xv, yv) accumulator */
    uint64_t n_member_entries; /* TRUE total length of the member lists of the reported vertices */
    uint32_t n_vertices;       /* TRUE number of vertices (may exceed cap_vertices) */
    uint32_t flags;            /* 1: vertices truncated, 2: member lists truncated (first cap_* kept, in order) */
    uint64_t reserved;
} hough_vertex_counts;

typedef struct hough_vertex_out { /* all [device], caller-owned */
    uint32_t *bin;            /* cap_vertices: lin = a*n_y + b */
    uint32_t *count;          /* cap_vertices */
    uint64_t *member_offset;  /* cap_vertices + 1 */
    uint32_t *member_index;   /* cap_members: positions in the peak arrays */
    hough_vertex_counts *counts;
} hough_vertex_out;

/* Bytes of [device] scratch hough_vertices needs (0 if vc is invalid).  Its first n_x*n_y uint32
 * words are the (xv, yv) accumulator, lin order, valid after the call's work has completed. */
size_t hough_vertex_workspace_bytes(const hough_vertex_config *vc);

/*
 * Enqueue the second transform over the peaks in `peaks` (the arrays hough_peaks filled for this
 * handle's grid: only bin[] and counts->n_peaks are read, on the device, so no host
 * synchronisation is needed between hough_peaks and this call).  `workspace`: [device], 256-byte
 * aligned, >= hough_vertex_workspace_bytes(vc), caller-owned, used only during the call's work.
 * Errors: HOUGH_EINVAL (NULL / bad vc), HOUGH_ENOMEM (workspace too small), HOUGH_ECUDA.
 */
int hough_vertices(hough_handle *h, const hough_vertex_config *vc, void *workspace, size_t workspace_bytes,
                   const hough_peaks_out *peaks, const hough_vertex_out *out, void *cuda_stream);

/*
 * ---- f2: fit of every peak's hit list, selection and removal of duplicates (section 8:
 * "find the locations of the peaks ... perform a fit of the hits to the candidate tracks";
 * "the track candidate collection is then cleaned to remove duplicate tracks or tracks
 * which share a large number of hits").  Recipes E4 / E5 of DESIGN.md section 8.
 *
 * E4, per reported peak p with hit list H(p) (ascending hit index, the arrays hough_peaks filled), all
 * in binary64, sums taken over the list in its order, never fused: means mx, my, mr of x, y, x^2+y^2;
 * central moments Cxx, Cxy, Cyy, Cxr, Cyr, Crr; q1 = Crr Cxy - Cxr Cyr; q2 = Crr (Cxx - Cyy) - Cxr^2 +
 * Cyr^2; phi = atan2(2 q1, q2)/2; khat = (-sin(phi) Cxr + cos(phi) Cyr)/Crr; delta = (-mx sin(phi) +
 * my cos(phi)) - khat mr; D = 1 - 4 delta khat; kappa = 2 khat/sqrt(D); d0 = 2 delta/(1 + sqrt(D));
 * rms = sqrt((sum eps^2/n)/D) with eps = khat w - (-sin(phi) u + cos(phi) v) over the centred hits;
 * the FORWARD representation is reported (mx cos(phi) + my sin(phi) >= 0, else phi -+ pi, d0 and kappa
 * negated -- exact sign flips, so the two mirror peaks of a track fit bit-identically).
 * status: 0 ok; 1 fewer than 3 hits; 2 degenerate (Crr = 0, D <= 0, non-finite result); 3 the peak's
 * list is not complete in hit_index (HOUGH_TRUNCATED_HITS cut it): not fitted.
 * E5: p is SELECTED iff status == 0 and rms <= rms_max; a selected p is a DUPLICATE iff another selected
 * o shares at least min_shared hits with it and is better (more layers in its mask; else smaller rms;
 * else lower position).  flag[p] = 0 not selected, 1 selected and kept, 2 selected but a duplicate.
 * kept[] lists the positions p with flag 1 in ascending order (the de-duplicated track collection:
 * what a host needs to read back instead of every peak).
 * Index results (status, flag, kept, counts) are exact given the rms values; the binary64 fit agrees
 * with the CPU oracle to the tolerance DESIGN.md section 8 derives (the moments are bit-identical; the
 * CUDA and host math libraries' atan2 / sin / cos differ in the last bits).
 */
typedef struct hough_fit_config {
    double rms_max;      /* [cm], >= 0 (may be +inf: every status-0 fit is selected) */
    uint32_t min_shared; /* >= 1 */
    uint32_t reserved;   /* 0 */
} hough_fit_config;

typedef struct hough_fit_counts { /* 32 bytes, same layout on host and device */
    uint32_t n_fitted;     /* candidates looked at = min(n_peaks, cap_peaks) */
    uint32_t n_ok;         /* status 0 */
    uint32_t n_selected;   /* flag 1 or 2 */
    uint32_t n_kept;       /* flag 1 = entries of kept[] */
    uint32_t n_duplicates; /* flag 2 */
    uint32_t n_truncated;  /* status 3 */
    uint64_t n_pair_tests; /* candidate pairs whose shared hits were counted (work of the duplicate rule) */
} hough_fit_counts;

typedef struct hough_fit_out { /* all [device], caller-owned, cap_peaks entries each (counts: 1) */
    double *kappa, *phi0, *d0, *rms; /* 0 where status != 0 */
    int32_t *status;
    uint8_t *flag;
    uint32_t *kept;
    hough_fit_counts *counts;
} hough_fit_out;

/* Bytes of [device] scratch hough_fit needs for this handle (its max_hits, cap_peaks, cap_hits);
 * 0 for a NULL handle or cap_hits >= 2^32. */
size_t hough_fit_workspace_bytes(const hough_handle *h);

/*
 * Enqueue E4 + E5 over the peaks and hit lists in `peaks` (the arrays hough_peaks filled for the event
 * last given to hough_vote on this handle: the hit coordinates are the handle's own device copy, so
 * the caller's x / y may already be gone).  Everything is read on the device: no host synchronisation
 * between hough_peaks and this call.  `workspace`: [device], 256-byte aligned, >=
 * hough_fit_workspace_bytes(h), caller-owned, used only during the call's work.
 * Errors: HOUGH_EINVAL (NULL / bad fc / cap_hits >= 2^32), HOUGH_ENOMEM, HOUGH_ESTATE (no hough_vote
 * before), HOUGH_ECUDA.
 */
int hough_fit(hough_handle *h, const hough_fit_config *fc, void *workspace, size_t workspace_bytes,
              const hough_peaks_out *peaks, const hough_fit_out *out, void *cuda_stream);

/*
 * ---- Peaks of an accumulator for callers that cannot allocate device memory.
 *
 * Everything above needs a handle, and a handle needs a workspace somebody got from cudaMalloc.  Some
 * users of a trigger library cannot call it: a plug-in inside a host framework that owns the whole
 * device-memory budget and only lends out input and output buffers; an event loop with real-time
 * constraints, where cudaMalloc / cudaFree are banned because they synchronise the whole device and
 * stall the events in flight on other streams; a thin C / Fortran client that is handed device
 * pointers and links no allocator.  This one call serves them.  It takes NO handle and NO workspace:
 * the scratch its scan needs (a ticket and one look-back word per 2048 bins, 65 792 bytes in all) is a
 * fixed array inside the library's own device code, so every GPU that loads libhough_b200.so holds
 * those 64 KiB from the moment the module is loaded until the process exits.  The call itself never
 * runs cudaMalloc, cudaFree or any library routine that allocates.
 *
 * The operation is the peak rule ("local maxima of the accumulator are the track
 * candidates"; PAPER.md:128 peak detection resident in GPU memory; north_star: popcount >= L_min and a
 * local maximum of the 3x3x3 neighbourhood, ties to the lower linear index; rule A6 of DESIGN.md
 * section 2) followed by the ordered compaction (A7 without the hit lists), i.e. what
 * hough_set_accumulator + hough_peaks_only compute, in one kernel launch:
 *   acc      [device] n_phi*n_d0*n_kappa uint32 masks, lin = (i*n_d0 + j)*n_kappa + k, read-only;
 *   bin,mask [device] cap_peaks entries each: the peaks in ascending lin and their masks; with more
 *            than cap_peaks peaks the first cap_peaks (in lin order) are written;
 *   n_peaks  [device] one uint32: the TRUE number of peaks (may exceed cap_peaks);
 *   n_kappa  any value >= 1 (no multiple-of-32 rule here); L_min 1..32; phi_wrap 1 needs n_phi >= 3.
 * All pointers are the caller's and must stay valid until the stream has passed the call's work.  The
 * call acts on the CURRENT device of the calling thread (cudaSetDevice), which must be the one the
 * pointers live on; it enqueues one 0-fill of the scratch and one kernel on `cuda_stream` and returns
 * without synchronising.
 *
 * Limits and rules that follow from the fixed array:
 *   - n_phi*n_d0*n_kappa <= HOUGH_NOALLOC_MAX_BINS (the 1024 x 64 x 256 grid of BASELINE.json configs
 *     2-4); a larger grid is refused with HOUGH_ENOMEM before anything is enqueued;
 *   - all calls on one GPU share the one array, from every thread and every stream.  Each call clears
 *     the part it uses first (the array keeps the previous call's contents), so calls in stream order
 *     are fine, but two calls whose work OVERLAPS on the same GPU race on it and return garbage or
 *     never finish: issue them on one stream, or order the streams with events;
 *   - the first call on each device looks up the array's device address (cudaGetSymbolAddress, which
 *     may load the module); make that first call before starting any stream capture.
 * Errors: HOUGH_EINVAL (NULL pointer, cap_peaks = 0, bad sizes / L_min / phi_wrap), HOUGH_ENOMEM (grid
 * beyond HOUGH_NOALLOC_MAX_BINS), HOUGH_ECUDA (no device, or a runtime call failed).
 */
#define HOUGH_NOALLOC_MAX_BINS (1u << 24)
int hough_peaks_noalloc(const uint32_t *acc, int32_t n_phi, int32_t n_d0, int32_t n_kappa, int32_t L_min,
                        int32_t phi_wrap, uint32_t *bin, uint32_t *mask, uint32_t cap_peaks, uint32_t *n_peaks,
                        void *cuda_stream);

/* Geometry the library chose (for reporting): tile_phi, tile_d0, n_tiles, threads per CTA,
 * dynamic shared memory bytes of the vote kernel, number of SMs.  Any pointer may be NULL. */
int hough_query(const hough_handle *h, int32_t *tile_phi, int32_t *tile_d0, int32_t *n_tiles,
                int32_t *threads, int32_t *smem_bytes, int32_t *n_sms);

/* Number of kernel launches enqueued by this handle since creation (for bench accounting). */
uint64_t hough_launch_count(const hough_handle *h);

/*
 * Per-kernel device times of the LAST hough_vote + hough_peaks pair, for handles created with
 * HOUGH_OPT_STAGE_TIMING (otherwise HOUGH_ESTATE).  Synchronises on the last recorded event.
 * ms[s] = milliseconds of stage s (0 for a stage that did not run), s < min(cap, HOUGH_N_STAGES);
 * returns the number of stages written or a negative error.  hough_stage_name(s) names stage s
 * (NULL if out of range).  Meant for measurement runs: the extra event records add launch gaps.
 */
#define HOUGH_N_STAGES 9
int hough_stage_times(hough_handle *h, float *ms, int cap);
const char *hough_stage_name(int stage);

const char *hough_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* HOUGH_B200_H */
