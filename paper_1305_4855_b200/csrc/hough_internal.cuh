// hough_internal.cuh -- shared declarations of the CUDA path (libhough_b200.so).
//
// Product code.  Shares nothing with oracle/ (see DESIGN.md section 3): the arithmetic
// recipe of the vote (A1..A7) is restated here with explicit
// round-to-nearest intrinsics so that nvcc can neither fuse nor reorder it.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/hough.h"

// ---------------------------------------------------------------------------------
// Geometry of one tiled sweep over the hits (vote, hit-list count, hit-list fill).
// A CTA owns a tile of P phi0 centres x D d0 centres x all kappa bins in shared memory.
// ---------------------------------------------------------------------------------
struct SweepGeom {
    int P, D;            // tile extent in cells
    int cells_pad;       // P*D rounded up to a multiple of 32 (one lane per cell)
    int groups;          // cells_pad / 32 : warps needed to cover the tile once
    int split;           // S : warp sets that share the surviving hits of a chunk
    int threads;         // 32 * groups * split
    int chunk;           // hits staged per TMA bulk copy
    int tiles_phi, tiles_d0, n_tiles;
    int n_big, P_small;  // the first n_big phi0 slabs are P rows high, the rest P_small
    int tile_words;      // 32-bit words of the bin tile in shared memory
    int smem_bytes;      // dynamic shared memory of the kernel
    int no_phi_cull;     // tile spans too wide an angle for the interval test
};

// Geometry of the hit-list sweep (hough_lists.cu): a warp owns a sub-tile of SP x SD = 32
// cells, a CTA a super-tile of WP x WD sub-tiles and one of S segments of the event's hits.
#define LIST_WARPS 16
#define LIST_MAX_SEGMENTS 16
struct ListGeom {
    int SP, SD, WP, WD;
    int warps;           // warps per CTA (<= LIST_WARPS)
    int tiles_phi, tiles_d0;
    int S;               // hit segments (sub-lists per peak)
    int max_pk;          // bound on the peaks of one sub-tile
    int warp_bytes;      // shared memory per warp
    int smem_bytes;      // dynamic shared memory of the kernel
    int no_phi_cull_tile, no_phi_cull_sub;
};

// vote variants (hough_handle::mode; hough_device.cuh variant_bins)
#define VOTE_CENTRE 0
#define VOTE_LINE 1
#define VOTE_INTERVAL 2

// Device-side constant block handed to every kernel by value.
struct GridDev {
    int n_phi, n_d0, n_kappa;
    int L_min, phi_wrap;
    int pack;            // masks per 32-bit word of the vote tile: 2 (n_layers <= 16) or 1
    float klo, khi, inv_dk;
    float kabs;          // max(|klo|, |khi|)
    float d0_absmax;     // max |d0 centre|
    const float *sn, *cs;            // [n_phi]
    const float *sne, *cse;          // [n_phi + 1] sin / cos of the phi0 bin EDGES (interval voting)
    const float *d0c, *twod0, *d0sq; // [n_d0]
};

// constants of the fast bin path (hough_device.cuh approx_bin; built by hough_create).
// t = trunc(e * rcp(den) * c1 + c0) is the kappa-bin coordinate in 16.16 fixed point, shifted by delta.
#define APPROX_FRAC_BITS 16
struct ApproxBin {
    float c1, c0;
    uint32_t lim;  // n_kappa * 2^16 + 2 delta: (unsigned)t >= lim -> no vote
    uint32_t edge; // 2 delta: (t & 0xffff) < edge -> the exact recipe decides
    int ok;        // 0: the fast path is off for this grid
};

struct HitsDev {         // prepared hits, SoA, padded with non-voting entries to a chunk multiple
    const float *x, *y, *r2;
    const uint32_t *bit;
    uint32_t n;          // real hits
    uint32_t n_pad;      // padded length (multiple of the chunk size)
};

// Per-event index of the hits by (layer label, azimuth bin) for the peak-driven hit lists
// (hough_peaklists.cu).  Pseudo-layer n_layers holds the hits outside the index's numeric range.
struct HitIndexDev {
    int NA;                 // azimuth bins per layer (power of two, 256 .. 16384)
    int n_keys;             // (n_layers + 1) * NA
    uint32_t *bin_cnt;      // [n_keys] histogram of the event (k_prep); k_index_scan leaves it zero for the next event
    uint32_t *bin_cur;      // [n_keys] scatter cursor (k_index_scan: rank of the first hit of the key)
    uint32_t *bin_start;    // [n_keys + 1] rank of the first hit of a key
    uint32_t *layer_r;      // [2 * 33] per layer: max of ~bits(r) and max of bits(r) over the hits of THIS event
                            // (one of hough_handle::layer_r2's two blocks; k_prep fills it and empties the other)
    uint32_t *key;          // [max_hits_pad] key of hit h, 0xffffffff = not indexed (bad layer)
    float4 *rec;            // [max_hits_pad] the hits in key order: (x, y, r2, bits of the hit index)
};

// Device counters of one event (internal; copied into the caller's hough_counts).
struct DevCounters {
    unsigned long long n_votes;
    unsigned long long n_hit_entries;
    unsigned long long n_evals;
    unsigned long long n_list_evals;
    unsigned int n_peaks;
    unsigned int n_bad_hits;
    unsigned int flags;
};

// stages of one event, in launch order (HOUGH_OPT_STAGE_TIMING)
enum {
    ST_PREP = 0, ST_VOTE, ST_PEAK_SWEEP, ST_SCAN_ROWS, ST_COMPACT, ST_LIST_SWEEP, ST_SCAN_LENS,
    ST_PLACE_LISTS, ST_FINISH
};

struct hough_handle {
    hough_config cfg;
    double *radii;       // host copy
    int device, n_sms;
    GridDev g;
    ApproxBin ab;
    SweepGeom vote_geom;
    ListGeom list_geom;
    // workspace carve-up (device)
    uint32_t *acc;
    float *t_sn, *t_cs, *t_d0c, *t_twod0, *t_d0sq, *t_phic, *t_sne, *t_cse;
    int mode;            // vote variant: 0 closed form at bin centres, 1 straight line, 2 interval (hough_device.cuh)
    HitIndexDev ix;
    uint32_t *layer_r2[2]; // the two alternating blocks behind ix.layer_r
    int rbuf;              // the block of the current event
    float *hx, *hy, *hr2;
    uint32_t *hbit;
    // staging of the host entry points' hit arrays, one set per in-flight slot
    float *raw_x[HOUGH_MAX_SLOTS], *raw_y[HOUGH_MAX_SLOTS];
    int32_t *raw_layer[HOUGH_MAX_SLOTS];
    uint32_t max_hits_pad;
    uint32_t *flags;      // 1 bit per bin
    uint32_t *row_base;   // [n_rows + 1] exclusive scan of peaks per (i, j) row
    uint32_t *list_len;   // [cap_peaks * S_max] length of sub-list (peak, segment), then its start in the peak's list
    uint32_t *peak_len;   // [cap_peaks] list length per peak
    uint32_t *ent_sub, *ent_hit, *ent_idx; // [cap_hits] entries (sub-list, hit, place) of the list sweep
    unsigned long long *n_pairs; // entries emitted (lives in the per-hough_peaks reset region)
    unsigned long long *scan_status; // look-back words of the chained scans
    unsigned int *scan_ticket;       // [4]
    DevCounters *counters;   // the current event's counters = cnt2[cbuf]
    DevCounters *cnt2[2];    // two blocks: k_finish clears the one the next hough_vote will use
    int cbuf, next_clean;
    int peaks_dirty;         // a hough_peaks call did not get as far as its k_finish: clear its scratch by memset
    uint32_t scan_blocks_max;
    // sweep tile geometry of the peak kernel
    int pk_JW, pk_Li, pk_smem;
    // hough_submit_host / hough_collect_*: three-way overlap.  The library owns one
    // non-blocking stream for the host->device copies; per slot: h2d_ev = inputs landed, slot_ev = the
    // slot's computation (and the copy of its counters into slot_counts) is complete, copy_ev = its
    // results have reached the host.  slot_busy: 0 free, 1 submitted, 2 results being copied.
    cudaStream_t h2d_stream;
    int pipeline_ready;          // every resource of the pipeline exists (pipeline_init is all or nothing)
    cudaEvent_t h2d_ev[HOUGH_MAX_SLOTS], slot_ev[HOUGH_MAX_SLOTS], copy_ev[HOUGH_MAX_SLOTS];
    unsigned char slot_busy[HOUGH_MAX_SLOTS];
    hough_counts *slot_counts;   // pinned host memory, one block per slot
    // the hit index of the peak-driven lists is built on a stream of the library's own, beside the vote
    // kernel (it is needed by hough_peaks only): ix_fork = hits prepared, ix_join = index built
    cudaStream_t aux_stream;
    cudaEvent_t ix_fork, ix_join;
    int ix_pending;
    // state
    uint32_t n_hits;
    int voted;
    int fused_valid;     // HOUGH_OPT_FUSED_PEAKS: the last hough_vote left the interior cells' peak flags
    uint64_t launches;
    // HOUGH_OPT_STAGE_TIMING: ev[0] = start of hough_vote, ev[s + 1] = end of stage s
    int timing;
    cudaEvent_t ev[HOUGH_N_STAGES + 2];
    unsigned char ev_set[HOUGH_N_STAGES + 2];
};

static inline void stage_mark(hough_handle *h, int slot, cudaStream_t st)
{
    if (h->timing) {
        cudaEventRecord(h->ev[slot], st);
        h->ev_set[slot] = 1;
    }
}

// Programmatic dependent launch (sm_90+): a kernel launched with launch_pdl may be scheduled while its
// predecessor in the stream is still draining; it must call pdl_wait() before it touches anything the
// predecessor wrote (the wait returns when the predecessor has completed and flushed), and a kernel
// lets its successor in early with pdl_trigger().  Without the attribute both are no-ops.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <typename... KArgs, typename... Args>
static inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                     Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}
#endif

// kernels' host launchers (each enqueues on `st`, returns cudaGetLastError())
cudaError_t launch_prep(hough_handle *h, const float *x, const float *y, const int32_t *layer,
                        uint32_t n, cudaStream_t st);
cudaError_t launch_vote(hough_handle *h, cudaStream_t st);
cudaError_t launch_clear(hough_handle *h, cudaStream_t st);
cudaError_t launch_peak_sweep(hough_handle *h, cudaStream_t st);
cudaError_t launch_peak_cells(hough_handle *h, int edge_cells_only, cudaStream_t st);
cudaError_t launch_compact(hough_handle *h, const hough_peaks_out *out, cudaStream_t st);
cudaError_t launch_scan_rows(hough_handle *h, cudaStream_t st);
cudaError_t launch_scan_lens(hough_handle *h, const hough_peaks_out *out, cudaStream_t st);
cudaError_t launch_list_sweep(hough_handle *h, cudaStream_t st);
cudaError_t launch_index_build(hough_handle *h, cudaStream_t st);
cudaError_t launch_peak_lists(hough_handle *h, const hough_peaks_out *out, cudaStream_t st);
cudaError_t launch_copy_lists(hough_handle *h, const hough_peaks_out *out, cudaStream_t st);
cudaError_t launch_check_lists(hough_handle *h, const hough_peaks_out *out, cudaStream_t st);
cudaError_t launch_lists_generic(hough_handle *h, const hough_peaks_out *out, cudaStream_t st);
cudaError_t launch_place_lists(hough_handle *h, const hough_peaks_out *out, cudaStream_t st);
cudaError_t launch_finish_counts(hough_handle *h, const hough_peaks_out *out, int with_lists,
                                 cudaStream_t st);

int sweep_geom_init(const hough_handle *h, SweepGeom *g, int P, int D, int split, int fit_waves);
int list_geom_init(hough_handle *h);
int list_segments_bound(const hough_config *c);
int list_config_ok(const hough_config *c);
int hough_vote_max_smem(void);
// Raise (never lower) a kernel's dynamic shared-memory limit on the current device.
cudaError_t ensure_dynamic_smem(const void *kernel, int bytes);

#define HOUGH_CHUNK 512       // hits per staged chunk
#define HOUGH_SCAN_ITEMS 512  // items per block of the chained scan
