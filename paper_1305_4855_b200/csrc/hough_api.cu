// hough_api.cu -- the C ABI of include/hough.h: configuration checks, the bin-centre
// tables (A1), the workspace carve-up, hit preparation (a1) and the call sequences of
// hough_vote / hough_peaks.  No torch types, no exceptions, no global state.
#include <math.h>
#include <mutex>
#include <new>
#include <stdlib.h>
#include <string.h>

#include "hough_internal.cuh"

// ------------------------------------------------------------------ a1: hit preparation
// r2 = x*x + y*y (three roundings, A2), layer bit, bad-hit count; entries n..n_pad are
// non-voting padding so that the staged chunks are always whole.
__global__ void __launch_bounds__(256) k_prep(const float *__restrict__ x, const float *__restrict__ y,
                                              const int32_t *__restrict__ layer, uint32_t n,
                                              uint32_t n_pad, int n_layers, float *__restrict__ hx,
                                              float *__restrict__ hy, float *__restrict__ hr2,
                                              uint32_t *__restrict__ hbit, DevCounters *counters, HitIndexDev ix,
                                              uint32_t *__restrict__ layer_r_next)
{
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    bool bad = false;
    __shared__ uint32_t s_layer_r[2 * 33]; // the CTA's share of the per-layer radius range
    pdl_trigger(); // the vote kernel may set up its tile meanwhile (it waits before it reads the hits)
    if (threadIdx.x < 2 * 33) {
        s_layer_r[threadIdx.x] = 0u;
        if (blockIdx.x == 0)
            layer_r_next[threadIdx.x] = 0u; // the range is per event: the next event's block starts empty
    }
    __syncthreads();
    if (i < n) {
        float xv = x[i], yv = y[i];
        float pp = __fmul_rn(xv, xv);
        float qq = __fmul_rn(yv, yv);
        float r2 = __fadd_rn(pp, qq);
        int l = layer[i];
        bad = (l < 0) || (l >= n_layers);
        hx[i] = xv;
        hy[i] = yv;
        hr2[i] = r2;
        hbit[i] = bad ? 0u : (1u << l);
        // index key for the peak-driven hit lists (hough_peaklists.cu): (layer label, azimuth bin);
        // hits whose r^2 is outside [2^-40, 2^80] (or not finite) go to pseudo-layer n_layers
        uint32_t key = 0xffffffffu;
        if (!bad) {
            if (!((r2 >= 9.094947017729282e-13f) && (r2 <= 1.2089258196146292e24f))) {
                key = (uint32_t)(n_layers * ix.NA);
            } else {
                const float r = sqrtf(r2);
                const float na_scale = (float)ix.NA * 0.15915494309189535f;
                const int ab = ((int)floorf((atan2f(yv, xv) + 3.14159265358979f) * na_scale)) & (ix.NA - 1);
                key = (uint32_t)(l * ix.NA + ab);
                atomicMax(&s_layer_r[2 * l], ~__float_as_uint(r));
                atomicMax(&s_layer_r[2 * l + 1], __float_as_uint(r));
            }
            atomicAdd(&ix.bin_cnt[key], 1u);
        }
        ix.key[i] = key;
    } else if (i < n_pad) {
        hx[i] = 0.f;
        hy[i] = 0.f;
        hr2[i] = __int_as_float(0x7fc00000);
        hbit[i] = 0u;
    }
    unsigned b = __ballot_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0 && b)
        atomicAdd(&counters->n_bad_hits, (unsigned int)__popc(b));
    __syncthreads();
    if (threadIdx.x < 2 * 33 && s_layer_r[threadIdx.x] != 0u)
        atomicMax(&ix.layer_r[threadIdx.x], s_layer_r[threadIdx.x]);
}

cudaError_t launch_prep(hough_handle *h, const float *x, const float *y, const int32_t *layer, uint32_t n,
                        cudaStream_t st)
{
    uint32_t n_pad = ((n + HOUGH_CHUNK - 1) / HOUGH_CHUNK) * HOUGH_CHUNK;
    if (n_pad == 0)
        return cudaSuccess;
    // the key histogram starts from zero: k_index_scan leaves it so; where no index is built (vote variants,
    // HOUGH_OPT_LIST_SWEEP) nobody reads it, but it is cleared all the same
    if ((h->cfg.options & HOUGH_OPT_LIST_SWEEP) || h->mode != VOTE_CENTRE) {
        cudaError_t e = cudaMemsetAsync(h->ix.bin_cnt, 0, (size_t)h->ix.n_keys * 4, st);
        if (e != cudaSuccess)
            return e;
    }
    // per-layer radius range of THIS event: the two blocks alternate, k_prep fills one and empties the other
    // (both start empty: hough_create).  The previous event's list kernel has read its block by now (stream order).
    h->rbuf ^= 1;
    h->ix.layer_r = h->layer_r2[h->rbuf];
    k_prep<<<(n_pad + 255) / 256, 256, 0, st>>>(x, y, layer, n, n_pad, h->cfg.n_layers, h->hx, h->hy, h->hr2,
                                                h->hbit, h->counters, h->ix, h->layer_r2[h->rbuf ^ 1]);
    h->launches += 1;
    return cudaGetLastError();
}

// cudaFuncAttributeMaxDynamicSharedMemorySize holds the LAST value set, not the largest: a
// handle with a small tile must not take the limit away from a live handle with a large one.
// The attribute belongs to the (kernel, device) pair, i.e. to the process, so the record of
// what has been set is process-wide too; it is the library's only static state and is
// guarded by a mutex (handles may be created from different threads).
cudaError_t ensure_dynamic_smem(const void *kernel, int bytes)
{
    struct Entry {
        const void *fn;
        int device, bytes;
    };
    static Entry table[128];
    static int n_entries = 0;
    static std::mutex mu;
    int device = 0;
    cudaGetDevice(&device);
    std::lock_guard<std::mutex> lock(mu);
    Entry *e = nullptr;
    for (int i = 0; i < n_entries; ++i)
        if (table[i].fn == kernel && table[i].device == device)
            e = &table[i];
    if (e && e->bytes >= bytes)
        return cudaSuccess;
    cudaError_t rc = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (rc != cudaSuccess)
        return rc;
    if (!e && n_entries < 128) {
        e = &table[n_entries++];
        e->fn = kernel;
        e->device = device;
    }
    if (e)
        e->bytes = bytes;
    return cudaSuccess;
}

// ------------------------------------------------------------------ configuration
static int cfg_valid(const hough_config *c)
{
    if (!c || !c->layer_radius_cm)
        return 0;
    if (c->n_layers < 1 || c->n_layers > 32)
        return 0;
    for (int l = 0; l < c->n_layers; ++l)
        if (!(c->layer_radius_cm[l] > 0.0))
            return 0;
    if (c->n_phi < 1 || c->n_d0 < 1 || c->n_kappa < 32 || (c->n_kappa % 32) != 0)
        return 0;
    if (!(c->phi_max > c->phi_min) || !(c->kappa_max > c->kappa_min))
        return 0;
    if (c->n_d0 == 1 ? !(c->d0_max >= c->d0_min) : !(c->d0_max > c->d0_min))
        return 0;
    if (!isfinite(c->phi_min) || !isfinite(c->phi_max) || !isfinite(c->d0_min) || !isfinite(c->d0_max) ||
        !isfinite(c->kappa_min) || !isfinite(c->kappa_max))
        return 0;
    double bins = (double)c->n_phi * (double)c->n_d0 * (double)c->n_kappa;
    if (bins >= 4294967296.0)
        return 0;
    if (c->L_min < 1 || c->L_min > c->n_layers)
        return 0;
    if (c->phi_wrap != 0 && c->phi_wrap != 1)
        return 0;
    if (c->phi_wrap && c->n_phi < 3)
        return 0;
    if (c->cap_peaks < 1 || c->cap_hits < 1)
        return 0;
    if (c->tile_phi < 0 || c->tile_d0 < 0)
        return 0;
    if (c->n_kappa > 16384)
        return 0; // one cell row must fit a shared-memory tile
    // magnitudes the conservative cull's interval arithmetic cannot overflow on (hough.h)
    if (fabs(c->d0_min) > 1e15 || fabs(c->d0_max) > 1e15 || fabs(c->kappa_min) > 1e15 || fabs(c->kappa_max) > 1e15)
        return 0;
    if (!list_config_ok(c))
        return 0; // max_hits beyond what the hit-list segmentation supports
    if ((c->options & HOUGH_OPT_LINE) && (c->options & HOUGH_OPT_INTERVAL))
        return 0;
    if ((c->options & HOUGH_OPT_FUSED_PEAKS) && (c->n_layers > 16 || (c->options & HOUGH_OPT_UNPACKED)))
        return 0; // the fused test works on the two-masks-per-word tile
    if ((c->options & HOUGH_OPT_LINE) && c->n_d0 != 1)
        return 0; // the straight-line transform has two parameters (theta, rho)
    return 1;
}

struct Carve {
    size_t off;
    unsigned char *base;
    void *take(size_t bytes)
    {
        off = (off + 255) & ~(size_t)255;
        void *p = base ? base + off : nullptr;
        off += bytes;
        return p;
    }
};

static uint32_t pad_hits(uint32_t n)
{
    uint32_t p = ((n + HOUGH_CHUNK - 1) / HOUGH_CHUNK) * HOUGH_CHUNK;
    return p ? p : HOUGH_CHUNK;
}

// Lays the workspace out; with base == NULL only the size is computed.
static size_t carve_workspace(const hough_config *c, unsigned char *base, hough_handle *h)
{
    Carve cv{0, base};
    size_t n_bins = (size_t)c->n_phi * c->n_d0 * c->n_kappa;
    size_t n_rows = (size_t)c->n_phi * c->n_d0;
    uint32_t hp = pad_hits(c->max_hits);
    uint32_t sb = (uint32_t)((n_rows + HOUGH_SCAN_ITEMS - 1) / HOUGH_SCAN_ITEMS);
    const size_t n_sub = (size_t)c->cap_peaks * (size_t)list_segments_bound(c);
    uint32_t sb2 = (uint32_t)(((size_t)c->cap_peaks + HOUGH_SCAN_ITEMS - 1) / HOUGH_SCAN_ITEMS);
    if (sb2 > sb)
        sb = sb2;
    sb += 1;
    void *acc = cv.take(n_bins * 4);
    void *t_sn = cv.take((size_t)c->n_phi * 4), *t_cs = cv.take((size_t)c->n_phi * 4);
    void *t_d0c = cv.take((size_t)c->n_d0 * 4), *t_twod0 = cv.take((size_t)c->n_d0 * 4);
    void *t_d0sq = cv.take((size_t)c->n_d0 * 4);
    void *hx = cv.take((size_t)hp * 4), *hy = cv.take((size_t)hp * 4), *hr2 = cv.take((size_t)hp * 4);
    void *hbit = cv.take((size_t)hp * 4);
    void *rx[HOUGH_MAX_SLOTS], *ry[HOUGH_MAX_SLOTS], *rl[HOUGH_MAX_SLOTS];
    for (int s = 0; s < HOUGH_MAX_SLOTS; ++s) {
        rx[s] = cv.take((size_t)hp * 4);
        ry[s] = cv.take((size_t)hp * 4);
        rl[s] = cv.take((size_t)hp * 4);
    }
    void *flags = cv.take(n_bins / 8);
    void *row_base = cv.take((n_rows + 1) * 4);
    void *list_len = cv.take(n_sub * 4);
    void *peak_len = cv.take((size_t)c->cap_peaks * 4);
    void *ent_sub = cv.take((size_t)c->cap_hits * 4), *ent_hit = cv.take((size_t)c->cap_hits * 4);
    void *ent_idx = cv.take((size_t)c->cap_hits * 4);
    // hit index of the peak-driven lists: azimuth bins per layer ~ 5 x hits per layer (a window touches
    // the bins it overlaps, so finer bins mean fewer candidates), a power of two
    int NA = 256;
    while (NA < 16384 && (uint64_t)NA * (uint64_t)c->n_layers < 5ull * c->max_hits)
        NA <<= 1;
    const int n_keys = (c->n_layers + 1) * NA;
    void *t_phic = cv.take((size_t)c->n_phi * 4);
    void *t_sne = cv.take((size_t)(c->n_phi + 1) * 4), *t_cse = cv.take((size_t)(c->n_phi + 1) * 4);
    void *ix_cnt = cv.take((size_t)n_keys * 4 + 2 * 2 * 33 * 4); // histogram | two blocks of per-layer radius range (one memset)
    void *ix_start = cv.take((size_t)(n_keys + 1) * 4);
    void *ix_cur = cv.take((size_t)n_keys * 4);
    void *ix_key = cv.take((size_t)hp * 4);
    void *ix_rec = cv.take((size_t)hp * 16);
    // reset region: counters | tickets | status words (kept contiguous for one memset)
    void *counters = cv.take(256 + (size_t)2 * sb * 8);
    if (h) {
        h->acc = (uint32_t *)acc;
        h->t_sn = (float *)t_sn;
        h->t_cs = (float *)t_cs;
        h->t_d0c = (float *)t_d0c;
        h->t_twod0 = (float *)t_twod0;
        h->t_d0sq = (float *)t_d0sq;
        h->hx = (float *)hx;
        h->hy = (float *)hy;
        h->hr2 = (float *)hr2;
        h->hbit = (uint32_t *)hbit;
        for (int s = 0; s < HOUGH_MAX_SLOTS; ++s) {
            h->raw_x[s] = (float *)rx[s];
            h->raw_y[s] = (float *)ry[s];
            h->raw_layer[s] = (int32_t *)rl[s];
        }
        h->max_hits_pad = hp;
        h->flags = (uint32_t *)flags;
        h->row_base = (uint32_t *)row_base;
        h->list_len = (uint32_t *)list_len;
        h->peak_len = (uint32_t *)peak_len;
        h->ent_sub = (uint32_t *)ent_sub;
        h->ent_hit = (uint32_t *)ent_hit;
        h->ent_idx = (uint32_t *)ent_idx;
        h->t_phic = (float *)t_phic;
        h->t_sne = (float *)t_sne;
        h->t_cse = (float *)t_cse;
        h->ix.NA = NA;
        h->ix.n_keys = n_keys;
        h->ix.bin_cnt = (uint32_t *)ix_cnt;
        h->layer_r2[0] = (uint32_t *)ix_cnt + n_keys;
        h->layer_r2[1] = h->layer_r2[0] + 2 * 33;
        h->ix.layer_r = h->layer_r2[0];
        h->rbuf = 0;
        h->ix.bin_start = (uint32_t *)ix_start;
        h->ix.bin_cur = (uint32_t *)ix_cur;
        h->ix.key = (uint32_t *)ix_key;
        h->ix.rec = (float4 *)ix_rec;
        h->n_pairs = (unsigned long long *)((unsigned char *)counters + 128);
        h->counters = (DevCounters *)counters;
        h->cnt2[0] = (DevCounters *)counters;
        h->cnt2[1] = (DevCounters *)((unsigned char *)counters + 192);
        h->scan_ticket = (unsigned int *)((unsigned char *)counters + 64);
        h->scan_status = (unsigned long long *)((unsigned char *)counters + 256);
        h->scan_blocks_max = sb;
    }
    return (cv.off + 255) & ~(size_t)255;
}

size_t hough_workspace_bytes(const hough_config *cfg)
{
    if (!cfg_valid(cfg))
        return 0;
    return carve_workspace(cfg, nullptr, nullptr);
}

// Tile shapes.  Defaults aim at two resident CTAs per SM (<= ~113 KB of shared memory
// each); cfg.tile_phi / tile_d0 override the vote tile.  All configuration comes from
// hough_config (no environment variables).
static int choose_geometry(hough_handle *h)
{
    const hough_config &c = h->cfg;
    const int nk = c.n_kappa;
    const int budget = 115 * 1024;
    const int staging = 4 * 1536 * 4 + (1536 + 8) * 16 + 1024; // hough_sweep.cu: VOTE_CHUNK hits staged + survivors
    // vote
    {
        int cell_bytes = nk * 4 / h->g.pack;
        int D = c.tile_d0 > 0 ? c.tile_d0 : (c.n_d0 < 8 ? c.n_d0 : 8);
        if (D > c.n_d0)
            D = c.n_d0;
        int P = c.tile_phi;
        if (P <= 0) {
            // whole cell groups (32 lanes) only: a padded group costs a full group of
            // shared memory and lanes (fine grid: 11 x 8 cells = 96 KB + staging -> 1 CTA/SM,
            // 41 % issue; 8 x 8 = 64 KB -> 2 CTAs/SM)
            int cells = ((budget - staging) / cell_bytes / 32) * 32;
            if (cells < 32)
                cells = (budget - staging) / cell_bytes;
            P = cells / D;
            if (P > 32)
                P = 32;
            if (P >= 16)
                P = (P / 8) * 8;
        }
        if (P < 1)
            P = 1;
        if (P > c.n_phi)
            P = c.n_phi;
        int groups = (P * D + 31) / 32;
        int split = 512 / (32 * groups);
        if (split < 1)
            split = 1;
        if (split > 8)
            split = 8;
        while (split > 1 && 32 * groups * split > 1024)
            --split;
        const int fit = c.tile_phi == 0 ? 1 : 0;
        if (!sweep_geom_init(h, &h->vote_geom, P, D, split, fit)) {
            // fall back to the smallest tile
            if (!sweep_geom_init(h, &h->vote_geom, 1, 1, 4, 0))
                return 0;
        }
    }
    // hit lists: warp sub-tiles, hit segments (hough_lists.cu)
    if (!list_geom_init(h))
        return 0;
    // peak sweep: JW warps x 2 rows per thread and CTA (2 of the rows are halo rows), Li phi0
    // planes per CTA
    {
        const int RJ = 2;
        int JW = 8;
        int need = (c.n_d0 + 2 + RJ - 1) / RJ; // warps that cover every row plus the two halo rows
        if (JW > need)
            JW = need;
        if (JW * RJ < 3)
            JW = (3 + RJ - 1) / RJ;
        // planes per CTA: 24 (8 % halo planes) when that still leaves >= 4 waves of CTAs, else 16
        const long long ctas24 = (long long)((c.n_kappa + 255) / 256) * ((c.n_d0 + RJ * JW - 3) / (RJ * JW - 2)) *
                                 ((c.n_phi + 23) / 24);
        int Li = ctas24 >= 8LL * h->n_sms ? 24 : 16;
        if (Li > c.n_phi)
            Li = c.n_phi;
        if (Li < 1)
            Li = 1;
        h->pk_JW = JW;
        h->pk_Li = Li;
        h->pk_smem = 2 * (RJ * JW) * 32 * 16;
    }
    return 1;
}

// Constants and admissibility of the fast bin path (hough_device.cuh approx_bin; DESIGN.md
// 4.5).  With klo, khi, inv_dk the fp32 constants of A1 taken as reals, the estimate is
//   t = trunc( e * rcp(den) * c1 + c0 ),  c1 = 2 inv_dk 2^16 (exact),  c0 = RN(-klo inv_dk 2^16 + delta).
// One binary32 rounding of a coordinate below n_kappa * 2^16 is at most U = n_kappa / 256
// steps.  Error budget against the exact qf * 2^16: E = (7A + 3) U + 1 with A = K / W; khi's
// own coordinate is within (2A + 1) U of n_kappa * 2^16; delta = ceil((12 A + 8) max(U, 1)).
static void approx_bin_init(hough_handle *h, const float *d0c, int nd)
{
    ApproxBin &ab = h->ab;
    memset(&ab, 0, sizeof(ab));
    if (h->cfg.options & HOUGH_OPT_EXACT_ONLY)
        return;
    const double klo = (double)h->g.klo, khi = (double)h->g.khi, inv = (double)h->g.inv_dk;
    const int nk = h->g.n_kappa;
    const double W = khi - klo, K = fmax(fabs(klo), fabs(khi));
    if (!(W > 0.0) || !(inv > 0.0) || K > 1048576.0 || W / nk < ldexp(1.0, -40))
        return;
    for (int j = 0; j < nd; ++j) { // den = r2 - 2 d0 s + d0^2 must be 0 or normal with a normal reciprocal
        const double a = fabs((double)d0c[j]);
        if (a != 0.0 && (a < ldexp(1.0, -20) || a > 1048576.0))
            return;
    }
    const double steps = 65536.0, U = fmax(nk / 256.0, 1.0);
    const double delta = ceil((12.0 * K / W + 8.0) * U);
    if (16.0 * delta > steps)
        return; // more than 1/8 of every bin would fall back to the exact recipe anyway
    // the bin coordinates of klo and khi must sit where the budget assumes them
    if (fabs((khi - klo) * inv - nk) * steps > 0.25 * delta)
        return;
    ab.c1 = (float)ldexp(inv, APPROX_FRAC_BITS + 1);
    ab.c0 = (float)(-klo * inv * steps + delta);
    ab.lim = (uint32_t)((double)nk * steps + 2.0 * delta);
    ab.edge = (uint32_t)(2.0 * delta);
    ab.ok = isfinite(ab.c1) && isfinite(ab.c0) ? 1 : 0;
}

int hough_create(const hough_config *cfg, void *workspace, size_t workspace_bytes, hough_handle **out)
{
    if (!out)
        return HOUGH_EINVAL;
    *out = nullptr;
    if (!cfg_valid(cfg) || !workspace)
        return HOUGH_EINVAL;
    if (((uintptr_t)workspace & 255) != 0)
        return HOUGH_EINVAL;
    size_t need = carve_workspace(cfg, nullptr, nullptr);
    if (workspace_bytes < need)
        return HOUGH_ENOMEM;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev) {
        cudaGetLastError();
        return HOUGH_ECUDA;
    }
    if (cudaSetDevice(cfg->device) != cudaSuccess)
        return HOUGH_ECUDA;
    hough_handle *h = new (std::nothrow) hough_handle();
    if (!h)
        return HOUGH_ENOMEM;
    memset(h, 0, sizeof(*h));
    h->cfg = *cfg;
    h->radii = (double *)malloc(sizeof(double) * cfg->n_layers);
    memcpy(h->radii, cfg->layer_radius_cm, sizeof(double) * cfg->n_layers);
    h->cfg.layer_radius_cm = h->radii;
    h->device = cfg->device;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess) {
        hough_destroy(h);
        return HOUGH_ECUDA;
    }
    h->n_sms = prop.multiProcessorCount;
    if (cfg->options & HOUGH_OPT_STAGE_TIMING) {
        for (int s = 0; s < HOUGH_N_STAGES + 2; ++s)
            if (cudaEventCreate(&h->ev[s]) != cudaSuccess) {
                cudaGetLastError();
                hough_destroy(h);
                return HOUGH_ECUDA;
            }
        h->timing = 1;
    }
    carve_workspace(cfg, (unsigned char *)workspace, h);
    if (cudaStreamCreateWithFlags(&h->aux_stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ix_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ix_join, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        hough_destroy(h);
        return HOUGH_ECUDA;
    }

    // A1: bin centres in fp64, one rounding to fp32
    const int np = cfg->n_phi, nd = cfg->n_d0;
    float *sn = (float *)malloc(sizeof(float) * np), *cs = (float *)malloc(sizeof(float) * np);
    float *d0c = (float *)malloc(sizeof(float) * nd), *twod0 = (float *)malloc(sizeof(float) * nd);
    float *d0sq = (float *)malloc(sizeof(float) * nd);
    float *phf = (float *)malloc(sizeof(float) * np);
    for (int i = 0; i < np; ++i) {
        double phic = cfg->phi_min + ((double)i + 0.5) * (cfg->phi_max - cfg->phi_min) / (double)np;
        sn[i] = (float)sin(phic);
        cs[i] = (float)cos(phic);
        phf[i] = (float)remainder(phic, 6.283185307179586); // the angle itself, in [-pi, pi] (azimuth windows)
    }
    // E2 (interval voting): the phi0 bin EDGES, the same way
    float *sne = (float *)malloc(sizeof(float) * (np + 1)), *cse = (float *)malloc(sizeof(float) * (np + 1));
    for (int i = 0; i <= np; ++i) {
        double pe = cfg->phi_min + (double)i * (cfg->phi_max - cfg->phi_min) / (double)np;
        sne[i] = (float)sin(pe);
        cse[i] = (float)cos(pe);
    }
    h->mode = (cfg->options & HOUGH_OPT_LINE) ? VOTE_LINE : (cfg->options & HOUGH_OPT_INTERVAL) ? VOTE_INTERVAL : VOTE_CENTRE;
    float d0abs = 0.f;
    for (int j = 0; j < nd; ++j) {
        volatile float c0 = (float)(cfg->d0_min + ((double)j + 0.5) * (cfg->d0_max - cfg->d0_min) / (double)nd);
        volatile float two = 2.0f * c0;
        volatile float sq = c0 * c0; // one binary32 multiply (volatile: no contraction, no excess precision)
        d0c[j] = c0;
        twod0[j] = two;
        d0sq[j] = sq;
        if (fabsf(c0) > d0abs)
            d0abs = fabsf(c0);
    }
    GridDev &g = h->g;
    g.n_phi = np;
    g.n_d0 = nd;
    g.n_kappa = cfg->n_kappa;
    g.L_min = cfg->L_min;
    g.phi_wrap = cfg->phi_wrap;
    g.pack = (cfg->n_layers <= 16 && !(cfg->options & HOUGH_OPT_UNPACKED)) ? 2 : 1;
    g.klo = (float)cfg->kappa_min;
    g.khi = (float)cfg->kappa_max;
    g.inv_dk = (float)((double)cfg->n_kappa / (cfg->kappa_max - cfg->kappa_min));
    g.kabs = fmaxf(fabsf(g.klo), fabsf(g.khi));
    g.d0_absmax = d0abs;
    g.sn = h->t_sn;
    g.cs = h->t_cs;
    g.sne = h->t_sne;
    g.cse = h->t_cse;
    g.d0c = h->t_d0c;
    g.twod0 = h->t_twod0;
    g.d0sq = h->t_d0sq;
    approx_bin_init(h, d0c, nd);
    if (h->mode != VOTE_CENTRE)
        h->ab.ok = 0; // the variants evaluate the exact recipe only
    int ok = 1;
    ok &= cudaMemcpy(h->t_sne, sne, sizeof(float) * (np + 1), cudaMemcpyHostToDevice) == cudaSuccess;
    ok &= cudaMemcpy(h->t_cse, cse, sizeof(float) * (np + 1), cudaMemcpyHostToDevice) == cudaSuccess;
    free(sne);
    free(cse);
    ok &= cudaMemcpy(h->t_sn, sn, sizeof(float) * np, cudaMemcpyHostToDevice) == cudaSuccess;
    ok &= cudaMemcpy(h->t_cs, cs, sizeof(float) * np, cudaMemcpyHostToDevice) == cudaSuccess;
    ok &= cudaMemcpy(h->t_phic, phf, sizeof(float) * np, cudaMemcpyHostToDevice) == cudaSuccess;
    free(phf);
    ok &= cudaMemcpy(h->t_d0c, d0c, sizeof(float) * nd, cudaMemcpyHostToDevice) == cudaSuccess;
    ok &= cudaMemcpy(h->t_twod0, twod0, sizeof(float) * nd, cudaMemcpyHostToDevice) == cudaSuccess;
    ok &= cudaMemcpy(h->t_d0sq, d0sq, sizeof(float) * nd, cudaMemcpyHostToDevice) == cudaSuccess;
    ok &= cudaMemset(h->counters, 0, 256 + (size_t)2 * h->scan_blocks_max * 8) == cudaSuccess;
    ok &= cudaMemset(h->ix.bin_cnt, 0, (size_t)h->ix.n_keys * 4 + 2 * 2 * 33 * 4) == cudaSuccess;
    h->cbuf = 0;
    h->next_clean = 1;
    free(sn);
    free(cs);
    free(d0c);
    free(twod0);
    free(d0sq);
    if (!ok) {
        cudaGetLastError();
        hough_destroy(h);
        return HOUGH_ECUDA;
    }
    if (!choose_geometry(h)) {
        hough_destroy(h);
        return HOUGH_EINVAL;
    }
    if (cudaDeviceSynchronize() != cudaSuccess) {
        hough_destroy(h);
        return HOUGH_ECUDA;
    }
    *out = h;
    return HOUGH_OK;
}

void hough_destroy(hough_handle *h)
{
    if (!h)
        return;
    if (h->timing)
        for (int s = 0; s < HOUGH_N_STAGES + 2; ++s)
            if (h->ev[s])
                cudaEventDestroy(h->ev[s]);
    for (int s = 0; s < HOUGH_MAX_SLOTS; ++s) {
        if (h->slot_ev[s])
            cudaEventDestroy(h->slot_ev[s]);
        if (h->h2d_ev[s])
            cudaEventDestroy(h->h2d_ev[s]);
        if (h->copy_ev[s])
            cudaEventDestroy(h->copy_ev[s]);
    }
    if (h->h2d_stream)
        cudaStreamDestroy(h->h2d_stream);
    if (h->aux_stream)
        cudaStreamDestroy(h->aux_stream);
    if (h->ix_fork)
        cudaEventDestroy(h->ix_fork);
    if (h->ix_join)
        cudaEventDestroy(h->ix_join);
    if (h->slot_counts)
        cudaFreeHost(h->slot_counts);
    free(h->radii);
    delete h;
}

#define CK(expr)                                                                                   \
    do {                                                                                           \
        cudaError_t e__ = (expr);                                                                  \
        if (e__ != cudaSuccess) {                                                                  \
            cudaGetLastError();                                                                    \
            return HOUGH_ECUDA;                                                                    \
        }                                                                                          \
    } while (0)

int hough_vote(hough_handle *h, const float *x, const float *y, const int32_t *layer, uint32_t n,
               void *cuda_stream)
{
    if (!h)
        return HOUGH_EINVAL;
    if (n > h->cfg.max_hits)
        return HOUGH_EINVAL;
    if (n > 0 && (!x || !y || !layer))
        return HOUGH_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    h->n_hits = n;
    if (h->timing)
        memset(h->ev_set, 0, sizeof(h->ev_set));
    if (h->ix_pending) { // an index build of a vote that no hough_peaks followed: k_prep resets its arrays
        CK(cudaStreamWaitEvent(st, h->ix_join, 0));
        h->ix_pending = 0;
    }
    stage_mark(h, 0, st);
    // the event's counters: the block the previous hough_peaks cleared (k_finish), else a memset
    h->cbuf ^= 1;
    h->counters = h->cnt2[h->cbuf];
    if (!h->next_clean)
        CK(cudaMemsetAsync(h->counters, 0, 64, st));
    h->next_clean = 0;
    CK(launch_prep(h, x, y, layer, n, st));
    if (!(h->cfg.options & HOUGH_OPT_LIST_SWEEP) && h->mode == VOTE_CENTRE && n > 0) {
        // beside the vote kernel, on the library's own stream (joined before the list kernel)
        CK(cudaEventRecord(h->ix_fork, st));
        CK(cudaStreamWaitEvent(h->aux_stream, h->ix_fork, 0));
        CK(launch_index_build(h, h->aux_stream));
        CK(cudaEventRecord(h->ix_join, h->aux_stream));
        h->ix_pending = 1;
    }
    stage_mark(h, ST_PREP + 1, st);
    CK(launch_vote(h, st));
    stage_mark(h, ST_VOTE + 1, st);
    h->voted = 1;
    return HOUGH_OK;
}

static int peaks_common(hough_handle *h, const hough_peaks_out *out, void *cuda_stream, int with_lists)
{
    if (!h || !out || !out->bin || !out->mask || !out->counts)
        return HOUGH_EINVAL;
    if (with_lists && (!out->hit_offset || !out->hit_index))
        return HOUGH_EINVAL;
    if (!h->voted)
        return HOUGH_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // tickets, work counter and look-back words were cleared by the previous call's k_finish -- unless that
    // call failed on the way
    if (h->peaks_dirty)
        CK(cudaMemsetAsync((unsigned char *)h->cnt2[0] + 64, 0, 128, st));
    if (h->peaks_dirty)
        CK(cudaMemsetAsync(h->scan_status, 0, (size_t)2 * h->scan_blocks_max * 8, st));
    h->peaks_dirty = 1;
    // a5: the streaming sweep; or, fused variant, only the cells on the vote tiles' edges (the others were
    // flagged by hough_vote's kernel -- not after hough_set_accumulator, which leaves no such flags)
    if ((h->cfg.options & HOUGH_OPT_FUSED_PEAKS) && h->fused_valid)
        CK(launch_peak_cells(h, 1, st));
    else if (h->cfg.options & HOUGH_OPT_CELL_PEAKS)
        CK(launch_peak_cells(h, 0, st));
    else
        CK(launch_peak_sweep(h, st));
    stage_mark(h, ST_PEAK_SWEEP + 1, st);
    CK(launch_scan_rows(h, st));
    stage_mark(h, ST_SCAN_ROWS + 1, st);
    CK(launch_compact(h, out, st));
    stage_mark(h, ST_COMPACT + 1, st);
    if (h->ix_pending) {
        CK(cudaStreamWaitEvent(st, h->ix_join, 0));
        h->ix_pending = 0;
    }
    if (with_lists) {
        // the vote variants (f3) take the generic lists: one warp per peak over all hits
        const int sweep = (h->cfg.options & HOUGH_OPT_LIST_SWEEP) && h->mode == VOTE_CENTRE ? 1 : 0;
        CK(h->mode != VOTE_CENTRE ? launch_lists_generic(h, out, st)
                                  : sweep ? launch_list_sweep(h, st) : launch_peak_lists(h, out, st));
        stage_mark(h, ST_LIST_SWEEP + 1, st);
        CK(launch_scan_lens(h, out, st));
        stage_mark(h, ST_SCAN_LENS + 1, st);
        CK(sweep ? launch_place_lists(h, out, st) : launch_copy_lists(h, out, st));
        stage_mark(h, ST_PLACE_LISTS + 1, st);
    }
    CK(launch_finish_counts(h, out, with_lists, st));
    h->next_clean = 1;
    h->peaks_dirty = 0;
    stage_mark(h, ST_FINISH + 1, st);
    if (with_lists && (h->cfg.options & HOUGH_OPT_CHECK_LISTS))
        CK(launch_check_lists(h, out, st)); // after k_finish: it ORs into the counters the caller reads
    return HOUGH_OK;
}

int hough_check_lists(hough_handle *h, const hough_peaks_out *out, void *cuda_stream)
{
    if (!h || !out || !out->mask || !out->counts || !out->hit_offset || !out->hit_index)
        return HOUGH_EINVAL;
    if (!h->voted)
        return HOUGH_ESTATE;
    CK(launch_check_lists(h, out, (cudaStream_t)cuda_stream));
    return HOUGH_OK;
}

int hough_peaks(hough_handle *h, const hough_peaks_out *out, void *cuda_stream)
{
    return peaks_common(h, out, cuda_stream, 1);
}

int hough_peaks_only(hough_handle *h, const hough_peaks_out *out, void *cuda_stream)
{
    return peaks_common(h, out, cuda_stream, 0);
}

const uint32_t *hough_accumulator(const hough_handle *h) { return h ? h->acc : nullptr; }

int hough_clear(hough_handle *h, void *cuda_stream)
{
    if (!h)
        return HOUGH_EINVAL;
    CK(launch_clear(h, (cudaStream_t)cuda_stream));
    return HOUGH_OK;
}

int hough_peak_sweep(hough_handle *h, void *cuda_stream)
{
    if (!h)
        return HOUGH_EINVAL;
    CK(launch_peak_sweep(h, (cudaStream_t)cuda_stream));
    return HOUGH_OK;
}

int hough_set_accumulator(hough_handle *h, const uint32_t *acc_dev, void *cuda_stream)
{
    if (!h || !acc_dev)
        return HOUGH_EINVAL;
    size_t n_bins = (size_t)h->g.n_phi * h->g.n_d0 * h->g.n_kappa;
    CK(cudaMemcpyAsync(h->acc, acc_dev, n_bins * 4, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
    CK(cudaMemsetAsync(h->counters, 0, 64, (cudaStream_t)cuda_stream));
    h->n_hits = 0;
    h->voted = 1;
    h->fused_valid = 0;
    return HOUGH_OK;
}

int hough_process_host(hough_handle *h, const float *x, const float *y, const int32_t *layer, uint32_t n,
                       const hough_peaks_out *dev, const hough_host_out *host, void *cuda_stream)
{
    if (!h || !dev || !host || !host->counts || !host->bin || !host->mask || !host->hit_offset)
        return HOUGH_EINVAL;
    if (n > h->cfg.max_hits || (n > 0 && (!x || !y || !layer)))
        return HOUGH_EINVAL;
    if (h->slot_busy[0]) // this call stages its hits where pipeline slot 0 does
        return HOUGH_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (n > 0) {
        CK(cudaMemcpyAsync(h->raw_x[0], x, (size_t)n * 4, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(h->raw_y[0], y, (size_t)n * 4, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(h->raw_layer[0], layer, (size_t)n * 4, cudaMemcpyHostToDevice, st));
    }
    int rc = hough_vote(h, h->raw_x[0], h->raw_y[0], h->raw_layer[0], n, cuda_stream);
    if (rc != HOUGH_OK)
        return rc;
    rc = hough_peaks(h, dev, cuda_stream);
    if (rc != HOUGH_OK)
        return rc;
    CK(cudaMemcpyAsync(host->counts, dev->counts, sizeof(hough_counts), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    uint64_t np = host->counts->n_peaks < h->cfg.cap_peaks ? host->counts->n_peaks : h->cfg.cap_peaks;
    uint64_t ne = host->counts->n_hit_entries < h->cfg.cap_hits ? host->counts->n_hit_entries : h->cfg.cap_hits;
    if (np > 0) {
        CK(cudaMemcpyAsync(host->bin, dev->bin, np * 4, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(host->mask, dev->mask, np * 4, cudaMemcpyDeviceToHost, st));
    }
    CK(cudaMemcpyAsync(host->hit_offset, dev->hit_offset, (np + 1) * 8, cudaMemcpyDeviceToHost, st));
    if (host->hit_index16 && dev->hit_index16 && (host->counts->flags & HOUGH_INDEX16)) {
        if (ne > 0)
            CK(cudaMemcpyAsync(host->hit_index16, dev->hit_index16, ne * 2, cudaMemcpyDeviceToHost, st));
    } else if (host->hit_index && ne > 0) {
        CK(cudaMemcpyAsync(host->hit_index, dev->hit_index, ne * 4, cudaMemcpyDeviceToHost, st));
    }
    CK(cudaStreamSynchronize(st));
    return HOUGH_OK;
}

// Lazily created resources of the pipelined host entry points.
// All or nothing: `pipeline_ready` is set only when every resource exists; a failure on the way
// releases what was created, so that the next call starts over instead of using half of them.
static void pipeline_release(hough_handle *h)
{
    for (int s = 0; s < HOUGH_MAX_SLOTS; ++s) {
        if (h->slot_ev[s])
            cudaEventDestroy(h->slot_ev[s]);
        if (h->h2d_ev[s])
            cudaEventDestroy(h->h2d_ev[s]);
        if (h->copy_ev[s])
            cudaEventDestroy(h->copy_ev[s]);
        h->slot_ev[s] = h->h2d_ev[s] = h->copy_ev[s] = nullptr;
    }
    if (h->h2d_stream)
        cudaStreamDestroy(h->h2d_stream);
    h->h2d_stream = nullptr;
    if (h->slot_counts)
        cudaFreeHost(h->slot_counts);
    h->slot_counts = nullptr;
    h->pipeline_ready = 0;
}

static int pipeline_init(hough_handle *h)
{
    if (h->pipeline_ready)
        return HOUGH_OK;
    bool ok = cudaStreamCreateWithFlags(&h->h2d_stream, cudaStreamNonBlocking) == cudaSuccess;
    for (int s = 0; ok && s < HOUGH_MAX_SLOTS; ++s) {
        ok = ok && cudaEventCreateWithFlags(&h->h2d_ev[s], cudaEventDisableTiming) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&h->slot_ev[s], cudaEventDisableTiming) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&h->copy_ev[s], cudaEventDisableTiming) == cudaSuccess;
    }
    ok = ok && cudaMallocHost((void **)&h->slot_counts, sizeof(hough_counts) * HOUGH_MAX_SLOTS) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        pipeline_release(h);
        return HOUGH_ECUDA;
    }
    h->pipeline_ready = 1;
    return HOUGH_OK;
}

int hough_submit_host(hough_handle *h, const float *x, const float *y, const int32_t *layer, uint32_t n,
                      const hough_peaks_out *dev, int32_t slot, void *cuda_stream)
{
    if (!h || !dev || slot < 0 || slot >= HOUGH_MAX_SLOTS)
        return HOUGH_EINVAL;
    if (n > h->cfg.max_hits || (n > 0 && (!x || !y || !layer)))
        return HOUGH_EINVAL;
    if (h->slot_busy[slot])
        return HOUGH_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = pipeline_init(h);
    if (rc != HOUGH_OK)
        return rc;
    // inputs: on the library's copy-in stream, into the slot's own staging arrays (free: the slot's
    // previous event has been collected, so its k_prep has long read them), ahead of whatever the
    // compute stream is still doing for the previous event
    if (n > 0) {
        CK(cudaMemcpyAsync(h->raw_x[slot], x, (size_t)n * 4, cudaMemcpyHostToDevice, h->h2d_stream));
        CK(cudaMemcpyAsync(h->raw_y[slot], y, (size_t)n * 4, cudaMemcpyHostToDevice, h->h2d_stream));
        CK(cudaMemcpyAsync(h->raw_layer[slot], layer, (size_t)n * 4, cudaMemcpyHostToDevice, h->h2d_stream));
    }
    CK(cudaEventRecord(h->h2d_ev[slot], h->h2d_stream));
    CK(cudaStreamWaitEvent(st, h->h2d_ev[slot], 0));
    rc = hough_vote(h, h->raw_x[slot], h->raw_y[slot], h->raw_layer[slot], n, cuda_stream);
    if (rc != HOUGH_OK)
        return rc;
    rc = hough_peaks(h, dev, cuda_stream);
    if (rc != HOUGH_OK)
        return rc;
    // the 48 bytes of counters follow the computation on its own stream, so that the collecting side
    // knows the sizes of the results without a round trip of its own
    CK(cudaMemcpyAsync(&h->slot_counts[slot], dev->counts, sizeof(hough_counts), cudaMemcpyDeviceToHost, st));
    CK(cudaEventRecord(h->slot_ev[slot], st));
    h->slot_busy[slot] = 1;
    return HOUGH_OK;
}

int hough_collect_begin(hough_handle *h, const hough_peaks_out *dev, const hough_host_out *host, int32_t slot,
                        void *copy_stream)
{
    if (!h || !dev || !host || !host->counts || !host->bin || !host->mask || !host->hit_offset || slot < 0 ||
        slot >= HOUGH_MAX_SLOTS)
        return HOUGH_EINVAL;
    if (h->slot_busy[slot] != 1)
        return HOUGH_ESTATE;
    cudaStream_t st = (cudaStream_t)copy_stream;
    CK(cudaEventSynchronize(h->slot_ev[slot]));
    const hough_counts c = h->slot_counts[slot];
    *host->counts = c;
    const uint64_t np = c.n_peaks < h->cfg.cap_peaks ? c.n_peaks : h->cfg.cap_peaks;
    const uint64_t ne = c.n_hit_entries < h->cfg.cap_hits ? c.n_hit_entries : h->cfg.cap_hits;
    if (np > 0) {
        CK(cudaMemcpyAsync(host->bin, dev->bin, np * 4, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(host->mask, dev->mask, np * 4, cudaMemcpyDeviceToHost, st));
    }
    CK(cudaMemcpyAsync(host->hit_offset, dev->hit_offset, (np + 1) * 8, cudaMemcpyDeviceToHost, st));
    if (host->hit_index16 && dev->hit_index16 && (host->counts->flags & HOUGH_INDEX16)) {
        if (ne > 0)
            CK(cudaMemcpyAsync(host->hit_index16, dev->hit_index16, ne * 2, cudaMemcpyDeviceToHost, st));
    } else if (host->hit_index && ne > 0) {
        CK(cudaMemcpyAsync(host->hit_index, dev->hit_index, ne * 4, cudaMemcpyDeviceToHost, st));
    }
    CK(cudaEventRecord(h->copy_ev[slot], st));
    h->slot_busy[slot] = 2;
    return HOUGH_OK;
}

int hough_collect_end(hough_handle *h, int32_t slot)
{
    if (!h || slot < 0 || slot >= HOUGH_MAX_SLOTS)
        return HOUGH_EINVAL;
    if (h->slot_busy[slot] != 2)
        return HOUGH_ESTATE;
    CK(cudaEventSynchronize(h->copy_ev[slot]));
    h->slot_busy[slot] = 0;
    return HOUGH_OK;
}

int hough_collect_host(hough_handle *h, const hough_peaks_out *dev, const hough_host_out *host, int32_t slot,
                       void *copy_stream)
{
    const int rc = hough_collect_begin(h, dev, host, slot, copy_stream);
    return rc != HOUGH_OK ? rc : hough_collect_end(h, slot);
}

int hough_query(const hough_handle *h, int32_t *tile_phi, int32_t *tile_d0, int32_t *n_tiles,
                int32_t *threads, int32_t *smem_bytes, int32_t *n_sms)
{
    if (!h)
        return HOUGH_EINVAL;
    if (tile_phi)
        *tile_phi = h->vote_geom.P;
    if (tile_d0)
        *tile_d0 = h->vote_geom.D;
    if (n_tiles)
        *n_tiles = h->vote_geom.n_tiles;
    if (threads)
        *threads = h->vote_geom.threads;
    if (smem_bytes)
        *smem_bytes = h->vote_geom.smem_bytes;
    if (n_sms)
        *n_sms = h->n_sms;
    return HOUGH_OK;
}

uint64_t hough_launch_count(const hough_handle *h) { return h ? h->launches : 0; }

static const char *const k_stage_names[HOUGH_N_STAGES] = {
    "prep", "vote", "peak_sweep", "scan_rows", "compact", "lists", "scan_lens", "place_lists",
    "finish"};

const char *hough_stage_name(int stage)
{
    return (stage >= 0 && stage < HOUGH_N_STAGES) ? k_stage_names[stage] : nullptr;
}

int hough_stage_times(hough_handle *h, float *ms, int cap)
{
    if (!h || !ms || cap < 1)
        return HOUGH_EINVAL;
    if (!h->timing)
        return HOUGH_ESTATE;
    int n = cap < HOUGH_N_STAGES ? cap : HOUGH_N_STAGES;
    int last = -1;
    for (int s = 0; s < HOUGH_N_STAGES + 1; ++s)
        if (h->ev_set[s])
            last = s;
    if (last < 0)
        return HOUGH_ESTATE;
    CK(cudaEventSynchronize(h->ev[last]));
    // a stage's time runs from the previous recorded event to its own
    int prev = -1;
    for (int s = 0; s < HOUGH_N_STAGES + 1; ++s) {
        if (!h->ev_set[s])
            continue;
        if (prev >= 0 && s - 1 < n) {
            float t = 0.f;
            CK(cudaEventElapsedTime(&t, h->ev[prev], h->ev[s]));
            ms[s - 1] = t;
        }
        prev = s;
    }
    for (int s = 0; s < n; ++s)
        if (!h->ev_set[s + 1])
            ms[s] = 0.f;
    return n;
}

const char *hough_strerror(int code)
{
    switch (code) {
    case HOUGH_OK:
        return "ok";
    case HOUGH_EINVAL:
        return "invalid argument or configuration";
    case HOUGH_ENOMEM:
        return "workspace or capacity too small";
    case HOUGH_ECUDA:
        return "CUDA runtime error (or no CUDA device)";
    case HOUGH_ESTATE:
        return "call order violated";
    default:
        return "unknown error code";
    }
}
