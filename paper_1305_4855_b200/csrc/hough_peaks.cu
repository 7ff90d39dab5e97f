// hough_peaks.cu -- accumulator sweep kernels (SURVEY.md section 8(a) rows a2, a5, a6 and
// the CSR bookkeeping of a7):
//   k_clear        zero the global accumulator (pure HBM write)
//   k_peak_sweep   popcount + 3x3x3 local-maximum test with ties to the lower linear index,
//                  one pass over the accumulator (4 B/bin read once), 1 flag bit per bin out
//   k_scan         single-pass chained prefix sum (decoupled look-back)
//   k_compact      flag bits -> (lin, mask) records in ascending lin
//   k_sort_lists   puts each peak's hit list into ascending hit index
//   k_finish       counters -> the caller's hough_counts
// The peak rule is BASELINE.json north_star's ("popcount reaches at least L_min and ...
// local maxima in the 3x3x3 neighbourhood (ties go to the lower linear index)"), restated
// in DESIGN.md section 2 A6: with key(b) = (popcount, -lin) a bin is a peak iff its key
// beats the key of every existing neighbour, i.e. popcount > every neighbour of lower lin
// and >= every neighbour of higher lin.
#include "hough_internal.cuh"

// ------------------------------------------------------------------ clear
__global__ void k_clear(uint4 *acc, size_t n_vec)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    size_t stride = (size_t)gridDim.x * blockDim.x;
    const uint4 z = make_uint4(0u, 0u, 0u, 0u);
    for (; i < n_vec; i += stride)
        acc[i] = z;
}

cudaError_t launch_clear(hough_handle *h, cudaStream_t st)
{
    size_t n_bins = (size_t)h->g.n_phi * h->g.n_d0 * h->g.n_kappa;
    size_t n_vec = n_bins / 4; // n_kappa is a multiple of 32
    int blocks = h->n_sms * 8;
    k_clear<<<blocks, 512, 0, st>>>(reinterpret_cast<uint4 *>(h->acc), n_vec);
    h->launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ peak sweep
// A CTA owns Tj d0 rows (plus one halo row on each side) and walks Li phi0 planes with a
// ring of three planes of byte popcounts in shared memory:
//   pc[r][w]  popcounts of 4 consecutive kappa bins packed in one word
//   m3[r][w]  max over kappa-1, kappa, kappa+1 of pc
//   bx[r][w]  max over the 3x3 (d0, kappa) box = max of m3 over r-1, r, r+1
// Missing neighbours (grid edges) are zero popcounts, which can never beat a bin with
// popcount >= L_min >= 1.
struct PeakParams {
    const uint32_t *acc;
    uint32_t *flags;
    int n_phi, n_d0, nk, L_min, wrap;
    int Tj, Li;
};

__device__ __forceinline__ uint32_t pack_popc(uint4 m)
{
    return (uint32_t)__popc(m.x) | ((uint32_t)__popc(m.y) << 8) | ((uint32_t)__popc(m.z) << 16) |
           ((uint32_t)__popc(m.w) << 24);
}

__global__ void __launch_bounds__(512) k_peak_sweep(const PeakParams p)
{
    extern __shared__ __align__(16) uint32_t sm[];
    const int WPR = p.nk >> 2;  // byte words per row
    const int RS = WPR + 2;     // row stride with one zero pad word on each side
    const int R = p.Tj + 2;
    const int plane_words = R * RS;
    uint32_t *pc = sm;                        // [3][R][RS]
    uint32_t *m3 = sm + 3 * plane_words;      // [3][R][RS]
    uint32_t *bx = sm + 6 * plane_words;      // [3][R][RS]
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int j0 = blockIdx.x * p.Tj;
    const int ia = blockIdx.y * p.Li, ib = min(ia + p.Li, p.n_phi);
    const int fw_per_row = p.nk >> 5;
    const uint32_t lmin4 = (uint32_t)p.L_min * 0x01010101u;

    for (int w = tid; w < 9 * plane_words; w += nthr)
        sm[w] = 0u;
    __syncthreads();

    // planes ia-1 .. ib ; plane index q = gi - (ia - 1)
    for (int gi = ia - 1; gi <= ib; ++gi) {
        const int q = gi - (ia - 1);
        const int slot = q % 3;
        int src = gi;
        bool exists = true;
        if (gi < 0) {
            src = p.n_phi - 1;
            exists = p.wrap != 0;
        } else if (gi >= p.n_phi) {
            src = 0;
            exists = p.wrap != 0;
        }
        uint32_t *pcs = pc + slot * plane_words;
        uint32_t *m3s = m3 + slot * plane_words;
        uint32_t *bxs = bx + slot * plane_words;
        // A: load masks, popcount, pack
        for (int idx = tid; idx < R * WPR; idx += nthr) {
            int r = idx / WPR, w = idx - r * WPR;
            int j = j0 - 1 + r;
            uint32_t v = 0u;
            if (exists && j >= 0 && j < p.n_d0) {
                const uint4 *rowp =
                    reinterpret_cast<const uint4 *>(p.acc + ((size_t)src * p.n_d0 + j) * p.nk);
                v = pack_popc(__ldg(rowp + w));
            }
            pcs[r * RS + 1 + w] = v;
        }
        __syncthreads();
        // B: max over kappa +-1
        for (int idx = tid; idx < R * WPR; idx += nthr) {
            int r = idx / WPR, w = idx - r * WPR;
            const uint32_t *row = pcs + r * RS + 1 + w;
            uint32_t cur = row[0], prev = row[-1], next = row[1];
            uint32_t left = (cur << 8) | (prev >> 24);
            uint32_t right = (cur >> 8) | (next << 24);
            m3s[r * RS + 1 + w] = __vmaxu4(cur, __vmaxu4(left, right));
        }
        __syncthreads();
        // C: max over d0 +-1 (interior rows only)
        for (int idx = tid; idx < p.Tj * WPR; idx += nthr) {
            int r = idx / WPR + 1, w = idx - (r - 1) * WPR;
            const uint32_t *c = m3s + r * RS + 1 + w;
            bxs[r * RS + 1 + w] = __vmaxu4(c[0], __vmaxu4(c[-RS], c[RS]));
        }
        __syncthreads();
        // OUT: plane gi-1 is now complete (needs planes gi-2, gi-1, gi)
        if (q >= 2) {
            const int io = gi - 1;
            const int smid = (q - 1) % 3, sprev = (q - 2) % 3, snext = slot;
            const uint32_t *pcm = pc + smid * plane_words;
            const uint32_t *m3m = m3 + smid * plane_words;
            const uint32_t *bxp = bx + sprev * plane_words;
            const uint32_t *bxn = bx + snext * plane_words;
            // With phi wrap, plane -1 of i = 0 is plane n_phi-1 (higher lin: ties lose to
            // us) and plane +1 of i = n_phi-1 is plane 0 (lower lin: ties win over us).
            const bool prev_is_high = (io == 0) && p.wrap;
            const bool next_is_low = (io == p.n_phi - 1) && p.wrap;
            const int items = p.Tj * WPR;
            const int items_pad = (items + 31) & ~31;
            for (int idx = tid; idx < items_pad; idx += nthr) {
                uint32_t nib = 0u;
                int r = 0, w = 0;
                bool ok = idx < items;
                if (ok) {
                    r = idx / WPR + 1;
                    w = idx - (r - 1) * WPR;
                    int o = r * RS + 1 + w;
                    uint32_t cur = pcm[o], prev = pcm[o - 1], next = pcm[o + 1];
                    uint32_t left = (cur << 8) | (prev >> 24);
                    uint32_t right = (cur >> 8) | (next << 24);
                    uint32_t lo = __vmaxu4(left, m3m[o - RS]);
                    uint32_t hi = __vmaxu4(right, m3m[o + RS]);
                    uint32_t bp = bxp[o], bn = bxn[o];
                    if (prev_is_high)
                        hi = __vmaxu4(hi, bp);
                    else
                        lo = __vmaxu4(lo, bp);
                    if (next_is_low)
                        lo = __vmaxu4(lo, bn);
                    else
                        hi = __vmaxu4(hi, bn);
                    uint32_t m = __vcmpgtu4(cur, lo) & __vcmpgeu4(cur, hi) & __vcmpgeu4(cur, lmin4);
                    nib = (((m & 0x01010101u) * 0x01020408u) >> 24) & 0xfu;
                }
                uint32_t bits = nib << ((idx & 7) << 2);
                bits |= __shfl_xor_sync(0xffffffffu, bits, 1);
                bits |= __shfl_xor_sync(0xffffffffu, bits, 2);
                bits |= __shfl_xor_sync(0xffffffffu, bits, 4);
                int j = j0 + r - 1;
                if (ok && (idx & 7) == 0 && j < p.n_d0)
                    p.flags[((size_t)io * p.n_d0 + j) * fw_per_row + (w >> 3)] = bits;
            }
        }
        // the slot written next (q+1) % 3 == (q-2) % 3 was last read by OUT above
        __syncthreads();
    }
}

cudaError_t launch_peak_sweep(hough_handle *h, cudaStream_t st)
{
    PeakParams p;
    p.acc = h->acc;
    p.flags = h->flags;
    p.n_phi = h->g.n_phi;
    p.n_d0 = h->g.n_d0;
    p.nk = h->g.n_kappa;
    p.L_min = h->g.L_min;
    p.wrap = h->g.phi_wrap;
    p.Tj = h->pk_Tj;
    p.Li = h->pk_Li;
    dim3 grid((h->g.n_d0 + p.Tj - 1) / p.Tj, (h->g.n_phi + p.Li - 1) / p.Li);
    static int configured = -1;
    if (configured < h->pk_smem) {
        cudaError_t e =
            cudaFuncSetAttribute(k_peak_sweep, cudaFuncAttributeMaxDynamicSharedMemorySize, h->pk_smem);
        if (e != cudaSuccess)
            return e;
        configured = h->pk_smem;
    }
    k_peak_sweep<<<grid, h->pk_threads, h->pk_smem, st>>>(p);
    h->launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ chained scan
// One pass, decoupled look-back: block t (ticket order) publishes its aggregate, then
// adds the inclusive prefixes / aggregates of its predecessors.  status word =
// (flag << 62) | value, flag 1 = aggregate, 2 = inclusive prefix; written with one
// 64-bit store so that no fence is needed between flag and value.
//   SCAN_ROWS : item i = number of flag bits of accumulator row i  -> row_base (u32)
//   SCAN_LENS : item i = list_len[i], i < min(n_peaks, cap_peaks)  -> hit_offset (u64)
#define SCAN_ROWS 0
#define SCAN_LENS 1
#define SCAN_THREADS 256
#define SCAN_PER_THREAD (HOUGH_SCAN_ITEMS / SCAN_THREADS)

struct ScanParams {
    const uint32_t *flags;
    int fw_per_row;
    uint32_t n_rows;
    uint32_t *row_base;
    const uint32_t *list_len;
    uint32_t cap_peaks;
    unsigned long long *hit_offset;
    unsigned long long cap_hits;
    DevCounters *counters;
    unsigned int *ticket;
    unsigned long long *status;
};

template <int KIND>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan(const ScanParams p)
{
    __shared__ unsigned int s_ticket;
    __shared__ unsigned long long s_warp[SCAN_THREADS / 32];
    __shared__ unsigned long long s_prefix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0)
        s_ticket = atomicAdd(p.ticket, 1u);
    __syncthreads();
    const unsigned int t = s_ticket;
    const uint32_t n = KIND == SCAN_ROWS ? p.n_rows : min(p.counters->n_peaks, p.cap_peaks);
    const unsigned long long base = (unsigned long long)t * HOUGH_SCAN_ITEMS;
    if (n == 0) {
        if (t == 0 && tid == 0) {
            if (KIND == SCAN_ROWS) {
                p.row_base[0] = 0u;
                p.counters->n_peaks = 0u;
            } else {
                p.hit_offset[0] = 0ull;
                p.counters->n_hit_entries = 0ull;
            }
        }
        return;
    }
    if (base >= n)
        return;

    uint32_t v[SCAN_PER_THREAD];
    unsigned long long tsum = 0;
#pragma unroll
    for (int q = 0; q < SCAN_PER_THREAD; ++q) {
        unsigned long long i = base + (unsigned long long)tid * SCAN_PER_THREAD + q;
        uint32_t x = 0u;
        if (i < n) {
            if (KIND == SCAN_ROWS) {
                const uint32_t *fw = p.flags + i * p.fw_per_row;
                for (int w = 0; w < p.fw_per_row; ++w)
                    x += __popc(fw[w]);
            } else {
                x = p.list_len[i];
            }
        }
        v[q] = x;
        tsum += x;
    }
    // block exclusive scan of tsum
    unsigned long long incl = tsum;
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o)
            incl += y;
    }
    if (lane == 31)
        s_warp[warp] = incl;
    __syncthreads();
    unsigned long long wbase = 0, agg = 0;
    for (int w = 0; w < SCAN_THREADS / 32; ++w) {
        unsigned long long x = s_warp[w];
        if (w < warp)
            wbase += x;
        agg += x;
    }
    unsigned long long texcl = wbase + incl - tsum;

    if (tid == 0) {
        volatile unsigned long long *status = p.status;
        unsigned long long prefix = 0;
        if (t == 0) {
            status[0] = (2ull << 62) | agg;
        } else {
            status[t] = (1ull << 62) | agg;
            long long q = (long long)t - 1;
            while (true) {
                unsigned long long s = status[q];
                unsigned long long flag = s >> 62;
                if (flag == 0ull)
                    continue; // predecessor (already scheduled: lower ticket) not there yet
                prefix += s & ((1ull << 62) - 1ull);
                if (flag == 2ull)
                    break;
                --q;
            }
            status[t] = (2ull << 62) | (prefix + agg);
        }
        s_prefix = prefix;
    }
    __syncthreads();
    unsigned long long run = s_prefix + texcl;
#pragma unroll
    for (int q = 0; q < SCAN_PER_THREAD; ++q) {
        unsigned long long i = base + (unsigned long long)tid * SCAN_PER_THREAD + q;
        if (i < n) {
            if (KIND == SCAN_ROWS)
                p.row_base[i] = (uint32_t)run;
            else
                p.hit_offset[i] = run;
            run += v[q];
            if (i == (unsigned long long)n - 1) { // the last item closes the scan
                if (KIND == SCAN_ROWS) {
                    p.row_base[n] = (uint32_t)run;
                    p.counters->n_peaks = (unsigned int)run;
                } else {
                    p.hit_offset[n] = run;
                    p.counters->n_hit_entries = run;
                }
            }
        }
    }
}

static void scan_params(hough_handle *h, ScanParams *p, const hough_peaks_out *out, int which)
{
    p->flags = h->flags;
    p->fw_per_row = h->g.n_kappa >> 5;
    p->n_rows = (uint32_t)h->g.n_phi * (uint32_t)h->g.n_d0;
    p->row_base = h->row_base;
    p->list_len = h->list_len;
    p->cap_peaks = h->cfg.cap_peaks;
    p->hit_offset = out ? reinterpret_cast<unsigned long long *>(out->hit_offset) : nullptr;
    p->cap_hits = h->cfg.cap_hits;
    p->counters = h->counters;
    p->ticket = h->scan_ticket + which;
    p->status = h->scan_status + (size_t)which * h->scan_blocks_max;
}

cudaError_t launch_scan_rows(hough_handle *h, cudaStream_t st)
{
    ScanParams p;
    scan_params(h, &p, nullptr, 0);
    uint32_t blocks = (p.n_rows + HOUGH_SCAN_ITEMS - 1) / HOUGH_SCAN_ITEMS;
    k_scan<SCAN_ROWS><<<blocks, SCAN_THREADS, 0, st>>>(p);
    h->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_scan_lens(hough_handle *h, const hough_peaks_out *out, cudaStream_t st)
{
    ScanParams p;
    scan_params(h, &p, out, 1);
    uint32_t blocks = (h->cfg.cap_peaks + HOUGH_SCAN_ITEMS - 1) / HOUGH_SCAN_ITEMS;
    k_scan<SCAN_LENS><<<blocks, SCAN_THREADS, 0, st>>>(p);
    h->launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ compaction (a6)
// One warp per accumulator row: ballot-free popcount prefix over the row's flag words,
// each lane expands the set bits of its word.  Records land in ascending lin because
// row_base is the exclusive scan of the rows in lin order.
__global__ void __launch_bounds__(256) k_compact(const uint32_t *__restrict__ flags,
                                                 const uint32_t *__restrict__ row_base,
                                                 const uint32_t *__restrict__ acc, uint32_t n_rows,
                                                 int nk, uint32_t cap_peaks, uint32_t *__restrict__ bin,
                                                 uint32_t *__restrict__ mask)
{
    const int lane = threadIdx.x & 31;
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    const int fw_per_row = nk >> 5;
    for (uint32_t row = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; row < n_rows; row += warps) {
        uint32_t gb = row_base[row];
        uint32_t cnt = row_base[row + 1] - gb;
        if (cnt == 0u || gb >= cap_peaks)
            continue;
        const uint32_t *fw = flags + (size_t)row * fw_per_row;
        uint32_t rank0 = gb;
        for (int wb = 0; wb < fw_per_row; wb += 32) {
            uint32_t f = (wb + lane < fw_per_row) ? fw[wb + lane] : 0u;
            uint32_t pc = __popc(f), incl = pc;
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o)
                    incl += t;
            }
            uint32_t rank = rank0 + incl - pc;
            while (f) {
                int b = __ffs(f) - 1;
                f &= f - 1;
                if (rank < cap_peaks) {
                    uint32_t lin = row * (uint32_t)nk + (uint32_t)(((wb + lane) << 5) + b);
                    bin[rank] = lin;
                    mask[rank] = acc[lin];
                }
                ++rank;
            }
            rank0 += __shfl_sync(0xffffffffu, incl, 31);
        }
    }
}

cudaError_t launch_compact(hough_handle *h, const hough_peaks_out *out, cudaStream_t st)
{
    uint32_t n_rows = (uint32_t)h->g.n_phi * (uint32_t)h->g.n_d0;
    uint32_t blocks = (n_rows + 7) / 8;
    uint32_t maxb = (uint32_t)h->n_sms * 16;
    if (blocks > maxb)
        blocks = maxb;
    k_compact<<<blocks, 256, 0, st>>>(h->flags, h->row_base, h->acc, n_rows, h->g.n_kappa,
                                      h->cfg.cap_peaks, out->bin, out->mask);
    h->launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ list order (a7)
// The fill pass appends with a shared-memory cursor, so a list is complete but in the
// order the warps happened to run.  One thread per peak sorts its (short) list.
__global__ void __launch_bounds__(256) k_sort_lists(const DevCounters *__restrict__ counters,
                                                    uint32_t cap_peaks,
                                                    const unsigned long long *__restrict__ hit_offset,
                                                    uint32_t *__restrict__ hit_index,
                                                    unsigned long long cap_hits)
{
    uint32_t n = min(counters->n_peaks, cap_peaks);
    uint32_t stride = gridDim.x * blockDim.x;
    for (uint32_t pk = blockIdx.x * blockDim.x + threadIdx.x; pk < n; pk += stride) {
        unsigned long long b = hit_offset[pk], e = hit_offset[pk + 1];
        if (e > cap_hits)
            continue; // a list cut by the capacity is not part of the valid output
        uint32_t *a = hit_index + b;
        int len = (int)(e - b);
        for (int i = 1; i < len; ++i) {
            uint32_t v = a[i];
            int j = i - 1;
            while (j >= 0 && a[j] > v) {
                a[j + 1] = a[j];
                --j;
            }
            a[j + 1] = v;
        }
    }
}

cudaError_t launch_sort_lists(hough_handle *h, const hough_peaks_out *out, cudaStream_t st)
{
    uint32_t blocks = (h->cfg.cap_peaks + 255) / 256;
    uint32_t maxb = (uint32_t)h->n_sms * 16;
    if (blocks > maxb)
        blocks = maxb;
    k_sort_lists<<<blocks, 256, 0, st>>>(h->counters, h->cfg.cap_peaks,
                                         reinterpret_cast<const unsigned long long *>(out->hit_offset),
                                         out->hit_index, h->cfg.cap_hits);
    h->launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ counters out
__global__ void k_finish(const DevCounters *c, hough_counts *out, uint32_t cap_peaks,
                         unsigned long long cap_hits, int with_lists)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        hough_counts r;
        r.n_votes = c->n_votes;
        r.n_hit_entries = with_lists ? c->n_hit_entries : 0ull;
        r.n_evals = c->n_evals;
        r.n_peaks = c->n_peaks;
        r.n_bad_hits = c->n_bad_hits;
        r.flags = 0u;
        if (r.n_peaks > cap_peaks)
            r.flags |= HOUGH_TRUNCATED_PEAKS;
        if (r.n_hit_entries > cap_hits)
            r.flags |= HOUGH_TRUNCATED_HITS;
        r.reserved = 0u;
        *out = r;
    }
}

cudaError_t launch_finish_counts(hough_handle *h, const hough_peaks_out *out, int with_lists,
                                 cudaStream_t st)
{
    k_finish<<<1, 32, 0, st>>>(h->counters, out->counts, h->cfg.cap_peaks, h->cfg.cap_hits, with_lists);
    h->launches += 1;
    return cudaGetLastError();
}
