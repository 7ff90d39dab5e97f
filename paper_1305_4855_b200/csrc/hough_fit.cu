// hough_fit.cu -- f2: fit of every peak's hit list, selection and removal of duplicates
// (section 8 "perform a fit of the hits to the candidate tracks"; "cleaned
// to remove duplicate tracks or tracks which share a large number of hits"; SURVEY.md section 8(f) f2;
// recipes E4 / E5 of DESIGN.md section 8, restated in include/hough.h).
//
// Six small kernels, everything read and decided on the device:
//   k_fit            E4, ONE THREAD per candidate: the three passes over the list run in list order in
//                    binary64 with explicit round-to-nearest intrinsics (no contraction), so the moments
//                    are the recipe's sums term by term; selection flag; per-hit histogram of the
//                    selected candidates.  (A config-3 list has ~12 hits: a warp per candidate would
//                    idle 20 lanes and change the summation order.)
//   k_inv_scan       exclusive scan of the per-hit histogram (one CTA)
//   k_inv_fill       inverted index hit -> selected candidates holding it
//   k_dedup          E5, ONE WARP per selected candidate: lanes walk the candidates that share a hit with
//                    it; a pair is examined once (at its first common hit) and only if the other one is
//                    better; shared hits are counted by merging the two ascending lists
//   k_kept_count / k_kept_compact   ordered compaction of the kept candidates
#include <math.h>

#include "hough_internal.cuh"

#define FIT_THREADS 256
#define FIT_CACHE 64 // hits of the warp's own candidate kept in shared memory by k_dedup

struct FitParams {
    const float *hx, *hy;
    uint32_t n_hits;
    const uint32_t *peak_mask;
    const unsigned long long *hit_offset;
    const uint32_t *hit_index;
    const hough_counts *peak_counts;
    uint32_t cap_peaks;
    unsigned long long cap_hits;
    double rms_max;
    uint32_t min_shared;
    // scratch
    uint32_t *inv_start; // [n_hits + 1] histogram, then exclusive scan
    uint32_t *inv_cur;   // [n_hits + 1] fill cursor
    uint32_t *inv;       // [cap_hits]
    uint32_t *block_cnt; // [n_blocks]
    // outputs
    double *kappa, *phi0, *d0, *rms;
    int32_t *status;
    unsigned char *flag;
    uint32_t *kept;
    hough_fit_counts *counts;
};

__device__ __forceinline__ double f_mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double f_add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double f_sub(double a, double b) { return __dsub_rn(a, b); }

// E4 for one list; the order of every operation is the recipe's
__device__ int fit_list(const float *__restrict__ hx, const float *__restrict__ hy, const uint32_t *__restrict__ idx,
                        uint32_t n, double &kappa, double &phi0, double &d0, double &rms)
{
    kappa = phi0 = d0 = rms = 0.0;
    if (n < 3)
        return 1;
    double sx = 0.0, sy = 0.0, sr = 0.0;
    for (uint32_t q = 0; q < n; ++q) {
        const uint32_t h = idx[q];
        const double xv = (double)hx[h], yv = (double)hy[h];
        sx = f_add(sx, xv);
        sy = f_add(sy, yv);
        sr = f_add(sr, f_add(f_mul(xv, xv), f_mul(yv, yv)));
    }
    const double dn = (double)n;
    const double mx = __ddiv_rn(sx, dn), my = __ddiv_rn(sy, dn), mr = __ddiv_rn(sr, dn);
    double Cxx = 0.0, Cxy = 0.0, Cyy = 0.0, Cxr = 0.0, Cyr = 0.0, Crr = 0.0;
    for (uint32_t q = 0; q < n; ++q) {
        const uint32_t h = idx[q];
        const double xv = (double)hx[h], yv = (double)hy[h];
        const double u = f_sub(xv, mx), v = f_sub(yv, my), w = f_sub(f_add(f_mul(xv, xv), f_mul(yv, yv)), mr);
        Cxx = f_add(Cxx, f_mul(u, u));
        Cxy = f_add(Cxy, f_mul(u, v));
        Cyy = f_add(Cyy, f_mul(v, v));
        Cxr = f_add(Cxr, f_mul(u, w));
        Cyr = f_add(Cyr, f_mul(v, w));
        Crr = f_add(Crr, f_mul(w, w));
    }
    Cxx = __ddiv_rn(Cxx, dn);
    Cxy = __ddiv_rn(Cxy, dn);
    Cyy = __ddiv_rn(Cyy, dn);
    Cxr = __ddiv_rn(Cxr, dn);
    Cyr = __ddiv_rn(Cyr, dn);
    Crr = __ddiv_rn(Crr, dn);
    if (!(Crr > 0.0))
        return 2;
    const double q1 = f_sub(f_mul(Crr, Cxy), f_mul(Cxr, Cyr));
    const double q2 = f_add(f_sub(f_mul(Crr, f_sub(Cxx, Cyy)), f_mul(Cxr, Cxr)), f_mul(Cyr, Cyr));
    double phi = f_mul(0.5, atan2(f_mul(2.0, q1), q2));
    double sp, cp;
    sincos(phi, &sp, &cp);
    const double khat = __ddiv_rn(f_add(f_mul(-sp, Cxr), f_mul(cp, Cyr)), Crr);
    const double delta = f_sub(f_add(f_mul(-mx, sp), f_mul(my, cp)), f_mul(khat, mr));
    const double D = f_sub(1.0, f_mul(f_mul(4.0, delta), khat));
    if (!(D > 0.0))
        return 2;
    const double sq = __dsqrt_rn(D);
    double kap = __ddiv_rn(f_mul(2.0, khat), sq);
    double dd = __ddiv_rn(f_mul(2.0, delta), f_add(1.0, sq));
    double see = 0.0;
    for (uint32_t q = 0; q < n; ++q) {
        const uint32_t h = idx[q];
        const double xv = (double)hx[h], yv = (double)hy[h];
        const double u = f_sub(xv, mx), v = f_sub(yv, my), w = f_sub(f_add(f_mul(xv, xv), f_mul(yv, yv)), mr);
        const double eps = f_sub(f_mul(khat, w), f_add(f_mul(-sp, u), f_mul(cp, v)));
        see = f_add(see, f_mul(eps, eps));
    }
    const double r = __dsqrt_rn(__ddiv_rn(__ddiv_rn(see, dn), D));
    if (f_add(f_mul(mx, cp), f_mul(my, sp)) < 0.0) { // backward representation: report the forward one
        const double pi = 3.14159265358979323846;
        phi = phi >= 0.0 ? f_sub(phi, pi) : f_add(phi, pi);
        dd = -dd;
        kap = -kap;
    }
    if (!(isfinite(kap) && isfinite(dd) && isfinite(r)))
        return 2;
    kappa = kap;
    phi0 = phi;
    d0 = dd;
    rms = r;
    return 0;
}

__global__ void __launch_bounds__(FIT_THREADS) k_fit(const FitParams p)
{
    const uint32_t n_rep = min(p.peak_counts->n_peaks, p.cap_peaks);
    const uint32_t c = blockIdx.x * FIT_THREADS + threadIdx.x;
    int st = -1;
    bool sel = false;
    if (c < n_rep) {
        const unsigned long long o0 = p.hit_offset[c], o1 = p.hit_offset[c + 1];
        double kappa = 0.0, phi0 = 0.0, d0 = 0.0, rms = 0.0;
        if (o1 > p.cap_hits || o1 < o0) {
            st = 3;
        } else {
            const uint32_t n = (uint32_t)min(o1 - o0, 0xffffffffull);
            st = fit_list(p.hx, p.hy, p.hit_index + o0, n, kappa, phi0, d0, rms);
            sel = st == 0 && rms <= p.rms_max;
            if (sel)
                for (uint32_t q = 0; q < n; ++q)
                    atomicAdd(&p.inv_start[p.hit_index[o0 + q]], 1u);
        }
        p.kappa[c] = kappa;
        p.phi0[c] = phi0;
        p.d0[c] = d0;
        p.rms[c] = rms;
        p.status[c] = st;
        p.flag[c] = sel ? 1 : 0;
    }
    const unsigned b_ok = __ballot_sync(0xffffffffu, st == 0), b_sel = __ballot_sync(0xffffffffu, sel),
                   b_tr = __ballot_sync(0xffffffffu, st == 3);
    if ((threadIdx.x & 31) == 0) {
        if (b_ok)
            atomicAdd(&p.counts->n_ok, (uint32_t)__popc(b_ok));
        if (b_sel)
            atomicAdd(&p.counts->n_selected, (uint32_t)__popc(b_sel));
        if (b_tr)
            atomicAdd(&p.counts->n_truncated, (uint32_t)__popc(b_tr));
    }
    if (blockIdx.x == 0 && threadIdx.x == 0)
        p.counts->n_fitted = n_rep;
}

// exclusive scan of inv_start[0 .. n_hits) in place, total at [n_hits]; copy into the fill cursor.
// One CTA; warp w owns the contiguous chunk [w * per, (w + 1) * per) and walks it 32 items at a time
// (coalesced), first for its sum, then -- after the scan of the 32 warp sums -- for the prefixes.
__global__ void __launch_bounds__(1024) k_inv_scan(const FitParams p)
{
    __shared__ uint32_t s_warp[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t n = p.n_hits, per = ((n + 1023u) / 1024u) * 32u;
    const uint32_t b0 = min((uint32_t)warp * per, n), b1 = min(b0 + per, n);
    uint32_t sum = 0;
    for (uint32_t q = b0 + lane; q < b1; q += 32)
        sum += p.inv_start[q];
    for (int o = 16; o > 0; o >>= 1)
        sum += __shfl_xor_sync(0xffffffffu, sum, o);
    if (lane == 0)
        s_warp[warp] = sum;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = s_warp[lane];
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, w, o);
            if (lane >= o)
                w += t;
        }
        s_warp[lane] = w; // inclusive over the warps
    }
    __syncthreads();
    uint32_t run = warp > 0 ? s_warp[warp - 1] : 0u;
    for (uint32_t q0 = b0; q0 < b1; q0 += 32) {
        const uint32_t q = q0 + lane;
        const uint32_t v = q < b1 ? p.inv_start[q] : 0u;
        uint32_t incl = v;
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o)
                incl += t;
        }
        if (q < b1) {
            p.inv_start[q] = run + incl - v;
            p.inv_cur[q] = run + incl - v;
        }
        run += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (threadIdx.x == 1023)
        p.inv_start[n] = s_warp[31];
}

__global__ void __launch_bounds__(FIT_THREADS) k_inv_fill(const FitParams p)
{
    const uint32_t n_rep = min(p.peak_counts->n_peaks, p.cap_peaks);
    const uint32_t c = blockIdx.x * FIT_THREADS + threadIdx.x;
    if (c >= n_rep || !p.flag[c])
        return;
    const unsigned long long o0 = p.hit_offset[c], o1 = p.hit_offset[c + 1];
    for (unsigned long long q = o0; q < o1; ++q)
        p.inv[atomicAdd(&p.inv_cur[p.hit_index[q]], 1u)] = c;
}

__device__ __forceinline__ bool fit_better(int la, double ra, uint32_t ia, int lb, double rb, uint32_t ib)
{ // is candidate a better than candidate b?
    if (la != lb)
        return la > lb;
    if (ra != rb)
        return ra < rb;
    return ia < ib;
}

__global__ void __launch_bounds__(FIT_THREADS) k_dedup(const FitParams p)
{
    __shared__ uint32_t s_list[FIT_THREADS / 32][FIT_CACHE];
    const uint32_t n_rep = min(p.peak_counts->n_peaks, p.cap_peaks);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t n_warps = gridDim.x * (FIT_THREADS / 32);
    unsigned long long tests = 0;
    // a warp looks at 32 candidates at a time (one coalesced read of their flags) and takes the selected
    // ones among them one after the other
    for (uint32_t c32 = (blockIdx.x * (FIT_THREADS / 32) + warp) * 32u; c32 < n_rep; c32 += n_warps * 32u) {
      unsigned todo = __ballot_sync(0xffffffffu, c32 + lane < n_rep && p.flag[c32 + lane] != 0);
      while (todo) {
        const uint32_t c = c32 + (uint32_t)(__ffs((int)todo) - 1);
        todo &= todo - 1;
        const unsigned long long o0 = p.hit_offset[c];
        const uint32_t np = (uint32_t)(p.hit_offset[c + 1] - o0);
        const uint32_t *A = p.hit_index + o0;
        const bool cached = np <= FIT_CACHE;
        __syncwarp();
        if (cached) {
            for (uint32_t q = lane; q < np; q += 32)
                s_list[warp][q] = A[q];
            __syncwarp();
        }
        const int lc = __popc(p.peak_mask[c]);
        const double rc = p.rms[c];
        bool dup = false;
        for (uint32_t q = 0; q < np && !dup; ++q) {
            const uint32_t h = cached ? s_list[warp][q] : A[q];
            const uint32_t zs = p.inv_start[h], ze = p.inv_start[h + 1];
            for (uint32_t zb = zs; zb < ze; zb += 32) {
                const uint32_t z = zb + lane;
                bool mine = false;
                if (z < ze) {
                    const uint32_t o = p.inv[z];
                    if (o != c && fit_better(__popc(p.peak_mask[o]), p.rms[o], o, lc, rc, c)) {
                        // shared hits by merging the two ascending lists; the pair is examined at its
                        // FIRST common hit only (an earlier one means it was examined in an earlier round)
                        const unsigned long long b0 = p.hit_offset[o];
                        const uint32_t nb = (uint32_t)(p.hit_offset[o + 1] - b0);
                        const uint32_t *B = p.hit_index + b0;
                        uint32_t i = 0, j = 0, shared = 0;
                        bool first_here = true;
                        while (i < np && j < nb) {
                            const uint32_t a = cached ? s_list[warp][i] : A[i], b = B[j];
                            if (a == b) {
                                if (shared == 0 && a != h) {
                                    first_here = false;
                                    break;
                                }
                                ++shared;
                                if (shared >= p.min_shared)
                                    break;
                                ++i;
                                ++j;
                            } else if (a < b) {
                                ++i;
                            } else {
                                ++j;
                            }
                        }
                        if (first_here) {
                            ++tests;
                            mine = shared >= p.min_shared;
                        }
                    }
                }
                if (__any_sync(0xffffffffu, mine)) {
                    dup = true;
                    break;
                }
            }
        }
        if (dup && lane == 0)
            p.flag[c] = 2;
      }
    }
    for (int o = 16; o > 0; o >>= 1)
        tests += __shfl_xor_sync(0xffffffffu, tests, o);
    if (lane == 0 && tests)
        atomicAdd(reinterpret_cast<unsigned long long *>(&p.counts->n_pair_tests), tests);
}

__global__ void __launch_bounds__(FIT_THREADS) k_kept_count(const FitParams p)
{
    __shared__ uint32_t s_cnt;
    if (threadIdx.x == 0)
        s_cnt = 0u;
    __syncthreads();
    const uint32_t n_rep = min(p.peak_counts->n_peaks, p.cap_peaks);
    const uint32_t c = blockIdx.x * FIT_THREADS + threadIdx.x;
    const bool k = c < n_rep && p.flag[c] == 1;
    const unsigned bal = __ballot_sync(0xffffffffu, k);
    if ((threadIdx.x & 31) == 0 && bal)
        atomicAdd(&s_cnt, (uint32_t)__popc(bal));
    __syncthreads();
    if (threadIdx.x == 0)
        p.block_cnt[blockIdx.x] = s_cnt;
}

__global__ void __launch_bounds__(FIT_THREADS) k_kept_compact(const FitParams p)
{
    __shared__ uint32_t s_red[FIT_THREADS / 32];
    __shared__ uint32_t s_wcnt[FIT_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t part = 0;
    for (uint32_t b = threadIdx.x; b < blockIdx.x; b += FIT_THREADS)
        part += p.block_cnt[b];
    for (int o = 16; o > 0; o >>= 1)
        part += __shfl_xor_sync(0xffffffffu, part, o);
    if (lane == 0)
        s_red[warp] = part;
    const uint32_t n_rep = min(p.peak_counts->n_peaks, p.cap_peaks);
    const uint32_t c = blockIdx.x * FIT_THREADS + threadIdx.x;
    const bool k = c < n_rep && p.flag[c] == 1;
    const unsigned bal = __ballot_sync(0xffffffffu, k);
    if (lane == 0)
        s_wcnt[warp] = (uint32_t)__popc(bal);
    __syncthreads();
    uint32_t base = 0, before = 0, all = 0;
    for (int w = 0; w < FIT_THREADS / 32; ++w) {
        base += s_red[w];
        before += w < warp ? s_wcnt[w] : 0u;
        all += s_wcnt[w];
    }
    if (k)
        p.kept[base + before + (uint32_t)__popc(bal & ((1u << lane) - 1u))] = c;
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) {
        const uint32_t kept = base + all;
        p.counts->n_kept = kept;
        p.counts->n_duplicates = p.counts->n_selected - kept;
    }
}

// ------------------------------------------------------------------ host side
static size_t fit_align(size_t b) { return (b + 255) & ~(size_t)255; }

size_t hough_fit_workspace_bytes(const hough_handle *h)
{
    if (!h || h->cfg.cap_hits >= 4294967296ull)
        return 0;
    const size_t nh = (size_t)h->cfg.max_hits + 1, n_blocks = ((size_t)h->cfg.cap_peaks + FIT_THREADS - 1) / FIT_THREADS;
    return 2 * fit_align(nh * 4) + fit_align((size_t)h->cfg.cap_hits * 4) + fit_align(n_blocks * 4);
}

int hough_fit(hough_handle *h, const hough_fit_config *fc, void *workspace, size_t workspace_bytes,
              const hough_peaks_out *peaks, const hough_fit_out *out, void *cuda_stream)
{
    if (!h || !fc || !workspace || !peaks || !peaks->mask || !peaks->hit_offset || !peaks->hit_index ||
        !peaks->counts || !out || !out->kappa || !out->phi0 || !out->d0 || !out->rms || !out->status ||
        !out->flag || !out->kept || !out->counts)
        return HOUGH_EINVAL;
    if (!(fc->rms_max >= 0.0) || fc->min_shared < 1 || fc->reserved != 0)
        return HOUGH_EINVAL;
    if (((uintptr_t)workspace & 255) != 0)
        return HOUGH_EINVAL;
    const size_t need = hough_fit_workspace_bytes(h);
    if (need == 0)
        return HOUGH_EINVAL;
    if (workspace_bytes < need)
        return HOUGH_ENOMEM;
    if (!h->voted)
        return HOUGH_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (cudaSetDevice(h->device) != cudaSuccess)
        return HOUGH_ECUDA;
    const size_t nh = (size_t)h->cfg.max_hits + 1, n_blocks = ((size_t)h->cfg.cap_peaks + FIT_THREADS - 1) / FIT_THREADS;
    unsigned char *w = (unsigned char *)workspace;
    FitParams p;
    p.hx = h->hx;
    p.hy = h->hy;
    p.n_hits = h->n_hits;
    p.peak_mask = peaks->mask;
    p.hit_offset = reinterpret_cast<const unsigned long long *>(peaks->hit_offset);
    p.hit_index = peaks->hit_index;
    p.peak_counts = peaks->counts;
    p.cap_peaks = h->cfg.cap_peaks;
    p.cap_hits = h->cfg.cap_hits;
    p.rms_max = fc->rms_max;
    p.min_shared = fc->min_shared;
    p.inv_start = (uint32_t *)w;
    w += fit_align(nh * 4);
    p.inv_cur = (uint32_t *)w;
    w += fit_align(nh * 4);
    p.inv = (uint32_t *)w;
    w += fit_align((size_t)h->cfg.cap_hits * 4);
    p.block_cnt = (uint32_t *)w;
    p.kappa = out->kappa;
    p.phi0 = out->phi0;
    p.d0 = out->d0;
    p.rms = out->rms;
    p.status = out->status;
    p.flag = out->flag;
    p.kept = out->kept;
    p.counts = out->counts;
#define FCK(call)                      \
    do {                               \
        if ((call) != cudaSuccess) {   \
            cudaGetLastError();        \
            return HOUGH_ECUDA;        \
        }                              \
    } while (0)
    FCK(cudaMemsetAsync(p.inv_start, 0, ((size_t)h->n_hits + 1) * 4, st));
    FCK(cudaMemsetAsync(out->counts, 0, sizeof(hough_fit_counts), st));
    k_fit<<<(unsigned)n_blocks, FIT_THREADS, 0, st>>>(p);
    k_inv_scan<<<1, 1024, 0, st>>>(p);
    k_inv_fill<<<(unsigned)n_blocks, FIT_THREADS, 0, st>>>(p);
    FCK(cudaGetLastError());
    k_dedup<<<h->n_sms * 8, FIT_THREADS, 0, st>>>(p);
    k_kept_count<<<(unsigned)n_blocks, FIT_THREADS, 0, st>>>(p);
    k_kept_compact<<<(unsigned)n_blocks, FIT_THREADS, 0, st>>>(p);
    FCK(cudaGetLastError());
#undef FCK
    h->launches += 6;
    return HOUGH_OK;
}
