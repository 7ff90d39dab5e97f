// hough_peaklists.cu -- a7, the hit lists of the reported peaks, PEAK-DRIVEN (SURVEY.md section
// 8(a)): "each peak is emitted with its sorted hit list" (BASELINE.json
// north_star); hit list of a peak = the hits whose own vote at the peak's (phi0, d0) cell lands
// in the peak's kappa bin, ascending hit index, CSR (A7).
//
// A second sweep of all hits over all cells repeats the whole vote to recover the 4 % of the
// votes that land in reported peaks.  Instead the hits are indexed once per event by
// (layer label, azimuth bin), and every peak looks only at the hits that can lie between the
// two circles that bound its bin:
//
//   with n = (-sin phi0, cos phi0), a hit X at radius r and w = sin(azimuth(X) - phi0):
//     kappa(X) >= kappa_1  <=>  2 e - kappa_1 den >= 0  <=>  w >= W(kappa_1, r)     (den = |X - P0|^2 > 0)
//     W(kappa, r) = A / r + B r,  A = d0 (2 + kappa d0) / (2 (1 + kappa d0)),  B = kappa / (2 (1 + kappa d0))
//   (the closed form solved for s = r w; needs 1 + kappa d0 > 0).  Over the radii [ra, rb] that
//   the hits of one layer label really have, min W(kappa_lo) and max W(kappa_hi) are taken at the
//   end points or at the stationary point sqrt(A / B); asin of that w-interval gives two azimuth
//   windows (the circle meets a radius twice: phi0 + asin w and phi0 + pi - asin w).
//
// The windows are SUPERSETS: the bin's kappa interval is widened by a bound on the binary32
// evaluation error of the recipe (which grows as 1 / den; hits closer than L0 to the point of
// closest approach P0 are taken through a third, "proximity" window around P0's azimuth instead),
// and every angle by 5e-5 rad (the azimuth bins of the index come from atan2f, 2 ulp ~ 1e-6 rad, and the
// window angles carry a few binary32 roundings of values below 2 pi).  Whatever cannot be
// bounded (1 + kappa d0 not safely positive, non-finite intermediate values, a window wider than
// the ring) falls back to the whole layer; hits outside the index's numeric range ("wild") are
// candidates of every peak.  Every candidate is then evaluated with the EXACT recipe
// (hough_device.cuh eval_kappa / kappa_bin), so the lists are bit-identical to the oracle's.
//
// Work split: ONE THREAD per peak; the warps draw 32 peaks at a time from a global counter.  The thread
// walks the layer labels set in the peak's mask (a hit of layer l in the bin sets bit l, so other
// layers cannot contribute), queues the candidate ranges of their windows in its 40 words of shared
// memory, evaluates all queued candidates in one flat loop and collects the matching hit indices at
// the top of the same words; it sorts them (insertion sort) and writes them to the peak's fixed slot
// of the staging buffer.  A list that outgrows shared memory spills to the slot in candidate order
// (PL_UNSORTED); one that outgrows the slot is only counted (PL_SLOW).  k_scan<LENS> turns the lengths
// into hit_offset and k_copy_lists moves the lists to their final place: a plain copy for sorted
// slots, ranks by counting for unsorted ones, and straight from the hits in index order (one warp per
// peak) for the rest.  (Round-2 history: a group of 16 lanes per peak with lane = layer spent 55 % of
// its instructions on the window arithmetic at 10 of 32 lanes active, plus three CTA barriers per
// batch: 2.8e8 warp instructions per pile-up event, 0.42 ms; now 1.2e8 and 0.17 ms.)
#include "hough_device.cuh"

#define PL_THREADS 256
#define PL_MAXSLOT 64 // entries of a staging slot (at most; hough_create sizes it from the capacities)
#define PL_SLOW 0xffffffffu
#define PI_F 3.14159265358979f

// ------------------------------------------------------------------ index build
// Histogram and per-layer radius range are accumulated by k_prep (hough_api.cu); here the
// prefix over the keys and the scatter into key order.
// Exclusive prefix over the keys by ONE CTA: per round every thread takes IS_V uint4 of the
// histogram (coalesced, all loads in flight together), the warps scan their uint4 sums with
// shuffles, warp 0 scans the IS_V x 32 warp totals, and the carry moves on to the next round.
// n_keys is a multiple of 256 (NA >= 256), so uint4 accesses never straddle the end.
#define IS_V 4
__global__ void __launch_bounds__(1024) k_index_scan(uint32_t *__restrict__ cnt, uint32_t *__restrict__ start,
                                                     uint32_t *__restrict__ cur, int n_keys)
{
    __shared__ uint32_t s_warp[IS_V][32];
    __shared__ uint32_t s_carry;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    uint32_t carry = 0;
    for (int base = 0; base < n_keys; base += IS_V * 4096) {
        uint4 v[IS_V];
        uint32_t incl[IS_V], sum[IS_V];
#pragma unroll
        for (int q = 0; q < IS_V; ++q) {
            const int k = base + q * 4096 + t * 4;
            v[q] = k < n_keys ? *reinterpret_cast<const uint4 *>(cnt + k) : make_uint4(0u, 0u, 0u, 0u);
        }
#pragma unroll
        for (int q = 0; q < IS_V; ++q) {
            sum[q] = v[q].x + v[q].y + v[q].z + v[q].w;
            incl[q] = sum[q];
        }
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
            for (int q = 0; q < IS_V; ++q) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, incl[q], o);
                if (lane >= o)
                    incl[q] += u;
            }
        }
        if (lane == 31) {
#pragma unroll
            for (int q = 0; q < IS_V; ++q)
                s_warp[q][warp] = incl[q];
        }
        __syncthreads();
        if (warp == 0) { // exclusive scan of the IS_V x 32 warp totals, in key order
            uint32_t run = carry;
#pragma unroll
            for (int q = 0; q < IS_V; ++q) {
                const uint32_t w = s_warp[q][lane];
                uint32_t wi = w;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t u = __shfl_up_sync(0xffffffffu, wi, o);
                    if (lane >= o)
                        wi += u;
                }
                s_warp[q][lane] = run + wi - w;
                run += __shfl_sync(0xffffffffu, wi, 31);
            }
            if (lane == 0)
                s_carry = run;
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < IS_V; ++q) {
            const int k = base + q * 4096 + t * 4;
            if (k < n_keys) {
                const uint32_t e0 = s_warp[q][warp] + incl[q] - sum[q];
                uint4 o;
                o.x = e0;
                o.y = e0 + v[q].x;
                o.z = o.y + v[q].y;
                o.w = o.z + v[q].z;
                *reinterpret_cast<uint4 *>(start + k) = o;
                *reinterpret_cast<uint4 *>(cur + k) = o;                          // the scatter cursor
                *reinterpret_cast<uint4 *>(cnt + k) = make_uint4(0u, 0u, 0u, 0u); // clean for the next event
            }
        }
        carry = s_carry;
        __syncthreads();
    }
    if (t == 0)
        start[n_keys] = carry;
}

__global__ void __launch_bounds__(256) k_index_scatter(HitIndexDev ix, const float *__restrict__ hx,
                                                       const float *__restrict__ hy,
                                                       const float *__restrict__ hr2, uint32_t n)
{
    const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n)
        return;
    const uint32_t key = ix.key[h];
    if (key == 0xffffffffu)
        return;
    const uint32_t rank = atomicAdd(&ix.bin_cur[key], 1u);
    ix.rec[rank] = make_float4(hx[h], hy[h], hr2[h], __uint_as_float(h));
}

cudaError_t launch_index_build(hough_handle *h, cudaStream_t st)
{
    if (h->n_hits == 0)
        return cudaSuccess;
    k_index_scan<<<1, 1024, 0, st>>>(h->ix.bin_cnt, h->ix.bin_start, h->ix.bin_cur, h->ix.n_keys);
    k_index_scatter<<<(h->n_hits + 255) / 256, 256, 0, st>>>(h->ix, h->hx, h->hy, h->hr2, h->n_hits);
    h->launches += 2;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ the peak-driven list kernel
struct PeakListParams {
    GridDev g;
    HitIndexDev ix;
    ApproxBin ab;
    const float *phic; // [n_phi] bin-centre angles
    uint32_t n_hits;
    const uint32_t *bin, *mask; // reported peaks (k_compact)
    const DevCounters *counters;
    uint32_t cap_peaks;
    uint32_t *peak_len; // [cap_peaks] list length
    uint32_t *peak_pos; // [cap_peaks] 0: the list is in the peak's slot in ascending order, PL_UNSORTED: in
                        // candidate order, PL_SLOW: it is not there
    uint32_t *slots;    // [cap_peaks][slot] staging
    uint32_t slot;
    unsigned long long *n_list_evals; // candidates evaluated
    unsigned long long *work;         // next peak to hand out (zeroed per hough_peaks)
    float dk, inv_dk_w; // kappa bin width (binary32) and its reciprocal (window arithmetic only)
    float edge_rel;     // slack on a bin edge, in bins
};

// The window arithmetic only has to produce SUPERSETS, with the margins stated below; it uses the
// approximate division / square root units (2 ulp) and a polynomial arc sine instead of the IEEE
// routines (a third of the instructions).  Nothing here decides a list entry: the exact recipe does.
__device__ __forceinline__ float fast_sqrt(float x)
{
    float r;
    asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
// asin on [-1, 1]: pi/2 - sqrt(1 - |x|) P7(|x|) (Abramowitz & Stegun 4.4.46, |error| <= 2e-8 in exact
// arithmetic, < 5e-7 in binary32 with the approximate square root; the windows carry 2e-5 rad of slack)
__device__ __forceinline__ float fast_asin(float x)
{
    const float a = fabsf(x);
    float p = -0.0012624911f;
    p = __fmaf_rn(p, a, 0.0066700901f);
    p = __fmaf_rn(p, a, -0.0170881256f);
    p = __fmaf_rn(p, a, 0.0308918810f);
    p = __fmaf_rn(p, a, -0.0501743046f);
    p = __fmaf_rn(p, a, 0.0889789874f);
    p = __fmaf_rn(p, a, -0.2145988016f);
    p = __fmaf_rn(p, a, 1.5707963050f);
    const float r = 1.5707963268f - fast_sqrt(fmaxf(1.0f - a, 0.0f)) * p;
    return copysignf(r, x);
}

struct PlWin { // an arc of azimuth bins [b, b + n) on the ring of NA bins; n = 0: absent
    int b, n;
};
// Azimuth window [a_lo, a_hi] (radians, a_lo <= a_hi, slack included) -> the bins it touches.
__device__ __forceinline__ PlWin window_bins(float a_lo, float a_hi, float na_scale, int NA)
{
    const float t0 = floorf((a_lo + PI_F) * na_scale), t1 = floorf((a_hi + PI_F) * na_scale);
    const float span = t1 - t0 + 1.0f;
    PlWin w;
    if (!(span < (float)NA)) { // also NaN: the whole ring
        w.b = 0;
        w.n = NA;
        return w;
    }
    w.b = (int)t0 & (NA - 1);
    w.n = (int)span;
    return w;
}
// If the two arcs overlap, a becomes their union and b disappears (so that no hit is a candidate twice).
__device__ __forceinline__ void merge_windows(PlWin &a, PlWin &b, int NA)
{
    if (a.n == 0 || b.n == 0)
        return;
    const int d = (b.b - a.b) & (NA - 1), d2 = (a.b - b.b) & (NA - 1);
    if (d < a.n) {
        a.n = max(a.n, d + b.n);
        b.n = 0;
    } else if (d2 < b.n) {
        a.b = b.b;
        a.n = max(b.n, d2 + a.n);
        b.n = 0;
    }
    if (a.n >= NA) {
        a.b = 0;
        a.n = NA;
    }
}

#define PL_QCAP 40 // words per thread: queued candidate ranges (first rank | count << 20) from the bottom,
                   // the list being collected from the top
#define PL_LCAP 24 // entries of a list collected (and sorted) in shared memory; longer lists spill to the slot
#define PL_UNSORTED 1u

__global__ void __launch_bounds__(PL_THREADS) k_peak_lists(const PeakListParams p)
{
    __shared__ uint32_t s_lbase[34]; // rank of the first hit of layer label l (label nL = the wild hits)
    __shared__ float s_ra[32], s_rb[32], s_ira[32], s_irb[32];
    __shared__ uint32_t s_q[PL_QCAP][PL_THREADS];

    const GridDev &g = p.g;
    const HitIndexDev &ix = p.ix;
    const int tid = threadIdx.x, lane = tid & 31;
    const int NA = ix.NA, nL = ix.n_keys / NA - 1;
    pdl_wait();
    pdl_trigger();
    if (tid <= nL)
        s_lbase[tid] = ix.bin_start[tid * NA];
    if (tid == nL + 1)
        s_lbase[tid] = ix.bin_start[nL * NA + 1];
    if (tid < nL) {
        const float ra = __uint_as_float(~ix.layer_r[2 * tid]) * (1.0f - 4e-6f);
        const float rb = __uint_as_float(ix.layer_r[2 * tid + 1]) * (1.0f + 4e-6f);
        s_ra[tid] = ra;
        s_rb[tid] = rb;
        s_ira[tid] = 1.0f / ra;
        s_irb[tid] = 1.0f / rb;
    }
    __syncthreads();
    const float na_scale = (float)NA * 0.15915494309189535f;
    const uint32_t n_rep = min(p.counters->n_peaks, p.cap_peaks);
    const int nk = g.n_kappa;
    const float klo = g.klo, khi = g.khi, inv_dk = g.inv_dk;
    const float U = 5.9604645e-08f; // 2^-24
    unsigned long long evals = 0;

    // the warps draw 32 peaks at a time from a global counter (lists differ in length: a static split
    // leaves the last wave of CTAs a third empty)
    for (;;) {
        unsigned long long base = 0;
        if (lane == 0)
            base = atomicAdd(p.work, 32ull);
        base = __shfl_sync(0xffffffffu, base, 0);
        if (base >= n_rep)
            break;
        const uint32_t pk = (uint32_t)base + lane;
        if (pk >= n_rep)
            continue;
        const uint32_t lin = p.bin[pk], pmask = p.mask[pk];
        const uint32_t k = lin % (uint32_t)nk, row = lin / (uint32_t)nk;
        const uint32_t j = row % (uint32_t)g.n_d0, i = row / (uint32_t)g.n_d0;
        const float c_sn = g.sn[i], c_cs = g.cs[i], c_d0 = g.d0c[j], c_2d0 = g.twod0[j], c_d0sq = g.d0sq[j];
        const float phi0 = p.phic[i], ad0 = fabsf(c_d0);
        uint32_t *slot = p.slots + (size_t)pk * p.slot;
        uint32_t cnt = 0;
        // the bin's kappa interval
        float ka = __fmaf_rn((float)k, p.dk, klo), kb = __fmaf_rn((float)(k + 1u), p.dk, klo);
        if (k == 0u)
            ka = fminf(ka, klo);
        if (k + 1u == (uint32_t)nk)
            kb = fmaxf(kb, khi);
        const float Kp = 1.01f * g.kabs + p.dk;
        const bool ab_ok = p.ab.ok != 0;
        int nq = 0;         // queued ranges of the current pass
        bool spill = false; // the list has outgrown shared memory
        uint32_t n_sm = 0;  // its entries in shared memory when that happened

        // one candidate with the exact recipe (the fixed-point estimate first where it is admissible,
        // as in the vote: hough_device.cuh approx_bin)
        auto consider = [&](const float4 r) {
            const float a = __fmul_rn(r.x, c_sn);
            const float b = __fmul_rn(r.y, c_cs);
            const float sv = __fsub_rn(b, a);
            const float ee = __fsub_rn(sv, c_d0);
            const float den = __fadd_rn(__fsub_rn(r.z, __fmul_rn(c_2d0, sv)), c_d0sq);
            bool match;
            uint32_t tb = 0;
            const bool fast = ab_ok && !hit_is_wild(r.z);
            if (fast)
                tb = approx_bin(ee, den, p.ab.c1, p.ab.c0);
            if (fast && !(tb < p.ab.lim)) {
                match = false;
            } else if (fast && (tb & 0xffffu) >= p.ab.edge) {
                match = (tb >> APPROX_FRAC_BITS) == k;
            } else {
                const float kappa = __fdiv_rn(__fadd_rn(ee, ee), den);
                match = (kappa >= klo) && (kappa < khi) && (uint32_t)kappa_bin(kappa, klo, inv_dk, nk - 1) == k;
            }
            if (match) {
                // collected at the top of the thread's queue words while it stays clear of the queued
                // ranges; after that straight into the slot (candidate order: k_copy_lists sorts those)
                const uint32_t hit = __float_as_uint(r.w);
                if (!spill && cnt < PL_LCAP && (uint32_t)nq + cnt < PL_QCAP) {
                    s_q[PL_QCAP - 1 - cnt][tid] = hit;
                } else {
                    if (!spill) {
                        spill = true;
                        n_sm = cnt;
                    }
                    if (cnt < p.slot)
                        slot[cnt] = hit;
                }
                ++cnt;
            }
        };

        int l = 0;
        while (l <= nL) {
            // ---- queue the candidate ranges (physical ranks of the key-ordered records) of as many
            // layers as fit; a range too long for a queue entry is walked on the spot
            nq = 0;
            auto push = [&](uint32_t rank0, uint32_t n) {
                if (n > 4095u) {
                    if (!spill) { // matches found now must not grow into the words the next pushes use
                        spill = true;
                        n_sm = cnt;
                    }
                    for (uint32_t c = 0; c < n; ++c)
                        consider(ix.rec[rank0 + c]);
                } else if (n) {
                    s_q[nq++][tid] = rank0 | (n << 20);
                }
                evals += n;
            };
            // virtual ranks [q0, q0 + n) of a layer whose hits are thought repeated twice
            auto push_virtual = [&](uint32_t lbase, uint32_t lcnt, uint32_t q0, uint32_t n) {
                if (q0 >= lcnt)
                    q0 -= lcnt;
                const uint32_t first = min(n, lcnt - q0);
                push(lbase + q0, first);
                push(lbase, n - first);
            };
            for (; l <= nL && (uint32_t)nq + 6u + (spill ? n_sm : min(cnt, (uint32_t)PL_LCAP)) <= PL_QCAP; ++l) {
                const uint32_t lbase = s_lbase[l], lcnt = s_lbase[l + 1] - lbase;
                if (l == nL) { // the wild hits (outside the index's numeric range): candidates of every peak
                    push(lbase, lcnt);
                    continue;
                }
                if (!((pmask >> l) & 1u) || !lcnt)
                    continue;
                const float ra = s_ra[l], rb = s_rb[l], ira = s_ira[l], irb = s_irb[l];
                // binary32 evaluation error of the recipe: |kappa_fp - kappa| <= errnum / den + 2 U K
                const float Gm = 1.4143f * rb + ad0;
                const float errnum = 2.0f * (12.0f * U * Gm + 16.0f * U * Kp * Gm * Gm);
                const float Lmin = fmaxf(0.0f, fmaxf(ra - ad0 * (1.0f + 1e-6f), ad0 * (1.0f - 1e-6f) - rb));
                const float L0sq = errnum * p.inv_dk_w * (1.0f + 1e-6f); // den >= L0sq: the error stays below one bin
                float D = Lmin * Lmin;
                const bool prox = !(D >= L0sq);
                if (prox)
                    D = L0sq;
                const float slack = __fdividef(errnum, D) * (1.0f + 1e-6f) + 2.0f * U * Kp + p.edge_rel * p.dk;
                const float k1 = ka - slack, k2 = kb + slack;
                const float g1 = __fmaf_rn(k1, c_d0, 1.0f), g2 = __fmaf_rn(k2, c_d0, 1.0f);
                bool whole = !(g1 > 0.01f && g2 > 0.01f);
                PlWin w0 = {0, 0}, w1 = {0, 0}, w2 = {0, 0};
                if (!whole) {
                    const float h1 = __fdividef(0.5f, g1), h2 = __fdividef(0.5f, g2);
                    const float A1 = c_d0 * __fmaf_rn(k1, c_d0, 2.0f) * h1, B1 = k1 * h1;
                    const float A2 = c_d0 * __fmaf_rn(k2, c_d0, 2.0f) * h2, B2 = k2 * h2;
                    float wlo = fminf(A1 * ira + B1 * ra, A1 * irb + B1 * rb);
                    float whi = fmaxf(A2 * ira + B2 * ra, A2 * irb + B2 * rb);
                    // W(k1, r) has its minimum 2 sqrt(A B) at r^2 = A / B (A, B > 0); the test interval is
                    // widened so that a rounded end point cannot hide the stationary point
                    if (A1 > 0.0f && B1 > 0.0f && A1 > 0.999f * ra * ra * B1 && A1 < 1.001f * rb * rb * B1)
                        wlo = fminf(wlo, 2.0f * fast_sqrt(A1 * B1) * (1.0f - 2e-6f));
                    // W(k2, r) has its maximum -2 sqrt(A B) at r^2 = A / B (A, B < 0)
                    if (A2 < 0.0f && B2 < 0.0f && A2 < 0.999f * ra * ra * B2 && A2 > 1.001f * rb * rb * B2)
                        whi = fmaxf(whi, -2.0f * fast_sqrt(A2 * B2) * (1.0f - 2e-6f));
                    const float ew = 1e-5f * (1.0f + fmaxf(fabsf(wlo), fabsf(whi)));
                    wlo -= ew;
                    whi += ew;
                    if (!(fabsf(wlo) < 3.0e38f) || !(fabsf(whi) < 3.0e38f) || !(wlo <= whi)) {
                        whole = true; // inf / NaN somewhere: no bound
                    } else if (!(wlo > 1.0f) && !(whi < -1.0f)) {
                        const float tlo = fast_asin(fmaxf(wlo, -1.0f)) - 5e-5f, thi = fast_asin(fminf(whi, 1.0f)) + 5e-5f;
                        w0 = window_bins(phi0 + tlo, phi0 + thi, na_scale, NA);
                        w1 = window_bins(phi0 + PI_F - thi, phi0 + PI_F - tlo, na_scale, NA);
                    }
                }
                if (!whole && prox) {
                    // hits closer than L0 to P0 (azimuth of P0 = phi0 +- pi/2): |X - P0|^2 >= 4 r |d0| sin^2(dpsi / 2)
                    const float arg = 0.5051f * fast_sqrt(__fdividef(L0sq, ra * ad0));
                    if (!(arg < 0.999f)) {
                        whole = true;
                    } else {
                        const float hw = 2.0f * fast_asin(arg) + 5e-5f, psi = phi0 + (c_d0 >= 0.0f ? 1.5707963f : -1.5707963f);
                        w2 = window_bins(psi - hw, psi + hw, na_scale, NA);
                    }
                }
                if (!whole) { // disjoint arcs
                    merge_windows(w0, w1, NA);
                    if (w2.n) {
                        merge_windows(w0, w2, NA);
                        merge_windows(w1, w2, NA);
                        merge_windows(w0, w1, NA);
                    }
                    whole = w0.n >= NA || w1.n >= NA || w2.n >= NA;
                }
                if (whole) {
                    push(lbase, lcnt);
                    continue;
                }
                // bins -> virtual ranks of the layer (its hits repeated twice, so an arc never wraps)
                const uint32_t *bs = ix.bin_start + l * NA;
                auto P2 = [&](int b) -> uint32_t { return b <= NA ? bs[b] - lbase : lcnt + bs[b - NA] - lbase; };
                if (w0.n) {
                    const uint32_t q0 = P2(w0.b);
                    push_virtual(lbase, lcnt, q0, P2(w0.b + w0.n) - q0);
                }
                if (w1.n) {
                    const uint32_t q0 = P2(w1.b);
                    push_virtual(lbase, lcnt, q0, P2(w1.b + w1.n) - q0);
                }
                if (w2.n) {
                    const uint32_t q0 = P2(w2.b);
                    push_virtual(lbase, lcnt, q0, P2(w2.b + w2.n) - q0);
                }
            }
            // ---- one flat loop over the queued candidates; the next record is loaded before the
            // current one is evaluated
            int e = 0;
            uint32_t rem = 0, rank = 0;
            float4 nxt = make_float4(0.f, 0.f, 0.f, 0.f);
            bool have = false;
            auto advance = [&]() {
                if (rem == 0u) {
                    if (e == nq) {
                        have = false;
                        return;
                    }
                    const uint32_t en = s_q[e++][tid];
                    rank = en & 0xfffffu;
                    rem = en >> 20;
                }
                nxt = ix.rec[rank];
                ++rank;
                --rem;
                have = true;
            };
            advance();
            while (have) {
                const float4 r = nxt;
                advance();
                consider(r);
            }
        }
        // ---- the list: sorted here when all of it is in shared memory (insertion sort, one thread per
        // list), then written to the peak's slot
        auto L = [&](uint32_t c) -> uint32_t & { return s_q[PL_QCAP - 1 - c][tid]; };
        const uint32_t in_sm = spill ? n_sm : cnt;
        if (!spill)
            for (uint32_t a = 1; a < cnt; ++a) {
                const uint32_t v = L(a);
                uint32_t b = a;
                while (b > 0 && L(b - 1) > v) {
                    L(b) = L(b - 1);
                    --b;
                }
                L(b) = v;
            }
        for (uint32_t c = 0; c < in_sm && c < p.slot; ++c)
            slot[c] = L(c);
        p.peak_len[pk] = cnt;
        p.peak_pos[pk] = cnt > p.slot ? PL_SLOW : spill ? PL_UNSORTED : 0u;
    }
    for (int o = 16; o > 0; o >>= 1)
        evals += __shfl_xor_sync(0xffffffffu, evals, o);
    if (lane == 0 && evals)
        atomicAdd(p.n_list_evals, evals);
}

// ------------------------------------------------------------------ placement
struct ListCopyParams {
    GridDev g;
    const float *hx, *hy, *hr2;
    const uint32_t *hbit;
    uint32_t n_hits;
    const DevCounters *counters;
    uint32_t cap_peaks;
    const uint32_t *bin;
    const uint32_t *peak_len, *peak_pos, *slots;
    uint32_t slot;
    const unsigned long long *hit_offset;
    uint32_t *hit_index;
    unsigned short *hit_index16; // optional 16-bit copy of the entries (NULL: not wanted)
    unsigned long long cap_hits;
};

// hit_index[hit_offset[p] ..] = the staged list of peak p in ascending hit index (half a warp per
// peak): a plain copy where k_peak_lists has sorted it, ranks by counting (hit indices are distinct)
// where the slot is in candidate order (PL_UNSORTED); a peak without a staged list (PL_SLOW) is
// written straight from the hits in index order by a whole warp.
template <int MODE>
__global__ void __launch_bounds__(256) k_copy_lists(const ListCopyParams p)
{
    const GridDev &g = p.g;
    const int lane = threadIdx.x & 31, hl = lane & 15;
    const unsigned hmask = 0xffffu << (lane & 16);
    pdl_wait();
    pdl_trigger();
    const uint32_t n = min(p.counters->n_peaks, p.cap_peaks);
    const uint32_t halves = (gridDim.x * blockDim.x) >> 4;
    auto put = [&](unsigned long long pos, uint32_t hit) {
        p.hit_index[pos] = hit;
        if (p.hit_index16)
            p.hit_index16[pos] = (unsigned short)hit;
    };
    // two pairs of peaks per warp and round (A and B), so that their loads are in flight together
    for (uint32_t pk0 = (((blockIdx.x * blockDim.x + threadIdx.x) >> 5) << 1); pk0 < n; pk0 += 2 * halves) {
        uint32_t pk[2], pos[2], len[2], v[2];
        unsigned long long dst[2];
        const uint32_t *src[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            pk[u] = pk0 + (uint32_t)u * halves + (lane >> 4);
            pos[u] = 0, len[u] = 0, dst[u] = 0;
            if (pk[u] < n) {
                pos[u] = p.peak_pos[pk[u]];
                len[u] = p.peak_len[pk[u]];
                dst[u] = p.hit_offset[pk[u]];
            }
            src[u] = p.slots + (size_t)pk[u] * p.slot;
        }
#pragma unroll
        for (int u = 0; u < 2; ++u)
            v[u] = (pos[u] != PL_SLOW && hl < len[u]) ? src[u][hl] : 0xffffffffu;
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            if (pos[u] == PL_SLOW || len[u] == 0u)
                continue;
            if (pos[u] == 0u) { // already in ascending order (sorted by k_peak_lists): a plain copy
                if (hl < len[u] && dst[u] + hl < p.cap_hits)
                    put(dst[u] + hl, v[u]);
                for (uint32_t a = hl + 16; a < len[u]; a += 16)
                    if (dst[u] + a < p.cap_hits)
                        put(dst[u] + a, src[u][a]);
            } else if (len[u] <= 16u) { // one entry per lane, ranks through shuffles
                uint32_t rk = 0;
#pragma unroll
                for (int b = 0; b < 16; ++b)
                    rk += __shfl_sync(hmask, v[u], b, 16) < v[u] ? 1u : 0u;
                if (hl < len[u] && dst[u] + rk < p.cap_hits)
                    put(dst[u] + rk, v[u]);
            } else {
                for (uint32_t a = hl; a < len[u]; a += 16) {
                    const uint32_t w = src[u][a];
                    uint32_t rk = 0;
                    for (uint32_t b = 0; b < len[u]; ++b)
                        rk += src[u][b] < w ? 1u : 0u;
                    if (dst[u] + rk < p.cap_hits)
                        put(dst[u] + rk, w);
                }
            }
        }
        // slow peaks of these pairs (rare), one after the other, by the whole warp
        if (!__any_sync(0xffffffffu, (pos[0] == PL_SLOW && len[0] != 0u) || (pos[1] == PL_SLOW && len[1] != 0u)))
            continue;
        for (int which = 0; which < 4; ++which) {
            const int u = which >> 1;
            const uint32_t spos = __shfl_sync(0xffffffffu, u ? pos[1] : pos[0], (which & 1) * 16);
            const uint32_t slen = __shfl_sync(0xffffffffu, u ? len[1] : len[0], (which & 1) * 16);
            const uint32_t spk = pk0 + (uint32_t)u * halves + (uint32_t)(which & 1);
            if (spk >= n || spos != PL_SLOW || slen == 0u)
                continue;
            unsigned long long w = p.hit_offset[spk];
            if (w >= p.cap_hits)
                continue;
            const uint32_t lin = p.bin[spk];
            const uint32_t k = lin % (uint32_t)g.n_kappa, row = lin / (uint32_t)g.n_kappa;
            const uint32_t j = row % (uint32_t)g.n_d0, i = row / (uint32_t)g.n_d0;
            const CellConst cc = cell_const(g, MODE, (int)i, (int)j);
            for (uint32_t base = 0; base < p.n_hits; base += 32) {
                const uint32_t hidx = base + lane;
                bool in = false;
                if (hidx < p.n_hits && p.hbit[hidx] != 0u) {
                    int k0, k1;
                    if (variant_bins<MODE>(p.hx[hidx], p.hy[hidx], p.hr2[hidx], cc, g.klo, g.khi, g.inv_dk,
                                           g.n_kappa - 1, k0, k1))
                        in = (uint32_t)k0 <= k && k <= (uint32_t)k1;
                }
                const unsigned bal = __ballot_sync(0xffffffffu, in);
                if (in) {
                    const unsigned long long q = w + __popc(bal & ((1u << lane) - 1u));
                    if (q < p.cap_hits)
                        put(q, hidx);
                }
                w += __popc(bal);
            }
        }
    }
}

// Entries of one staging slot: the three entry arrays of the legacy list sweep (3 x cap_hits words,
// contiguous in the workspace) shared out among cap_peaks peaks.
static uint32_t slot_entries(const hough_handle *h)
{
    const unsigned long long per = 3ull * h->cfg.cap_hits / h->cfg.cap_peaks;
    return (uint32_t)(per < PL_MAXSLOT ? per : PL_MAXSLOT);
}

cudaError_t launch_peak_lists(hough_handle *h, const hough_peaks_out *out, cudaStream_t st)
{
    if (h->n_hits == 0) // no event (hough_set_accumulator): every list is empty, the index is not built
        return cudaMemsetAsync(h->peak_len, 0, (size_t)h->cfg.cap_peaks * 4, st);
    PeakListParams p;
    p.g = h->g;
    p.ix = h->ix;
    p.phic = h->t_phic;
    p.n_hits = h->n_hits;
    p.bin = out->bin;
    p.mask = out->mask;
    p.counters = h->counters;
    p.cap_peaks = h->cfg.cap_peaks;
    p.peak_len = h->peak_len;
    p.peak_pos = h->list_len;
    p.slots = h->ent_sub;
    p.slot = slot_entries(h);
    p.n_list_evals = &h->counters->n_list_evals;
    p.ab = h->ab;
    p.dk = (float)(((double)h->g.khi - (double)h->g.klo) / (double)h->g.n_kappa);
    p.inv_dk_w = (float)((double)h->g.n_kappa / ((double)h->g.khi - (double)h->g.klo));
    // bin-edge slack in bins: the roundings of (kappa - klo) * inv_dk and of the edges computed here
    const double A = (double)h->g.kabs / ((double)h->g.khi - (double)h->g.klo);
    p.edge_rel = (float)(0.01 + 4e-7 * h->g.n_kappa * (1.0 + A));
    p.work = h->n_pairs;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_peak_lists, PL_THREADS, 0) != cudaSuccess || per_sm < 1)
        per_sm = 4;
    launch_pdl(k_peak_lists, dim3(h->n_sms * per_sm), dim3(PL_THREADS), 0, st, p);
    h->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_copy_lists(hough_handle *h, const hough_peaks_out *out, cudaStream_t st)
{
    ListCopyParams p;
    p.g = h->g;
    p.hx = h->hx;
    p.hy = h->hy;
    p.hr2 = h->hr2;
    p.hbit = h->hbit;
    p.n_hits = h->n_hits;
    p.counters = h->counters;
    p.cap_peaks = h->cfg.cap_peaks;
    p.bin = out->bin;
    p.peak_len = h->peak_len;
    p.peak_pos = h->list_len;
    p.slots = h->ent_sub;
    p.slot = slot_entries(h);
    p.hit_offset = reinterpret_cast<const unsigned long long *>(out->hit_offset);
    p.hit_index = out->hit_index;
    p.hit_index16 = (out->hit_index16 && h->n_hits <= 65536u) ? out->hit_index16 : nullptr;
    p.cap_hits = h->cfg.cap_hits;
    if (h->mode == VOTE_LINE)
        launch_pdl(k_copy_lists<VOTE_LINE>, dim3(h->n_sms * 16), dim3(256), 0, st, p);
    else if (h->mode == VOTE_INTERVAL)
        launch_pdl(k_copy_lists<VOTE_INTERVAL>, dim3(h->n_sms * 16), dim3(256), 0, st, p);
    else
        launch_pdl(k_copy_lists<VOTE_CENTRE>, dim3(h->n_sms * 16), dim3(256), 0, st, p);
    h->launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ generic lists (vote variants, f3)
// One warp per reported peak counts, over all hits, those whose vote at the peak's cell covers
// the peak's bin; every list is then written by k_copy_lists' whole-warp path (PL_SLOW).
template <int MODE>
__global__ void __launch_bounds__(256) k_list_count(const ListCopyParams p, uint32_t *peak_len, uint32_t *peak_pos,
                                                    unsigned long long *n_list_evals)
{
    const GridDev &g = p.g;
    const int lane = threadIdx.x & 31;
    const uint32_t n = min(p.counters->n_peaks, p.cap_peaks);
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t pk = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; pk < n; pk += warps) {
        const uint32_t lin = p.bin[pk];
        const uint32_t k = lin % (uint32_t)g.n_kappa, row = lin / (uint32_t)g.n_kappa;
        const uint32_t j = row % (uint32_t)g.n_d0, i = row / (uint32_t)g.n_d0;
        const CellConst cc = cell_const(g, MODE, (int)i, (int)j);
        uint32_t cnt = 0;
        for (uint32_t hidx = lane; hidx < p.n_hits; hidx += 32) {
            int k0, k1;
            if (p.hbit[hidx] != 0u && variant_bins<MODE>(p.hx[hidx], p.hy[hidx], p.hr2[hidx], cc, g.klo, g.khi,
                                                         g.inv_dk, g.n_kappa - 1, k0, k1))
                cnt += ((uint32_t)k0 <= k && k <= (uint32_t)k1) ? 1u : 0u;
        }
        for (int o = 16; o > 0; o >>= 1)
            cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
        if (lane == 0) {
            peak_len[pk] = cnt;
            peak_pos[pk] = PL_SLOW;
            atomicAdd(n_list_evals, (unsigned long long)p.n_hits);
        }
    }
}

cudaError_t launch_lists_generic(hough_handle *h, const hough_peaks_out *out, cudaStream_t st)
{
    if (h->n_hits == 0)
        return cudaMemsetAsync(h->peak_len, 0, (size_t)h->cfg.cap_peaks * 4, st);
    ListCopyParams p;
    p.g = h->g;
    p.hx = h->hx;
    p.hy = h->hy;
    p.hr2 = h->hr2;
    p.hbit = h->hbit;
    p.n_hits = h->n_hits;
    p.counters = h->counters;
    p.cap_peaks = h->cfg.cap_peaks;
    p.bin = out->bin;
    p.peak_len = p.peak_pos = p.slots = nullptr;
    p.slot = 0;
    p.hit_offset = nullptr;
    p.hit_index = nullptr;
    p.hit_index16 = nullptr;
    p.cap_hits = 0;
    unsigned long long *ev = &h->counters->n_list_evals;
    if (h->mode == VOTE_LINE)
        k_list_count<VOTE_LINE><<<h->n_sms * 16, 256, 0, st>>>(p, h->peak_len, h->list_len, ev);
    else if (h->mode == VOTE_INTERVAL)
        k_list_count<VOTE_INTERVAL><<<h->n_sms * 16, 256, 0, st>>>(p, h->peak_len, h->list_len, ev);
    else
        k_list_count<VOTE_CENTRE><<<h->n_sms * 16, 256, 0, st>>>(p, h->peak_len, h->list_len, ev);
    h->launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ list check (HOUGH_OPT_CHECK_LISTS)
// One warp per reported peak: its list, as written to the caller's arrays, is strictly ascending, names
// real hits, and the OR of their layer bits is the peak's mask.  Reads only final outputs, so it serves
// every list path (peak-driven, list sweep, vote variants).
__global__ void __launch_bounds__(256) k_check_lists(const hough_counts *counts_in, hough_counts *counts_out,
                                                     uint32_t cap_peaks, unsigned long long cap_hits,
                                                     const uint32_t *__restrict__ mask,
                                                     const unsigned long long *__restrict__ hit_offset,
                                                     const uint32_t *__restrict__ hit_index,
                                                     const uint32_t *__restrict__ hbit, uint32_t n_hits)
{
    const int lane = threadIdx.x & 31;
    const uint32_t n = min(counts_in->n_peaks, cap_peaks);
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    bool bad = false;
    for (uint32_t pk = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; pk < n; pk += warps) {
        const unsigned long long a = hit_offset[pk], b = hit_offset[pk + 1];
        if (b < a) {
            bad = true;
            continue;
        }
        if (b > cap_hits) // cut by the capacity: not a complete list
            continue;
        uint32_t m = 0;
        for (unsigned long long q = a + lane; q < b; q += 32) {
            const uint32_t hit = hit_index[q];
            if (hit >= n_hits || (q > a && hit_index[q - 1] >= hit))
                bad = true;
            else
                m |= hbit[hit];
        }
        for (int o = 16; o > 0; o >>= 1)
            m |= __shfl_xor_sync(0xffffffffu, m, o);
        if (m != mask[pk])
            bad = true;
    }
    if (__any_sync(0xffffffffu, bad) && lane == 0)
        atomicOr(&counts_out->flags, HOUGH_LIST_MISMATCH);
}

cudaError_t launch_check_lists(hough_handle *h, const hough_peaks_out *out, cudaStream_t st)
{
    if (h->n_hits == 0) // no event behind the accumulator (hough_set_accumulator): the lists are empty by design
        return cudaSuccess;
    k_check_lists<<<h->n_sms * 8, 256, 0, st>>>(out->counts, out->counts, h->cfg.cap_peaks,
                                                (unsigned long long)h->cfg.cap_hits, out->mask,
                                                reinterpret_cast<const unsigned long long *>(out->hit_offset),
                                                out->hit_index, h->hbit, h->n_hits);
    h->launches += 1;
    return cudaGetLastError();
}
