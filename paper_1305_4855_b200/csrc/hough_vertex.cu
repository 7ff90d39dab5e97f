// hough_vertex.cu -- f1, the SECOND Hough transform, over the peaks of the first
// (section 9; recipe E3 of DESIGN.md section 8).
//
// A reported peak (i, j, k) is the point (phi0_i, d0_j) of the parameter space; it votes along
// the line d0_j = -xv sin(phi0_i) + yv cos(phi0_i) of the (xv, yv) plane, once per bin centre of
// the axis the line is less steep against, into a uint32 count accumulator.  Five small kernels:
//   k_vertex_vote     peaks -> counts (a shared-memory copy of the accumulator per CTA when it
//                     fits, flushed with one global atomic per non-zero bin; global atomics otherwise)
//   k_vertex_flags    3x3 local-maximum test per bin, one flag byte per bin, count per block
//   k_vertex_compact  ordered compaction of the flagged bins (block bases from the block counts)
//   k_vertex_members<false>  list length per reported vertex (one CTA per vertex sweeps the peaks)
//   k_vertex_members<true>   offsets from the lengths, then the ordered fill
// Every floating-point operation that decides a bin is one binary32 round-to-nearest operation in
// the recipe's order; the bin-centre tables are computed in binary64 exactly as the recipe states.
#include "hough_device.cuh"

#define VX_THREADS 256
#define VX_SMEM_BINS 8192 // accumulator copy in shared memory up to this many bins (32 KB + <= 16 KB of tables)

struct VertexParams {
    // first transform
    int n_phi, n_d0, n_kappa;
    double d0_min, d0_max;
    const float *sn, *cs, *d0c;
    const uint32_t *peak_bin;
    const hough_counts *peak_counts;
    uint32_t cap_peaks;
    // vertex grid
    double x_min, x_max, y_min, y_max;
    int n_x, n_y;
    uint32_t V_min;
    float xlo, xhi, inv_dx, ylo, yhi, inv_dy;
    // scratch
    uint32_t *vacc;        // [n_x * n_y]
    unsigned char *flag;   // [n_x * n_y]
    uint32_t *block_cnt;   // [n_blocks]
    uint32_t *member_len;  // [cap_vertices]
    // outputs
    uint32_t cap_vertices;
    unsigned long long cap_members;
    uint32_t *out_bin, *out_count;
    unsigned long long *member_offset;
    uint32_t *member_index;
    hough_vertex_counts *counts;
};

__device__ __forceinline__ float vx_centre(double lo, double hi, int n, int q)
{
    return (float)(lo + ((double)q + 0.5) * (hi - lo) / (double)n);
}

// V2 for one peak cell at index q of the axis it iterates: the bin along the other axis, or -1
__device__ __forceinline__ int vx_vote_one(const VertexParams &p, float sn, float cs, float d, bool steep, float cq)
{
    if (!steep) {
        const float t = __fmul_rn(cq, sn);
        const float u = __fadd_rn(d, t);
        const float yv = __fdiv_rn(u, cs);
        if (!((yv >= p.ylo) && (yv < p.yhi)))
            return -1;
        return min(__float2int_rz(__fmul_rn(__fsub_rn(yv, p.ylo), p.inv_dy)), p.n_y - 1);
    }
    const float t = __fmul_rn(cq, cs);
    const float u = __fsub_rn(t, d);
    const float xv = __fdiv_rn(u, sn);
    if (!((xv >= p.xlo) && (xv < p.xhi)))
        return -1;
    return min(__float2int_rz(__fmul_rn(__fsub_rn(xv, p.xlo), p.inv_dx)), p.n_x - 1);
}

template <bool SMEM>
__global__ void __launch_bounds__(VX_THREADS) k_vertex_vote(const VertexParams p)
{
    extern __shared__ uint32_t s_dyn[];
    const int n_bins = p.n_x * p.n_y;
    float *s_xc = reinterpret_cast<float *>(s_dyn);
    float *s_yc = s_xc + p.n_x;
    uint32_t *s_acc = reinterpret_cast<uint32_t *>(s_yc + p.n_y);
    for (int a = threadIdx.x; a < p.n_x; a += blockDim.x)
        s_xc[a] = vx_centre(p.x_min, p.x_max, p.n_x, a);
    for (int b = threadIdx.x; b < p.n_y; b += blockDim.x)
        s_yc[b] = vx_centre(p.y_min, p.y_max, p.n_y, b);
    if (SMEM)
        for (int q = threadIdx.x; q < n_bins; q += blockDim.x)
            s_acc[q] = 0u;
    __syncthreads();
    const uint32_t n_rep = min(p.peak_counts->n_peaks, p.cap_peaks);
    // a group of 8 lanes shares one peak and strides the iterated axis.  The vote of a peak depends on
    // its (phi0, d0) cell only and the peaks are in ascending lin, so the peaks of one cell are
    // neighbours in the list: the first of them votes for all, with their number as the weight
    const uint32_t sub = threadIdx.x & 7u;
    const uint32_t grp = (blockIdx.x * blockDim.x + threadIdx.x) >> 3, n_grp = (gridDim.x * blockDim.x) >> 3;
    unsigned int votes = 0;
    for (uint32_t pk = grp; pk < n_rep; pk += n_grp) {
        const uint32_t row = p.peak_bin[pk] / (uint32_t)p.n_kappa;
        if (pk > 0 && p.peak_bin[pk - 1] / (uint32_t)p.n_kappa == row)
            continue;
        uint32_t weight = 1;
        while (pk + weight < n_rep && p.peak_bin[pk + weight] / (uint32_t)p.n_kappa == row)
            ++weight;
        const uint32_t j = row % (uint32_t)p.n_d0, i = row / (uint32_t)p.n_d0;
        const float sn = p.sn[i], cs = p.cs[i], d = p.d0c[j];
        const bool steep = !(fabsf(cs) >= fabsf(sn));
        const int nq = steep ? p.n_y : p.n_x;
        for (int q = (int)sub; q < nq; q += 8) {
            const int o = vx_vote_one(p, sn, cs, d, steep, steep ? s_yc[q] : s_xc[q]);
            if (o < 0)
                continue;
            const int lin = steep ? o * p.n_y + q : q * p.n_y + o;
            if (SMEM)
                atomicAdd(&s_acc[lin], weight);
            else
                atomicAdd(&p.vacc[lin], weight);
            votes += weight;
        }
    }
    for (int o = 16; o > 0; o >>= 1)
        votes += __shfl_xor_sync(0xffffffffu, votes, o);
    if ((threadIdx.x & 31) == 0 && votes)
        atomicAdd(reinterpret_cast<unsigned long long *>(&p.counts->n_vertex_votes), (unsigned long long)votes);
    if (SMEM) {
        __syncthreads();
        for (int q = threadIdx.x; q < n_bins; q += blockDim.x)
            if (s_acc[q])
                atomicAdd(&p.vacc[q], s_acc[q]);
    }
}

// V3: one thread per bin
__global__ void __launch_bounds__(VX_THREADS) k_vertex_flags(const VertexParams p)
{
    __shared__ uint32_t s_cnt;
    if (threadIdx.x == 0)
        s_cnt = 0u;
    __syncthreads();
    const int n_bins = p.n_x * p.n_y;
    const int lin = blockIdx.x * VX_THREADS + threadIdx.x;
    bool pk = false;
    if (lin < n_bins) {
        const int a = lin / p.n_y, b = lin - a * p.n_y;
        const uint32_t c = p.vacc[lin];
        pk = c >= p.V_min;
        if (pk)
            for (int da = -1; da <= 1; ++da)
                for (int db = -1; db <= 1; ++db) {
                    const int aa = a + da, bb = b + db;
                    if ((da == 0 && db == 0) || aa < 0 || aa >= p.n_x || bb < 0 || bb >= p.n_y)
                        continue;
                    const int ln = aa * p.n_y + bb;
                    const uint32_t cn = p.vacc[ln];
                    if (cn > c || (cn == c && ln < lin))
                        pk = false;
                }
        p.flag[lin] = pk ? 1 : 0;
    }
    const unsigned bal = __ballot_sync(0xffffffffu, pk);
    if ((threadIdx.x & 31) == 0 && bal)
        atomicAdd(&s_cnt, (uint32_t)__popc(bal));
    __syncthreads();
    if (threadIdx.x == 0)
        p.block_cnt[blockIdx.x] = s_cnt;
}

__device__ __forceinline__ unsigned long long block_sum_u64(unsigned long long v, unsigned long long *s_red)
{
    for (int o = 16; o > 0; o >>= 1)
        v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0)
        s_red[threadIdx.x >> 5] = v;
    __syncthreads();
    unsigned long long t = 0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w)
        t += s_red[w];
    __syncthreads();
    return t;
}

__global__ void __launch_bounds__(VX_THREADS) k_vertex_compact(const VertexParams p)
{
    __shared__ unsigned long long s_red[VX_THREADS / 32];
    __shared__ uint32_t s_wcnt[VX_THREADS / 32];
    // the vertices of the blocks before this one
    unsigned long long part = 0;
    for (uint32_t b = threadIdx.x; b < blockIdx.x; b += VX_THREADS)
        part += p.block_cnt[b];
    const uint32_t base = (uint32_t)block_sum_u64(part, s_red);
    const int n_bins = p.n_x * p.n_y;
    const int lin = blockIdx.x * VX_THREADS + threadIdx.x;
    const bool pk = lin < n_bins && p.flag[lin];
    const unsigned bal = __ballot_sync(0xffffffffu, pk);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0)
        s_wcnt[warp] = (uint32_t)__popc(bal);
    __syncthreads();
    uint32_t before = 0;
    for (int w = 0; w < warp; ++w)
        before += s_wcnt[w];
    if (pk) {
        const uint32_t pos = base + before + (uint32_t)__popc(bal & ((1u << lane) - 1u));
        if (pos < p.cap_vertices) {
            p.out_bin[pos] = (uint32_t)lin;
            p.out_count[pos] = p.vacc[lin];
        }
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) {
        uint32_t tot = base;
        for (int w = 0; w < VX_THREADS / 32; ++w)
            tot += s_wcnt[w];
        p.counts->n_vertices = tot;
        if (tot > p.cap_vertices)
            p.counts->flags |= 1u;
    }
}

// V4: one CTA per reported vertex.  The peaks are in ascending lin = ((i * n_d0 + j) * n_kappa + k), so the
// peaks of a (phi0, d0) cell are neighbours in the list and the cells of one phi0 row i follow each other.
// For the vertex bin (a, b) and a row i only the cells whose d0 centre lies within the bin's image
// d = -xv sin + yv cos can vote into it: thread = phi0 row finds that d0 interval (one d0 bin of margin on
// each side), brackets its peaks in the list by two binary searches and evaluates the EXACT V2 vote for
// them only; a block scan over the rows keeps the members in ascending peak position.
__device__ __forceinline__ uint32_t vx_lower_bound(const uint32_t *__restrict__ bin, uint32_t n, uint32_t key)
{
    uint32_t lo = 0, hi = n; // first position with bin[pos] >= key
    while (lo < hi) {
        const uint32_t mid = (lo + hi) >> 1;
        if (bin[mid] < key)
            lo = mid + 1;
        else
            hi = mid;
    }
    return lo;
}

template <bool FILL>
__global__ void __launch_bounds__(VX_THREADS) k_vertex_members(const VertexParams p)
{
    __shared__ unsigned long long s_red[VX_THREADS / 32];
    __shared__ uint32_t s_wcnt[VX_THREADS / 32];
    const uint32_t n_v = min(p.counts->n_vertices, p.cap_vertices);
    const uint32_t m = blockIdx.x;
    if (m >= n_v)
        return;
    unsigned long long w = 0;
    if (FILL) {
        unsigned long long part = 0;
        for (uint32_t q = threadIdx.x; q < m; q += VX_THREADS)
            part += p.member_len[q];
        w = block_sum_u64(part, s_red);
        if (threadIdx.x == 0) {
            p.member_offset[m] = w;
            if (m == n_v - 1) {
                const unsigned long long tot = w + p.member_len[m];
                p.member_offset[n_v] = tot;
                p.counts->n_member_entries = tot;
                if (tot > p.cap_members)
                    p.counts->flags |= 2u;
            }
        }
    }
    const uint32_t vlin = p.out_bin[m];
    const int va = (int)(vlin / (uint32_t)p.n_y), vb = (int)(vlin - (uint32_t)va * (uint32_t)p.n_y);
    const float xca = vx_centre(p.x_min, p.x_max, p.n_x, va), ycb = vx_centre(p.y_min, p.y_max, p.n_y, vb);
    // the bin's edges and the d0 grid, in binary64
    const double wx = (p.x_max - p.x_min) / (double)p.n_x, wy = (p.y_max - p.y_min) / (double)p.n_y;
    const double xe0 = p.x_min + va * wx, xe1 = xe0 + wx, ye0 = p.y_min + vb * wy, ye1 = ye0 + wy;
    const double dd0 = p.n_d0 > 1 ? (p.d0_max - p.d0_min) / (double)p.n_d0 : 1.0;
    const uint32_t n_rep = min(p.peak_counts->n_peaks, p.cap_peaks);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t total = 0;
    for (int i0 = 0; i0 < p.n_phi; i0 += VX_THREADS) {
        const int i = i0 + (int)threadIdx.x;
        uint32_t p0 = 0, p1 = 0, cnt = 0;
        float sn = 0.f, cs = 0.f;
        bool steep = false;
        if (i < p.n_phi) {
            sn = p.sn[i];
            cs = p.cs[i];
            steep = !(fabsf(cs) >= fabsf(sn));
            // image of the bin along the voted axis: d between these two values (either order)
            double da, db;
            if (!steep) { // yv = (d + xc sn) / cs in [ye0, ye1)  ->  d = yv cs - xc sn
                da = ye0 * (double)cs - (double)xca * (double)sn;
                db = ye1 * (double)cs - (double)xca * (double)sn;
            } else {      // xv = (yc cs - d) / sn in [xe0, xe1)  ->  d = yc cs - xv sn
                da = (double)ycb * (double)cs - xe0 * (double)sn;
                db = (double)ycb * (double)cs - xe1 * (double)sn;
            }
            const double dlo = fmin(da, db) - dd0, dhi = fmax(da, db) + dd0;
            int j0 = 0, j1 = p.n_d0 - 1;
            if (p.n_d0 > 1 && dlo == dlo && dhi == dhi) { // d0 centres d0_min + (j + 0.5) dd0 inside [dlo, dhi]
                const double t0 = floor((dlo - p.d0_min) / dd0 - 0.5), t1 = ceil((dhi - p.d0_min) / dd0 - 0.5);
                j0 = t0 < 0.0 ? 0 : (t0 > (double)(p.n_d0 - 1) ? p.n_d0 : (int)t0);
                j1 = t1 < 0.0 ? -1 : (t1 > (double)(p.n_d0 - 1) ? p.n_d0 - 1 : (int)t1);
            }
            if (j0 <= j1) {
                const uint32_t r0 = (uint32_t)i * (uint32_t)p.n_d0 + (uint32_t)j0, r1 = (uint32_t)i * (uint32_t)p.n_d0 + (uint32_t)j1;
                p0 = vx_lower_bound(p.peak_bin, n_rep, r0 * (uint32_t)p.n_kappa);
                // (r1 + 1) * n_kappa may be 2^32 for the very last row: then every remaining peak is in range
                const unsigned long long end = ((unsigned long long)r1 + 1ull) * (unsigned long long)p.n_kappa;
                p1 = end > 0xffffffffull ? n_rep : vx_lower_bound(p.peak_bin, n_rep, (uint32_t)end);
            }
            for (uint32_t pk = p0; pk < p1; ++pk) {
                const uint32_t row = p.peak_bin[pk] / (uint32_t)p.n_kappa;
                const uint32_t j = row % (uint32_t)p.n_d0;
                const int o = vx_vote_one(p, sn, cs, p.d0c[j], steep, steep ? ycb : xca);
                cnt += (o >= 0 && o == (steep ? va : vb)) ? 1u : 0u;
            }
        }
        // ordered placement: exclusive scan of the rows' counts over the block
        uint32_t incl = cnt;
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o)
                incl += t;
        }
        if (lane == 31)
            s_wcnt[warp] = incl;
        __syncthreads();
        uint32_t before = 0, all = 0;
        for (int q = 0; q < VX_THREADS / 32; ++q) {
            const uint32_t c = s_wcnt[q];
            before += q < warp ? c : 0u;
            all += c;
        }
        if (FILL && cnt) {
            unsigned long long pos = w + total + before + incl - cnt;
            for (uint32_t pk = p0; pk < p1; ++pk) {
                const uint32_t row = p.peak_bin[pk] / (uint32_t)p.n_kappa;
                const uint32_t j = row % (uint32_t)p.n_d0;
                const int o = vx_vote_one(p, sn, cs, p.d0c[j], steep, steep ? ycb : xca);
                if (o >= 0 && o == (steep ? va : vb)) {
                    if (pos < p.cap_members)
                        p.member_index[pos] = pk;
                    ++pos;
                }
            }
        }
        total += all;
        __syncthreads();
    }
    if (!FILL && threadIdx.x == 0)
        p.member_len[m] = total;
}

// the reported vertices are unknown on the host: with no vertex at all the fill kernel's first
// CTA still has to write member_offset[0] = 0
__global__ void k_vertex_finish(const VertexParams p)
{
    if (min(p.counts->n_vertices, p.cap_vertices) == 0u)
        p.member_offset[0] = 0ull;
}

// ------------------------------------------------------------------ host side
static int vcfg_valid(const hough_vertex_config *v)
{
    if (!v)
        return 0;
    if (!(v->x_max > v->x_min) || !(v->y_max > v->y_min) || !isfinite(v->x_min) || !isfinite(v->x_max) ||
        !isfinite(v->y_min) || !isfinite(v->y_max))
        return 0;
    if (v->n_x < 1 || v->n_y < 1 || v->n_x > 2048 || v->n_y > 2048)
        return 0;
    if (v->V_min < 1 || v->cap_vertices < 1 || v->cap_vertices > 65536u || v->cap_members < 1)
        return 0;
    return 1;
}

static size_t vx_align(size_t b) { return (b + 255) & ~(size_t)255; }

size_t hough_vertex_workspace_bytes(const hough_vertex_config *v)
{
    if (!vcfg_valid(v))
        return 0;
    const size_t n_bins = (size_t)v->n_x * v->n_y, n_blocks = (n_bins + VX_THREADS - 1) / VX_THREADS;
    return vx_align(n_bins * 4) + vx_align(n_bins) + vx_align(n_blocks * 4) + vx_align((size_t)v->cap_vertices * 4);
}

int hough_vertices(hough_handle *h, const hough_vertex_config *v, void *workspace, size_t workspace_bytes,
                   const hough_peaks_out *peaks, const hough_vertex_out *out, void *cuda_stream)
{
    if (!h || !vcfg_valid(v) || !workspace || !peaks || !peaks->bin || !peaks->counts || !out || !out->bin ||
        !out->count || !out->member_offset || !out->member_index || !out->counts)
        return HOUGH_EINVAL;
    if (((uintptr_t)workspace & 255) != 0)
        return HOUGH_EINVAL;
    if (workspace_bytes < hough_vertex_workspace_bytes(v))
        return HOUGH_ENOMEM;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (cudaSetDevice(h->device) != cudaSuccess)
        return HOUGH_ECUDA;
    const size_t n_bins = (size_t)v->n_x * v->n_y, n_blocks = (n_bins + VX_THREADS - 1) / VX_THREADS;
    unsigned char *w = (unsigned char *)workspace;
    VertexParams p;
    p.n_phi = h->cfg.n_phi;
    p.n_d0 = h->cfg.n_d0;
    p.n_kappa = h->cfg.n_kappa;
    p.d0_min = h->cfg.d0_min;
    p.d0_max = h->cfg.d0_max;
    p.sn = h->t_sn;
    p.cs = h->t_cs;
    p.d0c = h->t_d0c;
    p.peak_bin = peaks->bin;
    p.peak_counts = peaks->counts;
    p.cap_peaks = h->cfg.cap_peaks;
    p.x_min = v->x_min;
    p.x_max = v->x_max;
    p.y_min = v->y_min;
    p.y_max = v->y_max;
    p.n_x = v->n_x;
    p.n_y = v->n_y;
    p.V_min = (uint32_t)v->V_min;
    p.xlo = (float)v->x_min;
    p.xhi = (float)v->x_max;
    {
        volatile float ix = (float)((double)v->n_x / (v->x_max - v->x_min));
        volatile float iy = (float)((double)v->n_y / (v->y_max - v->y_min));
        p.inv_dx = ix;
        p.inv_dy = iy;
    }
    p.ylo = (float)v->y_min;
    p.yhi = (float)v->y_max;
    p.vacc = (uint32_t *)w;
    w += vx_align(n_bins * 4);
    p.flag = w;
    w += vx_align(n_bins);
    p.block_cnt = (uint32_t *)w;
    w += vx_align(n_blocks * 4);
    p.member_len = (uint32_t *)w;
    p.cap_vertices = v->cap_vertices;
    p.cap_members = v->cap_members;
    p.out_bin = out->bin;
    p.out_count = out->count;
    p.member_offset = reinterpret_cast<unsigned long long *>(out->member_offset);
    p.member_index = out->member_index;
    p.counts = out->counts;
#define VCK(call)                      \
    do {                               \
        if ((call) != cudaSuccess) {   \
            cudaGetLastError();        \
            return HOUGH_ECUDA;        \
        }                              \
    } while (0)
    VCK(cudaMemsetAsync(p.vacc, 0, n_bins * 4, st));
    VCK(cudaMemsetAsync(out->counts, 0, sizeof(hough_vertex_counts), st));
    const int vote_blocks = h->n_sms * 4;
    const size_t tab = (size_t)(v->n_x + v->n_y) * 4;
    if (n_bins <= VX_SMEM_BINS)
        k_vertex_vote<true><<<vote_blocks, VX_THREADS, tab + n_bins * 4, st>>>(p);
    else
        k_vertex_vote<false><<<vote_blocks, VX_THREADS, tab, st>>>(p);
    VCK(cudaGetLastError());
    k_vertex_flags<<<(unsigned)n_blocks, VX_THREADS, 0, st>>>(p);
    k_vertex_compact<<<(unsigned)n_blocks, VX_THREADS, 0, st>>>(p);
    k_vertex_members<false><<<v->cap_vertices, VX_THREADS, 0, st>>>(p);
    k_vertex_members<true><<<v->cap_vertices, VX_THREADS, 0, st>>>(p);
    k_vertex_finish<<<1, 1, 0, st>>>(p);
    VCK(cudaGetLastError());
#undef VCK
    h->launches += 6;
    return HOUGH_OK;
}
