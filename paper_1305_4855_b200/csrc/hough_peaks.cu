// hough_peaks.cu -- accumulator sweep kernels (SURVEY.md section 8(a) rows a2, a5, a6 and
// the CSR bookkeeping of a7):
//   k_clear        zero the global accumulator (pure HBM write)
//   k_peak_sweep   popcount + 3x3x3 local-maximum test with ties to the lower linear index,
//                  one pass over the accumulator (4 B/bin read once), 1 flag bit per bin out
//   k_scan         single-pass chained prefix sum (decoupled look-back)
//   k_compact      flag bits -> (lin, mask) records in ascending lin
//   k_finish       counters -> the caller's hough_counts
// The peak rule is BASELINE.json north_star's ("popcount reaches at least L_min and ...
// local maxima in the 3x3x3 neighbourhood (ties go to the lower linear index)"), restated
// in DESIGN.md section 2 A6: with key(b) = (popcount, -lin) a bin is a peak iff its key
// beats the key of every existing neighbour, i.e. popcount > every neighbour of lower lin
// and >= every neighbour of higher lin.
#include <type_traits>

#include "hough_device.cuh"

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
// Register-resident streaming stencil.
//   * popcounts travel as u16x2 pairs (two bins per register) so that the 3-way maxima are
//     single VIMNMX3.U16x2 instructions;
//   * a lane owns 8 consecutive kappa bins of a row (two 16-byte loads, four pair
//     registers), a warp 256 bins, a thread PEAK_RJ consecutive d0 rows; the CTA owns
//     PEAK_RJ*JW rows (first and last are halo rows) x 256 bins and walks Li phi0 planes
//     (+1 halo plane on each side);
//   * kappa neighbours come from the neighbouring lanes (two shuffles per row), d0
//     neighbours of the thread's outer rows through a double-buffered shared-memory
//     exchange (one barrier per plane), phi0 neighbours from the thread's own state;
//   * the raw masks of plane p+1 are loaded into registers before plane p is processed.
// With  m3 = max over kappa+-1 of pc,  bx = max over d0+-1 of m3  (the 3x3 box of a plane):
//   lower-lin neighbours of (i,j,k): box(i-1,j,k), m3(i,j-1,k), pc(i,j,k-1)    -> need pc >  them
//   higher-lin neighbours          : box(i+1,j,k), m3(i,j+1,k), pc(i,j,k+1)    -> need pc >= them
// (with phi wrap, plane i-1 of i = 0 is plane n_phi-1, which has HIGHER lin, and plane i+1
// of i = n_phi-1 is plane 0, which has LOWER lin).  "a > b" on pairs of small numbers is
// bit 15 / 31 of (a | 0x80008000) - b - 0x00010001, "a >= b" the same without the last term.

struct PeakParams {
    const uint32_t *acc;
    unsigned char *flags; // 1 bit per bin, byte q of a row = bins 8q .. 8q+7
    int n_phi, n_d0, nk, L_min, wrap;
    int JW, Li;
};

__device__ __forceinline__ uint32_t popc_pair(uint32_t a, uint32_t b)
{
    return (uint32_t)__popc(a) | ((uint32_t)__popc(b) << 16);
}

template <int PEAK_RJ>
struct PeakRaw { // raw masks of one plane for the thread's rows
    uint4 a[PEAK_RJ], b[PEAK_RJ];
    uint32_t e[PEAK_RJ]; // the one bin beyond the warp's 256-bin segment (lanes 0 and 31)
};

template <int PEAK_RJ, int MAXJW>
__global__ void __launch_bounds__(32 * MAXJW, 2) k_peak_sweep(const PeakParams p)
{
    extern __shared__ uint4 ex[]; // [2][rows][32] : m3 of every row of the current plane
    pdl_wait();
    pdl_trigger();
    // one warp per pair of d0 rows, 256 kappa bins wide
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int KW = 1;
    const int kw = 0, jw = warp;
    const int rows = PEAK_RJ * p.JW, Tj = rows - 2;
    const int k0 = (blockIdx.x * KW + kw) * 256 + lane * 8;
    const bool kact = k0 < p.nk;
    const int jfirst = blockIdx.y * Tj - 1;
    const int ia = blockIdx.z * p.Li, ib = min(ia + p.Li, p.n_phi);
    const uint32_t HB = 0x80008000u, ONE = 0x00010001u;
    const uint32_t lmin2 = (uint32_t)p.L_min * ONE;
    const uint32_t plane_stride = (uint32_t)p.n_d0 * (uint32_t)p.nk;

    // Rows or lanes outside the grid load a clamped (valid) address and are masked to zero.
    uint32_t roff[PEAK_RJ], rmask[PEAK_RJ], fbyte[PEAK_RJ];
    bool rout[PEAK_RJ];
#pragma unroll
    for (int t = 0; t < PEAK_RJ; ++t) {
        const int r = jw * PEAK_RJ + t, j = jfirst + r;
        const bool there = kact && j >= 0 && j < p.n_d0;
        const int jc = min(max(j, 0), p.n_d0 - 1);
        roff[t] = (uint32_t)jc * (uint32_t)p.nk + (uint32_t)(kact ? k0 : 0);
        rmask[t] = there ? 0xffffffffu : 0u;
        rout[t] = there && r >= 1 && r <= rows - 2;
        fbyte[t] = roff[t] >> 3;
    }
    const bool e_left = (lane == 0) && (k0 > 0);
    const bool e_right = (lane == 31) && (k0 + 8 < p.nk);
    const bool e_any = e_left || e_right;
    const int e_off = e_left ? -1 : 8;

    auto load_plane = [&](int pl, PeakRaw<PEAK_RJ> &R) {
        const int src = pl < 0 ? p.n_phi - 1 : (pl >= p.n_phi ? 0 : pl);
        const uint32_t *pb = p.acc + (size_t)src * plane_stride;
#pragma unroll
        for (int t = 0; t < PEAK_RJ; ++t) {
            const uint32_t *rp = pb + roff[t];
            R.a[t] = __ldg(reinterpret_cast<const uint4 *>(rp));
            R.b[t] = __ldg(reinterpret_cast<const uint4 *>(rp) + 1);
            R.e[t] = 0u;
            if (e_any)
                R.e[t] = __ldg(rp + e_off);
        }
    };

    // state of the open plane (the previous one): o = pc | HB, thr = what pc must reach
    // as far as known, bxp = box maxima of the previous plane
    uint32_t s_o[PEAK_RJ][4], s_thr[PEAK_RJ][4], s_bx[PEAK_RJ][4];
#pragma unroll
    for (int t = 0; t < PEAK_RJ; ++t)
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            s_o[t][q] = 0u;
            s_thr[t][q] = 0x7fff7fffu;
            s_bx[t][q] = 0u;
        }

    // shared-memory exchange through 32-bit addresses: this thread's rows, and the rows of
    // the warps below / above (r = 0 and r = rows-1 are halo rows and never output)
    const uint32_t ex0 = (uint32_t)__cvta_generic_to_shared(ex);
    const uint32_t ex_half = (uint32_t)rows * (uint32_t)KW * 512u;
    uint32_t ex_mine[PEAK_RJ];
#pragma unroll
    for (int t = 0; t < PEAK_RJ; ++t)
        ex_mine[t] = ex0 + (uint32_t)(((jw * PEAK_RJ + t) * KW + kw) * 32 + lane) * 16u;
    const uint32_t ex_dn = ex0 + (uint32_t)((max(jw * PEAK_RJ - 1, 0) * KW + kw) * 32 + lane) * 16u;
    const uint32_t ex_up = ex0 + (uint32_t)((min(jw * PEAK_RJ + PEAK_RJ, rows - 1) * KW + kw) * 32 + lane) * 16u;
    const int bar_dn = 1 + (jw - 1) * KW + kw, bar_up = 1 + jw * KW + kw;
    const bool has_dn = jw > 0, has_up = jw < p.JW - 1;
    // flag byte of the plane being closed, per row (advanced by one plane per step)
    long long fo[PEAK_RJ];
#pragma unroll
    for (int t = 0; t < PEAK_RJ; ++t)
        fo[t] = (long long)fbyte[t] + ((long long)ia - 3) * (long long)(plane_stride >> 3);
    uint32_t exo = 0;

    // One plane.  STEADY: an interior plane (0 < pl < n_phi) that is ours and whose predecessor
    // is ours too: masks and the strictness of the comparisons are compile-time constants.
    auto step = [&](int pl, const PeakRaw<PEAK_RJ> &C, PeakRaw<PEAK_RJ> &N, auto steady_tag) {
        constexpr bool STEADY = decltype(steady_tag)::value;
        if (!STEADY && pl > ib)
            return;
        if (STEADY || pl < ib)
            load_plane(pl + 1, N);
        const uint32_t pmask = STEADY ? 0xffffffffu : (((pl < 0 || pl >= p.n_phi) && !p.wrap) ? 0u : 0xffffffffu);
        const bool out_prev = STEADY ? true : (pl - 1 >= ia); // plane pl-1 is one of ours: close it
        // strictness of the comparison with the neighbouring planes (phi wrap changes lin order)
        const uint32_t d_next = STEADY ? 0u : (((pl - 1 == p.n_phi - 1) && p.wrap) ? ONE : 0u);
        const uint32_t d_prev = STEADY ? ONE : (((pl == 0) && p.wrap) ? 0u : ONE);

        // ---- phase A: pair popcounts, kappa shifts, m3; publish m3 of every row
        uint32_t c[PEAK_RJ][4], s[PEAK_RJ][5], m3[PEAK_RJ][4];
#pragma unroll
        for (int t = 0; t < PEAK_RJ; ++t) {
            const uint32_t m = rmask[t] & pmask;
            c[t][0] = popc_pair(C.a[t].x, C.a[t].y) & m;
            c[t][1] = popc_pair(C.a[t].z, C.a[t].w) & m;
            c[t][2] = popc_pair(C.b[t].x, C.b[t].y) & m;
            c[t][3] = popc_pair(C.b[t].z, C.b[t].w) & m;
            const uint32_t pe = (uint32_t)__popc(C.e[t]) & m;
            uint32_t pv = __shfl_up_sync(0xffffffffu, c[t][3], 1);
            uint32_t nx = __shfl_down_sync(0xffffffffu, c[t][0], 1);
            if (lane == 0)
                pv = pe << 16;
            if (lane == 31)
                nx = pe;
            s[t][0] = __funnelshift_r(pv, c[t][0], 16);      // bins (k0-1, k0)
            s[t][1] = __funnelshift_r(c[t][0], c[t][1], 16); // bins (k0+1, k0+2)
            s[t][2] = __funnelshift_r(c[t][1], c[t][2], 16);
            s[t][3] = __funnelshift_r(c[t][2], c[t][3], 16);
            s[t][4] = __funnelshift_r(c[t][3], nx, 16);      // bins (k0+7, k0+8)
#pragma unroll
            for (int q = 0; q < 4; ++q)
                m3[t][q] = __vimax3_u16x2(c[t][q], s[t][q], s[t][q + 1]);
            asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(ex_mine[t] + exo), "r"(m3[t][0]), "r"(m3[t][1]),
                         "r"(m3[t][2]), "r"(m3[t][3])
                         : "memory");
        }
        // A warp only needs the rows of the warps below and above it: pair barriers (named
        // barrier 1 + jw*KW + kw joins warps (jw, kw) and (jw+1, kw)) instead of a CTA-wide
        // one.  Lower id first on both sides, so the chain cannot deadlock; the exchange
        // buffer is double buffered, and passing the pair barriers of plane p+1 implies that
        // the neighbours have finished reading plane p.
        if (has_dn)
            asm volatile("bar.sync %0, 64;" ::"r"(bar_dn) : "memory");
        if (has_up)
            asm volatile("bar.sync %0, 64;" ::"r"(bar_up) : "memory");

        // ---- phase B: box maxima; close plane pl-1; open plane pl (always computed: a plane
        // that is not ours is simply never stored)
        uint4 vdn, vup;
        asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(vdn.x), "=r"(vdn.y), "=r"(vdn.z), "=r"(vdn.w) : "r"(ex_dn + exo));
        asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(vup.x), "=r"(vup.y), "=r"(vup.z), "=r"(vup.w) : "r"(ex_up + exo));
#pragma unroll
        for (int t = 0; t < PEAK_RJ; ++t) {
            uint32_t dn[4], up[4];
            if (t > 0) {
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    dn[q] = m3[t - 1][q];
            } else {
                dn[0] = vdn.x, dn[1] = vdn.y, dn[2] = vdn.z, dn[3] = vdn.w;
            }
            if (t < PEAK_RJ - 1) {
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    up[q] = m3[t + 1][q];
            } else {
                up[0] = vup.x, up[1] = vup.y, up[2] = vup.z, up[3] = vup.w;
            }
            uint32_t bits = 0u;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const uint32_t bx = __vimax3_u16x2(dn[q], m3[t][q], up[q]);
                const uint32_t thr = __vmaxu2(s_thr[t][q], bx + d_next);
                const uint32_t g = (s_o[t][q] - thr) >> (15 - 2 * q); // bin 2q -> bit 2q, 2q+1 -> bit 16+2q
                bits |= g & (ONE << (2 * q));
                const uint32_t lo = __vmaxu2(dn[q], s[t][q]);                  // lower lin: pc must exceed
                const uint32_t hi = __vimax3_u16x2(up[q], s[t][q + 1], lmin2); // higher lin: pc must reach
                s_thr[t][q] = __vimax3_u16x2(lo + ONE, hi, s_bx[t][q] + d_prev);
                s_o[t][q] = c[t][q] | HB;
                s_bx[t][q] = bx;
            }
            fo[t] += (long long)(plane_stride >> 3);
            if (out_prev && rout[t])
                p.flags[fo[t]] = (unsigned char)((bits | (bits >> 15)) & 0xffu);
        }
        exo ^= ex_half;
    };

    PeakRaw<PEAK_RJ> A, B;
    load_plane(ia - 1, A);
    const int st_lo = max(ia + 1, 1), st_hi = min(ib - 1, p.n_phi - 1); // steady planes: [st_lo, st_hi]
    for (int pl = ia - 1; pl <= ib; pl += 2) {
        if (pl >= st_lo && pl <= st_hi)
            step(pl, A, B, std::true_type());
        else
            step(pl, A, B, std::false_type());
        if (pl + 1 >= st_lo && pl + 1 <= st_hi)
            step(pl + 1, B, A, std::true_type());
        else
            step(pl + 1, B, A, std::false_type());
    }
}

cudaError_t launch_peak_sweep(hough_handle *h, cudaStream_t st)
{
    PeakParams p;
    p.acc = h->acc;
    p.flags = reinterpret_cast<unsigned char *>(h->flags);
    p.n_phi = h->g.n_phi;
    p.n_d0 = h->g.n_d0;
    p.nk = h->g.n_kappa;
    p.L_min = h->g.L_min;
    p.wrap = h->g.phi_wrap;
    p.JW = h->pk_JW;
    p.Li = h->pk_Li;
    const int Tj = 2 * p.JW - 2;
    dim3 grid((p.nk + 255) / 256, (p.n_d0 + Tj - 1) / Tj, (p.n_phi + p.Li - 1) / p.Li);
    launch_pdl(k_peak_sweep<2, 8>, grid, dim3(32 * p.JW), h->pk_smem, st, p);
    h->launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ cell-wise peak test
// The same rule, one warp per (cell, 256-bin segment), lane = 8 bins, straight from the global
// accumulator (9 cell rows per cell).  With HOUGH_OPT_FUSED_PEAKS it visits only the cells on the edge
// of a vote tile -- the others were decided by k_sweep's epilogue from shared memory -- and with
// HOUGH_OPT_CELL_PEAKS every cell (cross-check of k_peak_sweep, which reads every row once instead).
struct CellPeakParams {
    const uint32_t *acc;
    unsigned char *flags;
    int n_phi, n_d0, nk, L_min, wrap;
    int edge_only;
    int P, D, n_big, P_small; // vote tile geometry (SweepGeom)
};

__device__ __forceinline__ Strip strip_from_masks(const uint32_t *__restrict__ row, int k0, int nk)
{
    const uint4 a = *reinterpret_cast<const uint4 *>(row + k0), b = *reinterpret_cast<const uint4 *>(row + k0 + 4);
    Strip s;
    s.x[0] = popc_pair(a.x, a.y);
    s.x[1] = popc_pair(a.z, a.w);
    s.x[2] = popc_pair(b.x, b.y);
    s.x[3] = popc_pair(b.z, b.w);
    s.m = k0 > 0 ? ((uint32_t)__popc(row[k0 - 1]) << 16) : 0u;
    s.p = k0 + 8 < nk ? (uint32_t)__popc(row[k0 + 8]) : 0u;
    return s;
}

__global__ void __launch_bounds__(256) k_peak_cells(const CellPeakParams p)
{
    const int lane = threadIdx.x & 31;
    const int nseg = (p.nk + 255) >> 8;
    const uint32_t n_items = (uint32_t)p.n_phi * (uint32_t)p.n_d0 * (uint32_t)nseg;
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    const uint32_t lmin2 = (uint32_t)p.L_min * 0x00010001u;
    for (uint32_t item = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; item < n_items; item += warps) {
        const int cell = (int)(item / (uint32_t)nseg), seg = (int)(item - (uint32_t)cell * (uint32_t)nseg);
        const int i = cell / p.n_d0, j = cell - i * p.n_d0;
        if (p.edge_only) { // position of the cell in its vote tile (two slab heights)
            const int big = p.n_big * p.P;
            const int Pt = i < big ? p.P : p.P_small;
            const int i0 = i < big ? (i / p.P) * p.P : big + ((i - big) / p.P_small) * p.P_small;
            const int j0 = (j / p.D) * p.D;
            const int ni = min(Pt, p.n_phi - i0), nj = min(p.D, p.n_d0 - j0);
            const int il = i - i0, jl = j - j0;
            if (il > 0 && il < ni - 1 && jl > 0 && jl < nj - 1)
                continue;
        }
        const int k0 = seg * 256 + lane * 8;
        if (k0 >= p.nk)
            continue;
        const Strip C = strip_from_masks(p.acc + (size_t)cell * p.nk, k0, p.nk);
        Strip L, H;
        L.m = L.p = H.m = H.p = 0u;
#pragma unroll
        for (int t = 0; t < 4; ++t)
            L.x[t] = H.x[t] = 0u;
        for (int di = -1; di <= 1; ++di) {
            int ii = i + di;
            if (ii < 0 || ii >= p.n_phi) {
                if (!p.wrap)
                    continue;
                ii = ii < 0 ? ii + p.n_phi : ii - p.n_phi;
            }
            for (int dj = -1; dj <= 1; ++dj) {
                const int jj = j + dj;
                if ((di == 0 && dj == 0) || jj < 0 || jj >= p.n_d0)
                    continue;
                const int ncell = ii * p.n_d0 + jj; // the neighbour's own linear order decides the tie rule
                const Strip S = strip_from_masks(p.acc + (size_t)ncell * p.nk, k0, p.nk);
                if (ncell < cell)
                    strip_max(L, S);
                else
                    strip_max(H, S);
            }
        }
        p.flags[(size_t)cell * (size_t)(p.nk >> 3) + (size_t)(k0 >> 3)] = (unsigned char)peak_flags8(C, L, H, lmin2);
    }
}

cudaError_t launch_peak_cells(hough_handle *h, int edge_cells_only, cudaStream_t st)
{
    CellPeakParams p;
    p.acc = h->acc;
    p.flags = reinterpret_cast<unsigned char *>(h->flags);
    p.n_phi = h->g.n_phi;
    p.n_d0 = h->g.n_d0;
    p.nk = h->g.n_kappa;
    p.L_min = h->g.L_min;
    p.wrap = h->g.phi_wrap;
    p.edge_only = edge_cells_only;
    p.P = h->vote_geom.P;
    p.D = h->vote_geom.D;
    p.n_big = h->vote_geom.n_big;
    p.P_small = h->vote_geom.P_small;
    k_peak_cells<<<h->n_sms * 8, 256, 0, st>>>(p);
    h->launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ chained scan
// One pass, decoupled look-back: block t (ticket order) publishes its aggregate, then
// adds the inclusive prefixes / aggregates of its predecessors.  status word =
// (flag << 62) | value, flag 1 = aggregate, 2 = inclusive prefix; written with one
// 64-bit store so that no fence is needed between flag and value.
//   SCAN_ROWS : item i = number of flag bits of accumulator row i  -> row_base (u32)
//   SCAN_LENS : item i = peak_len[i] = length of peak i's list (k_sub_prefix),
//               i < min(n_peaks, cap_peaks)  -> hit_offset (u64)
#define SCAN_ROWS 0
#define SCAN_LENS 1
#define SCAN_THREADS 256
#define SCAN_PER_THREAD (HOUGH_SCAN_ITEMS / SCAN_THREADS)

struct ScanParams {
    const uint32_t *flags;
    int fw_per_row;
    uint32_t n_rows;
    uint32_t *row_base;
    const uint32_t *list_len; // LENS: peak_len
    uint32_t cap_peaks;
    unsigned long long *hit_offset;
    uint32_t S;
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
    pdl_wait();
    pdl_trigger();
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
                p.counters->n_list_evals = 0ull;
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

    if (warp == 0) {
        // decoupled look-back by a whole warp: 32 predecessors per round (lane 0 = the nearest)
        volatile unsigned long long *status = p.status;
        const unsigned long long VAL = (1ull << 62) - 1ull;
        unsigned long long prefix = 0;
        if (t == 0) {
            if (lane == 0)
                status[0] = (2ull << 62) | agg;
        } else {
            if (lane == 0)
                status[t] = (1ull << 62) | agg;
            long long q = (long long)t - 1;
            while (true) {
                const long long idx = q - lane;
                const unsigned long long sw = idx >= 0 ? status[idx] : (2ull << 62); // before block 0: prefix 0
                const unsigned long long flag = sw >> 62;
                const unsigned m2 = __ballot_sync(0xffffffffu, flag == 2ull);
                const unsigned m0 = __ballot_sync(0xffffffffu, flag == 0ull);
                const int first2 = m2 ? __ffs((int)m2) - 1 : 32;
                const unsigned need = first2 >= 31 ? 0xffffffffu : ((1u << (first2 + 1)) - 1u);
                if (m0 & need)
                    continue; // a predecessor this side of the nearest inclusive prefix is not there yet
                unsigned long long val = lane <= first2 ? (sw & VAL) : 0ull;
                for (int o = 16; o > 0; o >>= 1)
                    val += __shfl_xor_sync(0xffffffffu, val, o);
                prefix += val;
                if (first2 < 32)
                    break;
                q -= 32;
            }
            if (lane == 0)
                status[t] = (2ull << 62) | (prefix + agg);
        }
        if (lane == 0)
            s_prefix = prefix;
    }
    __syncthreads();
    unsigned long long run = s_prefix + texcl;
#pragma unroll
    for (int q = 0; q < SCAN_PER_THREAD; ++q) {
        unsigned long long i = base + (unsigned long long)tid * SCAN_PER_THREAD + q;
        if (i < n) {
            if (KIND == SCAN_ROWS) {
                p.row_base[i] = (uint32_t)run;
            } else {
                p.hit_offset[i] = run;
            }
            run += v[q];
            if (i == (unsigned long long)n - 1) { // the last item closes the scan
                if (KIND == SCAN_ROWS) {
                    p.row_base[n] = (uint32_t)run;
                    p.counters->n_peaks = (unsigned int)run;
                    // hough_peaks may be repeated on one vote: the list stage that follows counts from zero
                    p.counters->n_list_evals = 0ull;
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
    p->list_len = h->peak_len;
    p->cap_peaks = h->cfg.cap_peaks;
    p->hit_offset = out ? reinterpret_cast<unsigned long long *>(out->hit_offset) : nullptr;
    p->S = (uint32_t)h->list_geom.S;
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
    launch_pdl(k_scan<SCAN_ROWS>, dim3(blocks), dim3(SCAN_THREADS), 0, st, p);
    h->launches += 1;
    return cudaGetLastError();
}

// A peak's list is the concatenation of its S sub-lists (hough_lists.cu): replace the S
// lengths sub_len[p*S .. p*S+S) by their exclusive prefix and put the sum in peak_len[p].
// 256 peaks per block, staged through shared memory so that global traffic is coalesced.
__global__ void __launch_bounds__(256) k_sub_prefix(uint32_t *sub_len, uint32_t *peak_len,
                                                    const DevCounters *counters, uint32_t cap_peaks, uint32_t S)
{
    extern __shared__ uint32_t sp[]; // [256][S + 1]
    const uint32_t n = min(counters->n_peaks, cap_peaks);
    const uint32_t p0 = blockIdx.x * 256u;
    if (p0 >= n)
        return;
    const uint32_t np = min(256u, n - p0), words = np * S;
    uint32_t *g = sub_len + (size_t)p0 * S;
    for (uint32_t w = threadIdx.x; w < words; w += 256u)
        sp[(w / S) * (S + 1) + (w % S)] = g[w];
    __syncthreads();
    if (threadIdx.x < np) {
        uint32_t *row = sp + threadIdx.x * (S + 1), run = 0;
        for (uint32_t s = 0; s < S; ++s) {
            const uint32_t len = row[s];
            row[s] = run;
            run += len;
        }
        peak_len[p0 + threadIdx.x] = run;
    }
    __syncthreads();
    for (uint32_t w = threadIdx.x; w < words; w += 256u)
        g[w] = sp[(w / S) * (S + 1) + (w % S)];
}

cudaError_t launch_scan_lens(hough_handle *h, const hough_peaks_out *out, cudaStream_t st)
{
    if ((h->cfg.options & HOUGH_OPT_LIST_SWEEP) && h->mode == 0) { // the sweep's sub-lists -> list lengths (peak-driven lists write them directly)
        const uint32_t S = (uint32_t)h->list_geom.S;
        k_sub_prefix<<<(h->cfg.cap_peaks + 255) / 256, 256, 256 * (S + 1) * 4, st>>>(
            h->list_len, h->peak_len, h->counters, h->cfg.cap_peaks, S);
        h->launches += 1;
    }
    ScanParams p;
    scan_params(h, &p, out, 1);
    uint32_t blocks = (h->cfg.cap_peaks + HOUGH_SCAN_ITEMS - 1) / HOUGH_SCAN_ITEMS;
    launch_pdl(k_scan<SCAN_LENS>, dim3(blocks), dim3(SCAN_THREADS), 0, st, p);
    h->launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ compaction (a6)
// G lanes per accumulator row (G = the power of two that holds the row's flag words, at most 32), so a
// warp works on 32 / G rows at a time and their loads are in flight together: popcount prefix over the
// row's flag words inside the lane group, each lane expands the set bits of its word.  Records land in
// ascending lin because row_base is the exclusive scan of the rows in lin order.
template <int G>
__global__ void __launch_bounds__(256) k_compact(const uint32_t *__restrict__ flags,
                                                 const uint32_t *__restrict__ row_base,
                                                 const uint32_t *__restrict__ acc, uint32_t n_rows,
                                                 int nk, uint32_t cap_peaks, uint32_t *__restrict__ bin,
                                                 uint32_t *__restrict__ mask)
{
    constexpr int R = 32 / G; // rows per warp and round
    const int lane = threadIdx.x & 31, sl = lane % G, slot = lane / G;
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    const int fw_per_row = nk >> 5;
    pdl_wait();
    pdl_trigger();
    for (uint32_t row0 = ((blockIdx.x * blockDim.x + threadIdx.x) >> 5) * R; row0 < n_rows; row0 += warps * R) {
        const uint32_t row = row0 + (uint32_t)slot;
        uint32_t gb = 0, cnt = 0;
        if (row < n_rows) {
            gb = row_base[row];
            cnt = row_base[row + 1] - gb;
        }
        const bool live = cnt != 0u && gb < cap_peaks;
        const uint32_t *fw = flags + (size_t)row * fw_per_row;
        uint32_t rank0 = gb;
        for (int wb = 0; wb < fw_per_row; wb += G) { // one round unless a row has more than 32 flag words
            uint32_t f = (live && wb + sl < fw_per_row) ? fw[wb + sl] : 0u;
            uint32_t pc = __popc(f), incl = pc;
#pragma unroll
            for (int o = 1; o < G; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o, G);
                if (sl >= o)
                    incl += t;
            }
            uint32_t rank = rank0 + incl - pc;
            while (f) {
                const int b = __ffs(f) - 1;
                f &= f - 1;
                if (rank < cap_peaks) {
                    const uint32_t lin = row * (uint32_t)nk + (uint32_t)(((wb + sl) << 5) + b);
                    bin[rank] = lin;
                    mask[rank] = acc[lin];
                }
                ++rank;
            }
            rank0 += __shfl_sync(0xffffffffu, incl, G - 1, G);
        }
    }
}

cudaError_t launch_compact(hough_handle *h, const hough_peaks_out *out, cudaStream_t st)
{
    uint32_t n_rows = (uint32_t)h->g.n_phi * (uint32_t)h->g.n_d0;
    const int fwr = h->g.n_kappa >> 5, lanes = fwr <= 2 ? 2 : fwr <= 4 ? 4 : fwr <= 8 ? 8 : fwr <= 16 ? 16 : 32;
    uint32_t blocks = (n_rows + 8 * (32 / lanes) - 1) / (8 * (32 / lanes));
    uint32_t maxb = (uint32_t)h->n_sms * 16;
    if (blocks > maxb)
        blocks = maxb;
    const int fw = h->g.n_kappa >> 5;
    const uint32_t *fl = h->flags, *rb = h->row_base, *ac = h->acc;
#define COMPACT(G)                                                                                          \
    launch_pdl(k_compact<G>, dim3(blocks), dim3(256), 0, st, fl, rb, ac, n_rows, h->g.n_kappa, h->cfg.cap_peaks, \
               out->bin, out->mask)
    if (fw <= 2)
        COMPACT(2);
    else if (fw <= 4)
        COMPACT(4);
    else if (fw <= 8)
        COMPACT(8);
    else if (fw <= 16)
        COMPACT(16);
    else
        COMPACT(32);
#undef COMPACT
    h->launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ counters out
// Also clears what the next calls expect clean: the other counter block (the next hough_vote's), the scan
// tickets / work counter and the look-back words (the next hough_peaks').
__global__ void k_finish(const DevCounters *c, hough_counts *out, uint32_t cap_peaks,
                         unsigned long long cap_hits, int with_lists, int index16, uint32_t *next_counters,
                         uint32_t *reset, uint32_t reset_words, uint32_t *status, uint32_t status_words)
{
    pdl_wait();
    if (threadIdx.x < 16)
        next_counters[threadIdx.x] = 0u;
    for (uint32_t w = threadIdx.x; w < reset_words; w += blockDim.x)
        reset[w] = 0u;
    for (uint32_t w = threadIdx.x; w < status_words; w += blockDim.x)
        status[w] = 0u;
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        hough_counts r;
        r.n_votes = c->n_votes;
        r.n_hit_entries = with_lists ? c->n_hit_entries : 0ull;
        r.n_evals = c->n_evals;
        r.n_list_evals = with_lists ? c->n_list_evals : 0ull;
        r.n_peaks = c->n_peaks;
        r.n_bad_hits = c->n_bad_hits;
        r.flags = 0u;
        if (r.n_peaks > cap_peaks)
            r.flags |= HOUGH_TRUNCATED_PEAKS;
        if (r.n_hit_entries > cap_hits)
            r.flags |= HOUGH_TRUNCATED_HITS;
        if (index16)
            r.flags |= HOUGH_INDEX16;
        r.reserved = 0u;
        *out = r;
    }
}

cudaError_t launch_finish_counts(hough_handle *h, const hough_peaks_out *out, int with_lists,
                                 cudaStream_t st)
{
    // the 16-bit entries are written by k_copy_lists (not by the round-1 list sweep's placement kernel)
    const int sweep = (h->cfg.options & HOUGH_OPT_LIST_SWEEP) && h->mode == VOTE_CENTRE;
    const int index16 = with_lists && !sweep && out->hit_index16 && h->n_hits <= 65536u;
    unsigned char *base = (unsigned char *)h->cnt2[0];
    launch_pdl(k_finish, dim3(1), dim3(1024), 0, st, (const DevCounters *)h->counters, out->counts, h->cfg.cap_peaks,
               (unsigned long long)h->cfg.cap_hits, with_lists, index16, (uint32_t *)h->cnt2[h->cbuf ^ 1],
               (uint32_t *)(base + 64), 32u, (uint32_t *)h->scan_status, (uint32_t)(4 * h->scan_blocks_max));
    h->launches += 1;
    return cudaGetLastError();
}
