// hough_sweep.cu -- the tiled sweep of the hits over the (phi0, d0) cells:
//   MODE_VOTE  : a3 vote into a shared-memory tile with atomicOr, a4 coalesced write-out,
//                a8 vote count
//   MODE_LIST  : a7, one sweep that counts every reported peak's hit list (list_len) and
//                emits its (peak rank, hit index) pairs; k_scatter_pairs (hough_peaks.cu)
//                places them once the CSR offsets are known
// Both share the staging (TMA 1-D bulk copies of the SoA hit arrays into shared
// memory, double buffered), the conservative per-tile hit cull and the exact fp32
// evaluation of BASELINE.json north_star's closed form.
#include "hough_internal.cuh"

#define MODE_VOTE 0
#define MODE_LIST 1

#define PAIR_BUF 2048   // (peak, hit) pairs buffered per CTA between flushes
#define PAIR_FLUSH 1024 // flush at the end of a chunk once this many are waiting

#define EVAL_UNROLL 2

// ------------------------------------------------------------------ PTX helpers (TMA)
__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
// 1-D bulk copy global -> shared through the TMA unit; completion is signalled on `bar`.
__device__ __forceinline__ void tma_load_1d(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

// ------------------------------------------------------------------ the exact evaluation
// DESIGN.md section 2, A3: every operation is one binary32 round-to-nearest operation, in
// this order, never contracted.
__device__ __forceinline__ float eval_kappa(float x, float y, float r2, float sn, float cs, float d0c,
                                            float twod0, float d0sq)
{
    float a = __fmul_rn(x, sn);
    float b = __fmul_rn(y, cs);
    float s = __fsub_rn(b, a);
    float e = __fsub_rn(s, d0c);
    float num = __fadd_rn(e, e); // 2*e, exact
    float t = __fmul_rn(twod0, s);
    float u = __fsub_rn(r2, t);
    float den = __fadd_rn(u, d0sq);
    return __fdiv_rn(num, den);
}
// A4: the kappa bin of an in-range kappa (truncation, top clamp).
__device__ __forceinline__ int kappa_bin(float kappa, float klo, float inv_dk, int nk_minus_1)
{
    float qf = __fmul_rn(__fsub_rn(kappa, klo), inv_dk);
    return min(__float2int_rz(qf), nk_minus_1);
}
__device__ __forceinline__ void smem_red_or(uint32_t addr, uint32_t v)
{
    asm volatile("red.shared.or.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t smem_ld(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

// ------------------------------------------------------------------ conservative tile cull
// Can this hit cast a vote anywhere in the tile (phi0 centres between A and B, d0 centres
// in [dlo, dhi])?  Interval arithmetic on  2|e| <= K (e^2 + c^2),  e = s - d0,
// c^2 = r^2 - s^2, with slack that dominates every fp32 rounding of the exact recipe
// (DESIGN.md section 4.3).  May say yes too often, never no wrongly; any NaN says yes.
struct TileCull {
    float snA, csA, snB, csB;
    float dlo, dhi;
    int phi_all; // tile too wide in phi0: s ranges over [-r, r]
    int off;     // culling disabled (HOUGH_OPT_NO_CULL)
};

__device__ __forceinline__ bool hit_may_vote(float x, float y, float r2, const TileCull &tc, float K,
                                             float d0_absmax)
{
    if (tc.off)
        return true;
    const float EPS = 3.8146973e-06f; // 2^-18
    float ax = fabsf(x), ay = fabsf(y);
    if (!(ax <= 3.0e38f) || !(ay <= 3.0e38f))
        return false; // inf / NaN coordinates never vote (num/den is NaN)
    float r = sqrtf(r2);
    float smin, smax;
    if (tc.phi_all) {
        smin = -r;
        smax = r;
    } else {
        float sa = y * tc.csA - x * tc.snA, ca = x * tc.csA + y * tc.snA;
        float sb = y * tc.csB - x * tc.snB, cb = x * tc.csB + y * tc.snB;
        smin = fminf(sa, sb);
        smax = fmaxf(sa, sb);
        if (ca * cb <= 0.0f) { // s(phi0) has its extremum +-r inside the slab
            if (sa + sb >= 0.0f)
                smax = fmaxf(smax, r);
            else
                smin = fminf(smin, -r);
        }
    }
    float es = EPS * (ax + ay + d0_absmax) + 1e-30f;
    smin -= es;
    smax += es;
    float elo = smin - tc.dhi, ehi = smax - tc.dlo;
    float emin = (elo <= 0.0f && ehi >= 0.0f) ? 0.0f : fminf(fabsf(elo), fabsf(ehi));
    float emax = fmaxf(fabsf(elo), fabsf(ehi));
    float s2min = (smin <= 0.0f && smax >= 0.0f) ? 0.0f : fminf(smin * smin, smax * smax);
    float c2max = fmaxf(r2 - s2min, 0.0f);
    // g(e) = 2e - K e^2 is concave: its minimum over [emin, emax] is at an end point
    float g0 = 2.0f * emin - K * emin * emin;
    float g1 = 2.0f * emax - K * emax * emax;
    float gmin = fminf(g0, g1);
    float rhs = K * c2max * (1.0f + EPS) +
                K * EPS * (r2 + 2.0f * d0_absmax * (ax + ay) + d0_absmax * d0_absmax) + 1e-30f;
    return !(gmin > rhs);
}

// ------------------------------------------------------------------ kernel parameters
struct SweepParams {
    GridDev g;
    HitsDev hits;
    SweepGeom geom;
    int swz_mask; // XOR swizzle of the word index inside a cell row (vote tile)
    int no_cull;
    uint32_t *acc; // VOTE: global accumulator
    unsigned long long *n_votes;
    unsigned long long *n_evals;
    // hit lists (MODE_LIST)
    const uint32_t *flags;    // 1 bit per bin
    const uint32_t *row_base; // [n_rows + 1]
    const unsigned int *n_peaks_dev;
    uint32_t cap_peaks;
    uint32_t *list_len; // [cap_peaks], zeroed before the sweep
    uint2 *pairs;       // [pair_cap] (peak rank, hit index)
    unsigned long long *n_pairs;
    unsigned long long pair_cap;
};

template <int MODE, int PACK>
__global__ void __launch_bounds__(1024, 1) k_sweep(const SweepParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const GridDev &g = p.g;
    const SweepGeom &ge = p.geom;
    const int nk = g.n_kappa;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nwarps = ge.threads >> 5;
    const int wpr = nk >> 5; // flag words per cell row

    // ---- carve shared memory
    // VOTE: tile = masks [cells_pad][nk / PACK words];
    // LIST: tile = flag words [wpr][cells_pad] followed by their exclusive popcount prefix
    uint32_t *tile = reinterpret_cast<uint32_t *>(smem_raw);
    unsigned char *ptr = smem_raw + (size_t)ge.tile_words * 4;
    uint2 *pairbuf = nullptr;
    if (MODE == MODE_LIST) {
        pairbuf = reinterpret_cast<uint2 *>(ptr);
        ptr += (size_t)PAIR_BUF * 8;
    }
    float *stage = reinterpret_cast<float *>(ptr); // [2][4][chunk]
    ptr += (size_t)2 * 4 * ge.chunk * 4;
    float4 *surv = reinterpret_cast<float4 *>(ptr); // [chunk + EVAL_UNROLL]
    ptr += (size_t)(ge.chunk + EVAL_UNROLL) * 16;
    uint64_t *mbar = reinterpret_cast<uint64_t *>(ptr);
    ptr += 16;
    int *warp_cnt = reinterpret_cast<int *>(ptr); // [32]
    ptr += 32 * 4;
    unsigned int *s_npairs = reinterpret_cast<unsigned int *>(ptr); // [0] count, [1..2] flush base
    ptr += 16;

    // ---- which tile
    const int tp = blockIdx.x / ge.tiles_d0, td = blockIdx.x % ge.tiles_d0;
    const int i0 = tp * ge.P, j0 = td * ge.D;
    const int ni = min(ge.P, g.n_phi - i0), nj = min(ge.D, g.n_d0 - j0);

    // ---- this thread's cell and its constants (registers)
    const int grp = warp % ge.groups, set = warp / ge.groups;
    const int c = grp * 32 + lane;
    const int il = c / ge.D, jl = c - il * ge.D;
    const bool cell_ok = (il < ni) && (jl < nj);
    float c_sn = 0.f, c_cs = 0.f, c_d0 = 0.f, c_2d0 = 0.f, c_d0sq = __int_as_float(0x7fc00000);
    if (cell_ok) {
        c_sn = g.sn[i0 + il];
        c_cs = g.cs[i0 + il];
        c_d0 = g.d0c[j0 + jl];
        c_2d0 = g.twod0[j0 + jl];
        c_d0sq = g.d0sq[j0 + jl];
    }
    const float klo = g.klo, khi = g.khi, inv_dk = g.inv_dk;

    TileCull tc;
    tc.snA = g.sn[i0];
    tc.csA = g.cs[i0];
    tc.snB = g.sn[i0 + ni - 1];
    tc.csB = g.cs[i0 + ni - 1];
    tc.dlo = g.d0c[j0];
    tc.dhi = g.d0c[j0 + nj - 1];
    tc.phi_all = ge.no_phi_cull;
    tc.off = p.no_cull;

    const uint32_t n_chunks = p.hits.n_pad / ge.chunk;
    const uint32_t chunk_bytes = (uint32_t)ge.chunk * 4;

    if (tid == 0) {
        mbar_init(&mbar[0], 1);
        mbar_init(&mbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        s_npairs[0] = 0u;
    }
    __syncthreads();
    auto issue = [&](uint32_t ch) {
        float *dst = stage + (size_t)(ch & 1) * 4 * ge.chunk;
        uint64_t *bar = &mbar[ch & 1];
        mbar_expect_tx(bar, 4 * chunk_bytes);
        size_t off = (size_t)ch * ge.chunk;
        tma_load_1d(dst, p.hits.x + off, chunk_bytes, bar);
        tma_load_1d(dst + ge.chunk, p.hits.y + off, chunk_bytes, bar);
        tma_load_1d(dst + 2 * ge.chunk, p.hits.r2 + off, chunk_bytes, bar);
        tma_load_1d(dst + 3 * ge.chunk, p.hits.bit + off, chunk_bytes, bar);
    };
    if (tid == 0 && n_chunks > 0)
        issue(0);

    uint32_t c_gbase = 0u; // LIST: global rank of the first peak of this thread's cell
    if (MODE == MODE_VOTE) {
        // ---- clear the tile (a2, shared-memory part)
        for (int w = tid; w < ge.tile_words; w += ge.threads)
            tile[w] = 0u;
    } else {
        // ---- flag words of the reported peaks of every cell of the tile, and the number of
        // reported peaks below each word (peaks of global rank >= n_rep are not reported)
        const uint32_t n_rep = min(*p.n_peaks_dev, p.cap_peaks);
        uint32_t *ftile = tile, *ptile = tile + (size_t)wpr * ge.cells_pad;
        for (int cc = tid; cc < ge.cells_pad; cc += ge.threads) {
            const int cil = cc / ge.D, cjl = cc - cil * ge.D;
            uint32_t gb = 0, nr = 0;
            const uint32_t *fw = p.flags;
            if (cil < ni && cjl < nj) {
                size_t row = (size_t)(i0 + cil) * g.n_d0 + (j0 + cjl);
                gb = p.row_base[row];
                uint32_t cnt = p.row_base[row + 1] - gb;
                nr = gb >= n_rep ? 0u : min(cnt, n_rep - gb);
                fw += row * wpr;
            }
            uint32_t before = 0;
            for (int w = 0; w < wpr; ++w) {
                uint32_t f = nr ? fw[w] : 0u;
                while (before + (uint32_t)__popc(f) > nr) // the capacity cuts inside this word
                    f &= ~(0x80000000u >> __clz(f));
                ftile[(size_t)w * ge.cells_pad + cc] = f;
                ptile[(size_t)w * ge.cells_pad + cc] = before;
                before += (uint32_t)__popc(f);
            }
        }
        if (cell_ok)
            c_gbase = p.row_base[(size_t)(i0 + il) * g.n_d0 + (j0 + jl)];
    }
    __syncthreads();

    unsigned int my_votes = 0;
    unsigned long long tile_evals = 0; // thread 0: surviving hits x owned cells
    const int nkm1 = nk - 1;
    // VOTE: byte address of this cell's row in the tile and its word swizzle (in bytes)
    const int row_words = PACK == 2 ? (nk >> 1) : nk;
    const uint32_t row_addr = smem_u32(tile) + (uint32_t)c * (uint32_t)row_words * 4u;
    const uint32_t swzb = (uint32_t)(lane & p.swz_mask) << 2;
    // LIST: byte address of this cell's column in the flag tile; the prefix tile follows
    const uint32_t col_addr = smem_u32(tile) + (uint32_t)c * 4u;
    const uint32_t word_stride = (uint32_t)ge.cells_pad * 4u;
    const uint32_t prefix_off = (uint32_t)wpr * word_stride;

    for (uint32_t ch = 0; ch < n_chunks; ++ch) {
        const float *st = stage + (size_t)(ch & 1) * 4 * ge.chunk;
        mbar_wait(&mbar[ch & 1], (ch >> 1) & 1);
        if (tid == 0 && ch + 1 < n_chunks)
            issue(ch + 1); // the other buffer was released by the barrier ending chunk ch-1

        // ---- cull + order-preserving compaction of the survivors
        int total = 0;
        for (int base = 0; base < ge.chunk; base += ge.threads) {
            int hidx = base + tid;
            bool keep = false;
            float hx = 0.f, hy = 0.f, hr2 = 0.f;
            uint32_t hb = 0;
            if (hidx < ge.chunk) {
                hx = st[hidx];
                hy = st[ge.chunk + hidx];
                hr2 = st[2 * ge.chunk + hidx];
                hb = __float_as_uint(st[3 * ge.chunk + hidx]);
                keep = (hb != 0u) && hit_may_vote(hx, hy, hr2, tc, g.kabs, g.d0_absmax);
            }
            unsigned bal = __ballot_sync(0xffffffffu, keep);
            if (lane == 0)
                warp_cnt[warp] = __popc(bal);
            __syncthreads();
            int before = 0, all = 0;
            for (int w = 0; w < nwarps; ++w) {
                int cw = warp_cnt[w];
                before += (w < warp) ? cw : 0;
                all += cw;
            }
            if (keep) {
                int pos = total + before + __popc(bal & ((1u << lane) - 1u));
                uint32_t payload = (MODE == MODE_VOTE) ? hb : (uint32_t)(ch * ge.chunk + hidx);
                surv[pos] = make_float4(hx, hy, hr2, __uint_as_float(payload));
            }
            total += all;
            __syncthreads();
        }
        tile_evals += (unsigned long long)total * (unsigned)(ni * nj);
        if (tid < EVAL_UNROLL) // non-voting padding up to a multiple of the unroll factor
            surv[total + tid] = make_float4(0.f, 0.f, __int_as_float(0x7fc00000), 0.f);
        __syncthreads();

        // ---- evaluate: lane = cell, the warp walks the survivors
        for (int hs = set * EVAL_UNROLL; hs < total; hs += ge.split * EVAL_UNROLL) {
#pragma unroll
            for (int u = 0; u < EVAL_UNROLL; ++u) {
                const float4 hv = surv[hs + u];
                const float kappa = eval_kappa(hv.x, hv.y, hv.z, c_sn, c_cs, c_d0, c_2d0, c_d0sq);
                if ((kappa >= klo) && (kappa < khi)) {
                    const uint32_t k = (uint32_t)kappa_bin(kappa, klo, inv_dk, nkm1);
                    if (MODE == MODE_VOTE) {
                        const uint32_t bit = __float_as_uint(hv.w);
                        if (PACK == 2)
                            smem_red_or(row_addr + (((k << 1) ^ swzb) & ~3u), __funnelshift_l(0u, bit, k << 4));
                        else
                            smem_red_or(row_addr + ((k << 2) ^ swzb), bit);
                        ++my_votes;
                    } else {
                        const uint32_t wa = col_addr + (k >> 5) * word_stride;
                        const uint32_t f = smem_ld(wa);
                        if ((f >> (k & 31u)) & 1u) {
                            const uint32_t rank = smem_ld(wa + prefix_off) + (uint32_t)__popc(f & ((1u << (k & 31u)) - 1u));
                            const uint32_t gp = c_gbase + rank;
                            atomicAdd(&p.list_len[gp], 1u);
                            const uint2 pr = make_uint2(gp, __float_as_uint(hv.w));
                            const unsigned int pos = atomicAdd(&s_npairs[0], 1u);
                            if (pos < PAIR_BUF) {
                                pairbuf[pos] = pr;
                            } else { // buffer full inside one chunk: straight to global memory
                                unsigned long long gpos = atomicAdd(p.n_pairs, 1ull);
                                if (gpos < p.pair_cap)
                                    p.pairs[gpos] = pr;
                            }
                        }
                    }
                }
            }
        }
        __syncthreads(); // survivors and this stage buffer are free again

        if (MODE == MODE_LIST) {
            const unsigned int np = min(s_npairs[0], (unsigned int)PAIR_BUF);
            if (np >= PAIR_FLUSH || (ch + 1 == n_chunks && np > 0)) {
                if (tid == 0) {
                    unsigned long long b = atomicAdd(p.n_pairs, (unsigned long long)np);
                    s_npairs[1] = (unsigned int)b;
                    s_npairs[2] = (unsigned int)(b >> 32);
                }
                __syncthreads();
                const unsigned long long b = ((unsigned long long)s_npairs[2] << 32) | s_npairs[1];
                for (unsigned int q = tid; q < np; q += ge.threads)
                    if (b + q < p.pair_cap)
                        p.pairs[b + q] = pairbuf[q];
                __syncthreads();
                if (tid == 0)
                    s_npairs[0] = 0u;
                // the next write to s_npairs[0] / pairbuf is behind the barriers of the next cull
            }
        }
    }

    if (MODE == MODE_VOTE) {
        // ---- a4: write the tile out, kappa fastest, 16-byte stores
        if (PACK == 2) {
            const int W = nk >> 1;               // words per cell row
            const int pairs = (ge.P * ge.D) * (W >> 1);
            for (int q = tid; q < pairs; q += ge.threads) {
                int cc = q / (W >> 1), kw = (q - cc * (W >> 1)) << 1;
                int cil = cc / ge.D, cjl = cc - cil * ge.D;
                if (cil >= ni || cjl >= nj)
                    continue;
                int sw = (cc & 31) & p.swz_mask;
                uint32_t w0 = tile[(size_t)cc * W + (kw ^ sw)];
                uint32_t w1 = tile[(size_t)cc * W + ((kw + 1) ^ sw)];
                uint4 o = make_uint4(w0 & 0xffffu, w0 >> 16, w1 & 0xffffu, w1 >> 16);
                size_t lin = ((size_t)(i0 + cil) * g.n_d0 + (j0 + cjl)) * nk + (kw << 1);
                *reinterpret_cast<uint4 *>(p.acc + lin) = o;
            }
        } else {
            const int W = nk;
            const int quads = (ge.P * ge.D) * (W >> 2);
            for (int q = tid; q < quads; q += ge.threads) {
                int cc = q / (W >> 2), kw = (q - cc * (W >> 2)) << 2;
                int cil = cc / ge.D, cjl = cc - cil * ge.D;
                if (cil >= ni || cjl >= nj)
                    continue;
                int sw = (cc & 31) & p.swz_mask;
                const uint32_t *r = tile + (size_t)cc * W;
                uint4 o = make_uint4(r[kw ^ sw], r[(kw + 1) ^ sw], r[(kw + 2) ^ sw], r[(kw + 3) ^ sw]);
                size_t lin = ((size_t)(i0 + cil) * g.n_d0 + (j0 + cjl)) * nk + kw;
                *reinterpret_cast<uint4 *>(p.acc + lin) = o;
            }
        }
        // ---- a8: vote count (one global atomic per warp per tile)
        for (int o = 16; o > 0; o >>= 1)
            my_votes += __shfl_xor_sync(0xffffffffu, my_votes, o);
        if (lane == 0 && my_votes)
            atomicAdd(p.n_votes, (unsigned long long)my_votes);
        if (tid == 0 && tile_evals)
            atomicAdd(p.n_evals, tile_evals);
    }
}

// ------------------------------------------------------------------ host side
int hough_vote_max_smem(void) { return 227 * 1024; }

static int swizzle_mask_for(int row_words)
{
    int m = 31;
    while (m > 0 && (row_words % (m + 1)) != 0)
        m >>= 1;
    return m;
}

// Tile geometry.  Vote tile: cells_pad rows of n_kappa masks, PACK masks per word.
// List tile: the flag words and their popcount prefixes (2 words per 32 bins per cell)
// plus the pair buffer.
int sweep_geom_init(const hough_handle *h, SweepGeom *ge, int P, int D, int split, int list_mode)
{
    const hough_config &cfg = h->cfg;
    ge->P = P;
    ge->D = D;
    ge->cells_pad = ((P * D + 31) / 32) * 32;
    ge->groups = ge->cells_pad / 32;
    ge->split = split;
    ge->threads = 32 * ge->groups * split;
    ge->chunk = HOUGH_CHUNK;
    ge->tiles_phi = (cfg.n_phi + P - 1) / P;
    ge->tiles_d0 = (cfg.n_d0 + D - 1) / D;
    ge->n_tiles = ge->tiles_phi * ge->tiles_d0;
    size_t tile_bytes, extra = 0;
    if (list_mode) {
        tile_bytes = (size_t)2 * (cfg.n_kappa / 32) * ge->cells_pad * 4;
        extra = (size_t)PAIR_BUF * 8;
    } else {
        tile_bytes = (size_t)ge->cells_pad * cfg.n_kappa * 4 / h->g.pack;
    }
    ge->tile_words = (int)(tile_bytes / 4);
    size_t stage = (size_t)2 * 4 * ge->chunk * 4 + (size_t)(ge->chunk + EVAL_UNROLL) * 16 + 16 + 32 * 4 + 16 + 16;
    ge->smem_bytes = (int)(tile_bytes + extra + stage);
    // the interval test needs the slab to span well under a quarter turn
    double span = (cfg.phi_max - cfg.phi_min) * (double)(P - 1) / (double)cfg.n_phi;
    ge->no_phi_cull = (span > 1.0) ? 1 : 0;
    if (ge->threads > 1024 || ge->threads < 32)
        return 0;
    if (tile_bytes + extra + stage > (size_t)hough_vote_max_smem())
        return 0;
    return 1;
}

static void fill_params(hough_handle *h, SweepParams *p, const SweepGeom &ge)
{
    p->g = h->g;
    p->hits.x = h->hx;
    p->hits.y = h->hy;
    p->hits.r2 = h->hr2;
    p->hits.bit = h->hbit;
    p->hits.n = h->n_hits;
    p->hits.n_pad = ((h->n_hits + HOUGH_CHUNK - 1) / HOUGH_CHUNK) * HOUGH_CHUNK;
    p->geom = ge;
    int row_words = h->g.pack == 2 ? h->g.n_kappa / 2 : h->g.n_kappa;
    p->swz_mask = swizzle_mask_for(row_words);
    p->no_cull = (h->cfg.options & HOUGH_OPT_NO_CULL) ? 1 : 0;
    p->acc = h->acc;
    p->n_votes = &h->counters->n_votes;
    p->n_evals = &h->counters->n_evals;
    p->flags = h->flags;
    p->row_base = h->row_base;
    p->n_peaks_dev = &h->counters->n_peaks;
    p->cap_peaks = h->cfg.cap_peaks;
    p->list_len = h->list_len;
    p->pairs = h->pairs;
    p->n_pairs = h->n_pairs;
    p->pair_cap = h->cfg.cap_hits;
}

template <int MODE, int PACK>
static cudaError_t launch_one(const SweepParams &p, cudaStream_t st)
{
    static int configured_smem = -1; // per (MODE, PACK) instantiation
    if (configured_smem < p.geom.smem_bytes) {
        cudaError_t e = cudaFuncSetAttribute(k_sweep<MODE, PACK>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             p.geom.smem_bytes);
        if (e != cudaSuccess)
            return e;
        configured_smem = p.geom.smem_bytes;
    }
    k_sweep<MODE, PACK><<<p.geom.n_tiles, p.geom.threads, p.geom.smem_bytes, st>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_vote(hough_handle *h, cudaStream_t st)
{
    SweepParams p;
    fill_params(h, &p, h->vote_geom);
    h->launches += 1;
    return h->g.pack == 2 ? launch_one<MODE_VOTE, 2>(p, st) : launch_one<MODE_VOTE, 1>(p, st);
}

// One sweep: list_len[peak] (true lengths) and the (peak, hit) pairs.
cudaError_t launch_list_sweep(hough_handle *h, cudaStream_t st)
{
    SweepParams p;
    fill_params(h, &p, h->list_geom);
    h->launches += 1;
    return launch_one<MODE_LIST, 1>(p, st);
}
