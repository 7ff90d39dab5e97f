// hough_sweep.cu -- the tiled sweep of the hits over the (phi0, d0) cells:
//   MODE_VOTE  : a3 vote into a shared-memory tile with atomicOr, a4 coalesced write-out,
//                a8 vote count
//   MODE_COUNT : a7 pass 1, length of each reported peak's hit list
//   MODE_FILL  : a7 pass 2, the hit indices themselves
// All three share the staging (TMA 1-D bulk copies of the SoA hit arrays into shared
// memory, double buffered), the conservative per-tile hit cull and the exact fp32
// evaluation of BASELINE.json north_star's closed form.
#include "hough_internal.cuh"

#define MODE_VOTE 0
#define MODE_COUNT 1
#define MODE_FILL 2

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
// DESIGN.md section 2, A3 + A4: every operation is one binary32 round-to-nearest
// operation, in this order, never contracted.  Returns the kappa bin or -1.
__device__ __forceinline__ int eval_bin(float x, float y, float r2, float sn, float cs, float d0c,
                                        float twod0, float d0sq, float klo, float khi, float inv_dk,
                                        int nk_minus_1)
{
    float a = __fmul_rn(x, sn);
    float b = __fmul_rn(y, cs);
    float s = __fsub_rn(b, a);
    float e = __fsub_rn(s, d0c);
    float num = __fadd_rn(e, e); // 2*e, exact
    float t = __fmul_rn(twod0, s);
    float u = __fsub_rn(r2, t);
    float den = __fadd_rn(u, d0sq);
    float kappa = __fdiv_rn(num, den);
    if (!((kappa >= klo) && (kappa < khi)))
        return -1;
    float qf = __fmul_rn(__fsub_rn(kappa, klo), inv_dk);
    int k = __float2int_rz(qf);
    return min(k, nk_minus_1);
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
    int swz_mask;             // XOR swizzle of the word index inside a cell row (vote tile)
    int slot_swz;             // same for the u16 slot tile of the hit-list passes
    int no_cull;
    uint32_t *acc;            // VOTE: global accumulator
    unsigned long long *n_votes;
    unsigned long long *n_evals;
    // hit lists
    const uint32_t *flags;    // 1 bit per bin
    const uint32_t *row_base; // [n_rows + 1]
    const unsigned int *n_peaks_dev;
    uint32_t cap_peaks;
    uint32_t *list_len;       // COUNT out
    const unsigned long long *hit_offset; // FILL in
    uint32_t *hit_index;      // FILL out
    unsigned long long cap_hits;
    int max_tile_peaks;
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

    // ---- carve shared memory
    uint32_t *tile = reinterpret_cast<uint32_t *>(smem_raw);
    unsigned char *ptr = smem_raw + (size_t)ge.tile_words * 4;
    uint32_t *pk_cnt = nullptr, *cell_lbase = nullptr, *cell_gbase = nullptr, *cell_nrep = nullptr;
    if (MODE != MODE_VOTE) {
        pk_cnt = reinterpret_cast<uint32_t *>(ptr);
        ptr += (size_t)((p.max_tile_peaks + 3) & ~3) * 4;
        cell_lbase = reinterpret_cast<uint32_t *>(ptr);
        ptr += (size_t)ge.cells_pad * 4;
        cell_gbase = reinterpret_cast<uint32_t *>(ptr);
        ptr += (size_t)ge.cells_pad * 4;
        cell_nrep = reinterpret_cast<uint32_t *>(ptr);
        ptr += (size_t)ge.cells_pad * 4;
    }
    float *stage = reinterpret_cast<float *>(ptr); // [2][4][chunk]
    ptr += (size_t)2 * 4 * ge.chunk * 4;
    float4 *surv = reinterpret_cast<float4 *>(ptr); // [chunk + EVAL_UNROLL]
    ptr += (size_t)(ge.chunk + EVAL_UNROLL) * 16;
    uint64_t *mbar = reinterpret_cast<uint64_t *>(ptr);
    ptr += 16;
    int *warp_cnt = reinterpret_cast<int *>(ptr); // [32]
    ptr += 32 * 4;

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
    const int swz = lane & p.swz_mask, sswz = lane & p.slot_swz;

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

    // ---- clear the tile (a2, shared-memory part)
    for (int w = tid; w < ge.tile_words; w += ge.threads)
        tile[w] = 0u;

    uint32_t n_rep = 0;
    if (MODE != MODE_VOTE) {
        // Local peak ids of the reported peaks (global rank < n_rep) inside this tile.
        n_rep = min(*p.n_peaks_dev, p.cap_peaks);
        for (int cc = tid; cc < ge.cells_pad; cc += ge.threads) {
            int cil = cc / ge.D, cjl = cc - cil * ge.D;
            uint32_t gb = 0, nr = 0;
            if (cil < ni && cjl < nj) {
                size_t row = (size_t)(i0 + cil) * g.n_d0 + (j0 + cjl);
                gb = p.row_base[row];
                uint32_t cnt = p.row_base[row + 1] - gb;
                nr = gb >= n_rep ? 0u : min(cnt, n_rep - gb);
            }
            cell_gbase[cc] = gb;
            cell_nrep[cc] = nr;
        }
        for (int w = tid; w < p.max_tile_peaks; w += ge.threads)
            pk_cnt[w] = 0u;
        __syncthreads();
        if (warp == 0) { // exclusive scan of cell_nrep over the tile's cells
            uint32_t carry = 0;
            for (int base = 0; base < ge.cells_pad; base += 32) {
                uint32_t v = cell_nrep[base + lane], incl = v;
                for (int o = 1; o < 32; o <<= 1) {
                    uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
                    if (lane >= o)
                        incl += t;
                }
                cell_lbase[base + lane] = carry + incl - v;
                carry += __shfl_sync(0xffffffffu, incl, 31);
            }
        }
        __syncthreads();
        // slot[(cell, k)] = local peak id + 1 for reported peaks (u16), 0 otherwise
        unsigned short *slot = reinterpret_cast<unsigned short *>(tile);
        const int words_per_row = nk >> 5;
        for (int cc = warp; cc < ge.cells_pad; cc += nwarps) {
            uint32_t nr = cell_nrep[cc];
            if (nr == 0)
                continue;
            int cil = cc / ge.D, cjl = cc - cil * ge.D;
            size_t row = (size_t)(i0 + cil) * g.n_d0 + (j0 + cjl);
            const uint32_t *fw = p.flags + row * words_per_row;
            uint32_t rank0 = 0;
            const int cswz = (cc & 31) & p.slot_swz;
            for (int wb = 0; wb < words_per_row; wb += 32) {
                uint32_t f = (wb + lane < words_per_row) ? fw[wb + lane] : 0u;
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
                    if (rank < nr) {
                        int k = ((wb + lane) << 5) + b;
                        int ks = (((k >> 1) ^ cswz) << 1) | (k & 1);
                        slot[(size_t)cc * nk + ks] = (unsigned short)(cell_lbase[cc] + rank + 1);
                    }
                    ++rank;
                }
                rank0 += __shfl_sync(0xffffffffu, incl, 31);
            }
        }
    }
    __syncthreads();

    unsigned int my_votes = 0;
    unsigned long long tile_evals = 0; // thread 0: surviving hits x owned cells
    const int row_words = PACK == 2 ? (nk >> 1) : nk;
    uint32_t *my_row = tile + (size_t)c * row_words; // VOTE
    const unsigned short *my_slots = reinterpret_cast<const unsigned short *>(tile) + (size_t)c * nk;
    const int nkm1 = nk - 1;

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
                float4 hv = surv[hs + u];
                int k = eval_bin(hv.x, hv.y, hv.z, c_sn, c_cs, c_d0, c_2d0, c_d0sq, g.klo, g.khi,
                                 g.inv_dk, nkm1);
                if (k >= 0) {
                    if (MODE == MODE_VOTE) {
                        uint32_t bit = __float_as_uint(hv.w);
                        if (PACK == 2)
                            atomicOr(&my_row[(k >> 1) ^ swz], bit << ((k & 1) << 4));
                        else
                            atomicOr(&my_row[k ^ swz], bit);
                        ++my_votes;
                    } else {
                        int ks = (((k >> 1) ^ sswz) << 1) | (k & 1);
                        uint32_t sl = my_slots[ks];
                        if (sl) {
                            uint32_t lid = sl - 1;
                            uint32_t idx = atomicAdd(&pk_cnt[lid], 1u);
                            if (MODE == MODE_FILL) {
                                uint32_t gp = cell_gbase[c] + (lid - cell_lbase[c]);
                                unsigned long long pos = p.hit_offset[gp] + idx;
                                if (pos < p.cap_hits)
                                    p.hit_index[pos] = __float_as_uint(hv.w);
                            }
                        }
                    }
                }
            }
        }
        __syncthreads(); // survivors and this stage buffer are free again
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
    } else if (MODE == MODE_COUNT) {
        // ---- list lengths of this tile's reported peaks -> list_len[global rank]
        for (int cc = tid; cc < ge.cells_pad; cc += ge.threads) {
            uint32_t nr = cell_nrep[cc], lb = cell_lbase[cc], gb = cell_gbase[cc];
            for (uint32_t r = 0; r < nr; ++r)
                p.list_len[gb + r] = pk_cnt[lb + r];
        }
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

// bytes_per_bin_x2: twice the shared-memory bytes per bin of the tile (VOTE pack 2 -> 4,
// pack 1 -> 8; slots -> 4).
int sweep_geom_init(const hough_handle *h, SweepGeom *ge, int P, int D, int split, int bytes_per_bin_x2,
                    int list_mode)
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
    size_t tile_bytes = (size_t)ge->cells_pad * cfg.n_kappa * bytes_per_bin_x2 / 2;
    ge->tile_words = (int)(tile_bytes / 4);
    size_t extra = 0;
    if (list_mode) {
        size_t maxpk = (size_t)((P + 1) / 2) * ((D + 1) / 2) * (cfg.n_kappa / 2);
        extra = ((maxpk + 3) & ~(size_t)3) * 4 + (size_t)ge->cells_pad * 12;
    }
    size_t stage = (size_t)2 * 4 * ge->chunk * 4 + (size_t)(ge->chunk + EVAL_UNROLL) * 16 + 16 + 32 * 4 + 16;
    ge->smem_bytes = (int)(tile_bytes + extra + stage);
    // the interval test needs the slab to span well under a quarter turn
    double span = (cfg.phi_max - cfg.phi_min) * (double)(P - 1) / (double)cfg.n_phi;
    ge->no_phi_cull = (span > 1.0) ? 1 : 0;
    if (ge->threads > 1024 || ge->threads < 32)
        return 0;
    if (ge->smem_bytes > hough_vote_max_smem())
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
    p->slot_swz = swizzle_mask_for(h->g.n_kappa / 2);
    p->no_cull = (h->cfg.options & HOUGH_OPT_NO_CULL) ? 1 : 0;
    p->acc = h->acc;
    p->n_votes = &h->counters->n_votes;
    p->n_evals = &h->counters->n_evals;
    p->flags = h->flags;
    p->row_base = h->row_base;
    p->n_peaks_dev = &h->counters->n_peaks;
    p->cap_peaks = h->cfg.cap_peaks;
    p->list_len = h->list_len;
    p->hit_offset = nullptr;
    p->hit_index = nullptr;
    p->cap_hits = h->cfg.cap_hits;
    p->max_tile_peaks = ((ge.P + 1) / 2) * ((ge.D + 1) / 2) * (h->g.n_kappa / 2);
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

cudaError_t launch_list_count(hough_handle *h, cudaStream_t st)
{
    SweepParams p;
    fill_params(h, &p, h->list_geom);
    h->launches += 1;
    return h->g.pack == 2 ? launch_one<MODE_COUNT, 2>(p, st) : launch_one<MODE_COUNT, 1>(p, st);
}

cudaError_t launch_list_fill(hough_handle *h, const hough_peaks_out *out, cudaStream_t st)
{
    SweepParams p;
    fill_params(h, &p, h->list_geom);
    p.hit_offset = reinterpret_cast<const unsigned long long *>(out->hit_offset);
    p.hit_index = out->hit_index;
    h->launches += 1;
    return h->g.pack == 2 ? launch_one<MODE_FILL, 2>(p, st) : launch_one<MODE_FILL, 1>(p, st);
}
