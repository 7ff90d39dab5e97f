// hough_sweep.cu -- the tiled vote sweep of the hits over the (phi0, d0) cells: a3 vote into a
// shared-memory tile with shared atomic OR, a4 coalesced write-out, a8 vote count
// (DESIGN.md 4.1).  Hits are staged by TMA 1-D bulk copies of the
// SoA arrays into ONE shared-memory staging buffer (the survivors of a chunk are compacted out of it
// before they are evaluated, so the next chunk's copies land under the evaluation), culled per tile by
// the conservative interval test and evaluated with the exact fp32 recipe of BASELINE.json north_star's
// closed form (hough_device.cuh).
#include "hough_device.cuh"

#define EVAL_UNROLL 4
#define VOTE_CHUNK 1536 // hits staged per round of bulk copies (a multiple of HOUGH_CHUNK)

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
    ApproxBin ab;
    unsigned char *fused_flags; // HOUGH_OPT_FUSED_PEAKS: peak-flag bytes of the tile's interior cells (else NULL)
};

// APPROX: bins come from the fixed-point estimate wherever it provably equals the exact
// recipe (hough_device.cuh approx_bin); near a bin edge, and for hits whose
// r^2 is outside the estimate's admissible range, the exact recipe runs.
// MODE (with APPROX = false only): the vote variant, hough_device.cuh variant_bins.
template <int PACK, bool APPROX, int MODE>
__global__ void __launch_bounds__(1024, 1) k_sweep(const SweepParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const GridDev &g = p.g;
    const SweepGeom &ge = p.geom;
    const int nk = g.n_kappa;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nwarps = ge.threads >> 5;

    // ---- carve shared memory: tile = masks [P * D cells][nk / PACK words], then staging
    uint32_t *tile = reinterpret_cast<uint32_t *>(smem_raw);
    unsigned char *ptr = smem_raw + (size_t)ge.tile_words * 4;
    float *stage = reinterpret_cast<float *>(ptr); // [4][chunk]
    ptr += (size_t)4 * ge.chunk * 4;
    float4 *surv = reinterpret_cast<float4 *>(ptr); // [chunk + EVAL_UNROLL]
    ptr += (size_t)(ge.chunk + EVAL_UNROLL) * 16;
    uint64_t *mbar = reinterpret_cast<uint64_t *>(ptr);
    ptr += 16;
    ptr += 32 * 4;
    int *s_nwild = reinterpret_cast<int *>(ptr); // [4]: survivors of even / odd chunks, wild hits of even / odd chunks

    // ---- which tile: the first n_big phi0 slabs are P rows high, the others P_small
    // (two heights so that the CTAs fill whole waves)
    const int tp = blockIdx.x / ge.tiles_d0, td = blockIdx.x % ge.tiles_d0;
    const int Pt = tp < ge.n_big ? ge.P : ge.P_small;
    const int i0 = tp < ge.n_big ? tp * ge.P : ge.n_big * ge.P + (tp - ge.n_big) * ge.P_small;
    const int j0 = td * ge.D;
    const int ni = min(Pt, g.n_phi - i0), nj = min(ge.D, g.n_d0 - j0);

    // ---- this thread's cell and its constants (registers); warps beyond groups * split idle
    const int groups = (Pt * ge.D + 31) >> 5, split = nwarps / groups;
    const int grp = warp % groups, set = warp / groups;
    const int c = grp * 32 + lane;
    const int il = c / ge.D, jl = c - il * ge.D;
    const bool cell_ok = (il < ni) && (jl < nj);
    float c_sn = 0.f, c_cs = 0.f, c_d0 = 0.f, c_2d0 = 0.f, c_d0sq = __int_as_float(0x7fc00000);
    CellConst cc; // the same for the variants (MODE != 0); a padding lane's NaN never votes
    cc.sn = cc.cs = cc.snB = cc.csB = cc.d0c = cc.twod0 = cc.d0sq = __int_as_float(0x7fc00000);
    if (cell_ok) {
        c_sn = g.sn[i0 + il];
        c_cs = g.cs[i0 + il];
        c_d0 = g.d0c[j0 + jl];
        c_2d0 = g.twod0[j0 + jl];
        c_d0sq = g.d0sq[j0 + jl];
        if (MODE != VOTE_CENTRE)
            cc = cell_const(g, MODE, i0 + il, j0 + jl);
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
    const bool warp_ok = set < split;

    // chunks of ge.chunk hits; the padded hit count is a multiple of HOUGH_CHUNK, so the last chunk may
    // be shorter
    const uint32_t n_chunks = (p.hits.n_pad + ge.chunk - 1) / ge.chunk;

    if (tid < 4)
        s_nwild[tid] = 0; // survivor / wild counters of the even and odd chunks
    if (tid == 0) {
        mbar_init(&mbar[0], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // ONE staging buffer: the survivors of a chunk are compacted out of it before the evaluation, so
    // the next chunk's bulk copies are issued right after the cull and land under the evaluation
    auto issue = [&](uint32_t ch) {
        const size_t off = (size_t)ch * ge.chunk;
        const uint32_t bytes = (uint32_t)min((size_t)ge.chunk, (size_t)p.hits.n_pad - off) * 4u;
        mbar_expect_tx(&mbar[0], 4 * bytes);
        tma_load_1d(stage, p.hits.x + off, bytes, &mbar[0]);
        tma_load_1d(stage + ge.chunk, p.hits.y + off, bytes, &mbar[0]);
        tma_load_1d(stage + 2 * ge.chunk, p.hits.r2 + off, bytes, &mbar[0]);
        tma_load_1d(stage + 3 * ge.chunk, p.hits.bit + off, bytes, &mbar[0]);
    };
    // ---- clear the tile (a2, shared-memory part); everything up to here is independent of the hits,
    // so it may run while the preparation kernel is still draining (programmatic dependent launch)
    for (int w = tid; w < ge.tile_words; w += ge.threads)
        tile[w] = 0u;
    pdl_wait();
    if (tid == 0 && n_chunks > 0)
        issue(0);
    __syncthreads();

    const float ab_c1 = p.ab.c1, ab_c0 = p.ab.c0;
    const uint32_t ab_lim = p.ab.lim, ab_edge = p.ab.edge;
    unsigned int my_votes = 0;
    unsigned long long votes_wide = 0; // vote variants: my_votes is folded in after every hit (a whole-row fill is
                                       // up to 16384 votes, so 32 bits could wrap on very large events)
    unsigned long long tile_evals = 0; // thread 0: surviving hits x owned cells
    const int nkm1 = nk - 1;
    // byte address of this cell's row in the tile and its word swizzle (in bytes)
    const int row_words = PACK == 2 ? (nk >> 1) : nk;
    uint32_t row_addr = smem_u32(tile) + (uint32_t)c * (uint32_t)row_words * 4u;
    uint32_t swzb = (uint32_t)(lane & p.swz_mask) << 2;
    // keep both in registers: recomputing them inside the vote path costs more than it saves
    asm volatile("" : "+r"(row_addr), "+r"(swzb));

    for (uint32_t ch = 0; ch < n_chunks; ++ch) {
        const float *st = stage;
        const int len = (int)min((size_t)ge.chunk, (size_t)p.hits.n_pad - (size_t)ch * ge.chunk);
        mbar_wait(&mbar[0], ch & 1);

        // ---- cull + compaction of the survivors: ordinary hits from the front of surv, hits
        // outside the fast path's range ("wild") from its back.  Votes commute (OR), so the order
        // of the survivors is free: every warp reserves its places with one shared atomic (the
        // counter of chunk ch + 1 is cleared during the evaluation of chunk ch).
        int *s_total = s_nwild + (ch & 1), *s_wild = s_nwild + 2 + (ch & 1);
        for (int base = 0; base < len; base += ge.threads) {
            int hidx = base + tid;
            bool keep = false, wild = false;
            float hx = 0.f, hy = 0.f, hr2 = 0.f;
            uint32_t hb = 0;
            if (hidx < len) {
                hx = st[hidx];
                hy = st[ge.chunk + hidx];
                hr2 = st[2 * ge.chunk + hidx];
                hb = __float_as_uint(st[3 * ge.chunk + hidx]);
                keep = (hb != 0u) && hit_may_vote(hx, hy, hr2, tc, g.kabs, g.d0_absmax);
                if (APPROX) {
                    wild = keep && hit_is_wild(hr2);
                    keep = keep && !wild;
                }
            }
            const unsigned bal = __ballot_sync(0xffffffffu, keep);
            int wbase = 0;
            if (lane == 0 && bal)
                wbase = atomicAdd(s_total, __popc(bal));
            wbase = __shfl_sync(0xffffffffu, wbase, 0);
            if (keep)
                surv[wbase + __popc(bal & ((1u << lane) - 1u))] = make_float4(hx, hy, hr2, __uint_as_float(hb));
            if (APPROX && wild) // rare
                surv[ge.chunk + EVAL_UNROLL - 1 - atomicAdd(s_wild, 1)] = make_float4(hx, hy, hr2, __uint_as_float(hb));
        }
        __syncthreads();
        const int total = *s_total;
        const int n_wild = APPROX ? *s_wild : 0;
        if (tid == 0) {
            s_nwild[(ch + 1) & 1] = 0;
            s_nwild[2 + ((ch + 1) & 1)] = 0;
            if (ch + 1 < n_chunks)
                issue(ch + 1); // the staging buffer was released by the barrier above
        }
        tile_evals += (unsigned long long)(total + n_wild) * (unsigned)(ni * nj);
        if (!APPROX) {
            if (tid < EVAL_UNROLL) // non-voting padding up to a multiple of the unroll factor
                surv[total + tid] = make_float4(0.f, 0.f, __int_as_float(0x7fc00000), 0.f);
            __syncthreads();
        }

        // ---- evaluate: lane = cell, the `split` warps of a cell group interleave the survivors
        auto cast = [&](const uint32_t k, const uint32_t bit) {
            if (PACK == 2)
                smem_red_or(row_addr + (((k << 1) ^ swzb) & ~3u), __funnelshift_l(0u, bit, k << 4));
            else
                smem_red_or(row_addr + ((k << 2) ^ swzb), bit);
            ++my_votes;
        };
        auto exact = [&](const float4 hv) {
            if (MODE == VOTE_CENTRE) {
                const float kappa = eval_kappa(hv.x, hv.y, hv.z, c_sn, c_cs, c_d0, c_2d0, c_d0sq);
                if ((kappa >= klo) && (kappa < khi))
                    cast((uint32_t)kappa_bin(kappa, klo, inv_dk, nkm1), __float_as_uint(hv.w));
            } else {
                int k0, k1;
                if (__float_as_uint(hv.w) != 0u && variant_bins<MODE>(hv.x, hv.y, hv.z, cc, klo, khi, inv_dk, nkm1, k0, k1))
                    for (int k = k0; k <= k1; ++k)
                        cast((uint32_t)k, __float_as_uint(hv.w));
                votes_wide += my_votes;
                my_votes = 0;
            }
        };
        // the estimate of one (hit, cell): e and den are the exact binary32 values of the recipe (A3)
        auto estimate = [&](const float4 hv, float &e, float &den) -> uint32_t {
            const float a = __fmul_rn(hv.x, c_sn);
            const float b = __fmul_rn(hv.y, c_cs);
            const float sv = __fsub_rn(b, a);
            e = __fsub_rn(sv, c_d0);
            den = __fadd_rn(__fsub_rn(hv.z, __fmul_rn(c_2d0, sv)), c_d0sq);
            return approx_bin(e, den, ab_c1, ab_c0);
        };
        auto settle = [&](const uint32_t t, const float e, const float den, const uint32_t bit) {
            if (t < ab_lim) {
                if ((t & 0xffffu) < ab_edge) { // within delta of a bin edge: the exact recipe decides
                    const float kappa = __fdiv_rn(__fadd_rn(e, e), den);
                    if ((kappa >= klo) && (kappa < khi))
                        cast((uint32_t)kappa_bin(kappa, klo, inv_dk, nkm1), bit);
                } else {
                    cast(t >> APPROX_FRAC_BITS, bit);
                }
            }
        };
        if (warp_ok) {
            if (APPROX) {
                int hs = set * EVAL_UNROLL;
                for (; hs + EVAL_UNROLL <= total; hs += split * EVAL_UNROLL) {
                    // the four estimates first (independent chains), then the four votes
                    float4 hv[EVAL_UNROLL];
                    float e[EVAL_UNROLL], den[EVAL_UNROLL];
                    uint32_t t[EVAL_UNROLL];
#pragma unroll
                    for (int u = 0; u < EVAL_UNROLL; ++u) {
                        hv[u] = surv[hs + u];
                        t[u] = estimate(hv[u], e[u], den[u]);
                    }
#pragma unroll
                    for (int u = 0; u < EVAL_UNROLL; ++u)
                        settle(t[u], e[u], den[u], __float_as_uint(hv[u].w));
                }
                for (; hs < total; ++hs) { // the last, partial group of one set
                    const float4 hv = surv[hs];
                    float e, den;
                    const uint32_t t = estimate(hv, e, den);
                    settle(t, e, den, __float_as_uint(hv.w));
                }
                for (int w = set; w < n_wild; w += split)
                    exact(surv[ge.chunk + EVAL_UNROLL - 1 - w]);
            } else {
                for (int hs = set * EVAL_UNROLL; hs < total; hs += split * EVAL_UNROLL) {
#pragma unroll
                    for (int u = 0; u < EVAL_UNROLL; ++u)
                        exact(surv[hs + u]);
                }
            }
        }
        __syncthreads(); // survivors and this stage buffer are free again
    }

    {
        // ---- a4: write the tile out, kappa fastest, 16-byte stores
        if (PACK == 2) {
            const int W = nk >> 1;               // words per cell row
            const int pairs = (Pt * ge.D) * (W >> 1);
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
            const int quads = (Pt * ge.D) * (W >> 2);
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
        // ---- a5, fused variant (HOUGH_OPT_FUSED_PEAKS; BASELINE.json north_star: "peak finding is fused on
        // the tile"): the cells that are not on the tile's edge have all their 26 neighbours in this
        // tile, so their peak flags are decided here, from shared memory; the edge cells are left to
        // k_peak_cells (hough_peaks.cu).
        if (PACK == 2 && p.fused_flags != nullptr && ni > 2 && nj > 2) {
            const int W = nk >> 1, G = W >> 2; // words and 16-byte groups per cell row
            __syncthreads();                   // the write-out has read the masks
            // in place: masks -> popcount pairs, and the row swizzle undone (logical group q, word t sits
            // at group q ^ a, word t ^ b): groups q and q ^ a trade places, one thread does both
            for (int idx = tid; idx < Pt * ge.D * G; idx += ge.threads) {
                const int cc = idx / G, q = idx - cc * G;
                const int sw = (cc & 31) & p.swz_mask, q2 = q ^ (sw >> 2);
                if (q2 < q)
                    continue;
                uint4 *row = reinterpret_cast<uint4 *>(tile + (size_t)cc * W);
                auto conv = [&](uint4 v) -> uint4 {
                    if (sw & 1) {
                        uint32_t t0 = v.x; v.x = v.y; v.y = t0;
                        t0 = v.z; v.z = v.w; v.w = t0;
                    }
                    if (sw & 2) {
                        uint32_t t0 = v.x; v.x = v.z; v.z = t0;
                        t0 = v.y; v.y = v.w; v.w = t0;
                    }
                    v.x = (uint32_t)__popc(v.x & 0xffffu) | ((uint32_t)__popc(v.x >> 16) << 16);
                    v.y = (uint32_t)__popc(v.y & 0xffffu) | ((uint32_t)__popc(v.y >> 16) << 16);
                    v.z = (uint32_t)__popc(v.z & 0xffffu) | ((uint32_t)__popc(v.z >> 16) << 16);
                    v.w = (uint32_t)__popc(v.w & 0xffffu) | ((uint32_t)__popc(v.w >> 16) << 16);
                    return v;
                };
                const uint4 g1 = row[q], g2 = row[q2];
                row[q] = conv(g2);
                if (q2 != q)
                    row[q2] = conv(g1);
            }
            __syncthreads();
            const int nseg = (G + 31) >> 5, wj = nj - 2, n_items = (ni - 2) * wj * nseg;
            const uint32_t lmin2 = (uint32_t)g.L_min * 0x00010001u;
            auto load = [&](int cil, int cjl, int q) -> Strip {
                const uint32_t *row = tile + (size_t)(cil * ge.D + cjl) * W;
                const uint4 v = *reinterpret_cast<const uint4 *>(row + 4 * q);
                Strip s;
                s.x[0] = v.x, s.x[1] = v.y, s.x[2] = v.z, s.x[3] = v.w;
                s.m = q > 0 ? row[4 * q - 1] : 0u;
                s.p = q + 1 < G ? row[4 * q + 4] : 0u;
                return s;
            };
            for (int item = warp; item < n_items; item += nwarps) {
                const int ic = item / nseg, q = (item - ic * nseg) * 32 + lane;
                const int cil = 1 + ic / wj, cjl = 1 + ic % wj;
                if (q >= G)
                    continue;
                const Strip C = load(cil, cjl, q);
                Strip L = load(cil - 1, cjl - 1, q), H = load(cil + 1, cjl + 1, q);
                strip_max(L, load(cil - 1, cjl, q));
                strip_max(L, load(cil - 1, cjl + 1, q));
                strip_max(L, load(cil, cjl - 1, q));
                strip_max(H, load(cil, cjl + 1, q));
                strip_max(H, load(cil + 1, cjl - 1, q));
                strip_max(H, load(cil + 1, cjl, q));
                const size_t rowg = (size_t)(i0 + cil) * g.n_d0 + (j0 + cjl);
                p.fused_flags[rowg * (size_t)(nk >> 3) + q] = (unsigned char)peak_flags8(C, L, H, lmin2);
            }
        }
        // ---- a8: vote count (one global atomic per warp per tile)
        unsigned long long warp_votes = votes_wide + my_votes;
        for (int o = 16; o > 0; o >>= 1)
            warp_votes += __shfl_xor_sync(0xffffffffu, warp_votes, o);
        if (lane == 0 && warp_votes)
            atomicAdd(p.n_votes, warp_votes);
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

template <int PACK>
static const void *sweep_kernel_pack(const hough_handle *h)
{
    if (h->mode == VOTE_LINE)
        return (const void *)k_sweep<PACK, false, VOTE_LINE>;
    if (h->mode == VOTE_INTERVAL)
        return (const void *)k_sweep<PACK, false, VOTE_INTERVAL>;
    return h->ab.ok ? (const void *)k_sweep<PACK, true, VOTE_CENTRE> : (const void *)k_sweep<PACK, false, VOTE_CENTRE>;
}
static const void *sweep_kernel(const hough_handle *h)
{
    return h->g.pack == 2 ? sweep_kernel_pack<2>(h) : sweep_kernel_pack<1>(h);
}

// Tile geometry: P x D rows of n_kappa masks, PACK masks per word, plus the staging.
int sweep_geom_init(const hough_handle *h, SweepGeom *ge, int P, int D, int split, int fit_waves)
{
    const hough_config &cfg = h->cfg;
    ge->P = P;
    ge->D = D;
    ge->cells_pad = ((P * D + 31) / 32) * 32;
    ge->groups = ge->cells_pad / 32;
    ge->split = split;
    ge->threads = 32 * ge->groups * split;
    ge->chunk = VOTE_CHUNK;
    ge->tiles_phi = (cfg.n_phi + P - 1) / P;
    ge->tiles_d0 = (cfg.n_d0 + D - 1) / D;
    ge->n_tiles = ge->tiles_phi * ge->tiles_d0;
    // rows for the P x D cells only: padding lanes of the last cell group never vote
    const size_t tile_bytes = (size_t)(P * D) * cfg.n_kappa * 4 / h->g.pack, extra = 0;
    ge->tile_words = (int)(tile_bytes / 4);
    size_t stage = (size_t)4 * ge->chunk * 4 + (size_t)(ge->chunk + EVAL_UNROLL) * 16 + 16 + 32 * 4 + 16 + 16;
    ge->smem_bytes = (int)(tile_bytes + extra + stage);
    // the interval test needs the slab to span well under a quarter turn
    double span = (cfg.phi_max - cfg.phi_min) * (double)(P - 1) / (double)cfg.n_phi;
    ge->no_phi_cull = (span > 1.0) ? 1 : 0;
    if (ge->threads > 1024 || ge->threads < 32)
        return 0;
    if (tile_bytes + extra + stage > (size_t)hough_vote_max_smem())
        return 0;
    ge->n_big = ge->tiles_phi;
    ge->P_small = P;
    // Two slab heights: n_big slabs of P rows first, then slabs of P - (one cell group) rows,
    // chosen so that the CTAs fill whole waves (cost model: a wave takes as long as its
    // highest tile).
    const int step = (D <= 32 && 32 % D == 0) ? 32 / D : 0;
    if (fit_waves && step > 0 && P % step == 0 && P - step >= step) {
        int per_sm = 0;
        const void *fn = sweep_kernel(h);
        cudaError_t e = ensure_dynamic_smem(fn, ge->smem_bytes);
        if (e == cudaSuccess)
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, ge->threads, ge->smem_bytes);
        if (e != cudaSuccess || per_sm < 1) {
            cudaGetLastError();
            return 1;
        }
        const long long slots = (long long)h->n_sms * per_sm, T = ge->tiles_d0;
        const int Ps = P - step, n_phi = cfg.n_phi;
        const int ns_min = (n_phi + P - 1) / P, ns_max = (n_phi + Ps - 1) / Ps;
        long long best_cost = (long long)P * ((ns_min * T + slots - 1) / slots);
        for (int ns = ns_min + 1; ns <= ns_max; ++ns) {
            int a = (n_phi - ns * Ps + step - 1) / step;
            if (n_phi - ns * Ps <= 0)
                a = 0;
            if (a > ns)
                continue;
            if (ns > a && (long long)a * P + (long long)(ns - a - 1) * Ps >= n_phi)
                continue; // the last slab would be empty
            const long long w_big = (a * T + slots - 1) / slots, w_all = (ns * T + slots - 1) / slots;
            const long long cost = P * w_big + Ps * (w_all - w_big);
            if (cost < best_cost) {
                best_cost = cost;
                ge->tiles_phi = ns;
                ge->n_big = a;
                ge->P_small = Ps;
            }
        }
        ge->n_tiles = ge->tiles_phi * ge->tiles_d0;
    }
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
    p->no_cull = ((h->cfg.options & HOUGH_OPT_NO_CULL) || h->mode != VOTE_CENTRE) ? 1 : 0;
    p->acc = h->acc;
    p->n_votes = &h->counters->n_votes;
    p->n_evals = &h->counters->n_evals;
    p->ab = h->ab;
    p->fused_flags = (h->cfg.options & HOUGH_OPT_FUSED_PEAKS) ? reinterpret_cast<unsigned char *>(h->flags) : nullptr;
}

cudaError_t launch_vote(hough_handle *h, cudaStream_t st)
{
    SweepParams p;
    fill_params(h, &p, h->vote_geom);
    h->launches += 1;
    const void *fn = sweep_kernel(h);
    cudaError_t e = ensure_dynamic_smem(fn, p.geom.smem_bytes);
    if (e != cudaSuccess)
        return e;
    h->fused_valid = p.fused_flags != nullptr ? 1 : 0;
    void *args[] = {(void *)&p};
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(p.geom.n_tiles);
    cfg.blockDim = dim3(p.geom.threads);
    cfg.dynamicSmemBytes = (size_t)p.geom.smem_bytes;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelExC(&cfg, fn, args);
}
