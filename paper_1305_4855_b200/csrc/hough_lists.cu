// hough_lists.cu -- a7, the hit lists of the reported peaks (DESIGN.md
// section 4.4): "each peak is emitted with its sorted hit list" (BASELINE.json north_star),
// hit list of a peak = the hits whose own vote at the peak's (phi0, d0) cell lands in the
// peak's kappa bin, ascending hit index, CSR (A7).
//
// One sweep re-evaluates the votes and keeps those that land in a reported peak bin.  It
// is organised so that every entry already knows its final place in its list:
//   * a WARP owns a sub-tile of 32 (phi0, d0) cells (lane = cell) and walks the hits of ONE
//     segment of the event in ascending hit order, so the entries of a cell come out
//     ascending; a private shared-memory counter per peak hands out idx = 0, 1, 2, ...;
//   * the event's hits are cut into S segments (whole staged chunks); CTA = (super-tile of
//     LIST_WARPS sub-tiles, segment).  Sub-list (peak p, segment s) has the id p*S + s; the
//     concatenation of a peak's sub-lists in segment order is its ascending list;
//   * sub_len[p*S + s] is written at the end of the CTA; k_scan<LENS> sums a peak's S
//     lengths into hit_offset and leaves their exclusive prefix in sub_len;
//     k_scatter_entries drops entry (sub, hit, idx) at
//     hit_index[hit_offset[sub / S] + sub_len[sub] + idx].  No sort, no atomics on the lists.
// The hits are culled twice with the conservative interval test of DESIGN.md section 4.3:
// per CTA against the super-tile (lane = hit, order-preserving compaction) and per warp
// against its sub-tile (lane = hit, ballot), then the exact recipe runs on the survivors.
// If the entry buffer (cap_hits entries) overflows, the output is truncated anyway
// (n_hit_entries > cap_hits); k_scatter_entries then refills the lists that still fit
// directly from the hits, one warp per peak (list_slow).
#include "hough_device.cuh"

#define LIST_QUEUE 64  // entries a warp buffers before it flushes (>= 2 * 32)
#define LIST_ROUND 128 // CTA survivors a warp culls at a time
#define LIST_CHUNK 256 // hits staged per TMA bulk copy (divides HOUGH_CHUNK)
#define LIST_LQ 8      // pending votes per lane before the warp drains them

struct ListSweepParams {
    GridDev g;
    HitsDev hits;
    ListGeom geom;
    int no_cull;
    const uint32_t *flags;    // 1 bit per bin
    const uint32_t *row_base; // [n_rows + 1]
    const unsigned int *n_peaks_dev;
    uint32_t cap_peaks;
    uint32_t *sub_len;        // [cap_peaks * S], zeroed before the sweep
    uint32_t *ent_sub, *ent_hit, *ent_idx; // [ent_cap] entries
    unsigned long long *n_entries;
    unsigned long long ent_cap;
    unsigned long long *n_list_evals; // evaluations executed (hough_counts.n_list_evals)
    ApproxBin ab;
};

__device__ __forceinline__ unsigned short lds_u16(uint32_t addr)
{
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts_u16(uint32_t addr, unsigned short v)
{
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr), "h"(v) : "memory");
}

__device__ __forceinline__ void sts_u32(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// Per-warp shared-memory block; the fixed-size parts come first so that the hot loop
// addresses them with immediates off one register (wpr = n_kappa / 32):
//   widx    [LIST_ROUND + 4] u16   survivors of the warp-level cull (indices into surv)
//   laneq   [LIST_LQ][32] u32      per lane: pending (kappa bin << 10 | surv index)
//   flushq  [3][LIST_QUEUE] u32    finished entries on their way to global memory
//   flags   [wpr][32] u32   flag words of the reported peaks of the warp's cells
//   prefix  [wpr][32] u16   reported peaks of the cell below each word
//   count   [max_pk]  u16   entries handed out so far, per local peak id
#define OFF_WIDX 0
#define OFF_LANEQ 384
#define OFF_FLUSHQ (OFF_LANEQ + LIST_LQ * 128)
#define OFF_FLAGS (OFF_FLUSHQ + 3 * LIST_QUEUE * 4)
static_assert((LIST_ROUND + 4) * 2 <= OFF_LANEQ && OFF_FLAGS % 128 == 0, "per-warp block layout");

template <int OFF>
__device__ __forceinline__ uint32_t lds_off(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1+%2];" : "=r"(v) : "r"(addr), "n"(OFF));
    return v;
}
__device__ __forceinline__ float4 lds_f4(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
// WARPS: warps per CTA = sub-tiles per super-tile (ListGeom::warps).  APPROX: the hot loop
// finds the bin with the fixed-point estimate of hough_device.cuh; only
// candidates (the estimated bin is a reported peak, or the estimate is not decisive) reach
// the drain, which settles the undecided ones with the exact recipe.
template <int WARPS, bool APPROX>
__global__ void __launch_bounds__(32 * WARPS) k_list_sweep(const ListSweepParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const GridDev &g = p.g;
    const ListGeom &ge = p.geom;
    const int nk = g.n_kappa, wpr = nk >> 5;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int S = ge.S;

    // ---- which super-tile, which hit segment
    const int seg = blockIdx.x % S, tile_id = blockIdx.x / S;
    const int tp = tile_id / ge.tiles_d0, td = tile_id % ge.tiles_d0;
    const uint32_t n_chunks = p.hits.n_pad / LIST_CHUNK;
    const uint32_t ch0 = (uint32_t)(((unsigned long long)n_chunks * seg) / S);
    const uint32_t ch1 = (uint32_t)(((unsigned long long)n_chunks * (seg + 1)) / S);
    if (ch0 >= ch1)
        return; // empty segment: its sub-lists stay 0

    // ---- carve shared memory
    unsigned char *wbase = smem_raw + (size_t)warp * ge.warp_bytes;
    unsigned short *widx = reinterpret_cast<unsigned short *>(wbase + OFF_WIDX);
    uint32_t *wq = reinterpret_cast<uint32_t *>(wbase + OFF_FLUSHQ);
    uint32_t *wflags = reinterpret_cast<uint32_t *>(wbase + OFF_FLAGS);
    unsigned short *wpre = reinterpret_cast<unsigned short *>(wbase + OFF_FLAGS + (size_t)wpr * 128);
    unsigned short *wcnt = wpre + (size_t)wpr * 32;
    unsigned char *ptr = smem_raw + (size_t)WARPS * ge.warp_bytes;
    float *stage = reinterpret_cast<float *>(ptr); // [2][4][chunk]
    ptr += (size_t)2 * 4 * LIST_CHUNK * 4;
    float4 *surv = reinterpret_cast<float4 *>(ptr); // [chunk + 2]
    ptr += (size_t)(LIST_CHUNK + 2) * 16;
    uint64_t *mbar = reinterpret_cast<uint64_t *>(ptr);
    ptr += 16;
    int *warp_cnt = reinterpret_cast<int *>(ptr); // [LIST_WARPS]

    // ---- this warp's sub-tile and this lane's cell
    const int wp = warp / ge.WD, wd = warp % ge.WD;
    const int i0 = tp * ge.WP * ge.SP, j0 = td * ge.WD * ge.SD; // super-tile origin
    const int si0 = i0 + wp * ge.SP, sj0 = j0 + wd * ge.SD;
    const int sni = max(0, min(ge.SP, g.n_phi - si0)), snj = max(0, min(ge.SD, g.n_d0 - sj0));
    const int il = lane / ge.SD, jl = lane - il * ge.SD;
    const bool cell_ok = (il < sni) && (jl < snj);
    const bool warp_ok = sni > 0 && snj > 0;
    float c_sn = 0.f, c_cs = 0.f, c_d0 = 0.f, c_2d0 = 0.f, c_d0sq = __int_as_float(0x7fc00000);
    uint32_t c_row = 0;
    if (cell_ok) {
        c_sn = g.sn[si0 + il];
        c_cs = g.cs[si0 + il];
        c_d0 = g.d0c[sj0 + jl];
        c_2d0 = g.twod0[sj0 + jl];
        c_d0sq = g.d0sq[sj0 + jl];
        c_row = (uint32_t)(si0 + il) * (uint32_t)g.n_d0 + (uint32_t)(sj0 + jl);
    }
    const float klo = g.klo, khi = g.khi, inv_dk = g.inv_dk;
    const float ab_c1 = p.ab.c1, ab_c0 = p.ab.c0;
    const uint32_t ab_lim = p.ab.lim, ab_edge = p.ab.edge;

    // super-tile extent (CTA-level cull) and sub-tile extent (warp-level cull)
    const int ni = min(ge.WP * ge.SP, g.n_phi - i0), nj = min(ge.WD * ge.SD, g.n_d0 - j0);
    TileCull tc, wc;
    tc.snA = g.sn[i0];
    tc.csA = g.cs[i0];
    tc.snB = g.sn[i0 + ni - 1];
    tc.csB = g.cs[i0 + ni - 1];
    tc.dlo = g.d0c[j0];
    tc.dhi = g.d0c[j0 + nj - 1];
    tc.phi_all = ge.no_phi_cull_tile;
    tc.off = p.no_cull;
    wc = tc;
    if (warp_ok) {
        wc.snA = g.sn[si0];
        wc.csA = g.cs[si0];
        wc.snB = g.sn[si0 + sni - 1];
        wc.csB = g.cs[si0 + sni - 1];
        wc.dlo = g.d0c[sj0];
        wc.dhi = g.d0c[sj0 + snj - 1];
        wc.phi_all = ge.no_phi_cull_sub;
    }

    if (tid == 0) {
        mbar_init(&mbar[0], 1);
        mbar_init(&mbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t chunk_bytes = (uint32_t)LIST_CHUNK * 4;
    auto issue = [&](uint32_t ch) { // buffer and parity follow (ch - ch0)
        const uint32_t q = ch - ch0;
        float *dst = stage + (size_t)(q & 1) * 4 * LIST_CHUNK;
        uint64_t *bar = &mbar[q & 1];
        mbar_expect_tx(bar, 4 * chunk_bytes);
        size_t off = (size_t)ch * LIST_CHUNK;
        tma_load_1d(dst, p.hits.x + off, chunk_bytes, bar);
        tma_load_1d(dst + LIST_CHUNK, p.hits.y + off, chunk_bytes, bar);
        tma_load_1d(dst + 2 * LIST_CHUNK, p.hits.r2 + off, chunk_bytes, bar);
        tma_load_1d(dst + 3 * LIST_CHUNK, p.hits.bit + off, chunk_bytes, bar);
    };
    if (tid == 0)
        issue(ch0);

    // ---- per warp: flag words of the reported peaks of its 32 cells, the number of reported
    // peaks below each word, the local peak ids and their counters
    const uint32_t n_rep = min(*p.n_peaks_dev, p.cap_peaks);
    uint32_t c_gbase = 0, c_nrep = 0;
    {
        uint32_t nr = 0;
        const uint32_t *fw = p.flags;
        if (cell_ok) {
            c_gbase = p.row_base[c_row];
            const uint32_t cnt = p.row_base[c_row + 1] - c_gbase;
            nr = c_gbase >= n_rep ? 0u : min(cnt, n_rep - c_gbase);
            fw += (size_t)c_row * wpr;
        }
        uint32_t before = 0;
        for (int w = 0; w < wpr; ++w) {
            uint32_t f = nr ? fw[w] : 0u;
            while (before + (uint32_t)__popc(f) > nr) // the capacity cuts inside this word
                f &= ~(0x80000000u >> __clz(f));
            wflags[w * 32 + lane] = f;
            wpre[w * 32 + lane] = (unsigned short)before;
            before += (uint32_t)__popc(f);
        }
        c_nrep = before;
    }
    uint32_t c_lbase = c_nrep; // exclusive warp scan
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, c_lbase, o);
        if (lane >= o)
            c_lbase += t;
    }
    const uint32_t w_npk = __shfl_sync(0xffffffffu, c_lbase, 31);
    c_lbase -= c_nrep;
    for (uint32_t q = lane; q < w_npk; q += 32)
        wcnt[q] = 0;
    __syncwarp();

    const int nkm1 = nk - 1;
    const uint32_t wb = smem_u32(wbase);                              // the warp's block
    const uint32_t wl4 = wb + (uint32_t)lane * 4u;                    // this lane's column in it
    const uint32_t sv = smem_u32(surv);
    const uint32_t pre_addr = smem_u32(wpre) + (uint32_t)lane * 2u;   // + (k >> 5) * 64
    const uint32_t cnt_addr = smem_u32(wcnt) + c_lbase * 2u;          // + rank * 2
    const uint32_t sub0 = c_gbase * (uint32_t)S + (uint32_t)seg;      // + rank * S
    uint32_t *q_sub = wq, *q_hit = wq + LIST_QUEUE, *q_idx = wq + 2 * LIST_QUEUE;
    const uint32_t lt_mask = (1u << lane) - 1u;
    uint32_t qn = 0; // entries waiting in this warp's flush queue (warp-uniform)
    unsigned long long w_evals = 0; // hits x cells this warp evaluated (warp-uniform)
    uint32_t lqp = wl4; // + OFF_LANEQ: next free slot of this lane's queue (128 bytes apart)

    auto flush = [&]() {
        __syncwarp();
        unsigned long long b = 0;
        if (lane == 0)
            b = atomicAdd(p.n_entries, (unsigned long long)qn);
        b = __shfl_sync(0xffffffffu, b, 0);
        for (uint32_t e = lane; e < qn; e += 32)
            if (b + e < p.ent_cap) {
                p.ent_sub[b + e] = q_sub[e];
                p.ent_hit[b + e] = q_hit[e];
                p.ent_idx[b + e] = q_idx[e];
            }
        qn = 0;
        __syncwarp();
    };

    // Every lane turns its pending votes into entries, oldest first: rank of the bin among
    // the cell's reported peaks -> local peak id -> its counter (the place in the sub-list).
    auto drain = [&]() {
        const uint32_t nl = (lqp - wl4) >> 7;
        for (uint32_t e = 0;; ++e) {
            bool act = e < nl;
            if (!__any_sync(0xffffffffu, act))
                break;
            uint32_t k = 0, hit = 0;
            if (act) {
                const uint32_t ent = lds_off<OFF_LANEQ>(wl4 + e * 128u);
                if (APPROX) {
                    // ent = (t & ~511) | index: the bin is t >> 16 unless the coordinate is within
                    // edge (rounded up to a multiple of 512) steps above a bin edge, where the exact
                    // recipe decides
                    const float4 hv = surv[ent & 511u];
                    hit = __float_as_uint(hv.w);
                    k = ent >> APPROX_FRAC_BITS;
                    act = hit != 0xffffffffu; // the padding entry never counts
                    if ((ent & 0xfe00u) < ((ab_edge + 511u) & ~511u)) {
                        // r2 is recomputed from x, y (A2): the staged copy of a hit outside the
                        // estimate's range holds NaN instead
                        const float r2 = __fadd_rn(__fmul_rn(hv.x, hv.x), __fmul_rn(hv.y, hv.y));
                        const float kappa = eval_kappa(hv.x, hv.y, r2, c_sn, c_cs, c_d0, c_2d0, c_d0sq);
                        act = act && (kappa >= klo) && (kappa < khi);
                        k = act ? (uint32_t)kappa_bin(kappa, klo, inv_dk, nkm1) : 0u;
                        const uint32_t f = lds_off<OFF_FLAGS>(wl4 + ((k << 2) & ~127u));
                        act = act && ((f >> (k & 31u)) & 1u);
                    }
                } else {
                    hit = __float_as_uint(surv[ent & 1023u].w);
                    k = ent >> 10;
                }
            }
            const unsigned bh = __ballot_sync(0xffffffffu, act);
            if (act) {
                const uint32_t f = lds_off<OFF_FLAGS>(wl4 + ((k << 2) & ~127u));
                const uint32_t rank = lds_u16(pre_addr + (k >> 5) * 64u) + (uint32_t)__popc(f & ((1u << (k & 31u)) - 1u));
                const uint32_t ca = cnt_addr + rank * 2u;
                const unsigned short n = lds_u16(ca);
                sts_u16(ca, (unsigned short)(n + 1));
                const uint32_t pos = qn + (uint32_t)__popc(bh & lt_mask);
                q_sub[pos] = sub0 + rank * (uint32_t)S;
                q_hit[pos] = hit;
                q_idx[pos] = n;
            }
            qn += (uint32_t)__popc(bh);
            if (qn > LIST_QUEUE - 32)
                flush();
        }
        lqp = wl4;
    };

    // one hit against the warp's 32 cells: the bin, then the peak test of the bin
    auto process = [&](const float4 hv, const uint32_t sidx) {
        if (APPROX) {
            // e and den are the exact binary32 values of the recipe (A3)
            const float a = __fmul_rn(hv.x, c_sn);
            const float b = __fmul_rn(hv.y, c_cs);
            const float sv_ = __fsub_rn(b, a);
            const float e = __fsub_rn(sv_, c_d0);
            const float den = __fadd_rn(__fsub_rn(hv.z, __fmul_rn(c_2d0, sv_)), c_d0sq);
            const uint32_t t = approx_bin(e, den, ab_c1, ab_c0);
            if (t < ab_lim) {
                // flag word of bin t >> 16 (it may be n_kappa, just above khi: that word is not a
                // flag word, but then the estimate is undecided anyway)
                const uint32_t f = lds_off<OFF_FLAGS>(wl4 + ((t >> (APPROX_FRAC_BITS + 5)) << 7));
                const bool near = (t & 0xffffu) < ab_edge;
                if (near || ((f >> ((t >> APPROX_FRAC_BITS) & 31u)) & 1u)) {
                    // pending entry: the coordinate with its low 9 bits replaced by the index into surv
                    asm volatile("st.shared.u32 [%0+%1], %2;" ::"r"(lqp), "n"(OFF_LANEQ), "r"((t & ~511u) | sidx) : "memory");
                    lqp += 128u;
                }
            }
        } else {
            const float kappa = eval_kappa(hv.x, hv.y, hv.z, c_sn, c_cs, c_d0, c_2d0, c_d0sq);
            if ((kappa >= klo) && (kappa < khi)) {
                const uint32_t k = (uint32_t)kappa_bin(kappa, klo, inv_dk, nkm1);
                const uint32_t f = lds_off<OFF_FLAGS>(wl4 + ((k << 2) & ~127u));
                if ((f >> (k & 31u)) & 1u) {
                    asm volatile("st.shared.u32 [%0+%1], %2;" ::"r"(lqp), "n"(OFF_LANEQ), "r"((k << 10) | sidx) : "memory");
                    lqp += 128u;
                }
            }
        }
    };

    for (uint32_t ch = ch0; ch < ch1; ++ch) {
        const uint32_t q = ch - ch0;
        const float *st = stage + (size_t)(q & 1) * 4 * LIST_CHUNK;
        mbar_wait(&mbar[q & 1], (q >> 1) & 1);
        if (tid == 0 && ch + 1 < ch1)
            issue(ch + 1); // the other buffer was released by the barrier ending the previous chunk

        // ---- CTA-level cull against the super-tile, order-preserving compaction
        int total = 0;
        for (int base = 0; base < LIST_CHUNK; base += 32 * WARPS) {
            const int hidx = base + tid;
            float hx = 0.f, hy = 0.f, hr2 = 0.f;
            bool keep = false;
            if (hidx < LIST_CHUNK) {
                hx = st[hidx], hy = st[LIST_CHUNK + hidx], hr2 = st[2 * LIST_CHUNK + hidx];
                const uint32_t hb = __float_as_uint(st[3 * LIST_CHUNK + hidx]);
                keep = (hb != 0u) && hit_may_vote(hx, hy, hr2, tc, g.kabs, g.d0_absmax);
            }
            const unsigned bal = __ballot_sync(0xffffffffu, keep);
            if (lane == 0)
                warp_cnt[warp] = __popc(bal);
            __syncthreads();
            int all;
            const int before = warps_before(warp_cnt, WARPS, warp, lane, all);
            if (keep) // a hit outside the estimate's range is staged with r2 = NaN: every estimate says "undecided"
                surv[total + before + __popc(bal & lt_mask)] =
                    make_float4(hx, hy, (APPROX && hit_is_wild(hr2)) ? __int_as_float(0x7fc00000) : hr2,
                                __uint_as_float(ch * LIST_CHUNK + hidx));
            total += all;
            __syncthreads();
        }
        __syncthreads();
        if (tid == 0) { // the entry that pads odd batches: non-voting (exact path) / marked as padding
            if (APPROX) {
                const float4 h0 = surv[0]; // an ordinary evaluation whose entries the drain drops
                surv[total] = make_float4(h0.x, h0.y, h0.z, __uint_as_float(0xffffffffu));
            } else {
                surv[total] = make_float4(0.f, 0.f, __int_as_float(0x7fc00000), 0.f);
            }
        }
        __syncthreads();

        if (warp_ok) {
            for (int base = 0; base < total; base += LIST_ROUND) {
                // ---- warp-level cull against the sub-tile (lane = hit) -> widx[0 .. nw)
                int nw = 0;
#pragma unroll
                for (int r = 0; r < LIST_ROUND / 32 && base + r * 32 < total; ++r) {
                    const int idx = base + r * 32 + lane;
                    bool kw = false;
                    if (idx < total) {
                        const float4 hv = surv[idx];
                        kw = hit_may_vote(hv.x, hv.y, hv.z, wc, g.kabs, g.d0_absmax);
                    }
                    const unsigned bal = __ballot_sync(0xffffffffu, kw);
                    if (kw)
                        widx[nw + __popc(bal & lt_mask)] = (unsigned short)idx;
                    nw += __popc(bal);
                }
                w_evals += (unsigned long long)(nw * sni * snj);
                if (lane < 3)
                    widx[nw + lane] = (unsigned short)total; // pad to a multiple of 4 with the non-voting entry
                __syncwarp();
                // ---- lane = cell: the exact recipe on the survivors, four at a time
                for (int t = 0; t < nw; t += 4) {
                    const uint32_t wa = (wl4 & ~127u) + (uint32_t)t * 2u; // the block is 128-byte aligned
                    const uint32_t two0 = lds_off<OFF_WIDX>(wa), two1 = lds_off<OFF_WIDX + 4>(wa);
                    const uint32_t a = two0 & 0xffffu, b = two0 >> 16, c2 = two1 & 0xffffu, d2 = two1 >> 16;
                    const float4 h0 = lds_f4(sv + a * 16u), h1 = lds_f4(sv + b * 16u);
                    const float4 h2 = lds_f4(sv + c2 * 16u), h3 = lds_f4(sv + d2 * 16u);
                    process(h0, a);
                    process(h1, b);
                    process(h2, c2);
                    process(h3, d2);
                    if (__any_sync(0xffffffffu, lqp > wl4 + (LIST_LQ - 4) * 128u))
                        drain();
                }
                __syncwarp();
            }
            drain(); // surv is about to be reused
        }
        __syncthreads(); // survivors and this stage buffer are free again
    }

    if (qn)
        flush();
    if (lane == 0 && w_evals)
        atomicAdd(p.n_list_evals, w_evals);
    // ---- true lengths of this segment's sub-lists
    for (uint32_t r = 0; r < c_nrep; ++r)
        p.sub_len[(size_t)(c_gbase + r) * S + seg] = wcnt[c_lbase + r];
}

// ------------------------------------------------------------------ placement
struct ListPlaceParams {
    GridDev g;
    const float *hx, *hy, *hr2;
    const uint32_t *hbit;
    uint32_t n_hits;
    const unsigned long long *n_entries;
    unsigned long long ent_cap;
    const uint32_t *ent_sub, *ent_hit, *ent_idx;
    const uint32_t *sub_pre; // [n_rep * S] start of every sub-list inside its peak's list
    uint32_t S;
    const DevCounters *counters;
    uint32_t cap_peaks;
    const uint32_t *bin;
    const unsigned long long *hit_offset;
    uint32_t *hit_index;
    unsigned long long cap_hits;
};

// Entry buffer overflowed: write the lists that start below cap_hits straight from the
// hits, one warp per peak, ascending by construction.
__device__ void list_slow(const ListPlaceParams &p)
{
    const GridDev &g = p.g;
    const int lane = threadIdx.x & 31;
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    const uint32_t n = min(p.counters->n_peaks, p.cap_peaks);
    for (uint32_t pk = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; pk < n; pk += warps) {
        unsigned long long pos = p.hit_offset[pk];
        if (pos >= p.cap_hits)
            continue;
        const uint32_t lin = p.bin[pk];
        const uint32_t k = lin % (uint32_t)g.n_kappa, row = lin / (uint32_t)g.n_kappa;
        const uint32_t j = row % (uint32_t)g.n_d0, i = row / (uint32_t)g.n_d0;
        const float sn = g.sn[i], cs = g.cs[i], d0c = g.d0c[j], twod0 = g.twod0[j], d0sq = g.d0sq[j];
        for (uint32_t base = 0; base < p.n_hits; base += 32) {
            const uint32_t hidx = base + lane;
            bool in = false;
            if (hidx < p.n_hits && p.hbit[hidx] != 0u) {
                const float kappa = eval_kappa(p.hx[hidx], p.hy[hidx], p.hr2[hidx], sn, cs, d0c, twod0, d0sq);
                if ((kappa >= g.klo) && (kappa < g.khi))
                    in = (uint32_t)kappa_bin(kappa, g.klo, g.inv_dk, g.n_kappa - 1) == k;
            }
            const unsigned bal = __ballot_sync(0xffffffffu, in);
            if (in) {
                unsigned long long q = pos + __popc(bal & ((1u << lane) - 1u));
                if (q < p.cap_hits)
                    p.hit_index[q] = hidx;
            }
            pos += __popc(bal);
        }
    }
}

__global__ void __launch_bounds__(256) k_scatter_entries(const ListPlaceParams p)
{
    const unsigned long long n = *p.n_entries;
    if (n > p.ent_cap) {
        list_slow(p);
        return;
    }
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const uint32_t sub = p.ent_sub[i];
        const unsigned long long pos = p.hit_offset[sub / p.S] + p.sub_pre[sub] + p.ent_idx[i];
        if (pos < p.cap_hits)
            p.hit_index[pos] = p.ent_hit[i];
    }
}

// ------------------------------------------------------------------ host side
// Sub-tile = SP x SD = 32 cells (8 x 4 by default), super-tile = WP x WD sub-tiles, S hit
// segments chosen so that the CTAs fill a whole number of waves as nearly as possible.
static int list_segments_min(const hough_config *c)
{
    // u16 counters per (peak, segment): a segment is at most ceil(n_chunks / S) staged chunks
    // and must hold fewer than 65536 hits, i.e. at most 255 chunks of LIST_CHUNK = 256 hits
    const uint32_t hp = ((c->max_hits + HOUGH_CHUNK - 1) / HOUGH_CHUNK) * HOUGH_CHUNK;
    const uint32_t n_chunks = hp / LIST_CHUNK;
    const int s_min = (int)((n_chunks + 254u) / 255u);
    return s_min < 1 ? 1 : s_min;
}

// max_hits must leave S within LIST_MAX_SEGMENTS (k_sub_prefix stages 256 x (S + 1) words in
// static-limit shared memory): at most 16 x 255 x 256 = 1 044 480 hits per event.
int list_config_ok(const hough_config *c) { return list_segments_min(c) <= LIST_MAX_SEGMENTS; }

// Upper bound of S for a configuration (sizes the sub-list tables of the workspace).
int list_segments_bound(const hough_config *c)
{
    const int s_min = list_segments_min(c);
    int s_max = LIST_MAX_SEGMENTS;
    while (s_max > s_min && (unsigned long long)s_max * c->cap_peaks > (1ull << 26))
        --s_max;
    return s_max > s_min ? s_max : s_min;
}

template <bool APPROX>
static const void *list_sweep_fn_t(int warps)
{
    switch (warps) {
    case 16:
        return (const void *)k_list_sweep<16, APPROX>;
    case 8:
        return (const void *)k_list_sweep<8, APPROX>;
    case 4:
        return (const void *)k_list_sweep<4, APPROX>;
    case 2:
        return (const void *)k_list_sweep<2, APPROX>;
    default:
        return (const void *)k_list_sweep<1, APPROX>;
    }
}
static const void *list_sweep_fn(int warps, int approx)
{
    return approx ? list_sweep_fn_t<true>(warps) : list_sweep_fn_t<false>(warps);
}

int list_geom_init(hough_handle *h)
{
    const hough_config &c = h->cfg;
    ListGeom *ge = &h->list_geom;
    int SD = 4;
    while (SD > c.n_d0)
        SD >>= 1;
    int SP = 32 / SD, warps = LIST_WARPS;
    const int wpr = c.n_kappa / 32;
    // The per-warp tables grow with n_kappa: fewer warps per CTA first, then fewer cells per
    // warp (idle lanes), until the CTA fits (n_kappa = 256: 16 warps; 2048: 4; 16384: 1 warp
    // of 8 cells).
    for (;;) {
        ge->max_pk = ((SP + 1) / 2) * ((SD + 1) / 2) * ((c.n_kappa + 1) / 2);
        ge->warp_bytes = (OFF_FLAGS + wpr * 192 + ge->max_pk * 2 + 127) & ~127;
        ge->smem_bytes = warps * ge->warp_bytes + 2 * 4 * LIST_CHUNK * 4 + (LIST_CHUNK + 2) * 16 + 16 +
                         LIST_WARPS * 4 + 16;
        if (ge->smem_bytes <= hough_vote_max_smem())
            break;
        if (warps > 1)
            warps >>= 1;
        else if (SP > 1)
            SP >>= 1;
        else if (SD > 1)
            SD >>= 1;
        else
            return 0;
    }
    ge->SD = SD;
    ge->SP = SP;
    ge->warps = warps;
    ge->WD = 1;
    while (ge->WD < 4 && ge->WD * 2 <= warps && ge->WD * 2 * SD <= c.n_d0)
        ge->WD *= 2;
    ge->WP = warps / ge->WD;
    ge->tiles_phi = (c.n_phi + ge->WP * ge->SP - 1) / (ge->WP * ge->SP);
    ge->tiles_d0 = (c.n_d0 + ge->WD * ge->SD - 1) / (ge->WD * ge->SD);
    const double dphi = (c.phi_max - c.phi_min) / (double)c.n_phi;
    ge->no_phi_cull_tile = (dphi * (ge->WP * ge->SP - 1) > 1.0) ? 1 : 0;
    ge->no_phi_cull_sub = (dphi * (ge->SP - 1) > 1.0) ? 1 : 0;
    const void *fn = list_sweep_fn(ge->warps, h->ab.ok);
    if (ensure_dynamic_smem(fn, ge->smem_bytes) != cudaSuccess)
        return 0;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 32 * ge->warps, ge->smem_bytes) != cudaSuccess ||
        per_sm < 1)
        return 0;
    // segments: whole chunks, at most 65535 hits each (u16 counters), bounded sub-list table
    const uint32_t n_chunks_max = (h->max_hits_pad + LIST_CHUNK - 1) / LIST_CHUNK;
    const int s_min = list_segments_min(&c), s_bound = list_segments_bound(&c);
    int s_max = s_bound;
    if ((uint32_t)s_max > n_chunks_max)
        s_max = n_chunks_max > (uint32_t)s_min ? (int)n_chunks_max : s_min;
    const double slots = (double)h->n_sms * per_sm;
    const double tiles = (double)ge->tiles_phi * ge->tiles_d0;
    int best = s_min;
    double best_score = -1.0;
    for (int s = s_min; s <= s_max; ++s) {
        const double r = tiles * s / slots;
        const double eff = r / ceil(r);
        const double score = eff - 0.004 * s; // prefer fewer segments when the fill is equal
        if (score > best_score) {
            best_score = score;
            best = s;
        }
    }
    ge->S = best;
    return 1;
}

// sub_len[0 .. n_rep * S) = 0 (only the part this event uses)
__global__ void __launch_bounds__(256) k_zero_sub_len(uint32_t *sub_len, DevCounters *counters,
                                                      uint32_t cap_peaks, uint32_t S)
{
    if (blockIdx.x == 0 && threadIdx.x == 0)
        counters->n_list_evals = 0ull; // hough_peaks may be repeated on the same vote
    const size_t n = (size_t)min(counters->n_peaks, cap_peaks) * S;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        sub_len[i] = 0u;
}

cudaError_t launch_list_sweep(hough_handle *h, cudaStream_t st)
{
    ListSweepParams p;
    p.g = h->g;
    p.hits.x = h->hx;
    p.hits.y = h->hy;
    p.hits.r2 = h->hr2;
    p.hits.bit = h->hbit;
    p.hits.n = h->n_hits;
    p.hits.n_pad = ((h->n_hits + HOUGH_CHUNK - 1) / HOUGH_CHUNK) * HOUGH_CHUNK;
    p.geom = h->list_geom;
    p.no_cull = (h->cfg.options & HOUGH_OPT_NO_CULL) ? 1 : 0;
    p.flags = h->flags;
    p.row_base = h->row_base;
    p.n_peaks_dev = &h->counters->n_peaks;
    p.cap_peaks = h->cfg.cap_peaks;
    p.sub_len = h->list_len;
    p.ent_sub = h->ent_sub;
    p.ent_hit = h->ent_hit;
    p.ent_idx = h->ent_idx;
    p.n_entries = h->n_pairs;
    p.ent_cap = h->cfg.cap_hits;
    p.n_list_evals = &h->counters->n_list_evals;
    p.ab = h->ab;
    k_zero_sub_len<<<h->n_sms * 8, 256, 0, st>>>(h->list_len, h->counters, h->cfg.cap_peaks,
                                                 (uint32_t)h->list_geom.S);
    h->launches += 2;
    if (p.hits.n_pad == 0)
        return cudaGetLastError();
    const int blocks = h->list_geom.tiles_phi * h->list_geom.tiles_d0 * h->list_geom.S;
    void *args[] = {(void *)&p};
    return cudaLaunchKernel(list_sweep_fn(h->list_geom.warps, h->ab.ok), dim3(blocks), dim3(32 * h->list_geom.warps), args,
                            (size_t)h->list_geom.smem_bytes, st);
}

cudaError_t launch_place_lists(hough_handle *h, const hough_peaks_out *out, cudaStream_t st)
{
    ListPlaceParams p;
    p.g = h->g;
    p.hx = h->hx;
    p.hy = h->hy;
    p.hr2 = h->hr2;
    p.hbit = h->hbit;
    p.n_hits = h->n_hits;
    p.n_entries = h->n_pairs;
    p.ent_cap = h->cfg.cap_hits;
    p.ent_sub = h->ent_sub;
    p.ent_hit = h->ent_hit;
    p.ent_idx = h->ent_idx;
    p.sub_pre = h->list_len;
    p.S = (uint32_t)h->list_geom.S;
    p.counters = h->counters;
    p.cap_peaks = h->cfg.cap_peaks;
    p.bin = out->bin;
    p.hit_offset = reinterpret_cast<const unsigned long long *>(out->hit_offset);
    p.hit_index = out->hit_index;
    p.cap_hits = h->cfg.cap_hits;
    k_scatter_entries<<<h->n_sms * 16, 256, 0, st>>>(p);
    h->launches += 1;
    return cudaGetLastError();
}
