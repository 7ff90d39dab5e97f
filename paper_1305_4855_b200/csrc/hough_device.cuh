// hough_device.cuh -- device-side helpers shared by the sweep kernels (hough_sweep.cu,
// hough_lists.cu): TMA bulk-copy / mbarrier PTX wrappers, the exact fp32 evaluation of
// BASELINE.json north_star's closed form (A3/A4) and the conservative
// hit cull of DESIGN.md section 4.3.
#pragma once

#include "hough_internal.cuh"

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
// ------------------------------------------------------------------ vote variants (f3)
// SURVEY.md section 8(f) f3; recipes E1 / E2 of DESIGN.md section 8.  MODE 0: the closed form at
// the bin centres (one bin).  MODE 1: straight-line transform, the binned quantity is
// rho = y cos(theta) - x sin(theta) (Fig. 3).  MODE 2: interval voting, every bin
// between the closed-form values at the two phi0 bin EDGES (snB / csB = the upper edge).
struct CellConst {
    float sn, cs;   // bin centre (MODE 0, 1) or lower edge (MODE 2)
    float snB, csB; // upper edge (MODE 2)
    float d0c, twod0, d0sq;
};
// bins [k0, k1] that the hit votes into at this cell; false: no vote
template <int MODE>
__device__ __forceinline__ bool variant_bins(float x, float y, float r2, const CellConst &c, float klo, float khi,
                                             float inv_dk, int nkm1, int &k0, int &k1)
{
    if (MODE == VOTE_INTERVAL) {
        const float ka = eval_kappa(x, y, r2, c.sn, c.cs, c.d0c, c.twod0, c.d0sq);
        const float kb = eval_kappa(x, y, r2, c.snB, c.csB, c.d0c, c.twod0, c.d0sq);
        if (ka != ka || kb != kb)
            return false;
        const float lo = ka < kb ? ka : kb, hi = ka < kb ? kb : ka;
        if (hi < klo || lo >= khi)
            return false;
        k0 = (lo < klo) ? 0 : kappa_bin(lo, klo, inv_dk, nkm1);
        k1 = (hi >= khi) ? nkm1 : kappa_bin(hi, klo, inv_dk, nkm1);
        return true;
    }
    float v;
    if (MODE == VOTE_LINE)
        v = __fsub_rn(__fmul_rn(y, c.cs), __fmul_rn(x, c.sn));
    else
        v = eval_kappa(x, y, r2, c.sn, c.cs, c.d0c, c.twod0, c.d0sq);
    if (!((v >= klo) && (v < khi)))
        return false;
    k0 = k1 = kappa_bin(v, klo, inv_dk, nkm1);
    return true;
}
__device__ __forceinline__ CellConst cell_const(const GridDev &g, int mode, int i, int j)
{
    CellConst c;
    c.sn = mode == VOTE_INTERVAL ? g.sne[i] : g.sn[i];
    c.cs = mode == VOTE_INTERVAL ? g.cse[i] : g.cs[i];
    c.snB = mode == VOTE_INTERVAL ? g.sne[i + 1] : 0.f;
    c.csB = mode == VOTE_INTERVAL ? g.cse[i + 1] : 0.f;
    c.d0c = g.d0c[j];
    c.twod0 = g.twod0[j];
    c.d0sq = g.d0sq[j];
    return c;
}

// ------------------------------------------------------------------ the fast bin path
// The exact recipe costs ~14 issue slots for the IEEE divide, the two range compares and the
// bin.  The sweeps only need the BIN, so they first compute a 16.16 fixed-point estimate
//     t = trunc( e * rcp(den) * c1 + c0 )  ~=  (kappa - klo) * inv_dk * 2^16 + delta
// (MUFU.RCP + FMUL + FFMA + F2I; e and den are the exact binary32 values of the recipe) and
// use it only where it provably equals the exact result.  With U = n_kappa / 256 (one
// binary32 rounding of a coordinate below n_kappa * 2^16, in steps of 2^-16 bin) and
// A = max(|klo|, |khi|) / (khi - klo):  |estimate - exact qf * 2^16| <= E = (7A + 3) U + 1
// (2 ulp for the reciprocal, one rounding each for the product, the folded constant and the
// FMA, the truncation, plus the three roundings of the exact path itself).
// delta = ceil((12A + 8) max(U, 1)) > E + the offset of khi's own coordinate, so
//   (unsigned)t >= lim              kappa is outside [klo, khi) by more than E: no vote;
//   (t & 0xffff) <  edge = 2 delta   within delta of a bin edge (or of klo / khi; NaN gives
//                                    t = 0): the exact recipe decides;
//   otherwise                        the exact bin is t >> 16.
// Preconditions, checked on the host (approx_bin_init) and per hit (hit_is_wild): den is 0,
// +-inf, NaN or a normal number whose reciprocal is normal, so that MUFU.RCP's flush-to-zero
// never changes the outcome.  Hits outside that range take the exact recipe everywhere.
__device__ __forceinline__ uint32_t approx_bin(float e, float den, float c1, float c0)
{
    float rho;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rho) : "f"(den));
    const float p = __fmul_rn(e, rho);
    return (uint32_t)__float2int_rz(__fmaf_rn(p, c1, c0));
}
// r2 outside [2^-40, 2^80] (or NaN): the reciprocal of den could be flushed
__device__ __forceinline__ bool hit_is_wild(float r2)
{
    return !((r2 >= 9.094947017729282e-13f) && (r2 <= 1.2089258196146292e24f));
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

// Order-preserving compaction across the warps of a CTA: warp_cnt[w] holds the number of items
// warp w keeps (n_warps <= 32); every warp scans the counts with shuffles.  Returns the number
// of items of the warps before `warp`; `all` receives the CTA's total.
__device__ __forceinline__ int warps_before(const int *warp_cnt, int n_warps, int warp, int lane, int &all)
{
    const int cw = lane < n_warps ? warp_cnt[lane] : 0;
    int incl = cw;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o)
            incl += t;
    }
    all = __shfl_sync(0xffffffffu, incl, 31);
    return __shfl_sync(0xffffffffu, incl - cw, warp);
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
    if (!(ax <= 3.4028234664e38f) || !(ay <= 3.4028234664e38f))
        return false; // an inf / NaN coordinate never votes: s is +-inf or NaN, so num/den is NaN
    if (!(r2 <= 3.4028234664e38f))
        return true; // finite coordinates whose squares overflow: den = inf, kappa = +-0 may be in range
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


// ------------------------------------------------------------------ peak rule on popcount pairs
// A6 on 8 consecutive kappa bins of one (phi0, d0) cell (the fused / cell-wise peak test: k_sweep's
// epilogue and k_peak_cells).  A Strip holds popcounts as u16 pairs: word x[t] = bins 2t (low half) and
// 2t + 1 (high half) of the 8 bins, m = the word before (only its high half, bin -1, is used), p = the
// word after (only its low half, bin 8).  C = the cell itself, L = the bin-wise maximum over its
// neighbour cells of LOWER linear index, H = over those of HIGHER linear index (absent bins = 0).
// A bin is a peak iff pc >= L_min, pc > every lower-lin neighbour, pc >= every higher-lin neighbour.
struct Strip {
    uint32_t m, x[4], p;
};
__device__ __forceinline__ void strip_max(Strip &a, const Strip &b)
{
    a.m = __vmaxu2(a.m, b.m);
    a.p = __vmaxu2(a.p, b.p);
#pragma unroll
    for (int t = 0; t < 4; ++t)
        a.x[t] = __vmaxu2(a.x[t], b.x[t]);
}
__device__ __forceinline__ uint32_t peak_flags8(const Strip &C, const Strip &L, const Strip &H, uint32_t lmin2)
{
    const uint32_t HB = 0x80008000u, ONE = 0x00010001u;
    uint32_t byte = 0;
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        const uint32_t pC = t ? C.x[t - 1] : C.m, nC = t < 3 ? C.x[t + 1] : C.p;
        const uint32_t pL = t ? L.x[t - 1] : L.m, nL = t < 3 ? L.x[t + 1] : L.p;
        const uint32_t pH = t ? H.x[t - 1] : H.m, nH = t < 3 ? H.x[t + 1] : H.p;
        // (bin - 1, bin) and (bin + 1, bin + 2) re-paired so that every half sits beside its neighbour
        const uint32_t lfC = __byte_perm(pC, C.x[t], 0x5432), rtC = __byte_perm(C.x[t], nC, 0x5432);
        const uint32_t lfL = __byte_perm(pL, L.x[t], 0x5432), rtL = __byte_perm(L.x[t], nL, 0x5432);
        const uint32_t lfH = __byte_perm(pH, H.x[t], 0x5432), rtH = __byte_perm(H.x[t], nH, 0x5432);
        const uint32_t lo = __vmaxu2(__vimax3_u16x2(lfL, L.x[t], rtL), lfC);
        const uint32_t hi = __vimax3_u16x2(__vimax3_u16x2(lfH, H.x[t], rtH), rtC, lmin2);
        const uint32_t thr = __vmaxu2(lo + ONE, hi);
        const uint32_t res = (C.x[t] | HB) - thr; // bit 15 / 31: the half reaches its threshold
        byte |= ((res >> 15) & 1u) << (2 * t);
        byte |= (res >> 31) << (2 * t + 1);
    }
    return byte;
}
