/*
 * hough_ext_oracle.c -- CPU ORACLE for the rows SURVEY.md section 8(f) marks "next":
 *   f1  second Hough transform over the peaks (displaced-jet vertices)   PAPER.md:154-160 (section 9)
 *   f2  track fit of each peak's hit list + duplicate removal            PAPER.md:146 (section 8), :104
 *   f3  variants of the vote: straight-line transform, interval voting   PAPER.md:122 (Fig. 3), :124
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as hough_oracle.c: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load
 * or call it; it shares no code, header, table or constant generator with the CUDA path under
 * paper_1305_4855_b200/csrc/).  It is linked with hough_oracle.c, whose A1 tables
 * (oracle_tables) and A6 peak rule (oracle_peaks) it re-uses unchanged.
 *
 * The paper gives these steps in words only; DESIGN.md section 8 states the recipes
 * E1..E5 written out below and lists the readings taken.  Integer / index results are
 * defined bit-exactly: every floating-point operation that decides a bin is ONE IEEE-754
 * binary32 operation, round-to-nearest-even, in the order written, never fused
 * (build.py: -ffp-contract=off).  The fit (E5) is binary64 in a fixed summation order.
 *
 * Pins (tests/test_ext_oracle_pins.py, -m "not gpu"): fp64 geometry written differently
 * (line-through-column crossings, tangent lines of circles through a common vertex, the
 * point-on-circle test of the interval's end points), textbook reductions (rho = x cos
 * + y sin), exact-circle and straight-line recoveries and a Gauss-Newton geometric fit for
 * E5, brute-force set arithmetic for the duplicate rule.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t n_layers;
    int32_t n_phi, n_d0, n_kappa;
    int32_t L_min;
    int32_t phi_wrap;
    double phi_min, phi_max;
    double d0_min, d0_max;
    double kappa_min, kappa_max;
} oracle_grid; /* the struct of hough_oracle.c */

void oracle_tables(const oracle_grid *g, float *sn, float *cs, float *d0c, float *twod0, float *d0sq,
                   float *kscal);

typedef struct {
    float *sn, *cs, *d0c, *twod0, *d0sq;
    float ks[3];
} tables_t;

static void tables_make(const oracle_grid *g, tables_t *t)
{
    t->sn = malloc(sizeof(float) * g->n_phi);
    t->cs = malloc(sizeof(float) * g->n_phi);
    t->d0c = malloc(sizeof(float) * g->n_d0);
    t->twod0 = malloc(sizeof(float) * g->n_d0);
    t->d0sq = malloc(sizeof(float) * g->n_d0);
    oracle_tables(g, t->sn, t->cs, t->d0c, t->twod0, t->d0sq, t->ks);
}
static void tables_free(tables_t *t)
{
    free(t->sn); free(t->cs); free(t->d0c); free(t->twod0); free(t->d0sq);
}

/* ======================================================================================
 * E1/E2 -- variants of the vote (f3).
 *
 * mode 0  the closed form of hough_oracle.c (single bin per (hit, i, j)); here only so that
 *         the variants can be compared with it by the pins.
 * mode 1  E1, STRAIGHT-LINE transform (Fig. 3: "each hit results in a sinusoidal
 *         curve in the parameter space"): parameters (theta, rho); the grid's phi axis is
 *         theta, n_d0 must be 1 and the grid's kappa axis is rho [cm].  For hit h and theta
 *         centre i:   a = x*sn[i];  b = y*cs[i];  rho = b - a
 *         (the signed distance from the origin of the line with direction theta through the
 *         hit: the kappa -> 0 limit of the closed form, d0 = -x sin(phi0) + y cos(phi0)).
 *         Vote iff klo <= rho < khi, bin as A4.
 * mode 2  E2, INTERVAL voting for the circle transform ("fill
 *         the kappa range spanned across a phi0 bin"): with the phi0 bin EDGES
 *         phi_e[i] = phi_min + i (phi_max - phi_min)/n_phi  (fp64, sin/cos rounded once to
 *         binary32), ka = A3 at (edge i, d0 centre j), kb = A3 at (edge i+1, d0 centre j).
 *         No vote if either is NaN.  lo = min(ka, kb), hi = max(ka, kb); no vote if
 *         hi < klo or lo >= khi.  Otherwise every bin k0..k1 gets the bit, with
 *         k0 = (lo < klo) ? 0 : bin(lo),  k1 = (hi >= khi) ? n_kappa-1 : bin(hi)   (bin = A4).
 *         n_votes counts the bins set, one per (hit, i, j, k).  (A pole of kappa(phi0) inside
 *         the bin -- a hit within one bin's arc of the point of closest approach -- is not
 *         treated specially: DESIGN.md section 8, reading X2.)
 * ====================================================================================== */
static float kappa_A3(float x, float y, float r2, float sn, float cs, float d0c, float twod0, float d0sq)
{
    float a = x * sn;
    float b = y * cs;
    float s = b - a;
    float e = s - d0c;
    float num = 2.0f * e;
    float t = twod0 * s;
    float u = r2 - t;
    float den = u + d0sq;
    return num / den;
}

static int bin_A4(float v, float klo, float inv_dk, int n_kappa)
{
    float qf = (v - klo) * inv_dk;
    int k = (int)qf;
    if (k > n_kappa - 1)
        k = n_kappa - 1;
    return k;
}

/* bins [k0, k1] voted by (hit, i, j) under `mode`; returns 0 for no vote */
static int variant_bins(int mode, float x, float y, float r2, const tables_t *t, const float *sne,
                        const float *cse, int i, int j, int n_kappa, int *k0, int *k1)
{
    const float klo = t->ks[0], khi = t->ks[1], inv_dk = t->ks[2];
    if (mode == 0 || mode == 1) {
        float v;
        if (mode == 0) {
            v = kappa_A3(x, y, r2, t->sn[i], t->cs[i], t->d0c[j], t->twod0[j], t->d0sq[j]);
        } else {
            float a = x * t->sn[i];
            float b = y * t->cs[i];
            v = b - a;
        }
        if (!((v >= klo) && (v < khi)))
            return 0;
        *k0 = *k1 = bin_A4(v, klo, inv_dk, n_kappa);
        return 1;
    }
    float ka = kappa_A3(x, y, r2, sne[i], cse[i], t->d0c[j], t->twod0[j], t->d0sq[j]);
    float kb = kappa_A3(x, y, r2, sne[i + 1], cse[i + 1], t->d0c[j], t->twod0[j], t->d0sq[j]);
    if (ka != ka || kb != kb)
        return 0;
    float lo = ka < kb ? ka : kb, hi = ka < kb ? kb : ka;
    if (hi < klo || lo >= khi)
        return 0;
    *k0 = (lo < klo) ? 0 : bin_A4(lo, klo, inv_dk, n_kappa);
    *k1 = (hi >= khi) ? n_kappa - 1 : bin_A4(hi, klo, inv_dk, n_kappa);
    return 1;
}

static void edge_tables(const oracle_grid *g, float *sne, float *cse)
{
    for (int i = 0; i <= g->n_phi; ++i) {
        double pe = g->phi_min + (double)i * (g->phi_max - g->phi_min) / (double)g->n_phi;
        sne[i] = (float)sin(pe);
        cse[i] = (float)cos(pe);
    }
}

static void hit_prep(const oracle_grid *g, const float *x, const float *y, const int32_t *layer, uint32_t n,
                     float *r2, uint32_t *bit, uint32_t *n_bad)
{
    uint32_t bad = 0;
    for (uint32_t h = 0; h < n; ++h) {
        float p = x[h] * x[h];
        float q = y[h] * y[h];
        r2[h] = p + q;
        if (layer[h] < 0 || layer[h] >= g->n_layers) {
            bit[h] = 0u;
            ++bad;
        } else {
            bit[h] = 1u << layer[h];
        }
    }
    *n_bad = bad;
}

/* The variant vote over the whole grid (accumulator defined from scratch). Returns n_votes. */
uint64_t oracle_vote_variant(const oracle_grid *g, int mode, const float *x, const float *y,
                             const int32_t *layer, uint32_t n, uint32_t *acc, uint32_t *n_bad_out)
{
    const int np = g->n_phi, nd = g->n_d0, nk = g->n_kappa;
    tables_t t;
    tables_make(g, &t);
    float *sne = malloc(sizeof(float) * (np + 1)), *cse = malloc(sizeof(float) * (np + 1));
    edge_tables(g, sne, cse);
    float *r2 = malloc(sizeof(float) * (n ? n : 1));
    uint32_t *bit = malloc(sizeof(uint32_t) * (n ? n : 1));
    hit_prep(g, x, y, layer, n, r2, bit, n_bad_out);
    memset(acc, 0, sizeof(uint32_t) * (size_t)np * nd * nk);
    uint64_t n_votes = 0;
#pragma omp parallel for schedule(static) reduction(+ : n_votes)
    for (int i = 0; i < np; ++i)
        for (int j = 0; j < nd; ++j) {
            uint32_t *row = acc + ((size_t)i * nd + j) * nk;
            for (uint32_t h = 0; h < n; ++h) {
                int k0, k1;
                if (!bit[h] || !variant_bins(mode, x[h], y[h], r2[h], &t, sne, cse, i, j, nk, &k0, &k1))
                    continue;
                for (int k = k0; k <= k1; ++k)
                    row[k] |= bit[h];
                n_votes += (uint64_t)(k1 - k0 + 1);
            }
        }
    free(sne); free(cse); free(r2); free(bit);
    tables_free(&t);
    return n_votes;
}

/* A7 under a variant: H(peak) = hits whose vote at the peak's cell covers the peak's bin. */
uint64_t oracle_hitlists_variant(const oracle_grid *g, int mode, const float *x, const float *y,
                                 const int32_t *layer, uint32_t n, const uint32_t *peak_bin, uint64_t n_peaks,
                                 uint64_t *hit_offset, uint32_t *hit_index, uint64_t cap_hits)
{
    const int np = g->n_phi, nd = g->n_d0, nk = g->n_kappa;
    tables_t t;
    tables_make(g, &t);
    float *sne = malloc(sizeof(float) * (np + 1)), *cse = malloc(sizeof(float) * (np + 1));
    edge_tables(g, sne, cse);
    float *r2 = malloc(sizeof(float) * (n ? n : 1));
    uint32_t *bit = malloc(sizeof(uint32_t) * (n ? n : 1));
    uint32_t n_bad;
    hit_prep(g, x, y, layer, n, r2, bit, &n_bad);
    uint64_t w = 0;
    for (uint64_t p = 0; p < n_peaks; ++p) { /* ascending peaks, ascending hits: the CSR order */
        uint32_t lin = peak_bin[p];
        int k = (int)(lin % (uint32_t)nk);
        int j = (int)((lin / (uint32_t)nk) % (uint32_t)nd);
        int i = (int)(lin / ((uint32_t)nk * (uint32_t)nd));
        hit_offset[p] = w;
        for (uint32_t h = 0; h < n; ++h) {
            int k0, k1;
            if (!bit[h] || !variant_bins(mode, x[h], y[h], r2[h], &t, sne, cse, i, j, nk, &k0, &k1))
                continue;
            if (k0 <= k && k <= k1) {
                if (w < cap_hits)
                    hit_index[w] = h;
                ++w;
            }
        }
    }
    hit_offset[n_peaks] = w;
    free(sne); free(cse); free(r2); free(bit);
    tables_free(&t);
    return w;
}

/*
 * The same lists, walked cell by cell (the analogue of oracle_hitlists_cells in hough_oracle.c): peaks in
 * ascending lin, so the peaks of one (i, j) cell are consecutive; for every such run one pass over the hits,
 * variant_bins once per hit, and the hit joins every peak of the run whose bin lies in [k0, k1].  The
 * (peak, hit) pairs wait in a buffer until all lengths, hence the offsets, are known.  Pinned against
 * oracle_hitlists_variant (tests/test_ext_oracle_pins.py).
 */
uint64_t oracle_hitlists_variant_cells(const oracle_grid *g, int mode, const float *x, const float *y,
                                       const int32_t *layer, uint32_t n, const uint32_t *peak_bin, uint64_t n_peaks,
                                       uint64_t *hit_offset, uint32_t *hit_index, uint64_t cap_hits)
{
    const int np = g->n_phi, nd = g->n_d0, nk = g->n_kappa;
    tables_t t;
    tables_make(g, &t);
    float *sne = malloc(sizeof(float) * (np + 1)), *cse = malloc(sizeof(float) * (np + 1));
    edge_tables(g, sne, cse);
    float *r2 = malloc(sizeof(float) * (n ? n : 1));
    uint32_t *bit = malloc(sizeof(uint32_t) * (n ? n : 1));
    uint32_t n_bad;
    hit_prep(g, x, y, layer, n, r2, bit, &n_bad);
    uint64_t *len = calloc(n_peaks + 1, sizeof(uint64_t));
    uint64_t a = 0;
    /* pairs of all runs, run after run, in (run, h, peak) order */
    uint64_t cap_pairs = 1024, n_pairs = 0;
    uint64_t *pair_peak = malloc(sizeof(uint64_t) * cap_pairs);
    uint32_t *pair_hit = malloc(sizeof(uint32_t) * cap_pairs);
    while (a < n_peaks) {
        uint64_t b = a + 1;
        while (b < n_peaks && peak_bin[b] / (uint32_t)nk == peak_bin[a] / (uint32_t)nk)
            ++b;
        const uint32_t cell = peak_bin[a] / (uint32_t)nk;
        const int j = (int)(cell % (uint32_t)nd), i = (int)(cell / (uint32_t)nd);
        for (uint32_t h = 0; h < n; ++h) {
            int k0, k1;
            if (!bit[h] || !variant_bins(mode, x[h], y[h], r2[h], &t, sne, cse, i, j, nk, &k0, &k1))
                continue;
            for (uint64_t p = a; p < b; ++p) {
                const int k = (int)(peak_bin[p] % (uint32_t)nk);
                if (k < k0 || k > k1)
                    continue;
                if (n_pairs == cap_pairs) {
                    cap_pairs *= 2;
                    pair_peak = realloc(pair_peak, sizeof(uint64_t) * cap_pairs);
                    pair_hit = realloc(pair_hit, sizeof(uint32_t) * cap_pairs);
                }
                pair_peak[n_pairs] = p;
                pair_hit[n_pairs] = h;
                ++n_pairs;
                ++len[p];
            }
        }
        a = b;
    }
    uint64_t total = 0;
    for (uint64_t p = 0; p < n_peaks; ++p) {
        hit_offset[p] = total;
        total += len[p];
        len[p] = hit_offset[p]; /* becomes the write position */
    }
    hit_offset[n_peaks] = total;
    for (uint64_t c = 0; c < n_pairs; ++c) { /* a peak's pairs come in ascending h */
        const uint64_t w = len[pair_peak[c]]++;
        if (w < cap_hits)
            hit_index[w] = pair_hit[c];
    }
    free(len); free(pair_peak); free(pair_hit);
    free(sne); free(cse); free(r2); free(bit);
    tables_free(&t);
    return total;
}

/* ======================================================================================
 * E3 -- f1, the SECOND Hough transform, over the peaks of the first ("the
 * crossings all lie along a single sinusoidal curve in the parameter space ... that one
 * sinusoidal curve corresponds to a point in the original x-y space ... the vertex of the
 * displaced jet ... use the Hough transform a second time, this time applying it not to the
 * hits in the x-y space but the crossings in the parameter space").
 *
 * The sinusoid of a vertex V = (xv, yv) is d0 = -xv sin(phi0) + yv cos(phi0) (the tangent
 * line of a track at its point of closest approach passes through V; exact for kappa = 0,
 * off by kappa |V - P0|^2 / 2 otherwise: reading X3).  A peak at bin (i, j, k) is the point
 * (phi0_i, d0_j) of the parameter space (its kappa is not used); it votes along the line
 * it defines in the (xv, yv) plane, once per bin centre of the axis the line is less steep
 * against:
 *   V1 tables: xc[a] = (float)(x_min + (a + 0.5)(x_max - x_min)/n_x), yc[b] likewise;
 *      xlo = (float)x_min, xhi = (float)x_max, inv_dx = (float)(n_x/(x_max - x_min)); y likewise.
 *   V2 with sn = sn[i], cs = cs[i], d = d0c[j] (the A1 tables of the first transform):
 *      if |cs| >= |sn|:  for every a:  t = xc[a]*sn;  u = d + t;  yv = u / cs;
 *                        vote iff ylo <= yv < yhi into b = min((int)((yv - ylo)*inv_dy), n_y - 1);
 *      else:             for every b:  t = yc[b]*cs;  u = t - d;  xv = u / sn;
 *                        vote iff xlo <= xv < xhi into a = min((int)((xv - xlo)*inv_dx), n_x - 1).
 *      vacc[a*n_y + b] += 1 (uint32 counts; every reported peak has weight 1, so a track's
 *      mirror peak and plateau neighbours raise the same bins: reading X4).
 *   V3 vertex peaks: count >= V_min and, over the (up to 8) existing neighbours (no wrap),
 *      count(n) < count(b), or equal and lin(n) > lin(b); ascending lin = a*n_y + b.
 *   V4 members of a vertex bin (a, b): the peaks whose own V2 vote at column a (|cs| >= |sn|)
 *      or row b (otherwise) lands in (a, b); ascending peak position, CSR.
 * ====================================================================================== */
typedef struct {
    double x_min, x_max, y_min, y_max;
    int32_t n_x, n_y;
    int32_t V_min;
    int32_t reserved;
} oracle_vgrid;

void oracle_vertex_tables(const oracle_vgrid *v, float *xc, float *yc, float *scal /* xlo,xhi,inv_dx,ylo,yhi,inv_dy */)
{
    for (int a = 0; a < v->n_x; ++a)
        xc[a] = (float)(v->x_min + ((double)a + 0.5) * (v->x_max - v->x_min) / (double)v->n_x);
    for (int b = 0; b < v->n_y; ++b)
        yc[b] = (float)(v->y_min + ((double)b + 0.5) * (v->y_max - v->y_min) / (double)v->n_y);
    scal[0] = (float)v->x_min;
    scal[1] = (float)v->x_max;
    scal[2] = (float)((double)v->n_x / (v->x_max - v->x_min));
    scal[3] = (float)v->y_min;
    scal[4] = (float)v->y_max;
    scal[5] = (float)((double)v->n_y / (v->y_max - v->y_min));
}

/* V2 for one peak cell (sn, cs, d) at index q of the axis it iterates: the bin it votes
 * into along the other axis, or -1.  *steep = 1 when the iterated axis is y. */
static int vertex_vote_one(float sn, float cs, float d, int q, const float *xc, const float *yc,
                           const float *sc, int n_x, int n_y, int *steep)
{
    if (fabsf(cs) >= fabsf(sn)) {
        *steep = 0;
        float t = xc[q] * sn;
        float u = d + t;
        float yv = u / cs;
        if (!((yv >= sc[3]) && (yv < sc[4])))
            return -1;
        float qf = (yv - sc[3]) * sc[5];
        int b = (int)qf;
        return b > n_y - 1 ? n_y - 1 : b;
    }
    *steep = 1;
    float t = yc[q] * cs;
    float u = t - d;
    float xv = u / sn;
    if (!((xv >= sc[0]) && (xv < sc[1])))
        return -1;
    float qf = (xv - sc[0]) * sc[2];
    int a = (int)qf;
    return a > n_x - 1 ? n_x - 1 : a;
}

uint64_t oracle_vertex_vote(const oracle_grid *g, const oracle_vgrid *v, const uint32_t *peak_bin,
                            uint64_t n_peaks, uint32_t *vacc)
{
    tables_t t;
    tables_make(g, &t);
    float *xc = malloc(sizeof(float) * v->n_x), *yc = malloc(sizeof(float) * v->n_y), sc[6];
    oracle_vertex_tables(v, xc, yc, sc);
    memset(vacc, 0, sizeof(uint32_t) * (size_t)v->n_x * v->n_y);
    uint64_t votes = 0;
    for (uint64_t p = 0; p < n_peaks; ++p) {
        uint32_t row = peak_bin[p] / (uint32_t)g->n_kappa;
        int j = (int)(row % (uint32_t)g->n_d0), i = (int)(row / (uint32_t)g->n_d0);
        float sn = t.sn[i], cs = t.cs[i], d = t.d0c[j];
        int steep = fabsf(cs) >= fabsf(sn) ? 0 : 1;
        int nq = steep ? v->n_y : v->n_x;
        for (int q = 0; q < nq; ++q) {
            int st, o = vertex_vote_one(sn, cs, d, q, xc, yc, sc, v->n_x, v->n_y, &st);
            if (o < 0)
                continue;
            int a = steep ? o : q, b = steep ? q : o;
            vacc[(size_t)a * v->n_y + b] += 1u;
            ++votes;
        }
    }
    free(xc); free(yc);
    tables_free(&t);
    return votes;
}

uint64_t oracle_vertex_peaks(const oracle_vgrid *v, const uint32_t *vacc, uint32_t *vbin, uint32_t *vcount,
                             uint64_t cap)
{
    uint64_t n = 0;
    for (int a = 0; a < v->n_x; ++a)
        for (int b = 0; b < v->n_y; ++b) {
            size_t lin = (size_t)a * v->n_y + b;
            uint32_t c = vacc[lin];
            if (c < (uint32_t)v->V_min)
                continue;
            int ok = 1;
            for (int da = -1; da <= 1 && ok; ++da)
                for (int db = -1; db <= 1 && ok; ++db) {
                    int aa = a + da, bb = b + db;
                    if ((da == 0 && db == 0) || aa < 0 || aa >= v->n_x || bb < 0 || bb >= v->n_y)
                        continue;
                    size_t ln = (size_t)aa * v->n_y + bb;
                    if (vacc[ln] > c || (vacc[ln] == c && ln < lin))
                        ok = 0;
                }
            if (ok) {
                if (n < cap) {
                    vbin[n] = (uint32_t)lin;
                    vcount[n] = c;
                }
                ++n;
            }
        }
    return n;
}

uint64_t oracle_vertex_members(const oracle_grid *g, const oracle_vgrid *v, const uint32_t *peak_bin,
                               uint64_t n_peaks, const uint32_t *vbin, uint64_t n_vertices,
                               uint64_t *member_offset, uint32_t *member_index, uint64_t cap)
{
    tables_t t;
    tables_make(g, &t);
    float *xc = malloc(sizeof(float) * v->n_x), *yc = malloc(sizeof(float) * v->n_y), sc[6];
    oracle_vertex_tables(v, xc, yc, sc);
    uint64_t w = 0;
    for (uint64_t m = 0; m < n_vertices; ++m) {
        int a = (int)(vbin[m] / (uint32_t)v->n_y), b = (int)(vbin[m] % (uint32_t)v->n_y);
        member_offset[m] = w;
        for (uint64_t p = 0; p < n_peaks; ++p) {
            uint32_t row = peak_bin[p] / (uint32_t)g->n_kappa;
            int j = (int)(row % (uint32_t)g->n_d0), i = (int)(row / (uint32_t)g->n_d0);
            float sn = t.sn[i], cs = t.cs[i], d = t.d0c[j];
            int steep = fabsf(cs) >= fabsf(sn) ? 0 : 1, st;
            int o = vertex_vote_one(sn, cs, d, steep ? b : a, xc, yc, sc, v->n_x, v->n_y, &st);
            if (o >= 0 && o == (steep ? a : b)) {
                if (w < cap)
                    member_index[w] = (uint32_t)p;
                ++w;
            }
        }
    }
    member_offset[n_vertices] = w;
    free(xc); free(yc);
    tables_free(&t);
    return w;
}

/* ======================================================================================
 * E4/E5 -- f2, the fit of every peak's hit list and the removal of duplicates
 * ("perform a fit of the hits to the candidate tracks"; "the track
 * candidate collection is then cleaned to remove duplicate tracks or tracks which share a
 * large number of hits").
 *
 * E4 FIT.  The closed form of the transform, kappa (r^2 - 2 d0 s + d0^2) = 2 (s - d0) with
 * s = -x sin(phi0) + y cos(phi0), divided by 2 (1 + kappa d0), reads
 *        khat r^2 - s + delta = 0,   khat = kappa / (2 (1 + kappa d0)),
 *                                    delta = d0 (1 + kappa d0 / 2) / (1 + kappa d0),
 * which is linear in (khat, delta) for a given direction phi0.  Minimising the sum of its
 * squares over the list (unit weights) has the closed-form solution written below
 * (non-iterative circle fit in the track parameters, Karimaki's method restated for this
 * sign convention; derivation in DESIGN.md section 8).  All in binary64, sums taken over the
 * list in its (ascending hit) order, means first, then central moments:
 *   mx = sum x / n, my = sum y / n, mr = sum (x^2 + y^2) / n;
 *   u = x - mx, v = y - my, w = (x^2 + y^2) - mr;
 *   Cxx = sum u u / n, Cxy = sum u v / n, Cyy = sum v v / n, Cxr = sum u w / n, Cyr = sum v w / n,
 *   Crr = sum w w / n;
 *   q1 = Crr Cxy - Cxr Cyr;  q2 = Crr (Cxx - Cyy) - Cxr^2 + Cyr^2;  phi = atan2(2 q1, q2) / 2;
 *   sp = sin phi, cp = cos phi;  khat = (-sp Cxr + cp Cyr) / Crr;
 *   delta = (-mx sp + my cp) - khat mr;  D = 1 - 4 delta khat  (= 1/(1 + kappa d0)^2);
 *   kappa = 2 khat / sqrt(D);  d0 = 2 delta / (1 + sqrt(D));
 *   rms = sqrt((sum eps^2 / n) / D),  eps = khat w - (-sp u + cp v)   [cm]
 *   (eps is the residual khat r^2 - s + delta of the hit written with the centred moments; a
 *   third pass over the list.  Algebraically sum eps^2 / n = sp^2 Cxx - 2 sp cp Cxy + cp^2 Cyy
 *   - khat^2 Crr, but that difference of ~1e3 cm^2 terms leaves ~1e-7 relative rounding noise on
 *   a 1e-6 cm^2 variance, which would make the selection rms <= rms_max depend on the math
 *   library: DESIGN.md section 8, reading X6.)
 * phi is defined modulo pi; (phi + pi, -d0, -kappa) is the same circle.  The representation
 * reported is the FORWARD one: mx cp + my sp >= 0 (the hits lie ahead of the point of closest
 * approach), otherwise phi -= or += pi (into [-pi, pi)), d0 = -d0, kappa = -kappa -- exact
 * sign flips, so the two mirror peaks of a track with equal hit lists get
 * bit-identical kappa, d0 and rms.  status: 0 ok; 1 fewer than 3 hits; 2 degenerate
 * (Crr = 0, D <= 0 or a non-finite result).
 *
 * E5 SELECTION and DUPLICATES.  A candidate is selected iff status == 0 and rms <= rms_max.
 * A selected candidate c is a duplicate iff some other selected c' shares at least
 * `min_shared` hits with it and is better: more layers in its mask; else smaller rms; else
 * lower peak position.  (Domination, not a greedy chain: the rule has no order dependence.)
 * ====================================================================================== */
typedef struct {
    double kappa, phi0, d0, rms;
} oracle_fit;

static const double ORACLE_PI = 3.14159265358979323846; /* binary64 nearest to pi */

int oracle_fit_one(const float *x, const float *y, const uint32_t *idx, uint32_t n, oracle_fit *out)
{
    out->kappa = out->phi0 = out->d0 = out->rms = 0.0;
    if (n < 3)
        return 1;
    double sx = 0.0, sy = 0.0, sr = 0.0;
    for (uint32_t q = 0; q < n; ++q) {
        double xv = (double)x[idx[q]], yv = (double)y[idx[q]];
        sx += xv;
        sy += yv;
        sr += xv * xv + yv * yv;
    }
    const double dn = (double)n;
    const double mx = sx / dn, my = sy / dn, mr = sr / dn;
    double Cxx = 0.0, Cxy = 0.0, Cyy = 0.0, Cxr = 0.0, Cyr = 0.0, Crr = 0.0;
    for (uint32_t q = 0; q < n; ++q) {
        double xv = (double)x[idx[q]], yv = (double)y[idx[q]];
        double u = xv - mx, v = yv - my, w = (xv * xv + yv * yv) - mr;
        Cxx += u * u;
        Cxy += u * v;
        Cyy += v * v;
        Cxr += u * w;
        Cyr += v * w;
        Crr += w * w;
    }
    Cxx /= dn; Cxy /= dn; Cyy /= dn; Cxr /= dn; Cyr /= dn; Crr /= dn;
    if (!(Crr > 0.0))
        return 2;
    const double q1 = Crr * Cxy - Cxr * Cyr;
    const double q2 = Crr * (Cxx - Cyy) - Cxr * Cxr + Cyr * Cyr;
    double phi = 0.5 * atan2(2.0 * q1, q2);
    const double sp = sin(phi), cp = cos(phi);
    const double khat = (-sp * Cxr + cp * Cyr) / Crr;
    const double delta = (-mx * sp + my * cp) - khat * mr;
    const double D = 1.0 - 4.0 * delta * khat;
    if (!(D > 0.0))
        return 2;
    const double sq = sqrt(D);
    double kappa = 2.0 * khat / sq;
    double d0 = 2.0 * delta / (1.0 + sq);
    double see = 0.0;
    for (uint32_t q = 0; q < n; ++q) {
        double xv = (double)x[idx[q]], yv = (double)y[idx[q]];
        double u = xv - mx, v = yv - my, w = (xv * xv + yv * yv) - mr;
        double eps = khat * w - (-sp * u + cp * v);
        see += eps * eps;
    }
    double rms = sqrt((see / dn) / D);
    if (mx * cp + my * sp < 0.0) { /* backward representation: report the forward one */
        phi = phi >= 0.0 ? phi - ORACLE_PI : phi + ORACLE_PI;
        d0 = -d0;
        kappa = -kappa;
    }
    if (!(isfinite(kappa) && isfinite(d0) && isfinite(rms)))
        return 2;
    out->kappa = kappa;
    out->phi0 = phi;
    out->d0 = d0;
    out->rms = rms;
    return 0;
}

/* E4 for all peaks of a CSR. */
void oracle_fit_all(const float *x, const float *y, const uint64_t *hit_offset, const uint32_t *hit_index,
                    uint64_t n_peaks, oracle_fit *fit, int32_t *status)
{
#pragma omp parallel for schedule(dynamic, 256)
    for (uint64_t p = 0; p < n_peaks; ++p)
        status[p] = oracle_fit_one(x, y, hit_index + hit_offset[p], (uint32_t)(hit_offset[p + 1] - hit_offset[p]),
                                   &fit[p]);
}

static int better(int la, double ra, uint64_t ia, int lb, double rb, uint64_t ib)
{ /* is candidate a better than candidate b? */
    if (la != lb)
        return la > lb;
    if (ra != rb)
        return ra < rb;
    return ia < ib;
}

/* E5: flags[p] = 0 not selected, 1 selected and kept, 2 selected but a duplicate. */
void oracle_select_dedup(const uint64_t *hit_offset, const uint32_t *hit_index, const uint32_t *peak_mask,
                         uint64_t n_peaks, uint32_t n_hits, const oracle_fit *fit, const int32_t *status,
                         double rms_max, uint32_t min_shared, uint8_t *flags)
{
    /* inverted index: hit -> selected candidates holding it */
    uint64_t *cnt = calloc((size_t)n_hits + 1, sizeof(uint64_t));
    for (uint64_t p = 0; p < n_peaks; ++p) {
        flags[p] = (status[p] == 0 && fit[p].rms <= rms_max) ? 1 : 0;
        if (flags[p])
            for (uint64_t q = hit_offset[p]; q < hit_offset[p + 1]; ++q)
                cnt[hit_index[q] + 1]++;
    }
    for (uint32_t h = 0; h < n_hits; ++h)
        cnt[h + 1] += cnt[h];
    uint64_t *cur = malloc(sizeof(uint64_t) * ((size_t)n_hits + 1));
    memcpy(cur, cnt, sizeof(uint64_t) * ((size_t)n_hits + 1));
    uint32_t *inv = malloc(sizeof(uint32_t) * (cnt[n_hits] ? cnt[n_hits] : 1));
    for (uint64_t p = 0; p < n_peaks; ++p)
        if (flags[p])
            for (uint64_t q = hit_offset[p]; q < hit_offset[p + 1]; ++q)
                inv[cur[hit_index[q]]++] = (uint32_t)p;
    uint32_t *shared = calloc(n_peaks ? n_peaks : 1, sizeof(uint32_t));
    uint32_t *touched = malloc(sizeof(uint32_t) * (n_peaks ? n_peaks : 1));
    for (uint64_t p = 0; p < n_peaks; ++p) {
        if (!flags[p])
            continue;
        uint64_t nt = 0;
        for (uint64_t q = hit_offset[p]; q < hit_offset[p + 1]; ++q) {
            uint32_t h = hit_index[q];
            for (uint64_t z = cnt[h]; z < cnt[h + 1]; ++z) {
                uint32_t o = inv[z];
                if (o == p)
                    continue;
                if (shared[o]++ == 0)
                    touched[nt++] = o;
            }
        }
        int dup = 0;
        for (uint64_t z = 0; z < nt; ++z) {
            uint32_t o = touched[z];
            if (shared[o] >= min_shared &&
                better(__builtin_popcount(peak_mask[o]), fit[o].rms, o, __builtin_popcount(peak_mask[p]),
                       fit[p].rms, p))
                dup = 1;
            shared[o] = 0;
        }
        if (dup)
            flags[p] = 3; /* marked; turned into 2 below so that later candidates still see it as selected */
    }
    for (uint64_t p = 0; p < n_peaks; ++p)
        if (flags[p] == 3)
            flags[p] = 2;
    free(cnt); free(cur); free(inv); free(shared); free(touched);
}
