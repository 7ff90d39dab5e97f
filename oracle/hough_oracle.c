/*
 * hough_oracle.c -- CPU ORACLE for the Hough-transform track finder.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or constant generator with the CUDA path under
 * paper_1305_4855_b200/csrc/ and neither includes the other.
 *
 * What it is: the method written out step by step, in the order and notation of
 * SURVEY.md section 8(c) "A. Algorithm" (A1..A7), which restates BASELINE.json
 * north_star.  The paper itself (section 7, Fig. 3,
 * PAPER.md:138 section 8) defines the Hough transform for tracking only in words:
 * every hit maps to a curve in the track-parameter space, the curves of all hits are
 * accumulated, and local maxima of the accumulator are the track candidates.
 * north_star fixes the concrete form: parameters (phi0, d0, kappa), the closed form
 *     kappa = 2 (s - d0) / (r^2 - 2 d0 s + d0^2),   s = -x sin(phi0) + y cos(phi0),
 * evaluated at every (phi0, d0) bin centre, a uint32 layer-mask accumulator, the
 * popcount >= L_min / 3x3x3 local-maximum peak rule with ties to the lower linear
 * index, and a sorted hit list per peak.
 *
 * The method is a discretised voting heuristic, so the result has no definition other
 * than the algorithm itself: every arithmetic operation below is one IEEE-754 binary32
 * operation rounded to nearest-even, in the fixed order A3/A4, with no fused
 * multiply-add.  Build with:  gcc -O2 -ffp-contract=off -fno-fast-math  (see build.py).
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): fp64 point-on-circle geometry,
 * d0 = 0 and kappa -> 0 textbook reductions, single noiseless bin-centre track,
 * vote-count invariants, brute-force 27-neighbour peak rule, hit-list invariants
 * (oracle_hitlists_cells: equal to oracle_hitlists, and its total over every non-empty bin
 * equals n_votes).
 * PARITY UNPINNED: the paper's efficiency / purity numbers -- the
 * paper gives neither its peak rule nor its matching criterion, so they are not
 * reproduced here.
 *
 * Parallelism: `#pragma omp parallel for` over phi0 rows only (each thread owns whole
 * rows of the accumulator, so there is no race -- the paper's own CPU baseline is an
 * OpenMP Hough transform).  It is not tuned in any other way.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t n_layers;
    int32_t n_phi, n_d0, n_kappa;
    int32_t L_min;
    int32_t phi_wrap;
    double phi_min, phi_max;
    double d0_min, d0_max;
    double kappa_min, kappa_max;
} oracle_grid;

/* A1 -- tables: bin centres in fp64, one rounding to fp32. */
void oracle_tables(const oracle_grid *g, float *sn, float *cs, float *d0c, float *twod0,
                   float *d0sq, float *kscal /* klo, khi, inv_dk */)
{
    for (int i = 0; i < g->n_phi; ++i) {
        double phic = g->phi_min + ((double)i + 0.5) * (g->phi_max - g->phi_min) / (double)g->n_phi;
        sn[i] = (float)sin(phic);
        cs[i] = (float)cos(phic);
    }
    for (int j = 0; j < g->n_d0; ++j) {
        d0c[j] = (float)(g->d0_min + ((double)j + 0.5) * (g->d0_max - g->d0_min) / (double)g->n_d0);
        twod0[j] = 2.0f * d0c[j];
        d0sq[j] = d0c[j] * d0c[j];
    }
    kscal[0] = (float)g->kappa_min;
    kscal[1] = (float)g->kappa_max;
    kscal[2] = (float)((double)g->n_kappa / (g->kappa_max - g->kappa_min));
}

/* A3 + A4 for one (hit, i, j): returns the kappa bin voted into, or -1 for no vote. */
static int vote_bin(float x, float y, float r2, float sn, float cs, float d0c, float twod0,
                    float d0sq, float klo, float khi, float inv_dk, int n_kappa)
{
    float a = x * sn;
    float b = y * cs;
    float s = b - a;
    float e = s - d0c;
    float num = 2.0f * e;
    float t = twod0 * s;
    float u = r2 - t;
    float den = u + d0sq;
    float kappa = num / den;
    if (!((kappa >= klo) && (kappa < khi)))
        return -1;
    float qf = (kappa - klo) * inv_dk;
    int k = (int)qf;
    if (k > n_kappa - 1)
        k = n_kappa - 1;
    return k;
}

/* A2 -- per-hit quantities. layer outside [0, n_layers) => bad hit (bit 0, never votes). */
static void hit_prep(const oracle_grid *g, const float *x, const float *y, const int32_t *layer,
                     uint32_t n, float *r2, uint32_t *bit, uint32_t *n_bad)
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

/*
 * A3-A5 over the whole grid.  acc[(i*n_d0 + j)*n_kappa + k] |= bit_h.  The accumulator
 * is defined from scratch (zeroed here).  Returns n_votes (votes cast, bad hits excluded).
 */
uint64_t oracle_vote(const oracle_grid *g, const float *x, const float *y, const int32_t *layer,
                     uint32_t n, uint32_t *acc, uint32_t *n_bad_out)
{
    const int np = g->n_phi, nd = g->n_d0, nk = g->n_kappa;
    float *sn = malloc(sizeof(float) * np), *cs = malloc(sizeof(float) * np);
    float *d0c = malloc(sizeof(float) * nd), *twod0 = malloc(sizeof(float) * nd);
    float *d0sq = malloc(sizeof(float) * nd);
    float ks[3];
    oracle_tables(g, sn, cs, d0c, twod0, d0sq, ks);
    float *r2 = malloc(sizeof(float) * (n ? n : 1));
    uint32_t *bit = malloc(sizeof(uint32_t) * (n ? n : 1));
    hit_prep(g, x, y, layer, n, r2, bit, n_bad_out);
    memset(acc, 0, sizeof(uint32_t) * (size_t)np * nd * nk);
    uint64_t n_votes = 0;
#pragma omp parallel for schedule(static) reduction(+ : n_votes)
    for (int i = 0; i < np; ++i) {
        for (int j = 0; j < nd; ++j) {
            uint32_t *row = acc + ((size_t)i * nd + j) * nk;
            for (uint32_t h = 0; h < n; ++h) {
                if (!bit[h])
                    continue;
                int k = vote_bin(x[h], y[h], r2[h], sn[i], cs[i], d0c[j], twod0[j], d0sq[j],
                                 ks[0], ks[1], ks[2], nk);
                if (k >= 0) {
                    row[k] |= bit[h];
                    ++n_votes;
                }
            }
        }
    }
    free(sn); free(cs); free(d0c); free(twod0); free(d0sq); free(r2); free(bit);
    return n_votes;
}

/*
 * A3-A5 restricted to a list of cells (i, j): writes the n_kappa masks of each listed
 * cell to rows[c*n_kappa ..].  Used to check sampled rows of grids too large to
 * accumulate on the CPU in seconds.  Returns the votes cast in those cells.
 */
uint64_t oracle_vote_cells(const oracle_grid *g, const float *x, const float *y,
                           const int32_t *layer, uint32_t n, const int32_t *cell_i,
                           const int32_t *cell_j, uint32_t n_cells, uint32_t *rows)
{
    const int np = g->n_phi, nd = g->n_d0, nk = g->n_kappa;
    float *sn = malloc(sizeof(float) * np), *cs = malloc(sizeof(float) * np);
    float *d0c = malloc(sizeof(float) * nd), *twod0 = malloc(sizeof(float) * nd);
    float *d0sq = malloc(sizeof(float) * nd);
    float ks[3];
    oracle_tables(g, sn, cs, d0c, twod0, d0sq, ks);
    float *r2 = malloc(sizeof(float) * (n ? n : 1));
    uint32_t *bit = malloc(sizeof(uint32_t) * (n ? n : 1));
    uint32_t n_bad;
    hit_prep(g, x, y, layer, n, r2, bit, &n_bad);
    memset(rows, 0, sizeof(uint32_t) * (size_t)n_cells * nk);
    uint64_t n_votes = 0;
#pragma omp parallel for schedule(static) reduction(+ : n_votes)
    for (uint32_t c = 0; c < n_cells; ++c) {
        int i = cell_i[c], j = cell_j[c];
        uint32_t *row = rows + (size_t)c * nk;
        for (uint32_t h = 0; h < n; ++h) {
            if (!bit[h])
                continue;
            int k = vote_bin(x[h], y[h], r2[h], sn[i], cs[i], d0c[j], twod0[j], d0sq[j], ks[0],
                             ks[1], ks[2], nk);
            if (k >= 0) {
                row[k] |= bit[h];
                ++n_votes;
            }
        }
    }
    free(sn); free(cs); free(d0c); free(twod0); free(d0sq); free(r2); free(bit);
    return n_votes;
}

static inline int popc32(uint32_t v) { return __builtin_popcount(v); }

/* A6 for one bin. */
static int is_peak(const oracle_grid *g, const uint32_t *acc, int i, int j, int k)
{
    const int np = g->n_phi, nd = g->n_d0, nk = g->n_kappa;
    size_t lin = ((size_t)i * nd + j) * nk + k;
    int pc = popc32(acc[lin]);
    if (pc < g->L_min)
        return 0;
    for (int di = -1; di <= 1; ++di) {
        int ii = i + di;
        if (ii < 0 || ii >= np) {
            if (!g->phi_wrap)
                continue;
            ii = (ii + np) % np;
        }
        for (int dj = -1; dj <= 1; ++dj) {
            int jj = j + dj;
            if (jj < 0 || jj >= nd)
                continue;
            for (int dk = -1; dk <= 1; ++dk) {
                int kk = k + dk;
                if (kk < 0 || kk >= nk)
                    continue;
                if (di == 0 && dj == 0 && dk == 0)
                    continue;
                size_t ln = ((size_t)ii * nd + jj) * nk + kk;
                if (ln == lin)
                    continue; /* a wrapped neighbour that is the bin itself (n_phi < 3) */
                int pn = popc32(acc[ln]);
                if (pn > pc)
                    return 0;
                if (pn == pc && ln < lin)
                    return 0;
            }
        }
    }
    return 1;
}

/*
 * A6 + A7 (peak part): all peaks in ascending lin.  Writes at most cap records
 * (peak_bin, peak_mask) and returns the TRUE number of peaks.
 */
uint64_t oracle_peaks(const oracle_grid *g, const uint32_t *acc, uint32_t *peak_bin,
                      uint32_t *peak_mask, uint64_t cap)
{
    const int np = g->n_phi, nd = g->n_d0, nk = g->n_kappa;
    /* flags first (parallel over phi0 rows), then an ordered sweep */
    uint8_t *flag = malloc((size_t)np * nd * nk);
#pragma omp parallel for schedule(static)
    for (int i = 0; i < np; ++i)
        for (int j = 0; j < nd; ++j)
            for (int k = 0; k < nk; ++k)
                flag[((size_t)i * nd + j) * nk + k] = (uint8_t)is_peak(g, acc, i, j, k);
    uint64_t n_peaks = 0;
    size_t n_bins = (size_t)np * nd * nk;
    for (size_t lin = 0; lin < n_bins; ++lin) {
        if (flag[lin]) {
            if (n_peaks < cap) {
                peak_bin[n_peaks] = (uint32_t)lin;
                peak_mask[n_peaks] = acc[lin];
            }
            ++n_peaks;
        }
    }
    free(flag);
    return n_peaks;
}

/*
 * A7 (hit lists): for peak p at bin (i, j, k): H = { h : A3-A4 at (h, i, j) votes into k },
 * ascending h.  CSR: hit_offset[n_peaks + 1], hit_index[...].  Peaks must be given in
 * ascending lin (as oracle_peaks returns them).  Writes at most cap_hits indices (lists
 * are complete while they fit) and returns the TRUE total number of entries.
 */
uint64_t oracle_hitlists(const oracle_grid *g, const float *x, const float *y,
                         const int32_t *layer, uint32_t n, const uint32_t *peak_bin,
                         uint64_t n_peaks, uint64_t *hit_offset, uint32_t *hit_index,
                         uint64_t cap_hits)
{
    const int np = g->n_phi, nd = g->n_d0, nk = g->n_kappa;
    float *sn = malloc(sizeof(float) * np), *cs = malloc(sizeof(float) * np);
    float *d0c = malloc(sizeof(float) * nd), *twod0 = malloc(sizeof(float) * nd);
    float *d0sq = malloc(sizeof(float) * nd);
    float ks[3];
    oracle_tables(g, sn, cs, d0c, twod0, d0sq, ks);
    float *r2 = malloc(sizeof(float) * (n ? n : 1));
    uint32_t *bit = malloc(sizeof(uint32_t) * (n ? n : 1));
    uint32_t n_bad;
    hit_prep(g, x, y, layer, n, r2, bit, &n_bad);

    /* pass 1: list lengths */
    uint64_t *len = calloc(n_peaks + 1, sizeof(uint64_t));
#pragma omp parallel for schedule(dynamic, 1024)
    for (uint64_t p = 0; p < n_peaks; ++p) {
        uint32_t lin = peak_bin[p];
        int k = (int)(lin % (uint32_t)nk);
        int j = (int)((lin / (uint32_t)nk) % (uint32_t)nd);
        int i = (int)(lin / ((uint32_t)nk * (uint32_t)nd));
        uint64_t c = 0;
        for (uint32_t h = 0; h < n; ++h) {
            if (!bit[h])
                continue;
            if (vote_bin(x[h], y[h], r2[h], sn[i], cs[i], d0c[j], twod0[j], d0sq[j], ks[0], ks[1],
                         ks[2], nk) == k)
                ++c;
        }
        len[p] = c;
    }
    uint64_t total = 0;
    for (uint64_t p = 0; p < n_peaks; ++p) {
        hit_offset[p] = total;
        total += len[p];
    }
    hit_offset[n_peaks] = total;
    /* pass 2: fill, ascending h */
#pragma omp parallel for schedule(dynamic, 1024)
    for (uint64_t p = 0; p < n_peaks; ++p) {
        uint32_t lin = peak_bin[p];
        int k = (int)(lin % (uint32_t)nk);
        int j = (int)((lin / (uint32_t)nk) % (uint32_t)nd);
        int i = (int)(lin / ((uint32_t)nk * (uint32_t)nd));
        uint64_t w = hit_offset[p];
        for (uint32_t h = 0; h < n; ++h) {
            if (!bit[h])
                continue;
            if (vote_bin(x[h], y[h], r2[h], sn[i], cs[i], d0c[j], twod0[j], d0sq[j], ks[0], ks[1],
                         ks[2], nk) == k) {
                if (w < cap_hits)
                    hit_index[w] = h;
                ++w;
            }
        }
    }
    free(len);
    free(sn); free(cs); free(d0c); free(twod0); free(d0sq); free(r2); free(bit);
    return total;
}

/*
 * A7 once more, walked cell by cell instead of peak by peak -- the same definition and the same
 * outputs as oracle_hitlists, at the cost of ONE vote pass over the cells that hold a reported
 * peak instead of one pass per peak (which takes hours for the 4.9e5 peaks of a pile-up event).
 * Peaks come in ascending lin, so the peaks of one (i, j) cell are consecutive.  For every such
 * run of peaks: mark their kappa bins (which[k] = position in the run + 1), then go over the hits
 * in ascending h; a hit whose A3-A4 bin at (i, j) is marked belongs to that peak's list.  The
 * (peak, hit) pairs of a run wait in a buffer until all lengths, hence the offsets, are known.
 * No blocking and no index of the hits.
 * Pinned against oracle_hitlists and against n_votes (tests/test_oracle_pins.py).
 */
uint64_t oracle_hitlists_cells(const oracle_grid *g, const float *x, const float *y,
                               const int32_t *layer, uint32_t n, const uint32_t *peak_bin,
                               uint64_t n_peaks, uint64_t *hit_offset, uint32_t *hit_index,
                               uint64_t cap_hits)
{
    const int np = g->n_phi, nd = g->n_d0, nk = g->n_kappa;
    float *sn = malloc(sizeof(float) * np), *cs = malloc(sizeof(float) * np);
    float *d0c = malloc(sizeof(float) * nd), *twod0 = malloc(sizeof(float) * nd);
    float *d0sq = malloc(sizeof(float) * nd);
    float ks[3];
    oracle_tables(g, sn, cs, d0c, twod0, d0sq, ks);
    float *r2 = malloc(sizeof(float) * (n ? n : 1));
    uint32_t *bit = malloc(sizeof(uint32_t) * (n ? n : 1));
    uint32_t n_bad;
    hit_prep(g, x, y, layer, n, r2, bit, &n_bad);

    /* runs of peaks that share a cell: run r = peaks [run_first[r], run_first[r + 1]) */
    uint64_t *run_first = malloc(sizeof(uint64_t) * (n_peaks + 1));
    int64_t n_runs = 0;
    for (uint64_t p = 0; p < n_peaks; ++p)
        if (p == 0 || peak_bin[p] / (uint32_t)nk != peak_bin[p - 1] / (uint32_t)nk)
            run_first[n_runs++] = p;
    run_first[n_runs] = n_peaks;

    /* one pass over the hits per run: the (peak, hit) pairs of the run, in ascending h, kept until the
     * offsets are known (a hit votes at most once per cell, so a run has at most n pairs) */
    uint64_t *len = calloc(n_peaks + 1, sizeof(uint64_t));
    uint32_t **pair_peak = calloc(n_runs + 1, sizeof(uint32_t *)), **pair_hit = calloc(n_runs + 1, sizeof(uint32_t *));
    uint32_t *n_pairs = calloc(n_runs + 1, sizeof(uint32_t));
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t r = 0; r < n_runs; ++r) {
        const uint64_t a = run_first[r], b = run_first[r + 1];
        const uint32_t cell = peak_bin[a] / (uint32_t)nk;
        const int j = (int)(cell % (uint32_t)nd), i = (int)(cell / (uint32_t)nd);
        uint32_t *which = calloc(nk, sizeof(uint32_t));
        uint32_t *pp = malloc(sizeof(uint32_t) * (n ? n : 1)), *ph = malloc(sizeof(uint32_t) * (n ? n : 1));
        uint32_t c = 0;
        for (uint64_t p = a; p < b; ++p)
            which[peak_bin[p] % (uint32_t)nk] = (uint32_t)(p - a) + 1u;
        for (uint32_t h = 0; h < n; ++h) {
            if (!bit[h])
                continue;
            int k = vote_bin(x[h], y[h], r2[h], sn[i], cs[i], d0c[j], twod0[j], d0sq[j], ks[0],
                             ks[1], ks[2], nk);
            if (k < 0 || !which[k])
                continue;
            pp[c] = which[k] - 1u;
            ph[c] = h;
            ++c;
            ++len[a + which[k] - 1u];
        }
        n_pairs[r] = c;
        pair_peak[r] = realloc(pp, sizeof(uint32_t) * (c ? c : 1));
        pair_hit[r] = realloc(ph, sizeof(uint32_t) * (c ? c : 1));
        free(which);
    }
    uint64_t total = 0;
    for (uint64_t p = 0; p < n_peaks; ++p) {
        hit_offset[p] = total;
        total += len[p];
    }
    hit_offset[n_peaks] = total;
    /* fill: every run appends its pairs, still in ascending h, to its peaks' lists */
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t r = 0; r < n_runs; ++r) {
        const uint64_t a = run_first[r], b = run_first[r + 1];
        uint64_t *w = malloc(sizeof(uint64_t) * (b - a));
        for (uint64_t p = a; p < b; ++p)
            w[p - a] = hit_offset[p];
        for (uint32_t c = 0; c < n_pairs[r]; ++c) {
            uint64_t *dst = &w[pair_peak[r][c]];
            if (*dst < cap_hits)
                hit_index[*dst] = pair_hit[r][c];
            ++*dst;
        }
        free(w);
        free(pair_peak[r]);
        free(pair_hit[r]);
    }
    free(len); free(run_first); free(pair_peak); free(pair_hit); free(n_pairs);
    free(sn); free(cs); free(d0c); free(twod0); free(d0sq); free(r2); free(bit);
    return total;
}

/* kappa value (fp32, A3) and bin (A4) of one (hit, i, j) -- exposed for the pins. */
int oracle_vote_one(const oracle_grid *g, float x, float y, int i, int j, float *kappa_out)
{
    const int np = g->n_phi, nd = g->n_d0, nk = g->n_kappa;
    float *sn = malloc(sizeof(float) * np), *cs = malloc(sizeof(float) * np);
    float *d0c = malloc(sizeof(float) * nd), *twod0 = malloc(sizeof(float) * nd);
    float *d0sq = malloc(sizeof(float) * nd);
    float ks[3];
    oracle_tables(g, sn, cs, d0c, twod0, d0sq, ks);
    float p = x * x, q = y * y, r2 = p + q;
    float a = x * sn[i], b = y * cs[i], s = b - a;
    float e = s - d0c[j], num = 2.0f * e;
    float t = twod0[j] * s, u = r2 - t, den = u + d0sq[j];
    *kappa_out = num / den;
    int k = vote_bin(x, y, r2, sn[i], cs[i], d0c[j], twod0[j], d0sq[j], ks[0], ks[1], ks[2], nk);
    free(sn); free(cs); free(d0c); free(twod0); free(d0sq);
    return k;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int t)
{
#ifdef _OPENMP
    if (t > 0)
        omp_set_num_threads(t);
#else
    (void)t;
#endif
}
