"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

The paper defines the Hough transform for tracking in words (section 7;
PAPER.md:122 Fig. 3 "each hit results in a sinusoidal curve in the parameter space ...
local maxima"; PAPER.md:138 the 2-parameter curved case through the interaction point);
BASELINE.json north_star fixes the closed form, the mask vote and the peak rule.  None
of these tests re-types the oracle's formula: each one checks it against geometry in
fp64, a textbook special case, an invariant, or a brute force written differently
(SURVEY.md section 8(c) C).
"""
import math

import numpy as np
import pytest

from paper_1305_4855_b200 import synth

RADII = synth.LAYER_RADII_CM


def tiny_grid(n_phi=8, n_d0=4, n_kappa=8, L_min=2, **kw):
    return synth.Grid(n_phi=n_phi, n_d0=n_d0, n_kappa=n_kappa, L_min=L_min, **kw)


def centres(grid):
    phic = grid.phi_min + (np.arange(grid.n_phi) + 0.5) * (grid.phi_max - grid.phi_min) / grid.n_phi
    d0c = grid.d0_min + (np.arange(grid.n_d0) + 0.5) * (grid.d0_max - grid.d0_min) / grid.n_d0
    return phic, d0c


def signed_distance(X, phi0, d0, kappa):
    """fp64 signed distance (towards n) from point X to the track (phi0, d0, kappa):
    a circle of radius 1/|kappa| centred at (d0 + 1/kappa) n, n = (-sin phi0, cos phi0);
    the straight line through d0*n with direction (cos phi0, sin phi0) when kappa = 0.
    This is the point-on-circle test -- it never forms 2(s-d0)/(r^2-2 d0 s+d0^2)."""
    n = np.array([-math.sin(phi0), math.cos(phi0)])
    if kappa == 0.0:
        return float(np.dot(X, n) - d0)
    centre = (d0 + 1.0 / kappa) * n
    dist = math.hypot(X[0] - centre[0], X[1] - centre[1])
    return math.copysign(1.0, kappa) * (1.0 / abs(kappa) - dist)


def random_hits(rng, n, n_layers=10, rmax=80.0):
    r = rng.uniform(3.0, rmax, n)
    phi = rng.uniform(-math.pi, math.pi, n)
    x = (r * np.cos(phi)).astype(np.float32)
    y = (r * np.sin(phi)).astype(np.float32)
    layer = rng.integers(0, n_layers, n).astype(np.int32)
    return x, y, layer


# ---------------------------------------------------------------- closed form (A3/A4)

@pytest.mark.parametrize("seed", [0, 1, 2])
def test_vote_bin_is_where_the_circle_through_the_hit_lies(oracle, seed):
    """Point-on-circle pin: for every (hit, i, j) the signed distance from the hit to the
    track (phi0_i, d0_j, kappa) changes sign across exactly the voted kappa bin, and does
    not change sign inside [kappa_min, kappa_max) when no vote is cast."""
    rng = np.random.default_rng(seed)
    grid = tiny_grid(n_phi=12, n_d0=5, n_kappa=9)
    x, y, layer = random_hits(rng, 40)
    phic, d0c = centres(grid)
    edges = np.linspace(grid.kappa_min, grid.kappa_max, grid.n_kappa + 1)
    checked = voted = 0
    for h in range(len(x)):
        X = np.array([float(x[h]), float(y[h])])
        for i in range(grid.n_phi):
            for j in range(grid.n_d0):
                kap32, k = oracle.vote_one(grid, float(x[h]), float(y[h]), i, j)
                sd = [signed_distance(X, phic[i], d0c[j], e) for e in edges]
                # skip decisions within 1e-5 of an edge (fp32 vs fp64, table rounding)
                if min(abs(kap32 - e) for e in edges) < 1e-5 * grid.kappa_max:
                    continue
                checked += 1
                if k >= 0:
                    voted += 1
                    assert sd[k] * sd[k + 1] < 0, (h, i, j, k, kap32)
                    for kk in range(grid.n_kappa):
                        if kk != k:
                            assert sd[kk] * sd[kk + 1] > 0
                else:
                    assert sd[0] * sd[-1] > 0, (h, i, j, kap32)
    assert checked > 2000 and voted > 100


def test_d0_zero_reduces_to_through_origin_form(oracle):
    """Textbook 2-parameter case (tracks through the interaction point):
    a circle through the origin with direction phi0 passes through (r, phi) iff
    kappa = 2 sin(phi - phi0) / r."""
    grid = synth.Grid(n_phi=64, n_d0=1, n_kappa=128, L_min=3, d0_min=0.0, d0_max=0.0)
    phic, _ = centres(grid)
    rng = np.random.default_rng(5)
    for _ in range(300):
        r = rng.uniform(4.0, 80.0)
        phi = rng.uniform(-math.pi, math.pi)
        i = int(rng.integers(0, grid.n_phi))
        x32, y32 = np.float32(r * math.cos(phi)), np.float32(r * math.sin(phi))
        kap32, k = oracle.vote_one(grid, float(x32), float(y32), i, 0)
        expect = 2.0 * math.sin(phi - phic[i]) / r
        assert abs(kap32 - expect) <= 2e-6 * max(abs(expect), 1e-3), (r, phi, i)
        if grid.kappa_min + 1e-7 < expect < grid.kappa_max - 1e-7:
            q = (expect - grid.kappa_min) / (grid.kappa_max - grid.kappa_min) * grid.n_kappa
            if abs(q - round(q)) > 1e-2:
                assert k == int(q)
        elif expect < grid.kappa_min - 1e-7 or expect > grid.kappa_max + 1e-7:
            assert k == -1


def test_kappa_zero_reduces_to_straight_line_hough(oracle):
    """kappa -> 0 is the straight-line transform of PAPER.md:122 (Fig. 3): points on the
    line {d0 n + t (cos phi0, sin phi0)} have kappa = 0 at (phi0, d0) and therefore vote
    into the bin that contains 0 (n_kappa odd: the middle bin)."""
    grid = synth.Grid(n_phi=32, n_d0=9, n_kappa=65, L_min=3)
    phic, d0c = centres(grid)
    for i, j in [(3, 0), (17, 4), (30, 8)]:
        n = np.array([-math.sin(phic[i]), math.cos(phic[i])])
        u = np.array([math.cos(phic[i]), math.sin(phic[i])])
        for t in (5.0, 12.5, 33.0, 71.0):
            X = d0c[j] * n + t * u
            kap32, k = oracle.vote_one(grid, float(np.float32(X[0])), float(np.float32(X[1])), i, j)
            assert abs(kap32) < 2e-6
            assert k == grid.n_kappa // 2


def test_tables_are_fp64_centres_rounded_once(oracle):
    grid = synth.WORKLOADS["displaced3d"].grid
    sn, cs, d0c, twod0, d0sq, ks = oracle.tables(grid)
    phic, dc = centres(grid)
    # libm vs numpy sin may differ in the last fp64 bit: allow one fp32 ulp
    assert np.all(np.abs(sn - np.sin(phic)) <= np.spacing(np.abs(sn)))
    assert np.all(np.abs(cs - np.cos(phic)) <= np.spacing(np.abs(cs)))
    assert np.array_equal(d0c, dc.astype(np.float32))
    assert np.array_equal(twod0, np.float32(2.0) * d0c)
    assert np.array_equal(d0sq, d0c * d0c)
    assert ks[0] == np.float32(grid.kappa_min) and ks[1] == np.float32(grid.kappa_max)
    assert ks[2] == np.float32(grid.n_kappa / (grid.kappa_max - grid.kappa_min))
    # bin centres of a symmetric range are antisymmetric: catches an off-by-half in A1
    assert np.array_equal(d0c, -d0c[::-1])
    assert abs(phic[0] + math.pi - math.pi / grid.n_phi) < 1e-12


# ------------------------------------------------- generator <-> transform consistency

@pytest.mark.parametrize("gridname,i,j,kappa", [
    ("prompt2d", 37, 0, 0.0031), ("prompt2d", 200, 0, -0.0052),
    ("displaced3d", 100, 40, 0.0027), ("displaced3d", 700, 12, -0.0041),
    ("displaced3d", 5, 31, 0.0008),
])
def test_single_noiseless_track_peaks_in_its_own_bin_and_in_its_mirror(oracle, gridname, i, j, kappa):
    """north_star: 'a single noiseless generated track must peak in its own (phi0, d0,
    kappa) bin or an adjacent one' (phi0, d0 at bin centres: reading B9); the mirror
    description (phi0 + pi, -d0, -kappa) of the same circle does too (reading B8)."""
    grid = synth.WORKLOADS[gridname].grid
    x, y, layer = synth.single_track_event(grid, i, j, kappa)
    n_hits = len(x)
    assert n_hits >= 8
    ci = np.array([i, (i + grid.n_phi // 2) % grid.n_phi], np.int32)
    cj = np.array([j, grid.n_d0 - 1 - j], np.int32)
    rows, _ = oracle.vote_cells(grid, x, y, layer, ci, cj)
    full = sum(1 << int(l) for l in layer)
    kbin = (kappa - grid.kappa_min) / (grid.kappa_max - grid.kappa_min) * grid.n_kappa
    for row, kb in ((rows[0], kbin), (rows[1], grid.n_kappa - kbin)):
        k0 = int(kb)
        near = [k for k in (k0 - 1, k0, k0 + 1) if 0 <= k < grid.n_kappa]
        got = 0
        for k in near:
            got |= int(row[k])
        assert got == full                       # every layer votes within +-1 bin
        assert max(bin(int(row[k])).count("1") for k in near) >= n_hits - 2
        others = [int(row[k]) for k in range(grid.n_kappa) if k not in near]
        assert all(v == 0 for v in others)       # one hit -> one kappa per cell


def test_single_track_is_found_as_a_peak_with_all_its_hits(oracle):
    grid = synth.Grid(n_phi=64, n_d0=16, n_kappa=64, L_min=9)
    i, j, kappa = 21, 9, 0.0033
    x, y, layer = synth.single_track_event(grid, i, j, kappa)
    res = oracle.run(grid, x, y, layer)
    assert res["n_peaks"] >= 2                   # the track and its mirror
    bins = res["peak_bin"].astype(np.int64)
    pi, pj, pk = bins // (grid.n_d0 * grid.n_kappa), (bins // grid.n_kappa) % grid.n_d0, bins % grid.n_kappa
    k_true = int((kappa - grid.kappa_min) / (grid.kappa_max - grid.kappa_min) * grid.n_kappa)
    own = [p for p in range(len(bins)) if pi[p] == i and pj[p] == j and abs(pk[p] - k_true) <= 1]
    mir = [p for p in range(len(bins)) if pi[p] == (i + 32) % 64 and pj[p] == 15 - j
           and abs(pk[p] - (63 - k_true)) <= 1]
    assert own and mir
    p = own[0]
    lst = res["hit_index"][int(res["hit_offset"][p]):int(res["hit_offset"][p + 1])]
    assert len(lst) >= grid.L_min and len(set(lst.tolist())) == len(lst)


# ------------------------------------------------------------------------- vote count

def fp64_votes(grid, x, y):
    """In-range solutions counted on the host in fp64 with numpy (vectorised, written
    from the circle equation kappa |X - P0|^2 = 2 (X - P0).n); returns (k or -1, margin
    = distance of the decision from the nearest bin edge in units of bins)."""
    phic, d0c = centres(grid)
    X = np.stack([x.astype(np.float64), y.astype(np.float64)], 1)           # [h, 2]
    n = np.stack([-np.sin(phic), np.cos(phic)], 1)                         # [i, 2]
    P0 = d0c[None, :, None] * n[:, None, :]                                # [i, j, 2]
    D = X[:, None, None, :] - P0[None]                                     # [h, i, j, 2]
    proj = np.einsum("hijc,ic->hij", D, n)
    kap = 2.0 * proj / np.einsum("hijc,hijc->hij", D, D)
    q = (kap - grid.kappa_min) / (grid.kappa_max - grid.kappa_min) * grid.n_kappa
    k = np.floor(q).astype(np.int64)
    inr = (q >= 0) & (q < grid.n_kappa)
    margin = np.abs(q - np.round(q))
    return np.where(inr, k, -1), margin


@pytest.mark.parametrize("seed", [3, 4])
def test_vote_count_equals_host_counted_in_range_solutions(oracle, seed):
    """north_star: 'total votes must equal the host-counted in-range kappa solutions'."""
    rng = np.random.default_rng(seed)
    grid = tiny_grid(n_phi=24, n_d0=6, n_kappa=16)
    x, y, layer = random_hits(rng, 60)
    acc, n_votes, n_bad = oracle.vote(grid, x, y, layer)
    k64, margin = fp64_votes(grid, x, y)
    sure = margin > 2e-4
    lo = int(np.count_nonzero((k64 >= 0) & sure))
    hi = lo + int(np.count_nonzero(~sure))
    assert n_bad == 0 and lo <= n_votes <= hi and hi - lo < 20
    pc = sum(bin(int(v)).count("1") for v in acc.reshape(-1))
    assert pc <= n_votes <= len(x) * grid.n_phi * grid.n_d0
    # and the masks themselves, where fp64 is sure of the bin
    ref = np.zeros_like(acc)
    unsure = np.zeros(acc.shape, bool)
    for h in range(len(x)):
        for i in range(grid.n_phi):
            for j in range(grid.n_d0):
                k = k64[h, i, j]
                if not sure[h, i, j]:
                    unsure[i, j, :] = True
                elif k >= 0:
                    ref[i, j, k] |= np.uint32(1 << int(layer[h]))
    assert np.array_equal(acc[~unsure], ref[~unsure])
    assert np.count_nonzero(~unsure) > 0.8 * acc.size


def test_popcount_sum_equals_votes_for_a_single_track(oracle):
    grid = synth.Grid(n_phi=32, n_d0=8, n_kappa=32, L_min=5)
    x, y, layer = synth.single_track_event(grid, 11, 3, -0.004)
    acc, n_votes, _ = oracle.vote(grid, x, y, layer)
    assert sum(bin(int(v)).count("1") for v in acc.reshape(-1)) == n_votes


def test_vote_cells_equals_the_same_rows_of_the_whole_vote(oracle):
    """oracle_vote_cells (used where only part of a large grid is checked) must give exactly
    the rows oracle_vote gives, and its vote count the votes of those rows; listing every
    cell reproduces the whole accumulator and n_votes."""
    rng = np.random.default_rng(17)
    grid = synth.Grid(n_phi=24, n_d0=7, n_kappa=32, L_min=2)
    x, y, layer = random_hits(rng, 400)
    layer[::13] = -1                              # bad hits are skipped by both
    acc, n_votes, _ = oracle.vote(grid, x, y, layer)
    ci = rng.integers(0, grid.n_phi, 60)
    cj = rng.integers(0, grid.n_d0, 60)
    rows, nv = oracle.vote_cells(grid, x, y, layer, ci, cj)
    assert np.array_equal(rows, acc[ci, cj, :])
    # the same cells once more with single-hit events: votes in the listed cells add up
    per_hit = sum(oracle.vote_cells(grid, x[h:h + 1], y[h:h + 1], layer[h:h + 1], ci, cj)[1]
                  for h in range(len(x)))
    assert per_hit == nv
    ii, jj = np.meshgrid(np.arange(grid.n_phi), np.arange(grid.n_d0), indexing="ij")
    rows_all, nv_all = oracle.vote_cells(grid, x, y, layer, ii.ravel(), jj.ravel())
    assert np.array_equal(rows_all.reshape(acc.shape), acc) and nv_all == n_votes


def test_finite_coordinates_whose_squares_overflow_still_vote(oracle):
    """r2 = x*x + y*y = inf for |x| > ~1.8e19: den = inf, kappa = +-0, which is inside a kappa
    range that contains 0 (reading B4: no special case).  Checked against the definition: the
    vote of such a hit is bin(0) in every cell, for any finite coordinate up to FLT_MAX."""
    grid = synth.Grid(n_phi=16, n_d0=4, n_kappa=32, L_min=1)
    k0 = int((0.0 - grid.kappa_min) * (grid.n_kappa / (grid.kappa_max - grid.kappa_min)))
    for xv, yv in ((3.2e38, 1.0), (2.0, -3.3e38), (3.0e19, 0.0), (3.4028234e38, -3.4028234e38)):
        x = np.array([xv], np.float32)
        y = np.array([yv], np.float32)
        acc, n_votes, n_bad = oracle.vote(grid, x, y, np.array([3], np.int32))
        voted = acc[:, :, k0] == 8
        # every cell whose s is finite votes into the bin of kappa = 0; a cell whose s overflows
        # to +-inf (or whose 2*d0*s does) has num/den = inf/inf = NaN and casts no vote
        assert n_votes == int(voted.sum()) > 0 and n_bad == 0
        assert int((acc != 0).sum()) == n_votes


def test_bad_and_non_finite_hits_cast_no_vote(oracle):
    grid = tiny_grid()
    rng = np.random.default_rng(9)
    x, y, layer = random_hits(rng, 20)
    acc0, nv0, _ = oracle.vote(grid, x, y, layer)
    x2 = np.concatenate([x, np.float32([1.0, 2.0, np.nan, np.inf, 5.0])])
    y2 = np.concatenate([y, np.float32([1.0, 2.0, 1.0, 1.0, np.nan])])
    l2 = np.concatenate([layer, np.int32([-1, 10, 0, 1, 2])])
    acc1, nv1, nbad = oracle.vote(grid, x2, y2, l2)
    assert nbad == 2 and nv1 == nv0 and np.array_equal(acc0, acc1)
    acc2, nv2, _ = oracle.vote(grid, x[:0], y[:0], layer[:0])
    assert nv2 == 0 and not acc2.any()


# -------------------------------------------------------------------- peak rule (A6)

def brute_peaks(grid, acc):
    """27-neighbour rule written independently with a (popcount, -lin) ranking: a bin is a
    peak iff popcount >= L_min and its rank beats every distinct existing neighbour."""
    np_, nd, nk = grid.n_phi, grid.n_d0, grid.n_kappa
    a = np.asarray(acc, np.uint32).reshape(np_, nd, nk)
    pc = np.vectorize(lambda v: bin(int(v)).count("1"))(a)
    lin = np.arange(np_ * nd * nk).reshape(np_, nd, nk)
    out = []
    for i in range(np_):
        for j in range(nd):
            for k in range(nk):
                if pc[i, j, k] < grid.L_min:
                    continue
                me = (pc[i, j, k], -lin[i, j, k])
                nb = set()
                for di in (-1, 0, 1):
                    for dj in (-1, 0, 1):
                        for dk in (-1, 0, 1):
                            ii, jj, kk = i + di, j + dj, k + dk
                            if grid.phi_wrap:
                                ii %= np_
                            if 0 <= ii < np_ and 0 <= jj < nd and 0 <= kk < nk:
                                nb.add((ii, jj, kk))
                nb.discard((i, j, k))
                if all(me > (pc[n], -lin[n]) for n in nb):
                    out.append(lin[i, j, k])
    return np.asarray(out, np.uint32)


def rand_acc(rng, grid, density):
    bits = rng.random((grid.n_bins, 10)) < density
    return (bits * (1 << np.arange(10))).sum(1).astype(np.uint32)


@pytest.mark.parametrize("shape,wrap,L_min,density", [
    ((6, 5, 7), 1, 3, 0.4), ((6, 5, 7), 0, 3, 0.4), ((9, 1, 12), 1, 2, 0.3),
    ((9, 1, 12), 0, 5, 0.6), ((3, 3, 3), 1, 1, 0.5), ((4, 2, 2), 1, 1, 0.2),
    ((2, 3, 4), 1, 1, 0.5), ((1, 4, 5), 1, 1, 0.5), ((5, 6, 1), 0, 4, 0.5),
])
def test_peak_rule_against_brute_force(oracle, shape, wrap, L_min, density):
    rng = np.random.default_rng(hash(shape) % 1000 + wrap)
    grid = synth.Grid(n_phi=shape[0], n_d0=shape[1], n_kappa=shape[2], L_min=L_min, phi_wrap=wrap)
    for _ in range(6):
        acc = rand_acc(rng, grid, density)
        pb, pm, n = oracle.peaks(grid, acc)
        ref = brute_peaks(grid, acc)
        assert n == len(ref) and np.array_equal(pb, ref)
        assert np.array_equal(pm, acc[pb])
        assert np.all(np.diff(pb.astype(np.int64)) > 0)          # ascending lin (A7)


def test_peak_rule_plateaus_edges_and_threshold(oracle):
    g = synth.Grid(n_phi=5, n_d0=4, n_kappa=6, L_min=3, phi_wrap=1)
    acc = np.full(g.n_bins, 0b111, np.uint32)                    # all equal
    pb, _, n = oracle.peaks(g, acc)
    assert n == 1 and pb[0] == 0                                 # ties -> lowest lin only
    acc = np.zeros(g.n_bins, np.uint32)
    acc[[7, 8, 9]] = 0b1111                                      # 1-D plateau along kappa
    pb, _, _ = oracle.peaks(g, acc)
    assert pb.tolist() == [7]
    acc = np.zeros(g.n_bins, np.uint32)
    acc[0] = 0b111
    acc[g.n_bins - 1] = 0b111       # (4,3,5): a phi-wrap neighbour of (0,?,?) only via i
    pb, _, _ = oracle.peaks(g, acc)
    assert pb.tolist() == [0, g.n_bins - 1]                      # j, k never wrap
    acc = np.zeros(g.n_bins, np.uint32)
    lin = lambda i, j, k: (i * g.n_d0 + j) * g.n_kappa + k
    acc[lin(0, 1, 2)] = 0b111
    acc[lin(4, 1, 2)] = 0b111                                    # tie across the phi seam
    assert oracle.peaks(g, acc)[0].tolist() == [lin(0, 1, 2)]    # wrapped nb keeps its lin
    g0 = synth.Grid(n_phi=5, n_d0=4, n_kappa=6, L_min=3, phi_wrap=0)
    assert oracle.peaks(g0, acc)[0].tolist() == [lin(0, 1, 2), lin(4, 1, 2)]
    acc[lin(4, 1, 2)] = 0b11                                     # below L_min
    assert oracle.peaks(g, acc)[0].tolist() == [lin(0, 1, 2)]
    acc[lin(0, 1, 2)] = 0b1011                                   # popcount, not value
    acc[lin(0, 1, 3)] = 0b110000
    assert oracle.peaks(g, acc)[0].tolist() == [lin(0, 1, 2)]
    pb, pm, n = oracle.peaks(g, np.full(g.n_bins, 0b111, np.uint32), cap=0)
    assert n == 1 and len(pb) == 0                               # true count despite cap


# --------------------------------------------------------------------- hit lists (A7)

def test_hit_list_invariants_and_whole_pipeline_brute_force(oracle):
    rng = np.random.default_rng(11)
    grid = tiny_grid(n_phi=16, n_d0=4, n_kappa=8, L_min=2)
    x, y, layer = random_hits(rng, 50)
    res = oracle.run(grid, x, y, layer)
    acc = res["acc"].reshape(-1)
    off, idx = res["hit_offset"].astype(np.int64), res["hit_index"]
    assert res["n_peaks"] == len(res["peak_bin"]) > 3
    assert off[0] == 0 and off[-1] == res["n_hit_entries"] == len(idx)
    k64, margin = fp64_votes(grid, x, y)
    for p, b in enumerate(res["peak_bin"].astype(np.int64)):
        lst = idx[off[p]:off[p + 1]].astype(np.int64)
        assert np.all(np.diff(lst) > 0)                          # strictly ascending h
        m = 0
        for h in lst:
            m |= 1 << int(layer[h])
        assert m == int(acc[b]) == int(res["peak_mask"][p])      # OR of bits == mask
        assert len(lst) >= bin(m).count("1")
        i, j, k = b // (grid.n_d0 * grid.n_kappa), (b // grid.n_kappa) % grid.n_d0, b % grid.n_kappa
        sure = margin[:, i, j] > 2e-4                            # fp64 brute force of the list
        want = set(np.nonzero((k64[:, i, j] == k) & sure)[0].tolist())
        maybe = set(np.nonzero(~sure)[0].tolist())
        assert want <= set(lst.tolist()) <= want | maybe
    # sum of list lengths over ALL bins == n_votes (treat every non-empty bin as a peak)
    allbins = np.nonzero(acc)[0].astype(np.uint32)
    off2, idx2, tot2 = oracle.hitlists(grid, x, y, layer, allbins)
    assert tot2 == res["n_votes"] == len(idx2)
    off3, idx3, tot3 = oracle.hitlists(grid, x, y, layer, allbins, cap_hits=10)
    assert tot3 == tot2 and len(idx3) == 10 and np.array_equal(idx3, idx2[:10])
    assert np.array_equal(off3, off2)


def test_cellwise_hit_lists_equal_the_peakwise_ones(oracle):
    """oracle_hitlists_cells (one vote pass over the cells that hold a peak) against oracle_hitlists (one
    pass per peak), whose own pins are above: equal CSR on random grids with bad / non-finite hits, on the
    prompt2d and displaced3d events, with a cap that cuts a list, on the peak subsets a truncated GPU run
    reports, with no peaks and no hits; and its total over EVERY non-empty bin is the vote count."""
    rng = np.random.default_rng(12)
    cases = []
    for shape, n in [((16, 4, 8), 50), ((9, 1, 32), 200), ((24, 7, 64), 900), ((5, 3, 16), 1)]:
        d0 = dict(d0_min=0.0, d0_max=0.0) if shape[1] == 1 else {}
        grid = tiny_grid(n_phi=shape[0], n_d0=shape[1], n_kappa=shape[2], L_min=2, **d0)
        x, y, layer = random_hits(rng, n)
        if n >= 50:
            layer[::17] = 12                                    # bad layers cast no vote
            x[3], y[5] = np.nan, np.inf
        cases.append((grid, x, y, layer))
    for name, seed in (("prompt2d", 0), ("displaced3d", 1)):
        w = synth.WORKLOADS[name]
        cases.append((w.grid,) + tuple(synth.generate_event(w.event, seed)[:3]))
    for grid, x, y, layer in cases:
        acc, n_votes, _ = oracle.vote(grid, x, y, layer)
        pb, _pm, n_peaks = oracle.peaks(grid, acc)
        for bins in (pb, pb[: len(pb) // 2], pb[1::3], pb[:0]):
            off1, idx1, tot1 = oracle.hitlists(grid, x, y, layer, bins)
            off2, idx2, tot2 = oracle.hitlists_cells(grid, x, y, layer, bins)
            assert tot1 == tot2 and np.array_equal(off1, off2) and np.array_equal(idx1, idx2)
        if len(pb) > 2:
            offf, idxf, totf = oracle.hitlists(grid, x, y, layer, pb)
            cap = int(offf[len(pb) // 2]) + 1                   # cuts inside a list
            offc, idxc, totc = oracle.hitlists_cells(grid, x, y, layer, pb, cap_hits=cap)
            assert totc == totf and np.array_equal(offc, offf) and np.array_equal(idxc, idxf[:cap])
        if grid.n_bins <= 1 << 16:
            allbins = np.nonzero(acc.reshape(-1))[0].astype(np.uint32)
            _off, idx, tot = oracle.hitlists_cells(grid, x, y, layer, allbins)
            assert tot == n_votes == len(idx)
    g = cases[0][0]
    z = np.zeros(0, np.float32)
    off, idx, tot = oracle.hitlists_cells(g, z, z, np.zeros(0, np.int32), np.array([3, 40], np.uint32))
    assert tot == 0 and off.tolist() == [0, 0, 0] and len(idx) == 0


def test_oracle_is_deterministic_and_thread_count_independent(oracle):
    """OR of masks is order independent (the race remark of PAPER.md:126)."""
    w = synth.WORKLOADS["prompt2d"]
    x, y, layer, _ = synth.generate_event(w.event, 0)
    nt = oracle.num_threads()
    a = oracle.run(w.grid, x, y, layer)
    oracle.set_num_threads(1)
    b = oracle.run(w.grid, x, y, layer)
    oracle.set_num_threads(nt)
    for key in a:
        assert np.array_equal(a[key], b[key]), key
    perm = np.random.default_rng(1).permutation(len(x))
    c = oracle.run(w.grid, x[perm], y[perm], layer[perm])
    assert np.array_equal(a["acc"], c["acc"]) and a["n_votes"] == c["n_votes"]
    assert np.array_equal(a["peak_bin"], c["peak_bin"])
