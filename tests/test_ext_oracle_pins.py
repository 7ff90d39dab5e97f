"""Pins of oracle/hough_ext_oracle.c (the rows SURVEY.md 8(f) marks "next") -- CPU only.

The paper describes these steps in words (Fig. 3 straight-line transform,
PAPER.md:124 toy detector, PAPER.md:146 fit, PAPER.md:104 duplicate cleaning, PAPER.md:154-160
second transform over the crossings); DESIGN.md section 8 fixes the recipes E1..E5.  As in
test_oracle_pins.py no test re-types the oracle's formula: each checks it against fp64 geometry
written differently, a textbook special case, an invariant or a brute force.
"""
import dataclasses
import math

import numpy as np
import pytest

from paper_1305_4855_b200 import synth


def centres(lo, hi, n):
    return lo + (np.arange(n) + 0.5) * (hi - lo) / n


def lin_of(grid, i, j, k):
    return (i * grid.n_d0 + j) * grid.n_kappa + k


def signed_distance(X, phi0, d0, kappa):
    """fp64 signed distance (towards n) from X to the track (phi0, d0, kappa); the straight
    line through d0*n with direction (cos phi0, sin phi0) when kappa = 0 (same helper as
    test_oracle_pins.py: the point-on-circle test, never the closed form)."""
    n = np.array([-math.sin(phi0), math.cos(phi0)])
    if kappa == 0.0:
        return float(np.dot(X, n) - d0)
    centre = (d0 + 1.0 / kappa) * n
    dist = math.hypot(X[0] - centre[0], X[1] - centre[1])
    return math.copysign(1.0, kappa) * (1.0 / abs(kappa) - dist)


def random_hits(rng, n, n_layers=10, rmax=80.0):
    r = rng.uniform(3.0, rmax, n)
    phi = rng.uniform(-math.pi, math.pi, n)
    return ((r * np.cos(phi)).astype(np.float32), (r * np.sin(phi)).astype(np.float32),
            rng.integers(0, n_layers, n).astype(np.int32))


# ============================================================ E1: straight-line transform

LINE_GRID = synth.Grid(n_phi=48, n_d0=1, n_kappa=32, L_min=3, d0_min=0.0, d0_max=0.0, kappa_min=-20.0,
                       kappa_max=30.0)


def test_line_vote_is_the_signed_distance_of_the_line_through_the_hit(oracle):
    """For every (hit, theta centre): the voted rho bin contains the signed distance from the
    origin of the line of direction theta through the hit, computed in fp64 as the cross
    product dir x X; no vote iff that distance is outside [rho_min, rho_max)."""
    g = LINE_GRID
    rng = np.random.default_rng(5)
    x, y, layer = random_hits(rng, 40, rmax=35.0)
    th = centres(g.phi_min, g.phi_max, g.n_phi)
    edges = np.linspace(g.kappa_min, g.kappa_max, g.n_kappa + 1)
    checked = 0
    for h in range(len(x)):
        acc, nv, _ = oracle.vote_variant(g, oracle.MODE_LINE, x[h:h + 1], y[h:h + 1], layer[h:h + 1])
        for i in range(g.n_phi):
            rho = math.cos(th[i]) * float(y[h]) - math.sin(th[i]) * float(x[h])  # dir x X
            row = acc[i, 0]
            if np.min(np.abs(edges - rho)) < 1e-4:
                continue  # within rounding of an edge: either side is acceptable
            checked += 1
            if g.kappa_min <= rho < g.kappa_max:
                k = int(np.searchsorted(edges, rho, side="right") - 1)
                assert row[k] == (1 << int(layer[h])) and np.count_nonzero(row) == 1
            else:
                assert not row.any()
    assert checked > 1500


def test_line_transform_finds_collinear_hits_at_their_own_bin(oracle):
    """Hits placed exactly on the line (theta_c[i0], rho centre k0) peak in bin (i0, 0, k0) with
    every layer (peaks appear at the parameters of the actual trajectories)."""
    g = dataclasses.replace(LINE_GRID, L_min=8)
    th = centres(g.phi_min, g.phi_max, g.n_phi)
    rc = centres(g.kappa_min, g.kappa_max, g.n_kappa)
    for i0, k0 in [(3, 5), (20, 16), (47, 30)]:
        theta, rho = th[i0], rc[k0]
        t = np.linspace(5.0, 60.0, 10)
        x = (-rho * math.sin(theta) + t * math.cos(theta)).astype(np.float32)
        y = (rho * math.cos(theta) + t * math.sin(theta)).astype(np.float32)
        layer = np.arange(10, dtype=np.int32)
        res = oracle.run_variant(g, oracle.MODE_LINE, x, y, layer)
        assert res["acc"][i0, 0, k0] == 0x3ff
        assert lin_of(g, i0, 0, k0) in res["peak_bin"].tolist()
        p = res["peak_bin"].tolist().index(lin_of(g, i0, 0, k0))
        assert res["hit_index"][int(res["hit_offset"][p]):int(res["hit_offset"][p + 1])].tolist() == list(range(10))


def test_variant_mode0_is_the_base_oracle(oracle):
    g = synth.Grid(n_phi=16, n_d0=4, n_kappa=32, L_min=2)
    x, y, layer = random_hits(np.random.default_rng(1), 200)
    a0, n0, _ = oracle.vote(g, x, y, layer)
    a1, n1, _ = oracle.vote_variant(g, oracle.MODE_CIRCLE, x, y, layer)
    assert np.array_equal(a0, a1) and n0 == n1
    pb, _, _ = oracle.peaks(g, a0)
    o0, i0, t0 = oracle.hitlists(g, x, y, layer, pb)
    o1, i1, t1 = oracle.hitlists_variant(g, oracle.MODE_CIRCLE, x, y, layer, pb)
    assert np.array_equal(o0, o1) and np.array_equal(i0, i1) and t0 == t1


def test_cellwise_variant_hit_lists_equal_the_peakwise_ones(oracle):
    """oracle_hitlists_variant_cells against oracle_hitlists_variant (pinned above and below) in all three
    modes: random grids with bad and non-finite hits, whole peak lists, subsets, a cap that cuts a list,
    every non-empty bin (total = n_votes), no peaks."""
    rng = np.random.default_rng(40)
    for mode in (oracle.MODE_CIRCLE, oracle.MODE_LINE, oracle.MODE_INTERVAL):
        for shape, n in [((16, 4, 32), 120), ((24, 1, 64), 300), ((7, 3, 32), 2)]:
            if mode == oracle.MODE_LINE and shape[1] != 1:
                continue
            kw = dict(d0_min=0.0, d0_max=0.0) if shape[1] == 1 else {}
            if mode == oracle.MODE_LINE:
                kw.update(kappa_min=-90.0, kappa_max=90.0)
            g = synth.Grid(n_phi=shape[0], n_d0=shape[1], n_kappa=shape[2], L_min=2, **kw)
            x, y, layer = random_hits(rng, n)
            if n > 10:
                layer[::13] = -1
                x[1], y[2] = np.nan, np.inf
            acc, n_votes, _ = oracle.vote_variant(g, mode, x, y, layer)
            pb, _pm, _n = oracle.peaks(g, acc)
            allbins = np.nonzero(acc.reshape(-1))[0].astype(np.uint32)
            for bins in (pb, pb[1::2], allbins, pb[:0]):
                o1, i1, t1 = oracle.hitlists_variant(g, mode, x, y, layer, bins)
                o2, i2, t2 = oracle.hitlists_variant(g, mode, x, y, layer, bins, by_cell=True)
                assert t1 == t2 and np.array_equal(o1, o2) and np.array_equal(i1, i2)
            assert t1 == 0
            o1, i1, t1 = oracle.hitlists_variant(g, mode, x, y, layer, allbins)
            assert t1 == n_votes
            if len(pb) > 2:
                cap = int(oracle.hitlists_variant(g, mode, x, y, layer, pb)[0][len(pb) // 2]) + 1
                o3, i3, t3 = oracle.hitlists_variant(g, mode, x, y, layer, pb, cap_hits=cap, by_cell=True)
                of, idf, tf = oracle.hitlists_variant(g, mode, x, y, layer, pb)
                assert t3 == tf and np.array_equal(o3, of) and np.array_equal(i3, idf[:cap])


# ============================================================ E2: interval voting

def test_interval_vote_covers_the_curvatures_met_inside_the_phi0_bin(oracle):
    """Meaning of the interval: a kappa bin strictly inside the
    voted range has, by continuity, a phi0 inside the phi0 bin whose circle passes through the
    hit -- the fp64 signed distance from the hit to the track (phi0, d0_j, kappa_centre) has
    opposite signs at the two phi0 bin EDGES; two bins or more outside the range it has the
    same sign at both.  (Hits within 2 cm of the point of closest approach are left out: the
    pole of kappa(phi0), reading X2.)"""
    g = synth.Grid(n_phi=40, n_d0=4, n_kappa=48, L_min=2)
    rng = np.random.default_rng(11)
    x, y, layer = random_hits(rng, 12)
    pe = np.linspace(g.phi_min, g.phi_max, g.n_phi + 1)
    d0c = centres(g.d0_min, g.d0_max, g.n_d0)
    kc = centres(g.kappa_min, g.kappa_max, g.n_kappa)
    inside = outside = 0
    for h in range(len(x)):
        X = np.array([float(x[h]), float(y[h])])
        acc, nv, _ = oracle.vote_variant(g, oracle.MODE_INTERVAL, x[h:h + 1], y[h:h + 1], layer[h:h + 1])
        assert nv == np.count_nonzero(acc)
        for i in range(g.n_phi):
            for j in range(g.n_d0):
                near = False
                for pp in (pe[i], pe[i + 1], 0.5 * (pe[i] + pe[i + 1])):
                    P0 = d0c[j] * np.array([-math.sin(pp), math.cos(pp)])
                    near |= math.hypot(*(X - P0)) < 2.0
                if near:
                    continue
                ks = np.nonzero(acc[i, j])[0]
                if len(ks):
                    assert np.array_equal(ks, np.arange(ks[0], ks[-1] + 1))  # one contiguous range
                k0, k1 = (ks[0], ks[-1]) if len(ks) else (10 ** 6, -10 ** 6)
                for k in range(g.n_kappa):
                    fa = signed_distance(X, pe[i], d0c[j], kc[k])
                    fb = signed_distance(X, pe[i + 1], d0c[j], kc[k])
                    if k0 < k < k1:
                        assert fa * fb < 0.0
                        inside += 1
                    elif k < k0 - 1 or k > k1 + 1:
                        assert fa * fb > 0.0
                        outside += 1
    assert inside > 300 and outside > 10000


def test_interval_end_points_are_the_votes_at_the_bin_edges(oracle):
    """The range's end bins are the single-bin votes of the base oracle evaluated at the phi0
    EDGES: a grid shifted by half a bin (exactly representable numbers) has its centres there."""
    g = synth.Grid(n_phi=8, n_d0=3, n_kappa=64, L_min=2, phi_min=-1.0, phi_max=1.0)
    gs = dataclasses.replace(g, n_phi=9, phi_min=-1.125, phi_max=1.125)  # centres = g's edges
    rng = np.random.default_rng(3)
    x, y, layer = random_hits(rng, 60)
    n_checked = 0
    for h in range(len(x)):
        acc, _, _ = oracle.vote_variant(g, oracle.MODE_INTERVAL, x[h:h + 1], y[h:h + 1], layer[h:h + 1])
        edge, _, _ = oracle.vote(gs, x[h:h + 1], y[h:h + 1], layer[h:h + 1])
        for i in range(g.n_phi):
            for j in range(g.n_d0):
                ka, kb = np.nonzero(edge[i, j])[0], np.nonzero(edge[i + 1, j])[0]
                ks = np.nonzero(acc[i, j])[0]
                if len(ka) and len(kb):  # both edge votes in range: exactly the bins between them
                    lo, hi = min(ka[0], kb[0]), max(ka[0], kb[0])
                    assert np.array_equal(ks, np.arange(lo, hi + 1))
                    n_checked += 1
                elif len(ka) or len(kb):  # one end outside the kappa range: clipped at the grid's end
                    k_in = (ka if len(ka) else kb)[0]
                    assert len(ks) and (ks[0] == k_in or ks[-1] == k_in)
                    assert ks[0] == 0 or ks[-1] == g.n_kappa - 1
    assert n_checked > 100


def test_interval_hit_lists_are_the_hits_covering_the_peak_bin(oracle):
    g = synth.Grid(n_phi=24, n_d0=4, n_kappa=32, L_min=3)
    x, y, layer = random_hits(np.random.default_rng(8), 150)
    res = oracle.run_variant(g, oracle.MODE_INTERVAL, x, y, layer)
    assert res["n_peaks"] > 0
    off, idx = res["hit_offset"], res["hit_index"]
    for p, lin in enumerate(res["peak_bin"]):
        k = int(lin) % g.n_kappa
        j = (int(lin) // g.n_kappa) % g.n_d0
        i = int(lin) // (g.n_kappa * g.n_d0)
        hs = idx[int(off[p]):int(off[p + 1])]
        assert np.all(np.diff(hs.astype(np.int64)) > 0)
        m = 0
        for h in hs:
            m |= 1 << int(layer[h])
        assert m == int(res["peak_mask"][p])
        for h in range(len(x)):  # membership == the single hit's own vote covers the bin
            a, _, _ = oracle.vote_variant(g, oracle.MODE_INTERVAL, x[h:h + 1], y[h:h + 1], layer[h:h + 1])
            assert (a[i, j, k] != 0) == (h in hs)
        if p >= 3:
            break


# ============================================================ E3: the second transform (vertices)

VG = synth.VertexGrid(n_x=20, n_y=12, V_min=3, x_min=-5.0, x_max=7.0, y_min=-4.0, y_max=2.0)
PG = synth.Grid(n_phi=64, n_d0=16, n_kappa=8, L_min=2)


def test_vertex_vote_is_where_the_peaks_line_crosses_the_column(oracle):
    """A peak (phi0_i, d0_j) is the line {d0 n + t dir}; in fp64, written parametrically (never as
    (d0 + x sin)/cos), its crossing with the column x = xc[a] (row y = yc[b] for steep lines) lies
    in the voted bin; no vote iff the crossing is outside the vertex grid."""
    phic = centres(PG.phi_min, PG.phi_max, PG.n_phi)
    d0c = centres(PG.d0_min, PG.d0_max, PG.n_d0)
    xc, yc = centres(VG.x_min, VG.x_max, VG.n_x), centres(VG.y_min, VG.y_max, VG.n_y)
    xe, ye = np.linspace(VG.x_min, VG.x_max, VG.n_x + 1), np.linspace(VG.y_min, VG.y_max, VG.n_y + 1)
    rng = np.random.default_rng(2)
    sure = 0
    for _ in range(150):
        i, j, k = int(rng.integers(PG.n_phi)), int(rng.integers(PG.n_d0)), int(rng.integers(PG.n_kappa))
        vacc, nv = oracle.vertex_vote(PG, VG, [lin_of(PG, i, j, k)])
        assert nv == vacc.sum() and vacc.max() <= 1
        nvec = np.array([-math.sin(phic[i]), math.cos(phic[i])])
        dvec = np.array([math.cos(phic[i]), math.sin(phic[i])])
        base = d0c[j] * nvec
        if abs(dvec[0]) >= abs(dvec[1]):  # shallow: one vote per x column
            for a in range(VG.n_x):
                yv = base[1] + (xc[a] - base[0]) / dvec[0] * dvec[1]
                if np.min(np.abs(ye - yv)) < 1e-4:
                    continue
                sure += 1
                if VG.y_min <= yv < VG.y_max:
                    b = int(np.searchsorted(ye, yv, side="right") - 1)
                    assert vacc[a, b] == 1 and vacc[a].sum() == 1
                else:
                    assert vacc[a].sum() == 0
        else:
            for b in range(VG.n_y):
                xv = base[0] + (yc[b] - base[1]) / dvec[1] * dvec[0]
                if np.min(np.abs(xe - xv)) < 1e-4:
                    continue
                sure += 1
                if VG.x_min <= xv < VG.x_max:
                    a = int(np.searchsorted(xe, xv, side="right") - 1)
                    assert vacc[a, b] == 1 and vacc[:, b].sum() == 1
                else:
                    assert vacc[:, b].sum() == 0
    assert sure > 1500


def test_tracks_from_a_common_vertex_lie_on_its_sinusoid():
    """the crossings of a displaced jet lie on one sinusoid of the parameter space,
    d0 = -xv sin(phi0) + yv cos(phi0).  fp64 geometry: exact for straight tracks; for a circle the
    offset is kappa |V - P0|^2 / 2 (reading X3 of DESIGN.md section 8)."""
    rng = np.random.default_rng(4)
    for _ in range(200):
        xv, yv = rng.uniform(-6, 6, 2)
        psi = rng.uniform(-math.pi, math.pi)
        phi0, d0 = synth.track_from_vertex(xv, yv, psi, 0.0)
        assert abs(d0 - (-xv * math.sin(phi0) + yv * math.cos(phi0))) < 1e-12
        kappa = rng.uniform(-0.0114, 0.0114)
        phi0, d0 = synth.track_from_vertex(xv, yv, psi, kappa)
        assert abs(signed_distance(np.array([xv, yv]), phi0, d0, kappa)) < 1e-9  # V is on the circle
        P0 = d0 * np.array([-math.sin(phi0), math.cos(phi0)])
        L2 = (xv - P0[0]) ** 2 + (yv - P0[1]) ** 2
        s_v = -xv * math.sin(phi0) + yv * math.cos(phi0)
        assert abs((s_v - d0) - 0.5 * kappa * L2) < 1e-9


def _peaks_on_sinusoid(grid, xv, yv, rows):
    d0c = centres(grid.d0_min, grid.d0_max, grid.n_d0)
    phic = centres(grid.phi_min, grid.phi_max, grid.n_phi)
    out = []
    for i in rows:
        d = -xv * math.sin(phic[i]) + yv * math.cos(phic[i])
        j = int(np.argmin(np.abs(d0c - d)))
        out.append(lin_of(grid, i, j, int(i) % grid.n_kappa))
    return np.array(sorted(out), dtype=np.uint32)


def test_second_transform_finds_the_vertices_of_one_and_two_jets(oracle):
    """Fig. 7 / Fig. 8 in miniature: peaks placed on the sinusoid of a vertex (d0 snapped to its
    nearest bin centre) make that vertex's bin the maximum of the second accumulator and a
    reported vertex whose members are exactly those peaks; two jets give two vertices."""
    g = synth.Grid(n_phi=256, n_d0=128, n_kappa=8, L_min=2)  # d0 bins 0.16 cm << vertex bins 1 cm
    vg = synth.VertexGrid(n_x=16, n_y=16, V_min=10)
    xc, yc = centres(vg.x_min, vg.x_max, vg.n_x), centres(vg.y_min, vg.y_max, vg.n_y)
    a1, b1, a2, b2 = 11, 4, 3, 9
    rows1 = np.arange(5, 250, 7)   # 35 peaks, all directions
    rows2 = np.arange(2, 250, 11)  # 23 peaks
    p1 = _peaks_on_sinusoid(g, xc[a1], yc[b1], rows1)
    res = oracle.run_vertices(g, vg, p1)
    assert np.unravel_index(np.argmax(res["vacc"]), res["vacc"].shape) == (a1, b1)
    assert res["vacc"][a1, b1] == len(p1)
    assert (a1 * vg.n_y + b1) in res["vertex_bin"].tolist()
    m = res["vertex_bin"].tolist().index(a1 * vg.n_y + b1)
    assert res["vertex_count"][m] == len(p1)
    assert res["member_index"][int(res["member_offset"][m]):int(res["member_offset"][m + 1])].tolist() == list(range(len(p1)))
    both = np.array(sorted(set(p1.tolist()) | set(_peaks_on_sinusoid(g, xc[a2], yc[b2], rows2).tolist())), dtype=np.uint32)
    res2 = oracle.run_vertices(g, vg, both)
    top2 = set(np.argsort(res2["vacc"].ravel())[-2:].tolist())
    assert top2 == {a1 * vg.n_y + b1, a2 * vg.n_y + b2}
    assert top2 <= set(res2["vertex_bin"].tolist())


def test_mirror_peaks_vote_into_the_same_vertex_bins(oracle):
    """(phi0 + pi, -d0) is the same line, so the mirror image of a peak set
    fills the same second accumulator, up to votes that sit on a bin edge."""
    g = PG
    rng = np.random.default_rng(6)
    ii, jj = rng.integers(0, g.n_phi, 300), rng.integers(0, g.n_d0, 300)
    p = np.unique(np.array([lin_of(g, int(i), int(j), 0) for i, j in zip(ii, jj)], dtype=np.uint32))
    pm = np.unique(np.array([lin_of(g, (int(i) + g.n_phi // 2) % g.n_phi, g.n_d0 - 1 - int(j), 0)
                             for i, j in zip(ii, jj)], dtype=np.uint32))
    va, na = oracle.vertex_vote(g, VG, p)
    vb, nb = oracle.vertex_vote(g, VG, pm)
    assert na > 1000
    assert np.abs(va.astype(np.int64) - vb.astype(np.int64)).sum() <= 0.01 * na


def test_vertex_peak_rule_against_a_ranking_brute_force(oracle):
    """V3: count >= V_min and first in the (count desc, lin asc) ranking of its 3x3 neighbourhood."""
    rng = np.random.default_rng(9)
    for trial in range(30):
        vg = synth.VertexGrid(n_x=int(rng.integers(1, 9)), n_y=int(rng.integers(1, 9)), V_min=int(rng.integers(1, 4)))
        vacc = rng.integers(0, 5, (vg.n_x, vg.n_y)).astype(np.uint32)  # few values: many plateaus
        vb, vc, n = oracle.vertex_peaks(vg, vacc)
        want = []
        for a in range(vg.n_x):
            for b in range(vg.n_y):
                if vacc[a, b] < vg.V_min:
                    continue
                nb = [(-int(vacc[aa, bb]), aa * vg.n_y + bb) for aa in range(max(a - 1, 0), min(a + 2, vg.n_x))
                      for bb in range(max(b - 1, 0), min(b + 2, vg.n_y))]
                if min(nb) == (-int(vacc[a, b]), a * vg.n_y + b):
                    want.append(a * vg.n_y + b)
        assert n == len(want) and vb.tolist() == want
        assert vc.tolist() == [int(vacc.ravel()[w]) for w in want]
    vg = synth.VertexGrid(n_x=4, n_y=5, V_min=1)
    vb, vc, n = oracle.vertex_peaks(vg, np.full((4, 5), 7, np.uint32), cap=0)
    assert n == 1 and len(vb) == 0  # all equal: only lin 0; cap 0 still counts


def test_vertex_members_partition_the_votes(oracle):
    """V4 against V2: the members of EVERY bin, taken as a vertex, number that bin's count."""
    g, vg = PG, synth.VertexGrid(n_x=6, n_y=5, V_min=1, x_min=-3.0, x_max=3.0, y_min=-2.0, y_max=3.0)
    rng = np.random.default_rng(12)
    p = np.unique(rng.integers(0, g.n_bins, 80).astype(np.uint32))
    vacc, nv = oracle.vertex_vote(g, vg, p)
    allbins = np.arange(vg.n_x * vg.n_y, dtype=np.uint32)
    off, idx, tot = oracle.vertex_members(g, vg, p, allbins)
    assert tot == nv
    assert np.array_equal(np.diff(off.astype(np.int64)), vacc.ravel().astype(np.int64))
    for m in range(len(allbins)):
        assert np.all(np.diff(idx[int(off[m]):int(off[m + 1])].astype(np.int64)) > 0)
    off2, idx2, tot2 = oracle.vertex_members(g, vg, p, allbins, cap=7)
    assert tot2 == tot and np.array_equal(idx2, idx[:7])


# ============================================================ E4: the fit

def circle_points(phi0, d0, kappa, radii, sigma=0.0, rng=None):
    """Points of the track (phi0, d0, kappa) at the given radii (forward branch), fp64."""
    pts = []
    for r in radii:
        s = (kappa * (r * r + d0 * d0) + 2.0 * d0) / (2.0 * (1.0 + kappa * d0))
        phi = phi0 + math.asin(s / r)
        if sigma:
            phi += rng.normal(0.0, sigma) / r
        pts.append((r * math.cos(phi), r * math.sin(phi)))
    return np.array(pts)


def fit_points(oracle, pts, order=None):
    x = pts[:, 0].astype(np.float32)
    y = pts[:, 1].astype(np.float32)
    idx = np.arange(len(x), dtype=np.uint32) if order is None else np.asarray(order, dtype=np.uint32)
    return oracle.fit_one(x, y, idx)


def angle_diff(a, b):
    return (a - b + math.pi) % (2 * math.pi) - math.pi


@pytest.mark.parametrize("seed", [0, 1])
def test_fit_recovers_exact_circles_and_straight_lines(oracle, seed):
    rng = np.random.default_rng(seed)
    for trial in range(100):
        phi0 = rng.uniform(-math.pi, math.pi)
        d0 = rng.uniform(-2.5, 2.5)
        kappa = 0.0 if trial % 5 == 0 else rng.uniform(-0.0114, 0.0114)
        pts = circle_points(phi0, d0, kappa, synth.LAYER_RADII_CM)
        st, k, p, d, rms = fit_points(oracle, pts)
        assert st == 0
        # the only error is the rounding of the coordinates to binary32 (~4e-6 cm at 78 cm)
        assert abs(k - kappa) < 2e-8 and abs(d - d0) < 3e-5 and abs(angle_diff(p, phi0)) < 2e-6
        assert rms < 1e-5


def test_fit_agrees_with_a_geometric_least_squares_fit(oracle):
    """On smeared hits the closed-form fit agrees with Gauss-Newton on the fp64 signed distances
    (scipy) to a small fraction of the parameters' own uncertainties, and its rms is the rms
    of the signed distances."""
    from scipy.optimize import least_squares

    rng = np.random.default_rng(7)
    sig = 0.02  # 200 um, exaggerated so that the comparison is not dominated by fp32 rounding
    for trial in range(40):
        phi0, d0, kappa = rng.uniform(-math.pi, math.pi), rng.uniform(-2, 2), rng.uniform(-0.011, 0.011)
        pts = circle_points(phi0, d0, kappa, synth.LAYER_RADII_CM, sig, rng)
        pts32 = np.stack([pts[:, 0].astype(np.float32), pts[:, 1].astype(np.float32)], 1).astype(np.float64)
        st, k, p, d, rms = fit_points(oracle, pts)
        assert st == 0

        def resid(q):
            return [signed_distance(X, q[0], q[1], q[2]) for X in pts32]

        sol = least_squares(resid, [phi0, d0, kappa], x_scale=[1e-3, 1e-2, 1e-5], xtol=1e-15, ftol=1e-15, gtol=1e-15)
        pg, dg, kg = sol.x
        # parameter uncertainties at this smearing: ~1e-3 rad, ~2e-2 cm, ~3e-5 /cm
        assert abs(angle_diff(p, pg)) < 2e-5 and abs(d - dg) < 5e-4 and abs(k - kg) < 5e-7
        rms_geo = math.sqrt(np.mean(np.square(resid([p, d, k]))))
        assert abs(rms - rms_geo) < 0.02 * rms_geo + 1e-6


def test_fit_is_rotation_covariant_and_order_free_up_to_rounding(oracle):
    rng = np.random.default_rng(10)
    pts = circle_points(0.4, 1.2, 0.006, synth.LAYER_RADII_CM, 0.01, rng)
    st, k, p, d, rms = fit_points(oracle, pts)
    for alpha in (0.7, -2.1, 3.0):
        c, s = math.cos(alpha), math.sin(alpha)
        rot = pts @ np.array([[c, s], [-s, c]])
        st2, k2, p2, d2, rms2 = fit_points(oracle, rot)
        assert st2 == 0 and abs(k2 - k) < 2e-8 and abs(d2 - d) < 3e-5 and abs(angle_diff(p2, p + alpha)) < 1e-6
        assert abs(rms2 - rms) < 1e-6
    st3, k3, p3, d3, rms3 = fit_points(oracle, pts[::-1].copy())
    assert abs(k3 - k) < 1e-12 and abs(d3 - d) < 1e-9 and abs(angle_diff(p3, p)) < 1e-12


def test_fit_reports_the_forward_representation(oracle):
    """(phi + pi, -d0, -kappa) is the same circle; the hits must lie ahead of the point of closest
    approach.  Hits generated on the backward branch of (phi0, d0, kappa) are the forward branch
    of its mirror."""
    pts = circle_points(0.3, 1.0, 0.004, synth.LAYER_RADII_CM)
    mirrored = -pts  # point reflection: the forward branch of (phi0 + pi, d0, kappa)
    st, k, p, d, _ = fit_points(oracle, mirrored)
    assert st == 0 and abs(angle_diff(p, 0.3 + math.pi)) < 2e-6 and abs(d - 1.0) < 3e-5 and abs(k - 0.004) < 2e-8
    for q in (pts, mirrored):
        st, k, p, d, _ = fit_points(oracle, q)
        assert np.mean(q[:, 0] * math.cos(p) + q[:, 1] * math.sin(p)) > 0


def test_fit_rms_is_the_transverse_scatter(oracle):
    """Hits displaced by +-delta perpendicular to a straight track, alternating: rms ~ delta."""
    delta = 0.05
    t = np.linspace(5, 75, 12)
    phi0 = 0.9
    dirv = np.array([math.cos(phi0), math.sin(phi0)])
    nvec = np.array([-math.sin(phi0), math.cos(phi0)])
    pts = np.array([tt * dirv + (delta if q % 2 else -delta) * nvec for q, tt in enumerate(t)])
    st, k, p, d, rms = fit_points(oracle, pts)
    assert st == 0 and abs(rms - delta) < 0.15 * delta


def test_fit_status_codes(oracle):
    x = np.array([1, 2, 3, 4], np.float32)
    y = np.array([0, 0, 0, 0], np.float32)
    assert fit_points(oracle, np.stack([x, y], 1)[:2])[0] == 1        # fewer than 3 hits
    same = np.array([[3.0, 4.0]] * 4)
    assert fit_points(oracle, same)[0] == 2                            # all hits equal: Crr = 0
    ring = np.array([[5.0, 0.0], [0.0, 5.0], [-5.0, 0.0], [3.0, 4.0], [4.0, -3.0]])  # r^2 = 25 exactly
    assert fit_points(oracle, ring)[0] == 2                            # all at one radius: Crr = 0


# ============================================================ E5: selection and duplicates

def test_select_dedup_against_set_arithmetic(oracle):
    rng = np.random.default_rng(13)
    n_hits, n_c = 60, 120
    lists = []
    for c in range(n_c):
        base = lists[rng.integers(len(lists))] if lists and rng.random() < 0.5 else None
        if base is not None:  # a near-copy of an earlier candidate
            hs = set(base)
            for _ in range(int(rng.integers(0, 3))):
                hs.discard(int(rng.choice(sorted(hs)))) if len(hs) > 3 else None
                hs.add(int(rng.integers(n_hits)))
        else:
            hs = set(int(v) for v in rng.choice(n_hits, int(rng.integers(3, 9)), replace=False))
        lists.append(sorted(hs))
    off = np.zeros(n_c + 1, np.uint64)
    off[1:] = np.cumsum([len(l) for l in lists])
    idx = np.array([h for l in lists for h in l], np.uint32)
    mask = np.array([(1 << int(rng.integers(3, 8))) - 1 for _ in range(n_c)], np.uint32)
    fit = np.zeros(n_c, oracle.FIT_DTYPE)
    fit["rms"] = rng.choice([0.001, 0.002, 0.003, 0.5], n_c)  # ties on purpose
    status = rng.choice([0, 0, 0, 2], n_c).astype(np.int32)
    rms_max, min_shared = 0.01, 3
    flags = oracle.select_dedup(off, idx, mask, n_hits, fit, status, rms_max, min_shared)
    sel = [c for c in range(n_c) if status[c] == 0 and fit["rms"][c] <= rms_max]
    key = lambda c: (-bin(int(mask[c])).count("1"), float(fit["rms"][c]), c)
    for c in range(n_c):
        if c not in sel:
            assert flags[c] == 0
            continue
        dup = any(o != c and len(set(lists[c]) & set(lists[o])) >= min_shared and key(o) < key(c) for o in sel)
        assert flags[c] == (2 if dup else 1)
    assert {0, 1, 2} <= set(flags.tolist())


def test_mirror_twins_fit_identically_and_one_survives(oracle):
    """every track gives two peaks with the same hits; their fits are
    bit-identical (forward representation) and the duplicate rule keeps the lower one only."""
    g = synth.Grid(n_phi=64, n_d0=8, n_kappa=32, L_min=8)
    x, y, layer = synth.single_track_event(g, 9, 5, 0.004)
    res = oracle.run(g, x, y, layer)
    assert res["n_peaks"] >= 2
    fit, status = oracle.fit_all(x, y, res["hit_offset"], res["hit_index"])
    full = [p for p in range(res["n_peaks"]) if int(res["hit_offset"][p + 1] - res["hit_offset"][p]) == len(x)]
    assert len(full) >= 2 and all(status[p] == 0 for p in full)
    a, b = full[0], full[-1]
    assert fit[a] == fit[b]
    flags = oracle.select_dedup(res["hit_offset"], res["hit_index"], res["peak_mask"], len(x), fit, status, 0.01, 5)
    assert flags[a] == 1 and flags[b] == 2
