"""GPU parity of the rows SURVEY.md 8(f) marks "next" (f1 vertices, f2 fit + duplicates, f3 vote
variants) against oracle/hough_ext_oracle.c, through the C ABI (include/hough.h).

Index and integer results are compared bit for bit; the binary64 fit within the tolerance
DESIGN.md section 8 derives (different libm / CUDA math library sin, cos, atan2: a few ulp,
amplified by the cancellation in the transverse moment).
"""
import dataclasses
import math

import numpy as np
import pytest

from paper_1305_4855_b200 import synth

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def hough():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1305_4855_b200 import hough as hough_mod
    return hough_mod


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def random_hits(rng, n, n_layers=10, rmax=80.0):
    r = rng.uniform(0.5, rmax, n)
    phi = rng.uniform(-math.pi, math.pi, n)
    return ((r * np.cos(phi)).astype(np.float32), (r * np.sin(phi)).astype(np.float32),
            rng.integers(0, n_layers, n).astype(np.int32))


def make(hough, grid, x, y, layer, cap_peaks, cap_hits, **kw):
    h = hough.Hough(grid, max_hits=max(len(x), 1), cap_peaks=cap_peaks, cap_hits=cap_hits, **kw)
    h.vote(dev(x.astype(np.float32)), dev(y.astype(np.float32)), dev(layer.astype(np.int32)))
    h.peaks()
    return h


# ============================================================ f1: hough_vertices

def assert_vertices_same(res, ref):
    assert np.array_equal(res["vacc"], ref["vacc"])
    assert res["n_vertex_votes"] == ref["n_vertex_votes"]
    assert res["n_vertices"] == ref["n_vertices"]
    assert np.array_equal(res["vertex_bin"], ref["vertex_bin"])
    assert np.array_equal(res["vertex_count"], ref["vertex_count"])
    assert res["n_member_entries"] == ref["n_member_entries"]
    assert np.array_equal(res["member_offset"], ref["member_offset"])
    assert np.array_equal(res["member_index"], ref["member_index"])


@pytest.mark.parametrize("shape,vshape,n_hits,seed", [
    ((64, 16, 32), (20, 12), 300, 0),      # accumulator copy in shared memory, non-square
    ((50, 13, 64), (1, 37), 400, 1),       # a single column
    ((96, 8, 32), (130, 100), 500, 2),     # 13 000 bins: global atomics
    ((33, 9, 32), (257, 3), 200, 3),       # ragged blocks
])
def test_vertices_random_small(hough, oracle, shape, vshape, n_hits, seed):
    rng = np.random.default_rng(seed)
    g = synth.Grid(n_phi=shape[0], n_d0=shape[1], n_kappa=shape[2], L_min=2)
    vg = synth.VertexGrid(n_x=vshape[0], n_y=vshape[1], V_min=3, x_min=-5.0, x_max=7.0, y_min=-4.0, y_max=2.5)
    x, y, layer = random_hits(rng, n_hits)
    ref = oracle.run(g, x, y, layer)
    assert ref["n_peaks"] > 20
    h = make(hough, g, x, y, layer, 1 << 16, 1 << 20)
    res = h.read()
    assert np.array_equal(res["peak_bin"], ref["peak_bin"])
    vref = oracle.run_vertices(g, vg, ref["peak_bin"])
    assert vref["n_vertices"] > 0
    for rep in range(2):  # the call is repeatable on the same handle
        h.vertices(vg, cap_vertices=4096, cap_members=1 << 20)
        assert_vertices_same(h.read_vertices(), vref)
    h.close()


def test_vertices_jets_workload(hough, oracle):
    """The displaced-jet workload (PAPER.md:154 Fig. 7, :168 Fig. 8 in synthetic form)."""
    g, vg = synth.JETS_GRID, synth.JETS_VGRID
    for seed in (0, 1):
        x, y, layer, truth = synth.generate_jet_event(synth.JETS_SPEC, seed)
        ref = oracle.run(g, x, y, layer)
        vref = oracle.run_vertices(g, vg, ref["peak_bin"])
        h = make(hough, g, x, y, layer, 1 << 16, 1 << 20)
        h.vertices(vg)
        assert_vertices_same(h.read_vertices(), vref)
        h.close()


def test_vertices_over_the_peaks_of_a_pileup_event(hough, oracle):
    """4.9e5 peaks (BASELINE.json configs[2]) into 32 x 32 and 100 x 60 vertex grids: the member lists
    come from the d0 rows that can reach the vertex bin (binary searches in the sorted peak list)."""
    w = synth.WORKLOADS["pileup"]
    x, y, layer, _ = synth.generate_event(w.event, w.seeds[0])
    acc, _nv, _nb = oracle.vote(w.grid, x, y, layer)
    pb, _pm, n_peaks = oracle.peaks(w.grid, acc)
    h = hough.Hough(w.grid, len(x), w.cap_peaks, w.cap_hits)
    h.vote(dev(x), dev(y), dev(layer))
    h.peaks(lists=False)
    assert np.array_equal(h.read(lists=False)["peak_bin"], pb)
    for vg, cap_v in ((synth.JETS_VGRID, 1024), (synth.VertexGrid(n_x=100, n_y=60, V_min=2500, x_min=-9.0, x_max=11.0,
                                                                   y_min=-6.0, y_max=6.0), 4096)):
        vref = oracle.run_vertices(w.grid, vg, pb)
        assert vref["n_vertices"] > 10
        h.vertices(vg, cap_vertices=cap_v, cap_members=1 << 23)
        assert_vertices_same(h.read_vertices(), vref)
    h.close()


def test_vertices_truncation_and_no_peaks(hough, oracle):
    rng = np.random.default_rng(5)
    g = synth.Grid(n_phi=64, n_d0=16, n_kappa=32, L_min=2)
    vg = synth.VertexGrid(n_x=24, n_y=24, V_min=2)
    x, y, layer = random_hits(rng, 300)
    ref = oracle.run(g, x, y, layer)
    full = oracle.run_vertices(g, vg, ref["peak_bin"])
    assert full["n_vertices"] > 6 and full["n_member_entries"] > 40
    h = make(hough, g, x, y, layer, 1 << 16, 1 << 20)
    # vertex capacity smaller than the number of vertices: the first ones in lin order, with their lists
    cut = oracle.run_vertices(g, vg, ref["peak_bin"], cap_vertices=5)
    h.vertices(vg, cap_vertices=5, cap_members=1 << 16)
    res = h.read_vertices()
    assert res["flags"] & 1 and res["n_vertices"] == full["n_vertices"]
    assert np.array_equal(res["vertex_bin"], cut["vertex_bin"]) and np.array_equal(res["member_index"], cut["member_index"])
    assert np.array_equal(res["member_offset"], cut["member_offset"])
    # member capacity smaller than the total: true total reported, the first entries written
    h.vertices(vg, cap_vertices=4096, cap_members=17)
    res = h.read_vertices()
    assert res["flags"] & 2 and res["n_member_entries"] == full["n_member_entries"]
    assert np.array_equal(res["member_index"], full["member_index"][:17])
    assert np.array_equal(res["member_offset"], full["member_offset"])
    h.close()
    # an event without peaks: an all-zero accumulator, no vertex, member_offset[0] = 0
    g9 = dataclasses.replace(g, L_min=9)
    h = make(hough, g9, x[:5], y[:5], layer[:5], 1 << 10, 1 << 12)
    assert h.read()["n_peaks"] == 0
    h.vertices(vg)
    res = h.read_vertices()
    assert res["n_vertices"] == 0 and res["n_vertex_votes"] == 0 and not res["vacc"].any()
    assert res["member_offset"].tolist() == [0]
    h.close()


def test_vertices_rejects_bad_arguments(hough):
    g = synth.Grid(n_phi=16, n_d0=4, n_kappa=32, L_min=2)
    x, y, layer = random_hits(np.random.default_rng(0), 50)
    h = make(hough, g, x, y, layer, 1 << 10, 1 << 12)
    for bad in (synth.VertexGrid(n_x=0, n_y=4, V_min=1), synth.VertexGrid(n_x=4, n_y=4, V_min=0),
                synth.VertexGrid(n_x=4, n_y=4, V_min=1, x_min=1.0, x_max=1.0), synth.VertexGrid(n_x=4096, n_y=4, V_min=1)):
        with pytest.raises(hough.HoughError):
            h.vertices(bad)
    h.close()


# ============================================================ f3: vote variants

def read_all(h):
    res = h.read()
    res["acc"] = h.accumulator_host().copy()
    return res


def assert_same(res, ref):
    assert res["n_votes"] == ref["n_votes"]
    assert res["n_bad_hits"] == ref["n_bad_hits"]
    assert np.array_equal(res["acc"], ref["acc"])
    assert res["n_peaks"] == ref["n_peaks"]
    assert np.array_equal(res["peak_bin"], ref["peak_bin"])
    assert np.array_equal(res["peak_mask"], ref["peak_mask"])
    assert res["n_hit_entries"] == ref["n_hit_entries"]
    assert np.array_equal(res["hit_offset"], ref["hit_offset"])
    assert np.array_equal(res["hit_index"], ref["hit_index"])


@pytest.mark.parametrize("n_phi,n_rho,tile,n_hits,n_layers,seed", [
    (48, 32, 0, 300, 10, 0),
    (200, 64, 7, 1200, 10, 1),     # ragged phi slabs, several chunks
    (64, 96, 0, 600, 20, 2),       # more than 16 layers: unpacked tile
])
def test_line_transform_random(hough, oracle, n_phi, n_rho, tile, n_hits, n_layers, seed):
    rng = np.random.default_rng(seed)
    g = synth.Grid(n_phi=n_phi, n_d0=1, n_kappa=n_rho, L_min=3, d0_min=0.0, d0_max=0.0, kappa_min=-30.0,
                   kappa_max=45.0, layer_radii=tuple(float(3 + 4 * l) for l in range(n_layers)))
    x, y, layer = random_hits(rng, n_hits, n_layers=n_layers)
    layer[::17] = n_layers + 3  # some bad layers
    ref = oracle.run_variant(g, oracle.MODE_LINE, x, y, layer)
    assert ref["n_peaks"] > 5
    h = make(hough, g, x, y, layer, 1 << 16, 1 << 20, options=hough.OPT_LINE, tile_phi=tile)
    assert_same(read_all(h), ref)
    h.close()


def test_line_transform_toy_detector(hough, oracle):
    """The paper's own workload: the toy detector of PAPER.md:124 with straight tracks (Fig. 3)."""
    g = synth.TOY_LINE_GRID
    for spec, seed in ((synth.TOY_LINE_SPEC, 0), (synth.TOY_LINE_SPEC_5000, 1)):
        x, y, layer, truth = synth.generate_line_event(spec, seed)
        ref = oracle.run_variant(g, oracle.MODE_LINE, x, y, layer)
        h = make(hough, g, x, y, layer, 1 << 16, 1 << 20, options=hough.OPT_LINE)
        assert_same(read_all(h), ref)
        h.close()


def test_line_transform_needs_two_parameters(hough):
    g = synth.Grid(n_phi=16, n_d0=4, n_kappa=32, L_min=2)
    with pytest.raises(hough.HoughError):
        hough.Hough(g, 10, 10, 10, options=hough.OPT_LINE)
    g2 = synth.Grid(n_phi=16, n_d0=1, n_kappa=32, L_min=2, d0_min=0.0, d0_max=0.0)
    with pytest.raises(hough.HoughError):
        hough.Hough(g2, 10, 10, 10, options=hough.OPT_LINE | hough.OPT_INTERVAL)


@pytest.mark.parametrize("shape,tile,n_hits,n_layers,seed", [
    ((40, 4, 64), (0, 0), 200, 10, 0),
    ((50, 13, 64), (8, 4), 700, 10, 1),
    ((33, 9, 256), (4, 8), 300, 24, 2),    # unpacked tile
    ((64, 1, 128), (0, 0), 400, 10, 3),    # 2-parameter transform through the origin
])
def test_interval_voting_random(hough, oracle, shape, tile, n_hits, n_layers, seed):
    rng = np.random.default_rng(seed)
    d0 = dict(d0_min=0.0, d0_max=0.0) if shape[1] == 1 else {}
    g = synth.Grid(n_phi=shape[0], n_d0=shape[1], n_kappa=shape[2], L_min=4,
                   layer_radii=tuple(float(3 + 3 * l) for l in range(n_layers)), **d0)
    x, y, layer = random_hits(rng, n_hits, n_layers=n_layers)
    x[5], y[5] = np.float32(np.nan), np.float32(1.0)
    x[6], y[6] = np.float32(np.inf), np.float32(2.0)
    x[7], y[7] = np.float32(0.0), np.float32(0.0)
    ref = oracle.run_variant(g, oracle.MODE_INTERVAL, x, y, layer)
    assert ref["n_peaks"] > 0 and ref["n_votes"] > 5 * n_hits
    h = make(hough, g, x, y, layer, 1 << 18, 1 << 22, options=hough.OPT_INTERVAL, tile_phi=tile[0], tile_d0=tile[1])
    assert_same(read_all(h), ref)
    h.close()


def test_interval_voting_displaced3d(hough, oracle):
    """BASELINE.json configs[1] under interval voting, everything at full size: accumulator, n_votes, peaks
    and the whole CSR (the oracle's cell-wise lists; its peak-by-peak pass, O(peaks x hits), confirms them
    on the first 4096 peaks)."""
    w = synth.WORKLOADS["displaced3d"]
    x, y, layer, _ = synth.generate_event(w.event, w.seeds[0])
    acc, n_votes, n_bad = oracle.vote_variant(w.grid, oracle.MODE_INTERVAL, x, y, layer)
    pb, pm, n_peaks = oracle.peaks(w.grid, acc)
    h = make(hough, w.grid, x, y, layer, 1 << 22, 1 << 26, options=hough.OPT_INTERVAL)
    res = read_all(h)
    assert res["flags"] == 0
    assert res["n_votes"] == n_votes and np.array_equal(res["acc"], acc)
    assert res["n_peaks"] == n_peaks and np.array_equal(res["peak_bin"], pb) and np.array_equal(res["peak_mask"], pm)
    coff, cidx, ctot = oracle.hitlists_variant(w.grid, oracle.MODE_INTERVAL, x, y, layer, pb, cap_hits=1 << 26,
                                               by_cell=True)
    assert res["n_hit_entries"] == ctot <= 1 << 26
    assert np.array_equal(res["hit_offset"], coff) and np.array_equal(res["hit_index"], cidx)
    m = min(4096, n_peaks)
    off, idx, tot = oracle.hitlists_variant(w.grid, oracle.MODE_INTERVAL, x, y, layer, pb[:m])
    assert np.array_equal(coff[:m + 1], off) and np.array_equal(cidx[:tot], idx)
    h.close()


# ============================================================ f2: hough_fit (E4 fit, E5 selection + duplicates)
#
# Tolerance: the GPU sums the moments in the oracle's order without contraction,
# so they are bit-identical; the only difference is the last bits of atan2 / sin / cos (CUDA vs host
# libm, <= 2 ulp each = 4.4e-16 on sin(phi), cos(phi)), which enter every parameter multiplied by at
# most |m| ~ 80 cm (d0: mx sin - my cos), |u| ~ 80 cm (residuals), Cxr/Crr ~ 0.1 /cm (kappa).
FIT_TOL = {"kappa": 1e-15, "phi0": 4e-15, "d0": 5e-13, "rms": 5e-14}


def assert_fit_same(hough, oracle, res, x, y, g, rms_max, min_shared, exact_flags=True):
    fit, status = oracle.fit_all(x, y, res["hit_offset"], res["hit_index"])
    assert g["n_fitted"] == res["n_peaks"]
    assert np.array_equal(g["status"], status)
    assert g["n_ok"] == int((status == 0).sum()) and g["n_truncated"] == 0
    for k, tol in FIT_TOL.items():
        d = np.abs(g[k] - fit[k])
        if k == "phi0":
            d = np.minimum(d, np.abs(d - 2 * math.pi))  # a fit at +-pi may land on either side
        assert float(d.max(initial=0.0)) <= tol, (k, float(d.max()))
    # E5 is integer work given the rms values: the oracle's rule on the GPU's own fit must give the
    # GPU's flags bit for bit ...
    gfit = np.zeros(len(status), oracle.FIT_DTYPE)
    for k in FIT_TOL:
        gfit[k] = g[k]
    flags_g = oracle.select_dedup(res["hit_offset"], res["hit_index"], res["peak_mask"], len(x), gfit, status,
                                  rms_max, min_shared)
    assert np.array_equal(g["flag"], flags_g)
    # ... and the oracle's flags on its own fit agree wherever no rms comparison is a near-tie
    flags = oracle.select_dedup(res["hit_offset"], res["hit_index"], res["peak_mask"], len(x), fit, status,
                                rms_max, min_shared)
    if exact_flags:
        assert np.array_equal(g["flag"], flags)
    else:
        assert int((g["flag"] != flags).sum()) <= max(2, len(flags) // 200)
    kept = np.nonzero(g["flag"] == 1)[0].astype(np.uint32)
    assert np.array_equal(g["kept"], kept)
    assert g["n_selected"] == int((g["flag"] != 0).sum())
    assert g["n_kept"] == len(kept) and g["n_duplicates"] == int((g["flag"] == 2).sum())
    return fit, status, flags


@pytest.mark.parametrize("shape,n_hits,L_min,rms_max,min_shared,seed", [
    ((64, 16, 32), 400, 3, 5.0, 2, 0),            # random combinations: most lists have 3..5 hits
    ((64, 16, 32), 400, 3, float("inf"), 1, 0),   # every fit selected, one shared hit is enough
    ((50, 13, 64), 700, 2, 0.5, 3, 1),            # lists of 2 hits: status 1
    ((40, 4, 32), 3000, 6, 2.0, 4, 2),            # long lists (more than the 64 cached hits)
])
def test_fit_random_small(hough, oracle, shape, n_hits, L_min, rms_max, min_shared, seed):
    rng = np.random.default_rng(seed)
    g = synth.Grid(n_phi=shape[0], n_d0=shape[1], n_kappa=shape[2], L_min=L_min)
    x, y, layer = random_hits(rng, n_hits)
    h = make(hough, g, x, y, layer, 1 << 16, 1 << 21)
    res = h.read()
    assert res["n_peaks"] > 50 and res["flags"] == 0
    for rep in range(2):  # repeatable on the same handle
        h.fit(rms_max, min_shared)
        # 3-hit lists fit exactly (rms = rounding noise ~1e-16), so their rms order is a coin toss
        # between math libraries: near-ties are expected here, not in the physics workloads below
        fit, status, flags = assert_fit_same(hough, oracle, res, x, y, h.read_fit(), rms_max, min_shared,
                                             exact_flags=False)
    assert {1, 2} <= set(flags.tolist())
    h.close()


@pytest.mark.parametrize("name,seed", [("prompt2d", 0), ("displaced3d", 0), ("displaced3d", 4), ("pileup", 0)])
def test_fit_workloads(hough, oracle, name, seed):
    """BASELINE.json configs[0..2]: every peak fitted, tracks selected at rms <= 100 um, duplicates
    (mirror twins, plateau neighbours) removed when they share >= 3 hits with a better candidate."""
    w = synth.WORKLOADS[name]
    x, y, layer, _ = synth.generate_event(w.event, seed)
    h = make(hough, w.grid, x, y, layer, w.cap_peaks, w.cap_hits)
    res = h.read()
    h.fit(0.01, 3)
    g = h.read_fit()
    fit, status, flags = assert_fit_same(hough, oracle, res, x, y, g, 0.01, 3)
    assert g["n_kept"] > 0 and g["n_duplicates"] > 0
    h.close()


def test_fit_everything_selected_on_a_pileup_event(hough, oracle):
    """rms_max = 1 mm selects every candidate of a pile-up event (the bins are that small): 4.4e8 pairs
    of candidates are examined by the duplicate rule."""
    w = synth.WORKLOADS["pileup"]
    x, y, layer, _ = synth.generate_event(w.event, 1)
    h = make(hough, w.grid, x, y, layer, w.cap_peaks, w.cap_hits)
    res = read_all(h)
    # the oracle's fit below is fed with lists that are the ORACLE's too: the whole event is compared first
    ref = oracle.run(w.grid, x, y, layer, cap_hits=w.cap_hits, by_cell=True)
    res["acc"] = res["acc"].reshape(ref["acc"].shape)
    assert_same(res, ref)
    h.fit(0.1, 5)
    g = h.read_fit()
    assert_fit_same(hough, oracle, ref, x, y, g, 0.1, 5)
    assert g["n_selected"] == res["n_peaks"] and g["n_pair_tests"] > 10**8
    h.close()


def test_fit_mirror_twins_and_truncated_lists(hough, oracle):
    g = synth.Grid(n_phi=64, n_d0=8, n_kappa=32, L_min=8)
    x, y, layer = synth.single_track_event(g, 9, 5, 0.004)
    h = make(hough, g, x, y, layer, 1 << 10, 1 << 14)
    res = h.read()
    h.fit(0.01, 5)
    gf = h.read_fit()
    full = [p for p in range(res["n_peaks"]) if int(res["hit_offset"][p + 1] - res["hit_offset"][p]) == len(x)]
    a, b = full[0], full[-1]
    for k in FIT_TOL:  # exact sign flips: the twins fit bit-identically on the GPU too
        assert gf[k][a] == gf[k][b]
    assert gf["flag"][a] == 1 and gf["flag"][b] == 2
    h.close()
    # hit capacity smaller than the lists: peaks whose list is cut are status 3 and never selected
    rng = np.random.default_rng(3)
    g2 = synth.Grid(n_phi=64, n_d0=16, n_kappa=32, L_min=3)
    x, y, layer = random_hits(rng, 400)
    ref = oracle.run(g2, x, y, layer)
    cap = int(ref["n_hit_entries"]) // 2
    h = make(hough, g2, x, y, layer, 1 << 16, cap)
    res = h.read()
    assert res["flags"] & hough.TRUNCATED_HITS
    h.fit(5.0, 2)
    gf = h.read_fit()
    complete = ref["hit_offset"][1:] <= cap
    assert np.array_equal(gf["status"] == 3, ~complete) and gf["n_truncated"] == int((~complete).sum())
    m = int(complete.sum())  # lists are complete while they fit: the first m peaks, as without the cut
    fit, status = oracle.fit_all(x, y, ref["hit_offset"][:m + 1], ref["hit_index"])
    assert np.array_equal(gf["status"][:m], status)
    assert float(np.abs(gf["rms"][:m] - fit["rms"]).max()) <= FIT_TOL["rms"]
    assert not gf["flag"][m:].any()
    h.close()


def test_fit_no_peaks_and_bad_arguments(hough):
    g = synth.Grid(n_phi=16, n_d0=4, n_kappa=32, L_min=9)
    x, y, layer = random_hits(np.random.default_rng(0), 20)
    h = make(hough, g, x, y, layer, 1 << 10, 1 << 12)
    assert h.read()["n_peaks"] == 0
    h.fit(0.01, 3)
    gf = h.read_fit()
    assert gf["n_fitted"] == 0 and gf["n_kept"] == 0 and len(gf["kept"]) == 0
    for bad in ((-1.0, 3), (float("nan"), 3), (0.01, 0)):
        with pytest.raises(hough.HoughError):
            h.fit(*bad)
    h.close()
