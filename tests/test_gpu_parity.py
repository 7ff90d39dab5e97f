"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit for bit.

Every test drives libhough_b200.so through paper_1305_4855_b200.hough (ctypes marshalling
only) and compares accumulator masks, vote count, peak list and CSR hit lists with
oracle/ on the same seeded inputs (BASELINE.json north_star: "GPU results must match the
oracle bit-exactly (accumulator masks, peak list, hit lists)").
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


def run_gpu(hough, grid, x, y, layer, cap_peaks, cap_hits, **kw):
    h = hough.Hough(grid, max_hits=max(len(x), 1), cap_peaks=cap_peaks, cap_hits=cap_hits, **kw)
    h.vote(dev(x.astype(np.float32)), dev(y.astype(np.float32)), dev(layer.astype(np.int32)))
    h.peaks()
    res = h.read()
    res["acc"] = h.accumulator_host().copy()
    res["query"] = h.query()
    h.close()
    return res


def assert_same(res, ref, lists=True):
    assert not (res.get("flags", 0) & 8)             # HOUGH_LIST_MISMATCH (only ever set under OPT_CHECK_LISTS)
    assert res["n_votes"] == ref["n_votes"]
    assert res["n_bad_hits"] == ref["n_bad_hits"]
    assert np.array_equal(res["acc"], ref["acc"])
    assert res["n_peaks"] == ref["n_peaks"]
    assert np.array_equal(res["peak_bin"], ref["peak_bin"])
    assert np.array_equal(res["peak_mask"], ref["peak_mask"])
    if lists:
        assert res["n_hit_entries"] == ref["n_hit_entries"]
        assert np.array_equal(res["hit_offset"], ref["hit_offset"])
        assert np.array_equal(res["hit_index"], ref["hit_index"])


def random_hits(rng, n, n_layers=10, rmax=80.0):
    r = rng.uniform(0.5, rmax, n)
    phi = rng.uniform(-math.pi, math.pi, n)
    return ((r * np.cos(phi)).astype(np.float32), (r * np.sin(phi)).astype(np.float32),
            rng.integers(0, n_layers, n).astype(np.int32))


# ------------------------------------------------------------------ small grids, ragged tiles
@pytest.mark.parametrize("shape,tile,n_hits,seed", [
    ((8, 4, 32), (0, 0), 20, 0),          # one tile, phi slab wider than a quarter turn
    ((50, 13, 64), (8, 4), 700, 1),       # ragged in phi0 and d0, several chunks
    ((37, 5, 96), (6, 2), 1300, 2),       # n_kappa not a multiple of 64 (smaller swizzle)
    ((64, 1, 128), (16, 1), 300, 3),      # 2-D transform (n_d0 = 1)
    ((96, 24, 32), (32, 8), 513, 4),      # smallest row, hits = chunk + 1
    ((33, 9, 256), (4, 8), 100, 5),
])
# default, NO_CULL, EXACT_ONLY, LIST_SWEEP, both, FUSED_PEAKS, FUSED_PEAKS | NO_CULL, CELL_PEAKS
@pytest.mark.parametrize("options", [0, 1, 8, 16, 24, 128, 129, 256])
def test_random_hits_small_grids(hough, oracle, shape, tile, n_hits, seed, options):
    rng = np.random.default_rng(seed)
    d0 = dict(d0_min=0.0, d0_max=0.0) if shape[1] == 1 else {}
    grid = synth.Grid(n_phi=shape[0], n_d0=shape[1], n_kappa=shape[2], L_min=3, **d0)
    x, y, layer = random_hits(rng, n_hits)
    ref = oracle.run(grid, x, y, layer)
    res = run_gpu(hough, grid, x, y, layer, cap_peaks=grid.n_bins // 2 + 1,
                  cap_hits=max(ref["n_hit_entries"], 1) + 5, tile_phi=tile[0], tile_d0=tile[1],
                  options=options)
    assert_same(res, ref)


def test_no_wrap_and_asymmetric_kappa_range(hough, oracle):
    rng = np.random.default_rng(11)
    grid = synth.Grid(n_phi=40, n_d0=6, n_kappa=64, L_min=2, phi_min=-1.0, phi_max=2.0,
                      d0_min=-3.0, d0_max=7.0, kappa_min=-0.002, kappa_max=0.02, phi_wrap=0)
    x, y, layer = random_hits(rng, 900)
    ref = oracle.run(grid, x, y, layer)
    res = run_gpu(hough, grid, x, y, layer, cap_peaks=grid.n_bins // 2 + 1,
                  cap_hits=ref["n_hit_entries"] + 1, tile_phi=8, tile_d0=4)
    assert_same(res, ref)


def test_fused_peaks_needs_packed_tiles(hough):
    g = synth.Grid(n_phi=16, n_d0=4, n_kappa=32, L_min=2, layer_radii=tuple(float(3 + l) for l in range(20)))
    with pytest.raises(hough.HoughError):
        hough.Hough(g, 10, 10, 10, options=hough.OPT_FUSED_PEAKS)
    g = synth.Grid(n_phi=16, n_d0=4, n_kappa=32, L_min=2)
    with pytest.raises(hough.HoughError):
        hough.Hough(g, 10, 10, 10, options=hough.OPT_FUSED_PEAKS | hough.OPT_UNPACKED)


def test_more_than_16_layers_uses_unpacked_tiles(hough, oracle):
    rng = np.random.default_rng(12)
    radii = tuple(3.0 + 3.0 * i for i in range(24))
    grid = synth.Grid(n_phi=48, n_d0=10, n_kappa=64, L_min=4, layer_radii=radii)
    x, y, layer = random_hits(rng, 1500, n_layers=24)
    ref = oracle.run(grid, x, y, layer)
    res = run_gpu(hough, grid, x, y, layer, cap_peaks=grid.n_bins // 2 + 1,
                  cap_hits=ref["n_hit_entries"] + 1)
    assert_same(res, ref)


# ------------------------------------------------------------------ degenerate inputs
def test_empty_event(hough, oracle):
    grid = synth.Grid(n_phi=16, n_d0=4, n_kappa=32, L_min=1)
    e = np.zeros(0, np.float32)
    res = run_gpu(hough, grid, e, e, np.zeros(0, np.int32), cap_peaks=8, cap_hits=8)
    assert res["n_votes"] == 0 and res["n_peaks"] == 0 and res["n_hit_entries"] == 0
    assert not res["acc"].any() and res["hit_offset"].tolist() == [0]


def test_bad_layers_and_non_finite_hits(hough, oracle):
    rng = np.random.default_rng(13)
    grid = synth.Grid(n_phi=32, n_d0=8, n_kappa=64, L_min=2)
    x, y, layer = random_hits(rng, 400)
    layer[::7] = -1
    layer[3::11] = 10
    x[5] = np.nan
    y[6] = np.inf
    x[8] = -np.inf
    x[9] = 3.0e19            # x*x overflows: den = inf, kappa = 0 -> a legal vote
    x[10], y[10] = 0.0, 0.0  # hit at the origin
    # finite coordinates up to FLT_MAX still vote (r2 = inf => den = inf => kappa = +-0)
    x[12] = 3.2e38
    y[13] = -3.3e38
    x[14], y[14] = np.float32(3.4028234e38), np.float32(-3.4028234e38)
    x[15], y[15] = 1.0e19, 1.7e19      # r2 finite but huge
    layer[[9, 12, 13, 14, 15]] = [1, 2, 3, 4, 5]
    ref = oracle.run(grid, x, y, layer)
    assert ref["n_bad_hits"] > 0
    # the huge finite hits really vote in the oracle (so a cull that drops them is caught)
    solo = oracle.run(grid, x[12:15], y[12:15], layer[12:15])
    assert solo["n_votes"] > 0
    for opt in (0, 1):
        res = run_gpu(hough, grid, x, y, layer, cap_peaks=grid.n_bins // 2 + 1,
                      cap_hits=ref["n_hit_entries"] + 1, tile_phi=8, tile_d0=4, options=opt | hough.OPT_CHECK_LISTS)
        assert_same(res, ref)
    res = run_gpu(hough, grid, x, y, layer, cap_peaks=grid.n_bins // 2 + 1,
                  cap_hits=ref["n_hit_entries"] + 1)
    assert_same(res, ref)


def test_hits_at_the_point_of_closest_approach(hough, oracle):
    """den = |X - P0|^2 ~ 0: the quotient is ill-conditioned and the cull must stay a superset."""
    grid = synth.Grid(n_phi=64, n_d0=16, n_kappa=64, L_min=1)
    phic = grid.phi_min + (np.arange(grid.n_phi) + 0.5) * (grid.phi_max - grid.phi_min) / grid.n_phi
    d0c = grid.d0_min + (np.arange(grid.n_d0) + 0.5) * (grid.d0_max - grid.d0_min) / grid.n_d0
    rng = np.random.default_rng(14)
    xs, ys = [], []
    for _ in range(600):
        i, j = rng.integers(0, grid.n_phi), rng.integers(0, grid.n_d0)
        d = d0c[j] + rng.normal(0, 1e-4)
        t = rng.normal(0, 1e-3)
        xs.append(-d * math.sin(phic[i]) + t * math.cos(phic[i]))
        ys.append(d * math.cos(phic[i]) + t * math.sin(phic[i]))
    x, y = np.asarray(xs, np.float32), np.asarray(ys, np.float32)
    layer = rng.integers(0, 10, len(x)).astype(np.int32)
    ref = oracle.run(grid, x, y, layer)
    for opt in (0, 1):
        res = run_gpu(hough, grid, x, y, layer, cap_peaks=grid.n_bins // 2 + 1,
                      cap_hits=ref["n_hit_entries"] + 1, tile_phi=4, tile_d0=2, options=opt | hough.OPT_CHECK_LISTS)
        assert_same(res, ref)


def test_truncation_is_deterministic(hough, oracle):
    rng = np.random.default_rng(15)
    grid = synth.Grid(n_phi=32, n_d0=8, n_kappa=64, L_min=2)
    x, y, layer = random_hits(rng, 800)
    ref = oracle.run(grid, x, y, layer)
    assert ref["n_peaks"] > 40
    cap_p = 25
    full_len = int(ref["hit_offset"][cap_p])
    cap_h = int(ref["hit_offset"][cap_p - 5]) + 1      # cuts inside list cap_p-5
    res = run_gpu(hough, grid, x, y, layer, cap_peaks=cap_p, cap_hits=cap_h)
    assert res["flags"] == 3 and res["n_peaks"] == ref["n_peaks"]
    assert np.array_equal(res["peak_bin"], ref["peak_bin"][:cap_p])
    assert np.array_equal(res["peak_mask"], ref["peak_mask"][:cap_p])
    assert res["n_hit_entries"] == full_len
    assert np.array_equal(res["hit_offset"], ref["hit_offset"][:cap_p + 1])
    whole = int(ref["hit_offset"][cap_p - 5])           # lists that fit completely
    assert np.array_equal(res["hit_index"][:whole], ref["hit_index"][:whole])


@pytest.mark.parametrize("options", [0, 256, 128])  # streaming sweep, cell-wise kernel, (fused: falls back to the sweep)
def test_peak_rule_on_handmade_accumulators(hough, oracle, options):
    """Plateaus, ties, edges and phi wrap, through hough_set_accumulator + hough_peaks_only."""
    rng = np.random.default_rng(16)
    for (shape, wrap, L_min, dens) in [((6, 5, 32), 1, 1, 0.5), ((6, 5, 32), 0, 2, 0.9),
                                       ((3, 1, 64), 1, 1, 0.3), ((20, 17, 32), 1, 3, 1.0),
                                       ((5, 30, 64), 0, 1, 0.05)]:
        d0 = dict(d0_min=0.0, d0_max=0.0) if shape[1] == 1 else {}
        grid = synth.Grid(n_phi=shape[0], n_d0=shape[1], n_kappa=shape[2], L_min=L_min,
                          phi_wrap=wrap, **d0)
        for variant in range(3):
            acc = rng.integers(0, 1 << 10, grid.n_bins, dtype=np.uint32)
            acc[rng.random(grid.n_bins) > dens] = 0
            if variant == 1:
                acc[:] = 0x3ff                       # all equal: only lin 0 is a peak
            if variant == 2:
                acc &= 0x7                           # few distinct popcounts: many ties
            pb, pm, n = oracle.peaks(grid, acc)
            h = hough.Hough(grid, max_hits=1, cap_peaks=grid.n_bins, cap_hits=1, options=options)
            h.set_accumulator(dev(acc.view(np.int32)))
            h.peaks(lists=False)
            res = h.read(lists=False)
            h.close()
            assert res["n_peaks"] == n
            assert np.array_equal(res["peak_bin"], pb) and np.array_equal(res["peak_mask"], pm)


def test_repeat_runs_are_bit_identical(hough):
    """The race test of PAPER.md:126: OR of masks is order independent."""
    w = synth.WORKLOADS["displaced3d"]
    x, y, layer, _ = synth.generate_event(w.event, 3)
    h = hough.Hough(w.grid, len(x), w.cap_peaks, w.cap_hits)
    dx, dy, dl = dev(x), dev(y), dev(layer)
    outs = []
    for _ in range(3):
        h.vote(dx, dy, dl)
        h.peaks()
        r = h.read()
        outs.append((h.accumulator_host().copy(), r["n_votes"], r["peak_bin"].copy(),
                     r["hit_offset"].copy(), r["hit_index"].copy()))
    h.close()
    for o in outs[1:]:
        assert o[1] == outs[0][1]
        for a, b in zip(o, outs[0]):
            if isinstance(a, np.ndarray):
                assert np.array_equal(a, b)


# ------------------------------------------------------------------ the BASELINE.json configs
@pytest.mark.parametrize("name", ["prompt2d", "displaced3d", "pileup"])
def test_baseline_configs_full_parity(hough, oracle, name):
    w = synth.WORKLOADS[name]
    x, y, layer, _ = synth.generate_event(w.event, w.seeds[0])
    ref = oracle.run(w.grid, x, y, layer)
    res = run_gpu(hough, w.grid, x, y, layer, cap_peaks=w.cap_peaks, cap_hits=w.cap_hits)
    assert res["flags"] == 0
    assert_same(res, ref)


@pytest.mark.parametrize("name,options", [("displaced3d", 8), ("displaced3d", 16), ("pileup", 16 | 8),
                                          ("prompt2d", 128), ("displaced3d", 128), ("pileup", 128),
                                          ("displaced3d", 256), ("pileup", 256)])
def test_baseline_configs_alternative_paths(hough, oracle, name, options):
    """The same results from the alternative code paths the options select: exact recipe only
    (HOUGH_OPT_EXACT_ONLY: no fixed-point fast path), hit lists by a second sweep
    (HOUGH_OPT_LIST_SWEEP) instead of the peak-driven lists, peak flags fused into the vote tile
    plus the tile-edge pass (HOUGH_OPT_FUSED_PEAKS), peak flags by the cell-wise kernel
    (HOUGH_OPT_CELL_PEAKS)."""
    w = synth.WORKLOADS[name]
    x, y, layer, _ = synth.generate_event(w.event, w.seeds[0])
    ref = oracle.run(w.grid, x, y, layer)
    res = run_gpu(hough, w.grid, x, y, layer, cap_peaks=w.cap_peaks, cap_hits=w.cap_hits, options=options)
    assert res["flags"] == 0
    assert_same(res, ref)


def test_process_host_matches_device_path(hough, oracle):
    w = synth.WORKLOADS["displaced3d"]
    x, y, layer, _ = synth.generate_event(w.event, 1)
    ref = oracle.run(w.grid, x, y, layer)
    h = hough.Hough(w.grid, len(x), w.cap_peaks, w.cap_hits)
    res = h.process_host(x, y, layer)
    res["acc"] = h.accumulator_host().copy()
    h.close()
    assert_same(res, ref)


def test_batch_all_100_events_back_to_back_on_one_handle(hough, oracle):
    """BASELINE.json configs[3]: 100 events shaped like "pileup" (seeds 0..99), one handle, one
    stream, each with its own accumulator.  EVERY seed: whole accumulator, n_votes, n_bad_hits,
    peak list and masks, and the whole CSR (hit_offset, hit_index, n_hit_entries) against the oracle
    ("CSR hit lists equal ... config 4: all 100 seeds")."""
    w = synth.WORKLOADS["batch100"]
    assert w.seeds == tuple(range(100))
    h = hough.Hough(w.grid, 20000, w.cap_peaks, w.cap_hits)
    for seed in w.seeds:
        x, y, layer, _ = synth.generate_event(w.event, seed)
        h.vote(dev(x), dev(y), dev(layer))
        h.peaks()
        res = h.read()
        res["acc"] = h.accumulator_host()
        assert res["flags"] == 0, seed
        # the whole CSR of every seed: the oracle's lists walked cell by cell (one vote pass); on seed 0 the
        # peak-by-peak oracle (O(n_peaks x n_hits), minutes) confirms the cell-wise one at this size
        ref = oracle.run(w.grid, x, y, layer, cap_hits=w.cap_hits, by_cell=True)
        assert ref["n_hit_entries"] <= w.cap_hits
        if seed == 0:
            off1, idx1, tot1 = oracle.hitlists(w.grid, x, y, layer, ref["peak_bin"])
            assert tot1 == ref["n_hit_entries"]
            assert np.array_equal(off1, ref["hit_offset"]) and np.array_equal(idx1, ref["hit_index"])
        res["acc"] = res["acc"].reshape(ref["acc"].shape)
        assert_same(res, ref)
        # CSR consistency for every seed: n_hit_entries = sum of list lengths, OR of the
        # listed hits' layer bits = the peak's mask
        off = res["hit_offset"].astype(np.int64)
        assert off[0] == 0 and np.all(np.diff(off) > 0) and off[-1] == res["n_hit_entries"]
        bits = (np.uint32(1) << layer[res["hit_index"]].astype(np.uint32)).astype(np.uint32)
        assert np.array_equal(np.bitwise_or.reduceat(bits, off[:-1]), res["peak_mask"]), seed
    h.close()


def test_finegrid_full_accumulator_parity(hough, oracle):
    """BASELINE.json configs[4] at full size (134M bins, ~62k hits), in bench.py's launch
    configuration: the WHOLE 512 MiB accumulator, n_votes and n_bad_hits against the oracle's
    vote (1.6e10 evaluations: tens of seconds on the host cores); the whole peak list and masks
    against the oracle's peak rule on the ORACLE's accumulator; the whole CSR (every list of the
    ~3.6e6 peaks and n_hit_entries) against the oracle's cell-wise hit lists, which the
    peak-by-peak oracle (O(n_peaks x n_hits), infeasible in full here) confirms on 3000 sampled
    peaks plus the first and last 50.  Also the properties that hold at any size: offsets
    strictly increasing, ascending hit indices inside each list, OR of the listed hits' layer
    bits = the peak's mask."""
    w = synth.WORKLOADS["finegrid"]
    g = w.grid
    x, y, layer, _ = synth.generate_event(w.event, w.seeds[0])
    h = hough.Hough(g, len(x), w.cap_peaks, w.cap_hits)
    h.vote(dev(x), dev(y), dev(layer))
    h.peaks()
    res = h.read()
    acc = h.accumulator_host().reshape(g.n_phi, g.n_d0, g.n_kappa)
    h.close()
    assert res["flags"] == 0
    ref_acc, ref_votes, ref_bad = oracle.vote(g, x, y, layer)
    assert res["n_votes"] == ref_votes and res["n_bad_hits"] == ref_bad
    assert np.array_equal(acc, ref_acc)
    del acc
    pb, pm, n = oracle.peaks(g, ref_acc)
    del ref_acc
    assert res["n_peaks"] == n
    assert np.array_equal(res["peak_bin"], pb) and np.array_equal(res["peak_mask"], pm)
    off = res["hit_offset"].astype(np.int64)
    idx = res["hit_index"]
    assert off[0] == 0 and np.all(np.diff(off) > 0) and off[-1] == res["n_hit_entries"] == len(idx)
    inner = np.ones(len(idx), bool)
    inner[off[:-1]] = False                      # first entry of every list
    assert np.all(np.diff(idx.astype(np.int64))[inner[1:]] > 0)   # ascending inside each list
    bits = (np.uint32(1) << layer[idx].astype(np.uint32)).astype(np.uint32)
    assert np.array_equal(np.bitwise_or.reduceat(bits, off[:-1]), pm)
    # every list of every peak, and the total, against the oracle's cell-wise lists (one more vote pass) ...
    coff, cidx, ctot = oracle.hitlists_cells(g, x, y, layer, pb, cap_hits=w.cap_hits)
    assert ctot == res["n_hit_entries"] <= w.cap_hits
    assert np.array_equal(res["hit_offset"], coff) and np.array_equal(idx, cidx)
    # ... which the peak-by-peak oracle confirms on a sample at this size
    rng = np.random.default_rng(5)
    sel = np.unique(np.concatenate([rng.integers(0, n, 3000), np.arange(50), np.arange(n - 50, n)]))
    soff, sidx, _tot = oracle.hitlists(g, x, y, layer, pb[sel])
    for q, pk in enumerate(sel):
        assert np.array_equal(cidx[int(coff[pk]):int(coff[pk + 1])], sidx[int(soff[q]):int(soff[q + 1])]), pk
    del coff, cidx
    # the fused peak test (two 256-bin segments per cell row here) and the cell-wise kernel give the
    # same peaks and lists as the path just checked against the oracle
    for opt in (hough.OPT_FUSED_PEAKS, hough.OPT_CELL_PEAKS):
        h = hough.Hough(g, len(x), w.cap_peaks, w.cap_hits, options=opt)
        h.vote(dev(x), dev(y), dev(layer))
        h.peaks()
        alt = h.read()
        h.close()
        assert alt["n_peaks"] == n and alt["n_votes"] == ref_votes and alt["n_hit_entries"] == res["n_hit_entries"]
        assert np.array_equal(alt["peak_bin"], pb) and np.array_equal(alt["peak_mask"], pm)
        assert np.array_equal(alt["hit_offset"], res["hit_offset"]) and np.array_equal(alt["hit_index"], idx)


def test_unpacked_tile_option_with_few_layers(hough, oracle):
    """HOUGH_OPT_UNPACKED: the one-mask-per-word tile layout (used with 17..32 layers) on a
    10-layer detector, with and without the cull."""
    rng = np.random.default_rng(31)
    grid = synth.Grid(n_phi=50, n_d0=13, n_kappa=96, L_min=3)
    x, y, layer = random_hits(rng, 1100)
    ref = oracle.run(grid, x, y, layer)
    for opt in (hough.OPT_UNPACKED, hough.OPT_UNPACKED | hough.OPT_NO_CULL):
        res = run_gpu(hough, grid, x, y, layer, cap_peaks=grid.n_bins // 2 + 1,
                      cap_hits=ref["n_hit_entries"] + 1, options=opt)
        assert_same(res, ref)


def test_submit_collect_pipeline_matches_oracle(hough, oracle):
    """hough_submit_host / hough_collect_host with two events in flight: every event's results
    (copied on the second stream while the next event computes) equal the oracle's."""
    w = synth.WORKLOADS["displaced3d"]
    evs = [synth.generate_event(w.event, s)[:3] for s in (2, 3, 4, 5, 6)]
    refs = [oracle.run(w.grid, *e) for e in evs]
    pins = [[torch.from_numpy(a).pin_memory() for a in e] for e in evs]
    h = hough.Hough(w.grid, max(len(e[0]) for e in evs), w.cap_peaks, w.cap_hits)
    got = []
    for e, pe in enumerate(pins):
        h.submit_host(pe[0].numpy(), pe[1].numpy(), pe[2].numpy(), e & 1)
        if e > 0:
            r = h.collect_host((e - 1) & 1)
            got.append({k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in r.items()})
    r = h.collect_host((len(pins) - 1) & 1)
    got.append({k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in r.items()})
    with pytest.raises(hough.HoughError):
        h.collect_host(0)          # nothing submitted in that slot any more
    # the optional 16-bit copy of the lists holds the same entries as the 32-bit array
    d, hb, _out, _host = h._slot(0)
    n_e = int(hb["counts"].numpy().view(hough.COUNTS_DTYPE)[0]["n_hit_entries"])
    assert n_e > 0 and np.array_equal(d["hit_index"][:n_e].cpu().numpy().view(np.uint32),
                                      d["hit_index16"][:n_e].cpu().numpy().view(np.uint16))
    h.close()
    for res, ref in zip(got, refs):
        assert res["n_votes"] == ref["n_votes"] and res["n_peaks"] == ref["n_peaks"]
        assert np.array_equal(res["peak_bin"], ref["peak_bin"])
        assert np.array_equal(res["peak_mask"], ref["peak_mask"])
        assert np.array_equal(res["hit_offset"], ref["hit_offset"])
        assert np.array_equal(res["hit_index"], ref["hit_index"])


def test_three_slot_pipeline_with_pileup_events(hough, oracle):
    """hough_submit_host / hough_collect_begin / hough_collect_end with three events in flight (inputs
    of e+1 on the library's copy-in stream, e computing, results of e-1 on the copy-out stream;
    PAPER.md:128-130), on pile-up events of different sizes; the slot state machine rejects misuse."""
    w = synth.WORKLOADS["pileup"]
    specs = [w.event, dataclasses.replace(w.event, n_prompt=300, n_noise=900), w.event,
             dataclasses.replace(w.event, n_prompt=0, n_displaced=0, n_noise=40), w.event]
    evs = [synth.generate_event(sp, 11 + q)[:3] for q, sp in enumerate(specs)]
    pins = [[torch.from_numpy(a).pin_memory() for a in e] for e in evs]
    h = hough.Hough(w.grid, max(len(e[0]) for e in evs), w.cap_peaks, w.cap_hits)
    got = []

    def keep(r):
        got.append({k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in r.items()})

    n = len(pins)
    for e, pe in enumerate(pins):
        h.submit_host(pe[0].numpy(), pe[1].numpy(), pe[2].numpy(), e % 3)
        if e == 0:
            with pytest.raises(hough.HoughError):
                h.submit_host(pe[0].numpy(), pe[1].numpy(), pe[2].numpy(), 0)   # slot still in flight
            with pytest.raises(hough.HoughError):
                h.collect_end(0)                                                 # not begun
            with pytest.raises(hough.HoughError):
                h.process_host(pe[0].numpy(), pe[1].numpy(), pe[2].numpy())      # would reuse slot 0's staging
        if e > 0:
            h.collect_begin((e - 1) % 3)
        if e > 1:
            keep(h.collect_end((e - 2) % 3))
    h.collect_begin((n - 1) % 3)
    keep(h.collect_end((n - 2) % 3))
    keep(h.collect_end((n - 1) % 3))
    with pytest.raises(hough.HoughError):
        h.collect_begin(1)          # nothing submitted in that slot any more
    with pytest.raises(hough.HoughError):
        h.submit_host(pins[0][0].numpy(), pins[0][1].numpy(), pins[0][2].numpy(), 4)  # no such slot
    h.close()
    assert len(got) == n
    for res, ev in zip(got, evs):
        acc, n_votes, _ = oracle.vote(w.grid, *ev)
        pb, pm, n_peaks = oracle.peaks(w.grid, acc)
        # events of at most 65536 hits come back with their lists as 16-bit indices (hit_index16)
        assert res["n_votes"] == n_votes and res["n_peaks"] == n_peaks and res["flags"] == hough.INDEX16
        assert res["hit_index"].dtype == np.uint16
        assert np.array_equal(res["peak_bin"], pb) and np.array_equal(res["peak_mask"], pm)
        # every hit list (the oracle's cell-wise pass)
        coff, cidx, ctot = oracle.hitlists_cells(w.grid, *ev, pb, cap_hits=w.cap_hits)
        assert res["n_hit_entries"] == ctot <= w.cap_hits
        assert np.array_equal(res["hit_offset"], coff) and np.array_equal(res["hit_index"], cidx)


def test_second_vote_replaces_the_event_and_peaks_can_be_repeated(hough, oracle):
    """Reading B15: a second hough_vote before hough_peaks replaces the event; hough_peaks
    may be called again on the same accumulator and gives the same answer."""
    rng = np.random.default_rng(21)
    grid = synth.Grid(n_phi=48, n_d0=12, n_kappa=64, L_min=2)
    xa, ya, la = random_hits(rng, 900)
    xb, yb, lb = random_hits(rng, 350)
    ref = oracle.run(grid, xb, yb, lb)
    h = hough.Hough(grid, 900, grid.n_bins // 2 + 1, ref["n_hit_entries"] + 1000)
    h.vote(dev(xa), dev(ya), dev(la))
    h.vote(dev(xb), dev(yb), dev(lb))
    evals = []
    for _ in range(2):
        h.peaks()
        res = h.read()
        res["acc"] = h.accumulator_host().copy()
        assert_same(res, ref)
        evals.append(res["n_list_evals"])
    h.close()
    assert evals[0] > 0 and evals[1] == evals[0]      # the work counter of the list stage is per call


def test_an_outlier_radius_does_not_widen_the_list_windows_of_later_events(hough, oracle):
    """The per-layer radius range behind the peak-driven lists' azimuth windows belongs to ONE event: after
    an event with a far-away hit in a valid layer (and after an empty event, which runs no hit preparation),
    an ordinary event costs the list stage exactly what it costs a fresh handle."""
    w = synth.WORKLOADS["displaced3d"]
    x, y, layer, _ = synth.generate_event(w.event, 5)
    ref = oracle.run(w.grid, x, y, layer)

    def run(h, xs, ys, ls):
        h.vote(dev(xs), dev(ys), dev(ls))
        h.peaks()
        r = h.read()
        r["acc"] = h.accumulator_host().copy()
        return r

    fresh = hough.Hough(w.grid, len(x) + 10, w.cap_peaks, w.cap_hits)
    base = run(fresh, x, y, layer)
    fresh.close()
    assert_same(base, ref)
    xo, yo, lo = x.copy(), y.copy(), layer.copy()
    xo[:10], yo[:10] = 1.0e6, -3.0e5                   # finite, indexed (r^2 < 2^80), far outside the detector
    lo[:10] = np.arange(10, dtype=np.int32)            # one in every layer
    z = np.zeros(0, np.float32)
    h = hough.Hough(w.grid, len(x) + 10, w.cap_peaks, w.cap_hits)
    for pattern in ("outlier", "outlier+empty", "two outliers"):
        assert_same(run(h, xo, yo, lo), oracle.run(w.grid, xo, yo, lo))
        if pattern == "outlier+empty":
            assert run(h, z, z, np.zeros(0, np.int32))["n_peaks"] == 0
        if pattern == "two outliers":
            run(h, xo, yo, lo)
        after = run(h, x, y, layer)
        assert_same(after, ref)
        assert after["n_list_evals"] == base["n_list_evals"], pattern
    h.close()


def test_list_check_passes_on_real_lists_and_catches_tampering(hough, oracle):
    """hough_check_lists / HOUGH_OPT_CHECK_LISTS: clean on the lists of displaced3d and pile-up events (all
    three list paths), and HOUGH_LIST_MISMATCH once a list is tampered with: an entry replaced by a hit of
    another layer (the OR of the bits no longer gives the mask), two entries swapped (not ascending), an
    index beyond the event.  A capacity-cut list is not judged."""
    MIS = hough.LIST_MISMATCH
    for name, options in (("displaced3d", 0), ("displaced3d", hough.OPT_LIST_SWEEP), ("displaced3d", hough.OPT_INTERVAL),
                          ("pileup", 0)):
        w = synth.WORKLOADS[name]
        x, y, layer, _ = synth.generate_event(w.event, 4)
        cap_p, cap_h = (1 << 22, 1 << 26) if options == hough.OPT_INTERVAL else (w.cap_peaks, w.cap_hits)
        h = hough.Hough(w.grid, len(x), cap_p, cap_h, options=options | hough.OPT_CHECK_LISTS)
        h.vote(dev(x), dev(y), dev(layer))
        h.peaks()
        res = h.read()
        assert res["n_peaks"] > 0 and res["flags"] & ~hough.INDEX16 == 0, (name, options)
        h.check_lists()                                  # the explicit call agrees
        assert h.read_counts()["flags"] & MIS == 0
        if options:
            h.close()
            continue
        off = res["hit_offset"].astype(np.int64)
        lens = np.diff(off)
        p = int(np.argmax(lens >= 3))                    # a peak with at least three hits
        a = int(off[p])
        orig = h.hit_index[a:a + 3].clone()

        def tampered(values):
            h.peaks()                                    # fresh lists and a fresh flags word
            h.hit_index[a:a + len(values)] = torch.tensor(values, dtype=torch.int32, device=h.device)
            h.check_lists()
            flag = int(h.read_counts()["flags"]) & MIS
            h.hit_index[a:a + 3] = orig
            return flag

        o = [int(v) for v in orig.cpu().numpy()]
        assert tampered(o) == 0
        assert tampered([o[1], o[0]]) == MIS             # not ascending
        assert tampered([o[0], o[0]]) == MIS             # a repeated hit
        assert tampered([len(x) + 5]) == MIS             # no such hit
        # a later hit of a layer the mask does not have, in the third place: the OR gains a bit
        missing = [l for l in range(10) if not (int(res["peak_mask"][p]) >> l) & 1]
        cand = [hh for hh in range(o[1] + 1, len(x)) if layer[hh] in missing]
        if cand:
            assert tampered([o[0], o[1], cand[0]]) == MIS
        h.close()
    # a list cut by cap_hits is skipped, the complete ones before it are still judged
    w = synth.WORKLOADS["displaced3d"]
    x, y, layer, _ = synth.generate_event(w.event, 4)
    h = hough.Hough(w.grid, len(x), w.cap_peaks, 100, options=hough.OPT_CHECK_LISTS)
    h.vote(dev(x), dev(y), dev(layer))
    h.peaks()
    assert h.read()["flags"] == hough.TRUNCATED_HITS
    h.close()


def test_many_kappa_bins_and_single_cell_tiles(hough, oracle):
    """n_kappa = 2048 (a cell row of 4 KB: few cells per tile) and the 1 x 1 tile override."""
    rng = np.random.default_rng(22)
    grid = synth.Grid(n_phi=24, n_d0=6, n_kappa=2048, L_min=2)
    x, y, layer = random_hits(rng, 600)
    ref = oracle.run(grid, x, y, layer)
    for tile in ((0, 0), (1, 1)):
        res = run_gpu(hough, grid, x, y, layer, cap_peaks=grid.n_bins // 2 + 1,
                      cap_hits=ref["n_hit_entries"] + 1, tile_phi=tile[0], tile_d0=tile[1])
        assert_same(res, ref)
    # the largest n_kappa the library accepts: one warp of 8 cells per list CTA
    grid = synth.Grid(n_phi=6, n_d0=2, n_kappa=16384, L_min=1)
    x, y, layer = random_hits(rng, 300)
    ref = oracle.run(grid, x, y, layer)
    res = run_gpu(hough, grid, x, y, layer, cap_peaks=grid.n_bins // 2 + 1,
                  cap_hits=ref["n_hit_entries"] + 1, options=hough.OPT_CHECK_LISTS)
    assert_same(res, ref)


def test_random_configurations_share_the_process(hough, oracle):
    """60 random grids / detectors / tile overrides / hit counts in ONE process, handles created
    and destroyed back to back: besides parity this guards the per-kernel shared-memory limit
    (a small-tile handle must not lower it under a later large-tile one)."""
    for seed in range(60):
        rng = np.random.default_rng(1000 + seed)
        n_phi = int(rng.integers(3, 90))
        n_d0 = int(rng.choice([1, 2, 3, 5, 8, 13, 20, 33, 40]))
        nk = int(rng.choice([32, 64, 96, 128, 160, 256, 512, 1024]))
        nl = int(rng.choice([3, 10, 16, 17, 32]))
        wrap = int(rng.integers(0, 2))
        kw = dict(n_phi=n_phi, n_d0=n_d0, n_kappa=nk, L_min=int(rng.integers(1, min(nl, 4) + 1)),
                  layer_radii=tuple(2.0 + 70.0 * (i + 1) / nl for i in range(nl)), phi_wrap=wrap)
        if n_d0 == 1:
            kw.update(d0_min=0.0, d0_max=0.0)
        elif rng.random() < 0.5:
            kw.update(d0_min=float(rng.uniform(-20, 0)), d0_max=float(rng.uniform(1, 25)))
        if rng.random() < 0.5:
            a = float(rng.uniform(-0.03, 0.01))
            kw.update(kappa_min=a, kappa_max=a + float(rng.uniform(0.002, 0.05)))
        if not wrap or rng.random() < 0.3:
            a = float(rng.uniform(-3, 0))
            kw.update(phi_min=a, phi_max=a + float(rng.uniform(0.5, 6.0)))
        grid = synth.Grid(**kw)
        n = int(rng.choice([0, 1, 31, 200, 513, 1500, 3000]))
        r, ph = rng.uniform(0.3, 80, n), rng.uniform(-math.pi, math.pi, n)
        x, y = (r * np.cos(ph)).astype(np.float32), (r * np.sin(ph)).astype(np.float32)
        layer = rng.integers(-1 if rng.random() < 0.2 else 0, nl + (1 if rng.random() < 0.2 else 0),
                             n).astype(np.int32)
        ref = oracle.run(grid, x, y, layer)
        tile = (0, 0) if rng.random() < 0.5 else (int(rng.integers(1, 20)),
                                                  int(rng.integers(1, min(n_d0, 12) + 1)))
        opts = int(rng.integers(0, 2))          # NO_CULL or not
        peaks_by = int(rng.integers(0, 3))      # streaming sweep, fused (two-masks-per-word tiles only), cell-wise
        opts |= (128 if nl <= 16 else 0) if peaks_by == 1 else 256 if peaks_by == 2 else 0
        opts |= hough.OPT_CHECK_LISTS             # the device-side list invariant rides along
        res = run_gpu(hough, grid, x, y, layer, cap_peaks=grid.n_bins // 2 + 1,
                      cap_hits=max(ref["n_hit_entries"], 1) + 3, tile_phi=tile[0], tile_d0=tile[1],
                      options=opts)
        assert_same(res, ref)


def test_call_patterns_on_one_handle(hough, oracle):
    """Two long-lived handles (default and HOUGH_OPT_LIST_SWEEP) through 80 events of random sizes and
    call patterns -- vote twice, peaks twice, peaks without lists then with, a hand-made accumulator in
    between, the host entry point -- every result against the oracle.  The library keeps its per-event
    scratch clean without memsets (counters double-buffered, k_finish prepares the next calls): this
    is the test of that bookkeeping."""
    rng = np.random.default_rng(77)
    g = synth.Grid(n_phi=96, n_d0=12, n_kappa=64, L_min=4)
    handles = [hough.Hough(g, 4000, g.n_bins // 2 + 1, 1 << 22),
               hough.Hough(g, 4000, g.n_bins // 2 + 1, 1 << 22, options=hough.OPT_LIST_SWEEP)]

    def event():
        n = int(rng.choice([0, 1, 50, 700, 2500, 4000]))
        r, ph = rng.uniform(0.5, 80, n), rng.uniform(-math.pi, math.pi, n)
        return ((r * np.cos(ph)).astype(np.float32), (r * np.sin(ph)).astype(np.float32),
                rng.integers(-1, 11, n).astype(np.int32))

    for it in range(80):
        h = handles[0] if rng.random() < 0.7 else handles[1]
        x, y, layer = event()
        ref = oracle.run(g, x, y, layer)
        pat = int(rng.integers(0, 6))
        if pat == 0:      # a second vote replaces the first
            xa, ya, la = event()
            h.vote(dev(xa), dev(ya), dev(la))
            h.vote(dev(x), dev(y), dev(layer))
            h.peaks()
        elif pat == 1:    # peaks twice
            h.vote(dev(x), dev(y), dev(layer))
            h.peaks()
            h.peaks()
        elif pat == 2:    # without lists, then with
            h.vote(dev(x), dev(y), dev(layer))
            h.peaks(lists=False)
            h.peaks()
        elif pat == 3:    # a hand-made accumulator in between
            acc = rng.integers(0, 1 << 10, g.n_bins, dtype=np.uint32)
            h.set_accumulator(dev(acc.view(np.int32)))
            h.peaks(lists=False)
            pb, _pm, npk = oracle.peaks(g, acc)
            r0 = h.read(lists=False)
            assert r0["n_peaks"] == npk and r0["n_votes"] == 0 and np.array_equal(r0["peak_bin"], pb), it
            h.vote(dev(x), dev(y), dev(layer))
            h.peaks()
        elif pat == 4:    # host entry point
            res = h.process_host(x, y, layer)
            res = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in res.items()}
            res["acc"] = ref["acc"]
            assert_same(res, ref)
            continue
        else:
            h.vote(dev(x), dev(y), dev(layer))
            h.peaks()
        res = h.read()
        res["acc"] = h.accumulator_host()
        assert_same(res, ref)
    for h in handles:
        h.close()
