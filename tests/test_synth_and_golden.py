"""Input generator checks and the oracle regression fixture (CPU only)."""
import hashlib
import json
import math
import os

import numpy as np
import pytest

from paper_1305_4855_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden", "oracle_regression.json")


def test_workload_shapes_match_baseline_configs():
    w = synth.WORKLOADS
    assert (w["prompt2d"].grid.n_phi, w["prompt2d"].grid.n_d0, w["prompt2d"].grid.n_kappa) == (256, 1, 128)
    assert w["prompt2d"].grid.L_min == 8 and w["displaced3d"].grid.L_min == 6
    assert w["displaced3d"].grid.n_bins == 1024 * 64 * 256 == 16777216
    assert w["pileup"].grid.L_min == 7 and w["batch100"].seeds == tuple(range(100))
    assert w["finegrid"].grid.n_bins == 2048 * 128 * 512 == 134217728
    assert synth.LAYER_RADII_CM == (4.4, 7.3, 10.2, 25.5, 34.0, 42.0, 50.0, 60.8, 69.2, 78.0)
    assert abs(synth.KAPPA_PER_INV_PT - 0.0114) < 1e-12     # 0.003 * 3.8 T (reading B11)


@pytest.mark.parametrize("name,lo,hi", [("prompt2d", 240, 251), ("displaced3d", 1540, 1610),
                                        ("pileup", 15300, 15510)])
def test_event_sizes_and_determinism(name, lo, hi):
    w = synth.WORKLOADS[name]
    x, y, layer, truth = synth.generate_event(w.event, 0)
    assert lo <= len(x) <= hi and x.dtype == np.float32 and layer.dtype == np.int32
    x2, y2, l2, _ = synth.generate_event(w.event, 0)
    assert np.array_equal(x, x2) and np.array_equal(y, y2) and np.array_equal(layer, l2)
    x3, _, _, _ = synth.generate_event(w.event, 1)
    assert not np.array_equal(x[:100], x3[:100])
    r = np.hypot(x.astype(np.float64), y.astype(np.float64))
    assert np.allclose(r, np.asarray(synth.LAYER_RADII_CM)[layer], rtol=1e-6)
    assert all(abs(k) <= 0.0114 + 1e-12 for (_, _, k, _) in truth["tracks"])
    for (_, d0, _, nh) in truth["tracks"][w.event.n_prompt:]:
        assert nh == sum(1 for rr in synth.LAYER_RADII_CM if rr > abs(d0) + 2.0)


def test_generated_hits_lie_on_their_circle():
    """Generator geometry (configs[1] hit formula) checked with a distance, not the formula."""
    g = synth.WORKLOADS["displaced3d"].grid
    for (i, j, kappa) in [(10, 50, 0.004), (900, 3, -0.002)]:
        phi0 = g.phi_min + (i + 0.5) * (g.phi_max - g.phi_min) / g.n_phi
        d0 = g.d0_min + (j + 0.5) * (g.d0_max - g.d0_min) / g.n_d0
        x, y, _ = synth.single_track_event(g, i, j, kappa)
        cx, cy = -(d0 + 1 / kappa) * math.sin(phi0), (d0 + 1 / kappa) * math.cos(phi0)
        dist = np.hypot(x.astype(np.float64) - cx, y.astype(np.float64) - cy)
        assert np.allclose(dist, 1 / abs(kappa), rtol=0, atol=2e-4)


def test_oracle_regression_fixture(oracle):
    gold = json.load(open(GOLD))
    w = synth.WORKLOADS["prompt2d"]
    x, y, layer, _ = synth.generate_event(w.event, 0)
    cases = {"prompt2d_seed0": (w.grid, x, y, layer)}
    g = synth.Grid(n_phi=64, n_d0=16, n_kappa=64, L_min=9)
    cases["single_track_64x16x64_i21_j9_k0.0033"] = (g,) + synth.single_track_event(g, 21, 9, 0.0033)
    for name, (grid, x, y, layer) in cases.items():
        rec = gold[name]
        if synth.event_sha256(x, y, layer) != rec["hits_sha256"]:
            pytest.skip("numpy RNG/libm bitstream differs from the one that wrote the fixture")
        r = oracle.run(grid, x, y, layer)
        assert r["n_votes"] == rec["n_votes"]
        assert hashlib.sha256(r["acc"].tobytes()).hexdigest() == rec["acc_sha256"]
        assert r["peak_bin"].tolist() == rec["peak_bin"]
        assert r["peak_mask"].tolist() == rec["peak_mask"]
        assert r["hit_offset"].tolist() == rec["hit_offset"]
        assert r["hit_index"].tolist() == rec["hit_index"]


def test_first_batch_event_digest_is_stable():
    """The inputs bench.py measures are reproducible bit for bit (its JSON line carries the
    SHA-256 of the first event; this pins the generator's draw order and dtype handling)."""
    import bench
    w = synth.WORKLOADS["batch100"]
    e = synth.generate_event(w.event, w.seeds[0])[:3]
    assert bench.input_digest(e) == "6c3d9e0a77886577e984fbb164db541f5f97a879b8efe0c25b6346838d03ea5a"
