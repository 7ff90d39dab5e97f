"""hough_peaks_noalloc: the one entry point for callers that cannot allocate device memory.

A plug-in inside a framework that owns the device-memory budget, a real-time event loop where
cudaMalloc is banned because it synchronises the whole device, or a C client that is only handed
pointers can still find the peaks of an accumulator: this call takes no handle and no workspace, its
scan scratch is a fixed array built into the library's device code (include/hough.h states the limit,
HOUGH_NOALLOC_MAX_BINS, and the rule that overlapping calls on one GPU race on that array).

The GPU tests compare it with the existing path (hough_set_accumulator + hough_peaks_only), bit for bit
as every integer result in this repository, on several calls in a row: the array keeps the previous
call's contents, so a call after a LARGER one is the case that would expose a missing clear.

This file sorts last on purpose (`pytest --collect-only`): `pytest -x` stops at the first failure, and a
failure here must not hide the parity tests.
"""
import os

import numpy as np
import pytest

from paper_1305_4855_b200 import synth

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def hough():
    from paper_1305_4855_b200 import build
    build.build()
    from paper_1305_4855_b200 import hough as hough_mod
    return hough_mod


def test_noalloc_rejects_bad_sizes_before_touching_the_gpu(hough):
    """Argument checks come first, so they can be exercised without a device."""
    import ctypes as C
    f = hough._lib.hough_peaks_noalloc
    p = C.c_void_p(256)                                  # never dereferenced on these paths
    assert hough.NOALLOC_MAX_BINS == 1 << 24
    assert f(p, 2048, 128, 512, 7, 1, p, p, 10, p, None) == hough.HOUGH_ENOMEM   # the fine grid is too big
    assert f(p, 1024, 64, 257, 7, 1, p, p, 10, p, None) == hough.HOUGH_ENOMEM    # just above the limit
    assert f(None, 8, 8, 8, 1, 1, p, p, 10, p, None) == hough.HOUGH_EINVAL
    assert f(p, 8, 8, 8, 1, 1, p, p, 0, p, None) == hough.HOUGH_EINVAL           # cap_peaks = 0
    assert f(p, 2, 8, 8, 1, 1, p, p, 10, p, None) == hough.HOUGH_EINVAL          # wrap needs n_phi >= 3
    assert f(p, 8, 8, 8, 33, 0, p, p, 10, p, None) == hough.HOUGH_EINVAL
    assert f(p, 8, 0, 8, 1, 0, p, p, 10, p, None) == hough.HOUGH_EINVAL


def _existing_path(hough, grid, acc_dev, cap_peaks):
    h = hough.Hough(grid, max_hits=1, cap_peaks=cap_peaks, cap_hits=1)
    h.set_accumulator(acc_dev)
    h.peaks(lists=False)
    res = h.read(lists=False)
    h.close()
    return res


def _noalloc(hough, grid, acc_dev, cap_peaks, stream=None):
    i32 = dict(dtype=torch.int32, device=acc_dev.device)
    pb, pm = torch.full((cap_peaks,), -1, **i32), torch.full((cap_peaks,), -1, **i32)
    n = torch.full((1,), -1, **i32)
    hough.peaks_noalloc(acc_dev, grid.n_phi, grid.n_d0, grid.n_kappa, grid.L_min, grid.phi_wrap, pb, pm, n, stream)
    torch.cuda.synchronize()
    n_true = int(n.cpu().numpy().view(np.uint32)[0])
    k = min(n_true, cap_peaks)
    rest_untouched = bool((pb[k:] == -1).all()) and bool((pm[k:] == -1).all())
    return n_true, pb[:k].cpu().numpy().view(np.uint32), pm[:k].cpu().numpy().view(np.uint32), rest_untouched


def _random_acc(rng, grid, dens, bits):
    acc = rng.integers(0, 1 << bits, grid.n_bins, dtype=np.uint32)
    acc[rng.random(grid.n_bins) > dens] = 0
    return acc


CASES = [  # (n_phi, n_d0, n_kappa), wrap, L_min, density, mask bits; big ones first so later calls see stale scratch
    ((96, 12, 64), 1, 3, 0.6, 10),      # 36 blocks
    ((20, 17, 32), 1, 2, 1.0, 3),       # few distinct popcounts: many ties; 5.3 blocks (ragged tail)
    ((6, 5, 32), 0, 2, 0.9, 10),        # half a block, no wrap
    ((3, 1, 64), 1, 1, 0.3, 10),        # 2-D, the smallest wrapped grid
    ((48, 9, 96), 0, 4, 0.8, 10),       # 20.25 blocks
]


@pytest.mark.gpu
def test_noalloc_equals_existing_path_on_calls_in_a_row(hough):
    rng = np.random.default_rng(2024)
    dev = torch.device("cuda", 0)
    for (shape, wrap, L_min, dens, bits) in CASES:
        d0 = dict(d0_min=0.0, d0_max=0.0) if shape[1] == 1 else {}
        grid = synth.Grid(n_phi=shape[0], n_d0=shape[1], n_kappa=shape[2], L_min=L_min, phi_wrap=wrap, **d0)
        for rep in range(2):                            # two different accumulators, back to back
            acc = _random_acc(rng, grid, dens, bits)
            if rep == 1 and shape == (6, 5, 32):
                acc[:] = 0x3ff                          # all equal: only lin 0 is a peak
            acc_dev = torch.from_numpy(acc.view(np.int32)).to(dev)
            ref = _existing_path(hough, grid, acc_dev, grid.n_bins)
            n, pb, pm, clean = _noalloc(hough, grid, acc_dev, grid.n_bins)
            assert n == ref["n_peaks"], (shape, rep)
            assert np.array_equal(pb, ref["peak_bin"]) and np.array_equal(pm, ref["peak_mask"]), (shape, rep)
            assert clean
            n2, pb2, pm2, _ = _noalloc(hough, grid, acc_dev, grid.n_bins)    # and the very same call again
            assert n2 == n and np.array_equal(pb2, pb) and np.array_equal(pm2, pm)


@pytest.mark.gpu
def test_noalloc_truncates_like_the_existing_path_and_runs_on_a_side_stream(hough):
    rng = np.random.default_rng(7)
    dev = torch.device("cuda", 0)
    grid = synth.Grid(n_phi=64, n_d0=8, n_kappa=64, L_min=2)
    acc = _random_acc(rng, grid, 0.7, 10)
    acc_dev = torch.from_numpy(acc.view(np.int32)).to(dev)
    full = _existing_path(hough, grid, acc_dev, grid.n_bins)
    assert full["n_peaks"] > 100
    cap = 37
    st = torch.cuda.Stream(device=dev)
    n, pb, pm, clean = _noalloc(hough, grid, acc_dev, cap, stream=st)
    assert n == full["n_peaks"] and clean               # the true count, the first `cap` peaks in lin order
    assert np.array_equal(pb, full["peak_bin"][:cap]) and np.array_equal(pm, full["peak_mask"][:cap])


@pytest.mark.gpu
def test_noalloc_at_its_maximum_size(hough):
    """The largest grid the fixed scratch serves: the 1024 x 64 x 256 accumulator of configs 2-4, filled the
    way a pile-up event fills it (mean popcount about 5 of 10 layers), then a small call right after it."""
    w = synth.WORKLOADS["pileup"]
    grid = w.grid
    assert grid.n_bins == hough.NOALLOC_MAX_BINS
    rng = np.random.default_rng(99)
    dev = torch.device("cuda", 0)
    acc = rng.integers(0, 1 << 10, grid.n_bins, dtype=np.uint32)
    acc_dev = torch.from_numpy(acc.view(np.int32)).to(dev)
    ref = _existing_path(hough, grid, acc_dev, w.cap_peaks)
    assert ref["n_peaks"] <= w.cap_peaks
    n, pb, pm, _ = _noalloc(hough, grid, acc_dev, w.cap_peaks)
    assert n == ref["n_peaks"] and n > 10000
    assert np.array_equal(pb, ref["peak_bin"]) and np.array_equal(pm, ref["peak_mask"])
    small = synth.Grid(n_phi=12, n_d0=3, n_kappa=32, L_min=3)
    acc_s = torch.from_numpy(_random_acc(rng, small, 0.9, 10).view(np.int32)).to(dev)
    ref_s = _existing_path(hough, small, acc_s, small.n_bins)
    n_s, pb_s, pm_s, _ = _noalloc(hough, small, acc_s, small.n_bins)
    assert n_s == ref_s["n_peaks"] and np.array_equal(pb_s, ref_s["peak_bin"]) and np.array_equal(pm_s, ref_s["peak_mask"])
