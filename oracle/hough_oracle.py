"""ctypes front-end of the CPU oracle (oracle/hough_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this module and
this module never imports the product package.  All arithmetic of the method lives in
hough_oracle.c (restating BASELINE.json north_star; the
paper defines the transform in words only); this file only
marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import build as _build  # noqa: E402  (oracle/build.py)

sys.path.pop(0)


class _Grid(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("n_phi", C.c_int32), ("n_d0", C.c_int32),
                ("n_kappa", C.c_int32), ("L_min", C.c_int32), ("phi_wrap", C.c_int32),
                ("phi_min", C.c_double), ("phi_max", C.c_double), ("d0_min", C.c_double),
                ("d0_max", C.c_double), ("kappa_min", C.c_double), ("kappa_max", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_vote.restype = C.c_uint64
        _lib.oracle_vote_cells.restype = C.c_uint64
        _lib.oracle_peaks.restype = C.c_uint64
        _lib.oracle_hitlists.restype = C.c_uint64
        _lib.oracle_vote_one.restype = C.c_int
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def _g(grid) -> _Grid:
    return _Grid(grid.n_layers, grid.n_phi, grid.n_d0, grid.n_kappa, grid.L_min, grid.phi_wrap,
                 grid.phi_min, grid.phi_max, grid.d0_min, grid.d0_max, grid.kappa_min,
                 grid.kappa_max)


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _hits(x, y, layer):
    x = np.ascontiguousarray(x, dtype=np.float32)
    y = np.ascontiguousarray(y, dtype=np.float32)
    layer = np.ascontiguousarray(layer, dtype=np.int32)
    assert x.shape == y.shape == layer.shape and x.ndim == 1
    return x, y, layer


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(t: int) -> None:
    lib().oracle_set_num_threads(C.c_int(int(t)))


def tables(grid):
    """A1: (sn, cs, d0c, twod0, d0sq, (klo, khi, inv_dk)) as fp32 arrays."""
    g = _g(grid)
    sn = np.empty(grid.n_phi, np.float32)
    cs = np.empty(grid.n_phi, np.float32)
    d0c = np.empty(grid.n_d0, np.float32)
    twod0 = np.empty(grid.n_d0, np.float32)
    d0sq = np.empty(grid.n_d0, np.float32)
    ks = np.empty(3, np.float32)
    lib().oracle_tables(C.byref(g), _p(sn, C.c_float), _p(cs, C.c_float), _p(d0c, C.c_float),
                        _p(twod0, C.c_float), _p(d0sq, C.c_float), _p(ks, C.c_float))
    return sn, cs, d0c, twod0, d0sq, ks


def vote(grid, x, y, layer):
    """A2-A5 over the whole grid -> (acc uint32[n_phi, n_d0, n_kappa], n_votes, n_bad)."""
    x, y, layer = _hits(x, y, layer)
    g = _g(grid)
    acc = np.empty(grid.n_phi * grid.n_d0 * grid.n_kappa, np.uint32)
    n_bad = C.c_uint32(0)
    nv = lib().oracle_vote(C.byref(g), _p(x, C.c_float), _p(y, C.c_float), _p(layer, C.c_int32),
                           C.c_uint32(x.shape[0]), _p(acc, C.c_uint32), C.byref(n_bad))
    return acc.reshape(grid.n_phi, grid.n_d0, grid.n_kappa), int(nv), int(n_bad.value)


def vote_cells(grid, x, y, layer, cell_i, cell_j):
    """A2-A5 for listed cells only -> (rows uint32[n_cells, n_kappa], votes in them)."""
    x, y, layer = _hits(x, y, layer)
    ci = np.ascontiguousarray(cell_i, dtype=np.int32)
    cj = np.ascontiguousarray(cell_j, dtype=np.int32)
    g = _g(grid)
    rows = np.empty((ci.shape[0], grid.n_kappa), np.uint32)
    nv = lib().oracle_vote_cells(C.byref(g), _p(x, C.c_float), _p(y, C.c_float),
                                 _p(layer, C.c_int32), C.c_uint32(x.shape[0]),
                                 _p(ci, C.c_int32), _p(cj, C.c_int32), C.c_uint32(ci.shape[0]),
                                 _p(rows, C.c_uint32))
    return rows, int(nv)


def peaks(grid, acc, cap=None):
    """A6: (peak_bin uint32[m], peak_mask uint32[m], true n_peaks); m = min(n_peaks, cap)."""
    acc = np.ascontiguousarray(acc, dtype=np.uint32).reshape(-1)
    assert acc.shape[0] == grid.n_phi * grid.n_d0 * grid.n_kappa
    g = _g(grid)
    if cap is None:
        cap = acc.shape[0]
    pb = np.empty(max(cap, 1), np.uint32)
    pm = np.empty(max(cap, 1), np.uint32)
    n = int(lib().oracle_peaks(C.byref(g), _p(acc, C.c_uint32), _p(pb, C.c_uint32),
                               _p(pm, C.c_uint32), C.c_uint64(cap)))
    m = min(n, cap)
    return pb[:m].copy(), pm[:m].copy(), n


def hitlists(grid, x, y, layer, peak_bin, cap_hits=None):
    """A7: CSR (hit_offset uint64[m+1], hit_index uint32[min(total, cap)], true total)."""
    x, y, layer = _hits(x, y, layer)
    pb = np.ascontiguousarray(peak_bin, dtype=np.uint32)
    g = _g(grid)
    m = pb.shape[0]
    off = np.zeros(m + 1, np.uint64)
    if cap_hits is None:
        # first call sizes the output (cap 0 writes nothing), second fills it
        total = int(lib().oracle_hitlists(C.byref(g), _p(x, C.c_float), _p(y, C.c_float),
                                          _p(layer, C.c_int32), C.c_uint32(x.shape[0]),
                                          _p(pb, C.c_uint32), C.c_uint64(m), _p(off, C.c_uint64),
                                          _p(np.empty(1, np.uint32), C.c_uint32), C.c_uint64(0)))
        cap_hits = total
    idx = np.empty(max(cap_hits, 1), np.uint32)
    total = int(lib().oracle_hitlists(C.byref(g), _p(x, C.c_float), _p(y, C.c_float),
                                      _p(layer, C.c_int32), C.c_uint32(x.shape[0]),
                                      _p(pb, C.c_uint32), C.c_uint64(m), _p(off, C.c_uint64),
                                      _p(idx, C.c_uint32), C.c_uint64(cap_hits)))
    return off, idx[:min(total, cap_hits)].copy(), total


def vote_one(grid, x, y, i, j):
    """A3-A4 for one (hit, i, j): (kappa fp32, k or -1)."""
    g = _g(grid)
    kap = C.c_float(0)
    k = lib().oracle_vote_one(C.byref(g), C.c_float(x), C.c_float(y), C.c_int(i), C.c_int(j),
                              C.byref(kap))
    return float(kap.value), int(k)


def run(grid, x, y, layer, cap_peaks=None, cap_hits=None):
    """Whole path A1-A7 for one event; dict of outputs in the C-ABI's layout."""
    acc, n_votes, n_bad = vote(grid, x, y, layer)
    pb, pm, n_peaks = peaks(grid, acc, cap_peaks)
    off, idx, n_ent = hitlists(grid, x, y, layer, pb, cap_hits)
    return {"acc": acc, "n_votes": n_votes, "n_bad_hits": n_bad, "peak_bin": pb,
            "peak_mask": pm, "n_peaks": n_peaks, "hit_offset": off, "hit_index": idx,
            "n_hit_entries": n_ent}
