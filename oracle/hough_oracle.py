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
        _lib.oracle_hitlists_cells.restype = C.c_uint64
        _lib.oracle_vote_one.restype = C.c_int
        _lib.oracle_num_threads.restype = C.c_int
        for f in ("oracle_vote_variant", "oracle_hitlists_variant", "oracle_hitlists_variant_cells", "oracle_vertex_vote",
                  "oracle_vertex_peaks", "oracle_vertex_members"):
            getattr(_lib, f).restype = C.c_uint64
        _lib.oracle_fit_one.restype = C.c_int
        _lib.oracle_fit_all.restype = None
        _lib.oracle_select_dedup.restype = None
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


def hitlists(grid, x, y, layer, peak_bin, cap_hits=None, by_cell=False):
    """A7: CSR (hit_offset uint64[m+1], hit_index uint32[min(total, cap)], true total).
    by_cell: the same lists from oracle_hitlists_cells (one vote pass over the cells that hold a
    peak instead of one pass per peak: the only form that finishes on a pile-up event)."""
    x, y, layer = _hits(x, y, layer)
    fn = lib().oracle_hitlists_cells if by_cell else lib().oracle_hitlists
    pb = np.ascontiguousarray(peak_bin, dtype=np.uint32)
    g = _g(grid)
    m = pb.shape[0]
    off = np.zeros(m + 1, np.uint64)
    if cap_hits is None:
        # first call sizes the output (cap 0 writes nothing), second fills it
        total = int(fn(C.byref(g), _p(x, C.c_float), _p(y, C.c_float),
                                          _p(layer, C.c_int32), C.c_uint32(x.shape[0]),
                                          _p(pb, C.c_uint32), C.c_uint64(m), _p(off, C.c_uint64),
                                          _p(np.empty(1, np.uint32), C.c_uint32), C.c_uint64(0)))
        cap_hits = total
    idx = np.empty(max(cap_hits, 1), np.uint32)
    total = int(fn(C.byref(g), _p(x, C.c_float), _p(y, C.c_float),
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


def hitlists_cells(grid, x, y, layer, peak_bin, cap_hits=None):
    """A7 walked cell by cell (oracle_hitlists_cells); same outputs as hitlists."""
    return hitlists(grid, x, y, layer, peak_bin, cap_hits, by_cell=True)


def run(grid, x, y, layer, cap_peaks=None, cap_hits=None, by_cell=False):
    """Whole path A1-A7 for one event; dict of outputs in the C-ABI's layout."""
    acc, n_votes, n_bad = vote(grid, x, y, layer)
    pb, pm, n_peaks = peaks(grid, acc, cap_peaks)
    off, idx, n_ent = hitlists(grid, x, y, layer, pb, cap_hits, by_cell=by_cell)
    return {"acc": acc, "n_votes": n_votes, "n_bad_hits": n_bad, "peak_bin": pb,
            "peak_mask": pm, "n_peaks": n_peaks, "hit_offset": off, "hit_index": idx,
            "n_hit_entries": n_ent}


# ---------------------------------------------------------------------------------------
# hough_ext_oracle.c: the rows SURVEY.md 8(f) marks "next" (recipes E1..E5)

MODE_CIRCLE, MODE_LINE, MODE_INTERVAL = 0, 1, 2


class _VGrid(C.Structure):
    _fields_ = [("x_min", C.c_double), ("x_max", C.c_double), ("y_min", C.c_double),
                ("y_max", C.c_double), ("n_x", C.c_int32), ("n_y", C.c_int32),
                ("V_min", C.c_int32), ("reserved", C.c_int32)]


class _Fit(C.Structure):
    _fields_ = [("kappa", C.c_double), ("phi0", C.c_double), ("d0", C.c_double), ("rms", C.c_double)]


FIT_DTYPE = np.dtype([("kappa", np.float64), ("phi0", np.float64), ("d0", np.float64), ("rms", np.float64)])


def _vg(v) -> _VGrid:
    return _VGrid(v.x_min, v.x_max, v.y_min, v.y_max, v.n_x, v.n_y, v.V_min, 0)


def vote_variant(grid, mode, x, y, layer):
    """E1/E2: the vote under `mode` -> (acc[n_phi, n_d0, n_kappa], n_votes, n_bad)."""
    x, y, layer = _hits(x, y, layer)
    g = _g(grid)
    acc = np.empty(grid.n_phi * grid.n_d0 * grid.n_kappa, np.uint32)
    n_bad = C.c_uint32(0)
    nv = lib().oracle_vote_variant(C.byref(g), C.c_int(mode), _p(x, C.c_float), _p(y, C.c_float),
                                   _p(layer, C.c_int32), C.c_uint32(x.shape[0]), _p(acc, C.c_uint32),
                                   C.byref(n_bad))
    return acc.reshape(grid.n_phi, grid.n_d0, grid.n_kappa), int(nv), int(n_bad.value)


def hitlists_variant(grid, mode, x, y, layer, peak_bin, cap_hits=None, by_cell=False):
    """A7 under `mode`: CSR (hit_offset, hit_index[min(total, cap)], true total).
    by_cell: the same lists from oracle_hitlists_variant_cells (one pass over the hits per cell that
    holds a peak instead of one per peak)."""
    fn = lib().oracle_hitlists_variant_cells if by_cell else lib().oracle_hitlists_variant
    x, y, layer = _hits(x, y, layer)
    pb = np.ascontiguousarray(peak_bin, dtype=np.uint32)
    g = _g(grid)
    m = pb.shape[0]
    off = np.zeros(m + 1, np.uint64)

    def call(idx, cap):
        return int(fn(
            C.byref(g), C.c_int(mode), _p(x, C.c_float), _p(y, C.c_float), _p(layer, C.c_int32),
            C.c_uint32(x.shape[0]), _p(pb, C.c_uint32), C.c_uint64(m), _p(off, C.c_uint64),
            _p(idx, C.c_uint32), C.c_uint64(cap)))

    if cap_hits is None:
        cap_hits = call(np.empty(1, np.uint32), 0)
    idx = np.empty(max(cap_hits, 1), np.uint32)
    total = call(idx, cap_hits)
    return off, idx[:min(total, cap_hits)].copy(), total


def run_variant(grid, mode, x, y, layer, cap_peaks=None, cap_hits=None):
    """Whole path under a vote variant (peak rule A6 unchanged)."""
    acc, n_votes, n_bad = vote_variant(grid, mode, x, y, layer)
    pb, pm, n_peaks = peaks(grid, acc, cap_peaks)
    off, idx, n_ent = hitlists_variant(grid, mode, x, y, layer, pb, cap_hits)
    return {"acc": acc, "n_votes": n_votes, "n_bad_hits": n_bad, "peak_bin": pb,
            "peak_mask": pm, "n_peaks": n_peaks, "hit_offset": off, "hit_index": idx,
            "n_hit_entries": n_ent}


def vertex_tables(vgrid):
    v = _vg(vgrid)
    xc = np.empty(vgrid.n_x, np.float32)
    yc = np.empty(vgrid.n_y, np.float32)
    sc = np.empty(6, np.float32)
    lib().oracle_vertex_tables(C.byref(v), _p(xc, C.c_float), _p(yc, C.c_float), _p(sc, C.c_float))
    return xc, yc, sc


def vertex_vote(grid, vgrid, peak_bin):
    """E3 V2: (vacc uint32[n_x, n_y], votes cast)."""
    pb = np.ascontiguousarray(peak_bin, dtype=np.uint32)
    g, v = _g(grid), _vg(vgrid)
    vacc = np.empty(vgrid.n_x * vgrid.n_y, np.uint32)
    nv = lib().oracle_vertex_vote(C.byref(g), C.byref(v), _p(pb, C.c_uint32), C.c_uint64(pb.shape[0]),
                                  _p(vacc, C.c_uint32))
    return vacc.reshape(vgrid.n_x, vgrid.n_y), int(nv)


def vertex_peaks(vgrid, vacc, cap=None):
    """E3 V3: (vertex_bin[m], vertex_count[m], true n_vertices)."""
    vacc = np.ascontiguousarray(vacc, dtype=np.uint32).reshape(-1)
    v = _vg(vgrid)
    if cap is None:
        cap = vacc.shape[0]
    vb = np.empty(max(cap, 1), np.uint32)
    vc = np.empty(max(cap, 1), np.uint32)
    n = int(lib().oracle_vertex_peaks(C.byref(v), _p(vacc, C.c_uint32), _p(vb, C.c_uint32),
                                      _p(vc, C.c_uint32), C.c_uint64(cap)))
    m = min(n, cap)
    return vb[:m].copy(), vc[:m].copy(), n


def vertex_members(grid, vgrid, peak_bin, vertex_bin, cap=None):
    """E3 V4: CSR (member_offset[m+1], member_index[min(total, cap)], true total)."""
    pb = np.ascontiguousarray(peak_bin, dtype=np.uint32)
    vb = np.ascontiguousarray(vertex_bin, dtype=np.uint32)
    g, v = _g(grid), _vg(vgrid)
    off = np.zeros(vb.shape[0] + 1, np.uint64)

    def call(idx, c):
        return int(lib().oracle_vertex_members(
            C.byref(g), C.byref(v), _p(pb, C.c_uint32), C.c_uint64(pb.shape[0]), _p(vb, C.c_uint32),
            C.c_uint64(vb.shape[0]), _p(off, C.c_uint64), _p(idx, C.c_uint32), C.c_uint64(c)))

    if cap is None:
        cap = call(np.empty(1, np.uint32), 0)
    idx = np.empty(max(cap, 1), np.uint32)
    total = call(idx, cap)
    return off, idx[:min(total, cap)].copy(), total


def run_vertices(grid, vgrid, peak_bin, cap_vertices=None, cap_members=None):
    vacc, nv = vertex_vote(grid, vgrid, peak_bin)
    vb, vc, n = vertex_peaks(vgrid, vacc, cap_vertices)
    off, idx, tot = vertex_members(grid, vgrid, peak_bin, vb, cap_members)
    return {"vacc": vacc, "n_vertex_votes": nv, "vertex_bin": vb, "vertex_count": vc, "n_vertices": n,
            "member_offset": off, "member_index": idx, "n_member_entries": tot}


def fit_one(x, y, idx):
    """E4 for one list of hit indices -> (status, kappa, phi0, d0, rms)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    y = np.ascontiguousarray(y, dtype=np.float32)
    idx = np.ascontiguousarray(idx, dtype=np.uint32)
    f = _Fit()
    st = lib().oracle_fit_one(_p(x, C.c_float), _p(y, C.c_float), _p(idx, C.c_uint32),
                              C.c_uint32(idx.shape[0]), C.byref(f))
    return int(st), f.kappa, f.phi0, f.d0, f.rms


def fit_all(x, y, hit_offset, hit_index):
    """E4 for every list of a CSR -> (fit structured array[n_peaks], status int32[n_peaks])."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    y = np.ascontiguousarray(y, dtype=np.float32)
    off = np.ascontiguousarray(hit_offset, dtype=np.uint64)
    idx = np.ascontiguousarray(hit_index, dtype=np.uint32)
    m = off.shape[0] - 1
    fit = np.zeros(max(m, 1), FIT_DTYPE)
    status = np.zeros(max(m, 1), np.int32)
    if idx.shape[0] == 0:
        idx = np.zeros(1, np.uint32)
    lib().oracle_fit_all(_p(x, C.c_float), _p(y, C.c_float), _p(off, C.c_uint64), _p(idx, C.c_uint32),
                         C.c_uint64(m), fit.ctypes.data_as(C.POINTER(_Fit)), _p(status, C.c_int32))
    return fit[:m], status[:m]


def select_dedup(hit_offset, hit_index, peak_mask, n_hits, fit, status, rms_max, min_shared):
    """E5 -> flags uint8[n_peaks]: 0 not selected, 1 kept, 2 selected but a duplicate."""
    off = np.ascontiguousarray(hit_offset, dtype=np.uint64)
    idx = np.ascontiguousarray(hit_index, dtype=np.uint32)
    pm = np.ascontiguousarray(peak_mask, dtype=np.uint32)
    fit = np.ascontiguousarray(fit, dtype=FIT_DTYPE)
    status = np.ascontiguousarray(status, dtype=np.int32)
    m = off.shape[0] - 1
    flags = np.zeros(max(m, 1), np.uint8)
    if idx.shape[0] == 0:
        idx = np.zeros(1, np.uint32)
    lib().oracle_select_dedup(_p(off, C.c_uint64), _p(idx, C.c_uint32), _p(pm, C.c_uint32), C.c_uint64(m),
                              C.c_uint32(n_hits), fit.ctypes.data_as(C.POINTER(_Fit)), _p(status, C.c_int32),
                              C.c_double(rms_max), C.c_uint32(min_shared), flags.ctypes.data_as(C.POINTER(C.c_uint8)))
    return flags[:m]
