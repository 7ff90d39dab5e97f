"""Thin Python binding of the C ABI in include/hough.h (libhough_b200.so).

Argument marshalling only: every step of the path (hit preparation, staging, vote,
write-out, peak sweep, compaction, hit lists) runs in the CUDA kernels under ``csrc/``.
PyTorch is used for device memory and streams, nothing else.  There is no CPU fallback:
importing this module raises if the shared library cannot be loaded, and every call
raises ``HoughError`` on a non-zero return code.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libhough_b200.so")

HOUGH_OK, HOUGH_EINVAL, HOUGH_ENOMEM, HOUGH_ECUDA, HOUGH_ESTATE = 0, -1, -2, -3, -4
TRUNCATED_PEAKS, TRUNCATED_HITS, INDEX16, LIST_MISMATCH = 1, 2, 4, 8
OPT_NO_CULL = 1
OPT_STAGE_TIMING = 2
OPT_UNPACKED = 4
OPT_EXACT_ONLY = 8
OPT_LIST_SWEEP = 16
OPT_LINE = 32
OPT_INTERVAL = 64
OPT_FUSED_PEAKS = 128
OPT_CELL_PEAKS = 256
OPT_CHECK_LISTS = 512
N_STAGES = 9

# every symbol include/hough.h declares (checked by the CPU test-suite)
SYMBOLS = ("hough_workspace_bytes", "hough_create", "hough_destroy", "hough_vote", "hough_peaks",
           "hough_accumulator", "hough_process_host", "hough_submit_host", "hough_collect_begin", "hough_collect_end",
           "hough_collect_host", "hough_clear", "hough_peak_sweep",
           "hough_set_accumulator", "hough_peaks_only", "hough_microbench_smem", "hough_query",
           "hough_launch_count", "hough_stage_times", "hough_stage_name", "hough_strerror",
           "hough_vertex_workspace_bytes", "hough_vertices", "hough_fit_workspace_bytes", "hough_fit",
           "hough_peaks_noalloc", "hough_check_lists")


class HoughError(RuntimeError):
    pass


class Config(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("layer_radius_cm", C.POINTER(C.c_double)),
                ("phi_min", C.c_double), ("phi_max", C.c_double),
                ("d0_min", C.c_double), ("d0_max", C.c_double),
                ("kappa_min", C.c_double), ("kappa_max", C.c_double),
                ("n_phi", C.c_int32), ("n_d0", C.c_int32), ("n_kappa", C.c_int32),
                ("L_min", C.c_int32), ("phi_wrap", C.c_int32),
                ("max_hits", C.c_uint32), ("cap_peaks", C.c_uint32), ("cap_hits", C.c_uint64),
                ("tile_phi", C.c_int32), ("tile_d0", C.c_int32),
                ("options", C.c_uint32), ("device", C.c_int32)]


class Counts(C.Structure):
    _fields_ = [("n_votes", C.c_uint64), ("n_hit_entries", C.c_uint64), ("n_evals", C.c_uint64),
                ("n_list_evals", C.c_uint64), ("n_peaks", C.c_uint32), ("n_bad_hits", C.c_uint32), ("flags", C.c_uint32),
                ("reserved", C.c_uint32)]


class PeaksOut(C.Structure):
    _fields_ = [("bin", C.c_void_p), ("mask", C.c_void_p), ("hit_offset", C.c_void_p),
                ("hit_index", C.c_void_p), ("counts", C.c_void_p), ("hit_index16", C.c_void_p)]


class HostOut(C.Structure):
    _fields_ = [("bin", C.c_void_p), ("mask", C.c_void_p), ("hit_offset", C.c_void_p),
                ("hit_index", C.c_void_p), ("counts", C.c_void_p), ("hit_index16", C.c_void_p)]


class VertexConfig(C.Structure):
    _fields_ = [("x_min", C.c_double), ("x_max", C.c_double), ("y_min", C.c_double), ("y_max", C.c_double),
                ("n_x", C.c_int32), ("n_y", C.c_int32), ("V_min", C.c_int32), ("cap_vertices", C.c_uint32),
                ("cap_members", C.c_uint64)]


class VertexOut(C.Structure):
    _fields_ = [("bin", C.c_void_p), ("count", C.c_void_p), ("member_offset", C.c_void_p),
                ("member_index", C.c_void_p), ("counts", C.c_void_p)]


class FitConfig(C.Structure):
    _fields_ = [("rms_max", C.c_double), ("min_shared", C.c_uint32), ("reserved", C.c_uint32)]


class FitOut(C.Structure):
    _fields_ = [("kappa", C.c_void_p), ("phi0", C.c_void_p), ("d0", C.c_void_p), ("rms", C.c_void_p),
                ("status", C.c_void_p), ("flag", C.c_void_p), ("kept", C.c_void_p), ("counts", C.c_void_p)]


FIT_COUNTS_DTYPE = np.dtype([("n_fitted", "<u4"), ("n_ok", "<u4"), ("n_selected", "<u4"), ("n_kept", "<u4"),
                             ("n_duplicates", "<u4"), ("n_truncated", "<u4"), ("n_pair_tests", "<u8")])

VERTEX_COUNTS_DTYPE = np.dtype([("n_vertex_votes", "<u8"), ("n_member_entries", "<u8"), ("n_vertices", "<u4"),
                                ("flags", "<u4"), ("reserved", "<u8")])

COUNTS_DTYPE = np.dtype([("n_votes", "<u8"), ("n_hit_entries", "<u8"), ("n_evals", "<u8"),
                         ("n_list_evals", "<u8"), ("n_peaks", "<u4"), ("n_bad_hits", "<u4"), ("flags", "<u4"),
                         ("reserved", "<u4")])
COUNTS_WORDS = COUNTS_DTYPE.itemsize // 8  # int64 words of one hough_counts block


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "%s is missing: build it with `python -m paper_1305_4855_b200.build` "
            "(there is no CPU fallback)" % LIB_PATH)
    lib = C.CDLL(LIB_PATH)
    lib.hough_workspace_bytes.restype = C.c_size_t
    lib.hough_workspace_bytes.argtypes = [C.POINTER(Config)]
    lib.hough_create.restype = C.c_int
    lib.hough_create.argtypes = [C.POINTER(Config), C.c_void_p, C.c_size_t, C.POINTER(C.c_void_p)]
    lib.hough_destroy.restype = None
    lib.hough_destroy.argtypes = [C.c_void_p]
    lib.hough_vote.restype = C.c_int
    lib.hough_vote.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
    for name in ("hough_peaks", "hough_peaks_only", "hough_check_lists"):
        f = getattr(lib, name)
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, C.POINTER(PeaksOut), C.c_void_p]
    lib.hough_accumulator.restype = C.c_void_p
    lib.hough_accumulator.argtypes = [C.c_void_p]
    lib.hough_process_host.restype = C.c_int
    lib.hough_process_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32,
                                       C.POINTER(PeaksOut), C.POINTER(HostOut), C.c_void_p]
    lib.hough_submit_host.restype = C.c_int
    lib.hough_submit_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32,
                                      C.POINTER(PeaksOut), C.c_int32, C.c_void_p]
    for name in ("hough_collect_host", "hough_collect_begin"):
        f = getattr(lib, name)
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, C.POINTER(PeaksOut), C.POINTER(HostOut), C.c_int32, C.c_void_p]
    lib.hough_collect_end.restype = C.c_int
    lib.hough_collect_end.argtypes = [C.c_void_p, C.c_int32]
    for name in ("hough_clear", "hough_peak_sweep"):
        f = getattr(lib, name)
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, C.c_void_p]
    lib.hough_set_accumulator.restype = C.c_int
    lib.hough_set_accumulator.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.hough_microbench_smem.restype = C.c_int
    lib.hough_microbench_smem.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p,
                                          C.c_void_p, C.POINTER(C.c_uint64)]
    lib.hough_query.restype = C.c_int
    lib.hough_query.argtypes = [C.c_void_p] + [C.POINTER(C.c_int32)] * 6
    lib.hough_launch_count.restype = C.c_uint64
    lib.hough_launch_count.argtypes = [C.c_void_p]
    lib.hough_stage_times.restype = C.c_int
    lib.hough_stage_times.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.c_int]
    lib.hough_stage_name.restype = C.c_char_p
    lib.hough_stage_name.argtypes = [C.c_int]
    lib.hough_strerror.restype = C.c_char_p
    lib.hough_strerror.argtypes = [C.c_int]
    lib.hough_vertex_workspace_bytes.restype = C.c_size_t
    lib.hough_vertex_workspace_bytes.argtypes = [C.POINTER(VertexConfig)]
    lib.hough_vertices.restype = C.c_int
    lib.hough_vertices.argtypes = [C.c_void_p, C.POINTER(VertexConfig), C.c_void_p, C.c_size_t,
                                   C.POINTER(PeaksOut), C.POINTER(VertexOut), C.c_void_p]
    lib.hough_fit_workspace_bytes.restype = C.c_size_t
    lib.hough_fit_workspace_bytes.argtypes = [C.c_void_p]
    lib.hough_fit.restype = C.c_int
    lib.hough_fit.argtypes = [C.c_void_p, C.POINTER(FitConfig), C.c_void_p, C.c_size_t, C.POINTER(PeaksOut),
                              C.POINTER(FitOut), C.c_void_p]
    lib.hough_peaks_noalloc.restype = C.c_int
    lib.hough_peaks_noalloc.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32,
                                        C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p]
    return lib


_lib = _load()


def strerror(code: int) -> str:
    return _lib.hough_strerror(int(code)).decode()


def _check(rc: int, what: str):
    if rc != HOUGH_OK:
        raise HoughError("%s failed: %s (%d)" % (what, strerror(rc), rc))


def make_config(grid, max_hits, cap_peaks, cap_hits, device=0, tile_phi=0, tile_d0=0, options=0):
    """hough_config from any object with the Grid attributes (see synth.Grid).  Returns
    (Config, keep-alive objects)."""
    radii = (C.c_double * len(grid.layer_radii))(*[float(r) for r in grid.layer_radii])
    cfg = Config(len(grid.layer_radii), C.cast(radii, C.POINTER(C.c_double)),
                 grid.phi_min, grid.phi_max, grid.d0_min, grid.d0_max, grid.kappa_min, grid.kappa_max,
                 grid.n_phi, grid.n_d0, grid.n_kappa, grid.L_min, grid.phi_wrap,
                 int(max_hits), int(cap_peaks), int(cap_hits), int(tile_phi), int(tile_d0),
                 int(options), int(device))
    return cfg, radii


def workspace_bytes(grid, max_hits, cap_peaks, cap_hits, **kw) -> int:
    cfg, _keep = make_config(grid, max_hits, cap_peaks, cap_hits, **kw)
    return int(_lib.hough_workspace_bytes(C.byref(cfg)))


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


class Hough:
    """One grid on one device.  ``vote`` + ``peaks`` enqueue on a stream and return;
    ``read`` synchronises and returns numpy views of the results."""

    def __init__(self, grid, max_hits, cap_peaks, cap_hits, device=0, tile_phi=0, tile_d0=0,
                 options=0):
        if not torch.cuda.is_available():
            raise HoughError("no CUDA device: the Hough path has no CPU fallback")
        self.grid = grid
        self.device = torch.device("cuda", device)
        self.cap_peaks, self.cap_hits, self.max_hits = int(cap_peaks), int(cap_hits), int(max_hits)
        self.cfg, self._keep = make_config(grid, max_hits, cap_peaks, cap_hits, device, tile_phi,
                                           tile_d0, options)
        nbytes = int(_lib.hough_workspace_bytes(C.byref(self.cfg)))
        if nbytes == 0:
            raise HoughError("hough_workspace_bytes: invalid configuration")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self._h = C.c_void_p()
        _check(_lib.hough_create(C.byref(self.cfg), C.c_void_p(self.workspace.data_ptr()), nbytes,
                                 C.byref(self._h)), "hough_create")
        i32 = dict(dtype=torch.int32, device=self.device)
        self.peak_bin = torch.empty(self.cap_peaks, **i32)
        self.peak_mask = torch.empty(self.cap_peaks, **i32)
        self.hit_offset = torch.empty(self.cap_peaks + 1, dtype=torch.int64, device=self.device)
        self.hit_index = torch.empty(self.cap_hits, **i32)
        self.counts = torch.zeros(COUNTS_WORDS, dtype=torch.int64, device=self.device)
        self._out = PeaksOut(self.peak_bin.data_ptr(), self.peak_mask.data_ptr(),
                             self.hit_offset.data_ptr(), self.hit_index.data_ptr(),
                             self.counts.data_ptr())
        self._host = None

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            _lib.hough_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C-ABI calls
    def vote(self, x, y, layer, stream=None):
        """hough_vote: x, y float32 / layer int32 CUDA tensors of one event."""
        n = int(x.numel())
        assert x.is_cuda and y.is_cuda and layer.is_cuda
        assert x.dtype == torch.float32 and y.dtype == torch.float32 and layer.dtype == torch.int32
        assert y.numel() == n and layer.numel() == n
        assert x.is_contiguous() and y.is_contiguous() and layer.is_contiguous()
        _check(_lib.hough_vote(self._h, C.c_void_p(x.data_ptr()), C.c_void_p(y.data_ptr()),
                               C.c_void_p(layer.data_ptr()), n, _stream_ptr(stream)), "hough_vote")

    def peaks(self, stream=None, lists=True, counts_out=None):
        """hough_peaks (or hough_peaks_only): results land in this object's device arrays.
        counts_out: optional int64 CUDA tensor of COUNTS_WORDS words that receives this
        event's hough_counts instead of self.counts (lets a batch keep every event's counters)."""
        f = _lib.hough_peaks if lists else _lib.hough_peaks_only
        out = self._out
        if counts_out is not None:
            assert counts_out.is_cuda and counts_out.dtype == torch.int64
            assert counts_out.numel() == COUNTS_WORDS and counts_out.is_contiguous()
            out = PeaksOut(self._out.bin, self._out.mask, self._out.hit_offset, self._out.hit_index,
                           counts_out.data_ptr())
        _check(f(self._h, C.byref(out), _stream_ptr(stream)), "hough_peaks")

    def check_lists(self, stream=None):
        """hough_check_lists on this object's device arrays: a violated list invariant sets LIST_MISMATCH
        in the counters' flags (see ``read``)."""
        _check(_lib.hough_check_lists(self._h, C.byref(self._out), _stream_ptr(stream)), "hough_check_lists")

    def clear(self, stream=None):
        _check(_lib.hough_clear(self._h, _stream_ptr(stream)), "hough_clear")

    def peak_sweep(self, stream=None):
        _check(_lib.hough_peak_sweep(self._h, _stream_ptr(stream)), "hough_peak_sweep")

    def set_accumulator(self, acc, stream=None):
        assert acc.is_cuda and acc.dtype == torch.int32 and acc.numel() == self.grid.n_bins
        _check(_lib.hough_set_accumulator(self._h, C.c_void_p(acc.data_ptr()), _stream_ptr(stream)),
               "hough_set_accumulator")

    def accumulator(self) -> torch.Tensor:
        """Device view (int32 bit patterns of the uint32 masks), shape [n_phi, n_d0, n_kappa]."""
        ptr = _lib.hough_accumulator(self._h)
        off = ptr - self.workspace.data_ptr()
        g = self.grid
        return self.workspace[off:off + 4 * g.n_bins].view(torch.int32).view(g.n_phi, g.n_d0, g.n_kappa)

    def process_host(self, x, y, layer, stream=None, want_lists=True):
        """hough_process_host: numpy (ideally pinned) host arrays in, host results out."""
        x = np.ascontiguousarray(x, np.float32)
        y = np.ascontiguousarray(y, np.float32)
        layer = np.ascontiguousarray(layer, np.int32)
        n = x.shape[0]
        if self._host is None:
            pin = dict(pin_memory=True)
            self._host = dict(
                bin=torch.empty(self.cap_peaks, dtype=torch.int32, **pin),
                mask=torch.empty(self.cap_peaks, dtype=torch.int32, **pin),
                hit_offset=torch.empty(self.cap_peaks + 1, dtype=torch.int64, **pin),
                hit_index=torch.empty(self.cap_hits, dtype=torch.int32, **pin),
                counts=torch.zeros(COUNTS_WORDS, dtype=torch.int64, **pin))
        hb = self._host
        host = HostOut(hb["bin"].data_ptr(), hb["mask"].data_ptr(), hb["hit_offset"].data_ptr(),
                       hb["hit_index"].data_ptr() if want_lists else None, hb["counts"].data_ptr())
        _check(_lib.hough_process_host(self._h, C.c_void_p(x.ctypes.data), C.c_void_p(y.ctypes.data),
                                       C.c_void_p(layer.ctypes.data), n, C.byref(self._out),
                                       C.byref(host), _stream_ptr(stream)), "hough_process_host")
        cnt = hb["counts"].numpy().view(COUNTS_DTYPE)[0]
        return self._pack(cnt, hb["bin"].numpy(), hb["mask"].numpy(), hb["hit_offset"].numpy(),
                          hb["hit_index"].numpy() if want_lists else None)

    def _slot(self, slot):
        """Device and pinned host arrays of one in-flight event (submit_host / collect_host).  With at
        most 65536 hits per event the hit lists travel as 16-bit indices (hit_index16)."""
        if not hasattr(self, "_slots"):
            self._slots, self._copy_stream = {}, torch.cuda.Stream(device=self.device)
        if slot not in self._slots:
            i32 = dict(dtype=torch.int32, device=self.device)
            pin = dict(pin_memory=True)
            d = dict(bin=torch.empty(self.cap_peaks, **i32), mask=torch.empty(self.cap_peaks, **i32),
                     hit_offset=torch.empty(self.cap_peaks + 1, dtype=torch.int64, device=self.device),
                     hit_index=torch.empty(self.cap_hits, **i32),
                     counts=torch.zeros(COUNTS_WORDS, dtype=torch.int64, device=self.device))
            use16 = self.max_hits <= 65536
            if use16:
                d["hit_index16"] = torch.empty(self.cap_hits, dtype=torch.int16, device=self.device)
            hb = dict(bin=torch.empty(self.cap_peaks, dtype=torch.int32, **pin),
                      mask=torch.empty(self.cap_peaks, dtype=torch.int32, **pin),
                      hit_offset=torch.empty(self.cap_peaks + 1, dtype=torch.int64, **pin),
                      hit_index=torch.empty(self.cap_hits, dtype=torch.int32, **pin),
                      counts=torch.zeros(COUNTS_WORDS, dtype=torch.int64, **pin))
            if use16:
                hb["hit_index16"] = torch.empty(self.cap_hits, dtype=torch.int16, **pin)
            out = PeaksOut(d["bin"].data_ptr(), d["mask"].data_ptr(), d["hit_offset"].data_ptr(),
                           d["hit_index"].data_ptr(), d["counts"].data_ptr(),
                           d["hit_index16"].data_ptr() if use16 else None)
            host = HostOut(hb["bin"].data_ptr(), hb["mask"].data_ptr(), hb["hit_offset"].data_ptr(),
                           hb["hit_index"].data_ptr(), hb["counts"].data_ptr(),
                           hb["hit_index16"].data_ptr() if use16 else None)
            self._slots[slot] = (d, hb, out, host)
        return self._slots[slot]

    def submit_host(self, x, y, layer, slot, stream=None):
        """hough_submit_host: host arrays in (pinned for overlap), compute enqueued, returns at once."""
        x = np.ascontiguousarray(x, np.float32)
        y = np.ascontiguousarray(y, np.float32)
        layer = np.ascontiguousarray(layer, np.int32)
        _d, _hb, out, _host = self._slot(slot)
        _check(_lib.hough_submit_host(self._h, C.c_void_p(x.ctypes.data), C.c_void_p(y.ctypes.data),
                                      C.c_void_p(layer.ctypes.data), x.shape[0], C.byref(out), int(slot),
                                      _stream_ptr(stream)), "hough_submit_host")

    def collect_host(self, slot):
        """hough_collect_host: results of the event submitted in `slot`, copied on a second stream."""
        self.collect_begin(slot)
        return self.collect_end(slot)

    def collect_begin(self, slot):
        """hough_collect_begin: wait for the slot's computation, start copying its results to the host."""
        _d, _hb, out, host = self._slot(slot)
        _check(_lib.hough_collect_begin(self._h, C.byref(out), C.byref(host), int(slot),
                                        C.c_void_p(self._copy_stream.cuda_stream)), "hough_collect_begin")

    def collect_end(self, slot):
        """hough_collect_end: wait for the copies; returns numpy views of the slot's pinned host buffers."""
        _d, hb, _out, _host = self._slot(slot)
        _check(_lib.hough_collect_end(self._h, int(slot)), "hough_collect_end")
        cnt = hb["counts"].numpy().view(COUNTS_DTYPE)[0]
        if int(cnt["flags"]) & INDEX16 and "hit_index16" in hb:  # the lists came back as 16-bit indices
            idx = hb["hit_index16"].numpy().view(np.uint16)
        else:
            idx = hb["hit_index"].numpy()
        return self._pack(cnt, hb["bin"].numpy(), hb["mask"].numpy(), hb["hit_offset"].numpy(), idx)

    # -- f1: the second transform over the peaks (hough_vertices)
    def vertices(self, vgrid, cap_vertices=1024, cap_members=1 << 20, stream=None):
        """hough_vertices on the peaks of the last ``peaks`` call (device arrays of this object);
        ``vgrid`` has the synth.VertexGrid attributes.  Enqueues only; see ``read_vertices``."""
        key = (vgrid, int(cap_vertices), int(cap_members))
        if getattr(self, "_vx_key", None) != key:
            vc = VertexConfig(vgrid.x_min, vgrid.x_max, vgrid.y_min, vgrid.y_max, vgrid.n_x, vgrid.n_y,
                              vgrid.V_min, int(cap_vertices), int(cap_members))
            nbytes = int(_lib.hough_vertex_workspace_bytes(C.byref(vc)))
            if nbytes == 0:
                raise HoughError("hough_vertex_workspace_bytes: invalid configuration")
            i32 = dict(dtype=torch.int32, device=self.device)
            self._vx = dict(cfg=vc, nbytes=nbytes, ws=torch.empty(nbytes, dtype=torch.uint8, device=self.device),
                            bin=torch.empty(cap_vertices, **i32), count=torch.empty(cap_vertices, **i32),
                            member_offset=torch.empty(cap_vertices + 1, dtype=torch.int64, device=self.device),
                            member_index=torch.empty(cap_members, **i32),
                            counts=torch.zeros(VERTEX_COUNTS_DTYPE.itemsize // 8, dtype=torch.int64, device=self.device))
            v = self._vx
            v["out"] = VertexOut(v["bin"].data_ptr(), v["count"].data_ptr(), v["member_offset"].data_ptr(),
                                 v["member_index"].data_ptr(), v["counts"].data_ptr())
            self._vx_key = key
        v = self._vx
        _check(_lib.hough_vertices(self._h, C.byref(v["cfg"]), C.c_void_p(v["ws"].data_ptr()), v["nbytes"],
                                   C.byref(self._out), C.byref(v["out"]), _stream_ptr(stream)), "hough_vertices")

    def read_vertices(self):
        """Synchronise and copy the results of the last ``vertices`` call to the host."""
        torch.cuda.synchronize(self.device)
        v = self._vx
        vc = v["cfg"]
        cnt = v["counts"].cpu().numpy().view(VERTEX_COUNTS_DTYPE)[0]
        n_rep = min(int(cnt["n_vertices"]), int(vc.cap_vertices))
        n_mem = min(int(cnt["n_member_entries"]), int(vc.cap_members))
        return {"vacc": v["ws"][:4 * vc.n_x * vc.n_y].view(torch.int32).cpu().numpy().view(np.uint32).reshape(vc.n_x, vc.n_y),
                "n_vertex_votes": int(cnt["n_vertex_votes"]), "n_vertices": int(cnt["n_vertices"]),
                "n_member_entries": int(cnt["n_member_entries"]), "flags": int(cnt["flags"]),
                "vertex_bin": v["bin"][:n_rep].cpu().numpy().view(np.uint32),
                "vertex_count": v["count"][:n_rep].cpu().numpy().view(np.uint32),
                "member_offset": v["member_offset"][:n_rep + 1].cpu().numpy().view(np.uint64),
                "member_index": v["member_index"][:n_mem].cpu().numpy().view(np.uint32)}

    # -- f2: fit + duplicate removal (hough_fit)
    def fit(self, rms_max, min_shared, stream=None):
        """hough_fit on the peaks and hit lists of the last ``peaks`` call.  Enqueues only; see ``read_fit``."""
        if getattr(self, "_fit", None) is None:
            nbytes = int(_lib.hough_fit_workspace_bytes(self._h))
            if nbytes == 0:
                raise HoughError("hough_fit_workspace_bytes: cap_hits too large")
            f64 = dict(dtype=torch.float64, device=self.device)
            f = dict(nbytes=nbytes, ws=torch.empty(nbytes, dtype=torch.uint8, device=self.device),
                     kappa=torch.empty(self.cap_peaks, **f64), phi0=torch.empty(self.cap_peaks, **f64),
                     d0=torch.empty(self.cap_peaks, **f64), rms=torch.empty(self.cap_peaks, **f64),
                     status=torch.empty(self.cap_peaks, dtype=torch.int32, device=self.device),
                     flag=torch.empty(self.cap_peaks, dtype=torch.uint8, device=self.device),
                     kept=torch.empty(self.cap_peaks, dtype=torch.int32, device=self.device),
                     counts=torch.zeros(FIT_COUNTS_DTYPE.itemsize // 8, dtype=torch.int64, device=self.device))
            f["out"] = FitOut(f["kappa"].data_ptr(), f["phi0"].data_ptr(), f["d0"].data_ptr(), f["rms"].data_ptr(),
                              f["status"].data_ptr(), f["flag"].data_ptr(), f["kept"].data_ptr(),
                              f["counts"].data_ptr())
            self._fit = f
        f = self._fit
        fc = FitConfig(float(rms_max), int(min_shared), 0)
        _check(_lib.hough_fit(self._h, C.byref(fc), C.c_void_p(f["ws"].data_ptr()), f["nbytes"],
                              C.byref(self._out), C.byref(f["out"]), _stream_ptr(stream)), "hough_fit")

    def read_fit(self):
        """Synchronise and copy the results of the last ``fit`` call to the host."""
        torch.cuda.synchronize(self.device)
        f = self._fit
        cnt = f["counts"].cpu().numpy().view(FIT_COUNTS_DTYPE)[0]
        n = int(cnt["n_fitted"])
        out = {k: int(cnt[k]) for k in FIT_COUNTS_DTYPE.names}
        for k in ("kappa", "phi0", "d0", "rms", "status", "flag"):
            out[k] = f[k][:n].cpu().numpy()
        out["kept"] = f["kept"][:int(cnt["n_kept"])].cpu().numpy().view(np.uint32)
        return out

    # -- results
    def _pack(self, cnt, b, m, off, idx):
        n_rep = min(int(cnt["n_peaks"]), self.cap_peaks)
        n_ent = min(int(cnt["n_hit_entries"]), self.cap_hits)
        out = {"n_votes": int(cnt["n_votes"]), "n_hit_entries": int(cnt["n_hit_entries"]),
               "n_evals": int(cnt["n_evals"]), "n_list_evals": int(cnt["n_list_evals"]),
               "n_peaks": int(cnt["n_peaks"]), "n_bad_hits": int(cnt["n_bad_hits"]),
               "flags": int(cnt["flags"]),
               "peak_bin": b[:n_rep].view(np.uint32), "peak_mask": m[:n_rep].view(np.uint32),
               "hit_offset": off[:n_rep + 1].view(np.uint64)}
        if idx is not None:
            out["hit_index"] = idx[:n_ent] if idx.dtype == np.uint16 else idx[:n_ent].view(np.uint32)
        return out

    def read_counts(self):
        torch.cuda.synchronize(self.device)
        return self.counts.cpu().numpy().view(COUNTS_DTYPE)[0]

    def read(self, lists=True):
        """Synchronise and copy the results of the last vote + peaks to the host."""
        cnt = self.read_counts()
        n_rep = min(int(cnt["n_peaks"]), self.cap_peaks)
        n_ent = min(int(cnt["n_hit_entries"]), self.cap_hits) if lists else 0
        b = self.peak_bin[:n_rep].cpu().numpy()
        m = self.peak_mask[:n_rep].cpu().numpy()
        off = self.hit_offset[:n_rep + 1].cpu().numpy() if lists else np.zeros(n_rep + 1, np.int64)
        idx = self.hit_index[:n_ent].cpu().numpy() if lists else None
        return self._pack(cnt, b, m, off, idx)

    def accumulator_host(self) -> np.ndarray:
        torch.cuda.synchronize(self.device)
        return self.accumulator().cpu().numpy().view(np.uint32)

    def query(self):
        v = [C.c_int32() for _ in range(6)]
        _check(_lib.hough_query(self._h, *[C.byref(a) for a in v]), "hough_query")
        keys = ("tile_phi", "tile_d0", "n_tiles", "threads", "smem_bytes", "n_sms")
        return dict(zip(keys, [a.value for a in v]))

    def launch_count(self) -> int:
        return int(_lib.hough_launch_count(self._h))

    def stage_times(self) -> dict:
        """hough_stage_times: {stage name: ms} of the last vote + peaks (needs OPT_STAGE_TIMING)."""
        ms = (C.c_float * N_STAGES)()
        n = _lib.hough_stage_times(self._h, ms, N_STAGES)
        if n < 0:
            _check(n, "hough_stage_times")
        return {_lib.hough_stage_name(s).decode(): float(ms[s]) for s in range(n)}


NOALLOC_MAX_BINS = 1 << 24


def peaks_noalloc(acc, n_phi, n_d0, n_kappa, L_min, phi_wrap, peak_bin, peak_mask, n_peaks, stream=None):
    """hough_peaks_noalloc: peaks of the accumulator ``acc`` (int32 CUDA tensor of n_phi*n_d0*n_kappa
    masks) into the caller's ``peak_bin`` / ``peak_mask`` (int32, equal capacity) and ``n_peaks``
    (int32, one element), for callers that may not allocate device memory: the call takes no handle
    and no workspace, its scratch is a fixed array inside the library (at most NOALLOC_MAX_BINS bins;
    calls that overlap on one GPU race on it).  Every tensor here is the caller's; this wrapper
    allocates nothing either.  Enqueues on ``stream`` and returns."""
    for t in (acc, peak_bin, peak_mask, n_peaks):
        assert t.is_cuda and t.dtype == torch.int32 and t.is_contiguous() and t.device == acc.device
    assert acc.numel() == n_phi * n_d0 * n_kappa and peak_mask.numel() == peak_bin.numel() and n_peaks.numel() == 1
    with torch.cuda.device(acc.device):   # the call acts on the thread's current device
        _check(_lib.hough_peaks_noalloc(C.c_void_p(acc.data_ptr()), int(n_phi), int(n_d0), int(n_kappa), int(L_min),
                                        int(phi_wrap), C.c_void_p(peak_bin.data_ptr()),
                                        C.c_void_p(peak_mask.data_ptr()), int(peak_bin.numel()),
                                        C.c_void_p(n_peaks.data_ptr()), _stream_ptr(stream)),
               "hough_peaks_noalloc")


def microbench_smem(mode, threads=1024, ctas_per_sm=2, iters=4096, device=0, reps=5):
    """Times hough_microbench_smem with CUDA events; returns lane-ops per second (best of reps)."""
    st = torch.cuda.current_stream()
    ops = C.c_uint64()
    sink = torch.zeros(1, dtype=torch.int32, device=torch.device("cuda", device))
    best = None
    for _ in range(reps + 1):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        _check(_lib.hough_microbench_smem(device, mode, threads, ctas_per_sm, iters,
                                          C.c_void_p(sink.data_ptr()), C.c_void_p(st.cuda_stream),
                                          C.byref(ops)),
               "hough_microbench_smem")
        e1.record(st)
        e1.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None else min(best, ms)
    return ops.value / (best * 1e-3)
