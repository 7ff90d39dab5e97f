"""CPU-side checks of the boundary (no GPU, no compute calls): the C-ABI library loads, exports
every symbol include/hough.h declares, its host-only entry points behave as documented, and
the product path fails loudly without a CUDA device.  Also the multi-process plumbing of
bench.py (event sharding by seed, max-over-ranks time, summed work) on the gloo backend,
world_size 2 -- the path has no data-path collective.
"""
import ctypes as C
import os
import re
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def hough():
    from paper_1305_4855_b200 import build
    build.build()
    from paper_1305_4855_b200 import hough as hough_mod
    return hough_mod


def header_functions():
    src = open(os.path.join(ROOT, "include", "hough.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hough_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(hough):
    declared = header_functions()
    assert len(declared) >= 17
    assert sorted(hough.SYMBOLS) == declared
    lib = C.CDLL(hough.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name


def test_strerror_and_stage_names(hough):
    assert hough.strerror(0) == "ok"
    texts = {hough.strerror(c) for c in (0, -1, -2, -3, -4, -99)}
    assert len(texts) == 6
    names = [hough._lib.hough_stage_name(s) for s in range(hough.N_STAGES)]
    assert all(n for n in names) and len(set(names)) == hough.N_STAGES
    assert names[0] == b"prep" and names[1] == b"vote" and b"lists" in names
    assert hough._lib.hough_stage_name(hough.N_STAGES) is None
    assert hough._lib.hough_stage_name(-1) is None


def test_workspace_bytes_is_host_only_and_validates(hough):
    from paper_1305_4855_b200 import synth
    for name, w in synth.WORKLOADS.items():
        cfg, keep = hough.make_config(w.grid, 70000, w.cap_peaks, w.cap_hits)
        n = hough._lib.hough_workspace_bytes(C.byref(cfg))
        assert n >= w.grid.n_bins * 4 + w.grid.n_bins // 8, name
        assert n % 256 == 0
        assert n < 40 * 2 ** 30
    g = synth.Grid(n_phi=64, n_d0=4, n_kappa=48, L_min=3)      # n_kappa not a multiple of 32
    cfg, keep = hough.make_config(g, 10, 10, 10)
    assert hough._lib.hough_workspace_bytes(C.byref(cfg)) == 0
    g = synth.Grid(n_phi=64, n_d0=4, n_kappa=64, L_min=11)     # L_min > n_layers
    cfg, keep = hough.make_config(g, 10, 10, 10)
    assert hough._lib.hough_workspace_bytes(C.byref(cfg)) == 0
    g = synth.Grid(n_phi=2, n_d0=4, n_kappa=64, L_min=3)       # phi wrap needs n_phi >= 3
    cfg, keep = hough.make_config(g, 10, 10, 10)
    assert hough._lib.hough_workspace_bytes(C.byref(cfg)) == 0
    assert hough._lib.hough_workspace_bytes(None) == 0


def test_null_handles_are_rejected_not_dereferenced(hough):
    lib = hough._lib
    assert lib.hough_vote(None, None, None, None, 0, None) == hough.HOUGH_EINVAL
    assert lib.hough_clear(None, None) == hough.HOUGH_EINVAL
    assert lib.hough_peak_sweep(None, None) == hough.HOUGH_EINVAL
    assert lib.hough_accumulator(None) is None
    assert lib.hough_launch_count(None) == 0
    lib.hough_destroy(None)  # a no-op


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the behaviour WITHOUT a CUDA device")
def test_no_cpu_fallback_without_a_device(hough):
    """hough_create must fail with HOUGH_ECUDA (no silent CPU path)."""
    from paper_1305_4855_b200 import synth
    g = synth.Grid(n_phi=16, n_d0=4, n_kappa=32, L_min=2)
    cfg, keep = hough.make_config(g, 10, 10, 10)
    need = hough._lib.hough_workspace_bytes(C.byref(cfg))
    buf = np.zeros(need + 256, np.uint8)
    addr = (buf.ctypes.data + 255) & ~255
    h = C.c_void_p()
    rc = hough._lib.hough_create(C.byref(cfg), C.c_void_p(addr), need, C.byref(h))
    assert rc == hough.HOUGH_ECUDA and not h.value
    with pytest.raises((hough.HoughError, RuntimeError, AssertionError)):
        hough.Hough(g, 10, 10, 10)


# ------------------------------------------------------------------ multi-process plumbing
def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    n_ev = 3
    seeds = bench.shard_seeds(rank, n_ev)
    # stand-ins for this rank's measurements: time differs per rank, work is what the seeds give
    total_ms = 10.0 + 5.0 * rank
    votes, evals = float(sum(1000 + s for s in seeds)), float(100 * n_ev)
    agg = bench.aggregate(dist, torch.device("cpu"), total_ms, votes, evals, n_ev, world)
    out[rank] = (seeds, agg)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_events_and_reduce(tmp_path):
    import torch.multiprocessing as mp
    import sys
    if ROOT not in sys.path:
        sys.path.insert(0, ROOT)
    world, port = 2, _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    (s0, a0), (s1, a1) = out[0], out[1]
    assert s0 == [0, 1, 2] and s1 == [3, 4, 5]          # disjoint, rank-major
    assert a0 == a1                                      # every rank sees the same aggregate
    total_ms, votes, evals, events = a0
    assert total_ms == 15.0                              # max over ranks
    assert votes == float(sum(1000 + s for s in range(6)))
    assert evals == 600.0 and events == 6.0


def test_binding_structs_have_the_layout_of_the_header(hough, tmp_path):
    """The ctypes structures of the binding against sizeof / offsetof of include/hough.h as gcc sees it
    (a field added on one side only would shift every pointer after it)."""
    import subprocess
    structs = {
        "hough_config": (hough.Config, ["n_layers", "layer_radius_cm", "phi_min", "kappa_max", "n_phi", "L_min",
                                        "max_hits", "cap_peaks", "cap_hits", "tile_phi", "options", "device"]),
        "hough_counts": (hough.Counts, ["n_votes", "n_hit_entries", "n_evals", "n_list_evals", "n_peaks",
                                        "n_bad_hits", "flags"]),
        "hough_peaks_out": (hough.PeaksOut, ["bin", "mask", "hit_offset", "hit_index", "counts", "hit_index16"]),
        "hough_host_out": (hough.HostOut, ["bin", "mask", "hit_offset", "hit_index", "counts", "hit_index16"]),
        "hough_vertex_config": (hough.VertexConfig, ["x_min", "y_max", "n_x", "V_min", "cap_vertices", "cap_members"]),
        "hough_vertex_out": (hough.VertexOut, ["bin", "count", "member_offset", "member_index", "counts"]),
        "hough_fit_config": (hough.FitConfig, ["rms_max", "min_shared", "reserved"]),
        "hough_fit_out": (hough.FitOut, ["kappa", "phi0", "d0", "rms", "status", "flag", "kept", "counts"]),
    }
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "hough.h"', 'int main(void) {']
    for name, (_cls, fields) in structs.items():
        lines.append('printf("%s %%zu\\n", sizeof(%s));' % (name, name))
        for f in fields:
            lines.append('printf("%s.%s %%zu\\n", offsetof(%s, %s));' % (name, f, name, f))
    lines.append('printf("hough_vertex_counts %zu\\n", sizeof(hough_vertex_counts));')
    lines.append('printf("hough_fit_counts %zu\\n", sizeof(hough_fit_counts));')
    lines += ['return 0; }']
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    out = dict(l.split() for l in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.splitlines())
    for name, (cls, fields) in structs.items():
        assert int(out[name]) == C.sizeof(cls), name
        for f in fields:
            assert int(out["%s.%s" % (name, f)]) == getattr(cls, f).offset, (name, f)
    assert int(out["hough_counts"]) == hough.COUNTS_DTYPE.itemsize == 48
    assert int(out["hough_vertex_counts"]) == hough.VERTEX_COUNTS_DTYPE.itemsize
    assert int(out["hough_fit_counts"]) == hough.FIT_COUNTS_DTYPE.itemsize
