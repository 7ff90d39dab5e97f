#!/usr/bin/env python
"""bench.py -- throughput of the Hough-transform hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (hough_vote + hough_peaks: hit preparation,
staging, vote, write-out, peak sweep, compaction, hit lists) over one batch of the
workload: BASELINE.json configs[3], 100 independent pile-up events (seeds 0..99), each
with its own accumulator, back to back on one stream.  `value` is in-range votes cast per
second over all ranks (inputs resident in HBM); `events_per_s` and `evaluations_per_s`
(n * n_phi * n_d0 per event, the paper-level work) are reported beside it.  `e2e` is the
same metric through hough_submit_host + hough_collect_begin/_end (three events in flight):
pinned HOST buffers in, complete results copied back to the host, every event.
`per_config` gives events/s and votes/s of every BASELINE.json event shape.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload batch100|pileup|...]
    python bench.py --impl reference ...   # the CPU oracle, as it stands, on the host cores

N > 1 is launched with torch.distributed.run; ranks take disjoint seed ranges of the same
event recipe (weak scaling, no data-path collective: the paper runs one event per GPU).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1305_4855_b200 import synth  # noqa: E402  (input generator only)

METRIC = "hough_votes_per_s"
UNIT = "votes/s"
# fp32 operations of one closed-form evaluation counting the divide as one:
# 3 for s, 2 for num, 3 for den, 1 divide, 2 compares, 2 for the bin, 1 convert, 1 min
FLOP_PER_EVAL = 15.0


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)),
                "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        if self.thread is not None:
            self.thread.join(timeout=5)
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0]))
                smax.append(float(r[1]))
                power.append(float(r[2]))
            except ValueError:
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)),
                "power_w_max": float(max(power)), "samples": len(sm), "reasons": sorted(reasons)}


def shard_seeds(rank, n_ev):
    """Weak scaling: rank r takes seeds r*E .. r*E+E-1 of the same event recipe (no exchange)."""
    return [rank * n_ev + s for s in range(n_ev)]


def aggregate(dist, dev, total_ms, votes_step, evals_step, n_ev, world):
    """(max-over-ranks time, summed votes, summed evaluations, summed events) -- the only
    collectives of the job, outside the timed region."""
    if world <= 1:
        return float(total_ms), float(votes_step), float(evals_step), float(n_ev)
    import torch
    t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    v = torch.tensor([votes_step, evals_step, n_ev], dtype=torch.float64, device=dev)
    dist.all_reduce(v, op=dist.ReduceOp.SUM)
    votes_all, evals_all, events_all = [float(a) for a in v.tolist()]
    return float(t.item()), votes_all, evals_all, events_all


def ncu_profile():
    """Figures copied from the committed `ncu --set full` summaries (profiles/ncu_traffic.json):
    DRAM bytes and warp instructions per launch of the sweep kernels.  They are NOT measured in
    this run (ncu cannot run inside a timed bench); every use says so."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if not os.path.exists(p):
        return {}
    with open(p) as f:
        return json.load(f)


KERNEL_SOURCES = ("hough_sweep.cu", "hough_peaklists.cu", "hough_device.cuh", "hough_internal.cuh")


def kernel_source_digest():
    """SHA-256 over the sources of the two sweep kernels.  profiles/ncu_traffic.json stores the digest of
    the tree its ncu counts were captured on; a different digest here means those counts (and every
    fraction derived from them) describe other code, and the line says `stale`."""
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_1305_4855_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def input_digest(event):
    """SHA-256 over x, y, layer of one generated event (inputs are seeded and
    reproducible; the digest lets two runs prove they measured the same hits)."""
    import hashlib
    h = hashlib.sha256()
    for a in event:
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()


def oracle_module():
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    try:
        import hough_oracle
    finally:
        sys.path.pop(0)
    hough_oracle.lib()
    return hough_oracle


def time_oracle(workload, seed):
    """The oracle as it stands on one event of the workload (vote + peaks + hit lists)."""
    o = oracle_module()
    x, y, layer, _ = synth.generate_event(workload.event, seed)
    t0 = time.perf_counter()
    acc, n_votes, _ = o.vote(workload.grid, x, y, layer)
    pb, _pm, _n = o.peaks(workload.grid, acc, workload.cap_peaks)
    o.hitlists(workload.grid, x, y, layer, pb, workload.cap_hits)
    dt = time.perf_counter() - t0
    return n_votes, len(x), dt, o.num_threads()


def run_reference(args, workload, rank):
    """--impl reference: the CPU oracle on the host cores, one event per step (bounded sample)."""
    if rank != 0:
        return
    for s in range(args.warmup):  # W untimed steps, as printed
        time_oracle(workload, workload.seeds[s % len(workload.seeds)])
    votes, secs, cores = 0, 0.0, 1
    for s in range(args.steps):
        nv, _n, dt, cores = time_oracle(workload, workload.seeds[s % len(workload.seeds)])
        votes += nv
        secs += dt
    val = votes / secs
    sample = "1 event per step (seeds 0..%d of the batch): vote + peaks + hit lists" % (args.steps - 1)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": {"workload": workload.name, "sample": sample},
            "events_per_s": args.steps / secs,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": sample,
                             "note": "untuned correctness oracle (scalar -O2, O(n_peaks x n_hits) "
                                     "hit-list passes): a reported baseline, not a performance target"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="batch100", choices=sorted(synth.WORKLOADS))
    ap.add_argument("--events", type=int, default=0, help="events per step (default: the workload's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the stage-time, sweep-roofline and micro-benchmark legs")
    ap.add_argument("--kernel-digest", action="store_true",
                    help="print the digest of the sweep kernels' sources (see profiles/) and exit")
    args = ap.parse_args()
    if args.kernel_digest:
        print(kernel_source_digest())
        return

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    workload = synth.WORKLOADS[args.workload]

    if args.impl == "reference":
        run_reference(args, workload, rank)
        return

    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the Hough path has no CPU fallback)")
    from paper_1305_4855_b200 import hough

    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    peaks_info = load_peaks()

    # ---- inputs: this rank's events (weak scaling: rank r takes seeds r*E .. r*E+E-1)
    n_ev = args.events if args.events > 0 else len(workload.seeds)
    seeds = shard_seeds(rank, n_ev)
    events = [synth.generate_event(workload.event, s)[:3] for s in seeds]
    max_hits = max(len(e[0]) for e in events)
    d_events = [tuple(torch.from_numpy(a).to(dev) for a in e) for e in events]
    pin_events = [tuple(torch.from_numpy(a).pin_memory() for a in e) for e in events]
    h = hough.Hough(workload.grid, max_hits, workload.cap_peaks, workload.cap_hits, device=local_rank)
    counts_all = torch.zeros(n_ev, hough.COUNTS_WORDS, dtype=torch.int64, device=dev)
    st = torch.cuda.current_stream()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)  # > the 126 MB L2

    def step():
        for e in range(n_ev):
            x, y, layer = d_events[e]
            h.vote(x, y, layer)
            h.peaks(counts_out=counts_all[e])

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    cnt = counts_all.cpu().numpy().view(hough.COUNTS_DTYPE).reshape(n_ev)
    votes_step = int(cnt["n_votes"].sum())
    evals_step = sum(len(e[0]) for e in events) * workload.grid.n_phi * workload.grid.n_d0
    evals_done_step = int(cnt["n_evals"].sum())
    assert int(cnt["flags"].max()) == 0, "output capacities overflowed"

    # ---- timed region: K steps, one CUDA-event pair per step, L2 flushed between steps
    launches0 = h.launch_count()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    barrier()
    step_ms = []
    t_wall0 = time.perf_counter()
    for _ in range(args.steps):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        step()
        e1.record(st)
        e1.synchronize()
        step_ms.append(e0.elapsed_time(e1))
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop() if rank == 0 else None
    launches = h.launch_count() - launches0
    total_ms = float(sum(step_ms))
    total_ms, votes_all, evals_all, events_all = aggregate(dist, dev, total_ms, votes_step, evals_step,
                                                           n_ev, world)
    secs = total_ms * 1e-3
    value = votes_all * args.steps / secs

    # ---- e2e: host buffers in, host results out, every event (hough_process_host)
    def e2e_step():
        # three events in flight: inputs of e+1 on the library's copy-in stream,
        # e computing, results of e-1 on the copy-out stream; every event's complete results land in
        # pinned host memory before its slot is reused
        nv = 0
        for e in range(n_ev):
            x, y, layer = pin_events[e]
            h.submit_host(x.numpy(), y.numpy(), layer.numpy(), e % 3)
            if e > 0:
                h.collect_begin((e - 1) % 3)
            if e > 1:
                nv += h.collect_end((e - 2) % 3)["n_votes"]
        h.collect_begin((n_ev - 1) % 3)
        if n_ev > 1:
            nv += h.collect_end((n_ev - 2) % 3)["n_votes"]
        nv += h.collect_end((n_ev - 1) % 3)["n_votes"]
        return nv

    def e2e_step_sync():
        nv = 0
        for e in range(n_ev):
            x, y, layer = pin_events[e]
            nv += h.process_host(x.numpy(), y.numpy(), layer.numpy())["n_votes"]
        return nv

    e2e_step()
    barrier()
    t0 = time.perf_counter()
    nv_e2e = 0
    for _ in range(args.steps):
        nv_e2e += e2e_step()
    torch.cuda.synchronize(dev)
    e2e_secs = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([e2e_secs], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_secs = float(t.item())
    assert nv_e2e == votes_step * args.steps
    h2d = sum(len(e[0]) for e in events) * 12
    idx_bytes = 2 if max_hits <= 65536 else 4  # the lists come back as 16-bit indices when they fit (hit_index16)
    d2h = int(sum(48 + min(int(c["n_peaks"]), workload.cap_peaks) * 16 + 8 +
                  min(int(c["n_hit_entries"]), workload.cap_hits) * idx_bytes for c in cnt))
    e2e = {"value": votes_all * args.steps / e2e_secs, "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "events_per_s": events_all * args.steps / e2e_secs,
           "api": "hough_submit_host + hough_collect_begin/_end (three events in flight: copy-in, compute and "
                  "copy-out streams); complete results per event: counters, peak bins and masks, 64-bit list "
                  "offsets, hit lists as %d-bit indices" % (8 * idx_bytes)}
    if rank == 0 and world == 1:
        h.process_host(*[t.numpy() for t in pin_events[0]])  # allocates its pinned buffers
        t0 = time.perf_counter()
        e2e_step_sync()
        torch.cuda.synchronize(dev)
        e2e["events_per_s_one_at_a_time"] = n_ev / (time.perf_counter() - t0)  # hough_process_host


    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": workload.name, "events_per_step": n_ev,
                       "grid": [workload.grid.n_phi, workload.grid.n_d0, workload.grid.n_kappa],
                       "L_min": workload.grid.L_min, "hits_per_event": int(np.mean([len(e[0]) for e in events])),
                       "l2": "512 MiB flush buffer written between steps, outside the event pairs",
                       "parallelism": "replicas x%d (events sharded by seed, no collective)" % world},
            "ms_per_step_median": float(np.median(step_ms)), "ms_per_step_best": float(np.min(step_ms)),
            "inputs_sha256_first_event": input_digest(events[0]),
            "events_per_s": events_all * args.steps / secs,
            "evaluations_per_s": evals_all * args.steps / secs,
            "votes_per_event": votes_step / n_ev,
            "wall_s_timed_region": t_wall,
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks}

    if rank == 0 and not args.no_extras:
        line.update(extras(args, hough, torch, workload, d_events, n_ev, dev, local_rank, peaks_info,
                           votes_step, evals_step, evals_done_step, flush))
    if rank == 0 and not args.no_cpu_baseline and world == 1:
        # single-threaded oracle on the small 3-D config ("(a) single-threaded")
        o = oracle_module()
        small = synth.WORKLOADS["displaced3d"]
        nthr = o.num_threads()
        o.set_num_threads(1)
        nv1, _n1, dt1, _c = time_oracle(small, small.seeds[0])
        o.set_num_threads(nthr)
        line["cpu_baseline_1thread"] = {"value": nv1 / dt1, "unit": UNIT, "cores": 1, "kind": "oracle",
                                        "sample": "displaced3d (configs[1]), 1 event, %.1f s" % dt1}
        nv, _n, dt, cores = time_oracle(workload, workload.seeds[0])
        line["cpu_baseline"] = {"value": nv / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "events_per_s": 1.0 / dt,
                                "note": "untuned correctness oracle (scalar -O2, O(n_peaks x n_hits) "
                                        "hit-list passes): a reported baseline, not a performance target",
                                "sample": "1 of the %d events (seed 0), whole path: vote + peaks + "
                                          "hit lists, %.1f s" % (n_ev, dt)}
    h.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


def extras(args, hough, torch, workload, d_events, n_ev, dev, local_rank, peaks_info, votes_step,
           evals_step, evals_done_step, flush):
    """Per-kernel times measured live (CUDA events on the launching stream, recorded by the
    library around every kernel), the roofline of the measured dominant kernel, the
    shared-atomic micro-benchmark and the HBM roofline of the stand-alone accumulator sweeps."""
    out = {}
    g = workload.grid
    ht = hough.Hough(g, max(len(e[0]) for e in d_events), workload.cap_peaks,
                     workload.cap_hits, device=local_rank, options=hough.OPT_STAGE_TIMING)
    acc = {}
    reps = 2
    peak_cells, list_evals_done, hits_x_peak_cells = 0, 0, 0
    for r in range(reps + 1):
        for e in range(n_ev):
            x, y, layer = d_events[e]
            ht.vote(x, y, layer)
            ht.peaks()
            if r > 0:
                for k, v in ht.stage_times().items():
                    acc[k] = acc.get(k, 0.0) + v
            else:
                # algorithmic work of the hit-list sweep: every hit against
                # every (phi0, d0) cell that holds at least one reported peak
                res = ht.read(lists=False)
                cells = int(np.unique(res["peak_bin"] // np.uint32(g.n_kappa)).size)
                peak_cells += cells
                hits_x_peak_cells += cells * int(x.numel())
                list_evals_done += int(ht.read_counts()["n_list_evals"])
    ht.close()
    per_event = {k: v / (reps * n_ev) for k, v in acc.items()}
    out["stage_ms_per_event"] = {k: round(v, 5) for k, v in per_event.items()}
    tot = sum(per_event.values())
    dom = max(per_event, key=per_event.get)
    out["stage_share"] = {k: round(v / tot, 4) for k, v in per_event.items()}
    out["dominant_stage_measured"] = dom

    n_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    alu_peak = n_sms * 128 * peaks_info["sm_max_mhz"] * 1e6 / 1e12  # fp32 lanes x clock, no FMA
    issue_peak = n_sms * 4 * peaks_info["sm_max_mhz"] * 1e6          # warp instructions / s
    prof = ncu_profile()
    sweeps = prof.get("_sweeps", {})
    digest = kernel_source_digest()
    stale = sweeps.get("source_sha256") != digest  # the committed ncu counts were taken on other kernel sources
    out["kernel_source_sha256"] = digest
    alu_note = ("bound = plain fp32 ALU issue (no dense contraction, 0 HBM bytes per evaluation); "
                "algorithmic fp32 ops = 15 per closed-form evaluation (DESIGN.md 5.1) x the evaluations the "
                "method defines for this launch; peak = SMs x 128 fp32 lanes x sm_max_mhz without FMA (the "
                "recipe forbids contraction); " + peaks_info["source"] + ". `frac` follows the contract "
                "(algorithmic work / time / peak) and can exceed 1 because the conservative cull proves most "
                "evaluations cannot vote and skips them; `frac_executed` counts only evaluations actually "
                "run.  `frac` is the issue-slot fraction: warp instructions per launch (committed ncu capture, "
                "see `instructions_source`; `stale` is true when the kernel sources have changed since) / live "
                "CUDA-event time / (SMs x 4 schedulers x sm_max_mhz): the ceiling SURVEY.md 8(d) names for "
                "these kernels; `achieved`, `peak` and `algorithmic_equiv_frac` keep the algorithmic fp32 "
                "figure (which can exceed 1 because the conservative cull skips evaluations).")

    def sweep_roofline(kernel, stage, alg_evals, done_evals, key):
        secs = per_event[stage] * 1e-3
        achieved = FLOP_PER_EVAL * alg_evals / secs / 1e12
        r = {"kernel": kernel, "stage": stage, "bound": "alu", "achieved": achieved, "peak": alu_peak,
             "unit": "TFLOP/s", "frac": achieved / alu_peak,
             "traffic": prof.get(key), "traffic_source": "committed profile (profiles/ncu_traffic.json), "
                                                         "not measured in this run",
             "ms_per_launch": per_event[stage],
             "algorithmic_evaluations_per_launch": alg_evals,
             "executed_evaluations_per_launch": done_evals,
             "executed_frac": done_evals / alg_evals if alg_evals else None,
             "achieved_executed": FLOP_PER_EVAL * done_evals / secs / 1e12,
             "frac_executed": FLOP_PER_EVAL * done_evals / secs / 1e12 / alu_peak}
        instr = sweeps.get(key, {}).get("warp_instructions")
        r["algorithmic_equiv_frac"] = r["frac"]  # algorithmic fp32 work / time / ALU peak (can exceed 1: the cull)
        if instr:
            # the ceiling of these kernels is the issue slots: `frac` is the share of them
            # in use = warp instructions per launch (committed ncu capture) / live time / issue peak
            r["issue_slot_frac"] = instr / secs / issue_peak
            r["algorithmic_achieved_tflops"], r["alu_peak_tflops"] = r["achieved"], r["peak"]
            r["achieved"], r["peak"], r["unit"] = instr / secs, issue_peak, "warp-inst/s"
            r["frac"] = r["hardware_frac"] = r["issue_slot_frac"]
            r["frac_is"] = "issue slots used: warp instructions / time / (SMs x 4 schedulers x clock)"
            r["warp_instructions_per_launch"] = instr
            r["instructions_source"] = sweeps.get("source")
            r["issue_active_pct_ncu"] = sweeps.get(key, {}).get("issue_active_pct")
            r["stale"] = stale
        else:
            r["frac_is"] = "algorithmic fp32 work / time / ALU peak (no ncu instruction count committed)"
        return r

    rl_vote = sweep_roofline("k_sweep (vote)", "vote", evals_step / n_ev, evals_done_step / n_ev, "vote")
    rl_list = sweep_roofline("k_peak_lists (hit lists)", "lists", hits_x_peak_cells / n_ev,
                             list_evals_done / n_ev, "lists")
    rl_list["cells_with_reported_peaks_per_event"] = peak_cells / n_ev
    by_stage = {"vote": rl_vote, "lists": rl_list}
    # the contract's `roofline` describes the MEASURED dominant stage; the other sweep sits beside it
    primary = by_stage.get(dom, rl_vote)
    out["roofline"] = dict(primary, note=alu_note, dominant_stage_measured=dom)
    for k, v in by_stage.items():
        if v is not primary:
            out["roofline_" + k] = v

    # shared-atomic roofline: conflict-free no-return atomicOr micro-benchmark on this box
    vote_s = per_event["vote"] * 1e-3
    best = 0.0
    for thr, cps in ((1024, 2), (512, 4), (256, 8)):
        best = max(best, hough.microbench_smem(0, thr, cps, 4096, device=local_rank))
    rnd = hough.microbench_smem(1, 512, 4, 4096, device=local_rank)
    vps = (votes_step / n_ev) / vote_s
    out["roofline_smem_atomic"] = {"bound": "smem_atomic", "achieved": vps, "peak": best,
                                   "unit": "lane-atomics/s", "frac": vps / best,
                                   "peak_random_addresses": rnd,
                                   "note": "votes cast / vote-kernel time vs the conflict-free "
                                           "atomicOr micro-benchmark (hough_microbench_smem mode 0); "
                                           "structurally capped near 7 % by the issue slots of one exactly "
                                           "rounded divide per vote (DESIGN.md 5.1)"}

    # the unpruned sweep (HOUGH_OPT_NO_CULL: every hit x cell is evaluated), SURVEY.md 8(d):
    # "report the fraction honestly for both the pruned and unpruned kernels"
    hn = hough.Hough(g, max(len(e[0]) for e in d_events), workload.cap_peaks,
                     workload.cap_hits, device=local_rank,
                     options=hough.OPT_STAGE_TIMING | hough.OPT_NO_CULL)
    t_nc, n_nc = 0.0, min(n_ev, 3)
    for r in range(2):
        for e in range(n_nc):
            x, y, layer = d_events[e]
            hn.vote(x, y, layer)
            hn.peaks(lists=False)
            if r > 0:
                t_nc += hn.stage_times()["vote"]
    hn.close()
    vote_nc_s = t_nc / n_nc * 1e-3
    out["vote_unpruned"] = {
        "ms_per_event": vote_nc_s * 1e3, "evaluations_per_s": (evals_step / n_ev) / vote_nc_s,
        "alu_frac": FLOP_PER_EVAL * (evals_step / n_ev) / vote_nc_s / 1e12 / alu_peak,
        "smem_atomic_frac": (votes_step / n_ev) / vote_nc_s / best,
        "note": "same kernel with the conservative cull switched off: executed = algorithmic evaluations"}
    if sweeps:
        out["ncu_sweeps"] = dict(sweeps, note="copied from the committed ncu capture, not measured in this run")

    # the rows after the hot path, on the same events: f2 fit + duplicate removal, f1 second
    # transform over the peaks; device times per event, CUDA events around the C-ABI calls
    hx = hough.Hough(g, max(len(e[0]) for e in d_events), workload.cap_peaks, workload.cap_hits, device=local_rank)
    st0 = torch.cuda.current_stream()
    t_fit, t_vx, n_x, kept, nvx = 0.0, 0.0, 0, 0, 0
    for r in range(2):
        for ev in d_events[:min(n_ev, 5)]:
            hx.vote(*ev)
            hx.peaks()
            ea, eb, ec = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            ea.record(st0)
            hx.fit(0.01, 3)
            eb.record(st0)
            hx.vertices(synth.JETS_VGRID)
            ec.record(st0)
            ec.synchronize()
            if r > 0:
                t_fit += ea.elapsed_time(eb)
                t_vx += eb.elapsed_time(ec)
                n_x += 1
                kept += hx.read_fit()["n_kept"]
                nvx += hx.read_vertices()["n_vertices"]
    hx.close()
    out["next_rows"] = {"hough_fit_ms_per_event": t_fit / n_x, "hough_vertices_ms_per_event": t_vx / n_x,
                        "tracks_kept_per_event": kept / n_x, "vertices_per_event": nvx / n_x,
                        "note": "f2: circle fit of every peak's list, selection at rms <= 100 um, duplicates sharing "
                                ">= 3 hits removed; f1: second transform of all reported peaks into a 32 x 32 vertex "
                                "grid (parity against the oracle in tests/test_gpu_ext.py)"}

    # f4, second half (SURVEY.md 8(f) "multi-event"): two handles on two streams, events
    # alternating between them, so that the small latency-bound kernels of one event run beside the
    # issue-bound vote of the other.  Not the headline (BASELINE.json configs[3] is one stream, back to back).
    h2 = [hough.Hough(g, max(len(e[0]) for e in d_events), workload.cap_peaks, workload.cap_hits, device=local_rank)
          for _ in range(2)]
    s2 = [torch.cuda.Stream(device=dev) for _ in range(2)]

    def two_stream_pass():
        for e in range(n_ev):
            h2[e & 1].vote(*d_events[e], stream=s2[e & 1])
            h2[e & 1].peaks(stream=s2[e & 1])

    two_stream_pass()
    torch.cuda.synchronize(dev)
    t0 = time.perf_counter()
    for _ in range(3):
        two_stream_pass()
    torch.cuda.synchronize(dev)
    dt2 = time.perf_counter() - t0
    for hh in h2:
        hh.close()
    out["two_handles_two_streams"] = {"events_per_s": 3 * n_ev / dt2, "ms_per_event": dt2 / (3 * n_ev) * 1e3,
                                      "note": "device-resident, wall clock over 3 passes with a device synchronise on "
                                              "both sides; each handle has its own workspace and output arrays"}

    # every BASELINE.json event shape (north_star: "throughput on the synthetic event shapes ... as votes/s and
    # events/s"): device-resident, back to back on one stream (CUDA events), and one at a time through
    # hough_process_host with host buffers (wall clock)
    def shape_rate(wl, n_events, reps):
        evs_h = [synth.generate_event(wl.event, sd)[:3] for sd in range(n_events)]
        evs_d = [tuple(torch.from_numpy(a).to(dev) for a in e) for e in evs_h]
        hs = hough.Hough(wl.grid, max(len(e[0]) for e in evs_h), wl.cap_peaks, wl.cap_hits, device=local_rank)
        cs = torch.zeros(n_events, hough.COUNTS_WORDS, dtype=torch.int64, device=dev)
        stq = torch.cuda.current_stream()

        def one_pass():
            for q, ev in enumerate(evs_d):
                hs.vote(*ev)
                hs.peaks(counts_out=cs[q])

        one_pass()
        torch.cuda.synchronize(dev)
        c = cs.cpu().numpy().view(hough.COUNTS_DTYPE).reshape(n_events)
        assert int(c["flags"].max()) == 0
        ms = []
        for _ in range(reps):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stq)
            one_pass()
            e1.record(stq)
            e1.synchronize()
            ms.append(e0.elapsed_time(e1))
        secs = float(np.median(ms)) * 1e-3
        hs.process_host(*evs_h[0])
        t0 = time.perf_counter()
        for ev in evs_h:
            hs.process_host(*ev)
        dt_host = time.perf_counter() - t0
        hs.close()
        votes = int(c["n_votes"].sum())
        return {"events_per_s": n_events / secs, "votes_per_s": votes / secs, "ms_per_event": secs / n_events * 1e3,
                "hits_per_event": int(np.mean([len(e[0]) for e in evs_h])),
                "peaks_per_event": float(c["n_peaks"].mean()),
                "e2e_one_at_a_time_events_per_s": n_events / dt_host, "events_timed": n_events, "passes": reps}

    out["per_config"] = {name: shape_rate(synth.WORKLOADS[name], n, r)
                         for name, n, r in (("prompt2d", 100, 5), ("displaced3d", 100, 5), ("pileup", 10, 5),
                                            ("finegrid", 2, 3))}
    out["per_config"]["batch100"] = "the headline of this line (value, events_per_s, e2e)" \
        if workload.name == "batch100" else None
    out["per_config"]["note"] = ("seeds 0..n-1 of each shape, one handle, one stream, back to back, median of the "
                                 "passes, 512 MiB L2 flush before each pass; e2e_one_at_a_time = hough_process_host "
                                 "(pageable numpy inputs, full results back, synchronous): the small shapes are bound "
                                 "by the 11-launch chain and host latency, not by arithmetic")

    # a5 variants, measured: stand-alone streaming sweep, peak test fused into the
    # vote tile + tile-edge pass (HOUGH_OPT_FUSED_PEAKS), cell-wise kernel over every cell
    def peak_variant(wl, evs, options, reps=3):
        hv = hough.Hough(wl.grid, max(int(e[0].numel()) for e in evs), wl.cap_peaks, wl.cap_hits,
                         device=local_rank, options=hough.OPT_STAGE_TIMING | options)
        tv, tp, n = 0.0, 0.0, 0
        for r in range(reps + 1):
            for ev in evs:
                hv.vote(*ev)
                hv.peaks(lists=False)
                if r > 0:
                    t = hv.stage_times()
                    tv += t["vote"]
                    tp += t["peak_sweep"]
                    n += 1
        hv.close()
        return {"vote_ms": tv / n, "peak_flags_ms": tp / n, "sum_ms": (tv + tp) / n}

    fine = synth.WORKLOADS["finegrid"]
    x, y, layer = [torch.from_numpy(a).to(dev) for a in synth.generate_event(fine.event, 0)[:3]]
    variants = (("standalone_sweep", 0), ("fused_tile_plus_edge_cells", hough.OPT_FUSED_PEAKS),
                ("cellwise_all_cells", hough.OPT_CELL_PEAKS))
    out["peak_variants"] = {
        workload.name: {k: peak_variant(workload, d_events[:min(n_ev, 5)], o) for k, o in variants},
        "finegrid": {k: peak_variant(fine, [(x, y, layer)], o, reps=2) for k, o in variants},
        "note": "per event, CUDA events around the kernels (hough_stage_times); peak_flags_ms = k_peak_sweep, "
                "or k_peak_cells over the tile-edge cells / all cells; the fused variant's interior test "
                "is inside vote_ms"}

    # HBM roofline of the accumulator sweeps, on the fine grid (512 MiB > L2)
    hf = hough.Hough(fine.grid, len(x), fine.cap_peaks, fine.cap_hits, device=local_rank)
    hf.vote(x, y, layer)
    st = torch.cuda.current_stream()

    def timed(fn, n=10):
        fn()
        ts = []
        for _ in range(n):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st)
            fn()
            e1.record(st)
            e1.synchronize()
            ts.append(e0.elapsed_time(e1))
        return float(np.mean(ts)) * 1e-3

    nbytes = fine.grid.n_bins * 4
    t_sweep = timed(hf.peak_sweep)
    t_clear = timed(hf.clear)
    hf.close()
    hbm = peaks_info["hbm_gbs"]
    out["roofline_sweep"] = {
        "kernel": "k_peak_sweep", "workload": "finegrid (512 MiB accumulator, L2 flushed)",
        "bound": "hbm", "achieved": nbytes / t_sweep / 1e9, "peak": hbm, "unit": "GB/s",
        "frac": nbytes / t_sweep / 1e9 / hbm, "frac_of_8TBs_nominal": nbytes / t_sweep / 8e12,
        "traffic": prof.get("peak_sweep_finegrid"),
        "traffic_source": "committed profile (profiles/ncu_traffic.json), not measured in this run",
        "note": "algorithmic bytes = 4 B/bin read once; " + peaks_info["source"]}
    out["roofline_clear"] = {
        "kernel": "k_clear", "bound": "hbm", "achieved": nbytes / t_clear / 1e9, "peak": hbm,
        "unit": "GB/s", "frac": nbytes / t_clear / 1e9 / hbm, "traffic": None}
    return out


if __name__ == "__main__":
    main()
