#!/usr/bin/env python
"""bench.py -- whole hot path (vote -> peaks -> tracks -> jets) on synthetic trigger batches, one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5|C4|C3] [--events E] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch (BASELINE.json configs[4] by default: 4,096 events,
12-layer tracker, 128 x 1024 x 512 accumulator per event, processed in chunks of --chunk events).  `value` is
whole-job events/s with the hits already resident in HBM; `e2e` is the same metric through hough_trigger_host
with pinned HOST buffers (H2D of the hits and D2H of the per-event results inside the timed region).  N > 1:
one rank per GPU (torchrun), every rank processes its own batch of the same size (weak scaling, no data-path
collective -- events are independent); time = max over ranks, value = all ranks' events / that time.

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample per step.
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

# FP32-pipe instructions per vote of the normative O-2 sequence in scalar form: 3D = t, a, b,
# den, the 6 FMA-pipe instructions of the IEEE division, v, u, the floor add + the per-hit m1, m2, s, rs, r2 shared by
# the rows of a lane; 2D = m1, m2, s, division, v, u, floor.  (The kernel issues them two per instruction.)
I_FP32 = {"3d": 15.0, "2d": 15.0}
SM_COUNT, FP32_LANES = 148, 128


# ----------------------------------------------------------------------------------------------------
# multi-GPU helpers (also exercised by the world_size-2 gloo test)
# ----------------------------------------------------------------------------------------------------

def shard_range(n_items: int, rank: int, world: int):
    """Contiguous, balanced [lo, hi) slice of n_items for `rank` of `world` (strong-scaling helper)."""
    base, rem = divmod(n_items, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks(x: float, dist=None) -> float:
    if dist is None or not dist.is_initialized():
        return x
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([x], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, dist=None) -> float:
    if dist is None or not dist.is_initialized():
        return x
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([x], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


# ----------------------------------------------------------------------------------------------------
# clocks during the timed region
# ----------------------------------------------------------------------------------------------------

class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.lines, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.lines:
            if not (t0 - 0.05 <= ts <= t1 + 0.15):
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except Exception:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


# ----------------------------------------------------------------------------------------------------
# workloads
# ----------------------------------------------------------------------------------------------------

def make_workload(name: str, n_events):
    from paper_1309_6275_b200 import workloads as W
    k = {"C1": 1, "C2": 2, "C3": 3, "C4": 4, "C5": 5}[name]
    w = W.config(k)
    if n_events:
        w = W.scaled(w, n_events=int(n_events))
    return w


def cpu_oracle_rate(w, batch, budget_s: float = 15.0):
    """The oracle as it stands, event-parallel over the host cores, on a bounded sample of the same batch."""
    from oracle import hough_oracle as O
    cores = max(1, min(os.cpu_count() or 1, 64))
    g = O.Grid.from_workload(w)
    t0 = time.time()
    O.run_event(g, *batch.event(0), w.l_min, w.max_peaks, w.max_jets, w.cone_rad, w.d0_cut_mm, w.n_displaced_min,
                keep_planes=False)
    t_one = time.time() - t0
    n = int(max(1, min(batch.n_events, cores * max(1, int(budget_s / max(t_one, 1e-3))))))
    sub = batch.slice(0, n)
    t0 = time.time()
    O.run_batch(g, sub, w.l_min, w.max_peaks, w.max_jets, w.cone_rad, w.d0_cut_mm, w.n_displaced_min,
                keep_planes=False, workers=cores)
    dt = time.time() - t0
    return {"value": n / dt, "unit": "events/s", "cores": min(cores, n), "kind": "oracle",
            "sample": f"first {n} of {batch.n_events} events of {w.name}, one event per worker thread, "
                      f"{dt:.1f} s wall ({t_one:.2f} s/event single-thread)"}


# ----------------------------------------------------------------------------------------------------
# the two arms
# ----------------------------------------------------------------------------------------------------

def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import hough_oracle as O
    from paper_1309_6275_b200 import workloads as W
    w = make_workload(args.workload, args.events)
    cores = max(1, min(os.cpu_count() or 1, 64))
    g = O.Grid.from_workload(w)
    probe = W.generate(w, 1)
    t0 = time.time()
    O.run_event(g, *probe.event(0), w.l_min, w.max_peaks, w.max_jets, w.cone_rad, w.d0_cut_mm, w.n_displaced_min,
                keep_planes=False)
    t_one = time.time() - t0
    per_step = int(max(1, min(w.n_events, cores * max(1, int(12.0 / max(t_one * (args.steps + args.warmup), 1e-3))))))
    batch = W.generate(w, per_step)
    run = lambda: O.run_batch(g, batch, w.l_min, w.max_peaks, w.max_jets, w.cone_rad, w.d0_cut_mm,
                              w.n_displaced_min, keep_planes=False, workers=cores)
    for _ in range(args.warmup):
        run()
    t0 = time.time()
    for _ in range(args.steps):
        run()
    dt = time.time() - t0
    value = per_step * args.steps / dt
    sample = f"{per_step} events of {w.name} per step, one event per worker thread"
    print(json.dumps({
        "impl": "reference", "metric": "events_per_sec", "value": value, "unit": "events/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "events_per_step": per_step, "grid": [w.n_d0, w.n_phi0, w.n_kappa]},
        "cpu_baseline": {"value": value, "unit": "events/s", "cores": min(cores, per_step), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_ours(args):
    import torch
    from paper_1309_6275_b200 import binding as B
    from paper_1309_6275_b200 import workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", rank=rank, world_size=world)

    w = make_workload(args.workload, args.events)
    E = w.n_events
    # events per vote/peaks/jets launch: --chunk, else as many as fit in about 34 GB of planes (C5: 128 events)
    chunk = args.chunk if args.chunk > 0 else max(1, int(34.4e9 // (4 * w.bins_per_event)))
    chunk = min(chunk, E)
    mode = "3d" if w.n_d0 > 1 else "2d"
    # weak scaling: every rank owns a batch of E events (event indices continue across ranks)
    batch = W.generate(w, E, first_event=rank * E)
    H = batch.n_hits
    bins = w.bins_per_event

    h = B.Hough.for_workload(w, max_events=chunk, max_hits=H)
    offs = batch.hit_offsets.astype(np.int64)
    off, r, phi, layer = B.upload_batch(batch)
    count, mask = h.alloc_planes(chunk)
    out = h.alloc_outputs(E)
    stream = torch.cuda.current_stream()
    n_chunks = (E + chunk - 1) // chunk
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def one_step(stage_events=None, votes_acc=None):
        for ci in range(n_chunks):
            e0 = ci * chunk
            ne = min(chunk, E - e0)
            t = [ev() for _ in range(4)] if stage_events is not None else None
            if t: t[0].record(stream)
            hb, he = int(offs[e0]), int(offs[e0 + ne])
            h.hough_vote(ne, off[e0:e0 + ne + 1], he - hb, r[hb:he], phi[hb:he], layer[hb:he], count, mask, stream)
            if t: t[1].record(stream)
            h.hough_peaks(ne, count, mask, w.l_min, out["peaks"][e0:], out["n_peaks"][e0:], stream)
            if t: t[2].record(stream)
            h.hough_jets(ne, out["peaks"][e0:], out["n_peaks"][e0:], w.cone_rad, w.d0_cut_mm, w.n_displaced_min,
                         out["tracks"][e0:], out["jets"][e0:], out["n_jets"][e0:], out["flag"][e0:], stream)
            if t:
                t[3].record(stream)
                stage_events.append(t)
            if votes_acc is not None:
                votes_acc.append(int((count[:ne].to(torch.int32) & 0xFFFF).sum(dtype=torch.int64).item()))

    # warm-up (the first warm-up step also counts the votes, untimed)
    votes_chunks = []
    for i in range(args.warmup):
        one_step(votes_acc=votes_chunks if i == 0 else None)
    if not votes_chunks:
        one_step(votes_acc=votes_chunks)
    votes_per_step = float(sum(votes_chunks))
    torch.cuda.synchronize()
    if dist: dist.barrier()

    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    launches0 = h.hough_launch_count()
    stage_events = []
    t_start, t_stop = ev(), ev()
    torch.cuda.synchronize()
    wall0 = time.time()
    t_start.record(stream)
    for _ in range(args.steps):
        one_step(stage_events=stage_events)
    t_stop.record(stream)
    torch.cuda.synchronize()
    wall1 = time.time()
    if dist: dist.barrier()
    ms_total = t_start.elapsed_time(t_stop)
    clocks = sampler.stop(wall0, wall1)
    launches = h.hough_launch_count() - launches0
    status = h.hough_status()

    ms_vote = sum(t[0].elapsed_time(t[1]) for t in stage_events)
    ms_peaks = sum(t[1].elapsed_time(t[2]) for t in stage_events)
    ms_jets = sum(t[2].elapsed_time(t[3]) for t in stage_events)
    n_flag = int(out["flag"].sum().item())
    n_peaks_total = int(out["n_peaks"].to(torch.int64).sum().item())

    ms_max = max_over_ranks(ms_total, dist)
    total_events = sum_over_ranks(float(E * args.steps), dist)
    value = total_events / (ms_max * 1e-3)

    # ---- e2e: the same batch through hough_trigger_host with pinned host buffers ----
    del count, mask
    h.close()
    torch.cuda.empty_cache()
    h2 = B.Hough.for_workload(w, max_events=E, max_hits=H, host_chunk_events=chunk)
    pin = lambda a: torch.from_numpy(a).pin_memory()
    h_off, h_r, h_phi, h_layer = pin(batch.hit_offsets.view(np.int32)), pin(batch.r), pin(batch.phi), pin(batch.layer)
    h_np = torch.zeros(E, dtype=torch.int32).pin_memory(); h_nj = torch.zeros(E, dtype=torch.int32).pin_memory()
    h_fl = torch.zeros(E, dtype=torch.uint8).pin_memory()
    e2e_steps = max(1, min(args.steps, 3))
    call = lambda: h2.hough_trigger_host(E, h_off, H, h_r, h_phi, h_layer, w.l_min, w.cone_rad, w.d0_cut_mm,
                                         w.n_displaced_min, h_np, h_nj, h_fl, None, None, None, stream)
    call()
    torch.cuda.synchronize()
    if dist: dist.barrier()
    a, b = ev(), ev()
    a.record(stream)
    for _ in range(e2e_steps):
        call()
    b.record(stream)
    torch.cuda.synchronize()
    ms_e2e = max_over_ranks(a.elapsed_time(b), dist)
    e2e_value = sum_over_ranks(float(E * e2e_steps), dist) / (ms_e2e * 1e-3)
    e2e_ok = bool(np.array_equal(h_fl.numpy(), out["flag"].cpu().numpy()) and
                  np.array_equal(h_np.numpy(), out["n_peaks"].cpu().numpy()))
    h2_launches = h2.hough_launch_count()
    h2.close()

    if rank != 0:
        if dist: dist.destroy_process_group()
        return

    hbm_gbs, sm_max_mhz, peak_src = measured_peaks()
    # roofline of the dominant kernel (vote): FP32-pipe bound (max of atomics / FP32 / HBM-write terms)
    vote_s = ms_vote * 1e-3
    votes_timed = votes_per_step * args.steps
    fp32_peak = SM_COUNT * FP32_LANES * sm_max_mhz * 1e6            # thread-instructions / s, no FMA credit
    achieved_instr = votes_timed * I_FP32[mode] / vote_s
    t_hbm = 4.0 * bins * E * args.steps / (hbm_gbs * 1e9)
    t_fp32 = votes_timed * I_FP32[mode] / fp32_peak
    bound = "alu" if t_fp32 >= t_hbm else "hbm"
    # dram__bytes_read.sum + dram__bytes_write.sum of one vote launch (ncu --set full, profiles/r01c_summary.md);
    # only known for the launch shape that capture was taken on (C5, 128 events per launch)
    traffic = 34.33 if (w.name.startswith("C5") and chunk == 128) else None
    if bound == "alu":
        roofline = {"bound": "alu", "achieved": achieved_instr / 1e12, "peak": fp32_peak / 1e12, "unit": "Tinstr/s",
                    "frac": achieved_instr / fp32_peak, "traffic": None}
    else:
        ach = 4.0 * bins * E * args.steps / vote_s / 1e9
        roofline = {"bound": "hbm", "achieved": ach, "peak": hbm_gbs, "unit": "GB/s", "frac": ach / hbm_gbs,
                    "traffic": traffic, "traffic_unit": "GB per launch (algorithmic: %.2f)" % (4.0 * bins * chunk / 1e9)}
    roofline.update({"kernel": "vote_kernel", "peak_source": peak_src + "; FP32 peak = 148 SM x 128 lanes x sm_max clock",
                     "ms_per_launch": ms_vote / max(1, len(stage_events)), "launches": len(stage_events),
                     "i_fp32_per_vote": I_FP32[mode], "t_bound_terms_ms": {"fp32": t_fp32 * 1e3, "hbm_write": t_hbm * 1e3},
                     "note": "duration = CUDA events around hough_vote (includes the two small A0 prep kernels)"})
    stencil_bytes = 2.0 * bins * E * args.steps
    ach_st = stencil_bytes / (ms_peaks * 1e-3) / 1e9
    roofline_stencil = {"bound": "hbm", "kernel": "peak_stencil_kernel+peak_compact_kernel", "achieved": ach_st,
                        "peak": hbm_gbs, "unit": "GB/s", "frac": ach_st / hbm_gbs, "traffic": None,
                        "ms_per_launch": ms_peaks / max(1, len(stage_events))}

    cpu = cpu_oracle_rate(w, batch) if not args.no_cpu_baseline else None

    line = {
        "metric": "events_per_sec", "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "events_per_gpu": E, "chunk_events": chunk, "hits": H,
                   "grid": [w.n_d0, w.n_phi0, w.n_kappa], "l_min": w.l_min, "cone_rad": w.cone_rad,
                   "l2": "working set >> L2: 268 MB of planes per event, rewritten every chunk"},
        "votes_per_sec": votes_timed * world / (ms_max * 1e-3) if world == 1 else None,
        "votes_per_step": votes_per_step,
        "stage_ms_per_step": {"vote": ms_vote / args.steps, "peaks": ms_peaks / args.steps, "jets": ms_jets / args.steps},
        "events_flagged": n_flag, "peaks_total": n_peaks_total, "status_bits": status,
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "events/s", "h2d_bytes_per_step": int(H * 9 + (E + 1) * 4),
                "d2h_bytes_per_step": int(E * 9), "steps": e2e_steps, "matches_device_path": e2e_ok},
        "gpu_launches": int(launches), "gpu_launches_e2e": int(h2_launches),
        "roofline": roofline, "roofline_stencil": roofline_stencil,
    }
    if cpu:
        line["cpu_baseline"] = cpu
    print(json.dumps(line))
    if dist: dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C5", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--events", type=int, default=0, help="override the number of events per GPU (0 = the config's)")
    ap.add_argument("--chunk", type=int, default=0, help="events per vote/peaks/jets launch (0: what fits in 34 GB of planes)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
