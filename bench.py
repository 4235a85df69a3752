#!/usr/bin/env python
"""bench.py -- whole hot path (vote -> peaks -> tracks -> jets) on synthetic trigger batches, one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5|C4|C3|C2|C1|P4|F8|F9|F10] [--events E]
                  [--path fused|planes] [--impl ours|reference] [--tracks N]

A "step" is one pass of the whole hot path over one batch (BASELINE.json configs[4] by default: 4,096 events,
12-layer tracker, 128 x 1024 x 512 accumulator per event, processed in launches of --chunk events).  The default
path is the fused one (hough_vote_peaks + hough_jets: peaks are found while the accumulator tile is in shared memory,
no planes in HBM); --path planes times hough_vote + hough_peaks + hough_jets on accumulator planes instead, and a short
leg of it is measured in every run for the stencil's roofline.  `value` is whole-job events/s with the hits already
resident in HBM; `e2e` is the same metric through hough_trigger_host with pinned HOST buffers (H2D of the hits and
D2H of n_peaks / n_jets / flag / jets inside the timed region).

N > 1: one rank per GPU.  `python bench.py --gpus N` re-executes itself under torch.distributed.run when it was not
launched by it; every rank processes its own batch of the same size (weak scaling: events are independent, no
data-path collective), the per-event flags are all_gathered once per step (the only exchange),
time = max over ranks, value = all ranks' events / that time.

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample per step.
"""
from __future__ import annotations

import argparse
import csv
import glob
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

# FP32 (FMA-pipe) instructions per vote of the normative O-2 sequence written plainly: FADD / FMUL / FFMA in the SASS
# of the stand-alone function csrc/o2_count.cu (IEEE division = 5 FFMA + MUFU.RCP + FCHK; the compares, F2I, MUFU and
# FCHK run on other pipes and are not counted).  tests/test_abi_and_host.py::test_o2_instruction_count recounts them
# from the SASS; profiles/r02_o2_sass_count.md holds the listing.  (Round 1 used a hand count of 15.)
I_FP32 = {"3d": 17.0, "2d": 11.0}
# the same with the five per-(hit, column) operations of 3D (m1, m2, s, rs, r2) taken as shared by the d0 bins of the
# column (SURVEY.md 8(d) counts them "per (hit, ip)"): a stricter denominator, reported next to the contract's
I_FP32_SHARED = {"3d": 12.0, "2d": 11.0}
SM_COUNT, FP32_LANES = 148, 128
STAGES = ("prep", "vote", "peaks", "jets", "vertices")
SMEM_RED_PER_CLK = 32                                         # conflict-free 32-bit shared reductions per clock and SM


# ----------------------------------------------------------------------------------------------------
# multi-GPU helpers (exercised on CPU by the world_size-2 gloo test)
# ----------------------------------------------------------------------------------------------------

def shard_range(n_items: int, rank: int, world: int):
    """Contiguous, balanced [lo, hi) slice of n_items for `rank` of `world` (strong-scaling helper)."""
    base, rem = divmod(n_items, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def _dist_dev(dist):
    return "cuda" if dist.get_backend() == "nccl" else "cpu"


def max_over_ranks(x: float, dist=None) -> float:
    if dist is None or not dist.is_initialized():
        return x
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=_dist_dev(dist))
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, dist=None) -> float:
    if dist is None or not dist.is_initialized():
        return x
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=_dist_dev(dist))
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def first_event_of_rank(n_events_per_rank: int, rank: int) -> int:
    """Weak scaling: rank r owns the events [r * E, (r + 1) * E) of the synthetic stream."""
    return rank * n_events_per_rank


def gather_event_results(flag, n_peaks, n_jets, dist=None):
    """The one exchange of the sharded job: every rank contributes flag[E] (u8), n_peaks[E] and
    n_jets[E] (i32) of its own events; returns the three [world, E] tensors (identical on every rank; rank r's
    events are row r).  Without a process group the inputs come back as [1, E]."""
    import torch
    if dist is None or not dist.is_initialized():
        return flag[None], n_peaks[None], n_jets[None]
    world = dist.get_world_size()
    outs = []
    for t in (flag, n_peaks, n_jets):
        g = torch.empty(world * t.numel(), dtype=t.dtype, device=t.device)      # concatenation along dim 0
        dist.all_gather_into_tensor(g, t.contiguous().view(-1))
        outs.append(g.view((world,) + tuple(t.shape)))
    return tuple(outs)


def reexec_under_torchrun(args, argv):
    """`python bench.py --gpus N` (N > 1) without a launcher: start N ranks on this node and forward their output."""
    port = 29500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + argv
    raise SystemExit(subprocess.call(cmd))


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


def traffic_from_profiles(kernel_substr: str, tag: str = ""):
    """(dram__bytes_read.sum + dram__bytes_write.sum in GB per launch, file name, FMA-pipe busy fraction) of the newest
    committed `ncu --page raw --csv` export under profiles/ whose kernel name contains kernel_substr (e.g. "vote_kernel<1,"
    = the 3D kernels) and whose file name contains `tag` (the workload the capture was taken on); (None, None, None) if
    there is none.  The pipe fraction is sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_elapsed / 100: what
    the FP32 pipe was measured to do, next to the model-work fraction the roofline reports."""
    best = (None, None, None)
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_ncu_raw.csv"))):
        if tag and tag not in os.path.basename(path):
            continue
        try:
            rows = list(csv.reader(open(path, newline="")))
        except Exception:
            continue
        if len(rows) < 3:
            continue
        head, units = rows[0], rows[1]
        try:
            i_name = head.index("Kernel Name")
            i_r, i_w = head.index("dram__bytes_read.sum"), head.index("dram__bytes_write.sum")
        except ValueError:
            continue
        scale = {"byte": 1e-9, "Kbyte": 1e-6, "Mbyte": 1e-3, "Gbyte": 1.0, "Tbyte": 1e3}
        for row in rows[2:]:
            if kernel_substr in row[i_name]:
                try:
                    gb = float(row[i_r].replace(",", "")) * scale[units[i_r]] + \
                         float(row[i_w].replace(",", "")) * scale[units[i_w]]
                except Exception:
                    continue
                fma = None
                try:
                    fma = float(row[head.index("sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_elapsed")]) / 100.0
                except Exception:
                    pass
                best = (gb, os.path.basename(path), fma)
    return best


# ----------------------------------------------------------------------------------------------------
# workloads
# ----------------------------------------------------------------------------------------------------

def make_workload(name: str, n_events):
    from paper_1309_6275_b200 import workloads as W
    if name == "P4":
        return W.paper_timing(3000, int(n_events) if n_events else 32)
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
# the reference arm = the oracle
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


# ----------------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------------

class DeviceRun:
    """One workload resident on the device: context, uploaded hits, output tensors, and the step function."""

    def __init__(self, w, batch, chunk: int, path: str, vertices: bool = True):
        import torch
        from paper_1309_6275_b200 import binding as B
        self.torch, self.B, self.w, self.batch, self.path = torch, B, w, batch, path
        self.E = batch.n_events
        self.chunk = min(chunk, self.E)
        self.offs = batch.hit_offsets.astype(np.int64)
        self.n_chunks = (self.E + self.chunk - 1) // self.chunk
        hits_per_chunk = max(int(self.offs[min(c + self.chunk, self.E)] - self.offs[c]) for c in range(0, self.E, self.chunk))
        self.vertices = vertices and w.n_d0 > 1                  # the second Hough transform needs displaced tracks
        self.h = B.Hough.for_workload(w, max_events=self.chunk, max_hits=max(1, hits_per_chunk),
                                      vgrid=w.vgrid if self.vertices else None, max_vertices=w.max_vertices)
        self.off, self.r, self.phi, self.layer = B.upload_batch(batch)
        self.out = self.h.alloc_outputs(self.E)
        self.count = self.mask = None
        if path == "planes":
            self.count, self.mask = self.h.alloc_planes(self.chunk)
        self.stream = torch.cuda.current_stream()

    def step(self):
        h, w, out, st = self.h, self.w, self.out, self.stream
        for ci in range(self.n_chunks):
            e0 = ci * self.chunk
            ne = min(self.chunk, self.E - e0)
            hb, he = int(self.offs[e0]), int(self.offs[e0 + ne])
            a = (ne, self.off[e0:e0 + ne + 1], he - hb, self.r[hb:he], self.phi[hb:he], self.layer[hb:he])
            if self.path == "fused":
                h.hough_vote_peaks(*a, w.l_min, out["peaks"][e0:], out["n_peaks"][e0:], st)
            else:
                h.hough_vote(*a, self.count, self.mask, st)
                h.hough_peaks(ne, self.count, self.mask, w.l_min, out["peaks"][e0:], out["n_peaks"][e0:], st)
            h.hough_jets(ne, out["peaks"][e0:], out["n_peaks"][e0:], w.cone_rad, w.d0_cut_mm, w.n_displaced_min,
                         out["tracks"][e0:], out["jets"][e0:], out["n_jets"][e0:], out["flag"][e0:], st)
            if self.vertices:
                h.hough_vertices(ne, out["peaks"][e0:], out["n_peaks"][e0:], w.d0_cut_mm, w.vtx_n_min, out["vertices"][e0:],
                                 out["n_vertices"][e0:], out["vtx_flag"][e0:], None, st)

    def timed(self, steps: int, warmup: int, dist=None, after_step=None):
        """(ms total, stage ms {prep, vote, peaks, jets, vertices}, launches) for `steps` steps after `warmup` untimed ones."""
        torch = self.torch
        for _ in range(warmup):
            self.step()
            if after_step: after_step()
        torch.cuda.synchronize()
        if dist: dist.barrier()
        self.h.hough_profile(True)
        self.h.hough_profile_read()
        l0 = self.h.hough_launch_count()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record(self.stream)
        for _ in range(steps):
            self.step()
            if after_step: after_step()
        b.record(self.stream)
        torch.cuda.synchronize()
        if dist: dist.barrier()
        stage, _ = self.h.hough_profile_read()
        self.h.hough_profile(False)
        self.tile_kind = self.h.hough_last_tile_kind() if self.path == "fused" else 1
        return a.elapsed_time(b), stage, self.h.hough_launch_count() - l0

    def close(self):
        self.count = self.mask = None
        self.h.close()


def count_votes(w, batch, sub: int = 16):
    """Votes of the batch = sum of the count planes (untimed; accumulator path on `sub` events at a time)."""
    import torch
    from paper_1309_6275_b200 import binding as B
    E = batch.n_events
    sub = max(1, min(sub, E, int(8.6e9 // (4 * w.bins_per_event)) or 1))
    offs = batch.hit_offsets.astype(np.int64)
    hits = max(int(offs[min(c + sub, E)] - offs[c]) for c in range(0, E, sub))
    h = B.Hough.for_workload(w, max_events=sub, max_hits=max(1, hits))
    off, r, phi, layer = B.upload_batch(batch)
    count, mask = h.alloc_planes(sub)
    total = 0
    for e0 in range(0, E, sub):
        ne = min(sub, E - e0)
        hb, he = int(offs[e0]), int(offs[e0 + ne])
        h.hough_vote(ne, off[e0:e0 + ne + 1], he - hb, r[hb:he], phi[hb:he], layer[hb:he], count, mask)
        total += int((count[:ne].to(torch.int32) & 0xFFFF).sum(dtype=torch.int64).item())
    h.close()
    del count, mask
    torch.cuda.empty_cache()
    return float(total)


def vote_roofline(mode, votes, bins_written, ms_vote, launches, hbm_gbs, sm_max_mhz, peak_src, kernel, traffic=None,
                  tile_kind=1):
    """Roofline of the vote kernel: max of the FP32 term (I_FP32 instructions per vote on 148 x 128 lanes), the
    shared-reduction term (count + mask tiles: 2 per vote, mask tiles: 1 per vote, at 32 per clock and SM) and --
    accumulator path only -- the HBM-write term (4 B per bin).

    What `frac` is when the FP32 term binds: a MODEL-WORK fraction -- landed votes x the FP32 instructions the plain
    O-2 formulation spends per vote, over time x FP32 issue peak.  It is not the measured utilisation of the pipe: mirror
    tiles evaluate one O-2 chain for two votes and the packed fp32x2 arithmetic halves the issue count again, so the
    kernel issues fewer instructions per vote than the model charges and the fraction could exceed 1.  The measured
    pipe figure of the same kernel, where a committed ncu capture has it, is reported next to it as
    `fma_pipe_active_ncu`."""
    s = ms_vote * 1e-3
    clk = sm_max_mhz * 1e6
    fp32_peak = SM_COUNT * FP32_LANES * clk
    red_peak = SM_COUNT * SMEM_RED_PER_CLK * clk
    reds_per_vote = 1.0 if tile_kind == 2 else 2.0
    t_fp32 = votes * I_FP32[mode] / fp32_peak
    t_red = reds_per_vote * votes / red_peak
    t_hbm = 4.0 * bins_written / (hbm_gbs * 1e9)
    terms = {"fp32": t_fp32 * 1e3, "shared_reductions": t_red * 1e3, "hbm_write": t_hbm * 1e3}
    if t_hbm >= max(t_fp32, t_red):
        ach = 4.0 * bins_written / s / 1e9
        rl = {"bound": "hbm", "achieved": ach, "peak": hbm_gbs, "unit": "GB/s", "frac": ach / hbm_gbs}
    else:
        ach = votes * I_FP32[mode] / s
        rl = {"bound": "alu", "achieved": ach / 1e12, "peak": fp32_peak / 1e12, "unit": "Tinstr/s",
              "frac": ach / fp32_peak,
              "frac_kind": "model work: landed votes x I_FP32 (FP32 instructions per vote of the plain O-2 formulation) "
                           "/ (vote time x FP32 issue peak); not measured pipe utilisation, can exceed 1 on mirror / "
                           "packed tiles; evaluated (hit, row) pairs are not counted by the kernel"}
    rl.update({"traffic": traffic[0] if traffic else None, "traffic_source": traffic[1] if traffic else None,
               "fma_pipe_active_ncu": traffic[2] if traffic else None,
               "kernel": kernel, "ms_per_launch": ms_vote / max(1, launches), "launches": launches,
               "tiles": {0: None, 1: "count + mask", 2: "mask"}.get(tile_kind), "shared_reductions_per_vote": reds_per_vote,
               "i_fp32_per_vote": I_FP32[mode], "t_bound_terms_ms": terms,
               "frac_fp32_shared_hit_terms": votes * I_FP32_SHARED[mode] / s / fp32_peak,
               "peak_source": peak_src + "; FP32 peak = 148 SM x 128 lanes x sm_max clock (no FMA credit)",
               "note": "duration = CUDA events around the vote kernel alone (hough_profile, launching stream)"})
    return rl


def stencil_roofline(bins_read, ms_peaks, launches, hbm_gbs):
    ach = 2.0 * bins_read / (ms_peaks * 1e-3) / 1e9
    return {"bound": "hbm", "kernel": "peak_stencil_kernel+peak_compact_kernel", "achieved": ach, "peak": hbm_gbs,
            "unit": "GB/s", "frac": ach / hbm_gbs, "traffic": None, "ms_per_launch": ms_peaks / max(1, launches),
            "launches": launches}


def measure_config(name: str, hbm_gbs, sm_max_mhz, peak_src, steps: int = 3):
    """Short device-resident measurement of one of the other configs for the per_config block."""
    import torch
    from paper_1309_6275_b200 import workloads as W
    w = make_workload(name, None)
    batch = W.generate(w)
    mode = "3d" if w.n_d0 > 1 else "2d"
    chunk = max(1, min(w.n_events, int(34.4e9 // (4 * w.bins_per_event))))
    res = {"events": w.n_events, "hits": batch.n_hits, "grid": [w.n_d0, w.n_phi0, w.n_kappa], "l_min": w.l_min}
    votes = count_votes(w, batch)
    res["votes"] = votes
    single = w.n_events == 1
    reps = 200 if single else steps
    for path in ("fused", "planes"):
        run = DeviceRun(w, batch, chunk, path)
        ms, stage, launches = run.timed(reps, 20 if single else 2)
        n_launch = reps * run.n_chunks
        d = {"ms_per_step": ms / reps, "events_per_sec": w.n_events * reps / (ms * 1e-3),
             "stage_ms_per_step": {k: v / reps for k, v in zip(STAGES, stage)},
             "launches_per_step": launches // reps}
        if single:
            d["latency_us"] = 1e3 * ms / reps
        else:
            bins_w = 0 if path == "fused" else w.bins_per_event * w.n_events * reps
            # a committed capture of this config's fused launch (same events per launch), if there is one
            tr = traffic_from_profiles("vote_kernel<0," if mode == "2d" else "vote_kernel<1,", "_" + name.lower() + "_") \
                if path == "fused" else None
            d["roofline"] = vote_roofline(mode, votes * reps, bins_w, stage[1], n_launch, hbm_gbs, sm_max_mhz, peak_src,
                                          "vote_kernel<fused>" if path == "fused" else "vote_kernel",
                                          traffic=tr if tr and tr[0] is not None else None, tile_kind=run.tile_kind)
            if path == "planes":
                d["roofline_stencil"] = stencil_roofline(w.bins_per_event * w.n_events * reps, stage[2], n_launch, hbm_gbs)
        res[path] = d
        run.close()
        torch.cuda.empty_cache()
    return res


def p4_traffic(n_tracks: int, path: str, n_events: int):
    """The committed capture of the P4 fused launch with this many tracks per event (32 events per launch), if any."""
    if path != "fused" or n_events != 32:
        return None
    tr = traffic_from_profiles("vote_kernel<0,", f"_p4x{n_tracks}_")
    return tr if tr[0] is not None else None


def run_p4(args):
    """--workload P4: the paper's own timing benchmark (Fig. 4): time per event against tracks per
    event on the ten-layer toy detector with a 2048 x 2048 accumulator, fused path, one launch per batch."""
    import torch
    from paper_1309_6275_b200 import binding as B
    from paper_1309_6275_b200 import workloads as W
    if int(os.environ.get("WORLD_SIZE", "1")) != 1 or args.gpus != 1:
        raise SystemExit("bench.py --workload P4 is a single-GPU curve")
    torch.cuda.set_device(0)
    hbm_gbs, sm_max_mhz, peak_src = measured_peaks()
    points = [args.tracks] if args.tracks else [100, 300, 1000, 3000]
    E = args.events or 32
    curve, last = [], None
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.3)
    wall0 = time.time()
    for n in points:
        w = W.paper_timing(n, E)
        batch = W.generate(w)
        votes = count_votes(w, batch)
        d = {"tracks_per_event": n, "hits_per_event": batch.n_hits // E, "votes_per_event": votes / E}
        for path in ("fused", "planes"):
            run = DeviceRun(w, batch, E, path, vertices=False)
            ms, stage, launches = run.timed(args.steps, args.warmup)
            d[path] = {"ms_per_event": ms / args.steps / E, "events_per_sec": E * args.steps / (ms * 1e-3),
                       "stage_ms_per_event": {k: v / args.steps / E for k, v in zip(STAGES, stage)},
                       "roofline": vote_roofline("2d", votes * args.steps, 0 if path == "fused" else w.bins_per_event * E * args.steps,
                                                 stage[1], args.steps, hbm_gbs, sm_max_mhz, peak_src,
                                                 "vote_kernel<fused>" if path == "fused" else "vote_kernel",
                                                 traffic=p4_traffic(n, path, E), tile_kind=run.tile_kind)}
            if path == "fused":
                d["peaks_per_event"] = float(run.out["n_peaks"].float().mean().item())
                last = (w, batch, ms, stage, launches, votes)
            run.close()
            torch.cuda.empty_cache()
        curve.append(d)
    wall1 = time.time()
    clocks = sampler.stop(wall0, wall1)
    w, batch, ms, stage, launches, votes = last
    H = batch.n_hits
    # e2e at the last point
    h2 = B.Hough.for_workload(w, max_events=E, max_hits=H, host_chunk_events=E)
    pin = lambda a: torch.from_numpy(a).pin_memory()
    h_off, h_r, h_phi, h_layer = pin(batch.hit_offsets.view(np.int32)), pin(batch.r), pin(batch.phi), pin(batch.layer)
    h_np = torch.zeros(E, dtype=torch.int32).pin_memory(); h_nj = torch.zeros(E, dtype=torch.int32).pin_memory()
    h_fl = torch.zeros(E, dtype=torch.uint8).pin_memory()
    h_pk = torch.zeros((E, w.max_peaks, 8), dtype=torch.uint8).pin_memory()
    stream = torch.cuda.current_stream()
    call = lambda: h2.hough_trigger_host(E, h_off, H, h_r, h_phi, h_layer, w.l_min, w.cone_rad, w.d0_cut_mm,
                                         w.n_displaced_min, h_np, h_nj, h_fl, h_pk, None, None, stream)
    call(); torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(args.steps): call()
    b.record(stream); torch.cuda.synchronize()
    e2e_value = E * args.steps / (a.elapsed_time(b) * 1e-3)
    h2_launches = h2.hough_launch_count()
    h2.close()
    cpu = cpu_oracle_rate(w, batch, budget_s=10.0) if not args.no_cpu_baseline else None
    line = {"metric": "events_per_sec", "value": E * args.steps / (ms * 1e-3), "unit": "events/s", "n_gpus": 1,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "path": "fused", "events_per_gpu": E, "hits": H,
                       "grid": [w.n_d0, w.n_phi0, w.n_kappa], "l_min": w.l_min,
                       "detector": "PAPER.md:97-99: beam pipe 30 mm, 10 layers evenly spaced to 1100 mm, 0.4 mm resolution",
                       "l2": "no L2 flush needed: compute-bound, no planes in HBM on the fused path",
                       "note": "paper's Fig. 4 workload; its absolute times are in an unreadable figure (context only)"},
            "curve_time_vs_tracks": curve, "votes_per_step": votes, "clocks": clocks,
            "stage_ms_per_step": {k: v / args.steps for k, v in zip(STAGES, stage)},
            "e2e": {"value": e2e_value, "unit": "events/s", "h2d_bytes_per_step": int(H * 9 + (E + 1) * 4),
                    "d2h_bytes_per_step": int(E * 9 + E * w.max_peaks * 8), "steps": args.steps},
            "gpu_launches": int(launches), "gpu_launches_e2e": int(h2_launches),
            "roofline": curve[-1]["fused"]["roofline"]}
    if cpu:
        line["cpu_baseline"] = cpu
    print(json.dumps(line))


def match_vertices(found_r, found_phi, true_r, true_phi, tol_mm: float):
    """Truth matching of the efficiency studies: a simulated jet counts as identified if a found vertex lies within
    tol_mm of its vertex in the transverse plane (PAPER.md:137 'fraction of simulated jets successfully identified').
    Returns (true vertices matched, found vertices that match no true vertex)."""
    fx, fy = found_r * np.cos(found_phi), found_r * np.sin(found_phi)
    tx, ty = true_r * np.cos(true_phi), true_r * np.sin(true_phi)
    if tx.size == 0 or fx.size == 0:
        return 0, int(fx.size)
    d = np.hypot(fx[:, None] - tx[None, :], fy[:, None] - ty[None, :])
    return int((d.min(axis=0) <= tol_mm).sum()), int((d.min(axis=1) > tol_mm).sum())


def efficiency_point(w, batch, flags: int, steps: int, warmup: int, tol_mm: float):
    """One point of an efficiency study: the whole chain on the GPU for the batch, then truth matching on the host."""
    import torch
    from paper_1309_6275_b200 import binding as B
    E = batch.n_events
    stream = torch.cuda.current_stream()
    chunk = max(1, min(E, int(4e9 // (4 * w.bins_per_event))))
    off, r, phi, layer = B.upload_batch(batch)
    offs = batch.hit_offsets.astype(np.int64)
    hits_per_chunk = max(int(offs[min(c + chunk, E)] - offs[c]) for c in range(0, E, chunk))
    h = B.Hough.for_workload(w, max_events=chunk, max_hits=hits_per_chunk, vgrid=w.vgrid, max_vertices=w.max_vertices,
                             vote_flags=flags)
    count, mask = h.alloc_planes(chunk)
    out = h.alloc_outputs(E)

    def step():
        for e0 in range(0, E, chunk):
            ne = min(chunk, E - e0)
            hb, he = int(offs[e0]), int(offs[e0 + ne])
            h.hough_vote(ne, off[e0:e0 + ne + 1], he - hb, r[hb:he], phi[hb:he], layer[hb:he], count, mask, stream)
            h.hough_peaks(ne, count, mask, w.l_min, out["peaks"][e0:], out["n_peaks"][e0:], stream)
            h.hough_jets(ne, out["peaks"][e0:], out["n_peaks"][e0:], w.cone_rad, w.d0_cut_mm, w.n_displaced_min,
                         out["tracks"][e0:], out["jets"][e0:], out["n_jets"][e0:], out["flag"][e0:], stream)
            h.hough_vertices(ne, out["peaks"][e0:], out["n_peaks"][e0:], w.d0_cut_mm, w.vtx_n_min, out["vertices"][e0:],
                             out["n_vertices"][e0:], out["vtx_flag"][e0:], None, stream)
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    l0 = h.hough_launch_count()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(steps):
        step()
    b.record(stream)
    torch.cuda.synchronize()
    ms = a.elapsed_time(b) / steps
    nv = out["n_vertices"].cpu().numpy()
    vt = B.records(out["vertices"], B.VERTEX_DTYPE)
    npk = out["n_peaks"].cpu().numpy().astype(np.int64)
    found = fake = n_true = 0
    for e in range(E):
        k = min(int(nv[e]), w.max_vertices)
        t = batch.truth[e]
        tr = t.get("vertex_r", np.zeros(0)); tp = t.get("vertex_phi", np.zeros(0))
        m, f = match_vertices(vt[e, :k]["r"].astype(np.float64), vt[e, :k]["phi"].astype(np.float64), tr, tp, tol_mm)
        found += m; fake += f; n_true += int(tr.size)
    res = {"efficiency": found / max(1, n_true), "jets_found": found, "unmatched_vertices_per_event": fake / E,
           "peaks_per_event": float(npk.mean()), "peak_list_overflows": int((npk > w.max_peaks).sum()),
           "ms_per_event": ms / E, "status_bits": int(h.hough_status()), "launches": int(h.hough_launch_count() - l0)}
    h.close()
    del count, mask, out
    torch.cuda.empty_cache()
    return res


def run_efficiency(args):
    """--workload F8 | F9 | F10: the SHAPE of the paper's efficiency studies (Figs 8-10) on synthetic
    events of its toy detector: efficiency of displaced-jet detection against tracks per jet (F8), jets per event (F9),
    and jets per event among 3,000 tracks (F10).  Whole chain on the GPU through the C-ABI: hough_vote with the
    physics-quality voting variants (forward-hemisphere cut + kappa-range filling) -> hough_peaks ->
    hough_jets -> hough_vertices (second Hough transform, vertices inside the beam pipe dropped); the plain one-vote-per-
    column-centre vote is run next to it.  Only the truth matching happens on the host."""
    import torch
    from paper_1309_6275_b200 import binding as B
    from paper_1309_6275_b200 import workloads as W
    if int(os.environ.get("WORLD_SIZE", "1")) != 1 or args.gpus != 1:
        raise SystemExit("bench.py --workload F8/F9/F10 is a single-GPU study")
    torch.cuda.set_device(0)
    kind = args.workload
    xs = {"F8": [2, 4, 6, 8, 10, 12, 15, 20], "F9": [1, 2, 3, 4, 6, 8, 10], "F10": [1, 2, 4, 6, 8, 10]}[kind]
    if args.tracks:
        xs = [args.tracks]
    E = args.events or (32 if kind == "F10" else 64)
    tol_mm = 10.0
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.3)
    wall0 = time.time()
    curve, last_ms, launches = [], None, 0
    for x in xs:
        w = W.paper_efficiency(kind, x, E)
        batch = W.generate(w, keep_truth=True)
        d = {"x": x, "hits_per_event": batch.n_hits // E, "jets_simulated": int(sum(t["n_vertices"] for t in batch.truth))}
        for label, flags in (("variants", w.vote_flags), ("plain", 0)):
            d[label] = efficiency_point(w, batch, flags, args.steps, max(1, args.warmup), tol_mm)
            if label == "variants":
                last_ms, launches, last = d[label]["ms_per_event"] * E, d[label].pop("launches"), (w, batch)
            else:
                d[label].pop("launches")
        curve.append(d)
    clocks = sampler.stop(wall0, time.time())
    w, batch = last
    line = {"metric": "events_per_sec", "value": E / (last_ms * 1e-3), "unit": "events/s", "n_gpus": 1, "steps": args.steps,
            "warmup": max(1, args.warmup), "ms_per_step": last_ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "path": "planes (hough_vote with vote_flags %d)" % w.vote_flags,
                       "events_per_gpu": E, "hits": batch.n_hits, "grid": [w.n_d0, w.n_phi0, w.n_kappa], "l_min": w.l_min,
                       "vertex_grid": list(w.vgrid), "vtx_n_min": w.vtx_n_min, "d0_cut_mm": w.d0_cut_mm, "match_tol_mm": tol_mm,
                       "detector": "PAPER.md:97-99: beam pipe 30 mm, 10 layers evenly spaced to 1100 mm, 0.4 mm resolution",
                       "l2": "planes (67 MB per event, rewritten every launch) are larger than L2",
                       "note": "shape of the paper's efficiency studies (PAPER.md:137-151); its figures are not readable, "
                               "so there is no number to compare with"},
            "study": {"F8": "efficiency vs tracks per displaced jet (PAPER.md:137, Fig. 8)",
                      "F9": "efficiency vs displaced jets per event, 10 tracks each (PAPER.md:145, Fig. 9)",
                      "F10": "efficiency vs displaced jets per event among 3000 tracks (PAPER.md:147, Fig. 10)"}[kind],
            "curve_efficiency": curve, "clocks": clocks, "gpu_launches": int(launches)}
    print(json.dumps(line))


def run_ours(args):
    import torch
    from paper_1309_6275_b200 import binding as B
    from paper_1309_6275_b200 import workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; launch one rank per GPU "
                         f"(python bench.py --gpus N starts them itself)")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", rank=rank, world_size=world)

    w = make_workload(args.workload, args.events)
    E = w.n_events
    # events per launch: --chunk, else as many as would fit in about 34 GB of planes (C5: 128 events)
    chunk = args.chunk if args.chunk > 0 else max(1, int(34.4e9 // (4 * w.bins_per_event)))
    chunk = min(chunk, E)
    mode = "3d" if w.n_d0 > 1 else "2d"
    batch = W.generate(w, E, first_event=first_event_of_rank(E, rank))      # weak scaling: every rank its own events
    H = batch.n_hits
    bins = w.bins_per_event
    hbm_gbs, sm_max_mhz, peak_src = measured_peaks()

    votes_per_step = count_votes(w, batch)

    run = DeviceRun(w, batch, chunk, args.path, vertices=not args.no_vertices)
    gathered = {}

    def exchange():
        if dist is not None:
            gathered["v"] = gather_event_results(run.out["flag"], run.out["n_peaks"], run.out["n_jets"], dist)

    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    wall0 = time.time()
    ms_total, stage, launches = run.timed(args.steps, args.warmup, dist, exchange if dist else None)
    wall1 = time.time()
    clocks = sampler.stop(wall0 + 0.0, wall1)
    status = run.h.hough_status()
    n_flag = int(run.out["flag"].sum().item())
    n_vflag = int(run.out["vtx_flag"].sum().item()) if run.vertices else None
    n_vtx_total = int(run.out["n_vertices"].to(torch.int64).sum().item()) if run.vertices else None
    n_both = int((run.out["flag"].bool() & run.out["vtx_flag"].bool()).sum().item()) if run.vertices else None
    vflags_dev = run.out["vtx_flag"].cpu().numpy().copy()
    with_vtx = run.vertices
    n_peaks_total = int(run.out["n_peaks"].to(torch.int64).sum().item())
    flags_dev = run.out["flag"].cpu().numpy().copy()
    npk_dev = run.out["n_peaks"].cpu().numpy().copy()
    job_flags = None
    if dist is not None:
        gf = gathered["v"][0]
        assert gf.shape == (world, E) and bool((gf[rank] == run.out["flag"]).all())
        job_flags = int(gf.sum().item())

    ms_max = max_over_ranks(ms_total, dist)
    total_events = sum_over_ranks(float(E * args.steps), dist)
    value = total_events / (ms_max * 1e-3)
    n_launch = args.steps * run.n_chunks
    main_tile_kind = run.tile_kind
    run.close()
    torch.cuda.empty_cache()

    # ---- the accumulator path on a short leg (stencil roofline; vote kernel with the plane flush) ----
    planes = None
    if rank == 0 and args.path == "fused" and not args.no_planes_leg:
        n_ev = min(E, 2 * chunk)
        sub = batch.slice(0, n_ev)
        votes_sub = votes_per_step * (sub.n_hits / max(1, H))             # (estimate only used if it binds: it does not at C5/C3)
        prun = DeviceRun(w, sub, chunk, "planes")
        p_steps = 3
        p_ms, p_stage, p_launches = prun.timed(p_steps, 1)
        pl = p_steps * prun.n_chunks
        planes = {"events": n_ev, "ms_per_step": p_ms / p_steps, "events_per_sec": n_ev * p_steps / (p_ms * 1e-3),
                  "stage_ms_per_step": {k: v / p_steps for k, v in zip(STAGES, p_stage)},
                  "roofline_vote": vote_roofline(mode, votes_sub * p_steps, bins * n_ev * p_steps, p_stage[1], pl, hbm_gbs,
                                                 sm_max_mhz, peak_src, "vote_kernel"),
                  "roofline_stencil": stencil_roofline(bins * n_ev * p_steps, p_stage[2], pl, hbm_gbs)}
        same = bool(np.array_equal(prun.out["flag"].cpu().numpy(), flags_dev[:n_ev]) and
                    np.array_equal(prun.out["n_peaks"].cpu().numpy(), npk_dev[:n_ev]))
        planes["matches_fused_path"] = same
        prun.close()
        torch.cuda.empty_cache()

    # ---- e2e: the same batch through hough_trigger_host with pinned host buffers ----
    # max_plane_events = 1: this context never runs hough_peaks on a batch (only the one-event overflow fallback), so
    # it need not hold the peak finder's bitmap for max_events events (C5: 34 GB)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    h2 = B.Hough.for_workload(w, max_events=E, max_hits=H, host_chunk_events=chunk,
                              vgrid=w.vgrid if with_vtx else None, max_vertices=w.max_vertices, max_plane_events=1)
    e2e_ctx_bytes = int(free0 - torch.cuda.mem_get_info()[0])
    pin = lambda a: torch.from_numpy(a).pin_memory()
    h_off, h_r, h_phi, h_layer = pin(batch.hit_offsets.view(np.int32)), pin(batch.r), pin(batch.phi), pin(batch.layer)
    h_np = torch.zeros(E, dtype=torch.int32).pin_memory(); h_nj = torch.zeros(E, dtype=torch.int32).pin_memory()
    h_fl = torch.zeros(E, dtype=torch.uint8).pin_memory()
    h_jets = torch.zeros((E, w.max_jets, 20), dtype=torch.uint8).pin_memory()
    stream = torch.cuda.current_stream()
    e2e_steps = max(1, min(args.steps, 3))
    h_nv = torch.zeros(E, dtype=torch.int32).pin_memory(); h_vf = torch.zeros(E, dtype=torch.uint8).pin_memory()
    h_vtx = torch.zeros((E, w.max_vertices, 16), dtype=torch.uint8).pin_memory()
    if with_vtx:
        call = lambda: h2.hough_trigger_host_vtx(E, h_off, H, h_r, h_phi, h_layer, w.l_min, w.cone_rad, w.d0_cut_mm,
                                                 w.n_displaced_min, w.vtx_n_min, h_np, h_nj, h_fl, None, h_jets, h_nv,
                                                 h_vf, h_vtx, None, stream)
    else:
        call = lambda: h2.hough_trigger_host(E, h_off, H, h_r, h_phi, h_layer, w.l_min, w.cone_rad, w.d0_cut_mm,
                                             w.n_displaced_min, h_np, h_nj, h_fl, None, h_jets, None, stream)
    call()
    torch.cuda.synchronize()
    if dist: dist.barrier()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(e2e_steps):
        call()
    b.record(stream)
    torch.cuda.synchronize()
    ms_e2e = max_over_ranks(a.elapsed_time(b), dist)
    e2e_value = sum_over_ranks(float(E * e2e_steps), dist) / (ms_e2e * 1e-3)
    e2e_ok = bool(np.array_equal(h_fl.numpy(), flags_dev) and np.array_equal(h_np.numpy(), npk_dev) and
                  (not with_vtx or np.array_equal(h_vf.numpy(), vflags_dev)))
    h2_launches = h2.hough_launch_count()
    h2.close()
    torch.cuda.empty_cache()

    if rank != 0:
        if dist: dist.destroy_process_group()
        return

    votes_timed = votes_per_step * args.steps
    fused = args.path == "fused"
    kern = "vote_kernel<fused>" if fused else "vote_kernel"
    traffic = traffic_from_profiles("vote_kernel<1,") if (w.name == "C5" and chunk == 128) else None
    roofline = vote_roofline(mode, votes_timed, 0 if fused else bins * E * args.steps, stage[1], n_launch, hbm_gbs,
                             sm_max_mhz, peak_src, kern, traffic, tile_kind=main_tile_kind)

    per_config = None
    if not args.no_per_config and world == 1 and w.name == "C5" and not args.events:
        per_config = {}
        for name in ("C1", "C2", "C3", "C4"):
            per_config[name] = measure_config(name, hbm_gbs, sm_max_mhz, peak_src)

    cpu = cpu_oracle_rate(w, batch) if not args.no_cpu_baseline else None

    if fused:
        l2_note = (f"no L2 flush needed: the fused path streams nothing but the hits ({H * 25 / 1e6:.0f} MB of raw + "
                   f"prepared records per step, larger than the 126 MB L2 for C5) and is compute-bound")
    else:
        l2_note = f"working set >> L2: {4 * bins * chunk / 1e9:.1f} GB of planes rewritten and re-read every launch"
    line = {
        "metric": "events_per_sec", "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "path": args.path, "events_per_gpu": E, "chunk_events": chunk, "hits": H,
                   "grid": [w.n_d0, w.n_phi0, w.n_kappa], "l_min": w.l_min, "cone_rad": w.cone_rad, "l2": l2_note},
        "votes_per_sec": votes_timed * world / (ms_max * 1e-3) if world == 1 else None,
        "votes_per_step": votes_per_step,
        "stage_ms_per_step": {k: v / args.steps for k, v in zip(STAGES, stage)},
        "events_flagged": n_flag, "events_flagged_all_ranks": job_flags, "peaks_total": n_peaks_total,
        "second_transform": ({"vertex_grid": list(w.vgrid), "n_min": w.vtx_n_min, "d0_cut_mm": w.d0_cut_mm,
                              "events_flagged_vertex": n_vflag, "vertices_total": n_vtx_total,
                              "events_flagged_by_both": n_both} if with_vtx else None),
        "status_bits": status, "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "events/s", "h2d_bytes_per_step": int(H * 9 + (E + 1) * 4),
                "d2h_bytes_per_step": int(E * 9 + E * w.max_jets * 20 + (E * 5 + E * w.max_vertices * 16 if with_vtx else 0)),
                "steps": e2e_steps,
                "matches_device_path": e2e_ok},
        "e2e_context_device_bytes": e2e_ctx_bytes,
        "gpu_launches": int(launches), "gpu_launches_e2e": int(h2_launches),
        "roofline": roofline,
    }
    if planes:
        line["accumulator_path"] = planes
        line["roofline_stencil"] = planes["roofline_stencil"]
    if per_config:
        line["per_config"] = per_config
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
    ap.add_argument("--workload", default="C5", choices=["C1", "C2", "C3", "C4", "C5", "P4", "F8", "F9", "F10"])
    ap.add_argument("--tracks", type=int, default=0, help="P4 / F8 / F9 / F10: one point of the curve (0 = all of them)")
    ap.add_argument("--path", default="fused", choices=["fused", "planes"])
    ap.add_argument("--events", type=int, default=0, help="override the number of events per GPU (0 = the config's)")
    ap.add_argument("--chunk", type=int, default=0, help="events per launch (0: what would fit in 34 GB of planes)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true")
    ap.add_argument("--no-planes-leg", action="store_true")
    ap.add_argument("--no-vertices", action="store_true", help="leave the second Hough transform out of the step")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        reexec_under_torchrun(args, sys.argv[1:])
    if args.workload == "P4":
        run_p4(args)
    elif args.workload in ("F8", "F9", "F10"):
        run_efficiency(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
