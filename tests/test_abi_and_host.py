"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol include/hough.h
declares, the ctypes struct matches the header layout, the generators are deterministic, and the event-sharding
logic used for N > 1 GPUs is exercised with a world_size-2 gloo group (no compute calls without a GPU)."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "hough.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hough_[a-z_]+)\s*\(", text)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1309_6275_b200 import build, binding
    build.build()
    lib = C.CDLL(binding.LIB_PATH)
    declared = _declared_symbols()
    assert set(declared) == set(binding.EXPORTS), (declared, binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    # only sm_100a code is embedded
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out and not re.search(r"sm_(?!100a)\d+", out), out


def test_strerror_and_argument_validation_without_gpu():
    from paper_1309_6275_b200 import binding as B
    lib = B.load_library()
    assert B.strerror(0) == "ok" and "invalid" in B.strerror(-1)
    # a bad config is rejected before any CUDA call; null pointers likewise
    ctx = C.c_void_p()
    bad = B.HoughConfig(512, 250, 1, 1.14e-3, 0, 0, 3.8, 8, 1, 100, 16, 16, 0, 0, 0, 0, 0, 0, 0, 0)       # n_kappa % 8 != 0
    assert lib.hough_create(C.byref(bad), C.byref(ctx)) == -1
    bad2 = B.HoughConfig(512, 256, 1, 1.14e-3, 0, 0, 3.8, 17, 1, 100, 16, 16, 0, 0, 0, 0, 0, 0, 0, 0)     # n_layers > 16
    assert lib.hough_create(C.byref(bad2), C.byref(ctx)) == -1
    # a vertex grid counts tracks in 16 bits: a peak list that could overflow a bin is refused (hough.h)
    bad3 = B.HoughConfig(512, 256, 8, 1.14e-3, -10.0, 10.0, 3.8, 8, 1, 100, 65536, 16, 0, 0, 64, 32, 30.0, 430.0, 16, 0)
    assert lib.hough_create(C.byref(bad3), C.byref(ctx)) == -1
    assert lib.hough_create(None, C.byref(ctx)) == -1
    assert lib.hough_destroy(None) == -1
    assert lib.hough_plane_bytes(None, 3) == 0


def test_config_struct_layout_matches_header():
    from paper_1309_6275_b200 import binding as B
    # compile a 3-line C program against the real header and compare sizeof / offsets
    src = r'''
    #include <stdio.h>
    #include <stddef.h>
    #include "hough.h"
    int main(void){ printf("%zu %zu %zu %zu %zu %zu %zu %zu\n", sizeof(hough_config), offsetof(hough_config, max_hits),
        offsetof(hough_config, host_chunk_events), sizeof(hough_peak), sizeof(hough_track), sizeof(hough_jet),
        offsetof(hough_config, max_events), offsetof(hough_config, max_candidates_per_event));
        printf("%zu %zu %zu %zu %zu\n", offsetof(hough_config, vtx_r_min), offsetof(hough_config, max_vertices_per_event), sizeof(hough_vertex),
               offsetof(hough_config, vote_flags), offsetof(hough_config, debug_flags));
        printf("%zu\n", offsetof(hough_config, max_plane_events));
        return 0; }'''
    exe = "/tmp/hough_layout_probe"
    subprocess.run(["gcc", "-x", "c", "-", "-I", os.path.join(ROOT, "include"), "-o", exe], input=src, text=True, check=True)
    vals = list(map(int, subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()))
    assert vals[0] == C.sizeof(B.HoughConfig)
    assert vals[1] == B.HoughConfig.max_hits.offset and vals[2] == B.HoughConfig.host_chunk_events.offset
    assert vals[6] == B.HoughConfig.max_events.offset and vals[7] == B.HoughConfig.max_candidates_per_event.offset
    assert vals[8] == B.HoughConfig.vtx_r_min.offset and vals[9] == B.HoughConfig.max_vertices_per_event.offset
    assert vals[10] == B.VERTEX_DTYPE.itemsize == 16 and vals[11] == B.HoughConfig.vote_flags.offset
    assert vals[12] == B.HoughConfig.debug_flags.offset and vals[13] == B.HoughConfig.max_plane_events.offset
    assert vals[3] == B.PEAK_DTYPE.itemsize == 8 and vals[4] == B.TRACK_DTYPE.itemsize == 20
    assert vals[5] == B.JET_DTYPE.itemsize == 20


def test_packed_sweep_keeps_every_rounding_of_o2():
    """ptxas contracts mul.rn.f32x2 feeding add.rn.f32x2 into one FFMA2 (one rounding instead of the two O-2 asks
    for).  The 3D sweep therefore forms a = two_d0 * rs with scalar FMULs; what must survive in the SASS of every
    3D vote kernel is, per candidate pair, the three packed sums t, b, den (FADD2) next to the one round-down add
    of the bin floor (FADD2.RM), and no packed multiply may have been fused away: NQ0 and u stay FMUL2."""
    from paper_1309_6275_b200 import build
    lib = build.build()
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    # vote_kernel<MODE3D, KL, FUSED, MIRROR, VARIANT, MO>: the packed 3D kernels (the scalar voting-variant kernels are left out)
    kernels = []
    for body in sass.split("Function : ")[1:]:
        m = re.search(r"vote_kernelILb(\d)ELi(\d)ELb(\d)ELb(\d)ELb(\d)ELb(\d)EEEv", body.split("\n")[0])
        if m and m.group(1) == "1" and m.group(5) == "0":
            kernels.append((m.group(4) == "1", body))
    assert len(kernels) == 9                     # KL = 1, 2, 4 x {planes, fused} + the mirror kernels (planes, fused, fused mask tiles)
    n_mirror = 0
    for mirror, body in kernels:
        n_rm = len(re.findall(r"\bFADD2\.RM\b", body))
        n_add = len(re.findall(r"\bFADD2 ", body))
        n_mul = len(re.findall(r"\bFMUL2 ", body))
        n_fma = len(re.findall(r"\bFFMA2 ", body))
        assert n_rm > 0
        if mirror:                                               # per hit pair: 2 floors (row + mirror row), t, b, den,
            n_mirror += 1                                        # NQ0 + two u, the division's 4 FFMA2 + two v
            assert 2 * n_add == 3 * n_rm and 2 * n_mul == 3 * n_rm and n_fma == 3 * n_rm, (n_add, n_mul, n_fma, n_rm)
        else:
            assert n_add == 3 * n_rm, (n_add, n_rm)
            assert n_mul == 2 * n_rm, (n_mul, n_rm)
            assert n_fma == 5 * n_rm, (n_fma, n_rm)
    assert n_mirror == 3


def test_library_reads_no_environment_variable_and_rejects_unknown_debug_flags():
    """no environment variables, no global state.  Kernel variants are chosen through
    hough_config.debug_flags; nothing under csrc/ calls getenv."""
    from paper_1309_6275_b200 import binding as B
    csrc = os.path.join(ROOT, "paper_1309_6275_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f
    lib = B.load_library()
    ctx = C.c_void_p()
    for flags in (8, B.DEBUG_TILES_COUNT | B.DEBUG_TILES_MASK):
        bad = B.HoughConfig(512, 256, 1, 1.14e-3, 0, 0, 3.8, 8, 1, 100, 16, 16, 0, 0, 0, 0, 0, 0, 0, 0, 0, flags)
        assert lib.hough_create(C.byref(bad), C.byref(ctx)) == -1
    bad = B.HoughConfig(512, 256, 1, 1.14e-3, 0, 0, 3.8, 8, 4, 100, 16, 16, 0, 0, 0, 0, 0, 0, 0, 0, 5, 0)   # max_plane_events > max_events
    assert lib.hough_create(C.byref(bad), C.byref(ctx)) == -1


def test_product_path_never_touches_the_oracle():
    """No file of the package (or bench's product arm) imports oracle/; the oracle never imports the package."""
    pkg = os.path.join(ROOT, "paper_1309_6275_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "hough_oracle" not in text and "from oracle" not in text and "import oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1309_6275_b200 import" not in text and "import paper_1309_6275_b200" not in text
            assert "hough.h" not in text


def test_generators_are_deterministic_and_shaped_like_the_configs():
    from paper_1309_6275_b200 import workloads as W
    a = W.generate(W.config(1)); b = W.generate(W.config(1))
    assert a.n_hits == 180 and np.array_equal(a.phi, b.phi) and np.array_equal(a.layer, b.layer)
    assert a.r.dtype == np.float32 and a.layer.dtype == np.uint8 and a.hit_offsets.dtype == np.uint32
    assert set(np.unique(a.r).tolist()) <= set(np.float32(W.TRACKER_A).tolist())
    assert np.all((a.phi >= 0) & (a.phi <= np.float32(2 * np.pi)))
    c3 = W.generate(W.config(3), 3)
    assert c3.n_events == 3 and np.all(np.diff(c3.hit_offsets.astype(np.int64)) == 2600)
    c4 = W.generate(W.config(4), 2, keep_truth=True)
    assert 9000 < c4.n_hits / 2 < 9500 and c4.layer.max() == 11
    for t in c4.truth:
        assert t["n_vertices"] == 3 and 18 <= t["disp_kappa"].size <= 36
    c5 = W.generate(W.config(5), 40, keep_truth=True)
    n = np.diff(c5.hit_offsets.astype(np.int64))
    assert n.min() >= 500 + 50 * 8 and n.max() <= 2000 + 400 * 12 + 4 * 12 * 12
    assert 0 < sum(t["n_vertices"] > 0 for t in c5.truth) < 20
    # slicing keeps CSR consistent; events are independent of how many are generated
    s = c5.slice(3, 7)
    assert s.n_events == 4 and s.hit_offsets[0] == 0 and np.array_equal(s.event(1)[1], c5.event(4)[1])
    one = W.generate(W.config(5), 1, first_event=4)
    assert np.array_equal(one.phi, c5.event(4)[1])


def test_displaced_truth_geometry_is_self_consistent():
    """The generator's displaced tracks really pass through their vertex: closest-approach parameters (d0, phi0)
    reproduce the vertex position on the circle (pure geometry of the forward model, no voting arithmetic)."""
    from paper_1309_6275_b200 import workloads as W
    b = W.generate(W.config(2), keep_truth=True)
    t = b.truth[0]
    d0, phi0, kap = t["disp_d0"], t["disp_phi0"], t["disp_kappa"]
    v = t["disp_vertex"]
    vx = t["vertex_r"][v] * np.cos(t["vertex_phi"][v]); vy = t["vertex_r"][v] * np.sin(t["vertex_phi"][v])
    cx = (1 / kap - d0) * -np.sin(phi0); cy = (1 / kap - d0) * np.cos(phi0)
    assert np.allclose(np.hypot(vx - cx, vy - cy), 1 / np.abs(kap), rtol=1e-9)
    assert np.all(np.abs(d0) <= t["vertex_r"][v] + 1e-9)


_SHARD_SCRIPT = r'''
import os, sys
import numpy as np
import torch
import torch.distributed as dist
sys.path.insert(0, sys.argv[1])
import bench
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
# strong-scaling helper: every event owned by exactly one rank
lo, hi = bench.shard_range(37, rank, world)
mine = np.zeros(37, np.int64); mine[lo:hi] = 1
t = torch.from_numpy(mine); dist.all_reduce(t)
assert t.tolist() == [1] * 37, t.tolist()
# the path run_ours takes (weak scaling): rank r owns events [r*E, (r+1)*E) of the stream, generates exactly those,
# and the one exchange of the job gathers flag / n_peaks / n_jets of every rank.  The device calls are stubbed by
# tensors whose values are a known function of the global event index.
from paper_1309_6275_b200 import workloads as W
E = 5
w = W.scaled(W.config(5), n_events=E)
first = bench.first_event_of_rank(E, rank)
assert first == rank * E
batch = W.generate(w, E, first_event=first)
whole = W.generate(w, E * world)                                  # the stream every rank's slice comes from
assert np.array_equal(batch.phi, whole.slice(first, first + E).phi)
gidx = torch.arange(first, first + E)
flag = (gidx % 3 == 0).to(torch.uint8); n_peaks = (gidx * 7 + 1).to(torch.int32); n_jets = (gidx + 2).to(torch.int32)
gf, gp, gj = bench.gather_event_results(flag, n_peaks, n_jets, dist)
allidx = torch.arange(E * world).reshape(world, E)
assert gf.shape == (world, E) and torch.equal(gf, (allidx % 3 == 0).to(torch.uint8))
assert torch.equal(gp, (allidx * 7 + 1).to(torch.int32)) and torch.equal(gj, (allidx + 2).to(torch.int32))
ms = bench.max_over_ranks(10.0 + rank, dist)
assert ms == 10.0 + world - 1
tot = bench.sum_over_ranks(float(E), dist)
assert tot == float(E * world)
dist.destroy_process_group()
print("shard ok", rank, lo, hi)
'''


def test_event_sharding_and_flag_gather_world_size_2_gloo(tmp_path):
    script = tmp_path / "shard.py"
    script.write_text(_SHARD_SCRIPT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29611")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", "29611", str(script), ROOT],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.count("shard ok") == 2


def test_bench_gpus_flag_is_checked_against_the_launch():
    """--gpus N must match the number of ranks actually launched (round 1 silently ran one rank)."""
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "4", "--steps", "1", "--warmup", "1"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode != 0 and "WORLD_SIZE=1" in (r.stdout + r.stderr)
    import bench
    assert bench.gather_event_results.__doc__ and bench.reexec_under_torchrun.__doc__


def test_efficiency_workloads_and_truth_matching():
    """paper_efficiency: ten hits per track on the ten-layer toy detector, x tracks per jet / x jets /
    3000 tracks in total; bench.match_vertices counts a simulated jet as found iff a vertex lies within the tolerance."""
    import bench
    from paper_1309_6275_b200 import workloads as W
    w = W.paper_efficiency("F8", 6, 4)
    b = W.generate(w, keep_truth=True)
    assert b.n_hits == 4 * 6 * 10 and all(t["n_vertices"] == 1 for t in b.truth)
    assert all(40.0 <= t["vertex_r"][0] <= 130.0 for t in b.truth) and w.n_layers == 10 and w.vote_flags == 3
    w = W.paper_efficiency("F9", 5, 2)
    assert W.generate(w).n_hits == 2 * 5 * 10 * 10
    w = W.paper_efficiency("F10", 7, 1)
    b = W.generate(w, keep_truth=True)
    assert abs(b.n_hits - 30000) <= 300 and b.truth[0]["prompt_pt"].size == 3000 - 70     # a few 1 GeV loopers miss a layer
    # matching: vertices at (100 mm, 0) and (50 mm, pi/2); found ones 3 mm, 30 mm and far away
    tr, tp = np.array([100.0, 50.0]), np.array([0.0, np.pi / 2])
    fr, fp = np.array([103.0, 80.0, 200.0]), np.array([0.0, np.pi / 2, 3.0])
    assert bench.match_vertices(fr, fp, tr, tp, 10.0) == (1, 2)
    assert bench.match_vertices(fr, fp, tr, tp, 31.0) == (2, 1)
    assert bench.match_vertices(np.zeros(0), np.zeros(0), tr, tp, 10.0) == (0, 0)
    assert bench.match_vertices(fr, fp, np.zeros(0), np.zeros(0), 10.0) == (0, 3)


def test_o2_instruction_count():
    """bench.py's FP32 roofline term uses I_FP32 = FMA-pipe instructions (FADD / FMUL / FFMA) of the plain O-2 function
    compiled for sm_100a.  Recount them from the SASS of csrc/o2_count.cu: fast path only (up to the
    first EXIT; the slow path of the IEEE division sits behind it)."""
    import bench
    src = os.path.join(ROOT, "paper_1309_6275_b200", "csrc", "o2_count.cu")
    cubin = str(os.path.join("/tmp", "hough_o2_count.cubin"))
    subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "--fmad=false", "-prec-div=true",
                    "-ftz=false", "-cubin", src, "-o", cubin], check=True)
    sass = subprocess.run(["cuobjdump", "-sass", cubin], capture_output=True, text=True, check=True).stdout
    counts = {}
    for body in sass.split("Function : ")[1:]:
        name = body.split("\n")[0].strip()
        fast = body.split("EXIT")[0]
        ops = re.findall(r"^\s+/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d\s+)?([A-Z0-9_.]+)", fast, flags=re.M)
        fma_pipe = [o for o in ops if o.split(".")[0] in ("FADD", "FMUL", "FFMA")]
        other_fp = [o for o in ops if o.split(".")[0] in ("MUFU", "FCHK", "F2I", "FSETP")]
        counts[name] = (len(fma_pipe), len(other_fp))
    assert counts["o2_vote_3d"][0] == bench.I_FP32["3d"] == 17, counts
    assert counts["o2_vote_2d"][0] == bench.I_FP32["2d"] == 11, counts
    assert counts["o2_vote_3d"][1] == counts["o2_vote_2d"][1] == 5, counts        # MUFU.RCP, FCHK, F2I, 2 x FSETP
