"""ctypes wrapper around oracle/hough_oracle.c -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  It never imports the CUDA package and shares nothing with it.  All arithmetic lives in the C file
(each function there cites the passage it follows); this wrapper only marshals numpy arrays and, for
batches, runs the unchanged single-threaded per-event code on several events at once (one event per
worker thread; ctypes releases the GIL).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hough_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_hough.so")
CFLAGS = ["-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]

PEAK_DTYPE = np.dtype([("lin", "<u4"), ("count", "<u2"), ("mask", "<u2")])
TRACK_DTYPE = np.dtype([("pt", "<f4"), ("phi0", "<f4"), ("d0", "<f4"), ("q", "<i4"), ("jet", "<i4")])
JET_DTYPE = np.dtype([("seed_track", "<u4"), ("n_tracks", "<u4"), ("n_displaced", "<u4"),
                      ("phi", "<f4"), ("sum_pt", "<f4")])


VERTEX_DTYPE = np.dtype([("r", "<f4"), ("phi", "<f4"), ("n_tracks", "<u4"), ("lin", "<u4")])


class _VGrid(C.Structure):
    _fields_ = [("n_phi", C.c_uint32), ("n_r", C.c_uint32), ("r_min", C.c_float), ("r_max", C.c_float)]


class _Grid(C.Structure):
    _fields_ = [("n_phi0", C.c_uint32), ("n_kappa", C.c_uint32), ("n_d0", C.c_uint32),
                ("kappa_max", C.c_float), ("d0_min", C.c_float), ("d0_max", C.c_float),
                ("b_tesla", C.c_float), ("n_layers", C.c_uint32)]


def build(force: bool = False) -> str:
    """Compile the oracle shared object (gcc) if missing or older than its source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", *CFLAGS, _SRC, "-o", _LIB, "-lm"])
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        p = C.c_void_p
        lib.oracle_tables.argtypes = [C.POINTER(_Grid), p, p, p, p]
        lib.oracle_tables.restype = None
        lib.oracle_hit_prep.argtypes = [C.c_uint64, p, p, p]
        lib.oracle_hit_prep.restype = None
        lib.oracle_vote.argtypes = [C.POINTER(_Grid), C.c_uint64, p, p, p, C.c_uint32, C.c_uint32,
                                    C.c_uint32, C.c_uint32, p, p]
        lib.oracle_vote.restype = C.c_int64
        lib.oracle_vote_columns.argtypes = [C.POINTER(_Grid), C.c_uint64, p, p, p, C.c_uint32, p, p, p, p]
        lib.oracle_vote_columns.restype = C.c_int64
        lib.oracle_peaks.argtypes = [C.POINTER(_Grid), p, p, C.c_uint32, C.c_uint32, p]
        lib.oracle_peaks.restype = C.c_uint64
        lib.oracle_tracks.argtypes = [C.POINTER(_Grid), p, C.c_uint32, p]
        lib.oracle_tracks.restype = None
        lib.oracle_jets.argtypes = [C.POINTER(_Grid), p, C.c_uint32, C.c_float, C.c_float, C.c_uint32,
                                    C.c_uint32, p, p, p]
        lib.oracle_jets.restype = C.c_uint32
        lib.oracle_vote_variant.argtypes = [C.POINTER(_Grid), C.c_uint32, C.c_uint64, p, p, p, p, p]
        lib.oracle_vote_variant.restype = C.c_int64
        lib.oracle_angle_bin.argtypes = [C.POINTER(_VGrid), C.c_float, C.c_float]
        lib.oracle_angle_bin.restype = C.c_uint32
        lib.oracle_vertex_vote.argtypes = [C.POINTER(_VGrid), C.c_uint32, p, p, p, p, C.c_float, p]
        lib.oracle_vertex_vote.restype = C.c_int64
        lib.oracle_vertices.argtypes = [C.POINTER(_Grid), C.POINTER(_VGrid), p, C.c_uint32, C.c_float, C.c_uint32,
                                        C.c_uint32, p, p, p]
        lib.oracle_vertices.restype = C.c_uint32
        _lib = lib
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


@dataclass(frozen=True)
class Grid:
    """Accumulator geometry; n_d0 == 1 is the prompt 2D mode."""
    n_phi0: int
    n_kappa: int
    n_d0: int = 1
    kappa_max: float = 0.3e-3 * 3.8
    d0_min: float = 0.0
    d0_max: float = 0.0
    b_tesla: float = 3.8
    n_layers: int = 8

    def c(self) -> _Grid:
        return _Grid(self.n_phi0, self.n_kappa, self.n_d0, self.kappa_max, self.d0_min, self.d0_max,
                     self.b_tesla, self.n_layers)

    @property
    def shape(self) -> Tuple[int, int, int]:
        return (self.n_d0, self.n_phi0, self.n_kappa)

    @classmethod
    def from_workload(cls, w) -> "Grid":
        return cls(w.n_phi0, w.n_kappa, w.n_d0, w.kappa_max, w.d0_min, w.d0_max, w.b_tesla, w.n_layers)


@dataclass(frozen=True)
class VGrid:
    """Vertex space of the second Hough transform: phi_v x R_v bins, R_v over [r_min, r_max) (r_min = beam pipe)."""
    n_phi: int = 256
    n_r: int = 128
    r_min: float = 30.0
    r_max: float = 430.0

    def c(self) -> _VGrid:
        return _VGrid(self.n_phi, self.n_r, self.r_min, self.r_max)

    @property
    def shape(self) -> Tuple[int, int]:
        return (self.n_phi, self.n_r)


def angle_bin(v: VGrid, x: float, y: float) -> int:
    cv = v.c()
    return int(_load().oracle_angle_bin(C.byref(cv), x, y))


def vertex_vote(v: VGrid, d0, s0, c0, kappa, d0_cut: float = -1.0):
    """O-6 for tracks given by fp32 parameters: (count uint16 [n_phi, n_r], votes); tracks with |d0| <= d0_cut do not
    vote (the default -1 lets every track vote)."""
    d0 = np.ascontiguousarray(d0, np.float32); s0 = np.ascontiguousarray(s0, np.float32)
    c0 = np.ascontiguousarray(c0, np.float32); kappa = np.ascontiguousarray(kappa, np.float32)
    count = np.zeros(v.shape, np.uint16)
    cv = v.c()
    n = _load().oracle_vertex_vote(C.byref(cv), d0.size, _ptr(d0), _ptr(s0), _ptr(c0), _ptr(kappa), d0_cut, _ptr(count))
    return count, int(n)


def vertices(g: Grid, v: VGrid, pk: np.ndarray, d0_cut_mm: float, n_min: int, max_vertices: int):
    """O-6 + O-7 for ONE event's stored peaks: (stored vertices, total, flag, vertex plane)."""
    pk = np.ascontiguousarray(pk, PEAK_DTYPE)
    out = np.zeros(max_vertices, VERTEX_DTYPE)
    flag = np.zeros(1, np.uint8)
    count = np.zeros(v.shape, np.uint16)
    cg, cv = g.c(), v.c()
    n = int(_load().oracle_vertices(C.byref(cg), C.byref(cv), _ptr(pk), pk.size, d0_cut_mm, n_min, max_vertices,
                                    _ptr(out), _ptr(flag), _ptr(count)))
    return out[:min(n, max_vertices)].copy(), n, int(flag[0]), count


def tables(g: Grid):
    """O-0 tables: (c0[NPHI], s0[NPHI], d0c[ND], inv_dk) as fp32."""
    c0 = np.zeros(g.n_phi0, np.float32); s0 = np.zeros(g.n_phi0, np.float32)
    d0c = np.zeros(g.n_d0, np.float32); inv = np.zeros(1, np.float32)
    cg = g.c()
    _load().oracle_tables(C.byref(cg), _ptr(c0), _ptr(s0), _ptr(d0c), _ptr(inv))
    return c0, s0, d0c, np.float32(inv[0])


def _hits(r, phi, layer):
    r = np.ascontiguousarray(r, np.float32); phi = np.ascontiguousarray(phi, np.float32)
    layer = np.ascontiguousarray(layer, np.uint8)
    assert r.shape == phi.shape == layer.shape and r.ndim == 1
    return r, phi, layer


def hit_prep(phi):
    """O-1 for an array of hit azimuths: (sp, cp) = fp32 roundings of sin / cos evaluated in double (reading R6)."""
    phi = np.ascontiguousarray(phi, np.float32)
    sp = np.zeros(phi.size, np.float32); cp = np.zeros(phi.size, np.float32)
    _load().oracle_hit_prep(phi.size, _ptr(phi), _ptr(sp), _ptr(cp))
    return sp, cp


def vote(g: Grid, r, phi, layer, id_range: Optional[Tuple[int, int]] = None,
         ip_range: Optional[Tuple[int, int]] = None):
    """O-1 + O-2 for ONE event. Returns (count, mask) uint16 [ND, NPHI, NK] and the number of votes."""
    r, phi, layer = _hits(r, phi, layer)
    count = np.zeros(g.shape, np.uint16); mask = np.zeros(g.shape, np.uint16)
    id_lo, id_hi = id_range if id_range else (0, g.n_d0)
    ip_lo, ip_hi = ip_range if ip_range else (0, g.n_phi0)
    cg = g.c()
    n = _load().oracle_vote(C.byref(cg), r.size, _ptr(r), _ptr(phi), _ptr(layer), id_lo, id_hi, ip_lo, ip_hi,
                            _ptr(count), _ptr(mask))
    return count, mask, int(n)


VOTE_HEMI, VOTE_FILL = 1, 2


def vote_variant(g: Grid, flags: int, r, phi, layer):
    """O-2 with the physics-quality variants (VOTE_HEMI forward-hemisphere cut, VOTE_FILL kappa-range filling between
    the phi0 edges of a column) for ONE event: (count, mask) uint16 [ND, NPHI, NK], votes.  flags = 0 is O-2 itself."""
    r, phi, layer = _hits(r, phi, layer)
    count = np.zeros(g.shape, np.uint16); mask = np.zeros(g.shape, np.uint16)
    cg = g.c()
    n = _load().oracle_vote_variant(C.byref(cg), flags, r.size, _ptr(r), _ptr(phi), _ptr(layer), _ptr(count), _ptr(mask))
    return count, mask, int(n)


def vote_columns(g: Grid, r, phi, layer, col_id: Sequence[int], col_ip: Sequence[int]):
    """O-2 for sampled columns of ONE event: (count, mask) uint16 [n_cols, NK], votes."""
    r, phi, layer = _hits(r, phi, layer)
    cid = np.ascontiguousarray(col_id, np.uint32); cip = np.ascontiguousarray(col_ip, np.uint32)
    count = np.zeros((cid.size, g.n_kappa), np.uint16); mask = np.zeros_like(count)
    cg = g.c()
    n = _load().oracle_vote_columns(C.byref(cg), r.size, _ptr(r), _ptr(phi), _ptr(layer), cid.size,
                                    _ptr(cid), _ptr(cip), _ptr(count), _ptr(mask))
    return count, mask, int(n)


def peaks(g: Grid, count: np.ndarray, mask: np.ndarray, l_min: int, max_peaks: int):
    """O-3 for ONE event: (stored peaks [min(total, max_peaks)], total)."""
    count = np.ascontiguousarray(count, np.uint16).reshape(g.shape)
    mask = np.ascontiguousarray(mask, np.uint16).reshape(g.shape)
    out = np.zeros(max_peaks, PEAK_DTYPE)
    cg = g.c()
    total = int(_load().oracle_peaks(C.byref(cg), _ptr(count), _ptr(mask), l_min, max_peaks, _ptr(out)))
    return out[:min(total, max_peaks)].copy(), total


def tracks(g: Grid, pk: np.ndarray):
    """O-4 for ONE event's stored peaks."""
    pk = np.ascontiguousarray(pk, PEAK_DTYPE)
    out = np.zeros(pk.size, TRACK_DTYPE)
    cg = g.c()
    _load().oracle_tracks(C.byref(cg), _ptr(pk), pk.size, _ptr(out))
    return out


def jets(g: Grid, pk: np.ndarray, cone_rad: float, d0_cut_mm: float, n_displaced_min: int, max_jets: int):
    """O-4 + O-5 for ONE event: (tracks with .jet filled, stored jets, n_jets total, flag)."""
    pk = np.ascontiguousarray(pk, PEAK_DTYPE)
    trk = tracks(g, pk)
    out = np.zeros(max_jets, JET_DTYPE)
    flag = np.zeros(1, np.uint8)
    cg = g.c()
    n = int(_load().oracle_jets(C.byref(cg), _ptr(pk), pk.size, cone_rad, d0_cut_mm, n_displaced_min,
                                max_jets, _ptr(trk), _ptr(out), _ptr(flag)))
    return trk, out[:min(n, max_jets)].copy(), n, int(flag[0])


@dataclass
class EventResult:
    count: Optional[np.ndarray]
    mask: Optional[np.ndarray]
    votes: int
    peaks: np.ndarray
    n_peaks: int
    tracks: np.ndarray
    jets: np.ndarray
    n_jets: int
    flag: int


def run_event(g: Grid, r, phi, layer, l_min: int, max_peaks: int, max_jets: int, cone_rad: float,
              d0_cut_mm: float, n_displaced_min: int, keep_planes: bool = True) -> EventResult:
    """The whole chain vote -> peaks -> tracks -> jets for one event (PAPER.md:113 pipeline order)."""
    cnt, msk, nv = vote(g, r, phi, layer)
    pk, tot = peaks(g, cnt, msk, l_min, max_peaks)
    trk, jt, nj, fl = jets(g, pk, cone_rad, d0_cut_mm, n_displaced_min, max_jets)
    return EventResult(cnt if keep_planes else None, msk if keep_planes else None, nv, pk, tot, trk, jt, nj, fl)


def run_batch(g: Grid, batch, l_min: int, max_peaks: int, max_jets: int, cone_rad: float, d0_cut_mm: float,
              n_displaced_min: int, keep_planes: bool = True, workers: int = 1):
    """run_event over every event of a CSR batch (duck-typed: .n_events, .event(e)); `workers` events at once."""
    def one(e):
        r, phi, layer = batch.event(e)
        return run_event(g, r, phi, layer, l_min, max_peaks, max_jets, cone_rad, d0_cut_mm, n_displaced_min,
                         keep_planes)
    if workers <= 1:
        return [one(e) for e in range(batch.n_events)]
    with ThreadPoolExecutor(workers) as ex:
        return list(ex.map(one, range(batch.n_events)))
