"""Thin ctypes binding of libhough_b200.so -- argument marshalling only (include/hough.h is the contract).

PyTorch is used for device memory and streams, nothing else: every step of the path (hit preparation, vote,
peak stencil, compaction, tracks, jets) runs in the library's CUDA kernels.  There is no CPU fallback: if the
shared library is missing or no CUDA device is present, loading / hough_create fail loudly.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhough_b200.so")

PEAK_DTYPE = np.dtype([("lin", "<u4"), ("count", "<u2"), ("mask", "<u2")])
TRACK_DTYPE = np.dtype([("pt", "<f4"), ("phi0", "<f4"), ("d0", "<f4"), ("q", "<i4"), ("jet", "<i4")])
JET_DTYPE = np.dtype([("seed_track", "<u4"), ("n_tracks", "<u4"), ("n_displaced", "<u4"),
                      ("phi", "<f4"), ("sum_pt", "<f4")])
VERTEX_DTYPE = np.dtype([("r", "<f4"), ("phi", "<f4"), ("n_tracks", "<u4"), ("lin", "<u4")])

JETS_STATIC_MAX_TRACKS, JETS_STATIC_MAX_D0, ETOOLARGE = 1 << 19, 4096, -5
ST_EVENT_TOO_LARGE, ST_BAD_OFFSETS, ST_TRIG_ROUNDING, ST_CANDIDATE_OVERFLOW = 1, 2, 4, 8
ST_ERRORS = ST_EVENT_TOO_LARGE | ST_BAD_OFFSETS            # the bits that mean "results undefined"
N_PEAKS_OVERFLOW = 0xFFFFFFFF
VOTE_HEMI, VOTE_FILL = 1, 2
DEBUG_NO_MIRROR, DEBUG_TILES_COUNT, DEBUG_TILES_MASK = 1, 2, 4      # hough_config.debug_flags (tests, measurements)
EXPORTS = ["hough_create", "hough_destroy", "hough_plane_bytes", "hough_vote", "hough_peaks", "hough_vote_peaks",
           "hough_jets", "hough_jets_static", "hough_vertices", "hough_trigger_host_vtx",
           "hough_trigger_host", "hough_status", "hough_launch_count", "hough_last_tile_kind", "hough_microbench", "hough_strerror",
           "hough_debug_prepared_hits", "hough_debug_div_check", "hough_profile", "hough_profile_read"]


class HoughConfig(C.Structure):
    _fields_ = [("n_phi0", C.c_uint32), ("n_kappa", C.c_uint32), ("n_d0", C.c_uint32),
                ("kappa_max", C.c_float), ("d0_min", C.c_float), ("d0_max", C.c_float), ("b_tesla", C.c_float),
                ("n_layers", C.c_uint32), ("max_events", C.c_uint32), ("max_hits", C.c_uint64),
                ("max_peaks_per_event", C.c_uint32), ("max_jets_per_event", C.c_uint32),
                ("host_chunk_events", C.c_uint32), ("max_candidates_per_event", C.c_uint32),
                ("n_vtx_phi", C.c_uint32), ("n_vtx_r", C.c_uint32), ("vtx_r_min", C.c_float), ("vtx_r_max", C.c_float),
                ("max_vertices_per_event", C.c_uint32), ("vote_flags", C.c_uint32), ("max_plane_events", C.c_uint32),
                ("debug_flags", C.c_uint32)]


class HoughError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {strerror(code)} (code {code})")


_lib = None


def load_library() -> C.CDLL:
    """dlopen the in-tree CUDA library; never falls back to anything else."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1309_6275_b200.build` "
                "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        p, u32, u64, f32 = C.c_void_p, C.c_uint32, C.c_uint64, C.c_float
        lib.hough_create.argtypes = [C.POINTER(HoughConfig), C.POINTER(p)]
        lib.hough_destroy.argtypes = [p]
        lib.hough_plane_bytes.argtypes = [p, u32]
        lib.hough_plane_bytes.restype = C.c_size_t
        lib.hough_vote.argtypes = [p, u32, p, u64, p, p, p, p, p, p]
        lib.hough_peaks.argtypes = [p, u32, p, p, u32, p, p, p]
        lib.hough_vote_peaks.argtypes = [p, u32, p, u64, p, p, p, u32, p, p, p]
        lib.hough_jets.argtypes = [p, u32, p, p, f32, f32, u32, p, p, p, p, p]
        lib.hough_jets_static.argtypes = [C.POINTER(HoughConfig), u32, p, p, f32, f32, u32, p, p, p, p, p]
        lib.hough_trigger_host.argtypes = [p, u32, p, u64, p, p, p, u32, f32, f32, u32, p, p, p, p, p, p, p]
        lib.hough_trigger_host_vtx.argtypes = [p, u32, p, u64, p, p, p, u32, f32, f32, u32, u32, p, p, p, p, p, p, p, p, p, p]
        lib.hough_vertices.argtypes = [p, u32, p, p, f32, u32, p, p, p, p, p]
        lib.hough_status.argtypes = [p, C.POINTER(u32)]
        lib.hough_launch_count.argtypes = [p, C.POINTER(u64)]
        lib.hough_last_tile_kind.argtypes = [p, C.POINTER(C.c_int)]
        lib.hough_microbench.argtypes = [C.c_int, C.c_size_t, C.POINTER(C.c_double)]
        lib.hough_debug_prepared_hits.argtypes = [p, u64, p, C.POINTER(u32)]
        lib.hough_debug_div_check.argtypes = [u64, u64, f32, u32, C.POINTER(u64)]
        lib.hough_profile.argtypes = [p, C.c_int]
        lib.hough_profile_read.argtypes = [p, C.POINTER(f32), C.POINTER(u32)]
        lib.hough_strerror.argtypes = [C.c_int]
        lib.hough_strerror.restype = C.c_char_p
        for name in EXPORTS:
            if name not in ("hough_plane_bytes", "hough_strerror"):
                getattr(lib, name).restype = C.c_int
        _lib = lib
    return _lib


def strerror(code: int) -> str:
    return load_library().hough_strerror(code).decode()


def _check(code: int, where: str):
    if code != 0:
        raise HoughError(code, where)


def microbench(kind: int, nbytes: int = 0) -> float:
    """hough_microbench: 0 shared atomics/s, 1 fp32 non-FMA instr/s, 2 HBM read B/s, 3 HBM write B/s,
    4 packed fp32x2 instr/s, 5 / 6 bytes/s all SMs can store into L2 (coalesced / vote-flush pattern)."""
    out = C.c_double(0.0)
    _check(load_library().hough_microbench(kind, nbytes, C.byref(out)), "hough_microbench")
    return out.value


def debug_div_check(n_pairs: int, seed: int = 1, kappa_max: float = 0.3e-3 * 3.8, n_kappa: int = 512):
    """hough_debug_div_check -> (quotient mismatches, bin mismatches, pairs inside the kappa axis)."""
    out = (C.c_uint64 * 3)()
    _check(load_library().hough_debug_div_check(n_pairs, seed, kappa_max, n_kappa, out), "hough_debug_div_check")
    return int(out[0]), int(out[1]), int(out[2])


def _dptr(t) -> C.c_void_p:
    return C.c_void_p(t.data_ptr())


def _stream_ptr(stream=None) -> C.c_void_p:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def hough_jets_static(cfg: HoughConfig, n_events, d_peaks, d_n_peaks, cone_rad, d0_cut_mm, n_displaced_min, d_tracks,
                      d_jets, d_n_jets, d_flag, stream=None):
    """hough_jets for callers that may not allocate device memory (a process on a fixed memory budget, a real-time
    loop, a plug-in whose host owns the allocator): no context, hence no hough_create and no cudaMalloc.  `cfg` is a
    HoughConfig describing the grid (host side); the tensors are the caller's device buffers as for Hough.hough_jets.
    The scratch is a fixed array inside the library: HoughError(ETOOLARGE) if n_events * max_peaks_per_event >
    JETS_STATIC_MAX_TRACKS or n_d0 > JETS_STATIC_MAX_D0.  All calls on a device share that array, so keep them
    ordered on the GPU (one stream, or events between streams)."""
    _check(load_library().hough_jets_static(C.byref(cfg), n_events, _dptr(d_peaks), _dptr(d_n_peaks), cone_rad,
                                            d0_cut_mm, n_displaced_min, _dptr(d_tracks), _dptr(d_jets),
                                            _dptr(d_n_jets), _dptr(d_flag), _stream_ptr(stream)), "hough_jets_static")


class Hough:
    """Owner of one hough_ctx.  Methods mirror the C entry points one to one (same names, same order)."""

    def __init__(self, n_phi0: int, n_kappa: int, n_d0: int = 1, kappa_max: float = 0.3e-3 * 3.8,
                 d0_min: float = 0.0, d0_max: float = 0.0, b_tesla: float = 3.8, n_layers: int = 8,
                 max_events: int = 1, max_hits: int = 1 << 16, max_peaks_per_event: int = 4096,
                 max_jets_per_event: int = 256, host_chunk_events: int = 0, max_candidates_per_event: int = 0,
                 n_vtx_phi: int = 0, n_vtx_r: int = 0, vtx_r_min: float = 30.0, vtx_r_max: float = 430.0,
                 max_vertices_per_event: int = 64, vote_flags: int = 0, max_plane_events: int = 0,
                 debug_flags: int = 0):
        self.lib = load_library()
        self.cfg = HoughConfig(n_phi0, n_kappa, n_d0, kappa_max, d0_min, d0_max, b_tesla, n_layers, max_events,
                               max(1, max_hits), max_peaks_per_event, max_jets_per_event, host_chunk_events,
                               max_candidates_per_event, n_vtx_phi, n_vtx_r, vtx_r_min, vtx_r_max,
                               max_vertices_per_event, vote_flags, max_plane_events, debug_flags)
        self._ctx = C.c_void_p()
        _check(self.lib.hough_create(C.byref(self.cfg), C.byref(self._ctx)), "hough_create")

    @classmethod
    def for_workload(cls, w, max_events: Optional[int] = None, max_hits: Optional[int] = None,
                     host_chunk_events: int = 0, max_peaks: Optional[int] = None,
                     max_candidates: int = 0, vgrid=None, max_vertices: int = 64, vote_flags: int = 0,
                     max_plane_events: int = 0, debug_flags: int = 0) -> "Hough":
        """vgrid: None, or (n_vtx_phi, n_vtx_r, r_min, r_max) for the second Hough transform (hough_vertices)."""
        ne = w.n_events if max_events is None else max_events
        if max_hits is None:
            raise ValueError("for_workload: pass max_hits (the hit count of the largest batch per call); the context "
                             "allocates 36 B of workspace per hit")
        mh = max_hits
        return cls(w.n_phi0, w.n_kappa, w.n_d0, w.kappa_max, w.d0_min, w.d0_max, w.b_tesla, w.n_layers, ne,
                   min(mh, 0xFFFFFFFF), w.max_peaks if max_peaks is None else max_peaks, w.max_jets,
                   host_chunk_events, max_candidates, *((0, 0, 30.0, 430.0) if vgrid is None else vgrid), max_vertices, vote_flags,
                   max_plane_events, debug_flags)

    # -- lifetime ---------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx:
            self.lib.hough_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- sizes ------------------------------------------------------------------------------------
    @property
    def bins_per_event(self) -> int:
        return self.cfg.n_d0 * self.cfg.n_phi0 * self.cfg.n_kappa

    def hough_plane_bytes(self, n_events: int) -> int:
        return int(self.lib.hough_plane_bytes(self._ctx, n_events))

    def alloc_planes(self, n_events: int):
        """Two uint16 device tensors [E, ND, NPHI, NK] (torch has no uint16 arithmetic; int16 storage is used)."""
        import torch
        shape = (n_events, self.cfg.n_d0, self.cfg.n_phi0, self.cfg.n_kappa)
        return (torch.empty(shape, dtype=torch.int16, device="cuda"),
                torch.empty(shape, dtype=torch.int16, device="cuda"))

    def alloc_outputs(self, n_events: int):
        import torch
        mp, mj = self.cfg.max_peaks_per_event, self.cfg.max_jets_per_event
        dev = "cuda"
        return dict(
            peaks=torch.zeros((n_events, mp, PEAK_DTYPE.itemsize), dtype=torch.uint8, device=dev),
            n_peaks=torch.zeros(n_events, dtype=torch.int32, device=dev),
            tracks=torch.zeros((n_events, mp, TRACK_DTYPE.itemsize), dtype=torch.uint8, device=dev),
            jets=torch.zeros((n_events, mj, JET_DTYPE.itemsize), dtype=torch.uint8, device=dev),
            n_jets=torch.zeros(n_events, dtype=torch.int32, device=dev),
            flag=torch.zeros(n_events, dtype=torch.uint8, device=dev),
            vertices=torch.zeros((n_events, max(1, self.cfg.max_vertices_per_event), VERTEX_DTYPE.itemsize),
                                 dtype=torch.uint8, device=dev),
            n_vertices=torch.zeros(n_events, dtype=torch.int32, device=dev),
            vtx_flag=torch.zeros(n_events, dtype=torch.uint8, device=dev))

    # -- the hot path (device pointers + caller stream) -------------------------------------------
    def hough_vote(self, n_events, d_hit_offsets, n_hits_total, d_r, d_phi, d_layer, d_count, d_mask, stream=None):
        _check(self.lib.hough_vote(self._ctx, n_events, _dptr(d_hit_offsets), n_hits_total, _dptr(d_r), _dptr(d_phi),
                                   _dptr(d_layer), _dptr(d_count), _dptr(d_mask), _stream_ptr(stream)), "hough_vote")

    def hough_peaks(self, n_events, d_count, d_mask, l_min, d_peaks, d_n_peaks, stream=None):
        _check(self.lib.hough_peaks(self._ctx, n_events, _dptr(d_count), _dptr(d_mask), l_min, _dptr(d_peaks),
                                    _dptr(d_n_peaks), _stream_ptr(stream)), "hough_peaks")

    def hough_vote_peaks(self, n_events, d_hit_offsets, n_hits_total, d_r, d_phi, d_layer, l_min, d_peaks, d_n_peaks,
                         stream=None):
        _check(self.lib.hough_vote_peaks(self._ctx, n_events, _dptr(d_hit_offsets), n_hits_total, _dptr(d_r),
                                         _dptr(d_phi), _dptr(d_layer), l_min, _dptr(d_peaks), _dptr(d_n_peaks),
                                         _stream_ptr(stream)), "hough_vote_peaks")

    def hough_jets(self, n_events, d_peaks, d_n_peaks, cone_rad, d0_cut_mm, n_displaced_min, d_tracks, d_jets,
                   d_n_jets, d_flag, stream=None):
        _check(self.lib.hough_jets(self._ctx, n_events, _dptr(d_peaks), _dptr(d_n_peaks), cone_rad, d0_cut_mm,
                                   n_displaced_min, _dptr(d_tracks), _dptr(d_jets), _dptr(d_n_jets), _dptr(d_flag),
                                   _stream_ptr(stream)), "hough_jets")

    def hough_vertices(self, n_events, d_peaks, d_n_peaks, d0_cut_mm, n_min, d_vertices, d_n_vertices, d_flag,
                       d_vertex_plane=None, stream=None):
        plane = C.c_void_p(0) if d_vertex_plane is None else _dptr(d_vertex_plane)
        _check(self.lib.hough_vertices(self._ctx, n_events, _dptr(d_peaks), _dptr(d_n_peaks), d0_cut_mm, n_min,
                                       _dptr(d_vertices), _dptr(d_n_vertices), _dptr(d_flag), plane,
                                       _stream_ptr(stream)), "hough_vertices")

    def hough_trigger_host_vtx(self, n_events, h_hit_offsets, n_hits_total, h_r, h_phi, h_layer, l_min, cone_rad,
                               d0_cut_mm, n_displaced_min, vtx_n_min, h_n_peaks, h_n_jets, h_flag, h_peaks, h_jets,
                               h_n_vertices, h_vtx_flag, h_vertices=None, ms_stage=None, stream=None):
        """hough_trigger_host + the second Hough transform; HOST tensors / arrays in and out."""
        def hp(x):
            if x is None:
                return C.c_void_p(0)
            return C.c_void_p(x.ctypes.data) if isinstance(x, np.ndarray) else C.c_void_p(x.data_ptr())
        _check(self.lib.hough_trigger_host_vtx(self._ctx, n_events, hp(h_hit_offsets), n_hits_total, hp(h_r), hp(h_phi),
                                               hp(h_layer), l_min, cone_rad, d0_cut_mm, n_displaced_min, vtx_n_min,
                                               hp(h_n_peaks), hp(h_n_jets), hp(h_flag), hp(h_peaks), hp(h_jets),
                                               hp(h_n_vertices), hp(h_vtx_flag), hp(h_vertices), hp(ms_stage),
                                               _stream_ptr(stream)), "hough_trigger_host_vtx")

    def hough_trigger_host(self, n_events, h_hit_offsets, n_hits_total, h_r, h_phi, h_layer, l_min, cone_rad,
                           d0_cut_mm, n_displaced_min, h_n_peaks, h_n_jets, h_flag, h_peaks=None, h_jets=None,
                           ms_stage=None, stream=None):
        """HOST tensors / arrays in and out (torch CPU tensors, ideally pinned, or numpy arrays)."""
        def hp(x):
            if x is None:
                return C.c_void_p(0)
            return C.c_void_p(x.ctypes.data) if isinstance(x, np.ndarray) else C.c_void_p(x.data_ptr())
        _check(self.lib.hough_trigger_host(self._ctx, n_events, hp(h_hit_offsets), n_hits_total, hp(h_r), hp(h_phi),
                                           hp(h_layer), l_min, cone_rad, d0_cut_mm, n_displaced_min, hp(h_n_peaks),
                                           hp(h_n_jets), hp(h_flag), hp(h_peaks), hp(h_jets), hp(ms_stage),
                                           _stream_ptr(stream)), "hough_trigger_host")

    def hough_status(self) -> int:
        out = C.c_uint32(0)
        _check(self.lib.hough_status(self._ctx, C.byref(out)), "hough_status")
        return out.value

    def hough_debug_prepared_hits(self, n_hits: int):
        """(records float32 [n_hits, 4] = sp, cp, r, layer-bit pattern; number of hits flagged trig-rounding risk)."""
        rec = np.zeros((max(n_hits, 1), 4), np.float32)
        risk = C.c_uint32(0)
        _check(self.lib.hough_debug_prepared_hits(self._ctx, n_hits, C.c_void_p(rec.ctypes.data), C.byref(risk)),
               "hough_debug_prepared_hits")
        return rec[:n_hits], risk.value

    def hough_profile(self, enable: bool):
        _check(self.lib.hough_profile(self._ctx, 1 if enable else 0), "hough_profile")

    def hough_profile_read(self):
        """(ms per stage {prep, vote, peaks, jets, vertices} since the last read, number of calls)."""
        ms = (C.c_float * 5)(); n = C.c_uint32(0)
        _check(self.lib.hough_profile_read(self._ctx, ms, C.byref(n)), "hough_profile_read")
        return [float(x) for x in ms], int(n.value)

    def hough_last_tile_kind(self) -> int:
        """0 no fused launch yet, 1 count + mask tiles, 2 mask tiles (what the last fused launch started with)."""
        out = C.c_int(0)
        _check(self.lib.hough_last_tile_kind(self._ctx, C.byref(out)), "hough_last_tile_kind")
        return out.value

    def hough_launch_count(self) -> int:
        out = C.c_uint64(0)
        _check(self.lib.hough_launch_count(self._ctx, C.byref(out)), "hough_launch_count")
        return out.value


# -- conveniences used by tests / bench: upload a CSR batch, view raw output tensors as numpy records --------

def upload_batch(batch):
    """numpy CSR batch -> device tensors (offsets int32 storage of the uint32 values, r, phi, layer)."""
    import torch
    off = torch.from_numpy(batch.hit_offsets.view(np.int32)).cuda()
    r = torch.from_numpy(batch.r).cuda()
    phi = torch.from_numpy(batch.phi).cuda()
    layer = torch.from_numpy(batch.layer).cuda()
    return off, r, phi, layer


def records(t, dtype: np.dtype) -> np.ndarray:
    """Device uint8 tensor [..., itemsize] -> numpy structured array [...]."""
    a = t.cpu().numpy()
    return a.view(dtype).reshape(a.shape[:-1])


def planes_to_numpy(t) -> np.ndarray:
    return t.cpu().numpy().view(np.uint16)
