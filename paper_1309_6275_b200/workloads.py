"""Seeded synthetic tracker workloads (the five BASELINE.json configs) -- INPUT GENERATION ONLY.

This module serves both the CPU oracle (``oracle/``) and the CUDA path: it draws hits, nothing else.
It holds none of the method's arithmetic (no voting formula, no binning, no peak or jet logic); the
only geometry here is the *forward* model "where does a charged track cross a detector layer", which
is the detector simulation the paper calls its Monte-Carlo toy model (section 5), with
the tracker, field and multiplicities that BASELINE.json's ``configs`` fix.

Conventions:
  * units mm, rad, T, GeV; curvature kappa in 1/mm, kappa > 0 = counter-clockwise;
  * a particle of charge q and transverse momentum pT has kappa = -q * 0.3e-3 * B / pT;
  * a track is the circle through its point of closest approach P = d0*(sin phi0, -cos phi0)
    with tangent (cos phi0, sin phi0) there; centre = P + n/kappa, n = (-sin phi0, cos phi0);
  * one hit per forward layer crossing, phi smeared by N(0,1)*0.02/r rad, wrapped to [0, 2pi),
    stored as fp32; r is exactly the layer radius; noise hits: uniform layer, uniform phi;
  * event k of a config with seed S draws from numpy.random.default_rng([S, k]).

numpy only; no torch, no CUDA, no oracle import.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Dict, List, Optional, Tuple

import numpy as np

TWO_PI = 2.0 * np.pi

TRACKER_A = (40.0, 70.0, 110.0, 250.0, 330.0, 430.0, 520.0, 600.0)            # 8 barrel layers, mm
TRACKER_B = TRACKER_A + (700.0, 800.0, 900.0, 1000.0)                          # 12 layers
# the paper's toy detector (section 5): beam pipe of radius 30 mm, ten concentric evenly spaced layers,
# overall radius 1100 mm, hit resolution 0.4 mm
TRACKER_PAPER = tuple(30.0 + (i + 1) * (1100.0 - 30.0) / 10.0 for i in range(10))
B_TESLA = 3.8
KAPPA_MAX = 0.3e-3 * B_TESLA / 1.0        # |kappa| of a 1 GeV track, 1/mm  (configs: "0.3*3.8/1 GeV per m")


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config made concrete."""
    name: str
    seed: int
    n_events: int
    radii: Tuple[float, ...]
    # accumulator grid
    n_d0: int
    n_phi0: int
    n_kappa: int
    d0_min: float = 0.0
    d0_max: float = 0.0
    kappa_max: float = KAPPA_MAX
    b_tesla: float = B_TESLA
    # selection
    l_min: int = 6
    max_peaks: int = 4096
    max_jets: int = 256
    cone_rad: float = 0.4
    d0_cut_mm: float = 2.0
    n_displaced_min: int = 3
    # vertex space of the second Hough transform (beam pipe 30 mm) and its threshold
    vtx_n_phi: int = 256
    vtx_n_r: int = 128
    vtx_r_min: float = 30.0
    vtx_r_max: float = 430.0
    vtx_n_min: int = 4
    max_vertices: int = 64
    # event content
    n_prompt: Tuple[int, int] = (10, 10)            # inclusive integer range
    prompt_pt: str = "uniform_1_20"                 # or "exp2_trunc1"
    n_noise: Tuple[int, int] = (100, 100)
    n_llp: Tuple[int, int] = (0, 0)                 # displaced vertices per event (inclusive range)
    llp_prob: float = 1.0                           # probability that an event has any
    llp_radius: Tuple[float, float] = (10.0, 300.0)
    llp_tracks: Tuple[int, int] = (4, 4)
    llp_pt: Tuple[float, float] = (1.0, 10.0)
    llp_half_angle: float = 0.3
    llp_half_angle_range: Optional[Tuple[float, float]] = None   # if set: drawn per vertex, replaces llp_half_angle
    hit_sigma_mm: float = 0.02                      # azimuthal smearing of a hit: N(0,1) * hit_sigma_mm / r  (R27)
    vote_flags: int = 0                             # hough_config.vote_flags the workload is meant to be run with

    @property
    def n_layers(self) -> int:
        return len(self.radii)

    @property
    def bins_per_event(self) -> int:
        return self.n_d0 * self.n_phi0 * self.n_kappa

    @property
    def vgrid(self):
        return (self.vtx_n_phi, self.vtx_n_r, self.vtx_r_min, self.vtx_r_max)


def config(k: int) -> Workload:
    """BASELINE.json ``configs[k-1]`` (k = 1..5) with the readings R14, R15, R23, R29 filled in."""
    if k == 1:
        return Workload("C1", 1, 1, TRACKER_A, 1, 512, 256, l_min=6,
                        n_prompt=(10, 10), prompt_pt="uniform_1_20", n_noise=(100, 100))
    if k == 2:
        return Workload("C2", 2, 1, TRACKER_A, 64, 512, 256, -50.0, 50.0, l_min=4,
                        n_prompt=(20, 20), prompt_pt="uniform_1_20", n_noise=(300, 300),
                        n_llp=(2, 2), llp_radius=(10.0, 300.0), llp_tracks=(4, 4), llp_pt=(1.0, 10.0))
    if k == 3:
        return Workload("C3", 3, 1000, TRACKER_A, 1, 1024, 512, l_min=6,
                        n_prompt=(200, 200), prompt_pt="exp2_trunc1", n_noise=(1000, 1000))
    if k == 4:
        return Workload("C4", 4, 256, TRACKER_B, 128, 1024, 512, -100.0, 100.0, l_min=9, max_peaks=16384,
                        n_prompt=(500, 500), prompt_pt="exp2_trunc1", n_noise=(3000, 3000),
                        n_llp=(3, 3), llp_radius=(5.0, 400.0), llp_tracks=(6, 12), llp_pt=(1.0, 30.0))
    if k == 5:
        return Workload("C5", 5, 4096, TRACKER_B, 128, 1024, 512, -100.0, 100.0, l_min=9, max_peaks=16384,
                        n_prompt=(50, 400), prompt_pt="exp2_trunc1", n_noise=(500, 2000),
                        n_llp=(1, 4), llp_prob=0.10, llp_radius=(5.0, 400.0), llp_tracks=(6, 12),
                        llp_pt=(1.0, 30.0))
    raise ValueError("config index must be 1..5")


def paper_timing(n_tracks: int, n_events: int = 32) -> Workload:
    """"P4": the paper's own timing benchmark (Fig. 4 "Time vs. tracks per event, 2048x2048"): the
    ten-layer toy detector, 0.4 mm hit resolution, a 2048 x 2048 (phi0 x kappa) prompt accumulator, n_tracks tracks of
    10 hits each per event (the paper's curve runs to 3,000 tracks), no noise hits; the peak finder
    expects "7 or more hits per track".  pT is not stated: 1 + Exp(2) GeV as in the other configs."""
    return Workload(f"P4-{n_tracks}", 40, n_events, TRACKER_PAPER, 1, 2048, 2048, l_min=7, max_peaks=16384,
                    n_prompt=(n_tracks, n_tracks), prompt_pt="exp2_trunc1", n_noise=(0, 0), hit_sigma_mm=0.4)


def paper_efficiency(kind: str, x: int, n_events: int = 64) -> Workload:
    """The paper's three efficiency studies (section 7) on its toy detector (ten layers, 0.4 mm):
      "F8"  one displaced jet of x tracks, nothing else (Fig. 8: efficiency vs tracks per jet);
      "F9"  x displaced jets of 10 tracks each, nothing else (Fig. 9: efficiency vs jets per event);
      "F10" 3,000 tracks in total, x displaced jets of 10 tracks among them, the rest prompt (Fig. 10).
    Every track has 10 hits, so a displaced vertex lies between the 30 mm beam pipe and the first
    layer (137 mm): R_v uniform in [40, 130] mm.  "Dispersion angles between 15 and 60 degrees" is read
    as the full opening angle of a jet: its tracks leave the vertex within +- half of it around the radial direction.
    Not stated in the paper and chosen here (R43): jet-track pT uniform 1-30 GeV, prompt pT 1 + Exp(2) GeV, a
    3D accumulator of 64 d0 bins over [-80, 80] mm x 1024 x 512 voted with the forward-hemisphere cut and kappa-range
    filling (vote_flags 3), tracks = peaks with all 10 layers (with filled bands a lower threshold multiplies the
    duplicate peaks per track), vertices of 7 or more tracks (the paper's "7 or more", "simple reuse" of
    the peak finder's threshold) on a 256 x 128 (phi_v, R_v) grid over [30, 430) mm."""
    deg = np.pi / 180.0
    base = dict(n_events=n_events, radii=TRACKER_PAPER, n_d0=64, n_phi0=1024, n_kappa=512, d0_min=-80.0, d0_max=80.0,
                l_min=10, max_peaks=16384, max_jets=256, d0_cut_mm=2.5, vtx_n_min=7, max_vertices=256, n_noise=(0, 0),
                vote_flags=3,
                prompt_pt="exp2_trunc1", llp_radius=(40.0, 130.0), llp_pt=(1.0, 30.0), hit_sigma_mm=0.4,
                llp_half_angle_range=(7.5 * deg, 30.0 * deg))
    if kind == "F8":
        return Workload(f"F8-{x}", 80, n_prompt=(0, 0), n_llp=(1, 1), llp_tracks=(x, x), **base)
    if kind == "F9":
        return Workload(f"F9-{x}", 90, n_prompt=(0, 0), n_llp=(x, x), llp_tracks=(10, 10), **base)
    if kind == "F10":
        base["max_peaks"] = 65535                                # the most a context with a vertex grid accepts (hough.h)
        return Workload(f"F10-{x}", 100, n_prompt=(3000 - 10 * x, 3000 - 10 * x), n_llp=(x, x), llp_tracks=(10, 10), **base)
    raise ValueError("kind must be F8, F9 or F10")


def scaled(w: Workload, **kw) -> Workload:
    """Same recipe on a smaller grid / fewer events (parity-test cases the oracle finishes in seconds)."""
    return replace(w, **kw)


@dataclass
class EventBatch:
    """CSR batch of events: hits of event e are [hit_offsets[e], hit_offsets[e+1])."""
    hit_offsets: np.ndarray          # uint32 [E+1]
    r: np.ndarray                    # float32 [H]
    phi: np.ndarray                  # float32 [H]
    layer: np.ndarray                # uint8   [H]
    truth: List[Dict[str, np.ndarray]] = field(default_factory=list)   # per event; tests only

    @property
    def n_events(self) -> int:
        return int(self.hit_offsets.shape[0] - 1)

    @property
    def n_hits(self) -> int:
        return int(self.r.shape[0])

    def event(self, e: int) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
        a, b = int(self.hit_offsets[e]), int(self.hit_offsets[e + 1])
        return self.r[a:b], self.phi[a:b], self.layer[a:b]

    def slice(self, e0: int, e1: int) -> "EventBatch":
        a, b = int(self.hit_offsets[e0]), int(self.hit_offsets[e1])
        off = (self.hit_offsets[e0:e1 + 1].astype(np.int64) - a).astype(np.uint32)
        return EventBatch(off, self.r[a:b].copy(), self.phi[a:b].copy(), self.layer[a:b].copy(),
                          self.truth[e0:e1] if self.truth else [])


# ----------------------------------------------------------------------------------------------
# detector forward model
# ----------------------------------------------------------------------------------------------

def _prompt_hits(kappa: np.ndarray, phi0: np.ndarray, radii: np.ndarray):
    """Forward crossings of tracks from the origin (d0 = 0): phi = phi0 + asin(kappa r / 2)  (R26)."""
    a = 0.5 * kappa[:, None] * radii[None, :]
    ok = np.abs(a) <= 1.0
    phi = phi0[:, None] + np.arcsin(np.clip(a, -1.0, 1.0))
    lay = np.broadcast_to(np.arange(radii.size)[None, :], a.shape)
    rr = np.broadcast_to(radii[None, :], a.shape)
    return rr[ok], phi[ok], lay[ok]


def _displaced_hits(vx, vy, psi, kappa, radii, r_vertex):
    """First forward crossing of every layer with r > r_vertex by circles starting at V heading psi (R28).

    Position after arc length L: x(L) = C + (1/kappa) * (sin(psi + kappa L), -cos(psi + kappa L)),
    C = V + (1/kappa) * (-sin psi, cos psi).  |x(L)| = r  <=>  sin(theta - gamma) = rhs with
    theta = psi + kappa L, C = |C| (cos gamma, sin gamma), rhs = (r^2 - |C|^2 - 1/kappa^2) kappa / (2 |C|).
    """
    inv_k = 1.0 / kappa
    cx = vx - inv_k * np.sin(psi)
    cy = vy + inv_k * np.cos(psi)
    cn = np.hypot(cx, cy)
    gam = np.arctan2(cy, cx)
    rhs = (radii[None, :] ** 2 - (cn ** 2 + inv_k ** 2)[:, None]) * (kappa / (2.0 * cn))[:, None]
    reach = (np.abs(rhs) <= 1.0) & (radii[None, :] > r_vertex[:, None])
    beta = np.arcsin(np.clip(rhs, -1.0, 1.0))
    period = (TWO_PI / np.abs(kappa))[:, None]
    best = np.full(rhs.shape, np.inf)
    for th in (gam[:, None] + beta, gam[:, None] + np.pi - beta):
        L = np.mod((th - psi[:, None]) * inv_k[:, None], period)
        best = np.minimum(best, L)
    theta = psi[:, None] + kappa[:, None] * best
    x = cx[:, None] + inv_k[:, None] * np.sin(theta)
    y = cy[:, None] - inv_k[:, None] * np.cos(theta)
    phi = np.arctan2(y, x)
    lay = np.broadcast_to(np.arange(radii.size)[None, :], rhs.shape)
    rr = np.broadcast_to(radii[None, :], rhs.shape)
    return rr[reach], phi[reach], lay[reach]


def track_params_from_circle(vx, vy, psi, kappa):
    """(d0, phi0) of the circle through V with direction psi and curvature kappa (truth for tests).

    centre C = (1/kappa - d0) * (-sin phi0, cos phi0)  =>  d0 = 1/kappa - sg*|C|, sg = sign(1/kappa - d0);
    the physical branch is the one with |d0| < |1/kappa| i.e. sg = sign(kappa).
    """
    inv_k = 1.0 / kappa
    cx = vx - inv_k * np.sin(psi)
    cy = vy + inv_k * np.cos(psi)
    sg = np.sign(kappa)
    cn = np.hypot(cx, cy)
    d0 = inv_k - sg * cn
    phi0 = np.mod(np.arctan2(-cx * sg, cy * sg), TWO_PI)
    return d0, phi0


def _draw_pt(rng, kind: str, n: int) -> np.ndarray:
    if kind == "uniform_1_20":
        return rng.uniform(1.0, 20.0, n)
    if kind == "exp2_trunc1":                       # exponential mean 2 truncated at >= 1 (memoryless form, R29)
        return 1.0 + rng.exponential(2.0, n)
    raise ValueError(kind)


def _randint_incl(rng, lo_hi: Tuple[int, int]) -> int:
    lo, hi = lo_hi
    return int(lo) if lo == hi else int(rng.integers(lo, hi + 1))


def generate_event(w: Workload, k: int, seed: Optional[int] = None):
    """Hits of event k: (r f32, phi f32, layer u8, truth dict)."""
    rng = np.random.default_rng([w.seed if seed is None else seed, k])
    radii = np.asarray(w.radii, dtype=np.float64)
    rs, phis, lays = [], [], []

    n_p = _randint_incl(rng, w.n_prompt)
    pt = _draw_pt(rng, w.prompt_pt, n_p)
    phi0 = rng.uniform(0.0, TWO_PI, n_p)
    q = rng.choice(np.array([-1.0, 1.0]), n_p)
    kap = -q * 0.3e-3 * w.b_tesla / pt
    r_, p_, l_ = _prompt_hits(kap, phi0, radii)
    rs.append(r_); phis.append(p_); lays.append(l_)
    truth = {"prompt_pt": pt, "prompt_phi0": phi0, "prompt_kappa": kap}

    n_v = 0
    if w.n_llp[1] > 0 and (w.llp_prob >= 1.0 or rng.uniform() < w.llp_prob):
        n_v = _randint_incl(rng, w.n_llp)
    v_r = rng.uniform(w.llp_radius[0], w.llp_radius[1], n_v)
    v_phi = rng.uniform(0.0, TWO_PI, n_v)
    d_v, d_psi, d_kap, d_rv = [], [], [], []
    for j in range(n_v):
        n_t = _randint_incl(rng, w.llp_tracks)
        half = w.llp_half_angle if w.llp_half_angle_range is None else rng.uniform(*w.llp_half_angle_range)
        d_psi.append(v_phi[j] + rng.uniform(-half, half, n_t))
        dq = rng.choice(np.array([-1.0, 1.0]), n_t)
        dpt = rng.uniform(w.llp_pt[0], w.llp_pt[1], n_t)
        d_kap.append(-dq * 0.3e-3 * w.b_tesla / dpt)
        d_v.append(np.full(n_t, j))
        d_rv.append(np.full(n_t, v_r[j]))
    if n_v:
        d_v = np.concatenate(d_v); d_psi = np.concatenate(d_psi)
        d_kap = np.concatenate(d_kap); d_rv = np.concatenate(d_rv)
        vx = v_r[d_v] * np.cos(v_phi[d_v]); vy = v_r[d_v] * np.sin(v_phi[d_v])
        r_, p_, l_ = _displaced_hits(vx, vy, d_psi, d_kap, radii, d_rv)
        rs.append(r_); phis.append(p_); lays.append(l_)
        dd0, dphi0 = track_params_from_circle(vx, vy, d_psi, d_kap)
        truth.update(disp_vertex=d_v, disp_kappa=d_kap, disp_d0=dd0, disp_phi0=dphi0,
                     vertex_r=v_r, vertex_phi=v_phi)
    truth["n_vertices"] = n_v

    r_sig = np.concatenate(rs); p_sig = np.concatenate(phis); l_sig = np.concatenate(lays)
    p_sig = p_sig + rng.standard_normal(p_sig.size) * (w.hit_sigma_mm / r_sig)   # R27

    n_n = _randint_incl(rng, w.n_noise)
    l_n = rng.integers(0, radii.size, n_n)
    p_n = rng.uniform(0.0, TWO_PI, n_n)
    r_all = np.concatenate([r_sig, radii[l_n]])
    p_all = np.mod(np.concatenate([p_sig, p_n]), TWO_PI)
    l_all = np.concatenate([l_sig, l_n])
    perm = rng.permutation(r_all.size)                # hit order carries no information (R25)
    return (r_all[perm].astype(np.float32), p_all[perm].astype(np.float32),
            l_all[perm].astype(np.uint8), truth)


def generate(w: Workload, n_events: Optional[int] = None, first_event: int = 0,
             keep_truth: bool = False) -> EventBatch:
    """Events first_event .. first_event+n_events-1 of workload w as one CSR batch."""
    n = w.n_events if n_events is None else n_events
    rs, ps, ls, tr = [], [], [], []
    off = np.zeros(n + 1, dtype=np.int64)
    for i in range(n):
        r, p, l, t = generate_event(w, first_event + i)
        rs.append(r); ps.append(p); ls.append(l)
        off[i + 1] = off[i] + r.size
        if keep_truth:
            tr.append(t)
    if n == 0:
        return EventBatch(np.zeros(1, np.uint32), np.zeros(0, np.float32), np.zeros(0, np.float32),
                          np.zeros(0, np.uint8), [])
    assert off[-1] < 2 ** 32
    return EventBatch(off.astype(np.uint32), np.concatenate(rs), np.concatenate(ps), np.concatenate(ls), tr)


def batch_from_events(events) -> EventBatch:
    """Build a CSR batch from a list of (r, phi, layer) triples (hand-made test events)."""
    off = np.zeros(len(events) + 1, dtype=np.int64)
    for i, (r, _, _) in enumerate(events):
        off[i + 1] = off[i] + len(r)
    cat = lambda j, dt: (np.concatenate([np.asarray(ev[j], dtype=dt) for ev in events])
                         if events else np.zeros(0, dt))
    return EventBatch(off.astype(np.uint32), cat(0, np.float32), cat(1, np.float32), cat(2, np.uint8), [])
