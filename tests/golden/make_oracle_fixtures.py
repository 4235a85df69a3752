#!/usr/bin/env python
"""Writes tests/golden/oracle_regression.json: a few small seeded events run through the CPU oracle (oracle/ only, plus the
seeded input generator), so that an accidental change of the oracle's arithmetic, of a reading or of
the generator shows up as a diff of this file.  These are NOT paper values: the paper prints no worked example, no
equation and no table for this path (PAPER.md:85-123 describe it in words; its figures are not in the container), so
there is no paper fixture to store; what pins the oracle's correctness are P1-P20 in tests/test_oracle_pins.py.

    python tests/golden/make_oracle_fixtures.py          # rewrites the file; commit it with the change that explains it
"""
import hashlib
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import hough_oracle as O                      # noqa: E402
from paper_1309_6275_b200 import workloads as W           # noqa: E402

CASES = [
    ("C1", W.config(1), 0, 0),
    ("C2 on 16 x 128 x 64", W.scaled(W.config(2), n_d0=16, n_phi0=128, n_kappa=64), 0, 0),
    ("C4 content on 8 x 96 x 72, L_min 6", W.scaled(W.config(4), n_d0=8, n_phi0=96, n_kappa=72, l_min=6), 1, 0),
    ("C2 on 8 x 128 x 64, hemisphere cut + kappa-range filling", W.scaled(W.config(2), n_d0=8, n_phi0=128, n_kappa=64), 0, 3),
]


def digest(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


def run_case(name, w, event, flags):
    g = O.Grid.from_workload(w)
    r, phi, layer, _ = W.generate_event(w, event)
    if flags:
        count, mask, votes = O.vote_variant(g, flags, r, phi, layer)
    else:
        count, mask, votes = O.vote(g, r, phi, layer)
    peaks, n_peaks = O.peaks(g, count, mask, w.l_min, w.max_peaks)
    _, jets, n_jets, flag = O.jets(g, peaks, w.cone_rad, w.d0_cut_mm, w.n_displaced_min, w.max_jets)
    vtx, n_vtx, vflag, vplane = O.vertices(g, O.VGrid(*w.vgrid), peaks, w.d0_cut_mm, w.vtx_n_min, w.max_vertices)
    return {"case": name, "event": event, "vote_flags": flags, "hits": int(r.size), "votes": int(votes),
            "count_sha256": digest(count), "mask_sha256": digest(mask), "count_max": int(count.max()),
            "n_peaks": int(n_peaks), "first_peaks_lin": [int(x) for x in peaks["lin"][:8]],
            "first_peaks_count": [int(x) for x in peaks["count"][:8]], "n_jets": int(n_jets), "flag": int(flag),
            "jet_seeds": [int(x) for x in jets["seed_track"][:8]], "n_vertices": int(n_vtx), "vertex_flag": int(vflag),
            "vertex_plane_sha256": digest(vplane)}


def make():
    return [run_case(*c) for c in CASES]


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.json")
    with open(out, "w") as f:
        json.dump(make(), f, indent=1)
        f.write("\n")
    print("wrote", out)
