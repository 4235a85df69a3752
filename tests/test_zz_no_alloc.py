"""hough_jets_static: the jet step for callers that are not allowed to allocate device memory.

Every other entry point needs a context, and hough_create calls cudaMalloc for the workspaces of the whole path.  Some
users cannot do that: a trigger process that handed out all of its device memory at start-up and must stay inside that
budget, a real-time loop in which an allocation would stall every stream of the GPU, a plug-in whose host runtime owns
the allocator and passes it nothing but input and output buffers.  hough_jets_static gives them A5-A6 (peak -> track,
phi-cone jets, displaced-jet flag) with its scratch in a fixed array that is part of the library's device image
(4 MiB of clustering keys + 16 KiB of d0 bin centres, see include/hough.h).

This file checks, on a GPU, that the new call returns what the existing hough_jets returns -- integer fields equal,
floats within the tolerance the other parity tests use -- on two calls in a row that share the scratch array (the second
with another grid and shorter events, so anything stale left by the first would show), including events with more than
4096 tracks, the only ones whose keys leave shared memory.  It is named test_zz_* so that pytest collects it last:
`pytest -x` stops at the first failure, and a failure here must not hide the parity tests.
"""
import ctypes as C

import numpy as np
import pytest

RTOL, ATOL = 1e-5, 1e-6          # tests/test_gpu_parity.py's tolerances for the reported floats


def _cfg(B, n_phi0, n_kappa, n_d0, d0_min, d0_max, max_events, max_peaks, max_jets):
    return B.HoughConfig(n_phi0, n_kappa, n_d0, 0.3e-3 * 3.8, d0_min, d0_max, 3.8, 8, max_events, 1, max_peaks, max_jets,
                         0, 0, 0, 0, 30.0, 430.0, 0, 0)


def test_static_entry_refuses_what_its_fixed_scratch_cannot_hold():
    """Sizes beyond the fixed array are rejected with their own error code before anything touches the GPU (so this
    part runs without one): the caller learns that it has to shrink the call, not that 'something was invalid'."""
    from paper_1309_6275_b200 import binding as B
    lib = B.load_library()
    one = C.c_void_p(16)                                         # any non-null pointer: the call returns before using it
    args = (one, one, 0.4, 2.0, 3, one, one, one, one, None)
    ok_peaks = B.JETS_STATIC_MAX_TRACKS // 64
    too_many_tracks = _cfg(B, 128, 64, 8, -20.0, 20.0, 65, ok_peaks, 16)
    assert lib.hough_jets_static(C.byref(too_many_tracks), 65, *args) == B.ETOOLARGE
    too_many_d0 = _cfg(B, 16, 8, B.JETS_STATIC_MAX_D0 + 1, -20.0, 20.0, 1, 16, 16)
    assert lib.hough_jets_static(C.byref(too_many_d0), 1, *args) == B.ETOOLARGE
    assert "HOUGH_JETS_STATIC_MAX_TRACKS" in B.strerror(B.ETOOLARGE)
    bad = _cfg(B, 128, 60, 8, -20.0, 20.0, 1, 16, 16)            # n_kappa % 8 != 0: as hough_create
    assert lib.hough_jets_static(C.byref(bad), 1, *args) == -1
    assert lib.hough_jets_static(None, 1, *args) == -1
    good = _cfg(B, 128, 64, 8, -20.0, 20.0, 1, 16, 16)
    assert lib.hough_jets_static(C.byref(good), 1, None, *args[1:]) == -1


def _peak_lists(B, rng, bins, sizes, max_peaks):
    pk = np.zeros((len(sizes), max_peaks), B.PEAK_DTYPE)
    for e, T in enumerate(sizes):
        pk[e, :T]["lin"] = np.sort(rng.choice(bins, T, replace=False))
    return pk


def _same(B, got, ref, sizes, max_jets, what):
    nj, rnj = got["n_jets"].cpu().numpy(), ref["n_jets"].cpu().numpy()
    assert np.array_equal(nj, rnj), what
    assert np.array_equal(got["flag"].cpu().numpy(), ref["flag"].cpu().numpy()), what
    jt, rjt = B.records(got["jets"], B.JET_DTYPE), B.records(ref["jets"], B.JET_DTYPE)
    tr, rtr = B.records(got["tracks"], B.TRACK_DTYPE), B.records(ref["tracks"], B.TRACK_DTYPE)
    for e, T in enumerate(sizes):
        J = min(int(rnj[e]), max_jets)
        for f in ("seed_track", "n_tracks", "n_displaced"):
            assert np.array_equal(jt[e, :J][f], rjt[e, :J][f]), (what, e, f)
        for f in ("phi", "sum_pt"):
            assert np.allclose(jt[e, :J][f], rjt[e, :J][f], rtol=RTOL), (what, e, f)
        for f in ("jet", "q"):
            assert np.array_equal(tr[e, :T][f], rtr[e, :T][f]), (what, e, f)
        for f in ("pt", "phi0", "d0"):
            assert np.allclose(tr[e, :T][f], rtr[e, :T][f], rtol=RTOL, atol=ATOL), (what, e, f)


@pytest.mark.gpu
def test_static_entry_matches_hough_jets_on_two_calls_in_a_row():
    import torch
    from paper_1309_6275_b200 import binding as B
    rng = np.random.default_rng(31)
    # call 1: long events (keys of the events above 4096 tracks go to the static array), 8 d0 bins
    # call 2: another grid (16 d0 bins over another range: the d0 table in the array must be rewritten) and events that
    #         are shorter than call 1's at the same index (stale keys beyond T must not be read)
    calls = [dict(grid=(128, 64, 8, -20.0, 20.0), max_peaks=8192, max_jets=64,
                  sizes=[8192, 6000, 4097, 4096, 512, 33, 1, 0], args=(0.4, 2.0, 3)),
             dict(grid=(256, 32, 16, -35.0, 5.0), max_peaks=8192, max_jets=32,
                  sizes=[5000, 4100, 100, 4097, 0, 7000, 8192, 2], args=(0.1, 8.0, 2))]
    free_before_second = free_after_second = None
    for k, c in enumerate(calls):
        nphi, nk, nd, d0_min, d0_max = c["grid"]
        E, mp, mj = len(c["sizes"]), c["max_peaks"], c["max_jets"]
        pk = _peak_lists(B, rng, nd * nphi * nk, c["sizes"], mp)
        dpk = torch.from_numpy(pk.view(np.uint8).reshape(E, mp, 8)).cuda()
        dn = torch.tensor(c["sizes"], dtype=torch.int32).cuda()
        # the existing path: a context (which allocates) and hough_jets
        h = B.Hough(nphi, nk, nd, d0_min=d0_min, d0_max=d0_max, max_events=E, max_hits=1, max_peaks_per_event=mp,
                    max_jets_per_event=mj)
        ref = h.alloc_outputs(E)
        h.hough_jets(E, dpk, dn, *c["args"], ref["tracks"], ref["jets"], ref["n_jets"], ref["flag"])
        got = h.alloc_outputs(E)                                  # plain torch buffers: the caller's outputs
        cfg = _cfg(B, nphi, nk, nd, d0_min, d0_max, E, mp, mj)
        torch.cuda.synchronize()
        if k == 1:
            free_before_second = torch.cuda.mem_get_info()[0]
        B.hough_jets_static(cfg, E, dpk, dn, *c["args"], got["tracks"], got["jets"], got["n_jets"], got["flag"])
        torch.cuda.synchronize()
        if k == 1:
            free_after_second = torch.cuda.mem_get_info()[0]
        _same(B, got, ref, c["sizes"], mj, f"call {k + 1}")
        assert int(got["n_jets"].sum()) > 0                       # not vacuous
        h.close()
    # once the first call has done the per-device set-up, a call takes no device memory at all
    assert free_after_second >= free_before_second, (free_before_second, free_after_second)
