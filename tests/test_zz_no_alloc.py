"""tpc_slice_frames_static (include/tpc_tracker.h): the frame slicer for callers that cannot allocate.  Its scratch
is a file-scope static device array of the library (TPC_SLICE_STATIC_MAX_ENTRIES uint32), shared by every call.

The GPU test compares its output with the existing path's (tpc_slice_frames with a caller workspace) on two calls
in a row that differ in size and in number of slices, so the second call runs on the first call's leftovers in
the array.  The slicer is index and byte work (SPEC 11 SLICE: an fp32 slice formula, then a stable partition), so
the bar is the one the other slicer tests use: every output array bit-identical.

This file is named so that pytest collects it last (the suite runs with pytest -x); it holds for a fresh process
(`pytest tests/test_zz_no_alloc.py`) and after the other tests alike.
"""
from __future__ import annotations

import ctypes as C

import numpy as np
import pytest


def _frame(n_events, seed, t_shifts, n_slices_in=1):
    from tpc_workload import default_geometry, generate_event, make_frame, CONFIGS
    geom = default_geometry()
    evs = [generate_event(geom, CONFIGS[1]["spec"], seed + i) for i in range(n_events)]
    return geom, make_frame(evs, t_shifts, 1000.0, n_slices_in, seed=seed)


def test_static_slicer_rejects_sizes_beyond_its_array():
    """The size check comes before any CUDA call, so it is checked without a GPU: n_tasks_in*n_rows*n_slices + 2
    entries must fit TPC_SLICE_STATIC_MAX_ENTRIES; beyond it the call returns TPC_ERR_WORKSPACE with a text."""
    from paper_1712_09434_b200 import load_library, SLICE_STATIC_MAX_ENTRIES
    lib = load_library()
    dummy = C.c_void_p(256)  # never dereferenced: the call is refused first
    ns, nr, n_sl = 36, 159, 4
    frames = SLICE_STATIC_MAX_ENTRIES // (ns * nr * n_sl) + 1
    rc = lib.tpc_slice_frames_static(dummy, dummy, dummy, 1, ns * frames, ns, nr, 250.0, n_sl, dummy, dummy, dummy,
                                     dummy, None)
    assert rc == -2, rc  # TPC_ERR_WORKSPACE
    text = lib.tpc_last_error(None).decode()
    assert "static array" in text and str(SLICE_STATIC_MAX_ENTRIES) in text, text


@pytest.mark.gpu
def test_static_slicer_equals_the_workspace_path_on_two_calls_in_a_row():
    import torch
    from paper_1712_09434_b200 import slice_frames, slice_frames_static, slice_static_setup
    dev = torch.device("cuda:0")
    slice_static_setup()          # once per device, at set-up
    slice_static_setup()          # idempotent
    cases = [
        (_frame(5, 700, [0.0, 130.0, 377.0, 512.0, 740.0]), 250.0, 4),   # first call: 4 slices
        (_frame(2, 810, [0.0, 444.0]), 125.0, 7),                        # second: other size, 7 slices, stale scratch
    ]
    for (geom, fr), slice_len, n_sl in cases:
        ns, nr, n = geom.n_sectors, geom.n_rows, fr.n_clusters
        y = torch.from_numpy(np.ascontiguousarray(fr.y)).to(dev)
        z = torch.from_numpy(np.ascontiguousarray(fr.z)).to(dev)
        ro = torch.from_numpy(fr.row_offsets.astype(np.uint32).view(np.int32)).to(dev)
        ref = slice_frames(y, z, ro, ns, ns, nr, slice_len, n_sl)        # existing path: caller workspace
        # the caller's own outputs, poisoned so that an entry the call does not write shows
        y_o = torch.full_like(y, float("nan")); z_o = torch.full_like(z, float("nan"))
        src = torch.full((n,), -7, dtype=torch.int32, device=dev)
        ro_o = torch.full((ns * n_sl * nr + 1,), -7, dtype=torch.int32, device=dev)
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated(dev)
        slice_frames_static(y, z, ro, ns, ns, nr, slice_len, n_sl, y_o, z_o, src, ro_o)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated(dev) == before               # nothing came from torch's allocator either
        for name, a, b in (("y", y_o, ref[0]), ("z", z_o, ref[1]), ("src_index", src, ref[2]),
                           ("row_offsets", ro_o, ref[3])):
            ga, gb = a.cpu().numpy(), b.cpu().numpy()
            assert ga.shape == gb.shape, name
            assert np.array_equal(ga.view(np.uint32), gb.view(np.uint32)), name   # bit-identical
        assert int(ro_o[-1]) == n and int(ro_o[0]) == 0
    # an empty frame goes through as well (no cluster, offsets all zero)
    geom = cases[0][0][0]
    ns, nr = geom.n_sectors, geom.n_rows
    e = torch.empty(0, dtype=torch.float32, device=dev)
    ei = torch.empty(0, dtype=torch.int32, device=dev)
    ro_e = torch.full((ns * 3 * nr + 1,), -7, dtype=torch.int32, device=dev)
    slice_frames_static(e, e, torch.zeros(ns * nr + 1, dtype=torch.int32, device=dev), ns, ns, nr, 250.0, 3, e, e, ei, ro_e)
    torch.cuda.synchronize()
    assert int(ro_e.abs().sum()) == 0
