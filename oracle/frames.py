"""CPU ORACLE of the frame slicer (docs/ARITH_SPEC.md section 11, SLICE; "slice the time frames
along the time / beam axis") - TEST INFRASTRUCTURE.  The definition written out: fp32 slice formula, then a stable
sort by (frame, slice, sector, row).  Shares nothing with paper_1712_09434_b200/.
Pins: tests/test_oracle_frames.py (hand-built rows, permutation / stability / offsets properties).
"""
from __future__ import annotations

import numpy as np


def slice_frames(y, zeta, row_offsets, n_tasks_in: int, n_sectors: int, n_rows: int, slice_len: float, n_slices: int):
    """Returns (y_out, z_out, src_index, row_offsets_out); n_tasks_out = n_tasks_in * n_slices."""
    y = np.asarray(y, np.float32)
    zeta = np.asarray(zeta, np.float32)
    ro = np.asarray(row_offsets, np.int64)
    n = y.shape[0]
    tr = np.repeat(np.arange(n_tasks_in * n_rows), np.diff(ro))
    task, row = tr // n_rows, tr % n_rows
    frame, sec = task // n_sectors, task % n_sectors
    inv = np.float32(1.0) / np.float32(slice_len)
    f = np.fmin(np.fmax(np.abs(zeta) * inv, np.float32(0)), np.float32(n_slices - 1))
    f = np.where(np.isnan(f), np.float32(0), f)
    sl = f.astype(np.int64)
    out_tr = ((frame * n_slices + sl) * n_sectors + sec) * n_rows + row
    order = np.argsort(out_tr, kind="stable")
    counts = np.bincount(out_tr, minlength=n_tasks_in * n_slices * n_rows)
    ro_out = np.zeros(n_tasks_in * n_slices * n_rows + 1, np.uint32)
    ro_out[1:] = np.cumsum(counts)
    assert int(ro_out[-1]) == n
    return y[order], zeta[order], order.astype(np.uint32), ro_out
