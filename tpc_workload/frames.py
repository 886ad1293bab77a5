"""Synthetic time frames (docs/ARITH_SPEC.md section 11; continuous read-out, "time frames with
many overlapping events", sliced "along the time / beam axis").  Seeded INPUT only: events of ``events.py`` are
overlaid with a shift of their z coordinate (a cluster of an event that happened dt later is read out dt later, i.e.
v_drift*dt further along the frame axis) and every cluster is filed under the slice its frame coordinate falls in.
None of the tracker's arithmetic lives here.
"""
from __future__ import annotations

import dataclasses
from typing import Sequence

import numpy as np

from .events import ClusterBatch


def make_frame(events: Sequence[ClusterBatch], shifts_cm: Sequence[float], slice_len_cm: float, n_slices: int,
               seed: int = 0) -> ClusterBatch:
    """Overlay single-event batches (n_tasks = n_sectors each) into ONE frame.

    The frame coordinate of a cluster is zeta = z + shift on the A side (z >= 0) and z - shift on the C side, so
    |zeta| grows with the shift on both sides; its slice is floor(|zeta| / slice_len_cm), clipped to n_slices - 1.
    Returns a batch with n_tasks = n_slices * n_sectors, task = slice*n_sectors + sector, ``z`` = zeta (fp32), the
    geometry's z_max enlarged to the frame length, truth kept per cluster (truth_track unique over the frame;
    truth_state[:, 1] shifted like z).  Order inside a row: a seeded shuffle.
    """
    g = events[0].geometry
    ns, nr = g.n_sectors, g.n_rows
    parts = []
    base = 0
    for ev, sh in zip(events, shifts_cm):
        assert ev.n_tasks == ns
        tr = np.repeat(np.arange(ns * nr), np.diff(ev.row_offsets.astype(np.int64)))
        sec, row = tr // nr, tr % nr
        sgn = np.where(2 * sec < ns, 1.0, -1.0) if ns >= 2 else np.ones(len(tr))
        zeta = ev.z.astype(np.float64) + sgn * sh
        st = ev.truth_state.copy()
        st[:, 1] += sgn * sh
        tt = ev.truth_track.astype(np.int64)
        tt = np.where(tt >= 0, tt + base, -1)
        base += int(ev.truth_track.max()) + 1 if len(ev.truth_track) else 0
        parts.append((sec, row, ev.y, zeta, ev.charge, tt, ev.truth_leg, st, ev.x))
    sec, row, y, zeta, q, tt, leg, st, x = (np.concatenate(c) for c in zip(*parts))
    sl = np.minimum((np.abs(zeta) / slice_len_cm).astype(np.int64), n_slices - 1)
    key = (sl * ns + sec) * nr + row
    rng = np.random.Generator(np.random.PCG64(seed))
    perm = np.lexsort((rng.random(len(key)), key))
    counts = np.bincount(key, minlength=n_slices * ns * nr)
    ro = np.zeros(n_slices * ns * nr + 1, np.uint32)
    ro[1:] = np.cumsum(counts)
    z_len = float(slice_len_cm * n_slices)
    return ClusterBatch(geometry=dataclasses.replace(g, z_max=z_len), n_tasks=n_slices * ns,
                        x=x[perm].astype(np.float32), y=y[perm].astype(np.float32), z=zeta[perm].astype(np.float32),
                        charge=q[perm], row_offsets=ro, sigma_y=events[0].sigma_y, sigma_z=events[0].sigma_z,
                        truth_track=tt[perm].astype(np.int32), truth_leg=leg[perm], truth_state=st[perm], tracks={})
