"""Shared test helpers: hand-built events, closed-form helix (fp64), result comparison."""
from __future__ import annotations

import dataclasses

import numpy as np

from tpc_workload import ClusterBatch, default_geometry, generate_tracks_event, concat_batches

A_PER_KG = -0.000299792458


def batch_from_rows(geom, task_row_points, n_tasks=None):
    """Build a ClusterBatch from {(task,row): [(y,z), ...]} keeping list order as gid order."""
    n_tasks = n_tasks or geom.n_sectors
    nr = geom.n_rows
    ys, zs, xs = [], [], []
    offs = np.zeros(n_tasks * nr + 1, np.uint32)
    k = 0
    for t in range(n_tasks):
        for r in range(nr):
            pts = task_row_points.get((t, r), [])
            for (y, z) in pts:
                ys.append(y); zs.append(z); xs.append(geom.row_x[r])
            k += len(pts)
            offs[t * nr + r + 1] = k
    n = len(ys)
    return ClusterBatch(geometry=geom, n_tasks=n_tasks, x=np.array(xs, np.float32), y=np.array(ys, np.float32),
                        z=np.array(zs, np.float32), charge=np.full(n, 50, np.uint16), row_offsets=offs,
                        sigma_y=0.1, sigma_z=0.15, truth_track=np.full(n, -1, np.int32),
                        truth_leg=np.full(n, -1, np.int8), truth_state=np.zeros((n, 5)))


def helix_closed_form(x, p, xnew, a):
    """Exact helix propagation in fp64 with libm (y, z, sinphi, dz/dl, q/pT)."""
    y, z, s, t, q = [float(v) for v in p]
    k = a * q
    dx = xnew - x
    s1 = s + k * dx
    if abs(k) < 1e-14:
        c = np.sqrt(1 - s * s)
        return np.array([y + dx * s / c, z + t * dx / c, s1, t, q])
    ph0, ph1 = np.arcsin(s), np.arcsin(s1)
    # cos(ph0) - cos(ph1) = 2 sin((ph0+ph1)/2) sin((ph1-ph0)/2): same value, no cancellation
    dy = 2.0 * np.sin(0.5 * (ph0 + ph1)) * np.sin(0.5 * (ph1 - ph0)) / k
    return np.array([y + dy, z + t * (ph1 - ph0) / k, s1, t, q])


def unpack_cov(c15):
    m = np.zeros((5, 5))
    k = 0
    for i in range(5):
        for j in range(i + 1):
            m[i, j] = m[j, i] = c15[k]
            k += 1
    return m


def pack_cov(m):
    return np.array([m[i, j] for i in range(5) for j in range(i + 1)])


def single_track_events(n_events, rng, pt_range=(0.3, 5.0), sigma_y=0.1, sigma_z=0.15, eta_max=0.9,
                        geom=None):
    """n_events events of ONE primary each (no crossings, no noise), stacked into one batch."""
    geom = geom or default_geometry()
    evs = []
    for e in range(n_events):
        pt = np.exp(rng.uniform(np.log(pt_range[0]), np.log(pt_range[1]), 1))
        ch = np.where(rng.random(1) < 0.5, -1.0, 1.0)
        ph = rng.uniform(0, 2 * np.pi, 1)
        et = rng.uniform(-eta_max, eta_max, 1)
        evs.append(generate_tracks_event(geom, pt, ch, ph, et, np.zeros(1), sigma_y, sigma_z, 0.0, rng,
                                         track_id_base=e * 10))
    return concat_batches(evs)


def tracks_as_dict(res):
    """{(task, tuple(hit gids))} -> index, for set-wise comparison of two results."""
    out = {}
    for t in range(len(res.track_task)):
        b = int(res.track_hit_begin[t]); n = int(res.track_nhits[t])
        out[(int(res.track_task[t]), tuple(int(h) for h in res.hit_cluster[b:b + n]))] = t
    return out
