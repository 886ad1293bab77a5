"""Synthetic Pb-Pb-shaped TPC events: geometry, helices, clusters, truth.

Stands in for the paper's 2015 Pb-Pb selection (Table 1), which
does not exist on this box.  Recipe = SURVEY.md section 8(d) / BASELINE.json
``configs``; every deviation is listed in DESIGN.md ("Input recipe").

Only inputs are made here.  All helix maths is fp64 closed form (circle in
x-y, linear in z); the result is smeared and cast to fp32.  Nothing in this
file is used by the tracker arithmetic of either implementation.

Conventions
-----------
* Global frame: beam along z, B = (0, 0, +Bz).  Signed curvature
  ``kappa = -c * Bz[kG] * charge / pT`` [1/cm], c = 0.000299792458, so the
  direction angle obeys d(psi)/d(s_xy) = kappa.
* Sector k (0..17) is centred at azimuth (k + 0.5) * 20 deg.  Sector index
  ``s = k`` for z > 0 (A side) and ``s = k + 18`` for z < 0 (C side).
  Local frame of a sector: x along its centre line, y across, z = global z.
* Pad row r is the plane ``x_local = row_x[r]``, limited to
  ``|y_local| <= row_x[r] * tan(10 deg)``.
* task = event * n_sectors + sector; clusters are stored sorted by
  (task, row) with a seeded random order inside every row.
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

C_KAPPA = 0.000299792458  # GeV / (kG * cm)
SECTOR_PITCH = np.deg2rad(20.0)
N_PHI_FULL = 18
R_OUT = 252.0  # cm: a track that reaches this radius has left the TPC


# --------------------------------------------------------------------------
# geometry
# --------------------------------------------------------------------------
@dataclass(frozen=True)
class Geometry:
    n_sectors: int
    n_rows: int
    row_x: np.ndarray  # float32 [n_rows], strictly increasing
    tan_half_angle: np.float32
    z_max: float
    bz_kgauss: float

    @property
    def n_phi(self) -> int:
        return max(self.n_sectors // 2, 1)

    @property
    def two_sided(self) -> bool:
        return self.n_sectors >= 2

    def sector_angle(self, sector: int) -> float:
        return (sector % self.n_phi + 0.5) * SECTOR_PITCH


def default_geometry(n_sectors: int = 36, n_rows: int = 159,
                     bz_kgauss: float = 5.0) -> Geometry:
    """36 sectors x 159 rows, radii uniform 85..247 cm, Bz = 0.5 T."""
    r = np.arange(n_rows, dtype=np.float64)
    denom = max(n_rows - 1, 1)
    row_x = (85.0 + 162.0 * r / denom).astype(np.float32)
    return Geometry(n_sectors=n_sectors, n_rows=n_rows, row_x=row_x,
                    tan_half_angle=np.float32(np.tan(np.deg2rad(10.0))),
                    z_max=250.0, bz_kgauss=bz_kgauss)


# --------------------------------------------------------------------------
# event recipe
# --------------------------------------------------------------------------
@dataclass(frozen=True)
class EventSpec:
    n_primaries: int
    pt_range: Tuple[float, float]
    eta_max: float = 0.9
    n_loopers: int = 0
    looper_pt_range: Tuple[float, float] = (0.05, 0.1)
    noise_frac: float = 0.0
    sigma_y: float = 0.1
    sigma_z: float = 0.15
    vertex_z_spread: float = 0.0  # uniform +- this
    phi_in_first_sector: bool = False  # config 0: phi within the one sector


@dataclass
class ClusterBatch:
    """Tracker input (x, y, z, charge, row_offsets) plus generator truth."""
    geometry: Geometry
    n_tasks: int
    x: np.ndarray          # float32 [N]
    y: np.ndarray          # float32 [N]
    z: np.ndarray          # float32 [N]
    charge: np.ndarray     # uint16  [N]
    row_offsets: np.ndarray  # uint32 [n_tasks * n_rows + 1]
    sigma_y: float
    sigma_z: float
    # truth (never shown to a tracker)
    truth_track: np.ndarray  # int32 [N]; -1 = noise; unique per (event, track)
    truth_leg: np.ndarray    # int8  [N]; 0 outgoing (+x), 1 incoming, -1 noise
    truth_state: np.ndarray  # float64 [N,5]: y, z, sinphi, dz/ds, q/pT (local, +x going)
    tracks: Dict[str, np.ndarray] = field(default_factory=dict)

    @property
    def n_clusters(self) -> int:
        return int(self.x.shape[0])

    @property
    def n_events(self) -> int:
        return self.n_tasks // self.geometry.n_sectors


# --------------------------------------------------------------------------
# helix -> row crossings (fp64, closed form)
# --------------------------------------------------------------------------
def _track_sector_pairs(phi0, sgn, theta_max, n_phi):
    """(track, k) pairs whose 20-degree wedge the arc can touch.

    Seen from the origin, a point of a circle through the origin at turning
    angle theta sits at azimuth phi0 + sgn*theta/2 (chord angle = half the
    turning angle), so the arc covers azimuths [phi0, phi0 + sgn*theta_max/2].
    """
    a0 = phi0
    a1 = phi0 + sgn * 0.5 * theta_max
    lo = np.minimum(a0, a1)
    hi = np.maximum(a0, a1)
    klo = np.floor(lo / SECTOR_PITCH - 1e-9).astype(np.int64)
    khi = np.floor(hi / SECTOR_PITCH + 1e-9).astype(np.int64)
    cnt = np.minimum(khi - klo + 1, N_PHI_FULL)
    ti = np.repeat(np.arange(phi0.shape[0]), cnt)
    first = np.cumsum(cnt) - cnt
    k = np.repeat(klo, cnt) + (np.arange(ti.shape[0]) - np.repeat(first, cnt))
    k = np.mod(k, N_PHI_FULL)
    keep = k < n_phi
    return ti[keep], k[keep]


def _crossings(geom: Geometry, pt, charge, phi0, eta, z0):
    """All (track, sector, row, branch) crossings; returns dict of flat arrays."""
    n_trk = pt.shape[0]
    X = geom.row_x.astype(np.float64)
    tan_h = np.tan(np.deg2rad(10.0))
    kappa = -C_KAPPA * geom.bz_kgauss * charge / pt
    sgn = np.sign(kappa)
    radius = 1.0 / np.abs(kappa)
    theta_max = np.where(2.0 * radius <= R_OUT, 2.0 * np.pi,
                         2.0 * np.arcsin(np.minimum(R_OUT / (2.0 * radius), 1.0)))
    t = np.sinh(eta)
    if not geom.two_sided:
        t = np.abs(t)  # single-sector geometry: fold eta onto the A side

    ti_all, k_all = _track_sector_pairs(phi0, sgn, theta_max, geom.n_phi)
    out = {n: [] for n in ("trk", "sec", "row", "leg", "y", "z", "s", "sin", "t", "q")}
    rows = np.arange(geom.n_rows)
    chunk = 4096
    for c0 in range(0, ti_all.shape[0], chunk):
        ti = ti_all[c0:c0 + chunk]
        k = k_all[c0:c0 + chunk]
        alpha = (k + 0.5) * SECTOR_PITCH
        kap = kappa[ti][:, None]
        ph = phi0[ti][:, None]
        al = alpha[:, None]
        v = np.sin(ph - al) + kap * X[None, :]           # sin(psi - alpha) on the row
        ok_v = np.abs(v) <= 1.0
        av = np.arcsin(np.clip(v, -1.0, 1.0))
        for leg in (0, 1):
            psi = al + (av if leg == 0 else (np.pi - av))
            theta = np.mod(sgn[ti][:, None] * (psi - ph), 2.0 * np.pi)
            s_xy = theta * radius[ti][:, None]
            xg = (np.sin(psi) - np.sin(ph)) / kap
            yg = -(np.cos(psi) - np.cos(ph)) / kap
            yl = -xg * np.sin(al) + yg * np.cos(al)
            xl = xg * np.cos(al) + yg * np.sin(al)
            zz = z0[ti][:, None] + t[ti][:, None] * s_xy
            ok = (ok_v & (theta > 1e-12) & (theta < theta_max[ti][:, None])
                  & (np.abs(xl - X[None, :]) < 1e-6)       # rejects the 2*pi alias
                  & (np.abs(yl) <= X[None, :] * tan_h)
                  & (np.abs(zz) <= geom.z_max) & (zz != 0.0))
            if not geom.two_sided:
                ok &= zz > 0.0
            pi_, ri_ = np.nonzero(ok)
            zsel = zz[pi_, ri_]
            side = (zsel < 0.0).astype(np.int64) if geom.two_sided else 0
            flip = -1.0 if leg == 1 else 1.0
            out["trk"].append(ti[pi_])
            out["sec"].append(k[pi_] + side * geom.n_phi)
            out["row"].append(rows[ri_])
            out["leg"].append(np.full(pi_.shape[0], leg, dtype=np.int8))
            out["y"].append(yl[pi_, ri_])
            out["z"].append(zsel)
            out["s"].append(s_xy[pi_, ri_])
            out["sin"].append(flip * v[pi_, ri_])
            out["t"].append(flip * t[ti][pi_])
            out["q"].append(flip * (charge / pt)[ti][pi_])
    return {n: (np.concatenate(a) if a else np.zeros(0)) for n, a in out.items()}, n_trk


def _crossings_straight(geom: Geometry, pt, charge, phi0, eta, z0):
    """Bz = 0: straight lines from (0, 0, z0); same output as ``_crossings`` (leg 0 only)."""
    X = geom.row_x.astype(np.float64)
    tan_h = np.tan(np.deg2rad(10.0))
    t = np.sinh(eta)
    if not geom.two_sided:
        t = np.abs(t)
    out = {n: [] for n in ("trk", "sec", "row", "leg", "y", "z", "s", "sin", "t", "q")}
    rows = np.arange(geom.n_rows)
    for i in range(pt.shape[0]):
        for k in range(geom.n_phi):
            d = np.mod(phi0[i] - (k + 0.5) * SECTOR_PITCH + np.pi, 2.0 * np.pi) - np.pi
            if abs(d) >= 0.5 * np.pi:
                continue
            yl = X * np.tan(d)
            s_xy = X / np.cos(d)
            zz = z0[i] + t[i] * s_xy
            ok = (np.abs(yl) <= X * tan_h) & (np.abs(zz) <= geom.z_max) & (zz != 0.0) & (s_xy < R_OUT)
            if not geom.two_sided:
                ok &= zz > 0.0
            ri_ = np.nonzero(ok)[0]
            side = (zz[ri_] < 0.0).astype(np.int64) if geom.two_sided else 0
            n = ri_.shape[0]
            out["trk"].append(np.full(n, i)); out["sec"].append(k + side * geom.n_phi)
            out["row"].append(rows[ri_]); out["leg"].append(np.zeros(n, np.int8))
            out["y"].append(yl[ri_]); out["z"].append(zz[ri_]); out["s"].append(s_xy[ri_])
            out["sin"].append(np.full(n, np.sin(d))); out["t"].append(np.full(n, t[i]))
            out["q"].append(np.full(n, charge[i] / pt[i]))
    return {n: (np.concatenate([np.atleast_1d(v) for v in a]) if a else np.zeros(0)) for n, a in out.items()}, pt.shape[0]


def _moyal_charge(rng, n, mpv=50.0, width=10.0):
    """Moyal(mpv, width) stand-in for a Landau: x = mpv - width*ln(Z^2)."""
    zn = rng.standard_normal(n)
    q = mpv - width * np.log(np.maximum(zn * zn, 1e-300))
    return np.clip(np.rint(q), 1, 65535).astype(np.uint16)


def generate_tracks_event(geom: Geometry, pt, charge, phi0, eta, z0,
                          sigma_y: float, sigma_z: float, noise_frac: float,
                          rng: np.random.Generator, track_id_base: int = 0,
                          shuffle: bool = True) -> ClusterBatch:
    """Clusters of ONE event for explicitly given tracks (all arrays fp64)."""
    pt = np.asarray(pt, np.float64)
    charge = np.asarray(charge, np.float64)
    phi0 = np.asarray(phi0, np.float64)
    eta = np.asarray(eta, np.float64)
    z0 = np.asarray(z0, np.float64)
    if geom.bz_kgauss == 0.0:
        cr, _ = _crossings_straight(geom, pt, charge, phi0, eta, z0)
    else:
        cr, _ = _crossings(geom, pt, charge, phi0, eta, z0)
    n_rows = geom.n_rows
    n_sr = geom.n_sectors * n_rows
    sr = cr["sec"].astype(np.int64) * n_rows + cr["row"].astype(np.int64)
    # canonical order before any draw: (sector,row), then track, leg, path length
    order = np.lexsort((cr["s"], cr["leg"], cr["trk"], sr))
    for n in cr:
        cr[n] = cr[n][order]
    sr = sr[order]
    n_hit = sr.shape[0]
    y = cr["y"] + sigma_y * rng.standard_normal(n_hit)
    z = cr["z"] + sigma_z * rng.standard_normal(n_hit)
    # noise: Poisson(frac * n_row) per (sector,row), uniform over the row's y-z extent
    per_row = np.bincount(sr, minlength=n_sr)
    n_noise = rng.poisson(noise_frac * per_row) if noise_frac > 0 else np.zeros(n_sr, np.int64)
    tot_noise = int(n_noise.sum())
    sr_n = np.repeat(np.arange(n_sr), n_noise)
    row_n = sr_n % n_rows
    sec_n = sr_n // n_rows
    half_w = geom.row_x.astype(np.float64)[row_n] * np.tan(np.deg2rad(10.0))
    y_n = (2.0 * rng.random(tot_noise) - 1.0) * half_w
    z_n = rng.random(tot_noise) * geom.z_max
    if geom.two_sided:
        z_n = np.where(sec_n >= geom.n_phi, -z_n, z_n)
    # merge
    sr_all = np.concatenate([sr, sr_n])
    y_all = np.concatenate([y, y_n])
    z_all = np.concatenate([z, z_n])
    trk_all = np.concatenate([cr["trk"].astype(np.int64) + track_id_base,
                              np.full(tot_noise, -1, np.int64)])
    leg_all = np.concatenate([cr["leg"].astype(np.int8), np.full(tot_noise, -1, np.int8)])
    state = np.zeros((n_hit + tot_noise, 5), np.float64)
    state[:n_hit, 0] = cr["y"]
    state[:n_hit, 1] = cr["z"]
    state[:n_hit, 2] = cr["sin"]
    state[:n_hit, 3] = cr["t"]
    state[:n_hit, 4] = cr["q"]
    n_all = sr_all.shape[0]
    q_adc = _moyal_charge(rng, n_all)
    key = rng.random(n_all) if shuffle else np.arange(n_all, dtype=np.float64)
    perm = np.lexsort((key, sr_all))
    sr_all = sr_all[perm]
    row_offsets = np.zeros(n_sr + 1, np.uint32)
    row_offsets[1:] = np.cumsum(np.bincount(sr_all, minlength=n_sr))
    return ClusterBatch(
        geometry=geom, n_tasks=geom.n_sectors,
        x=geom.row_x[(sr_all % n_rows)].astype(np.float32),
        y=y_all[perm].astype(np.float32), z=z_all[perm].astype(np.float32),
        charge=q_adc[perm], row_offsets=row_offsets,
        sigma_y=sigma_y, sigma_z=sigma_z,
        truth_track=trk_all[perm].astype(np.int32), truth_leg=leg_all[perm],
        truth_state=state[perm],
        tracks={"pt": pt, "charge": charge, "phi0": phi0, "eta": eta, "z0": z0})


def generate_event(geom: Geometry, spec: EventSpec, seed: int,
                   track_id_base: int = 0) -> ClusterBatch:
    """One event drawn from ``spec`` with ``PCG64(seed)`` in a fixed draw order."""
    rng = np.random.Generator(np.random.PCG64(seed))

    def draw(n, pt_lo, pt_hi):
        pt = np.exp(rng.uniform(np.log(pt_lo), np.log(pt_hi), n))
        ch = np.where(rng.random(n) < 0.5, -1.0, 1.0)
        if spec.phi_in_first_sector:
            ph = rng.uniform(0.0, SECTOR_PITCH, n)
        else:
            ph = rng.uniform(0.0, 2.0 * np.pi, n)
        et = rng.uniform(-spec.eta_max, spec.eta_max, n)
        if spec.vertex_z_spread > 0:
            zv = rng.uniform(-spec.vertex_z_spread, spec.vertex_z_spread, n)
        else:
            zv = np.zeros(n)
        return pt, ch, ph, et, zv

    parts = [draw(spec.n_primaries, *spec.pt_range)]
    if spec.n_loopers > 0:
        parts.append(draw(spec.n_loopers, *spec.looper_pt_range))
    pt, ch, ph, et, zv = (np.concatenate(c) for c in zip(*parts))
    return generate_tracks_event(geom, pt, ch, ph, et, zv, spec.sigma_y, spec.sigma_z,
                                 spec.noise_frac, rng, track_id_base=track_id_base)


def concat_batches(batches: Sequence[ClusterBatch]) -> ClusterBatch:
    """Stack events into one multi-event batch (task = event*n_sectors + sector)."""
    g = batches[0].geometry
    offs = [np.zeros(1, np.uint32)]
    base = 0
    for b in batches:
        offs.append((b.row_offsets[1:].astype(np.uint64) + base).astype(np.uint32))
        base += b.n_clusters
    cat = lambda n: np.concatenate([getattr(b, n) for b in batches])  # noqa: E731
    return ClusterBatch(
        geometry=g, n_tasks=sum(b.n_tasks for b in batches),
        x=cat("x"), y=cat("y"), z=cat("z"), charge=cat("charge"),
        row_offsets=np.concatenate(offs), sigma_y=batches[0].sigma_y,
        sigma_z=batches[0].sigma_z, truth_track=cat("truth_track"),
        truth_leg=cat("truth_leg"), truth_state=cat("truth_state"), tracks={})


def take_tasks(batch: ClusterBatch, tasks: Sequence[int]):
    """Same task layout, but only the clusters of ``tasks`` (others become empty).

    Tasks are independent, so a tracker run on the result must
    reproduce, task by task, what it finds in the full batch.  Returns
    ``(sub_batch, sel)`` with ``sel[i]`` = index in ``batch`` of sub-cluster i.
    """
    nr = batch.geometry.n_rows
    keep = np.zeros(batch.n_tasks, bool)
    keep[np.asarray(list(tasks), np.int64)] = True
    counts = np.diff(batch.row_offsets.astype(np.int64))
    counts = counts * np.repeat(keep, nr)
    offs = np.zeros(batch.n_tasks * nr + 1, np.uint32)
    offs[1:] = np.cumsum(counts)
    task_of = np.repeat(np.arange(batch.n_tasks), np.add.reduceat(
        np.diff(batch.row_offsets.astype(np.int64)), np.arange(0, batch.n_tasks * nr, nr)))
    sel = np.nonzero(keep[task_of])[0]
    sub = dataclasses.replace(
        batch, x=batch.x[sel], y=batch.y[sel], z=batch.z[sel],
        charge=batch.charge[sel], row_offsets=offs,
        truth_track=batch.truth_track[sel], truth_leg=batch.truth_leg[sel],
        truth_state=batch.truth_state[sel])
    return sub, sel


# --------------------------------------------------------------------------
# BASELINE.json configs
# --------------------------------------------------------------------------
CONFIGS: Dict[int, dict] = {
    0: dict(name="config0_single_sector", n_sectors=1, seeds=[1],
            spec=EventSpec(n_primaries=200, pt_range=(0.2, 5.0), noise_frac=0.01,
                           phi_in_first_sector=True)),
    1: dict(name="config1_peripheral", n_sectors=36, seeds=[2],
            spec=EventSpec(n_primaries=1000, pt_range=(0.2, 5.0), noise_frac=0.02)),
    2: dict(name="config2_central", n_sectors=36, seeds=[100],
            spec=EventSpec(n_primaries=15000, pt_range=(0.1, 10.0), n_loopers=1500,
                           noise_frac=0.05)),
    3: dict(name="config3_batch16_central", n_sectors=36, seeds=list(range(100, 116)),
            spec=EventSpec(n_primaries=15000, pt_range=(0.1, 10.0), n_loopers=1500,
                           noise_frac=0.05)),
    4: dict(name="config4_stress", n_sectors=36, seeds=[4],
            spec=EventSpec(n_primaries=50000, pt_range=(0.1, 10.0), noise_frac=0.20,
                           sigma_y=0.15, sigma_z=0.2, vertex_z_spread=10.0)),
}


def _gen_one(args):
    n_sectors, spec, seed, ev = args
    return generate_event(default_geometry(n_sectors=n_sectors), spec, seed,
                          track_id_base=ev * 1_000_000)


def generate_config(config: int, n_events: Optional[int] = None,
                    workers: int = 1) -> ClusterBatch:
    """The clusters of BASELINE.json ``configs[config]`` (optionally its first events)."""
    c = CONFIGS[config]
    seeds: List[int] = c["seeds"] if n_events is None else c["seeds"][:n_events]
    jobs = [(c["n_sectors"], c["spec"], s, i) for i, s in enumerate(seeds)]
    if workers > 1 and len(jobs) > 1:
        import multiprocessing as mp
        with mp.get_context("fork").Pool(min(workers, len(jobs))) as pool:
            evs = pool.map(_gen_one, jobs)
    else:
        evs = [_gen_one(j) for j in jobs]
    return evs[0] if len(evs) == 1 else concat_batches(evs)
