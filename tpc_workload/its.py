"""Seeded synthetic ITS events (docs/ARITH_SPEC.md section 12): INPUT only.  Six cylindrical
layers, primary tracks as exact fp64 helices from the event vertex, one cluster per crossed layer smeared along
r-phi and z, uniform noise clusters.  None of the tracker's arithmetic lives here.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict

import numpy as np

C_KAPPA = 0.000299792458


@dataclass
class ItsGeometry:
    R: np.ndarray         # float32 [6] cm
    sig_rphi: np.ndarray  # float32 [6] cm
    sig_z: np.ndarray     # float32 [6] cm
    xx0: np.ndarray       # float32 [6] radiation lengths
    half_z: np.ndarray    # float32 [6] cm (noise only)
    bz_kgauss: float = 5.0


def default_its_geometry(xx0: float = 0.011) -> ItsGeometry:
    """SPD (2 layers), SDD (2), SSD (2): radii and resolutions of the Run-2 ITS."""
    return ItsGeometry(R=np.array([3.9, 7.6, 15.0, 23.9, 38.0, 43.0], np.float32),
                       sig_rphi=np.array([0.0012, 0.0012, 0.0035, 0.0035, 0.0020, 0.0020], np.float32),
                       sig_z=np.array([0.0100, 0.0100, 0.0025, 0.0025, 0.0830, 0.0830], np.float32),
                       xx0=np.full(6, xx0, np.float32),
                       half_z=np.array([14.1, 14.1, 22.2, 29.7, 43.1, 48.9], np.float32))


@dataclass
class ItsBatch:
    geometry: ItsGeometry
    n_events: int
    x: np.ndarray            # float32 [N] global
    y: np.ndarray
    z: np.ndarray
    layer_offsets: np.ndarray  # uint32 [n_events*6 + 1]
    vertex: np.ndarray       # float32 [n_events, 3]
    truth_track: np.ndarray  # int32 [N], -1 noise, unique over the batch
    truth_xyz: np.ndarray    # float64 [N, 3] exact crossing
    tracks: Dict[str, np.ndarray] = field(default_factory=dict)   # per generated track: event, pt, charge, phi0, eta

    @property
    def n_clusters(self) -> int:
        return int(self.x.shape[0])


def _crossings(geom, vtx, pt, charge, phi0, eta):
    """Exact crossing of every helix with every cylinder (Newton on the turning angle); NaN where it curls back."""
    kappa = -C_KAPPA * geom.bz_kgauss * charge / pt
    t = np.sinh(eta)
    n = pt.shape[0]
    out = np.full((n, 6, 3), np.nan)
    for l in range(6):
        R = float(geom.R[l])
        arg = 0.5 * kappa * R
        ok = np.abs(arg) < 0.98
        dpsi = np.where(ok, 2.0 * np.arcsin(np.clip(arg, -0.98, 0.98)), np.nan)   # vertex at the origin
        for _ in range(6):                                                       # correct for the vertex offset
            psi = phi0 + dpsi
            px = vtx[0] + (np.sin(psi) - np.sin(phi0)) / kappa
            py = vtx[1] - (np.cos(psi) - np.cos(phi0)) / kappa
            f = px * px + py * py - R * R
            df = 2.0 * (px * np.cos(psi) + py * np.sin(psi)) / kappa
            dpsi = dpsi - f / df
        psi = phi0 + dpsi
        px = vtx[0] + (np.sin(psi) - np.sin(phi0)) / kappa
        py = vtx[1] - (np.cos(psi) - np.cos(phi0)) / kappa
        s_xy = dpsi / kappa
        pz = vtx[2] + t * s_xy
        good = ok & (s_xy > 0) & (np.abs(pz) <= float(geom.half_z[l]))
        out[good, l, 0], out[good, l, 1], out[good, l, 2] = px[good], py[good], pz[good]
    return out


def generate_its_events(geom: ItsGeometry, n_events: int, n_tracks: int, seed: int, pt_range=(0.2, 5.0), eta_max=0.9,
                        noise_frac: float = 0.05, smear: bool = True, vertex_sigma=(0.01, 0.01, 5.0)) -> ItsBatch:
    rng = np.random.Generator(np.random.PCG64(seed))
    xs, ys, zs, tt, txyz, offs = [], [], [], [], [], [0]
    vtxs = np.zeros((n_events, 3))
    trk = {k: [] for k in ("event", "pt", "charge", "phi0", "eta")}
    base = 0
    for e in range(n_events):
        v = rng.normal(0.0, 1.0, 3) * np.asarray(vertex_sigma)
        vtxs[e] = v
        pt = np.exp(rng.uniform(np.log(pt_range[0]), np.log(pt_range[1]), n_tracks))
        ch = np.where(rng.random(n_tracks) < 0.5, -1.0, 1.0)
        ph = rng.uniform(0.0, 2.0 * np.pi, n_tracks)
        et = rng.uniform(-eta_max, eta_max, n_tracks)
        cr = _crossings(geom, v, pt, ch, ph, et)
        for k, a in (("event", np.full(n_tracks, e)), ("pt", pt), ("charge", ch), ("phi0", ph), ("eta", et)):
            trk[k].append(a)
        for l in range(6):
            hit = ~np.isnan(cr[:, l, 0])
            P = cr[hit, l, :]
            ids = np.nonzero(hit)[0] + base
            X, Y, Zc = P[:, 0].copy(), P[:, 1].copy(), P[:, 2].copy()
            if smear:
                r = np.hypot(X, Y)
                d = rng.normal(0.0, 1.0, len(X)) * float(geom.sig_rphi[l])
                X, Y = X - d * Y / r, Y + d * X / r
                Zc = Zc + rng.normal(0.0, 1.0, len(X)) * float(geom.sig_z[l])
            n_noise = int(rng.poisson(noise_frac * len(X))) if noise_frac > 0 else 0
            phn = rng.uniform(0, 2 * np.pi, n_noise)
            X = np.concatenate([X, float(geom.R[l]) * np.cos(phn)])
            Y = np.concatenate([Y, float(geom.R[l]) * np.sin(phn)])
            Zc = np.concatenate([Zc, rng.uniform(-1, 1, n_noise) * float(geom.half_z[l])])
            ids = np.concatenate([ids, np.full(n_noise, -1)])
            exact = np.concatenate([P, np.full((n_noise, 3), np.nan)])
            perm = rng.permutation(len(X))
            xs.append(X[perm]); ys.append(Y[perm]); zs.append(Zc[perm]); tt.append(ids[perm]); txyz.append(exact[perm])
            offs.append(offs[-1] + len(X))
        base += n_tracks
    cat = np.concatenate
    return ItsBatch(geometry=geom, n_events=n_events, x=cat(xs).astype(np.float32), y=cat(ys).astype(np.float32),
                    z=cat(zs).astype(np.float32), layer_offsets=np.array(offs, np.uint32), vertex=vtxs.astype(np.float32),
                    truth_track=cat(tt).astype(np.int32), truth_xyz=cat(txyz),
                    tracks={k: cat(v) for k, v in trk.items()})
