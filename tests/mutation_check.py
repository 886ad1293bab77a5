"""Mutation check of the oracle pins (test infrastructure; not collected by pytest).

    python tests/mutation_check.py [--write]        # about 10 minutes on 8 cores

Copies oracle/, tests/ and tpc_workload/ to a scratch directory, injects ONE plausible mistake at a time into the
copy of oracle/tpc_oracle.cpp (a textual replacement that must match exactly once), rebuilds it and runs the CPU pin
suites (tests/test_oracle_units.py, test_oracle_tracker.py, test_oracle_following.py).  A mutant is KILLED when at
least one test fails.  --write stores the table as tests/mutants.md.  The repo's own oracle is never touched.
"""
from __future__ import annotations

import argparse
import os
import shutil
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SUITES = ["tests/test_oracle_units.py", "tests/test_oracle_tracker.py", "tests/test_oracle_following.py",
          "tests/test_oracle_merge.py", "tests/test_oracle_its.py"]

# (name, SPEC tag, text in oracle/tpc_oracle.cpp, replacement)
MUTANTS = [
    ("search metric weights swapped", "H5",
     "const R d = (dy2 * ez) + (dz2 * ey);", "const R d = (dy2 * ey) + (dz2 * ez);"),
    ("search metric plain Euclid", "H5",
     "const R d = (dy2 * ez) + (dz2 * ey);", "const R d = dy2 + dz2;"),
    ("search tie goes to the larger gid", "H6",
     "(d == best && c < bg)", "(d == best && c > bg)"),
    ("search tie: first visited wins", "H6",
     "|| (d == best && c < bg)", ""),
    ("y window: cap removed", "H2",
     "const R hy2 = rmin(R(T.prm.accept_k2) * ey, T.smax2);", "const R hy2 = R(T.prm.accept_k2) * ey;"),
    ("z window halved", "H2",
     "const R hz2 = rmin(R(T.prm.accept_k2) * ez, T.smax2);",
     "const R hz2 = R(0.5) * rmin(R(T.prm.accept_k2) * ez, T.smax2);"),
    ("windows: max instead of min", "H2",
     "const R hy2 = rmin(R(T.prm.accept_k2) * ey, T.smax2);", "const R hy2 = rmax(R(T.prm.accept_k2) * ey, T.smax2);"),
    ("y window from ez", "H1/H2",
     "const R hy2 = rmin(R(T.prm.accept_k2) * ey, T.smax2);", "const R hy2 = rmin(R(T.prm.accept_k2) * ez, T.smax2);"),
    ("window test: and -> or", "H4",
     "if (!(dy2 <= hy2 && dz2 <= hz2)) return;", "if (!(dy2 <= hy2 || dz2 <= hz2)) return;"),
    ("window test: strict", "H4",
     "if (!(dy2 <= hy2 && dz2 <= hz2)) return;", "if (!(dy2 < hy2 && dz2 < hz2)) return;"),
    ("up pass stops at gap >= max_row_gap", "K3",
     "else if (++gap > T.prm.max_row_gap) break;", "else if (++gap >= T.prm.max_row_gap) break;"),
    ("up pass never resets the gap", "K3",
     "tk.last_row = r; tk.n_hits++; gap = 0; }", "tk.last_row = r; tk.n_hits++; }"),
    ("up pass: last_row follows the misses", "K3",
     "else if (++gap > T.prm.max_row_gap) break;", "else { tk.last_row = r; if (++gap > T.prm.max_row_gap) break; }"),
    ("down pass counts in-span misses towards the gap", "K5",
     "} else if (r < tk.first_row) {\n          if (++gap", "} else {\n          if (++gap"),
    ("down pass never resets the gap", "K5",
     "if (r < tk.first_row) { tk.first_row = r; gap = 0; }", "if (r < tk.first_row) { tk.first_row = r; }"),
    ("down pass skips the search inside the span", "K5",
     "if (tk.map[r] >= 0) { apply_hit(st, (uint32_t)tk.map[r]); continue; }",
     "if (tk.map[r] >= 0) { apply_hit(st, (uint32_t)tk.map[r]); continue; }\n        if (r > tk.first_row) continue;"),
    ("down pass stops at gap >= max_row_gap", "K5",
     "          if (++gap > T.prm.max_row_gap) break;\n        }", "          if (++gap >= T.prm.max_row_gap) break;\n        }"),
    ("down pass: first_row not updated", "K5",
     "if (r < tk.first_row) { tk.first_row = r; gap = 0; }", "if (r < tk.first_row) { gap = 0; }"),
    ("chain hits beyond a failed transport still taken", "K2",
     "if (!transport(st, T.X[r], T.a, R(T.prm.max_sinphi))) { chain_ok = false; break; }\n        apply_hit",
     "if (!transport(st, T.X[r], T.a, R(T.prm.max_sinphi))) { chain_ok = false; }\n        apply_hit"),
    ("turn-around scales only the diagonal", "K4 / R15",
     "      for (int i = 0; i < 15; ++i) st.c[i] = st.c[i] * R(T.prm.turn_cov_scale);\n",
     "      for (int i : {0, 2, 5, 9, 14}) st.c[i] = st.c[i] * R(T.prm.turn_cov_scale);\n"),
    ("turn-around: lastRow hit not re-fitted", "K4 / D3",
     "if (st.x == T.X[tk.last_row]) apply_hit(st, (uint32_t)tk.map[tk.last_row]);", ""),
    ("turn-around: no transport back to lastRow", "K4",
     "if (st.x != T.X[tk.last_row]) transport(st, T.X[tk.last_row], T.a, R(T.prm.max_sinphi));", ""),
    ("turn-around: chi2 not reset", "K4 / R26",
     "st.chi2 = R(0); st.ndf = -5;\n      // the hit", "st.ndf = -5;\n      // the hit"),
    ("finish: no transport back to firstRow", "K6",
     "if (st.x != T.X[tk.first_row]) transport(st, T.X[tk.first_row], T.a, R(T.prm.max_sinphi));  // K6", ""),
    ("transport fails only on |s1|", "P4 / D2",
     "if (!(rabs(s) <= max_sinphi && rabs(s1) <= max_sinphi)) return false;",
     "if (!(rabs(s1) <= max_sinphi)) return false;"),
    ("ownership tie goes to the larger start gid", "K7 / R16",
     "| (uint64_t)(0xFFFFFFFFu - h0);", "| (uint64_t)h0;"),
    ("ownership: gid before length", "K7 / R16",
     "((uint64_t)tk.n_hits << 32) | (uint64_t)(0xFFFFFFFFu - h0);",
     "((uint64_t)(0xFFFFFFFFu - h0) << 32) | (uint64_t)tk.n_hits;"),
    ("selector keeps hits it does not own", "L1",
     "if (tk.map[r] >= 0 && owner[tk.map[r]] == keys[i]) hits.push_back", "if (tk.map[r] >= 0) hits.push_back"),
    ("selector minimum on tracklet hits only", "L2",
     "if ((int)hits.size() < p->min_track_hits) continue;", ""),
    # the first half of the path (killed since round 1; kept as regression)
    ("neighbour tie-break by larger gid", "N5",
     "(u < bu || (u == bu && d < bd))", "(u > bu || (u == bu && d > bd))"),
    ("neighbour window: z not projected", "N1",
     "const R zu = z * T.ratio_up[r], zd = z * T.ratio_dn[r];", "const R zu = z, zd = z;"),
    ("neighbour chi2: weights swapped", "N4",
     "const R chi = ((dy * dy) * T.wy) + ((dz * dz) * T.wz);", "const R chi = ((dy * dy) * T.wz) + ((dz * dz) * T.wy);"),
    ("cleaner: one-sided links survive", "C1",
     "cu[h] = (up[h] >= 0 && dn[up[h]] == (int32_t)h) ? up[h] : -1;", "cu[h] = up[h];"),
    ("seed length cut off by one", "S3",
     "if (len < T.prm.min_seed_hits) return false;", "if (len <= T.prm.min_seed_hits) return false;"),
    ("seed q/pT variance", "K1",
     "st.c[14] = R(T.prm.c0_qpt);", "st.c[14] = R(1);"),
    ("arc length unsigned", "P9",
     "const R dl = dx * rsqrt_(R(1) + tt * tt);", "const R dl = rabs(dx) * rsqrt_(R(1) + tt * tt);"),
    ("f04 denominator", "P16",
     "const R f04 = ((a * dx) * g) / (c1 * cs);", "const R f04 = ((a * dx) * g) / (c * cs);"),
    ("P24 term dropped", "P24",
     "n[2] = m11 + f12 * m12 + f13 * m13 + f14 * m14;", "n[2] = m11 + f12 * m12 + f13 * m13;"),
    ("update gain sign", "U5",
     "st.p[j] = st.p[j] + k[j] * res;", "st.p[j] = st.p[j] - k[j] * res;"),
    # ---- SPEC 9: merger and refit ----
    ("rotation: y' with the wrong sign of sa", "R4",
     "st.p[0] = y * ca - x * sa;", "st.p[0] = y * ca + x * sa;"),
    ("rotation: sin(phi) turned the other way", "R2",
     "const R s1 = s * ca - c * sa;                                // R2", "const R s1 = s * ca + c * sa;"),
    ("rotation: x' not moved", "R4",
     "st.x = x * ca + y * sa;                                      // R4", "st.x = x * ca;"),
    ("rotation jacobian: point not taken back along the track (j00 = ca)", "R5",
     "const R j00 = ca - (s1 / c1) * sa;                           // R5", "const R j00 = ca;"),
    ("rotation jacobian: j10 dropped", "R5",
     "const R j10 = -((t / c1) * sa);", "const R j10 = R(0);"),
    ("rotation jacobian: j20 dropped", "R5",
     "const R j20 = -((a * q) * sa);", "const R j20 = R(0);"),
    ("rotation jacobian: j22 = ca", "R5",
     "const R j22 = ca + (s / c) * sa;", "const R j22 = ca;"),
    ("rotation covariance: c21' loses m21", "R7",
     "st.c[4] = m20 * j10 + m21;", "st.c[4] = m20 * j10;"),
    ("rotation: angle limit not tested", "R3",
     "if (!(c1 > R(0) && rabs(s1) <= max_sinphi)) return false;    // R3", "if (!(c1 > R(0))) return false;"),
    ("merger: rows may overlap (rl_i <= rf_j)", "G2",
     "if (!(rl[i] < rf[j] && rf[j] <= rl[i] + max_row_gap)) continue;", "if (!(rl[i] <= rf[j] && rf[j] <= rl[i] + max_row_gap)) continue;"),
    ("merger: row gap off by one", "G2",
     "if (!(rl[i] < rf[j] && rf[j] <= rl[i] + max_row_gap)) continue;", "if (!(rl[i] < rf[j] && rf[j] < rl[i] + max_row_gap)) continue;"),
    ("merger: matched at the outer end's x, no transport to the first row of j", "G3",
     "if (q.x != sj_state.x && !transport(q, sj_state.x, T.a, R(p->max_sinphi))) continue;", ""),
    ("merger: chi2 without the q/pT term", "G4",
     "for (int k = 0; k < 5; ++k) {\n        const R dk = q.p[k] - sj_state.p[k];", "for (int k = 0; k < 4; ++k) {\n        const R dk = q.p[k] - sj_state.p[k];"),
    ("merger: chi2 cut not applied", "G4",
     "if (!(chi < R(chi2_max))) continue;", ""),
    ("merger: tie goes to the larger first hit", "G5",
     "(chi == chi_in[j] && gid_first[i] < gid_first[best_in[j]])", "(chi == chi_in[j] && gid_first[i] > gid_first[best_in[j]])"),
    ("merger: links need not be mutual", "G6",
     "if (j >= 0 && best_in[j] == (int32_t)i) {", "if (j >= 0) {"),
    ("refit: covariance not inflated", "F1",
     "for (int i = 0; i < 15; ++i) st.c[i] = st.c[i] * R(T.prm.turn_cov_scale);                       // F1", ""),
    ("refit: no rotation at the sector change", "F2",
     "if (d == 0 || !rotate(st, d, MT.ca, MT.sa, T.a, R(T.prm.max_sinphi))) break;\n      sector = h.sector;", "sector = h.sector;"),
    # ---- SPEC 12: ITS standalone tracker ----
    ("ITS tracklet: opposite side accepted", "V3",
     "if (!(cd > R(0) && rabs(sd) <= R(p->max_sinphi_pair) && rabs(tb - ta) <= R(p->max_dtan))) continue;  // V3",
     "if (!(rabs(sd) <= R(p->max_sinphi_pair) && rabs(tb - ta) <= R(p->max_dtan))) continue;"),
    ("ITS tracklet: angle window strict", "V3",
     "rabs(sd) <= R(p->max_sinphi_pair)", "rabs(sd) < R(p->max_sinphi_pair) * R(0.99)"),
    ("ITS tracklet: tie goes to the larger gid", "V5",
     "(m == m0[B - a1] && A < (uint32_t)b0B)", "(m == m0[B - a1] && A > (uint32_t)b0B)"),
    ("ITS tracklet: not mutual", "V5",
     "if (Bq < 0 || best0[(uint32_t)Bq - a1] != (int64_t)A) continue;", "if (Bq < 0) continue;"),
    ("ITS seed: curvature sign", "W2",
     "const R kap = -((R(2) * (ya * xb)) / ((ra * rb) * dab));", "const R kap = ((R(2) * (ya * xb)) / ((ra * rb) * dab));"),
    ("ITS seed: local y with the wrong sign", "W1",
     "auto loc_y = [&](uint32_t P) { return (Y[P] - vy) * ca - (X[P] - vx) * sa; };",
     "auto loc_y = [&](uint32_t P) { return (Y[P] - vy) * ca + (X[P] - vx) * sa; };"),
    ("ITS seed: beam axis not moved by the vertex", "W1",
     "const R ox = -(vx * ca + vy * sa), oy = -(vy * ca - vx * sa);", "const R ox = R(0), oy = R(0);"),
    ("ITS outward: one missed layer already drops the track", "O2",
     "if (++miss == 2) alive = false;", "if (++miss == 1) alive = false;"),
    ("ITS outward: misses are never reset", "O2",
     "cl[l] = (int32_t)best; ++n_cl; miss = 0;", "cl[l] = (int32_t)best; ++n_cl;"),
    ("ITS outward: minimum number of clusters off by one", "O3",
     "if (!alive || n_cl < p->min_clusters) continue;", "if (!alive || n_cl <= p->min_clusters) continue;"),
    ("ITS outward: chi2 cut ignored", "O2",
     "if (!(rabs(dx) <= R(p->max_dx) && chi < R(p->chi2_max))) continue;", "if (!(rabs(dx) <= R(p->max_dx))) continue;"),
    ("ITS outward: residual without the slope term", "O2",
     "const R dy = loc_y(P) - (st.p[0] + dx * (st.p[2] / c));", "const R dy = loc_y(P) - st.p[0];"),
    ("ITS inward: covariance not inflated", "N1",
     "for (int i = 0; i < 15; ++i) st.c[i] = st.c[i] * R(p->turn_cov_scale);                              // N1", ""),
    ("ITS inward: no transport to the vertex plane", "N3",
     "if (st.x != R(0)) transport(st, R(0), a, R(p->max_sinphi));                                         // N3", ""),
    ("ITS: material ignored", "O / SCATTER",
     "st.c[5] = st.c[5] + th * (R(1) - st.p[2] * st.p[2]);", ""),
]

# Not a mutant: semantically equivalent to the SPEC text, listed so that nobody tries to kill it again.
EQUIVALENT = [
    ("a chain-fit transport failure continues into the up pass (chain_ok ignored)", "K2 -> K4",
     "the up pass would start with the transport from lastRow to lastRow+1 on the unchanged state - the very call "
     "that just failed - and stop at once: same result for every input"),
    ("refit: starts from the inner-end state of the outermost segment instead of its outer end", "F1",
     "F2 then transports that state to the row of the outermost hit itself: the covariance is multiplied by "
     "turn_cov_scale before the transport instead of after it, which is the same matrix up to rounding"),
]


def run_mutant(idx: int) -> tuple:
    name, tag, old, new = MUTANTS[idx]
    src = open(os.path.join(ROOT, "oracle", "tpc_oracle.cpp")).read()
    if src.count(old) != 1:
        return (name, tag, f"ERROR: pattern matches {src.count(old)} times", "")
    tmp = tempfile.mkdtemp(prefix=f"mut{idx:02d}_")
    try:
        for d in ("oracle", "tests", "tpc_workload"):
            shutil.copytree(os.path.join(ROOT, d), os.path.join(tmp, d),
                            ignore=shutil.ignore_patterns("*.so", "__pycache__", ".pytest_cache"))
        with open(os.path.join(tmp, "oracle", "tpc_oracle.cpp"), "w") as f:
            f.write(src.replace(old, new))
        env = dict(os.environ, PYTHONPATH=tmp, PYTHONDONTWRITEBYTECODE="1")
        b = subprocess.run([sys.executable, "-m", "oracle.build", "--force"], cwd=tmp, env=env, capture_output=True, text=True)
        if b.returncode != 0:
            return (name, tag, "ERROR: mutant does not compile", b.stderr[-300:])
        r = subprocess.run([sys.executable, "-m", "pytest", "-q", "-x", "-p", "no:cacheprovider", *SUITES],
                           cwd=tmp, env=env, capture_output=True, text=True)
        failed = [ln.split(" ")[1] for ln in r.stdout.splitlines() if ln.startswith("FAILED ")]
        if r.returncode == 0:
            return (name, tag, "SURVIVES", "")
        return (name, tag, "killed", failed[0].split("::")[-1] if failed else "?")
    finally:
        shutil.rmtree(tmp, ignore_errors=True)


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--write", action="store_true")
    ap.add_argument("--jobs", type=int, default=max(1, (os.cpu_count() or 2) // 2))
    ap.add_argument("--only", default="", help="run only the mutants whose SPEC tag starts with one of these letters, e.g. RGF")
    args = ap.parse_args()
    todo = [i for i, m in enumerate(MUTANTS) if not args.only or m[1][0] in args.only]
    with ThreadPoolExecutor(args.jobs) as ex:
        rows = list(ex.map(run_mutant, todo))
    lines = ["# Mutants of `oracle/tpc_oracle.cpp` and the CPU pin that kills each",
             "",
             "Written by `python tests/mutation_check.py --write` (one textual mistake at a time in a scratch copy of the",
             "oracle, rebuilt, then `pytest -x` over `" + "`, `".join(s.split("/")[-1] for s in SUITES) + "`).",
             "SPEC tags are those of `docs/ARITH_SPEC.md`.",
             "",
             "| # | mutant | SPEC | result | first failing test |", "|---|---|---|---|---|"]
    for i, (name, tag, res, test) in enumerate(rows):
        lines.append(f"| {i + 1} | {name} | {tag} | {res} | `{test}` |" if test else f"| {i + 1} | {name} | {tag} | {res} | |")
    lines += ["", "Equivalent to the SPEC text (cannot be killed, not a different reading):", ""]
    for name, tag, why in EQUIVALENT:
        lines.append(f"* {name} ({tag}): {why}.")
    n_alive = sum(1 for r in rows if r[2] != "killed")
    lines += ["", f"{len(rows) - n_alive} of {len(rows)} killed."]
    text = "\n".join(lines) + "\n"
    print(text)
    if args.write:
        open(os.path.join(ROOT, "tests", "mutants.md"), "w").write(text)
    return 1 if n_alive else 0


if __name__ == "__main__":
    sys.exit(main())
