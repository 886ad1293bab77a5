"""Workload for compute-sanitizer (SURVEY.md section 4 test tiers, section 5 race detection).

    PYTORCH_NO_CUDA_MEMORY_CACHING=1 compute-sanitizer --tool memcheck|racecheck|initcheck|synccheck \
        python tests/sanitize_run.py [small|host]

Runs the CUDA path through the C ABI binding without any comparison (parity is tests/test_gpu_parity.py's job):
`small` = configs 0 and 1 with every debug output, the hand-built ragged rows with ties, empty input and empty
tasks, a capacity overflow; `host` = tpc_track_batch_host on one central event (the chunked, three-stream path).
PYTORCH_NO_CUDA_MEMORY_CACHING=1 makes every torch tensor its own cudaMalloc, so that an out-of-bounds access
of a workspace or output array is seen by memcheck instead of landing in a neighbouring cached block.
"""
from __future__ import annotations

import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def small():
    import gpu_helpers as G
    from helpers import batch_from_rows
    from tpc_workload import generate_config, default_geometry
    for cfg in (0, 1):
        b = generate_config(cfg)
        g = G.run_gpu(b, counters=True)
        print(f"config {cfg}: {b.n_clusters} clusters -> {g['n_tracks']} tracks, status {g['status']}", flush=True)
        assert g["status"] == 0 and g["n_tracks"] > 0
    geom = default_geometry(n_sectors=1, n_rows=12)
    pts = {}
    for r in range(12):
        x = float(geom.row_x[r])
        row = [(0.01 * x, 0.5 * x), (-0.02 * x, 0.2 * x)]
        if r % 2 == 0:
            row.append((0.01 * x, 0.5 * x))
        if r >= 3:
            row.append((5.0 + 0.03 * x, 0.9 * x))
        pts[(0, r)] = row
    g = G.run_gpu(batch_from_rows(geom, pts, n_tasks=1))
    print(f"hand-built rows: {g['n_tracks']} tracks", flush=True)
    g = G.run_gpu(batch_from_rows(default_geometry(n_sectors=2), {}, n_tasks=2))
    assert g["n_tracks"] == 0
    b = generate_config(0)
    for kw in (dict(max_tracklets=16), dict(track_capacity=8), dict(hit_capacity=100)):
        g = G.run_gpu(b, debug=False, debug_tracklets=False, **kw)
        assert g["status"] != 0
    print("empty input and overflow cases done", flush=True)


def host():
    import torch
    import gpu_helpers as G
    from paper_1712_09434_b200 import Tracker
    from tpc_workload import generate_config
    b = generate_config(2)
    dev = torch.device("cuda:0")
    trk = Tracker(b.geometry, G.tracker_params_for(b))
    n = b.n_clusters
    y = torch.from_numpy(np.ascontiguousarray(b.y)).pin_memory()
    z = torch.from_numpy(np.ascontiguousarray(b.z)).pin_memory()
    ro = torch.from_numpy(b.row_offsets.astype(np.uint32).view(np.int32)).pin_memory()
    out = trk.alloc_outputs(n, dev, pinned_host=True)
    ws = trk.alloc_workspace(trk.host_workspace_bytes(n, b.n_tasks, 0, out.track_task.shape[0],
                                                      out.hit_cluster.shape[0]), dev)
    for _ in range(2):
        up, down = trk.track_batch_host(y, z, ro, b.n_tasks, out, ws)
    print(f"host path: {n} clusters, h2d {up} d2h {down}, header {out.header.tolist()}", flush=True)
    assert int(out.header[2]) == 0
    trk.close()


if __name__ == "__main__":
    which = sys.argv[1] if len(sys.argv) > 1 else "small"
    {"small": small, "host": host}[which]()
    print("sanitize_run done", flush=True)
