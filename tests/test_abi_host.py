"""CPU-side checks of the boundary (no compute calls): the C-ABI library loads and exports every
symbol include/tpc_tracker.h declares, argument validation works, the product path has no CPU
fallback and never touches ``oracle/``, and the N > 1 sharding logic (gloo, world_size 2)."""
from __future__ import annotations

import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _has_cuda():
    import torch
    return torch.cuda.is_available()


def test_library_exports_every_declared_symbol():
    from paper_1712_09434_b200 import exported_symbols, load_library
    from paper_1712_09434_b200.build import build
    build()
    names = exported_symbols()
    assert {"tpc_tracker_create", "tpc_tracker_destroy", "tpc_workspace_bytes", "tpc_track_batch",
            "tpc_track_batch_host", "tpc_last_error", "tpc_default_params"} <= set(names)
    lib = load_library()
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in include/tpc_tracker.h but not exported"


def test_default_params_match_spec_section_8():
    from paper_1712_09434_b200 import load_library
    from paper_1712_09434_b200.binding import _Params
    p = _Params()
    load_library().tpc_default_params(C.byref(p))
    want = dict(sigma_y=0.1, sigma_z=0.15, nf_hy=2.0, nf_hz=1.5, nf_chi2_max=75.0, grid_bin_min=2.0,
                grid_bin_max=20.0, max_sinphi=0.95, c0_sinphi=1.0, c0_dzds=1.0, c0_qpt=100.0, accept_k2=16.0,
                search_max=3.0, turn_cov_scale=100.0, min_seed_hits=5, max_row_gap=4, min_track_hits=10)
    for k, v in want.items():
        assert getattr(p, k) == (np.float32(v) if isinstance(v, float) else v), k


def test_create_rejects_bad_geometry_and_reports_text():
    from paper_1712_09434_b200 import load_library
    from paper_1712_09434_b200.binding import _Geometry
    lib = load_library()
    h = C.c_void_p()
    row_x = (C.c_float * 3)(3.0, 2.0, 1.0)  # not increasing
    g = _Geometry(1, 3, row_x, 0.17, 250.0)
    assert lib.tpc_tracker_create(C.byref(g), 5.0, None, C.byref(h)) == -1
    assert b"increasing" in lib.tpc_last_error(None)
    assert not h.value
    assert lib.tpc_tracker_create(None, 5.0, None, C.byref(h)) == -1


@pytest.mark.skipif(_has_cuda(), reason="only meaningful without a device")
def test_no_cpu_fallback_without_a_device():
    """Without a CUDA device tpc_tracker_create fails with TPC_ERR_CUDA: there is no CPU path."""
    from paper_1712_09434_b200 import Tracker, TpcError
    from tpc_workload import default_geometry
    with pytest.raises(TpcError, match=r"\(-3\)"):
        Tracker(default_geometry(n_sectors=1))


def test_product_never_imports_the_oracle():
    """The package and bench.py's product arm may not import, link or run anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1712_09434_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), f
                assert "tpc_oracle" not in text, f
                assert not re.search(r"\b_work[/\\.]", text), f
    code = ("import sys; sys.path.insert(0, %r); import paper_1712_09434_b200; "
            "assert not any(m == 'oracle' or m.startswith('oracle.') for m in sys.modules), 'oracle imported'" % ROOT)
    subprocess.run([sys.executable, "-c", code], check=True)


def test_shard_events_partitions_exactly():
    from paper_1712_09434_b200 import shard_events
    for n in (0, 1, 7, 16, 17):
        for w in (1, 2, 3, 8):
            got = [e for r in range(w) for e in shard_events(n, w, r)]
            assert got == list(range(n))
            sizes = [len(shard_events(n, w, r)) for r in range(w)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_events(4, 2, 2)


_GLOO_WORKER = r"""
import os, sys
sys.path.insert(0, %(root)r)
import numpy as np, torch, torch.distributed as dist
from paper_1712_09434_b200.sharding import shard_events, gather_counts
from tpc_workload import generate_config
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%(port)d", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
mine = shard_events(3, 2, rank)
# every rank generates ONLY its events of the 3-event peripheral batch (seeds are per event)
from tpc_workload.events import CONFIGS, generate_event, default_geometry
spec = CONFIGS[1]["spec"]
n = sum(generate_event(default_geometry(), spec, 200 + e).n_clusters for e in mine)
tot = gather_counts([n, len(mine), 0, 0])
full = sum(generate_event(default_geometry(), spec, 200 + e).n_clusters for e in range(3))
assert tot[0] == full and tot[1] == 3, (tot, full)
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_sharding_world_size_2_gloo(tmp_path):
    """The N > 1 path of bench.py: events sharded by rank, no data-path collective, one gather of counters."""
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    script = tmp_path / "w.py"
    script.write_text(_GLOO_WORKER % dict(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT)
             for r in range(2)]
    outs = [p.communicate(timeout=240)[0].decode() for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o
        assert "ok" in o


def test_bench_gpus_2_launches_two_ranks_dry_run():
    """`python bench.py --gpus 2` starts two ranks by itself (torch.distributed.run, 127.0.0.1) and its control flow -
    rendezvous, barriers, MAX-reduce of the durations, gather of the counters, rank-0 print - runs on gloo with
    --dry-run (no CUDA call, no tracking: the line says dry_run and carries no value)."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-run"], env=env,
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout  # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["dry_run"] is True and d["value"] is None and d["n_gpus"] == 2
    assert d["max_ms_over_ranks"] == [11.0, 21.0]          # max over ranks of (10 + rank, 20 + rank)
    assert d["summed_counts"] == [3000, 2, 30, 300]        # sums over ranks
    # a rank count that contradicts --gpus is refused, not silently reported
    env2 = dict(env, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "4", "--dry-run"], env=env2,
                       capture_output=True, text=True, timeout=120)
    assert r.returncode != 0 and "WORLD_SIZE" in r.stderr


def test_ncu_summary_is_tied_to_the_source_hash(tmp_path, monkeypatch):
    """bench.py reports ncu figures only while the CUDA sources still hash to what the capture was taken on."""
    import json
    import bench
    import bench_profile
    f = tmp_path / "k.json"
    monkeypatch.setattr(bench, "NCU_SUMMARY", str(f))
    assert bench.load_ncu_summary("w")[0] == {}
    f.write_text(json.dumps({"workload": "w", "source_hash": bench_profile.source_hash(),
                             "kernels": {"tracklet_up_pass": {"dram_bytes": 1.0}}}))
    assert bench.load_ncu_summary("w")[0]["tracklet_up_pass"]["dram_bytes"] == 1.0
    assert bench.load_ncu_summary("other")[0] == {}
    f.write_text(json.dumps({"workload": "w", "source_hash": "stale", "kernels": {"tracklet_up_pass": {}}}))
    assert bench.load_ncu_summary("w")[0] == {}
