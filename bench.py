"""bench.py - throughput of the TPC sector tracker hot path (a1..a7) on synthetic Pb-Pb-shaped batches.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C] [--events E]

A step is one pass of the whole hot path (one tpc_track_batch call: grid build, neighbour finder, cleaner,
start hits, tracklet constructor, selector + output) over one batch.  Default workload: BASELINE.json
configs[3], 16 central-Pb-Pb-like events = 576 sector tasks, about 40.7 M clusters, per GPU (weak scaling:
every rank tracks its own 16 events, no data-path collective - DESIGN.md section 8).
Prints ONE JSON line (rank 0).  DESIGN.md section 6 states the algorithmic-bytes formula used for `roofline`.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "tpc_clusters_tracked_per_s"
UNIT = "clusters/s"
FALLBACK_HBM_GBS = 6650.0  # B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent
# ncu figures of the dominant kernel (DRAM bytes, thread instructions per launch) are NOT constants of this file:
# bench_profile.py writes them from an `ncu --set full` capture into profiles/r02_ncu_kernels.json together with a
# hash of the CUDA sources they were measured on; they are reported only while that hash is the built sources' hash.
NCU_SUMMARY = os.path.join(ROOT, "profiles", "r02_ncu_kernels.json")
ALU_PEAK_THREAD_INST_PER_S = 148 * 4 * 32 * 1.965e9  # SMs x schedulers x lanes x SM clock


def load_ncu_summary(workload):
    """{stage name: {"dram_bytes", "thread_inst", ...}} from the committed ncu summary, or {} when it is absent,
    was taken on another workload, or the CUDA sources have changed since (stale numbers are not reported)."""
    from bench_profile import source_hash
    try:
        d = json.load(open(NCU_SUMMARY))
    except (OSError, ValueError):
        return {}, "no ncu summary"
    if d.get("workload") != workload:
        return {}, f"ncu summary is for {d.get('workload')}"
    if d.get("source_hash") != source_hash():
        return {}, "ncu summary is older than the CUDA sources (hash differs)"
    return d.get("kernels", {}), os.path.relpath(NCU_SUMMARY, ROOT)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (default 3: the batch)")
    ap.add_argument("--events", type=int, default=None, help="use only the first E events of the config")
    ap.add_argument("--cpu-events", type=int, default=4, help="events in the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-merge", action="store_true", help="skip the merger + refit leg (SURVEY 8(f)1)")
    ap.add_argument("--no-transform", action="store_true", help="skip the cluster transformation leg (SURVEY 8(f)3)")
    ap.add_argument("--no-its", action="store_true", help="skip the ITS standalone tracker leg (SURVEY 8(f)4)")
    ap.add_argument("--cpu-workers", type=int, default=0, help="worker processes of the all-cores cpu_baseline leg (0 = all)")
    ap.add_argument("--dry-run", action="store_true",
                    help="control flow only (rendezvous, barriers, MAX-reduce, counter gather) on the gloo backend with "
                         "no CUDA call and no tracking; prints a line marked dry_run with value null (used by the CPU tests)")
    return ap.parse_args()


def workload_name(config, n_events):
    from tpc_workload.events import CONFIGS
    return f"{CONFIGS[config]['name']}[{n_events} events]"


def make_workload(config, n_events, rank):
    """Seeded synthetic batch of this rank: the config's seeds shifted by 1000*rank (rank 0 = the config itself)."""
    from tpc_workload.events import CONFIGS, generate_event, default_geometry, concat_batches
    c = CONFIGS[config]
    seeds = [s + 1000 * rank for s in (c["seeds"] if n_events is None else c["seeds"][:n_events])]
    jobs = [(c["n_sectors"], c["spec"], s, i) for i, s in enumerate(seeds)]
    workers = max(1, min(len(jobs), (os.cpu_count() or 1) // max(int(os.environ.get("WORLD_SIZE", "1")), 1), 16))
    if workers > 1:
        import multiprocessing as mp
        from tpc_workload.events import _gen_one
        with mp.get_context("fork").Pool(workers) as pool:
            evs = pool.map(_gen_one, jobs)
    else:
        evs = [generate_event(default_geometry(n_sectors=j[0]), j[1], j[2], track_id_base=j[3] * 1_000_000) for j in jobs]
    return evs[0] if len(evs) == 1 else concat_batches(evs)


# ---------------------------------------------------------------------------------------------
# algorithmic bytes (SURVEY.md section 8(d) / DESIGN.md section 6), from the device counters
# ---------------------------------------------------------------------------------------------
def algorithmic_bytes(c):
    """SURVEY.md section 8(d) / DESIGN.md section 6.  The tracklet constructor (a5) runs as four kernels; its
    formula is split by what each kernel must move (chain: link + (y,z) per chain hit; up pass: bin bounds and
    candidates of its searches; refit: (y,z) of the hits re-read; the last kernel: the rest - its searches, the
    map, the ownership words, the record), so the four parts add up to the a5 formula exactly."""
    N, B, T0, T = c["clusters"], c["bins"], c["start_hits"], c["tracklets_built"]
    Hc, S, K, Ht = c["chain_hits"], c["searches"], c["candidates"], c["tracklet_hits"]
    Ho, To = c["out_hits"], c["out_tracks"]
    a5 = 12 * Hc + 16 * S + 8 * K + 8 * Ht + 4 * Ht + 8 * Ht + 8 * N + 88 * T
    chain = 12 * Hc
    up = 16 * c["searches_up"] + 8 * c["candidates_up"]
    refit = 8 * min(c["refit_steps"], Ht)
    return {
        "grid_build": 8 * N + 8 * N + 4 * N + 4 * B,
        "neighbour_finder": 8 * N + 4 * B + 8 * N,
        "cleaner": 8 * N,
        "start_hits": 4 * T0,
        "tracklet_chain_fit": chain,
        "tracklet_up_pass": up,
        "tracklet_refit": refit,
        # K7 (ownership words, 8 B per hit and 8 B per cluster) is its own kernel now; it takes the selector's
        # map and ownership reads (12 B per hit) along
        "tracklet_down_finish": a5 - chain - up - refit - 8 * Ht - 8 * N,
        "ownership": 8 * Ht + 8 * N + 4 * Ht + 8 * Ht,
        "selector_output": 4 * Ho + 100 * To,
    }


class ClockSampler:
    """nvidia-smi clocks/throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "20", "-i", str(gpu_index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [ln.split(",") for ln in open(self.f.name).read().splitlines() if ln.count(",") >= 8]
        os.unlink(self.f.name)
        sm, mx, pw, reasons = [], [], [], set()
        for r in rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); pw.append(float(r[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                if v.strip().lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------
# the oracle, timed as it stands (cpu_baseline leg and --impl reference): the ONLY use of oracle/ here
# ---------------------------------------------------------------------------------------------
def time_oracle(batch, events):
    """Single-threaded CPU oracle over the given events of ``batch``; returns (seconds, clusters)."""
    import oracle
    from tpc_workload import take_tasks
    ns = batch.geometry.n_sectors
    tasks = [e * ns + s for e in events for s in range(ns)]
    sub, _ = take_tasks(batch, tasks)
    prm = oracle.OracleParams(sigma_y=batch.sigma_y, sigma_z=batch.sigma_z)
    t0 = time.perf_counter()
    oracle.track(sub.geometry, sub.y, sub.z, sub.row_offsets, sub.n_tasks, params=prm)
    return time.perf_counter() - t0, sub.n_clusters


def _oracle_one_task(task):
    import oracle
    from tpc_workload import take_tasks
    b = _POOL_BATCH
    sub, _ = take_tasks(b, [task])
    oracle.track(sub.geometry, sub.y, sub.z, sub.row_offsets, sub.n_tasks,
                 params=oracle.OracleParams(sigma_y=b.sigma_y, sigma_z=b.sigma_z))
    return sub.n_clusters


_POOL_BATCH = None


def time_oracle_all_cores(batch, workers=0):
    """The oracle as it stands over every (event, sector) task of ``batch``, one task per worker process at a time
    (tasks are independent; the oracle itself stays single-threaded).  Returns (s, clusters, workers)."""
    global _POOL_BATCH
    import multiprocessing as mp
    import oracle  # noqa: F401  (builds the library before the fork)
    oracle.oracle._load()
    cores = len(os.sched_getaffinity(0))
    workers = workers or cores
    _POOL_BATCH = batch
    with mp.get_context("fork").Pool(workers) as pool:
        pool.map(_oracle_one_task, range(min(workers, batch.n_tasks)), chunksize=1)  # warm the workers
        t0 = time.perf_counter()
        done = pool.map(_oracle_one_task, range(batch.n_tasks), chunksize=1)
        s = time.perf_counter() - t0
    _POOL_BATCH = None
    return s, int(sum(done)), workers


def cpu_model():
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def run_reference(args):
    """--impl reference: the oracle on the host cores; one step = one event (36 sector tasks) of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from tpc_workload.events import CONFIGS
    n_cfg = len(CONFIGS[args.config]["seeds"]) if args.events is None else args.events
    n_gen = min(n_cfg, 4)
    batch = make_workload(args.config, n_gen, 0)
    for i in range(args.warmup):
        time_oracle(batch, [i % n_gen])
    tot_s, tot_c = 0.0, 0
    for i in range(args.steps):
        s, c = time_oracle(batch, [i % n_gen])
        tot_s += s
        tot_c += c
    value = tot_c / tot_s
    sample = f"one event (36 sector tasks) of the workload per step, events 0..{n_gen - 1} in turn"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(args.config, n_cfg), "step_sample": sample},
        "events_per_s": args.steps / tot_s,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------
# the product arm
# ---------------------------------------------------------------------------------------------
def reduce_over_ranks(ms_pair, counts, dev):
    """The ONLY exchanges of the N > 1 path (reporting, not data): MAX over ranks of the timed durations and the
    sum of (clusters, events, tracks, hits).  dev = a CUDA device under nccl, None under gloo."""
    import torch
    import torch.distributed as dist
    from paper_1712_09434_b200.sharding import gather_counts
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor(list(ms_pair), dtype=torch.float64, device=dev if dev is not None else "cpu")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_pair = [float(v) for v in t.cpu()]
    return ms_pair, gather_counts(counts)


def run_dry(args, rank, world):
    """--dry-run: the control flow of run_ours (rendezvous, barriers, MAX-reduce, counter gather, rank-0 print)
    on gloo, with no CUDA call and NO tracking.  The line carries "dry_run": true and "value": null."""
    import torch.distributed as dist
    if world > 1:
        dist.init_process_group("gloo")
        dist.barrier()
    fake_ms, fake_counts = [10.0 + rank, 20.0 + rank], [1000 * (rank + 1), 1, 10 * (rank + 1), 100 * (rank + 1)]
    if world > 1:
        dist.barrier()
    ms, tot = reduce_over_ranks(fake_ms, fake_counts, None)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"dry_run": True, "metric": METRIC, "value": None, "unit": UNIT, "n_gpus": world,
                          "max_ms_over_ranks": ms, "summed_counts": tot}))
    return 0


def run_ours(args):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise RuntimeError(f"--gpus {args.gpus} but WORLD_SIZE={world}: launch with one rank per GPU")
    if args.dry_run:
        return run_dry(args, rank, world)
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the tracker has no CPU path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    from paper_1712_09434_b200 import Tracker, TrackerParams
    from paper_1712_09434_b200.build import build as build_cuda
    from tpc_workload.events import CONFIGS
    if rank == 0:
        build_cuda()
    if world > 1:
        dist.barrier()
    n_cfg = len(CONFIGS[args.config]["seeds"]) if args.events is None else args.events
    batch = make_workload(args.config, args.events, rank)
    n, n_tasks, nr = batch.n_clusters, batch.n_tasks, batch.geometry.n_rows
    n_events = batch.n_events

    trk = Tracker(batch.geometry, TrackerParams(sigma_y=batch.sigma_y, sigma_z=batch.sigma_z))
    y_h = torch.from_numpy(np.ascontiguousarray(batch.y)).pin_memory()
    z_h = torch.from_numpy(np.ascontiguousarray(batch.z)).pin_memory()
    ro_h = torch.from_numpy(batch.row_offsets.astype(np.uint32).view(np.int32)).pin_memory()
    y, z, ro = y_h.to(dev), z_h.to(dev), ro_h.to(dev)
    out = trk.alloc_outputs(n, dev)
    ws = trk.alloc_workspace(trk.workspace_bytes(n, n_tasks), dev)
    stream = torch.cuda.current_stream(dev)

    # one untimed counted pass: the counters of the algorithmic-bytes formula, and the result sizes
    trk.enable_counters(True)
    trk.track_batch(y, z, ro, n_tasks, out, ws)
    counters = trk.read_counters(stream)
    trk.enable_counters(False)
    hdr = out.header.cpu().numpy().astype(np.int64)
    if int(hdr[2]) != 0:
        raise RuntimeError(f"tracker status bits {int(hdr[2])}: capacity overflow in the bench workload")
    counters["out_tracks"], counters["out_hits"] = int(hdr[0]), int(hdr[1])
    alg = algorithmic_bytes(counters)

    for _ in range(args.warmup):
        trk.track_batch(y, z, ro, n_tasks, out, ws)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    trk.enable_stage_timing(True)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record(stream)
    for _ in range(args.steps):
        trk.track_batch(y, z, ro, n_tasks, out, ws)
    ev1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms_total = ev0.elapsed_time(ev1)
    stage_ms, stage_calls = trk.read_stage_ms(stream)
    trk.enable_stage_timing(False)
    clocks = sampler.stop() if sampler else None

    # end to end through tpc_track_batch_host: pinned host inputs -> device -> tracks back on the host
    e2e = e2e_pipe = None
    if not args.no_e2e:
        out_h = trk.alloc_outputs(n, dev, pinned_host=True)
        tcap, hcap = out_h.track_task.shape[0], out_h.hit_cluster.shape[0]
        ws_h = trk.alloc_workspace(trk.host_workspace_bytes(n, n_tasks, 0, tcap, hcap), dev)
        for _ in range(min(args.warmup, 2)):
            up, down = trk.track_batch_host(y_h, z_h, ro_h, n_tasks, out_h, ws_h)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            up, down = trk.track_batch_host(y_h, z_h, ro_h, n_tasks, out_h, ws_h)
        e1.record(stream)
        torch.cuda.synchronize()
        e2e_ms = e0.elapsed_time(e1)
        e2e = (e2e_ms, up, down)
        # the same with two batches in flight (tpc_host_submit / tpc_host_collect): every step still uploads its
        # inputs from pinned host memory and downloads its tracks and hits, but under the kernels of its neighbours
        out_h2 = trk.alloc_outputs(n, dev, pinned_host=True)
        ws_h2 = trk.alloc_workspace(trk.host_workspace_bytes(n, n_tasks, 0, tcap, hcap), dev)
        outs_p, wss_p = (out_h, out_h2), (ws_h, ws_h2)

        def run_pipeline(steps):
            trk.host_submit(0, y_h, z_h, ro_h, n_tasks, tcap, hcap, wss_p[0])
            for i in range(1, steps):
                trk.host_submit(i % 2, y_h, z_h, ro_h, n_tasks, tcap, hcap, wss_p[i % 2])
                trk.host_collect((i - 1) % 2, outs_p[(i - 1) % 2])
            return trk.host_collect((steps - 1) % 2, outs_p[(steps - 1) % 2])
        run_pipeline(2)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        t_p0 = time.perf_counter()
        up_p, down_p = run_pipeline(args.steps)
        torch.cuda.synchronize()
        pipe_ms = (time.perf_counter() - t_p0) * 1e3
        assert int(out_h.header[0]) == int(hdr[0]) and int(out_h2.header[1]) == int(hdr[1])
        e2e_pipe = (pipe_ms, up_p, down_p)
        del ws_h2, out_h2
        del ws_h, out_h

    # sector-segment merger + final refit behind a7 (tpc_merge_refit), timed on its own: tracker call +
    # merger call per step, CUDA events around the merger on the launching stream
    merge = None
    if not args.no_merge:
        tcap = int(out.track_task.shape[0])
        mg = trk.alloc_merged(tcap, dev)
        mws = trk.alloc_workspace(trk.merge_workspace_bytes(tcap, n_tasks), dev)
        pairs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                 for _ in range(args.steps)]
        for _ in range(2):
            trk.track_batch(y, z, ro, n_tasks, out, ws)
            trk.merge_refit(y, z, ro, n_tasks, out, mg, ws, mws)
        torch.cuda.synchronize()
        m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        m0.record(stream)
        for a, b in pairs:
            trk.track_batch(y, z, ro, n_tasks, out, ws)
            a.record(stream)
            trk.merge_refit(y, z, ro, n_tasks, out, mg, ws, mws)
            b.record(stream)
        m1.record(stream)
        torch.cuda.synchronize()
        mh = mg.header.cpu().numpy().astype(np.int64)
        merge_ms = sum(a.elapsed_time(b) for a, b in pairs) / args.steps
        # what the merger must move once: the state of every sector track in and its outer end out and in again
        # (3 x 84 B), the kept hits of the refit (4 B map entry + 8 B cluster), the merged record out (104 B)
        merge_bytes = 252 * int(hdr[0]) + 12 * int(hdr[1]) + 104 * int(mh[0])
        merge = {"ms_per_step": merge_ms, "tracker_plus_merger_ms_per_step": m0.elapsed_time(m1) / args.steps,
                 "sector_tracks": int(hdr[0]), "links": int(mh[1]), "merged_tracks": int(mh[0]), "status": int(mh[2]),
                 "algorithmic_bytes": merge_bytes, "achieved_gbs": merge_bytes / (merge_ms / 1e3) / 1e9,
                 "launches": 8, "note": "runs on the tracker's workspace: no track, hit or cluster leaves the device"}
        del mg, mws

    # cluster transformation (pad, time) -> (y, z) in front of a1 (tpc_transform_clusters), timed on its
    # own with CUDA events on the launching stream: 8 B read + 8 B written per cluster, the 6 MB map stays in L2
    xform = None
    if not args.no_transform:
        from paper_1712_09434_b200 import ClusterTransform
        from tpc_workload import default_calibration, raw_from_yz
        raw = default_calibration(batch.geometry, seed=7)
        pad_h, time_h = raw_from_yz(batch.geometry, raw, batch.y, batch.z, batch.row_offsets, n_tasks)
        xf = ClusterTransform(batch.geometry, raw)
        pad_d, time_d = torch.from_numpy(pad_h).to(dev), torch.from_numpy(time_h).to(dev)
        y2, z2 = torch.empty_like(pad_d), torch.empty_like(time_d)
        for _ in range(3):
            xf.transform(pad_d, time_d, ro, n_tasks, y2, z2)
        torch.cuda.synchronize()
        x0, x1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        x0.record(stream)
        for _ in range(args.steps):
            xf.transform(pad_d, time_d, ro, n_tasks, y2, z2)
        x1.record(stream)
        torch.cuda.synchronize()
        x_ms = x0.elapsed_time(x1) / args.steps
        xform = {"ms_per_step": x_ms, "algorithmic_bytes": 16 * n, "achieved_gbs": 16 * n / (x_ms / 1e3) / 1e9,
                 "clusters_per_s": n / (x_ms / 1e3), "launches": 1,
                 "note": "back-to-back launches over 651 MB: the arrays exceed the 126 MB L2"}
        xf.close()
        del pad_d, time_d, y2, z2

    # ITS standalone tracker on 16 synthetic events of 1 500 primaries (about 9 000 clusters per layer
    # and event with 10 % noise), timed on its own with CUDA events on the launching stream
    its = None
    if not args.no_its:
        from paper_1712_09434_b200 import ItsTracker
        from tpc_workload import default_its_geometry, generate_its_events
        ig = default_its_geometry()
        ib = generate_its_events(ig, 16, 1500, seed=3, pt_range=(0.15, 5.0), noise_frac=0.1)
        it = ItsTracker(ig)
        tt = lambda a_: torch.from_numpy(np.ascontiguousarray(a_)).to(dev)  # noqa: E731
        ix, iy, iz = tt(ib.x), tt(ib.y), tt(ib.z)
        ilo, ivt = tt(ib.layer_offsets.astype(np.uint32).view(np.int32)), tt(ib.vertex.astype(np.float32).reshape(-1))
        for _ in range(3):
            io = it.track_batch(ix, iy, iz, ilo, ivt, ib.n_events)
        torch.cuda.synchronize()
        i0, i1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        i0.record(stream)
        for _ in range(args.steps):
            io = it.track_batch(ix, iy, iz, ilo, ivt, ib.n_events)
        i1.record(stream)
        torch.cuda.synchronize()
        ih = io["header"].cpu().numpy()
        i_ms = i0.elapsed_time(i1) / args.steps
        its = {"ms_per_step": i_ms, "events": ib.n_events, "clusters": ib.n_clusters, "tracklets": int(ih[1]),
               "tracks": int(ih[0]), "status": int(ih[2]), "events_per_s": ib.n_events / (i_ms / 1e3), "launches": 4,
               "note": "includes the allocation of outputs and workspace by the binding (torch caching allocator)"}
        it.close()

    # max over ranks, totals over ranks
    (ms_total, e2e_ms_max, e2e_pipe_ms_max), tot = reduce_over_ranks([ms_total, e2e[0] if e2e else 0.0,
                                                                       e2e_pipe[0] if e2e else 0.0],
                                                    [n, n_events, int(hdr[0]), int(hdr[1])], dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        peak_gbs, peak_src = float(json.load(open(peaks_path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    else:
        peak_gbs, peak_src = FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"
    secs = ms_total / 1e3
    ms_step = ms_total / args.steps
    value = tot[0] * args.steps / secs
    top = max(stage_ms, key=stage_ms.get)
    top_gbs = alg[top] / (stage_ms[top] / 1e3) / 1e9 if stage_ms[top] > 0 else 0.0
    path_bytes = sum(alg.values())
    path_gbs = path_bytes / (ms_step / 1e3) / 1e9
    ncu_all, ncu_src = load_ncu_summary(CONFIGS[args.config]["name"] if args.events is None else "partial")
    ncu = ncu_all.get(top)  # None unless the committed capture was taken on exactly these sources and this workload
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": workload_name(args.config, n_cfg), "events_per_gpu": n_events,
                   "sector_tasks_per_gpu": n_tasks, "clusters_per_gpu": n, "tracks_per_gpu": int(hdr[0]),
                   "parallelism": f"events sharded over {world} GPU(s), no collective",
                   "l2": "inputs (8 B/cluster) and every intermediate array are larger than the 126 MB L2"
                         if 8 * n > 126e6 else "inputs smaller than L2: latency case, not the headline"},
        "events_per_s": tot[1] * args.steps / secs,
        "tracks_per_s": tot[2] * args.steps / secs,
        "hbm_roofline_frac_path": path_gbs / peak_gbs,
        "roofline": {"bound": "hbm", "kernel": top, "achieved": top_gbs, "peak": peak_gbs, "unit": "GB/s",
                     "frac": top_gbs / peak_gbs, "traffic": ncu.get("dram_bytes") if ncu else None,
                     "traffic_source": ncu_src, "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": alg[top], "ms_per_launch": stage_ms[top],
                     "traffic_gbs": (ncu["dram_bytes"] / (stage_ms[top] / 1e3) / 1e9) if ncu and "dram_bytes" in ncu else None,
                     "note": "achieved = ALGORITHMIC bytes over the live launch time (the metric's definition); traffic = "
                             "the DRAM bytes ncu saw this kernel move (with the wavefront order of the tracklet queue about the "
                             "algorithmic bytes). The kernel is bound by the latency of the two dependent gathers of a search, "
                             "mostly L2 hits, and by instruction issue (DESIGN.md section 6); \"alu\" shows how far it is from "
                             "the plain-ALU ceiling",
                     "share_of_step": stage_ms[top] / max(sum(stage_ms.values()), 1e-9)},
        "roofline_path": {"bound": "hbm", "achieved": path_gbs, "peak": peak_gbs, "unit": "GB/s",
                          "frac": path_gbs / peak_gbs, "algorithmic_bytes_per_step": path_bytes,
                          "bytes_per_cluster": path_bytes / max(n, 1)},
        # the dominant kernel is bound by plain (non-FMA) ALU issue, not by HBM: thread
        # instructions per launch from the committed ncu capture over the live launch time, against the ALU ceiling
        "alu": ({"bound": "alu", "kernel": top, "achieved": ncu["thread_inst"] / (stage_ms[top] / 1e3) / 1e12,
                 "peak": ALU_PEAK_THREAD_INST_PER_S / 1e12, "unit": "T thread-instructions/s",
                 "frac": ncu["thread_inst"] / (stage_ms[top] / 1e3) / ALU_PEAK_THREAD_INST_PER_S,
                 "thread_inst_per_launch": ncu["thread_inst"], "source": ncu_src}
                if ncu and "thread_inst" in ncu else None),
        "stages_ms": stage_ms, "stages_algorithmic_bytes": alg, "stage_calls_averaged": stage_calls,
        "counters": counters,
        "clocks": clocks,
        "gpu_launches": trk.launches_per_batch() * args.steps,
    }
    if its:
        line["its_standalone"] = its
    if xform:
        xform["hbm_frac"] = xform["achieved_gbs"] / peak_gbs
        line["cluster_transform"] = xform
    if merge:
        merge["hbm_frac"] = merge["achieved_gbs"] / peak_gbs
        line["merge_refit"] = merge
    if e2e:
        # headline end-to-end number: the pipelined entry point (what a caller with a stream of batches uses); every
        # step uploads its own inputs and downloads its own result inside the timed region (wall clock between two
        # device synchronisations: the copies run on the library's own streams).  e2e_sync: one batch at a time.
        line["e2e"] = {"value": tot[0] * args.steps / (e2e_pipe_ms_max / 1e3), "unit": UNIT,
                       "h2d_bytes_per_step": e2e_pipe[1], "d2h_bytes_per_step": e2e_pipe[2],
                       "ms_per_step": e2e_pipe_ms_max / args.steps,
                       "api": "tpc_host_submit / tpc_host_collect (pinned host buffers, two batches in flight)"}
        line["e2e_sync"] = {"value": tot[0] * args.steps / (e2e_ms_max / 1e3), "unit": UNIT,
                            "h2d_bytes_per_step": e2e[1], "d2h_bytes_per_step": e2e[2],
                            "ms_per_step": e2e_ms_max / args.steps,
                            "api": "tpc_track_batch_host (pinned host buffers, one batch at a time, three chunks)"}
    if world == 1 and not args.no_cpu_baseline:
        # the oracle as it stands, (i) over all host cores, one (event, sector) task per worker process at a time, on
        # every event of the workload, (ii) on one thread on the first events
        s_all, c_all, workers = time_oracle_all_cores(batch, args.cpu_workers)
        ne = max(1, min(args.cpu_events, n_events))
        s1, c1 = time_oracle(batch, list(range(ne)))
        line["cpu_baseline"] = {
            "value": c_all / s_all, "unit": UNIT, "cores": workers, "kind": "oracle",
            "sample": f"all {n_events} event(s) of the workload ({c_all} clusters, {n_tasks} sector tasks), one task per "
                      f"worker process, {workers} workers, {s_all:.1f} s",
            "events_per_s": n_events / s_all, "cores_available": len(os.sched_getaffinity(0)), "cpu_model": cpu_model(),
            "single_thread": {"value": c1 / s1, "unit": UNIT, "cores": 1,
                              "sample": f"first {ne} event(s) ({c1} clusters), one thread, {s1:.1f} s"}}
    trk.close()
    if world > 1:
        dist.destroy_process_group()
    print(json.dumps(line))
    return 0


def relaunch_under_torchrun(args):
    """`python bench.py --gpus N` (N > 1) outside a launcher: start N ranks, one per GPU, as the driver would."""
    import socket
    sock = socket.socket()
    sock.bind(("127.0.0.1", 0))
    port = sock.getsockname()[1]
    sock.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    return subprocess.call(cmd)


def main():
    args = parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return relaunch_under_torchrun(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
