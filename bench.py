#!/usr/bin/env python
"""bench.py -- one JSON line for the hot path of arXiv 2507.23700 on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C3]

A STEP is one pass of the whole hot path (every row of SURVEY.md §8(a)) over one synthetic
batch, through the C ABI:
    arbx_build(N prims)                      B1..B6
    arbx_query_spatial(Q queries) -> CSR     Q1,Q2,T1,T2,T3
    arbx_query_count(Q queries)              Q1,Q2,T1 (= T4, the count-only callback path)
    arbx_query_knn(Q points, k)              Q1,Q2,K1,K2      (when the workload has a k)
    arbx_destroy
The default workload is BASELINE.json configs[2] ("C3": N = Q = 10^7 3-D fp32 points, hollow
sphere queries, radius with ~16 neighbours, kNN k = 16) -- the configuration BASELINE.json's
metric is quoted on ("... at N=10M fp32 3D").

value       = queries answered per second over the whole step (3 query batches; the build
              is inside the step), inputs resident in HBM, device-timed.
e2e         = the same with pinned-HOST inputs copied to the device and every result copied
              back to pinned host memory inside the timed region, every step; three streams
              and two buffer sets let step i's compute overlap step i+1's copy-in and step
              i-1's copy-out (the per-call stream argument of the ABI).
breakdown   = per-call rates: build Mprims/s, radius/count/kNN queries/s, and per hot-path
              step milliseconds + achieved algorithmic GB/s (arbx_profile_*, CUDA events).
roofline    = the dominant kernel (largest share of the step) against the measured HBM peak.
cpu_baseline= the oracle (oracle/, never tuned) on the host cores, bounded sample.

N > 1 (torchrun): replicas only -- every rank runs the same step on its own data (rank
seeds), no data-path collective; value = all ranks' queries / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "BVH build Mprims/s; radius & kNN(k=16) queries/s at N=10M fp32 3D; HBM GB/s"
UNIT = "queries/s"


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---- algorithmic HBM bytes per hot-path step -------------
def sort_passes(n, D):
    """8-bit digit passes of the build sort: code width adapted to n (csrc/build.cu, reading A15)."""
    lg = max(0, int(n - 1).bit_length())
    bmax = min(32, 64 // D)
    b = min(bmax, (lg + D - 1) // D + 4)
    b = min(bmax, max(b, 8 * ((D * b + 7) // 8) // D))
    return (D * b + 7) // 8


def query_sort_passes(D):
    return (D * min(16, 32 // D) + 7) // 8


def algorithmic_bytes(cfg, totals):
    """COMPULSORY bytes the method itself must move per step, per kernel id of
    arbx_profile_kernel_name: SURVEY.md §8(d)'s per-primitive / per-query figures times the
    units one step processes.  A traversal reads the part of the tree its queries can reach
    ONCE: (leaf record + one child box + 8 bytes of links) per TOUCHED primitive, where
    `touched` = distinct primitives that appear in this workload's results (measured, passed
    in `totals`); `whole_tree` (every leaf and every node slot) is reported beside it."""
    n, nq, D = cfg["n"], cfg["nq"], cfg["dim"]
    pk, qk = cfg["pkind"], cfg["qkind"]
    pw = D if pk == 0 else 2 * D if pk == 1 else D + 1          # floats per primitive row
    qw = D if qk == 0 else 2 * D if qk == 1 else D + 1          # floats per spatial query row
    lw = (pw + 1 + 1) // 2 * 2                                  # floats per leaf record as SURVEY.md counts it
                                                                # (geometry + index, 8-byte granules: 16 / 32 / 24 B for
                                                                # 3-D points / 3-D boxes / 5-D points; ours pads to 16 B)
    npass = sort_passes(n, D)                                   # 8-bit digit passes, build sort
    qpass = query_sort_passes(D)                                # digit passes, query sort
    nbatches = 3 if cfg["k"] else 2                             # query batches per step
    pairs = totals["pairs"]
    per_touched = 4 * lw + 8 * D + 8                            # leaf + child box + links
    tree_sp = per_touched * totals.get("touched_spatial", n)
    tree_knn = per_touched * totals.get("touched_knn", n)
    b = {
        "B1_bounds": 4 * pw * n,
        "B2_codes": 4 * pw * n + 8 * n,
        "B3_sort_hist": 8 * n,
        # pass 0 reads keys only (values are positions), later passes read and write (key,val)
        "B3_sort_pass": (8 + 12) * n + (npass - 1) * 24 * n,
        "B4_leaves": 4 * n + 4 * pw * n + 4 * lw * n,
        # B5: codes 8 + links 8 + parent 4; B6: leaf read + flag RMW 8 + box write + box read by the parent
        "B5B6_hierarchy_refit": n * (20 + 4 * lw + 8 + 16 * D),
        "T2_scan": 4 * nq + 4 * nq + 4 * (nq + 1),
    }
    q1_spatial = 4 * qw * nq + 4 * nq
    q1_knn = 4 * D * nq + 4 * nq
    b["Q1_qcodes"] = 2 * q1_spatial + (q1_knn if cfg["k"] else 0)
    b["Q2_qsort_hist"] = nbatches * 4 * nq
    b["Q2_qsort_pass"] = nbatches * ((4 + 8) * nq + (qpass - 1) * 16 * nq)
    # traversal: order 4 + query row + count 4; the reachable part of the tree once per traversal
    per_count = nq * (4 + 4 * qw + 4) + tree_sp
    # arbx_query_count: one count traversal; arbx_query_spatial: one traversal that also stores
    # the hits in scratch rows (both under the T1 id), then the rows are copied into the CSR
    # slices (T3 id: rows read + indices written + counts and offsets read)
    b["T1_spatial_count"] = per_count + (per_count + 4 * pairs)
    b["T3_spatial_fill"] = 4 * pairs + 4 * pairs + 8 * nq
    if cfg["k"]:
        b["K1K2_knn"] = nq * (4 + 4 * D + 8 * cfg["k"]) + tree_knn
    nw = 4 * (D + 1)
    b["_whole_tree"] = 4 * (n * lw + (n - 1) * nw)
    return b


# kernel id -> substring of the CUDA kernel name in the committed ncu launch list
_NCU_KERNEL = {"K1K2_knn": "knn_", "T1_spatial_count": "spatial_kernel", "T3_spatial_fill": "compact_rows",
               "B5B6_hierarchy_refit": "hierarchy_kernel", "B3_sort_pass": "onesweep_pass<unsigned long long",
               "Q2_qsort_pass": "onesweep_pass<unsigned int"}


def ncu_traffic(kernel_id: str, workload: str, launches_per_step: float = 1.0):
    """dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel id per bracketed launch,
    from the committed ncu launch list of this same workload (profiles/r2_launches_<workload>.csv
    holds the rows of ONE step): the sum over every CUDA kernel of that id (K1K2_knn = packet +
    per-lane kernel) divided by the number of bracketed launches per step; None if absent."""
    path = os.path.join(ROOT, "profiles", f"r2_launches_{workload}.csv")
    pat = _NCU_KERNEL.get(kernel_id)
    if not pat or not os.path.exists(path):
        return None
    import csv
    tot, cnt = 0.0, 0
    with open(path) as f:
        for r in csv.DictReader(f):
            if pat in r["kernel"]:
                tot += float(r["dram_read_bytes"]) + float(r["dram_write_bytes"])
                cnt += 1
    return int(tot / max(launches_per_step, 1.0)) if cnt else None


def max_over_ranks(vals, device=None):
    """MAX over all ranks of each entry of `vals` (identity without a process group)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in vals]
    t = torch.tensor(list(vals), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def rank_seed_offset(rank: int) -> int:
    """Replicas draw distinct inputs of the same law."""
    return 1000 * rank


class ClockSampler:
    """SM clock and throttle reasons DURING the timed region (B200_PROFILING.md).
    Sampling from another thread or process (a looping `nvidia-smi --query-gpu`, or NVML polled
    from a thread) was measured to stall this process's CUDA calls by 2-60 ms per step: NVML
    queries and the CUDA allocator contend for a driver lock.  So the samples are taken through
    NVML by the BENCH THREAD ITSELF, in three of the timed steps, right after that step's last kernel has been
    enqueued: the GPU is busy with that kernel (milliseconds of queued work) while the host
    asks.  Without pynvml the fallback is a looping nvidia-smi at 200 ms."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index: int):
        self.rows = []          # (time, sm_mhz, reasons bitmask)
        self.smax = None
        self.proc = None
        self.nv = None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.smax = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.nv = pynvml
        except Exception:
            try:
                q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                     "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
                self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "200",
                                              "-i", str(index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
                threading.Thread(target=self._read, daemon=True).start()
            except Exception:
                self.proc = None

    def sample(self):
        """One in-thread NVML sample (call while the GPU has queued work)."""
        if self.nv is None:
            return
        try:
            mhz = float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
            try:
                bits = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
            except Exception:
                bits = int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
            self.rows.append((time.time(), mhz, bits))
        except Exception:
            pass

    def _read(self):
        names = [0x8, 0x40, 0x20, 0x4]
        for line in self.proc.stdout:
            f = [x.strip() for x in line.split(",")]
            try:
                bits = 0
                for nm, v in zip(names, f[2:6]):
                    if v.lower().startswith("active"):
                        bits |= nm
                self.smax = float(f[1])
                self.rows.append((time.time(), float(f[0]), bits))
            except Exception:
                continue

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is not None:
            time.sleep(0.25)
            self.proc.terminate()
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": self.smax, "reasons": ["clock sampling unavailable"], "samples": 0}
        rows = [r for r in self.rows if t0 <= r[0] <= t1 + 0.1] or self.rows
        bits = 0
        for r in rows:
            bits |= r[2]
        return {"sm_mhz": float(np.median([r[1] for r in rows])), "sm_max_mhz": self.smax,
                "reasons": sorted(v for k, v in self.REASONS.items() if bits & k), "samples": len(rows),
                "source": "nvml, sampled by the bench thread in the first, middle and last timed step while that step's last kernel runs" if self.nv is not None else "nvidia-smi -lms 200"}


# ---- the oracle, timed (cpu_baseline leg and --impl reference) ----------------------------------
def oracle_step(cfg, sample: int):
    """One bounded oracle 'step': grid build(s) over all N primitives + `sample` queries of each
    batch kind (sample >= Q: the whole step, nothing extrapolated).  Returns (seconds of the full
    step -- extrapolated linearly in the number of queries when sample < Q --, full-step
    queries/s, detail incl. the wall time this call really took)."""
    import oracle
    prims, pk = cfg["prims"], cfg["pkind"]
    nq = cfg["nq"]
    s = min(sample, nq)
    t_begin = time.perf_counter()
    t0 = time.perf_counter()
    grid = oracle.Grid(prims, pk, oracle.default_cell(prims, pk, "spatial", cfg["r"] if cfg["r"] else None))
    t_build = time.perf_counter() - t0
    t0 = time.perf_counter()
    off, _, _ = oracle.spatial(prims, pk, cfg["queries"][:s], cfg["qkind"], grid)
    t_spatial = time.perf_counter() - t0
    t0 = time.perf_counter()
    off2, _, _ = oracle.spatial(prims, pk, cfg["queries"][:s], cfg["qkind"], grid)   # count-only = same search
    t_count = time.perf_counter() - t0
    del grid
    t_knn = t_kbuild = 0.0
    if cfg["k"]:
        t0 = time.perf_counter()
        kgrid = oracle.Grid(prims, pk, oracle.default_cell(prims, pk, "knn"))
        t_kbuild = time.perf_counter() - t0
        t0 = time.perf_counter()
        oracle.knn(prims, pk, cfg["qpoints"][:s], cfg["k"], kgrid)
        t_knn = time.perf_counter() - t0
        del kgrid
    wall = time.perf_counter() - t_begin
    nb = 3 if cfg["k"] else 2
    full = t_build + t_kbuild + (nq / s) * (t_spatial + t_count + t_knn)
    detail = dict(sample_queries_per_batch=s, extrapolated=bool(s < nq), wall_s=round(wall, 3),
                  t_grid_build_s=round(t_build + t_kbuild, 3),
                  t_spatial_s=round(t_spatial, 3), t_count_s=round(t_count, 3), t_knn_s=round(t_knn, 3),
                  build_mprims_s=round(cfg["n"] / max(t_build, 1e-9) / 1e6, 3),
                  radius_qps=round(s / max(t_spatial, 1e-9), 1),
                  knn_qps=round(s / t_knn, 1) if t_knn else None)
    return full, nb * nq / full, detail


def bench_config(cfg):
    """The `config` object of the JSON line: the workload only, identical in both arms."""
    return dict(workload=cfg["name"], n=cfg["n"], nq=cfg["nq"], dim=cfg["dim"], k=cfg["k"], r=cfg["r"])


def run_reference(args, cfg):
    """Reference arm = the oracle as it stands on the host cores.  Every step builds the grids
    over all N primitives and answers a bounded sample of each query batch; the LAST timed step
    answers ALL queries (nothing extrapolated) unless --ref-no-full-step.  `value` is the
    full-step rate: measured in that last step, else extrapolated linearly in the query count."""
    import oracle
    oracle.build()
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = oracle.num_threads()
    fulls, walls, detail, full_detail = [], [], None, None
    t_run0 = time.perf_counter()
    for i in range(args.warmup + args.steps):
        last = i == args.warmup + args.steps - 1
        whole = last and not args.ref_no_full_step
        full, v, d = oracle_step(cfg, cfg["nq"] if whole else args.ref_sample)
        if i >= args.warmup:
            walls.append(d["wall_s"])
            if whole:
                full_detail = d
                full_step_s = full
            else:
                fulls.append(full)
                detail = d
    nb = 3 if cfg["k"] else 2
    if full_detail is not None:
        step_s, src = full_step_s, "measured: the last timed step answered all queries"
    else:
        step_s, src = float(np.mean(fulls)), "extrapolated linearly from the sampled queries"
    value = nb * cfg["nq"] / step_s
    ms_wall = 1e3 * float(np.mean(walls))
    d0 = detail or full_detail
    sample = (f"per step: uniform-grid build over all {cfg['n']} primitives + first {d0['sample_queries_per_batch']} "
              f"queries of each of the {nb} batches; value = full-step rate ({src})")
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=ms_wall, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic", config=bench_config(cfg),
                ms_per_full_step=1e3 * step_s, full_step_source=src,
                extrapolated_from_queries=None if full_detail is not None else d0["sample_queries_per_batch"],
                sampled_steps_extrapolated_ms=[round(1e3 * f, 1) for f in fulls],
                run_wall_s=round(time.perf_counter() - t_run0, 1),
                cpu_baseline=dict(value=value, unit=UNIT, cores=cores, kind="oracle", sample=sample,
                                  detail=full_detail or detail),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                gpu_launches=0)
    print(json.dumps(line), flush=True)


def quick_config(arbx, torch, dg, name, dev, stream, steps=5, warmup=3):
    """One configuration, device-resident inputs, the same step as the headline (build + CSR
    radius/box query + count-only + kNN), CUDA events around every C-ABI call; median of `steps`."""
    cfg = dg.config(name, 1.0)
    n, nq, D, k, pk, qk = cfg["n"], cfg["nq"], cfg["dim"], cfg["k"], cfg["pkind"], cfg["qkind"]
    prims, queries = torch.from_numpy(cfg["prims"]).to(dev), torch.from_numpy(cfg["queries"]).to(dev)
    qpoints = torch.from_numpy(cfg["qpoints"]).to(dev) if k else None
    offsets = torch.empty(nq + 1, dtype=torch.int32, device=dev)
    counts = torch.empty(nq, dtype=torch.int32, device=dev)
    kidx = torch.empty((nq, k), dtype=torch.int32, device=dev) if k else None
    kdist = torch.empty((nq, k), dtype=torch.float32, device=dev) if k else None
    rec = []
    with torch.cuda.stream(stream):
        h = arbx.arbx_build(prims, D, pk, stream)
        _, total = arbx.arbx_query_spatial(h, queries, nq, qk, offsets, None, 0, stream)
        arbx.arbx_destroy(h, stream)
        indices = torch.empty(max(int(total), 1), dtype=torch.int32, device=dev)
        for i in range(warmup + steps):
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(5)]
            ev[0].record(stream)
            h = arbx.arbx_build(prims, D, pk, stream); ev[1].record(stream)
            arbx.arbx_query_spatial(h, queries, nq, qk, offsets, indices, int(total), stream); ev[2].record(stream)
            arbx.arbx_query_count(h, queries, nq, qk, counts, stream); ev[3].record(stream)
            if k:
                arbx.arbx_query_knn(h, qpoints, nq, k, kidx, kdist, stream)
            ev[4].record(stream)
            arbx.arbx_destroy(h, stream)
            if i >= warmup:
                rec.append(ev)
        torch.cuda.synchronize()
    t = np.median(np.array([[e[j].elapsed_time(e[j + 1]) for j in range(4)] + [e[0].elapsed_time(e[4])] for e in rec]), axis=0)
    out = dict(n=n, nq=nq, dim=D, k=k, ms_per_step=round(float(t[4]), 4), build_ms=round(float(t[0]), 4),
               build_mprims_s=round(n / t[0] / 1e3, 2), radius_csr_qps=round(nq / t[1] * 1e3, 1),
               count_only_qps=round(nq / t[2] * 1e3, 1), knn_qps=round(nq / t[3] * 1e3, 1) if k else None,
               pairs=int(total), steps=steps, warmup=warmup)
    del prims, queries, qpoints, offsets, counts, kidx, kdist, indices
    torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C3", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--scale", type=float, default=1.0, help="shrink N and Q (debugging only; a scaled run is not a bench value)")
    ap.add_argument("--ref-sample", type=int, default=200_000, help="oracle queries per batch per step")
    ap.add_argument("--cpu-sample", type=int, default=500_000, help="cpu_baseline queries per batch")
    ap.add_argument("--ref-no-full-step", action="store_true", help="reference arm: do not run the last step on all queries")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short C1/C2/C4/C5 runs after the timed region")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print(f"note: --warmup {args.warmup} < 3 breaks the timing rules; use >= 3 for a reportable number", file=sys.stderr)

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` outside torchrun: start the N ranks ourselves (one per GPU)
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        os.execvp(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
                                   f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
                                   "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])

    from paper_2507_23700_b200 import datagen as dg
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = dg.config(args.workload, args.scale, seed_offset=0 if args.impl == "reference" else rank_seed_offset(rank))

    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    import torch.distributed as dist
    from paper_2507_23700_b200 import binding as arbx

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    if torch.cuda.device_count() < world:
        raise SystemExit(f"bench.py: {world} ranks but only {torch.cuda.device_count()} CUDA devices (one rank per GPU)")
    arbx.lib()   # fail loudly if the extension is missing
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    n, nq, D, k = cfg["n"], cfg["nq"], cfg["dim"], cfg["k"]
    pk, qk = cfg["pkind"], cfg["qkind"]
    stream = torch.cuda.Stream()
    # pinned host inputs (e2e leg) and device-resident copies (value leg)
    h_prims = torch.from_numpy(cfg["prims"]).pin_memory()
    h_queries = torch.from_numpy(cfg["queries"]).pin_memory()
    h_qpoints = torch.from_numpy(cfg["qpoints"]).pin_memory() if k else None
    d_prims, d_queries = h_prims.to(dev), h_queries.to(dev)
    d_qpoints = h_qpoints.to(dev) if k else None

    # size the CSR buffer once (an untimed query: count + scan only)
    with torch.cuda.stream(stream):
        h0 = arbx.arbx_build(d_prims, D, pk, stream)
        offsets = torch.empty(nq + 1, dtype=torch.int32, device=dev)
        _, total = arbx.arbx_query_spatial(h0, d_queries, nq, qk, offsets, None, 0, stream)
        arbx.arbx_destroy(h0, stream)
    capacity = int(total)
    indices = torch.empty(max(capacity, 1), dtype=torch.int32, device=dev)
    touched = {}     # distinct primitives in the results: the part of the tree a traversal must read
    counts = torch.empty(nq, dtype=torch.int32, device=dev)
    kidx = torch.empty((nq, k), dtype=torch.int32, device=dev) if k else None
    kdist = torch.empty((nq, k), dtype=torch.float32, device=dev) if k else None
    nbatches = 3 if k else 2

    marks = []   # (name, event) per step, on `stream`
    sampler_box = [None]
    step_no = [0]
    # NVML calls take ~10 us but were seen to take 4-17 ms about once in 300 calls: three samples
    # (first, middle and last timed step) keep that risk out of the timing
    sample_steps = set()

    def mark(name):
        e = torch.cuda.Event(enable_timing=True)
        e.record(stream)
        marks.append((name, e))

    def step(prims, queries, qpoints, timed_marks, out=None):
        o_off, o_idx, o_cnt, o_ki, o_kd = out if out is not None else (offsets, indices, counts, kidx, kdist)
        h = arbx.arbx_build(prims, D, pk, stream)
        if timed_marks: mark("build")
        arbx.arbx_query_spatial(h, queries, nq, qk, o_off, o_idx, capacity, stream)
        if timed_marks: mark("spatial")
        arbx.arbx_query_count(h, queries, nq, qk, o_cnt, stream)
        if timed_marks: mark("count")
        if k:
            arbx.arbx_query_knn(h, qpoints, nq, k, o_ki, o_kd, stream)
            if timed_marks: mark("knn")
        if timed_marks and sampler_box[0] is not None and step_no[0] in sample_steps:
            sampler_box[0].sample()      # the GPU is busy with the kernels just enqueued
        step_no[0] += 1
        arbx.arbx_destroy(h, stream)

    # ---- value leg: inputs resident in HBM --------------------------------------------------------
    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            step(d_prims, d_queries, d_qpoints, False)
        barrier()
        sampler = ClockSampler(local_rank) if rank == 0 and not os.environ.get("ARBX_BENCH_NO_SMI") else None
        sampler_box[0] = sampler
        step_no[0] = 0
        sample_steps.update({0, args.steps // 2, args.steps - 1})
        arbx.arbx_profile_enable(True)
        arbx.arbx_profile_read()
        l0 = arbx.arbx_launch_count()
        t_wall0 = time.time()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            mark("begin")
            step(d_prims, d_queries, d_qpoints, True)
        e1.record(stream)
        barrier()
        t_wall1 = time.time()
        launches = arbx.arbx_launch_count() - l0
        prof = arbx.arbx_profile_read()
        arbx.arbx_profile_enable(False)
        sampler_box[0] = None
        clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    ms_total = e0.elapsed_time(e1)
    seen = torch.zeros(n, dtype=torch.bool, device=dev)
    if capacity:
        seen[indices[:capacity].long()] = True
    touched["touched_spatial"] = int(seen.sum())
    if k:
        seen.zero_()
        seen[kidx.reshape(-1).clamp_(min=0).long()] = True
        touched["touched_knn"] = int(seen.sum())
    del seen
    calls = {}
    for (na, ea), (nb_, eb) in zip(marks[:-1], marks[1:]):
        if nb_ != "begin":
            calls[nb_] = calls.get(nb_, 0.0) + ea.elapsed_time(eb)
    calls = {c: v / args.steps for c, v in calls.items()}
    # per-step durations (begin of step i -> begin of step i+1; the last one ends at e1): a host
    # hiccup (the storage query synchronises once per call) shows up as max >> median
    begins = [e for (nm, e) in marks if nm == "begin"]
    per_step = [a.elapsed_time(b) for a, b in zip(begins[:-1], begins[1:])] + [begins[-1].elapsed_time(e1)]
    step_stats = dict(min=round(min(per_step), 4), median=round(float(np.median(per_step)), 4), max=round(max(per_step), 4),
                      all=[round(x, 3) for x in per_step])
    marks.clear()

    # ---- outside the step: the capped count (NEXT-1, arbx_query_count_upto), device-timed ---------------
    extras = {}
    with torch.cuda.stream(stream):
        hx = arbx.arbx_build(d_prims, D, pk, stream)
        for limit in (1, 8):
            for rep in range(3):
                a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
                a.record(stream)
                arbx.arbx_query_count_upto(hx, d_queries, nq, qk, limit, counts, stream)
                b.record(stream)
            torch.cuda.synchronize()
            extras[f"count_upto_{limit}_qps"] = round(nq / a.elapsed_time(b) * 1e3, 1)
        if pk == 0 and qk == 2 and cfg["r"]:
            # NEXT-2 self-join over the primitives themselves with the workload's radius (device-timed)
            poff = torch.empty(n + 1, dtype=torch.int32, device=dev)
            _, ptotal = arbx.arbx_query_pairs(hx, float(cfg["r"]), poff, None, 0, stream)
            pidx = torch.empty(max(ptotal, 1), dtype=torch.int32, device=dev)
            for rep in range(3):
                a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
                a.record(stream)
                arbx.arbx_query_pairs(hx, float(cfg["r"]), poff, pidx, pidx.numel(), stream)
                b.record(stream)
            torch.cuda.synchronize()
            lab = torch.empty(n, dtype=torch.int32, device=dev)
            for rep in range(2):
                c = torch.cuda.Event(enable_timing=True); d = torch.cuda.Event(enable_timing=True)
                c.record(stream)
                arbx.arbx_dbscan(hx, float(cfg["r"]), 8, lab, stream)
                d.record(stream)
            torch.cuda.synchronize()
            extras["dbscan_minpts8_prims_per_s"] = round(n / c.elapsed_time(d) * 1e3, 1)
            extras["dbscan_clusters"] = int((lab == torch.arange(n, device=dev, dtype=torch.int32)).sum())
            extras["self_join_pairs"] = int(ptotal)
            extras["self_join_prims_per_s"] = round(n / a.elapsed_time(b) * 1e3, 1)
            del poff, pidx
        arbx.arbx_destroy(hx, stream)
        # NEXT-4 fp64 coordinates (arbx_*_f64: exact fp64 leaf tests over the fp32 tree), device-timed on
        # the same primitives and the first 10^6 queries of the batch, converted to fp64
        nq64 = min(nq, 1_000_000)
        p64, q64 = d_prims.double(), d_queries[:nq64].double().contiguous()
        c64 = torch.empty(nq64, dtype=torch.int32, device=dev)
        for rep in range(2):
            a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True); c = torch.cuda.Event(enable_timing=True)
            a.record(stream)
            h64 = arbx.arbx_build_f64(p64, D, pk, stream)
            b.record(stream)
            arbx.arbx_query_count_f64(h64, q64, nq64, qk, c64, stream)
            c.record(stream)
            arbx.arbx_destroy(h64, stream)
        torch.cuda.synchronize()
        extras["f64_build_mprims_s"] = round(n / a.elapsed_time(b) / 1e3, 2)
        extras["f64_count_qps"] = round(nq64 / b.elapsed_time(c) * 1e3, 1)
        del p64, q64, c64
    torch.cuda.synchronize()

    # ---- e2e leg: pinned host inputs in, every result back to pinned host memory ---------------------
    e2e = None
    if not args.no_e2e:
        ho = torch.empty(nq + 1, dtype=torch.int32).pin_memory()
        hi = torch.empty(max(capacity, 1), dtype=torch.int32).pin_memory()
        hc = torch.empty(nq, dtype=torch.int32).pin_memory()
        hki = torch.empty((nq, k), dtype=torch.int32).pin_memory() if k else None
        hkd = torch.empty((nq, k), dtype=torch.float32).pin_memory() if k else None
        # Three streams, double-buffered: while step i computes, the inputs of step i+1 are coming
        # in and the results of step i-1 are going out (H2D and D2H use separate copy engines).
        # Every step still copies all of its inputs in and all of its results out.
        s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
        inb = [(torch.empty_like(d_prims), torch.empty_like(d_queries), torch.empty_like(d_qpoints) if k else None)
               for _ in range(2)]
        outb = [(offsets, indices, counts, kidx, kdist),
                (torch.empty_like(offsets), torch.empty_like(indices), torch.empty_like(counts),
                 torch.empty_like(kidx) if k else None, torch.empty_like(kdist) if k else None)]
        ev_in, ev_comp, ev_out = [None, None], [None, None], [None, None]

        def enqueue_in(i):
            b = i % 2
            with torch.cuda.stream(s_in):
                if ev_comp[b] is not None: s_in.wait_event(ev_comp[b])     # step i-2 is done with this buffer
                inb[b][0].copy_(h_prims, non_blocking=True)
                inb[b][1].copy_(h_queries, non_blocking=True)
                if k: inb[b][2].copy_(h_qpoints, non_blocking=True)
                ev_in[b] = torch.cuda.Event(); ev_in[b].record(s_in)

        def run(i):
            b = i % 2
            stream.wait_event(ev_in[b])
            if ev_out[b] is not None: stream.wait_event(ev_out[b])          # results of step i-2 have left
            with torch.cuda.stream(stream):
                step(inb[b][0], inb[b][1], inb[b][2], False, outb[b])
            ev_comp[b] = torch.cuda.Event(); ev_comp[b].record(stream)

        def enqueue_out(i):
            b = i % 2
            o_off, o_idx, o_cnt, o_ki, o_kd = outb[b]
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_comp[b])
                ho.copy_(o_off, non_blocking=True)
                hi[:capacity].copy_(o_idx[:capacity], non_blocking=True)
                hc.copy_(o_cnt, non_blocking=True)
                if k:
                    hki.copy_(o_ki, non_blocking=True)
                    hkd.copy_(o_kd, non_blocking=True)
                ev_out[b] = torch.cuda.Event(); ev_out[b].record(s_out)

        def pipeline(nsteps):
            enqueue_in(0)
            for i in range(nsteps):
                if i + 1 < nsteps: enqueue_in(i + 1)
                run(i)
                enqueue_out(i)

        pipeline(2)                       # warm-up (allocator, second buffer set)
        barrier()
        a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
        a.record(s_in)
        pipeline(args.steps)
        b.record(s_out)
        barrier()
        ms_e2e = a.elapsed_time(b) / args.steps
        h2d = h_prims.numel() * 4 + h_queries.numel() * 4 + (h_qpoints.numel() * 4 if k else 0)
        d2h = ho.numel() * 4 + capacity * 4 + hc.numel() * 4 + (hki.numel() * 8 if k else 0)
        assert int(ho[-1]) == capacity and int(hc.sum()) == capacity, "e2e results inconsistent"
    # ---- the other BASELINE.json configurations, same process, after the timed region ------------------
    l2_note = ("inputs and outputs exceed L2 (no flush needed)" if (d_prims.numel() + d_queries.numel()) * 4 > 126e6
               else "working set fits L2")
    others = None
    if rank == 0 and world == 1 and not args.no_other_configs and args.scale == 1.0:
        del d_prims, d_queries, d_qpoints, indices, counts, kidx, kdist, offsets
        if not args.no_e2e:
            del inb, outb, ho, hi, hc, hki, hkd
        torch.cuda.empty_cache()
        others = {}
        for name in ("C1", "C2", "C3", "C4", "C5"):
            if name != cfg["name"]:
                others[name] = quick_config(arbx, torch, dg, name, dev, stream)

    # max over ranks
    ms_step = ms_total / args.steps
    ms_step, ms_e2e_max = max_over_ranks([ms_step, ms_e2e if not args.no_e2e else 0.0], dev)
    if not args.no_e2e:
        e2e = dict(value=world * nbatches * nq / (ms_e2e_max / 1e3), unit=UNIT, ms_per_step=ms_e2e_max,
                   h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h))

    if rank == 0:
        peak, peak_src = _peaks()
        ab = algorithmic_bytes(cfg, dict(pairs=capacity, **touched))
        kern = {}
        for name, (ms, ncalls) in prof.items():
            ms_s = ms / args.steps
            by = ab.get(name)
            kern[name] = dict(ms_per_step=round(ms_s, 4), launches_per_step=ncalls / args.steps,
                              share=round(ms_s / ms_step, 4),
                              algorithmic_gb=round(by / 1e9, 4) if by else None,
                              achieved_gbs=round(by / 1e6 / ms_s, 1) if by and ms_s > 0 else None,
                              frac_of_peak=round(by / 1e6 / ms_s / peak, 4) if by and ms_s > 0 else None)
        dom = max(kern, key=lambda x: kern[x]["ms_per_step"])
        dk = kern[dom]
        # per-LAUNCH figures for the dominant kernel
        lps = max(dk["launches_per_step"], 1)
        roofline = dict(bound="hbm", kernel=dom, achieved=dk["achieved_gbs"], peak=peak, unit="GB/s",
                        frac=dk["frac_of_peak"], traffic=ncu_traffic(dom, cfg["name"], lps), peak_source=peak_src,
                        algorithmic_bytes_per_launch=int(ab[dom] / lps) if ab.get(dom) else None,
                        ms_per_launch=round(dk["ms_per_step"] / lps, 4), share_of_step=dk["share"])
        build_bytes = sum(ab[x] for x in ab if x.startswith("B"))
        breakdown = dict(
            build_mprims_s=round(n / calls["build"] / 1e3, 2), build_ms=round(calls["build"], 4),
            build_algorithmic_gbs=round(build_bytes / 1e6 / calls["build"], 1),
            build_frac_of_peak=round(build_bytes / 1e6 / calls["build"] / peak, 4),
            radius_csr_qps=round(nq / calls["spatial"] * 1e3, 1), radius_csr_ms=round(calls["spatial"], 4),
            count_only_qps=round(nq / calls["count"] * 1e3, 1), count_only_ms=round(calls["count"], 4),
            knn_qps=round(nq / calls["knn"] * 1e3, 1) if k else None, knn_ms=round(calls["knn"], 4) if k else None,
            pairs=capacity, step_ms=step_stats, extras_outside_step=extras, kernels=kern,
            byte_model=dict(model="SURVEY.md 8(d) compulsory bytes; a traversal reads (leaf + child box + links) of the TOUCHED primitives once",
                            whole_tree_bytes=int(ab["_whole_tree"]), **touched))
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            import oracle
            oracle.build()
            _, v, detail = oracle_step(cfg, args.cpu_sample)
            cpu = dict(value=v, unit=UNIT, cores=oracle.num_threads(), kind="oracle",
                       sample=(f"uniform-grid build over all {n} primitives + first {detail['sample_queries_per_batch']} "
                               f"queries of each of the {nbatches} batches of this workload, query time extrapolated linearly to Q={nq}"),
                       detail=detail)
        line = dict(metric=METRIC, value=world * nbatches * nq / (ms_step / 1e3), unit=UNIT, n_gpus=world,
                    steps=args.steps, warmup=args.warmup, ms_per_step=ms_step, higher_is_better=True,
                    scaling="weak", vs_baseline=None, dtype="f32", data="synthetic",
                    config=bench_config(cfg),
                    run=dict(scale=args.scale, parallelism=f"replicas x{world}" if world > 1 else "single GPU",
                             l2=l2_note),
                    clocks=clocks, e2e=e2e, gpu_launches=int(launches), roofline=roofline,
                    cpu_baseline=cpu, breakdown=breakdown, other_configs=others)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
