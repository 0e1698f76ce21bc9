#!/usr/bin/env python
"""bench.py — times the ETC migration hot path on B200.

A step = one pass of the whole hot path over one synthetic model state:
  (a1) etc_layout_create x2 -> (a2) etc_cost_matrix -> (a3) etc_sketch -> (a4) etc_plan_create -> (a5,a6) etc_migrate.
metric = migrate GB/s counting read+write bytes: (2*direct + 4*staged payload bytes) / step time, plus the fraction of the
measured HBM copy bandwidth the dominant copy kernel reaches (roofline) and the cost-matrix + sketch time.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config c2] [--impl reference]
N > 1 (torchrun): independent replicas, one per GPU ("replicas only": the path's only exchange step is closed by
BASELINE.json, so there is no data-path collective); value = all ranks' bytes / max-over-ranks time.
"""
from __future__ import annotations
import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "migrate GB/s (read+write)"
UNIT = "GB/s"

def ncu_traffic(workload_name: str, mode: str, kernel_prefix: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed ncu --set full
    captures (profiles/ncu_traffic.csv names the capture each row was read from).  None where no capture exists."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    try:
        import csv
        for row in csv.DictReader(open(p)):
            if row["workload"] == workload_name and row["mode"] == mode and kernel_prefix.startswith(row["kernel"]):
                return int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
    except Exception:
        pass
    return None


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.idx, self.proc, self.path = gpu_index, None, None

    def start(self):
        try:
            f = tempfile.NamedTemporaryFile("w", suffix=".csv", delete=False)
            self.path = f.name
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.idx}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=f,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if not self.proc:
            return out
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        try:
            for line in open(self.path):
                c = [x.strip() for x in line.split(",")]
                if len(c) < 9:
                    continue
                try:
                    sm.append(float(c[1])); mx.append(float(c[2]))
                except ValueError:
                    continue
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def max_over_ranks(ms: float, world: int, device=None) -> float:
    """Timing of a multi-rank run = the slowest rank's device time (the only data `torch.distributed` carries here:
    "replicas only").  Works on any backend (nccl on the GPU box, gloo in the CPU tests)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(world: int, hbm_bytes_per_replica: int, ms_per_step: float) -> float:
    """Whole-job GB/s: every rank migrates one replica of the workload (weak scaling), time = max over ranks."""
    return world * hbm_bytes_per_replica / (ms_per_step * 1e-3) / 1e9


# ------------------------------------------------------------------------------------------------ reference arm (oracle)
def oracle_sample(w, budget_elems=6_000_000, threads=1):
    """Time the CPU oracle, as it stands, on a bounded sample of the workload: cost matrix + sketch on the full layout
    (they are metadata), then the element-wise migration of the first `m` elements of every new buffer.  threads > 1:
    the (new rank, kind) buffers are independent, so they are handed to that many host threads (the oracle's C code
    runs outside the GIL); each task counts into its own traffic matrix."""
    import numpy as np
    from concurrent.futures import ThreadPoolExecutor
    from oracle import oracle as O
    oo, on = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
    t0 = time.perf_counter()
    ov, need, hold = O.overlap(oo, on, method="ranges")
    t1 = time.perf_counter()
    dm, val = O.sketch_hungarian(ov)
    t2 = time.perf_counter()
    bufs = [(n, k, on.buffer_elems(n, k)) for n in range(on.n_dev) for k in on.kinds()]
    bufs = [b for b in bufs if b[2] > 0]
    m = max(1, budget_elems // max(1, len(bufs)))
    # position-stamped source buffers would need the full state in host RAM; the oracle's migration time does not
    # depend on the values, so the sample runs in traffic-counting mode plus a copy into a destination window.
    src = None
    P = max(oo.n_dev, on.n_dev)
    moved = sum(min(m, cnt) * on.elem_bytes(k) for n, k, cnt in bufs)

    def one(b):
        n, k, cnt = b
        O.migrate_range(oo, on, dm, n, k, 0, min(m, cnt), src, None, np.zeros((P, P), np.int64), None)

    threads = max(1, min(int(threads), len(bufs)))
    t3 = time.perf_counter()
    if threads == 1:
        for b in bufs:
            one(b)
    else:
        with ThreadPoolExecutor(threads) as ex:
            list(ex.map(one, bufs))
    t4 = time.perf_counter()
    return dict(cost_ms=(t1 - t0) * 1e3, sketch_ms=(t2 - t1) * 1e3, migrate_s=t4 - t3, payload_bytes=moved,
                elems_per_buffer=m, n_buffers=len(bufs), local_opt=val, threads=O.max_threads(), migrate_threads=threads)


def oracle_metadata(w):
    """CPU side of cost matrix + sketch on the full layout of workload w: the oracle's plain range-overlap routine, its
    plain O(k^3) Hungarian, and (where SciPy is installed) linear_sum_assignment, the routine the paper itself calls
    (PAPER.md:134)."""
    from oracle import oracle as O
    oo, on = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
    O.overlap(oo, on, method="ranges")                      # untimed: starts the OpenMP thread pool
    t0 = time.perf_counter()
    ov, need, hold = O.overlap(oo, on, method="ranges")
    t1 = time.perf_counter()
    dm, val = O.sketch_hungarian(ov)
    t2 = time.perf_counter()
    out = {"devices": [oo.n_dev, on.n_dev], "cost_matrix_ms": (t1 - t0) * 1e3, "cost_matrix_threads": O.max_threads(),
           "hungarian_ms": (t2 - t1) * 1e3, "local_bytes": int(val)}
    try:
        from scipy.optimize import linear_sum_assignment
        t3 = time.perf_counter()
        r, c = linear_sum_assignment(ov, maximize=True)
        out["scipy_linear_sum_assignment_ms"] = (time.perf_counter() - t3) * 1e3
        out["scipy_agrees"] = bool(int(ov[r, c].sum()) == int(val))
    except ImportError:
        pass
    return out


def run_reference(args, w):
    rank, _, world = dist_env()
    if rank != 0:
        return
    from oracle import oracle as O
    O.build()
    times, last = [], None
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        last = oracle_sample(w, budget_elems=args.ref_elems, threads=os.cpu_count() or 1)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
    ms = statistics.mean(times) * 1e3
    # same metric: read+write bytes per second; the oracle copies each sampled payload byte once (1R + 1W)
    val = 2 * last["payload_bytes"] / (ms / 1e3) / 1e9
    cores = last["migrate_threads"]   # one host thread per (new rank, kind) buffer; the cost matrix uses OpenMP (below)
    sample = (f"first {last['elems_per_buffer']} elements of each of {last['n_buffers']} new buffers "
              f"({last['payload_bytes']} payload bytes, {cores} host threads) + full cost matrix (ranges routine, {last['threads']} OpenMP "
              f"threads) + Hungarian, per step")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u8", "data": "synthetic", "config": {"workload": w["name"], "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "cost_matrix_ms": last["cost_ms"], "sketch_ms": last["sketch_ms"]},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------ CUDA arm
def run_cuda(args, w):
    import numpy as np
    import torch
    import paper_2607_04749_b200 as E
    from etc_inputs import bench_fill_torch

    rank, local_rank, world = dist_env()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    E.init(local_rank)
    model = w["model"]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- resident inputs: every old shard buffer filled with the workload's value distribution
    lay_old, lay_new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
    src = E.alloc_buffers(lay_old, dev)
    dst = E.alloc_buffers(lay_new, dev)
    for (d, k), t in src.items():
        view = t.view(torch.bfloat16 if (k == 0 and model["param_bytes"] == 2) else torch.float32)
        bench_fill_torch(view, k, w["seed"] + d * 4 + k)
    P = max(lay_old.n_dev, lay_new.n_dev)
    out_cost = (torch.empty((lay_new.n_dev, P), dtype=torch.int64, device=dev),
                torch.empty(lay_new.n_dev, dtype=torch.int64, device=dev), torch.empty(P, dtype=torch.int64, device=dev))
    out_sk = (torch.empty(lay_new.n_dev, dtype=torch.int32, device=dev), torch.empty(1, dtype=torch.int64, device=dev))
    flags = E.ETC_ALL_STAGED if args.all_staged else E.ETC_LOCAL_DIRECT
    # staging sized once from a first plan (allocation is not part of the path)
    ov, _, _ = E.etc_cost_matrix(lay_old, lay_new, out=out_cost)
    dm, _ = E.etc_sketch(ov, out=out_sk)
    plan0 = E.etc_plan_create(lay_old, lay_new, dm, flags)
    st0 = plan0.stats
    staging = torch.empty(max(st0.staging_bytes, 16), dtype=torch.uint8, device=dev)
    from paper_2607_04749_b200.binding import pointer_tables
    src_tab, dst_tab = pointer_tables(plan0, src, dst)
    hbm_bytes = st0.hbm_bytes
    del plan0

    stream = torch.cuda.current_stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)

    plan_stream = torch.cuda.Stream(dev, priority=-1)     # high priority: its small kernels cut in front of copy CTAs
    planned = [torch.cuda.Event() for _ in range(4)]
    step_no = [0]

    def step(record=None):
        """One pass of the whole hot path.  Planning (a1-a4, metadata only, one host sync for table sizes) is enqueued
        on its own stream so that its host sync does not wait for the previous step's copy kernels; the copy stream waits
        for the plan by event.  record: list to which this step's timing events are appended."""
        e = [ev() for _ in range(8)] if record is not None else None
        with torch.cuda.stream(plan_stream):
            if e: e[0].record(plan_stream)
            lo, ln = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])     # (a1)
            if e: e[1].record(plan_stream)
            ov, need, hold = E.etc_cost_matrix(lo, ln, out=out_cost, stream=plan_stream)             # (a2)
            if e: e[2].record(plan_stream)
            dm, lb = E.etc_sketch(ov, out=out_sk, stream=plan_stream)                                # (a3)
            if e: e[3].record(plan_stream)
            plan = E.etc_plan_create(lo, ln, dm, flags, stream=plan_stream)                          # (a4)
            if e: e[4].record(plan_stream)
            done = planned[step_no[0] % len(planned)]
            done.record(plan_stream)
        step_no[0] += 1
        stream.wait_event(done)
        if e: e[7].record(stream)
        E.etc_migrate(plan, src_tab, dst_tab, staging, E.ETC_PHASE_PACK, stream=stream)          # (a5) + local
        if e: e[5].record(stream)
        E.etc_migrate(plan, src_tab, dst_tab, staging, E.ETC_PHASE_UNPACK, stream=stream)        # (a6)
        if e: e[6].record(stream)
        if record is not None:
            record.append(e)
        return plan

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = E.kernel_launches()
    recs = []
    t_begin, t_end = ev(), ev()
    barrier()
    t_begin.record(stream)
    for _ in range(args.steps):
        plan = step(recs)
    t_end.record(stream)
    barrier()
    launches = E.kernel_launches() - launches0
    clocks = sampler.stop()
    total_ms = t_begin.elapsed_time(t_end)
    total_ms = max_over_ranks(total_ms, world, dev)
    ms_per_step = total_ms / args.steps
    stats = plan.stats
    phase = lambda a, b: statistics.mean(r[a].elapsed_time(r[b]) for r in recs)
    bd = {"layout_ms": phase(0, 1), "cost_matrix_ms": phase(1, 2), "sketch_ms": phase(2, 3), "plan_ms": phase(3, 4),
          "pack_local_ms": phase(7, 5), "unpack_ms": phase(5, 6)}
    value = job_value(world, hbm_bytes, ms_per_step)

    # ---- roofline of the dominant kernel, timed live with CUDA events over the timed region
    peak, peak_src = measured_peak()
    direct = stats.local_bytes + stats.remote_bytes - stats.staged_bytes
    k1_bytes = 2 * (stats.staged_bytes + direct)       # launch 1: pack (staged payload) + local (direct payload): 1R+1W
    k2_bytes = 2 * stats.staged_bytes                  # launch 2: unpack
    if bd["pack_local_ms"] >= bd["unpack_ms"]:
        kname, kbytes, kms = "migrate_copy_kernel<false> (pack + local)", k1_bytes, bd["pack_local_ms"]
    else:
        kname, kbytes, kms = "migrate_copy_kernel<true> (unpack)", k2_bytes, bd["unpack_ms"]
    achieved = kbytes / (kms * 1e-3) / 1e9 if kms > 0 else 0.0
    roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "peak_source": peak_src, "algorithmic_bytes_per_launch": kbytes,
                "avg_launch_ms": kms, "traffic": ncu_traffic(w["name"], "ALL_STAGED" if args.all_staged else "LOCAL_DIRECT", kname),
                "frac_of_8TBs_nominal": achieved / 8000.0}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u8", "data": "synthetic",
            "config": {"workload": w["name"], "old": w["old"], "new": w["new"],
                       "mode": "ALL_STAGED" if args.all_staged else "LOCAL_DIRECT", "l2": "inputs_larger_than_L2",
                       "pipelining": "planning (a1-a4) of step i+1 on its own stream overlaps the copy kernels of step i",
                       "parallelism": "replicas only" if world > 1 else "1 GPU, all virtual devices in one HBM"},
            "hbm_bytes_per_step": hbm_bytes, "payload": {"local": stats.local_bytes, "remote": stats.remote_bytes,
                                                         "staged": stats.staged_bytes},
            "breakdown_ms": bd, "cost_sketch_ms": bd["cost_matrix_ms"] + bd["sketch_ms"],
            "roofline": roofline, "clocks": clocks, "gpu_launches": launches}

    del staging
    torch.cuda.empty_cache()
    if rank == 0 and not args.no_extras:
        line["extras"] = extras(E, torch, w, dev, src, dst, lay_old, lay_new, peak)

    # ---- e2e: the same step through the C ABI with HOST buffers; H2D of every old shard and D2H of every new shard
    #      are inside the timed region
    if not args.no_e2e:
        try:
            line["e2e"] = e2e(E, torch, args, w, dev, src, dst, hbm_bytes, world, barrier)
        except Exception as ex:       # e.g. not enough pinned host memory on the box
            line["e2e"] = {"value": None, "unit": UNIT, "error": repr(ex)[:200]}
    if rank == 0 and not args.no_extras:
        try:                          # destroys src: last GPU leg
            del dst
            torch.cuda.empty_cache()
            line["extras"]["chunked_eager_release"] = chunked(E, torch, w, dev, src, lay_old, lay_new, args.e2e_staging)
        except Exception as ex:
            line["extras"]["chunked_eager_release"] = {"error": repr(ex)[:200]}

    if rank == 0:
        if world == 1 and not args.no_cpu:
            from oracle import oracle as O
            ncores = os.cpu_count() or 1
            o = oracle_sample(w, budget_elems=args.cpu_elems, threads=ncores)          # all host cores
            o1 = oracle_sample(w, budget_elems=max(1, args.cpu_elems // 8), threads=1)  # single-thread figure
            line["cpu_baseline"] = {
                "value": 2 * o["payload_bytes"] / o["migrate_s"] / 1e9, "unit": UNIT, "cores": o["migrate_threads"],
                "kind": "oracle",
                "sample": f"element-wise oracle migration of the first {o['elems_per_buffer']} elements of each of "
                          f"{o['n_buffers']} new buffers ({o['payload_bytes']} payload bytes, 1R+1W each), the independent "
                          f"buffers spread over {o['migrate_threads']} host threads; host has {ncores} cores",
                "single_thread_value": 2 * o1["payload_bytes"] / o1["migrate_s"] / 1e9,
                "single_thread_sample": f"first {o1['elems_per_buffer']} elements of each buffer, 1 thread",
                "cost_matrix_ms": o["cost_ms"], "sketch_ms": o["sketch_ms"], "cost_matrix_threads": o["threads"]}
            try:
                from etc_inputs import workload as _wl
                line["cpu_baseline"]["metadata"] = {w["name"]: oracle_metadata(w), "c5b": oracle_metadata(_wl("c5b"))}
            except Exception as ex:
                line["cpu_baseline"]["metadata"] = {"error": repr(ex)[:200]}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def extras(E, torch, w, dev, src, dst, lay_old, lay_new, peak):
    """Context numbers outside the timed region: pack / unpack kernel rates with everything staged, and the
    metadata-only cost matrix + sketch of the 512 -> 384 device layout (BASELINE.json configs[4])."""
    from etc_inputs import workload
    out = {}
    ev = lambda: torch.cuda.Event(enable_timing=True)
    stream = torch.cuda.current_stream()
    try:
        ov, _, _ = E.etc_cost_matrix(lay_old, lay_new)
        dm, _ = E.etc_sketch(ov)
        plan = E.etc_plan_create(lay_old, lay_new, dm, E.ETC_ALL_STAGED)
        stg = torch.empty(max(plan.stats.staging_bytes, 16), dtype=torch.uint8, device=dev)
        tp, tu = [], []
        for i in range(8):
            a, b, c = ev(), ev(), ev()
            a.record(stream); E.etc_migrate(plan, src, dst, stg, E.ETC_PHASE_PACK)
            b.record(stream); E.etc_migrate(plan, src, dst, stg, E.ETC_PHASE_UNPACK)
            c.record(stream); torch.cuda.synchronize()
            if i >= 3:
                tp.append(a.elapsed_time(b)); tu.append(b.elapsed_time(c))
        nbytes = 2 * plan.stats.staged_bytes
        out["all_staged"] = {"staged_bytes": plan.stats.staged_bytes, "pack_ms": statistics.mean(tp),
                             "unpack_ms": statistics.mean(tu),
                             "pack_GBs": nbytes / statistics.mean(tp) / 1e6, "unpack_GBs": nbytes / statistics.mean(tu) / 1e6,
                             "pack_frac_of_measured_peak": nbytes / statistics.mean(tp) / 1e6 / peak,
                             "unpack_frac_of_measured_peak": nbytes / statistics.mean(tu) / 1e6 / peak}
        del stg, plan
    except Exception as ex:
        out["all_staged"] = {"error": repr(ex)[:200]}
    try:
        # one migration, cold start to finish, nothing overlapped: (a1)-(a6) on one stream, host wall clock from the
        # first call to the synchronise after the last kernel (the latency a single reconfiguration sees)
        walls = []
        for i in range(8):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            lo, ln = E.etc_layout_create(w["model"], w["old"]), E.etc_layout_create(w["model"], w["new"])
            ov, _, _ = E.etc_cost_matrix(lo, ln)
            dm, _ = E.etc_sketch(ov)
            plan = E.etc_plan_create(lo, ln, dm, 0)
            if i == 0:
                stg = torch.empty(max(plan.stats.staging_bytes, 16), dtype=torch.uint8, device=dev)
            E.etc_migrate(plan, src, dst, stg)
            torch.cuda.synchronize()
            if i >= 3:
                walls.append((time.perf_counter() - t0) * 1e3)
        hb = 2 * plan.stats.local_bytes + 4 * plan.stats.remote_bytes
        out["one_shot"] = {"wall_ms_median": statistics.median(walls), "wall_ms_best": min(walls),
                           "GBs": hb / statistics.median(walls) / 1e6,
                           "note": "a1-a6 serially on one stream, host wall clock incl. every host-side step, no overlap "
                                   "with a previous migration"}
        del stg, plan
    except Exception as ex:
        out["one_shot"] = {"error": repr(ex)[:200]}
    try:
        # (f1) virtual rank allocator on config 3's pre-emption (16 -> 12 devices, 4 per node), metadata only: bytes
        # that change device under the sketch alone, under the sketch composed with Algorithm 2 (one hop: communication
        # coalescing), and if the defragmentation were a second migration stage
        w3 = workload("c3")
        lo, ln = E.etc_layout_create(w3["model"], w3["old"]), E.etc_layout_create(w3["model"], w3["new"])
        ov, need, _ = E.etc_cost_matrix(lo, ln)
        dm, _ = E.etc_sketch(ov)
        E.etc_defrag(dm, lo.n_dev, ln.n_dev, 4, E.ETC_DEFRAG_BOTH); torch.cuda.synchronize()     # untimed: loads the kernel
        a, b = ev(), ev()
        a.record(stream)
        final, n_ops, _ = E.etc_defrag(dm, lo.n_dev, ln.n_dev, 4, E.ETC_DEFRAG_BOTH)
        b.record(stream); torch.cuda.synchronize()
        p0, p1 = E.etc_plan_create(lo, ln, dm), E.etc_plan_create(lo, ln, final)
        dm_h, fin_h, need_h = dm.cpu().tolist(), final.cpu().tolist(), need.cpu().tolist()
        moved = sum(need_h[r] for r in range(ln.n_dev) if dm_h[r] != fin_h[r])
        out["defrag_c3_16_to_12"] = {"devices_per_node": 4, "sketch_map": dm_h, "final_map": fin_h,
                                     "operators": [int(x) for x in n_ops.cpu().tolist()], "defrag_ms": a.elapsed_time(b),
                                     "remote_bytes_sketch_only": p0.stats.remote_bytes,
                                     "remote_bytes_coalesced": p1.stats.remote_bytes,
                                     "remote_bytes_two_stage": p0.stats.remote_bytes + moved,
                                     "nodes_occupied": [len({p // 4 for p in dm_h}), len({p // 4 for p in fin_h})]}
        del p0, p1
    except Exception as ex:
        out["defrag_c3_16_to_12"] = {"error": repr(ex)[:200]}
    try:
        wb = workload("c5b")
        lo, ln = E.etc_layout_create(wb["model"], wb["old"]), E.etc_layout_create(wb["model"], wb["new"])
        tc, ts = [], []
        for i in range(6):
            a, b, c = ev(), ev(), ev()
            a.record(stream); ov, _, _ = E.etc_cost_matrix(lo, ln)
            b.record(stream); dm, lb = E.etc_sketch(ov)
            c.record(stream); torch.cuda.synchronize()
            if i >= 2:
                tc.append(a.elapsed_time(b)); ts.append(b.elapsed_time(c))
        out["c5b_512_to_384"] = {"cost_matrix_ms": statistics.mean(tc), "sketch_ms": statistics.mean(ts),
                                 "local_bytes": int(lb.item()), "pieces": [lo.n_pieces, ln.n_pieces]}
    except Exception as ex:
        out["c5b_512_to_384"] = {"error": repr(ex)[:200]}
    return out


def e2e(E, torch, args, w, dev, src, dst, hbm_bytes, world, barrier):
    """The same metric through the public API with HOST buffers: old shards in pinned host memory -> whole path (a1-a6,
    as kind-by-kind rounds of a kind-major plan) -> new shards in pinned host memory, everything inside the timed region.
    Headline: zero-copy (host_pipeline.HostMigration(zero_copy=True)): the pinned host buffers ARE the source and
    destination tables of the C-ABI call, the copy kernels move every byte over PCIe, no device copy of any shard exists.
    Beside it: the DMA pipelines (cudaMemcpyAsync of every old shard byte / of only the regions the plan reads, rounds
    on device buffers, cudaMemcpyAsync of the new shards; three streams)."""
    from paper_2607_04749_b200.host_pipeline import HostMigration
    # pinning the host copies is the step that can fail on one rank only (host memory): agree on it before any
    # collective, so that no rank is left waiting in a barrier
    ok, h_src, h_dst = 1.0, {}, {}
    try:
        h_src = {k: torch.empty(t.shape, dtype=t.dtype, pin_memory=True) for k, t in src.items()}
        h_dst = {k: torch.empty(t.shape, dtype=t.dtype, pin_memory=True) for k, t in dst.items()}
    except Exception:
        ok = 0.0
    if -max_over_ranks(-ok, world, dev) < 0.5:
        h_src = h_dst = None
        raise RuntimeError("pinned host buffers for the old and new shards could not be allocated on every rank")
    for k, t in src.items():
        h_src[k].copy_(t)
    torch.cuda.synchronize()
    n = max(1, min(args.steps, args.e2e_steps))
    flags = E.ETC_ALL_STAGED if args.all_staged else E.ETC_LOCAL_DIRECT

    def leg(**kw):
        mk = lambda: HostMigration(w["model"], w["old"], w["new"], h_src, h_dst, dev, args.e2e_staging, flags, **kw)
        warm = mk(); warm.run(); barrier()
        hm = mk()
        del warm
        barrier()
        for _ in range(n):
            plan = hm.run()
        barrier()
        ms = max_over_ranks(hm.begin.elapsed_time(hm.done) / n, world, dev)
        return {"value": job_value(world, hbm_bytes, ms), "unit": UNIT, "ms_per_step": ms, "steps": n,
                "h2d_bytes_per_step": hm.h2d_bytes, "d2h_bytes_per_step": hm.d2h_bytes,
                "pcie_GBs_each_way": [hm.h2d_bytes / ms / 1e6, hm.d2h_bytes / ms / 1e6],
                "rounds": len(plan.rounds), "staging_bytes": args.e2e_staging}

    out = leg(zero_copy=True)
    out["note"] = ("zero-copy: pinned host old shards -> [copy kernels read them over PCIe, only the bytes their chunks "
                   "name] -> whole path (kind-major rounds, staging on the device) -> [copy kernels write over PCIe] -> "
                   "pinned host new shards; h2d / d2h = bytes the kernels read from / write to host memory")
    for key, kw, note in (
            ("dma_full_upload", dict(d_src=src, d_dst=dst),
             "cudaMemcpyAsync of EVERY old shard byte -> rounds on device buffers -> cudaMemcpyAsync of the new shards; "
             "upload, rounds and download of different kinds overlap on three streams"),
            ("dma_needed_only", dict(d_src=src, d_dst=dst, needed_only=True),
             "plan first, then cudaMemcpy2DAsync of only the source regions the plan's slices read (etc_upload_sources)")):
        if world > 1:
            continue                                            # context legs: single-GPU runs only
        try:
            out[key] = leg(**kw)
            out[key]["note"] = note
        except Exception as ex:
            out[key] = {"error": repr(ex)[:200]}
    return out


def chunked(E, torch, w, dev, src, lay_old, lay_new, cap):
    """(f2) device-resident state chunking with eager release: DESTROYS `src` (run last).  Reports the peak of live
    bytes relative to the old state, the quantity of the paper's Fig. 12 (1.25x there)."""
    from paper_2607_04749_b200.host_pipeline import migrate_chunked
    stream = torch.cuda.current_stream()
    ov, _, _ = E.etc_cost_matrix(lay_old, lay_new)
    dm, _ = E.etc_sketch(ov)
    plan = E.etc_plan_create(lay_old, lay_new, dm, E.ETC_KIND_MAJOR)
    torch.cuda.synchronize()
    torch.cuda.reset_peak_memory_stats(dev)
    base = torch.cuda.memory_allocated(dev)
    old_bytes = sum(t.numel() for t in src.values())
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    dst, info = migrate_chunked(plan, lay_new, src, cap, dev)
    b.record(stream)
    torch.cuda.synchronize()
    ms = a.elapsed_time(b)
    peak_alloc = torch.cuda.max_memory_allocated(dev) - (base - old_bytes)
    return {"staging_cap_bytes": cap, "rounds": info["rounds"], "ms": ms, "GBs": plan.stats.hbm_bytes / ms / 1e6,
            "peak_live_over_old": info["peak_live_bytes"] / info["old_bytes"],
            "torch_peak_allocated_over_old": peak_alloc / old_bytes,
            "all_at_once_over_old": (info["old_bytes"] + info["new_bytes"] + plan.stats.staging_bytes) / info["old_bytes"],
            "note": "includes on-demand allocation of the new buffers (torch caching allocator) inside the timed region"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", default="c2", help="workload: c1..c5 (BASELINE.json configs[0..4]); default configs[1]")
    ap.add_argument("--all-staged", action="store_true", help="ETC_ALL_STAGED: every slice goes through pack/unpack")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=6)
    ap.add_argument("--e2e-staging", type=int, default=1 << 30, help="staging bound (bytes) of the e2e / chunked legs")
    ap.add_argument("--ref-elems", type=int, default=48_000_000, help="--impl reference: oracle sample (elements) per step")
    ap.add_argument("--cpu-elems", type=int, default=300_000_000, help="cpu_baseline leg: oracle sample (elements), ~10 s")
    args = ap.parse_args()
    from etc_inputs import workload
    w = workload(args.config)
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_cuda(args, w)


if __name__ == "__main__":
    main()
