#!/usr/bin/env python
"""bench.py — DASH 4D hash encoder, fwd + bwd, on B200 (metric: BASELINE.json "4D hash encode fwd+bwd
Mqueries/s at 1 B200; achieved GB/s vs HBM peak").

One STEP = one pass of the whole hot path over one batch of synthetic queries:
    zero the table gradient  ->  dash_hash4d_fwd  ->  dash_hash4d_bwd
all through the C ABI (include/dash_hash4d.h), on one stream.  Default workload: BASELINE.json configs[3]
("C4": N=1M, L=16, F=4, T=2^21, fp16 table) — the config the north_star's roofline bar is quoted on.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C1..C5] [--impl reference]

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/) instead — the only
place besides the cpu_baseline leg where this file executes oracle code.
N > 1: replicas (the path needs no exchange step) — every rank runs the same workload on its
own GPU, value = N * queries / max-over-ranks time, scaling "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from dash_inputs import CONFIGS, make_workload  # noqa: E402

METRIC = "4d_hash_encode_fwd_bwd_mqueries_per_s"
UNIT = "Mqueries/s"
REFERENCE_SAMPLE_QUERIES = 100_000     # per step of --impl reference
REFERENCE_BUDGET_SECONDS = 240.0       # --impl reference stops timing further steps after this long
CPU_BASELINE_QUERIES = 1_000_000       # bounded sample of the cpu_baseline leg (3 runs, ~10 s of CPU work)
CPU_BASELINE_QUERIES_1T = 100_000      # ... of its single-thread run


# ------------------------------------------------------------------------------------------ helpers

def algorithmic_bytes(enc, has_index: bool):
    """SURVEY.md §8d / DESIGN.md §6: bytes the method itself must move, per query and fixed."""
    s_table = 2 if enc.table_dtype == "fp16" else 4
    inp = 20 if has_index else 16
    fwd = inp + 16 * enc.L * enc.F * s_table + 4 * enc.L * enc.F
    bwd = inp + 4 * enc.L * enc.F + 16 * enc.L * enc.F * 4
    zero = 4 * enc.L * enc.T * enc.F
    return fwd, bwd, zero


def profiled_traffic(config: str, key: str):
    """ncu dram__bytes_read.sum + dram__bytes_write.sum, from the committed summary profiles/traffic.json —
    written by `python -m paper_2507_19141_b200.ncu_summary` from the raw-page CSV of the ncu capture it names.
    Keys: "fwd_call", "bwd_call" (all launches of one C-ABI call), "step"."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as fh:
            return float(json.load(fh)[config][key])
    except Exception:  # noqa: BLE001
        return None


def compulsory_bytes(dh, torch, cfg, enc, N, xyz, t, index):
    """B_min of SURVEY.md §8d: HBM bytes an ideal cache would still move.  fwd: query inputs once + every TOUCHED
    32-byte table sector once + `out` once; bwd: query inputs + `dout` once + the whole gradient buffer written
    once.  The touched sectors are counted exactly, from the library's own corner indices (dash_hash4d_indices)."""
    s_table = 2 if enc.table_dtype == "fp16" else 4
    slot_bytes = enc.F * s_table
    n_sectors = (enc.L * enc.T * slot_bytes + 31) // 32
    seen = torch.zeros(n_sectors, dtype=torch.bool, device=xyz.device)
    level_base = (torch.arange(enc.L, device=xyz.device, dtype=torch.int64) * enc.T).view(1, enc.L, 1)
    chunk = 1 << 16
    rows_seen = torch.zeros(xyz.shape[0], dtype=torch.bool, device=xyz.device) if index is not None else None
    for a in range(0, N, chunk):
        z = min(N, a + chunk)
        if index is not None:
            idx, _ = dh.dash_hash4d_indices(cfg, xyz, t[a:z], index=index[a:z], want_weights=False)
            rows_seen[index[a:z].long()] = True
        else:
            idx, _ = dh.dash_hash4d_indices(cfg, xyz[a:z], t[a:z], want_weights=False)
        slot = idx.long() & 0xffffffff
        seen[((slot + level_base) * slot_bytes) // 32] = True
    table_touched = int(seen.sum()) * 32
    if index is not None:
        inputs = N * 4 + N * 4 + int(rows_seen.sum()) * 12          # index + t + touched xyz rows
    else:
        inputs = N * 16
    row = enc.L * enc.F * 4
    fwd = inputs + table_touched + N * row
    bwd = inputs + N * row + enc.L * enc.T * enc.F * 4
    return {"fwd": fwd, "bwd": bwd, "step": fwd + bwd, "table_sectors_touched_bytes": table_touched}


def time_step_of(dh, torch, wl, peak, l2_bytes, sort_coarse: bool, steps: int = 20):
    """The timed step of run_cuda (ZERO_GRAD backward, SORT_COARSE forward, ORDER_READY backward, one shared workspace)
    on another workload `wl`, in the same launch configuration, `steps` times after 3 warm-up steps.  CUDA events per
    step; a 2 x L2 buffer is written between steps (outside the timed segments) when the working set is smaller than that."""
    enc, N = wl.spec.enc, wl.N
    flags = dh.FLAG_DENSE_COARSE | dh.FLAG_ZERO_GRAD | (dh.FLAG_SORT_COARSE if sort_coarse else 0)
    cfg = dh.config_from_params(enc, flags=flags)
    cfg_bwd = dh.with_flags(cfg, flags | dh.FLAG_ORDER_READY) if sort_coarse else cfg
    need = dh.dash_hash4d_workspace_bytes(cfg, N, dh.OP_BWD)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda") if need else None
    to_dev = lambda a: None if a is None else torch.from_numpy(a).cuda()
    xyz, t, index, table, dout = to_dev(wl.xyz), to_dev(wl.t), to_dev(wl.index), to_dev(wl.table), to_dev(wl.dout)
    out = torch.empty((N, enc.L * enc.F), dtype=torch.float32, device="cuda")
    dtable = torch.empty((enc.L, enc.T, enc.F), dtype=torch.float32, device="cuda")
    nbytes = lambda x: 0 if x is None else x.numel() * x.element_size()
    working_set = sum(nbytes(x) for x in (xyz, t, table, dout, out, dtable))
    flush = torch.empty(2 * l2_bytes, dtype=torch.uint8, device="cuda") if working_set < 2 * l2_bytes else None
    ev = lambda: torch.cuda.Event(enable_timing=True)
    seg = []
    for i in range(steps + 3):
        if flush is not None:
            flush.zero_()
        m = [ev(), ev(), ev()]
        m[0].record()
        dh.dash_hash4d_fwd(cfg, xyz, t, table, out=out, index=index, workspace=ws)
        m[1].record()
        dh.dash_hash4d_bwd(cfg_bwd, xyz, t, dout, dtable, index=index, workspace=ws)
        m[2].record()
        if i >= 3:
            seg.append(m)
    torch.cuda.synchronize()
    ms_fwd = sum(m[0].elapsed_time(m[1]) for m in seg) / steps
    ms_bwd = sum(m[1].elapsed_time(m[2]) for m in seg) / steps
    ms = sum(m[0].elapsed_time(m[2]) for m in seg) / steps
    b_fwd, b_bwd, b_zero = algorithmic_bytes(enc, index is not None)
    step_bytes = (b_fwd + b_bwd) * N + b_zero
    return {"N": N, "ms_per_step": ms, "Mqueries_per_s": N / (ms * 1e-3) / 1e6, "fwd_ms": ms_fwd, "bwd_ms": ms_bwd,
            "step_frac_of_hbm_peak": step_bytes / (ms * 1e-3) / 1e9 / peak,
            "sorted_path_taken": bool(sort_coarse and need), "steps": steps,
            "l2_flush_between_steps": flush is not None}


def measured_hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:  # noqa: BLE001
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={self.FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:  # noqa: BLE001
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:  # noqa: BLE001
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for name, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm), "reasons": sorted(reasons)}


def time_oracle(wl, n_queries: int, repeats: int = 1):
    """Oracle fwd+bwd on the first n_queries queries of the workload, as it stands.  -> (seconds, threads)."""
    import oracle
    enc = wl.spec.enc
    cfg = oracle.config_from_params(enc)
    n = min(n_queries, wl.N)
    t = np.ascontiguousarray(wl.t[:n])
    dout = np.ascontiguousarray(wl.dout[:n])
    if wl.index is not None:
        xyz, index = wl.xyz, np.ascontiguousarray(wl.index[:n])
    else:
        xyz, index = np.ascontiguousarray(wl.xyz[:n]), None
    best = float("inf")
    for _ in range(repeats):
        t0 = time.perf_counter()
        oracle.oracle_fwd(cfg, n, xyz, t, wl.table, index=index)
        oracle.oracle_bwd(cfg, n, xyz, t, dout, index=index)
        best = min(best, time.perf_counter() - t0)
    return best, n, oracle.threads()


# ------------------------------------------------------------------------------------------ reference arm

def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = make_workload(args.config)
    times = []
    n = threads = 0
    began = time.perf_counter()
    for i in range(args.warmup + args.steps):
        sec, n, threads = time_oracle(wl, REFERENCE_SAMPLE_QUERIES)
        if i >= args.warmup:
            times.append(sec)
        # the oracle is deliberately slow: never let this arm run longer than a few minutes
        if times and time.perf_counter() - began > REFERENCE_BUDGET_SECONDS:
            break
    sec = sum(times) / len(times)
    value = n / sec / 1e6
    enc = wl.spec.enc
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": len(times), "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "steps_requested": args.steps,
        "config": {"workload": f"{args.config}: first {n} of {wl.N} queries per step, L={enc.L} F={enc.F} "
                               f"T=2^{enc.T.bit_length() - 1} table {enc.table_dtype}",
                   "queries_per_step": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": f"first {n} queries of {args.config}, fwd+bwd, mean of {len(times)} steps"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------ launcher

def launch_replicas(args):
    """`python bench.py --gpus N` without torchrun: re-exec this command under torch.distributed.run with N ranks
    on this node (one process per GPU).  Refuses N above the number of visible devices."""
    import socket
    if args.impl != "plumbing":
        import torch
        have = torch.cuda.device_count()
        if args.gpus > have:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but only {have} CUDA device(s) are visible")
    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        port = sock.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")            # communicator lines: the driver's rank check reads them
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


def run_plumbing(args):
    """Launcher self-test (CPU, gloo): every rank joins, barriers, contributes a fake per-rank time; rank 0 prints
    the rank count it really saw.  No kernel runs and no number here is a measurement."""
    from paper_2507_19141_b200.replicas import Replicas
    rep = Replicas(backend="gloo")
    rep.barrier()
    ms = rep.max_over_ranks(1.0 + rep.rank)
    if rep.is_reporter:
        print(json.dumps({"impl": "plumbing", "n_gpus": rep.world, "max_over_ranks_ms": ms,
                          "config": {"parallelism": f"replicas x{rep.world}"}}), flush=True)
    rep.close()
    return 0


# ------------------------------------------------------------------------------------------ ceilings / sweeps

def run_ceilings(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --ceilings: no CUDA device")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    from paper_2507_19141_b200 import ceilings
    res = ceilings.full()
    if args.md:
        with open(args.md, "w") as fh:
            fh.write(ceilings.to_markdown(res, "python bench.py --ceilings --md " + args.md))
    print(json.dumps({"ceilings": res}), flush=True)
    return 0


def run_group_sweep(args):
    """ms per call of fwd, zero+bwd and bwd(ZERO_GRAD) for G = 1..16 on --config (reproduces profiles/group_sweep_*)."""
    import torch
    import paper_2507_19141_b200 as dh
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --sweep-groups: no CUDA device")
    wl = make_workload(args.config)
    enc, N = wl.spec.enc, wl.N
    cfg = dh.config_from_params(enc, flags=dh.FLAG_DENSE_COARSE)
    cfg_z = dh.config_from_params(enc, flags=dh.FLAG_DENSE_COARSE | dh.FLAG_ZERO_GRAD)
    to_dev = lambda a: None if a is None else torch.from_numpy(a).cuda()
    xyz, t, index, table, dout = (to_dev(a) for a in (wl.xyz, wl.t, wl.index, wl.table, wl.dout))
    out = torch.empty((N, enc.L * enc.F), dtype=torch.float32, device="cuda")
    dtable = torch.empty((enc.L, enc.T, enc.F), dtype=torch.float32, device="cuda")

    def timed(fn, iters=20):
        for _ in range(3):
            fn()
        a, z = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(iters):
            fn()
        z.record(); z.synchronize()
        return a.elapsed_time(z) / iters

    rows = {}
    for g in (1, 2, 4, 8, 16):
        dh.dash_hash4d_set_debug(dh.DEBUG_FWD_GROUP, g)
        dh.dash_hash4d_set_debug(dh.DEBUG_BWD_GROUP, g)
        rows[f"G={g}"] = {
            "fwd_ms": timed(lambda: dh.dash_hash4d_fwd(cfg, xyz, t, table, out=out, index=index)),
            "zero+bwd_ms": timed(lambda: (dh.dash_hash4d_zero(cfg, dtable),
                                          dh.dash_hash4d_bwd(cfg, xyz, t, dout, dtable, index=index))),
            "bwd_zero_grad_ms": timed(lambda: dh.dash_hash4d_bwd(cfg_z, xyz, t, dout, dtable, index=index)),
        }
    dh.dash_hash4d_set_debug(dh.DEBUG_FWD_GROUP, 0)
    dh.dash_hash4d_set_debug(dh.DEBUG_BWD_GROUP, 0)
    rows["library_choice"] = {
        "fwd_ms": timed(lambda: dh.dash_hash4d_fwd(cfg, xyz, t, table, out=out, index=index)),
        "bwd_zero_grad_ms": timed(lambda: dh.dash_hash4d_bwd(cfg_z, xyz, t, dout, dtable, index=index)),
    }
    print(json.dumps({"group_sweep": {"config": args.config, "rows": rows}}), flush=True)
    return 0


def run_sorted_experiment(args):
    """VERDICT r1 item 4 / SURVEY §7 step 7, decided on kernels: the hand-written counting sort
    (dash_hash4d_sort_queries) is timed by itself, then fwd and bwd(ZERO_GRAD) are timed on the queries in the given
    order and in the sorted order (same kernels, `index` = the sorted order; t / dout permuted outside the timing)."""
    import torch
    import paper_2507_19141_b200 as dh
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --sorted-experiment: no CUDA device")
    out_rows = {}
    for name in args.config.split(","):
        wl = make_workload(name)
        enc, N = wl.spec.enc, wl.N
        cfg = dh.config_from_params(enc, flags=dh.FLAG_DENSE_COARSE | dh.FLAG_ZERO_GRAD)
        to_dev = lambda a: None if a is None else torch.from_numpy(a).cuda()
        xyz, t, index, table, dout = (to_dev(a) for a in (wl.xyz, wl.t, wl.index, wl.table, wl.dout))
        out = torch.empty((N, enc.L * enc.F), dtype=torch.float32, device="cuda")
        dtable = torch.empty((enc.L, enc.T, enc.F), dtype=torch.float32, device="cuda")

        def timed(fn, iters=20):
            for _ in range(3):
                fn()
            a, z = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(iters):
                fn()
            z.record(); z.synchronize()
            return a.elapsed_time(z) / iters

        row = {"N": N,
               "fwd_ms": timed(lambda: dh.dash_hash4d_fwd(cfg, xyz, t, table, out=out, index=index)),
               "bwd_ms": timed(lambda: dh.dash_hash4d_bwd(cfg, xyz, t, dout, dtable, index=index))}
        for bits in (5, 6, 7):
            order = torch.empty((N,), dtype=torch.int32, device="cuda")
            ws = torch.empty(max(16, dh.binding._load().dash_hash4d_sort_workspace_bytes(N, bits)), dtype=torch.uint8,
                             device="cuda")
            sort_ms = timed(lambda: dh.dash_hash4d_sort_queries(xyz, index=index, bits=bits, N=N, order=order,
                                                                workspace=ws))
            o64 = order.long()
            index_s = (index[o64] if index is not None else order).contiguous()
            t_s, dout_s = t[o64].contiguous(), dout[o64].contiguous()
            row[f"bits={bits}"] = {
                "sort_ms": sort_ms,
                "fwd_sorted_ms": timed(lambda: dh.dash_hash4d_fwd(cfg, xyz, t_s, table, out=out, index=index_s)),
                "bwd_sorted_ms": timed(lambda: dh.dash_hash4d_bwd(cfg, xyz, t_s, dout_s, dtable, index=index_s)),
            }
            r = row[f"bits={bits}"]
            r["step_delta_ms_if_sorted_each_step"] = (r["sort_ms"] + r["fwd_sorted_ms"] + r["bwd_sorted_ms"]
                                                      - row["fwd_ms"] - row["bwd_ms"])
        out_rows[name] = row
    print(json.dumps({"sorted_experiment": out_rows}), flush=True)
    return 0


# ------------------------------------------------------------------------------------------ CUDA arm

def run_cuda(args):
    import torch
    import paper_2507_19141_b200 as dh

    from paper_2507_19141_b200.replicas import Replicas

    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
    torch.cuda.set_device(local)
    rep = Replicas(backend="nccl", device=torch.device("cuda", local))
    world, rank = rep.world, rep.rank

    debug_keys = {"fwd_group": dh.DEBUG_FWD_GROUP, "bwd_group": dh.DEBUG_BWD_GROUP,
                  "smooth_group": dh.DEBUG_SMOOTH_GROUP, "deform_path": dh.DEBUG_DEFORM_PATH,
                  "bwd_variant": dh.DEBUG_BWD_VARIANT,
                  "bwd_coarse_levels": dh.DEBUG_BWD_COARSE_LEVELS, "bwd_run_chunk": dh.DEBUG_BWD_RUN_CHUNK,
                  "fwd_ordered_levels": dh.DEBUG_FWD_ORDERED_LEVELS, "sort_key_bits": dh.DEBUG_SORT_KEY_BITS}
    for item in args.set_debug:
        key, _, val = item.partition("=")
        dh.dash_hash4d_set_debug(debug_keys[key], int(val))

    wl = make_workload(args.config)
    enc, N = wl.spec.enc, wl.N
    flags = dh.FLAG_DENSE_COARSE | (dh.FLAG_ZERO_GRAD if args.zero_grad_fused else 0)
    if args.sort_coarse:
        flags |= dh.FLAG_SORT_COARSE
    cfg = dh.config_from_params(enc, flags=flags)
    # SORT_COARSE: the forward sorts the queries by coarse cell, the backward of the same step reuses that order
    cfg_bwd = dh.with_flags(cfg, flags | dh.FLAG_ORDER_READY) if args.sort_coarse else cfg
    bwd_ws_bytes = dh.dash_hash4d_workspace_bytes(cfg, N, dh.OP_BWD)
    bwd_ws = torch.empty(bwd_ws_bytes, dtype=torch.uint8, device="cuda") if bwd_ws_bytes else None
    to_dev = lambda a: None if a is None else torch.from_numpy(a).cuda()
    xyz, t, index = to_dev(wl.xyz), to_dev(wl.t), to_dev(wl.index)
    table, dout = to_dev(wl.table), to_dev(wl.dout)
    out = torch.empty((N, enc.L * enc.F), dtype=torch.float32, device="cuda")
    dtable = torch.empty((enc.L, enc.T, enc.F), dtype=torch.float32, device="cuda")

    ev = lambda: torch.cuda.Event(enable_timing=True)

    nbytes = lambda x: 0 if x is None else x.numel() * x.element_size()
    ws_bytes = nbytes(table) + nbytes(dtable) + nbytes(out) + nbytes(dout) + nbytes(xyz) + nbytes(t)
    l2_bytes = torch.cuda.get_device_properties(local).L2_cache_size
    # timing hygiene: inputs larger than L2 (C3-C5), else write a buffer of 2 x L2 between iterations
    flush = torch.empty(2 * l2_bytes, dtype=torch.uint8, device="cuda") if ws_bytes < 2 * l2_bytes else None

    def step(marks=None):
        if flush is not None:
            flush.zero_()
        if marks is not None:
            marks[0].record()
        if not args.zero_grad_fused:
            dh.dash_hash4d_zero(cfg, dtable)
        if marks is not None:
            marks[1].record()
        dh.dash_hash4d_fwd(cfg, xyz, t, table, out=out, index=index, workspace=bwd_ws)
        if marks is not None:
            marks[2].record()
        dh.dash_hash4d_bwd(cfg_bwd, xyz, t, dout, dtable, index=index, workspace=bwd_ws)
        if marks is not None:
            marks[3].record()

    barrier = rep.barrier

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    marks = [[ev() for _ in range(4)] for _ in range(args.steps)]
    start, stop = ev(), ev()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler is not None:
        time.sleep(0.25)                       # let the sampler come up before the timed region
    dh.dash_hash4d_launch_count(reset=True)
    barrier()
    start.record()
    for i in range(args.steps):
        step(marks[i])
    stop.record()
    barrier()
    launches = dh.dash_hash4d_launch_count()
    clocks = sampler.stop() if sampler is not None else None
    seg = np.array([[m[0].elapsed_time(m[1]), m[1].elapsed_time(m[2]), m[2].elapsed_time(m[3])]
                    for m in marks])
    ms_zero, ms_fwd, ms_bwd = (float(v) for v in seg.mean(0))
    if flush is None:
        ms_total = start.elapsed_time(stop)                      # K back-to-back steps, one event pair
    else:
        ms_total = float(np.array([m[0].elapsed_time(m[3]) for m in marks]).sum())   # flushes excluded
    ms_step = rep.max_over_ranks(ms_total) / args.steps

    # ---- roofline of the dominant kernel (the bwd scatter), live CUDA-event durations
    b_fwd, b_bwd, b_zero = algorithmic_bytes(enc, index is not None)
    peak, peak_src = measured_hbm_peak()
    dominant = "bwd" if ms_bwd >= ms_fwd else "fwd"
    dom_bytes = (b_bwd if dominant == "bwd" else b_fwd) * N
    if dominant == "bwd" and args.zero_grad_fused:
        dom_bytes += b_zero
    dom_ms = ms_bwd if dominant == "bwd" else ms_fwd
    kernel_name = f"hash4d_{dominant}_kernel"
    sorted_path = bool(args.sort_coarse) and bwd_ws is not None
    if dominant == "bwd" and args.zero_grad_fused:
        kernel_name = "hash4d_bwd_kernel+zero_kernel (one dash_hash4d_bwd call, ZERO_GRAD)"
        if sorted_path:
            kernel_name = ("hash4d_bwd_kernel+hash4d_bwd_runs_kernel+zero_kernel (one dash_hash4d_bwd call, ZERO_GRAD, "
                           "SORT_COARSE with the forward's order)")
    achieved = dom_bytes / (dom_ms * 1e-3) / 1e9
    step_bytes = (b_fwd + b_bwd) * N + b_zero
    roofline = {
        "bound": "hbm", "kernel": kernel_name, "achieved": achieved, "peak": peak,
        "unit": "GB/s", "frac": achieved / peak,
        "traffic": args.traffic_bytes if args.traffic_bytes is not None
        else profiled_traffic(args.config, "bwd_call" if dominant == "bwd" else "fwd_call"),
        "peak_source": peak_src,
        "algorithmic_bytes_per_launch": dom_bytes,
        "step": {"algorithmic_bytes": step_bytes, "achieved": step_bytes / (ms_step * 1e-3) / 1e9,
                 "frac": step_bytes / (ms_step * 1e-3) / 1e9 / peak,
                 "ms": {"zero": ms_zero, "fwd": ms_fwd, "bwd": ms_bwd}},
    }

    # `achieved` / `frac` divide the ALGORITHMIC bytes (one access per corner per query and level) by the
    # time.  On the sorted path the kernels issue fewer accesses than that count (lines shared between neighbouring
    # lanes, runs merged in registers), so the figure is a work-equivalent throughput, not HBM utilisation; the DRAM
    # bytes ncu saw for the same call, over the same live time, are given beside it.
    roofline["achieved_kind"] = ("algorithmic bytes / time" if not sorted_path else
                                 "algorithmic bytes / time = work-equivalent throughput: SORT_COARSE issues fewer "
                                 "accesses than the algorithmic count; see `dram` for the profiled DRAM bytes")
    if roofline["traffic"]:
        dram_gbs = roofline["traffic"] / (dom_ms * 1e-3) / 1e9
        roofline["dram"] = {"bytes_per_call_ncu": roofline["traffic"], "GBps": dram_gbs, "frac": dram_gbs / peak,
                            "note": "profiles/traffic.json bytes (ncu, cold-cache replay) over the live CUDA-event time of "
                                    "the same call; the per-call write split under-counts late write-backs, so the step "
                                    "figure (traffic_step) is the one to quote"}

    # ---- the stricter figures of SURVEY.md §8d, beside the algorithmic-bytes fraction
    bmin = compulsory_bytes(dh, torch, dh.config_from_params(enc, flags=dh.FLAG_DENSE_COARSE), enc, N, xyz, t, index)
    roofline["b_min"] = {"bytes": bmin, "step_GBps": bmin["step"] / (ms_step * 1e-3) / 1e9,
                         "step_frac_of_hbm_peak": bmin["step"] / (ms_step * 1e-3) / 1e9 / peak,
                         "note": "compulsory HBM bytes with an ideal cache; touched table sectors counted exactly"}
    roofline["traffic_step"] = profiled_traffic(args.config, "step")
    roofline["traffic_fwd_call"] = profiled_traffic(args.config, "fwd_call")
    from paper_2507_19141_b200 import ceilings as ceil_mod
    ceil = ceil_mod.quick()
    lane_ops = 16 * enc.L * N                                    # corner gathers (fwd) / corner reductions (bwd)
    red_key = "red16_pair_xcorner_L2" if enc.F * 4 >= 16 else "red8_pair_xcorner_L2"
    roofline["ceilings"] = {
        "gather_G_lane_loads_per_s": ceil["gather8_pair_xcorner_L2"]["G_lane_ops_per_s"],
        "red_G_lane_reds_per_s": ceil[red_key]["G_lane_ops_per_s"], "red_kernel": red_key,
        "fwd_G_lane_loads_per_s": lane_ops / (ms_fwd * 1e-3) / 1e9,
        "bwd_G_lane_reds_per_s": lane_ops / (ms_bwd * 1e-3) / 1e9,
        "fwd_frac_of_gather_ceiling": lane_ops / (ms_fwd * 1e-3) / 1e9 / ceil["gather8_pair_xcorner_L2"]["G_lane_ops_per_s"],
        "bwd_frac_of_red_ceiling": lane_ops / (ms_bwd * 1e-3) / 1e9 / ceil[red_key]["G_lane_ops_per_s"],
        "note": "microbenchmarks of include/dash_ceilings.h run in this process (L2-resident 32 MiB footprint, "
                "x-corner lane pairs, 8 accesses in flight per lane, RANDOM addresses); bwd time includes the fused zero "
                "passes, fwd time the coarse sort; with sort_coarse the path shares lines between neighbouring lanes and "
                "merges reductions, so a fraction above 1 means fewer accesses reach L1 / L2 than the method names",
    }

    # ---- deterministic mode (DETERMINISTIC_BWD, 64-bit fixed point): what it costs on this workload
    det_ms = None
    if args.deterministic_leg:
        cfg_det = dh.config_from_params(enc, flags=flags | dh.FLAG_DETERMINISTIC_BWD)
        need = dh.dash_hash4d_workspace_bytes(cfg_det, N, dh.OP_BWD)
        try:
            ws_det = torch.empty(need, dtype=torch.uint8, device="cuda")
            run_det = lambda: dh.dash_hash4d_bwd(cfg_det, xyz, t, dout, dtable, index=index, workspace=ws_det)
            run_det(); run_det()
            torch.cuda.synchronize()
            d0, d1 = ev(), ev()
            d0.record()
            for _ in range(5):
                run_det()
            d1.record()
            torch.cuda.synchronize()
            det_ms = d0.elapsed_time(d1) / 5
            del ws_det
        except torch.OutOfMemoryError:
            det_ms = None
    roofline["deterministic_bwd_ms"] = det_ms

    # ---- what the coarse sort costs inside the forward call: the same forward on the order already in the workspace
    if sorted_path:
        def avg_ms(fn, iters=20):
            fn(); fn()
            torch.cuda.synchronize()
            a, b = ev(), ev()
            a.record()
            for _ in range(iters):
                fn()
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b) / iters
        with_sort = avg_ms(lambda: dh.dash_hash4d_fwd(cfg, xyz, t, table, out=out, index=index, workspace=bwd_ws))
        ready = avg_ms(lambda: dh.dash_hash4d_fwd(cfg_bwd, xyz, t, table, out=out, index=index, workspace=bwd_ws))
        roofline["step"]["ms"]["fwd_sort_part"] = with_sort - ready

    # ---- e2e: HOST (pinned) buffers through the binding's *_host calls, copies inside the timed region
    pin = lambda a: None if a is None else torch.from_numpy(a).pin_memory()
    xyz_h, t_h, index_h, dout_h = pin(wl.xyz), pin(wl.t), pin(wl.index), pin(wl.dout)
    out_h = torch.empty((N, enc.L * enc.F), dtype=torch.float32).pin_memory()
    dtable_h = torch.empty((enc.L, enc.T, enc.F), dtype=torch.float32).pin_memory()
    host_step = dh.HostStep(cfg)

    def e2e_step():
        host_step(xyz_h, t_h, table, dout_h, out_h, dtable_h, index_h=index_h)

    e2e_steps = max(3, min(args.steps, 10))
    e2e_step(); e2e_step()
    barrier()
    e0, e1 = ev(), ev()
    e0.record()
    for _ in range(e2e_steps):
        e2e_step()
    e1.record()
    barrier()
    e2e_ms = rep.max_over_ranks(e0.elapsed_time(e1) / e2e_steps)
    h2d = nbytes(xyz_h) + nbytes(t_h) + nbytes(index_h) + nbytes(dout_h)
    d2h = nbytes(out_h) + nbytes(dtable_h)

    # ---- extras (information only, not part of the metric): the NEXT-row calls on the same workload
    extras = None
    if args.extras:
        def timed(fn, iters=10):
            fn(); fn()
            torch.cuda.synchronize()
            a, b = ev(), ev()
            a.record()
            for _ in range(iters):
                fn()
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b) / iters
        dq = torch.empty((N, 4), dtype=torch.float32, device="cuda")
        loss = torch.empty((N,), dtype=torch.float32, device="cuda")
        cfg_acc = dh.config_from_params(enc, flags=dh.FLAG_DENSE_COARSE)
        gen = torch.Generator(device="cuda"); gen.manual_seed(1234)
        cfg_x = dh.with_flags(cfg, flags & ~dh.FLAG_SORT_COARSE)   # the extras time the calls without the coarse sort
        extras = {"bwd_input_ms": timed(lambda: dh.dash_hash4d_bwd_input(cfg_x, xyz, t, table, dout, dq=dq,
                                                                           index=index))}
        if sorted_path:   # the coordinate gradient walking the order the step's forward left in the workspace
            extras["bwd_input_ms_sort_coarse_order_ready"] = timed(
                lambda: dh.dash_hash4d_bwd_input(cfg_bwd, xyz, t, table, dout, dq=dq, index=index, workspace=bwd_ws))
        for delta in (1e-4, 1e-3, 1e-2):
            eps = (torch.rand((N, 4), device="cuda", generator=gen) * 2 - 1) * delta
            extras[f"smooth_loss+grad_ms(eps=U(-{delta:g},{delta:g}))"] = timed(
                lambda: dh.dash_hash4d_smooth(cfg_acc, xyz, t, eps, table, grad_scale=0.1, loss=loss,
                                              dtable=dtable, index=index))
        extras["smooth_unfused_equivalent_ms"] = 2 * (ms_fwd + ms_bwd)
        one_t = t[:1].contiguous()
        extras["fwd_one_timestamp_ms"] = timed(lambda: dh.dash_hash4d_fwd(cfg_x, xyz, one_t, table, out=out,
                                                                           index=index, t_stride=0))
        # every other BASELINE.json config's step in this bench's launch configuration (a bar per config)
        if args.config == "C4":
            extras["configs"] = {}
            for name in ("C2", "C3", "C5"):
                extras["configs"][name] = time_step_of(dh, torch, make_workload(name), peak, l2_bytes,
                                                       bool(args.sort_coarse))
            # The rule that turns the sorted path on (N*F >= 2^21, levels with Ns^3 Nt <= 2N) was fitted on clustered
            # inputs (PAPER.md:241 is the basis for clustering).  A/B on C4's encoder with C1's distribution: 1M
            # iid-uniform queries, where runs of queries in one cell are short.
            import copy
            wl_u = copy.copy(wl)
            q_u = np.random.default_rng(20).random(size=(wl.N, 4), dtype=np.float32)
            wl_u.xyz, wl_u.t, wl_u.index = np.ascontiguousarray(q_u[:, :3]), np.ascontiguousarray(q_u[:, 3]), None
            extras["uniform_1M_on_C4_encoder"] = {
                "sort_coarse_1": time_step_of(dh, torch, wl_u, peak, l2_bytes, True),
                "sort_coarse_0": time_step_of(dh, torch, wl_u, peak, l2_bytes, False)}
            del wl_u, q_u
        # G_3D of the decomposition stage on its own workload (dash_inputs.G3D_SPEC)
        from dash_inputs import make_g3d_workload
        g3 = make_g3d_workload()
        e3 = g3.spec.enc
        cfg3 = dh.make_config(e3.L, e3.F, e3.T, e3.res_s_min, e3.res_s_max, 1, 1, e3.table_dtype,
                              flags=dh.FLAG_DENSE_COARSE | dh.FLAG_ZERO_GRAD)
        p3, tab3, dy3 = to_dev(g3.xyz), to_dev(g3.table), to_dev(g3.dout)
        out3 = torch.empty((g3.N, e3.L * e3.F), dtype=torch.float32, device="cuda")
        dt3 = torch.empty((e3.L, e3.T, e3.F), dtype=torch.float32, device="cuda")
        t_zero = torch.zeros(1, device="cuda")
        extras["g3d"] = {
            "workload": f"N={g3.N} points, L={e3.L} F={e3.F} T=2^{e3.T.bit_length() - 1}, {e3.res_s_min}->{e3.res_s_max}",
            "fwd_ms": timed(lambda: dh.dash_hash3d_fwd(cfg3, p3, tab3, out=out3)),
            "bwd_ms": timed(lambda: dh.dash_hash3d_bwd(cfg3, p3, dy3, dt3)),
            "fwd_ms_via_4d_kernels_nt1_t0": timed(lambda: dh.dash_hash4d_fwd(cfg3, p3, t_zero, tab3, out=out3,
                                                                               t_stride=0)),
            "bwd_ms_via_4d_kernels_nt1_t0": timed(lambda: dh.dash_hash4d_bwd(cfg3, p3, t_zero, dy3, dt3,
                                                                               t_stride=0)),
        }
        # the same with SORT_COARSE: the forward sorts the points by 3D cell, the backward reuses the order
        cfg3s = dh.with_flags(cfg3, cfg3.flags | dh.FLAG_SORT_COARSE)
        cfg3r = dh.with_flags(cfg3, cfg3.flags | dh.FLAG_SORT_COARSE | dh.FLAG_ORDER_READY)
        ws3 = torch.empty(max(16, dh.dash_hash3d_workspace_bytes(cfg3s, g3.N, dh.OP_FWD)), dtype=torch.uint8, device="cuda")
        extras["g3d"]["sort_coarse"] = {
            "fwd_ms_with_sort": timed(lambda: dh.dash_hash3d_fwd(cfg3s, p3, tab3, out=out3, workspace=ws3)),
            "fwd_ms_order_ready": timed(lambda: dh.dash_hash3d_fwd(cfg3r, p3, tab3, out=out3, workspace=ws3)),
            "bwd_ms_order_ready": timed(lambda: dh.dash_hash3d_bwd(cfg3r, p3, dy3, dt3, workspace=ws3)),
        }
        del ws3
        del p3, tab3, dy3, out3, dt3
        # sparse Adam over the touched entries of the step's own gradient (dtable as the timed bwd left it)
        th32 = table.float().contiguous()
        m1, v1 = torch.zeros_like(th32), torch.zeros_like(th32)
        t16 = table if enc.table_dtype == "fp16" else None
        g_keep = dtable.clone()
        touched = int((g_keep != 0).sum())
        def adam_once():
            dtable.copy_(g_keep)
        def adam_timed(iters=5):
            tot = 0.0
            for k in range(iters + 1):
                dtable.copy_(g_keep)
                a, b = ev(), ev()
                a.record()
                dh.dash_hash4d_adam_step(cfg, th32, dtable, m1, v1, k + 1, table16=t16)
                b.record()
                torch.cuda.synchronize()
                if k:
                    tot += a.elapsed_time(b)
            return tot / iters
        ms_adam = adam_timed()
        n_el = th32.numel()
        adam_bytes = 4 * n_el + touched * (12 + 12 + 4 + (2 if t16 is not None else 0))
        extras["adam_step"] = {"ms": ms_adam, "touched_fraction": touched / n_el,
                               "algorithmic_GBps": adam_bytes / (ms_adam * 1e-3) / 1e9,
                               "frac_of_hbm_peak": adam_bytes / (ms_adam * 1e-3) / 1e9 / peak}
        del th32, m1, v1, g_keep
        # render path (Eq. 9-10): G_4D -> phi_d -> heads in one kernel, one timestamp per frame
        from dash_inputs import make_mlp_params
        extras["deform"] = {}
        for name in ("C2", "C3"):
            w2 = make_workload(name, with_dout=False)
            e2 = w2.spec.enc
            widths = [e2.L * e2.F, 128, 128, 10]
            cfg2 = dh.config_from_params(e2, flags=dh.FLAG_DENSE_COARSE)
            mlp = dh.make_mlp_config(widths)
            x2, tab2 = to_dev(w2.xyz), to_dev(w2.table)
            one = to_dev(w2.t[:1].copy())
            prm = to_dev(make_mlp_params(11, widths))
            o2 = torch.empty((w2.N, 10), dtype=torch.float32, device="cuda")
            f2 = torch.empty((w2.N, e2.L * e2.F), dtype=torch.float32, device="cuda")
            ws2 = torch.empty(w2.N * e2.L * e2.F * 4, dtype=torch.uint8, device="cuda")
            row = {"workload": f"{name}: N={w2.N}, one timestamp, MLP {widths}"}
            dh.dash_hash4d_set_debug(dh.DEBUG_DEFORM_PATH, 1)
            row["fused_ms"] = timed(lambda: dh.dash_deform_fwd(cfg2, mlp, x2, one, tab2, prm, out=o2, t_stride=0), 20)
            dh.dash_hash4d_set_debug(dh.DEBUG_DEFORM_PATH, 2)
            row["two_pass_ms"] = timed(lambda: dh.dash_deform_fwd(cfg2, mlp, x2, one, tab2, prm, out=o2, t_stride=0,
                                                                  workspace=ws2), 20)
            dh.dash_hash4d_set_debug(dh.DEBUG_DEFORM_PATH, 0)
            row["encoder_only_ms"] = timed(lambda: dh.dash_hash4d_fwd(cfg2, x2, one, tab2, out=f2, t_stride=0), 20)
            row["mlp_only_ms"] = timed(lambda: dh.dash_mlp_fwd(mlp, f2, prm, out=o2), 20)
            sl2 = torch.empty((e2.L, e2.T, e2.F), dtype=torch.float32, device="cuda")
            row["slice_t_ms"] = timed(lambda: dh.dash_hash4d_slice_t(cfg2, one, tab2, slice_out=sl2), 20)
            row["slice_encoder_only_ms"] = timed(lambda: dh.dash_hash4d_slice_fwd(cfg2, x2, sl2, out=f2), 20)
            row["slice_fused_ms"] = timed(lambda: dh.dash_deform_slice_fwd(cfg2, mlp, x2, sl2, prm, out=o2), 20)
            row["frame_ms_slice_path"] = row["slice_t_ms"] + row["slice_fused_ms"]
            # The Gaussians of a scene do not move between rendered frames: a spatial (Morton) order computed ONCE
            # (dash_hash4d_sort_queries) serves every frame, either as the call's index list or as the order the scene
            # is stored in.  With one timestamp per frame neighbouring lanes then share cells on every coarse level.
            order2 = dh.dash_hash4d_sort_queries(x2, bits=7)
            xs2 = x2[order2.long()].contiguous()
            row["sorted_once"] = {
                "sort_ms_once_per_scene": timed(lambda: dh.dash_hash4d_sort_queries(x2, bits=7, order=order2), 10),
                "fused_ms_index_list": timed(lambda: dh.dash_deform_fwd(cfg2, mlp, x2, one, tab2, prm, out=o2, t_stride=0,
                                                                        index=order2), 20),
                "fused_ms_stored_in_order": timed(lambda: dh.dash_deform_fwd(cfg2, mlp, xs2, one, tab2, prm, out=o2,
                                                                             t_stride=0), 20),
                "encoder_only_ms_stored_in_order": timed(lambda: dh.dash_hash4d_fwd(cfg2, xs2, one, tab2, out=f2,
                                                                                    t_stride=0), 20),
                "slice_fused_ms_stored_in_order": timed(lambda: dh.dash_deform_slice_fwd(cfg2, mlp, xs2, sl2, prm,
                                                                                         out=o2), 20),
            }
            del order2, xs2
            row["mlp_tflops"] = 2.0 * w2.N * sum(a * b for a, b in zip(widths[:-1], widths[1:])) / (
                row["mlp_only_ms"] * 1e-3) / 1e12
            # training direction (Q30): backward through the chain, and the whole deformation backward
            dy2 = torch.randn((w2.N, 10), device="cuda", generator=gen)
            dprm = torch.zeros_like(prm)
            dft = torch.empty((w2.N, e2.L * e2.F), dtype=torch.float32, device="cuda")
            row["mlp_bwd_ms"] = timed(lambda: dh.dash_mlp_bwd(mlp, f2, prm, dy2, dprm, dfeat=dft), 20)
            # forward recompute (1x) + dgrad (1x) + wgrad (1x) of every layer
            row["mlp_bwd_tflops"] = 3.0 * 2.0 * w2.N * sum(a * b for a, b in zip(widths[:-1], widths[1:])) / (
                row["mlp_bwd_ms"] * 1e-3) / 1e12
            dt2 = torch.empty((e2.L, e2.T, e2.F), dtype=torch.float32, device="cuda")
            tq = to_dev(w2.t)
            cfg2z = dh.config_from_params(e2, flags=dh.FLAG_DENSE_COARSE | dh.FLAG_ZERO_GRAD)
            wsb = torch.empty(2 * w2.N * e2.L * e2.F * 4 + 64, dtype=torch.uint8, device="cuda")
            row["deform_bwd_ms_per_query_t"] = timed(lambda: dh.dash_deform_bwd(cfg2z, mlp, x2, tq, tab2, prm, dy2, dt2,
                                                                              dprm, workspace=wsb), 20)
            del dy2, dprm, dft, dt2, wsb
            extras["deform"][name] = row
            del x2, tab2, o2, f2, ws2, sl2

    if not rep.is_reporter:
        rep.close()
        return 0

    # ---- cpu_baseline: the oracle as it stands, bounded sample, on this box's host cores
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        sec, n_s, threads = time_oracle(wl, CPU_BASELINE_QUERIES, repeats=3)
        oracle.set_threads(1)
        sec1, n_1, _ = time_oracle(wl, CPU_BASELINE_QUERIES_1T)
        oracle.set_threads(threads)
        cpu = {"value": n_s / sec / 1e6, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": f"first {n_s} of {N} queries of {args.config}, fwd+bwd, best of 3 ({sec:.2f} s)",
               "one_thread": {"value": n_1 / sec1 / 1e6, "unit": UNIT, "cores": 1,
                              "sample": f"first {n_1} queries, fwd+bwd once ({sec1:.2f} s)"}}

    value = N * world / (ms_step * 1e-3) / 1e6
    ws_mb = ws_bytes / 1e6
    l2_note = (f"working set {ws_mb:.0f} MB > 2 x L2 ({l2_bytes / 1e6:.0f} MB): no flush between iterations"
               if flush is None else
               f"working set {ws_mb:.0f} MB: a {2 * l2_bytes / 1e6:.0f} MB buffer is written between iterations "
               f"(outside the timed segments)")
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{args.config}: N={N} queries, L={enc.L} F={enc.F} T=2^{enc.T.bit_length() - 1} "
                               f"table {enc.table_dtype}, spatial {enc.res_s_min}->{enc.res_s_max}, "
                               f"temporal {enc.res_t_min}->{enc.res_t_max}; step = zero(dtable)+fwd+bwd",
                   "queries_per_step_per_gpu": N, "parallelism": f"replicas x{world}",
                   "l2": l2_note,
                   "zero_grad_fused": bool(args.zero_grad_fused),
                   "sort_coarse": sorted_path,
                   **({"debug_overrides": args.set_debug} if args.set_debug else {})},
        "roofline": roofline,
        "e2e": {"value": N * world / (e2e_ms * 1e-3) / 1e6, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms, "steps": e2e_steps},
        "gpu_launches": int(launches),
        "clocks": clocks,
    }
    if cpu is not None:
        line["cpu_baseline"] = cpu
    if extras is not None:
        line["extras"] = extras
    print(json.dumps(line), flush=True)
    rep.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="default 200 (cuda arm) / 10 (reference arm)")
    ap.add_argument("--warmup", type=int, default=None, help="default 20 (cuda arm) / 2 (reference arm)")
    ap.add_argument("--config", default="C4",
                    help="C1..C5 (BASELINE.json configs); --sorted-experiment takes a comma-separated list")
    ap.add_argument("--sorted-experiment", action="store_true",
                    help="time dash_hash4d_sort_queries and fwd / bwd in the given vs the sorted order (JSON line)")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference", "plumbing"],
                    help="cuda: the product; reference: the CPU oracle; plumbing: launcher/rank self-test on gloo "
                         "(no kernels, no measurement; tests/test_replicas_gloo.py)")
    ap.add_argument("--zero-grad-fused", type=int, default=1,
                    help="1: bwd zeroes each level group itself (DASH_HASH4D_FLAG_ZERO_GRAD)")
    ap.add_argument("--sort-coarse", type=int, default=1,
                    help="1: DASH_HASH4D_FLAG_SORT_COARSE — fwd sorts the queries by coarse 4D cell and walks them in that "
                         "order, bwd reuses the order (ORDER_READY) and merges runs on the coarse levels; the library "
                         "ignores the flag when N*F < 2^21 (C2, C3).  0: the plain path (A/B)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--extras", type=int, default=1,
                    help="1: also time bwd_input / smooth / one-timestamp fwd (information only)")
    ap.add_argument("--deterministic-leg", type=int, default=1,
                    help="1: also time dash_hash4d_bwd with DETERMINISTIC_BWD (information only)")
    ap.add_argument("--traffic-bytes", type=float, default=None,
                    help="ncu dram bytes per launch of the dominant kernel (from profiles/), else null")
    ap.add_argument("--set-debug", action="append", default=[], metavar="KEY=VALUE",
                    help="dash_hash4d_set_debug override for A/B runs, e.g. bwd_group=1, bwd_variant=2 "
                         "(keys: fwd_group bwd_group smooth_group deform_path bwd_variant bwd_coarse_levels bwd_run_chunk fwd_ordered_levels sort_key_bits)")
    ap.add_argument("--ceilings", action="store_true",
                    help="run the microbenchmarks of include/dash_ceilings.h and print their JSON line instead")
    ap.add_argument("--md", default=None, help="with --ceilings: also write the table as markdown to this path")
    ap.add_argument("--sweep-groups", action="store_true",
                    help="time fwd / bwd for every level-group size G (dash_hash4d_set_debug) and print a JSON line")
    args = ap.parse_args()
    if args.gpus < 1:
        ap.error("--gpus must be >= 1")
    if not args.sorted_experiment and args.config not in CONFIGS:
        ap.error(f"--config must be one of {sorted(CONFIGS)}")
    if args.impl in ("cuda", "plumbing") and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return launch_replicas(args)
    if "WORLD_SIZE" in os.environ and int(os.environ["WORLD_SIZE"]) != args.gpus:
        ap.error(f"--gpus {args.gpus} but the launcher started WORLD_SIZE={os.environ['WORLD_SIZE']} ranks")
    if args.impl == "plumbing":
        return run_plumbing(args)
    if args.ceilings:
        return run_ceilings(args)
    if args.sweep_groups:
        return run_group_sweep(args)
    if args.sorted_experiment:
        return run_sorted_experiment(args)
    if args.steps is None:
        args.steps = 10 if args.impl == "reference" else 200
    if args.warmup is None:
        args.warmup = 2 if args.impl == "reference" else 20
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
