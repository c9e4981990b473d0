"""Chip ceilings of the encoder's access patterns, measured by the microbenchmark kernels of csrc/ceilings.cu
(include/dash_ceilings.h).  `python bench.py --ceilings` prints the dict below as one JSON
line; `bench.py` also calls `quick()` to put the three ceilings the hot path is compared against into the normal
bench line.  CUDA events on the launching stream, one warm-up launch, best of `reps` launches.
"""
from __future__ import annotations

import torch

from . import binding as b

MiB = 1 << 20
L2_RESIDENT = 32 * MiB      # one C4 gradient level (33.5 MB) / two fp16 table levels
HBM_RESIDENT = 1024 * MiB   # far beyond the 126 MB L2


def _time(fn, reps=5):
    fn()
    best = float("inf")
    for _ in range(reps):
        a, z = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        ops = fn()
        z.record()
        z.synchronize()
        best = min(best, a.elapsed_time(z))
    return ops, best


def _rate(kind, buf, sink, width, pattern, footprint, iters, reps=5, **kw):
    ops, ms = _time(lambda: b.dash_ceiling_launch(kind, buf, sink, width=width, pattern=pattern,
                                                  footprint_bytes=footprint, iters=iters, **kw), reps)
    return {"G_lane_ops_per_s": ops / (ms * 1e-3) / 1e9, "payload_GBps": ops * width / (ms * 1e-3) / 1e9,
            "ms": ms, "lane_ops": ops}


def _buffers(nbytes):
    dev = torch.device("cuda", torch.cuda.current_device())
    return torch.zeros(nbytes, dtype=torch.uint8, device=dev), torch.zeros(nbytes, dtype=torch.uint8, device=dev)


PATTERNS = {"independent": b.CEIL_INDEPENDENT, "pair_aligned": b.CEIL_PAIR_ALIGNED, "pair_xcorner": b.CEIL_PAIR_XCORNER}


def quick():
    """The three ceilings the bench line compares the hot path against (about 50 ms of GPU time)."""
    buf, sink = _buffers(L2_RESIDENT)
    sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    out = {
        "gather8_pair_xcorner_L2": _rate(b.CEIL_GATHER, buf, sink, 8, b.CEIL_PAIR_XCORNER, L2_RESIDENT, 32),
        "red16_pair_xcorner_L2": _rate(b.CEIL_RED, buf, sink, 16, b.CEIL_PAIR_XCORNER, L2_RESIDENT, 32),
        "red8_pair_xcorner_L2": _rate(b.CEIL_RED, buf, sink, 8, b.CEIL_PAIR_XCORNER, L2_RESIDENT, 32),
    }
    for v in out.values():
        v["per_sm_cycle_note"] = f"{sms} SMs"
    return out


def full():
    sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    buf, sink = _buffers(HBM_RESIDENT)
    res = {"device": torch.cuda.get_device_name(), "sms": sms,
           "method": "CUDA events, 1 warm-up + best of 5 launches; 8 x SMs CTAs x 256 threads x iters x 8 accesses "
                     "unless a grid is named; L2 = 32 MiB footprint, HBM = 1 GiB footprint"}
    threads = 8 * sms * 256
    iters_copy = max(1, HBM_RESIDENT // 16 // (threads * 8))
    ops, ms = _time(lambda: b.dash_ceiling_launch(b.CEIL_COPY, buf, sink, width=16, footprint_bytes=HBM_RESIDENT,
                                                  iters=iters_copy))
    moved = min(ops, HBM_RESIDENT // 16) * 16
    res["copy"] = {"GBps_read_plus_write": 2 * moved / (ms * 1e-3) / 1e9, "ms": ms, "bytes_each_way": moved}

    gather, red = {}, {}
    for where, fp, it in (("L2", L2_RESIDENT, 32), ("HBM", HBM_RESIDENT, 8)):
        for width in (8, 16, 32):
            for name, pat in PATTERNS.items():
                if width == 32 and pat != b.CEIL_INDEPENDENT:
                    continue
                gather[f"{width}B_{name}_{where}"] = _rate(b.CEIL_GATHER, buf, sink, width, pat, fp, it)
        for width in (4, 8, 16):
            for name, pat in PATTERNS.items():
                red[f"{width}B_{name}_{where}"] = _rate(b.CEIL_RED, buf, sink, width, pat, fp, it)
    res["gather"], res["red"] = gather, red

    # same-address contention: all lanes of the chip draw from a footprint of 1, 64, 4096 16-byte slots
    res["red_contention_16B"] = {f"{n}_slots": _rate(b.CEIL_RED, buf, sink, 16, b.CEIL_INDEPENDENT, 16 * n, 4)
                                 for n in (1, 64, 4096, 262144)}
    # is the limit per SM or chip-wide?  1 CTA of 1024 threads per SM (160 KB of dynamic smem), 1/4 .. 4/4 of the SMs
    sweep = {}
    for frac in (4, 2, 1):
        grid = max(1, sms // frac)
        for kind, nm, width in ((b.CEIL_RED, "red16", 16), (b.CEIL_GATHER, "gather8", 8)):
            sweep[f"{nm}_{grid}_SMs"] = _rate(kind, buf, sink, width, b.CEIL_INDEPENDENT, L2_RESIDENT, 64,
                                              grid=grid, block=1024, dyn_smem=160 * 1024)
    res["sm_count_sweep_L2"] = sweep
    # shared-memory atomics (what CTA-private accumulators would cost) and TMA bulk gathers (a second path past L1?)
    res["smem_atomic_f32"] = _rate(b.CEIL_SMEM_ATOMIC, buf, sink, 4, b.CEIL_INDEPENDENT, L2_RESIDENT, 8)
    res["smem_atomic_u64"] = _rate(b.CEIL_SMEM_ATOMIC_U64, buf, sink, 8, b.CEIL_INDEPENDENT, L2_RESIDENT, 8)
    res["tma_gather_16B_L2"] = _rate(b.CEIL_TMA_GATHER, buf, sink, 16, b.CEIL_INDEPENDENT, L2_RESIDENT, 8)
    res["tma_gather_16B_L2_2_ctas_per_sm"] = _rate(b.CEIL_TMA_GATHER, buf, sink, 16, b.CEIL_INDEPENDENT, L2_RESIDENT,
                                                   8, grid=2 * sms, block=256)
    return res


def to_markdown(res: dict, command: str) -> str:
    """The `full()` dict as the table `profiles/ceilings_rNN.md` holds (written by `bench.py --ceilings --md PATH`)."""
    sms = res["sms"]
    ghz = res.get("sm_clock_ghz", 1.965)
    per = lambda g: g / (sms * ghz)          # lane accesses per SM per cycle at the max SM clock
    out = [f"# Chip ceilings of the encoder's access patterns — {res['device']}, {sms} SMs", "",
           "Command:", "", "```", command, "```", "", res["method"] + ".",
           f"Per-SM-cycle figures assume {ghz} GHz (the max SM clock of this pool's B200s).", "",
           f"Stream copy (1 GiB each way): **{res['copy']['GBps_read_plus_write']:.0f} GB/s** read + write.", "",
           "| kernel / pattern | footprint | G lane accesses / s | per SM per cycle | payload GB/s | ms |",
           "|---|---|---|---|---|---|"]

    def row(name, where, v):
        out.append(f"| {name} | {where} | {v['G_lane_ops_per_s']:.1f} | {per(v['G_lane_ops_per_s']):.2f} | "
                   f"{v['payload_GBps']:.0f} | {v['ms']:.3f} |")
    for sec, label in (("gather", "ld.global.nc"), ("red", "red.global.add.f32")):
        for k, v in res[sec].items():
            width, rest = k.split("_", 1)
            pat, where = rest.rsplit("_", 1)
            row(f"{label} {width} {pat}", where, v)
    for k, v in res["red_contention_16B"].items():
        row(f"red.v4.f32, all lanes into {k.replace('_', ' ')}", "contention", v)
    for k, v in res["sm_count_sweep_L2"].items():
        row(f"{k.replace('_', ' ')} (1 CTA x 1024 threads per SM)", "L2", v)
    row("atomicAdd(float) on 32 KB of shared memory (ATOMS.CAST.SPIN loop)", "smem", res["smem_atomic_f32"])
    row("atomicAdd(u64) on 32 KB of shared memory", "smem", res["smem_atomic_u64"])
    row("cp.async.bulk 16 B global -> shared (TMA), 8 CTAs/SM", "L2", res["tma_gather_16B_L2"])
    row("cp.async.bulk 16 B global -> shared (TMA), 2 CTAs/SM", "L2", res["tma_gather_16B_L2_2_ctas_per_sm"])
    return "\n".join(out) + "\n"
