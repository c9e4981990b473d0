"""Tolerance checks shared by the GPU parity tests (DESIGN.md §3 Q17).

rtol: BASELINE.json north_star states rel 1e-5 (fp32 tables) / 2e-3 (fp16 tables, fp32 accumulate).
Both checks must pass:
  normwise per level:  ||a - ref||_2 / ||ref||_2 <= rtol
  elementwise:         |a - ref| <= rtol * A * max(1, sqrt(hits/1e4)) + 1e-30,
                       A = sum |W * v| over the terms of that element (computed by the oracle).
The fp32 arithmetic of the kernels (3 multiplies per weight, 16-term FMA chain / n-term fp32 atomic sum)
gives |err| <~ (5 + 16) * 2^-24 * A = 1.3e-6 * A in fwd, and ~2^-24 * sqrt(n) * A in bwd: inside 1e-5.
"""
import numpy as np

RTOL_FP32 = 1e-5
RTOL_FP16 = 2e-3


def fixed_point_quantum(n_queries: int, absmax: float) -> float:
    """Quantum 2^-s of the DETERMINISTIC_BWD fixed-point accumulators (DESIGN.md §3 Q23):
    s = 61 - e - k with absmax < 2^e and n_queries <= 2^k, clamped to [-100, 100]."""
    import math
    e = math.frexp(absmax)[1] if absmax > 0 else 0
    k = 0
    while (1 << k) < n_queries:
        k += 1
    return 2.0 ** -max(-100, min(100, 61 - e - k))


def check_close(got, ref, mag, rtol, L, hits=None, what="", quantum=0.0):
    """got/ref: arrays with a leading or trailing level structure flattened by the caller into
    shape [L][...]; mag: same shape, the conditioning term A; hits: optional [L][...] counts;
    quantum: fixed-point step of the deterministic mode (each of `hits` contributions is rounded to it)."""
    got = np.asarray(got, np.float64).reshape(L, -1)
    ref64 = np.asarray(ref, np.float64).reshape(L, -1)
    mag = np.asarray(mag, np.float64).reshape(L, -1)
    assert np.isfinite(got).all(), f"{what}: non-finite values"
    err = np.abs(got - ref64)
    for l in range(L):
        den = np.linalg.norm(ref64[l])
        num = np.linalg.norm(got[l] - ref64[l])
        assert num <= rtol * den + 1e-30, f"{what}: level {l} normwise {num / max(den, 1e-300):.3e} > {rtol}"
    allow = rtol * mag
    if hits is not None:
        h = np.asarray(hits, np.float64).reshape(L, -1)
        if h.shape[1] != mag.shape[1]:                       # hits per slot, mag per (slot, f)
            h = np.repeat(h, mag.shape[1] // h.shape[1], axis=1)
        allow = allow * np.maximum(1.0, np.sqrt(h / 1e4)) + 0.5 * quantum * h
    bad = err > allow + 1e-30
    assert not bad.any(), (f"{what}: {bad.sum()} elements out of tolerance; worst ratio "
                           f"{(err / (mag + 1e-300)).max():.3e} (rtol {rtol})")
    return float((err / (mag + 1e-300)).max())
