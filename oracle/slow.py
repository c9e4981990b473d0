"""Second, even slower transcription of the encoder definition — pure Python loops, numpy scalars.

TEST INFRASTRUCTURE.  Exists only to guard oracle/dash_oracle.c against transcription mistakes on
tiny inputs (tests/test_oracle_bruteforce.py).  It follows PAPER.md:125-135 literally:
Eq. 7 resolutions, floor(x*N_l) cell location, Eq. 8 hash, quadrilinear interpolation, Eq. 9
concatenation; readings Q1-Q21 as in DESIGN.md §3.  Written independently of the C file:
the hash is a Python-int computation reduced mod 2^32, the weights use fractions of Python floats.
"""
from __future__ import annotations

import math

import numpy as np

DEFAULT_PRIMES = (1, 2654435761, 805459861, 3674653429)   # Q7
MAXF = float(np.nextafter(np.float32(1), np.float32(0)))  # 1 - 2^-24


def resolutions(n_min: int, n_max: int, L: int) -> list[int]:
    """Eq. 7 with the exponent restored (Q1) and the +1e-6 guard (Q2)."""
    if L == 1:
        return [n_min]
    return [int(math.floor(n_min * math.pow(n_max / n_min, l / (L - 1)) + 1e-6)) for l in range(L)]


def is_dense(ns: int, nt: int, T: int) -> bool:
    return (ns + 1) ** 3 * (nt + 1) <= T   # Q10 (exact integer arithmetic)


def clamp(v) -> np.float32:
    v = np.float32(v)
    if np.isnan(v):
        return np.float32(0)
    return np.float32(min(max(float(v), 0.0), MAXF))   # Q12


def locate(x, n: int):
    pos = np.float32(clamp(x)) * np.float32(n)          # one binary32 multiply (Q4)
    assert pos.dtype == np.float32
    c = int(math.floor(float(pos)))
    w = float(pos) - c                                  # exact
    return c, w


def slot_of(g, ns: int, T: int, dense: bool, primes=DEFAULT_PRIMES) -> int:
    if dense:
        S = ns + 1
        return g[0] + S * (g[1] + S * (g[2] + S * g[3]))
    h = 0
    for gi, pi in zip(g, primes):
        h ^= (gi * pi) & 0xFFFFFFFF                      # Q8: uint32 wraparound
    return h % T                                         # Eq. 8


def corners(q, ns: int, nt: int, T: int, dense: bool, primes=DEFAULT_PRIMES):
    """16 (slot, weight) pairs; corner k has bit d set => +1 along d (x,y,z,t)."""
    cw = [locate(q[d], ns if d < 3 else nt) for d in range(4)]
    res = []
    for k in range(16):
        g, w = [], 1.0
        for d in range(4):
            up = (k >> d) & 1
            g.append(cw[d][0] + up)
            w *= cw[d][1] if up else (1.0 - cw[d][1])
        res.append((slot_of(g, ns, T, dense, primes), w))
    return res


def plan(L, T, rs_min, rs_max, rt_min, rt_max, dense_coarse=True):
    rs, rt = resolutions(rs_min, rs_max, L), resolutions(rt_min, rt_max, L)
    dn = [dense_coarse and is_dense(a, b, T) for a, b in zip(rs, rt)]
    return rs, rt, dn


def forward(queries, table, L, F, T, rs_min, rs_max, rt_min, rt_max, dense_coarse=True,
            primes=DEFAULT_PRIMES):
    """queries [n][4]; table [L][T][F] (any float dtype).  Returns float64 [n][L*F] (unrounded)."""
    rs, rt, dn = plan(L, T, rs_min, rs_max, rt_min, rt_max, dense_coarse)
    out = np.zeros((len(queries), L * F))
    for n, q in enumerate(queries):
        for l in range(L):
            for s, w in corners(q, rs[l], rt[l], T, dn[l], primes):
                for f in range(F):
                    out[n, l * F + f] += w * float(table[l, s, f])
    return out


def backward(queries, dout, L, F, T, rs_min, rs_max, rt_min, rt_max, dense_coarse=True,
             primes=DEFAULT_PRIMES):
    """Returns float64 [L][T][F]: sum over queries and corners of w * dout."""
    rs, rt, dn = plan(L, T, rs_min, rs_max, rt_min, rt_max, dense_coarse)
    g = np.zeros((L, T, F))
    for n, q in enumerate(queries):
        for l in range(L):
            for s, w in corners(q, rs[l], rt[l], T, dn[l], primes):
                for f in range(F):
                    g[l, s, f] += w * float(dout[n, l * F + f])
    return g


def backward_input(queries, table, dout, L, F, T, rs_min, rs_max, rt_min, rt_max, dense_coarse=True,
                   primes=DEFAULT_PRIMES):
    """dq[n][d] = sum_{l,f} dout * N_{l,d} * sum_k s_d(k) prod_{e!=d} omega_e(k) * table  (float64 [n][4]).
    Coordinates moved by the clamp get 0 (Q24)."""
    rs, rt, dn = plan(L, T, rs_min, rs_max, rt_min, rt_max, dense_coarse)
    dq = np.zeros((len(queries), 4))
    for n, q in enumerate(queries):
        for l in range(L):
            res = [rs[l]] * 3 + [rt[l]]
            cw = [locate(q[d], res[d]) for d in range(4)]
            for k in range(16):
                g = [cw[d][0] + ((k >> d) & 1) for d in range(4)]
                s = slot_of(g, rs[l], T, dn[l], primes)
                for d in range(4):
                    w = 1.0 if (k >> d) & 1 else -1.0
                    for e in range(4):
                        if e != d:
                            w *= cw[e][1] if (k >> e) & 1 else 1.0 - cw[e][1]
                    for f in range(F):
                        dq[n, d] += float(dout[n, l * F + f]) * res[d] * w * float(table[l, s, f])
        for d in range(4):
            v = np.float32(q[d])
            if np.isnan(v) or v < 0 or float(v) > MAXF:
                dq[n, d] = 0.0
    return dq


def smooth(queries, eps, table, L, F, T, rs_min, rs_max, rt_min, rt_max, dense_coarse=True, grad_scale=1.0,
           primes=DEFAULT_PRIMES):
    """Eq. 11: loss[n] = ||G(x_n) - G(fl32(x_n + eps_n))||^2 (float64 [n]) and the gradient of
    grad_scale * sum_n loss[n] with respect to the table (float64 [L][T][F])."""
    rs, rt, dn = plan(L, T, rs_min, rs_max, rt_min, rt_max, dense_coarse)
    eps = np.asarray(eps, np.float32).reshape(-1, 4)
    loss = np.zeros(len(queries))
    grad = np.zeros((L, T, F))
    for n, q in enumerate(queries):
        e = eps[n if len(eps) > 1 else 0]
        q2 = [np.float32(np.float32(q[d]) + e[d]) for d in range(4)]
        for l in range(L):
            c1 = corners(q, rs[l], rt[l], T, dn[l], primes)
            c2 = corners(q2, rs[l], rt[l], T, dn[l], primes)
            for f in range(F):
                d = sum(w * float(table[l, s, f]) for s, w in c1) - sum(w * float(table[l, s, f]) for s, w in c2)
                loss[n] += d * d
                for s, w in c1:
                    grad[l, s, f] += 2.0 * grad_scale * w * d
                for s, w in c2:
                    grad[l, s, f] -= 2.0 * grad_scale * w * d
    return loss, grad
