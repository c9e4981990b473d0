"""Pins for the oracle's host-side pieces: Eq. 7 schedule, Eq. 8 hash, dense index, cell location,
fp16 decode (readings DESIGN.md §3).  CPU only."""
import math
import os

import numpy as np
import pytest

import oracle
from dash_inputs import CONFIGS


def _read_rows(path):
    rows = []
    with open(path) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line)
    return rows


# ---------------------------------------------------------------- Eq. 7 resolutions

def exact_floor_geometric(n_min, n_max, l, L):
    """Largest n with n^(L-1) <= n_min^(L-1-l) * n_max^l: the exact floor of
    n_min*(n_max/n_min)^(l/(L-1)) in integer arithmetic (no floating point at all)."""
    if L == 1:
        return n_min
    rhs = n_min ** (L - 1 - l) * n_max ** l
    n = int(round(rhs ** (1.0 / (L - 1))))
    while n ** (L - 1) > rhs:
        n -= 1
    while (n + 1) ** (L - 1) <= rhs:
        n += 1
    return n


def test_resolutions_match_printed_lists(golden_dir):
    for row in _read_rows(os.path.join(golden_dir, "resolutions.txt")):
        head, vals = row.split(":")
        _, n_min, n_max, L = head.split()
        n_min, n_max, L = int(n_min), int(n_max), int(L)
        want = [int(v) for v in vals.split()]
        cfg = oracle.make_config(L, 2, 1 << 12, n_min, n_max, n_min, n_max)
        rs, rt, _ = oracle.oracle_resolutions(cfg)
        assert list(rs) == want
        assert list(rt) == want
        # and the printed lists themselves equal the exact mathematical floor
        assert want == [exact_floor_geometric(n_min, n_max, l, L) for l in range(L)]


@pytest.mark.parametrize("n_min,n_max,L", [(16, 512, 10), (4, 4096, 11), (8, 8, 5), (3, 1000, 7),
                                           (16, 2048, 8), (1, 8192, 14), (5, 5000, 32), (2, 300, 2)])
def test_resolutions_exact_floor_other_ranges(n_min, n_max, L):
    cfg = oracle.make_config(L, 1, 64, n_min, n_max, n_min, n_max)
    rs, rt, _ = oracle.oracle_resolutions(cfg)
    want = [exact_floor_geometric(n_min, n_max, l, L) for l in range(L)]
    assert list(rs) == want and list(rt) == want
    assert rs[0] == n_min and rs[-1] == n_max
    assert all(a <= b for a, b in zip(rs, rs[1:]))


def test_single_level_is_nmin():
    cfg = oracle.make_config(1, 2, 64, 7, 99, 3, 50)
    rs, rt, _ = oracle.oracle_resolutions(cfg)
    assert list(rs) == [7] and list(rt) == [3]


def test_spatial_and_temporal_ranges_are_separate():
    enc = CONFIGS["C2"].enc
    rs, rt, _ = oracle.oracle_resolutions(oracle.config_from_params(enc))
    assert rs[0] == 16 and rs[-1] == 2048 and rt[0] == 8 and rt[-1] == 150


def test_dense_levels_per_config():
    """Q10: dense iff (Ns+1)^3 (Nt+1) <= T.  SURVEY §8c: C1 none; C2 l=0,1; C3/C5 l=0..2; C4 l=0..3."""
    want = {"C1": [], "C2": [0, 1], "C3": [0, 1, 2], "C4": [0, 1, 2, 3], "C5": [0, 1, 2]}
    for name, levels in want.items():
        enc = CONFIGS[name].enc
        rs, rt, dn = oracle.oracle_resolutions(oracle.config_from_params(enc))
        assert [l for l in range(enc.L) if dn[l]] == levels
        for l in range(enc.L):
            assert bool(dn[l]) == ((int(rs[l]) + 1) ** 3 * (int(rt[l]) + 1) <= enc.T)
        _, _, dn_off = oracle.oracle_resolutions(oracle.config_from_params(enc, dense_coarse=False))
        assert not dn_off.any()


# ---------------------------------------------------------------- Eq. 8 hash

def test_hash_golden_values(golden_dir):
    for row in _read_rows(os.path.join(golden_dir, "hash_values.txt")):
        gx, gy, gz, gt, T, want = (int(v) for v in row.split())
        cfg = oracle.make_config(1, 2, T, 4096, 4096, 300, 300, dense_coarse=False)
        assert oracle.oracle_vertex_slot(cfg, 0, (gx, gy, gz, gt)) == want, row


def test_hash_xor_structure():
    """h(g) ^ h(g') depends only on the coordinates that differ (XOR of per-axis terms), T = 2^32-free
    check done at T = 2^31 so 'mod T' only drops the top bit."""
    T = 1 << 31
    cfg = oracle.make_config(1, 1, T, 4096, 4096, 300, 300, dense_coarse=False)
    rng = np.random.default_rng(11)
    for _ in range(50):
        g = rng.integers(0, 4097, size=4)
        g2 = g.copy()
        g2[1] = rng.integers(0, 4097)
        other = rng.integers(0, 4097, size=4)
        o1, o2 = other.copy(), other.copy()
        o1[1], o2[1] = g[1], g2[1]
        a = oracle.oracle_vertex_slot(cfg, 0, g) ^ oracle.oracle_vertex_slot(cfg, 0, g2)
        b = oracle.oracle_vertex_slot(cfg, 0, o1) ^ oracle.oracle_vertex_slot(cfg, 0, o2)
        assert a == b


def test_custom_primes_and_x_adjacency():
    T = 1 << 16
    cfg = oracle.make_config(1, 1, T, 64, 64, 8, 8, primes=(1, 3, 5, 7), dense_coarse=False)
    assert oracle.oracle_vertex_slot(cfg, 0, (2, 1, 1, 1)) == (2 ^ 3 ^ 5 ^ 7)
    assert oracle.oracle_vertex_slot(cfg, 0, (10, 20, 30, 4)) == (10 ^ 60 ^ 150 ^ 28) % T
    # default pi1 = 1: even gx and gx+1 are adjacent slots
    cfg = oracle.make_config(1, 1, T, 64, 64, 8, 8, dense_coarse=False)
    for g in [(4, 9, 2, 3), (62, 0, 63, 8)]:
        a = oracle.oracle_vertex_slot(cfg, 0, g)
        b = oracle.oracle_vertex_slot(cfg, 0, (g[0] + 1,) + g[1:])
        assert b == a ^ 1


# ---------------------------------------------------------------- dense index

@pytest.mark.parametrize("level", [0, 1])
def test_dense_index_is_a_bijection_on_c2(level):
    """Brute force over every vertex of C2's dense levels: 17^3*9 = 44217 and 23^3*10 = 121670."""
    enc = CONFIGS["C2"].enc
    cfg = oracle.config_from_params(enc)
    rs, rt, dn = oracle.oracle_resolutions(cfg)
    assert dn[level]
    S, St = int(rs[level]) + 1, int(rt[level]) + 1
    count = S ** 3 * St
    assert count == (44217, 121670)[level]
    seen = np.zeros(count, bool)
    for gt in range(St):
        for gz in range(S):
            for gy in range(S):
                base = oracle.oracle_vertex_slot(cfg, level, (0, gy, gz, gt))
                last = oracle.oracle_vertex_slot(cfg, level, (S - 1, gy, gz, gt))
                assert last == base + S - 1          # x is the fastest axis
                assert not seen[base:base + S].any()
                seen[base:base + S] = True
    assert seen.all()


def test_dense_index_golden():
    cfg = oracle.config_from_params(CONFIGS["C2"].enc)   # level 0: Ns=16, Nt=8, S=17
    assert oracle.oracle_vertex_slot(cfg, 0, (16, 16, 16, 8)) == 44216
    assert oracle.oracle_vertex_slot(cfg, 0, (3, 5, 7, 2)) == 11937
    assert oracle.oracle_vertex_slot(cfg, 0, (0, 0, 0, 0)) == 0
    assert oracle.oracle_vertex_slot(cfg, 0, (0, 1, 0, 0)) == 17
    assert oracle.oracle_vertex_slot(cfg, 0, (0, 0, 1, 0)) == 289
    assert oracle.oracle_vertex_slot(cfg, 0, (0, 0, 0, 1)) == 4913


# ---------------------------------------------------------------- cell location

def test_locate_is_one_fp32_multiply():
    """Frame-aligned timestamps t = j/300 at Nt = 300: floor(fl32(fl32(j/300)*300)) — numpy's binary32
    multiply is the independent witness; some frames land in cell j-1."""
    short = 0
    for j in range(300):
        tj = np.float32(j / 300.0)
        pos = np.float32(tj * np.float32(300))
        cell, frac = oracle.oracle_locate(float(tj), 300)
        assert cell == int(math.floor(float(pos)))
        assert frac == float(pos) - cell
        short += cell == j - 1
    assert short > 0      # the hazard is real: a double-precision product would never give j-1


def test_locate_clamp_and_edges():
    one_m = float(np.nextafter(np.float32(1), np.float32(0)))
    for n in list(range(1, 600)) + [1023, 1024, 2048, 4095, 4096, 8191, 8192]:
        cell, frac = oracle.oracle_locate(one_m, n)
        assert cell <= n - 1 and 0.0 <= frac < 1.0
        assert oracle.oracle_locate(1.0, n) == (cell, frac)         # clamped to 1-2^-24
        assert oracle.oracle_locate(7.5, n) == (cell, frac)
        assert oracle.oracle_locate(0.0, n) == (0, 0.0)
        assert oracle.oracle_locate(-3.0, n) == (0, 0.0)
        assert oracle.oracle_locate(float("nan"), n) == (0, 0.0)    # Q12: NaN -> 0
    assert oracle.oracle_locate(0.5, 16) == (8, 0.0)
    assert oracle.oracle_locate(0.53125, 16) == (8, 0.5)


# ---------------------------------------------------------------- fp16 decode (Q13)

def test_half_decode_all_patterns():
    bits = np.arange(65536, dtype=np.uint16)
    want = bits.view(np.float16).astype(np.float64)
    for b in range(0, 65536, 7):
        got = oracle.oracle_half_to_double(b)
        if np.isnan(want[b]):
            assert np.isnan(got)
        else:
            assert got == want[b] and np.signbit(got) == np.signbit(want[b])
    for b in (0x0000, 0x8000, 0x0001, 0x03ff, 0x0400, 0x3c00, 0x7bff, 0x7c00, 0xfc00, 0xfbff):
        assert oracle.oracle_half_to_double(b) == want[b]
