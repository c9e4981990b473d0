"""Pins of the G_3D oracle (oracle/dash_oracle.c `dash_oracle3d_*`; Eq. 3: "a 3D hash encoder
G_3D from Instant-NGP"; Q26 = Eq. 7-9 with d = 3).  CPU only.

What fixes it, other than itself:
  * it must equal the (already pinned) 4D oracle at temporal resolution 1, t = 0, Eq. 8 on every level:
    g_t = 0 adds 0 to the XOR and the upper t-corners carry weight exactly 0;
  * hand-derived hash values of tests/golden/hash_values.txt (rows with g_t = 0);
  * scipy's RegularGridInterpolator on dense levels; bijection of the dense index by brute force;
  * multi-affine reproduction, weights sum to 1, adjoint identity, an 8-corner brute force written here."""
import os

import numpy as np
import pytest
from scipy.interpolate import RegularGridInterpolator

import oracle
from dash_inputs import make_queries_uniform

P3 = (1, 2654435761, 805459861)


def brute_level(xyz, table_l, res, T, dense):
    out = np.zeros((len(xyz), table_l.shape[1]))
    for n, p in enumerate(xyz):
        pos = (np.float32(p) * np.float32(res)).astype(np.float32)
        c = np.floor(pos).astype(np.int64)
        w = (pos - np.floor(pos)).astype(np.float64)
        for k in range(8):
            g = [int(c[d]) + ((k >> d) & 1) for d in range(3)]
            wk = np.prod([w[d] if (k >> d) & 1 else 1 - w[d] for d in range(3)])
            if dense:
                S = res + 1
                s = g[0] + S * (g[1] + S * g[2])
            else:
                s = (((g[0] * P3[0]) & 0xFFFFFFFF) ^ ((g[1] * P3[1]) & 0xFFFFFFFF)
                     ^ ((g[2] * P3[2]) & 0xFFFFFFFF)) % T
            out[n] += wk * table_l[s].astype(np.float64)
    return out


@pytest.mark.parametrize("half", [False, True])
def test_equals_4d_oracle_at_nt1_t0(half):
    L, F, T, n = 6, 2, 1 << 12, 300
    c3 = oracle.make_config(L, F, T, 4, 200, 1, 1, "fp16" if half else "fp32", dense_coarse=False)
    xyz, _ = make_queries_uniform(11, n)
    xyz[0] = [0.0, 1.0, np.float32(1) - np.float32(2.0 ** -24)]
    xyz[1] = [np.nan, -1.0, 2.0]
    rng = np.random.default_rng(3)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16 if half else np.float32)
    dout = rng.standard_normal((n, L * F)).astype(np.float32)
    t0 = np.zeros(1, np.float32)
    i3, w3 = oracle.oracle3d_indices(c3, n, xyz)
    i4, w4 = oracle.oracle_indices(c3, n, xyz, t0, t_stride=0)
    np.testing.assert_array_equal(i3, i4[:, :, :8])
    np.testing.assert_array_equal(w3, w4[:, :, :8])
    assert (w4[:, :, 8:] == 0).all()
    np.testing.assert_array_equal(oracle.oracle3d_fwd(c3, n, xyz, table),
                                  oracle.oracle_fwd(c3, n, xyz, t0, table, t_stride=0))
    np.testing.assert_array_equal(oracle.oracle3d_bwd(c3, n, xyz, dout),
                                  oracle.oracle_bwd(c3, n, xyz, t0, dout, t_stride=0))


def test_golden_hash_values_with_gt_zero(golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "hash_values.txt")) if l.strip() and l[0] != "#"]
    used = 0
    for gx, gy, gz, gt, T, want in (tuple(int(v) for v in r) for r in rows):
        if gt != 0 or max(gx, gy, gz) >= 16:
            continue
        cfg = oracle.make_config(1, 1, T, 16, 16, 1, 1, dense_coarse=False)
        p = np.array([[gx / 16.0, gy / 16.0, gz / 16.0]], np.float32)      # exactly on vertex g
        idx, w = oracle.oracle3d_indices(cfg, 1, p)
        assert idx[0, 0, 0] == want and w[0, 0, 0] == 1.0
        used += 1
    assert used >= 8


def test_dense_rule_is_the_three_dimensional_one():
    # (Ns+1)^3 <= T decides, not the 4D product: 17^3 = 4913 <= 8192 < 2*4913
    cfg = oracle.make_config(3, 2, 8192, 16, 64, 1, 1)
    rs, dn = oracle.oracle3d_resolutions(cfg)
    assert list(rs) == [16, 32, 64] and list(dn) == [True, False, False]
    _, _, dn4 = oracle.oracle_resolutions(cfg)
    assert not dn4[0]
    # bijection of the dense index onto [0, S^3) by brute force over all vertices of level 0
    S = 17
    g = np.stack(np.meshgrid(np.arange(16), np.arange(16), np.arange(16), indexing="ij"), -1).reshape(-1, 3)
    idx, _ = oracle.oracle3d_indices(cfg, len(g), (g / 16.0).astype(np.float32))
    seen = np.unique(idx[:, 0, :])
    assert seen.min() == 0 and seen.max() == S ** 3 - 1 and len(seen) == S ** 3
    assert idx[0, 0, 7] == 1 + S * (1 + S * 1)            # cell (0,0,0), corner (1,1,1)


def test_scipy_trilinear_on_dense_levels_and_bruteforce_everywhere():
    L, F, T, n = 4, 2, 1 << 15, 400
    cfg = oracle.make_config(L, F, T, 5, 90, 1, 1)
    rs, dn = oracle.oracle3d_resolutions(cfg)
    assert dn[0] and dn[1] and not dn[3]
    rng = np.random.default_rng(5)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float32)
    xyz, _ = make_queries_uniform(6, n)
    out, mag = oracle.oracle3d_fwd(cfg, n, xyz, table, want_abs=True)
    for l in range(L):
        res = int(rs[l])
        want = brute_level(xyz, table[l], res, T, bool(dn[l]))
        np.testing.assert_allclose(out[:, l * F:(l + 1) * F], want, rtol=0, atol=3e-7)
        if dn[l]:
            S = res + 1
            grid = table[l, :S ** 3].reshape(S, S, S, F).transpose(2, 1, 0, 3)   # [x][y][z][f], x fastest in memory
            axes = [np.arange(S, dtype=np.float64)] * 3
            pos = (xyz * np.float32(res)).astype(np.float32).astype(np.float64)
            for f in range(F):
                rgi = RegularGridInterpolator(axes, grid[..., f].astype(np.float64), method="linear")
                np.testing.assert_allclose(out[:, l * F + f], rgi(pos), rtol=0, atol=3e-7)
    assert (mag >= np.abs(out) - 1e-7).all()


def test_multi_affine_reproduction_weights_and_adjoint():
    L, F, T, n = 3, 4, 1 << 14, 500
    cfg = oracle.make_config(L, F, T, 8, 20, 1, 1)
    rs, dn = oracle.oracle3d_resolutions(cfg)
    assert dn.all()
    a, b = np.array([0.3, -1.1, 0.7]), np.array([1.9, 0.4, -0.8])
    table = np.zeros((L, T, F), np.float32)
    for l in range(L):
        S = int(rs[l]) + 1
        gz, gy, gx = np.meshgrid(np.arange(S), np.arange(S), np.arange(S), indexing="ij")
        vals = np.prod([a[d] + b[d] * g / float(rs[l]) for d, g in enumerate((gx, gy, gz))], axis=0)
        for f in range(F):
            table[l, :S ** 3, f] = ((f + 1) * vals).reshape(-1)
    xyz, _ = make_queries_uniform(9, n)
    out = oracle.oracle3d_fwd(cfg, n, xyz, table)
    for l in range(L):
        x = (xyz * np.float32(rs[l])).astype(np.float32).astype(np.float64) / float(rs[l])   # the located point
        want = np.prod(a + b * x, axis=1)
        for f in range(F):
            np.testing.assert_allclose(out[:, l * F + f], (f + 1) * want, rtol=2e-6, atol=2e-6)
    _, w = oracle.oracle3d_indices(cfg, n, xyz)
    assert (w >= 0).all() and np.abs(w.sum(-1) - 1).max() < 1e-15
    # adjoint identity on a hashed configuration
    cfg2 = oracle.make_config(5, 2, 1 << 10, 4, 300, 1, 1)
    rng = np.random.default_rng(2)
    theta = rng.standard_normal((5, 1 << 10, 2)).astype(np.float32)
    g = rng.standard_normal((n, 10)).astype(np.float32)
    lhs = float((oracle.oracle3d_fwd(cfg2, n, xyz, theta).astype(np.float64) * g).sum())
    rhs = float((oracle.oracle3d_bwd(cfg2, n, xyz, g).astype(np.float64) * theta).sum())
    assert abs(lhs - rhs) <= 2e-6 * max(abs(lhs), 1.0)
    # index list = gather of rows
    index = rng.integers(0, n, 77).astype(np.int32)
    np.testing.assert_array_equal(oracle.oracle3d_fwd(cfg2, 77, xyz, theta, index=index),
                                  oracle.oracle3d_fwd(cfg2, 77, np.ascontiguousarray(xyz[index]), theta))


def test_coordinate_gradient_equals_the_4d_oracle_and_exact_central_differences():
    """oracle3d_bwd_input pinned (i) to the 4D coordinate gradient at Nt = 1, t = 0 with Eq. 8 on every level (g_t = 0
    adds nothing to the XOR; the t-derivative is dropped), (ii) by central differences of the pinned 3D forward on
    power-of-two grids (the interpolant is affine in x inside a cell, steps of 2^-14 stay inside), (iii) a clamped
    coordinate has gradient 0 and the magnitude term is the value itself when every term has one sign."""
    L, F, T = 4, 2, 1 << 11
    rng = np.random.default_rng(21)
    n = 300
    cfg3 = oracle.make_config(L, F, T, 8, 64, 1, 1, dense_coarse=False)
    cfg4 = oracle.make_config(L, F, T, 8, 64, 1, 1, dense_coarse=False)
    xyz, _ = make_queries_uniform(21, n)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float32)
    dout = rng.standard_normal((n, L * F)).astype(np.float32)
    dq3, mag3 = oracle.oracle3d_bwd_input(cfg3, n, xyz, table, dout, want_abs=True)
    dq4, mag4 = oracle.oracle_bwd_input(cfg4, n, xyz, np.zeros(1, np.float32), table, dout, t_stride=0, want_abs=True)
    np.testing.assert_array_equal(dq3, dq4[:, :3])
    np.testing.assert_allclose(mag3, mag4[:, :3], rtol=1e-14)
    # (ii) exact central differences on a dense + hashed power-of-two schedule
    cfgd = oracle.make_config(3, 1, 1 << 10, 4, 16, 1, 1)                       # levels 4, 8, 16: (8+1)^3 = 729 dense
    tab = rng.uniform(-1, 1, (3, 1 << 10, 1)).astype(np.float32)
    pts = (rng.integers(1, 60, (200, 3)) / 64.0 + 2.0 ** -9).astype(np.float32)  # strictly inside cells of every level
    dy = rng.standard_normal((200, 3)).astype(np.float32)
    dq = oracle.oracle3d_bwd_input(cfgd, 200, pts, tab, dy)
    h = np.float32(2.0 ** -14)
    for d in range(3):
        pp, pm = pts.copy(), pts.copy()
        pp[:, d] += h; pm[:, d] -= h
        fd = ((oracle.oracle3d_fwd(cfgd, 200, pp, tab).astype(np.float64) - oracle.oracle3d_fwd(cfgd, 200, pm, tab)) * dy).sum(1) / (2.0 * float(h))
        np.testing.assert_allclose(dq[:, d], fd, rtol=0, atol=2e-3)             # the forward's fp32 rounding / 2^-13
    # (iii) clamp and sign structure
    bad = np.array([[-0.5, 0.3, 0.4], [0.2, np.nan, 0.4], [0.2, 0.3, 1.5]], np.float32)
    dqb = oracle.oracle3d_bwd_input(cfgd, 3, bad, tab, np.ones((3, 3), np.float32))
    assert dqb[0, 0] == 0 and dqb[1, 1] == 0 and dqb[2, 2] == 0 and np.abs(dqb).sum() > 0
    S = 5
    gx = np.arange(1 << 10) % S
    mono = np.zeros((1, 1 << 10, 1), np.float32); mono[0, :, 0] = 1.0 + gx       # v = 1 + g_x on the level-4 dense grid
    c1 = oracle.make_config(1, 1, 1 << 10, 4, 4, 1, 1)
    q, m = oracle.oracle3d_bwd_input(c1, 100, xyz[:100], mono, np.ones((100, 1), np.float32), want_abs=True)
    np.testing.assert_allclose(q[:, 0], 4.0, rtol=1e-6)
    cell = np.floor(xyz[:100, 0] * np.float32(4)).astype(np.float64)
    np.testing.assert_allclose(m[:, 0], 4 * (2 * (1 + cell) + 1), rtol=1e-12)
