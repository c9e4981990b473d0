"""Pins for the oracle's smoothness regulariser (Eq. 11; Q25): composition from
the pinned forward/backward, closed form on a multi-affine table, exact central differences (the loss is
quadratic in the table), degenerate perturbations, Python brute force.  CPU only."""
import numpy as np

import oracle
from oracle import slow
from dash_inputs import make_queries_uniform


def _setup(seed=0, n=300, L=4, F=2, T=1 << 13, scale=2e-3):
    cfg = oracle.make_config(L, F, T, 8, 256, 4, 32)
    rng = np.random.default_rng(seed)
    xyz, t = make_queries_uniform(seed, n)
    eps = rng.uniform(-scale, scale, (n, 4)).astype(np.float32)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float32)
    return cfg, xyz, t, eps, table


def test_equals_composition_of_pinned_forward_and_backward():
    cfg, xyz, t, eps, table = _setup()
    n = len(t)
    loss, grad, la, fa, ga = oracle.oracle_smooth(cfg, n, xyz, t, eps, table, grad_scale=0.75, want_abs=True)
    x2 = (xyz + eps[:, :3]).astype(np.float32); t2 = (t + eps[:, 3]).astype(np.float32)   # fp32 adds (numpy)
    y1 = oracle.oracle_fwd(cfg, n, xyz, t, table).astype(np.float64)
    y2 = oracle.oracle_fwd(cfg, n, x2, t2, table).astype(np.float64)
    d = y1 - y2
    # forward outputs are fp32-rounded (6e-8 relative each): the oracle's own tolerance terms cover it
    assert (np.abs(loss - (d * d).sum(1)) <= 2e-7 * la + 1e-12).all()
    d32 = d.astype(np.float32)
    g = 1.5 * (oracle.oracle_bwd(cfg, n, xyz, t, d32).astype(np.float64)
               - oracle.oracle_bwd(cfg, n, x2, t2, d32).astype(np.float64))
    assert (np.abs(grad - g) <= 4e-7 * ga + 1e-12).all()
    assert np.abs(grad).max() > 1e-3 and (loss > 0).all()
    # levels whose cell is shared by x and x+eps still contribute (weights differ): coarse level non-zero
    assert np.abs(grad[0]).max() > 0


def test_closed_form_on_multi_affine_table():
    ns, nt = 12, 5
    S, St = ns + 1, nt + 1
    cfg = oracle.make_config(1, 1, S ** 3 * St, ns, ns, nt, nt)
    a = np.array([0.3, -1.2, 0.7, 2.0]); b = np.array([1.5, 0.4, -2.2, 0.9])
    gx, gy, gz, gt = np.meshgrid(np.arange(S), np.arange(S), np.arange(S), np.arange(St), indexing="ij")
    vals = ((a[0] + b[0] * gx / ns) * (a[1] + b[1] * gy / ns) * (a[2] + b[2] * gz / ns) * (a[3] + b[3] * gt / nt))
    table = np.zeros((1, cfg.T, 1), np.float32)
    table[0, (gx + S * (gy + S * (gz + S * gt))).ravel(), 0] = vals.ravel()
    n = 1500
    xyz, t = make_queries_uniform(3, n)
    eps = np.random.default_rng(4).uniform(-0.05, 0.05, (n, 4)).astype(np.float32)
    loss, _ = oracle.oracle_smooth(cfg, n, xyz, t, eps, table, want_grad=False)

    def g_at(x, tt):
        x = np.clip(x, 0, np.float32(1) - np.float32(2.0 ** -24)); tt = np.clip(tt, 0, np.float32(1) - np.float32(2.0 ** -24))
        p = np.concatenate([(x * np.float32(ns)).astype(np.float64) / ns,
                            ((tt * np.float32(nt)).astype(np.float64) / nt)[:, None]], 1)
        return np.prod(a[None] + b[None] * p, axis=1)
    want = (g_at(xyz, t) - g_at((xyz + eps[:, :3]).astype(np.float32), (t + eps[:, 3]).astype(np.float32))) ** 2
    np.testing.assert_allclose(loss, want, rtol=0, atol=3e-6 * np.abs(vals).max() * np.sqrt(want.max()) + 1e-12)


def test_central_differences_are_exact_for_a_quadratic():
    cfg, xyz, t, eps, table = _setup(seed=2, n=150, L=3, T=1 << 11)
    n = len(t)
    _, grad = oracle.oracle_smooth(cfg, n, xyz, t, eps, table, grad_scale=1.0)
    idx, _ = oracle.oracle_indices(cfg, n, xyz, t)
    h = np.float32(0.5)
    rng = np.random.default_rng(0)
    for l in range(3):
        for s in rng.choice(np.unique(idx[:, l]), 5, replace=False):
            for f in range(2):
                tp, tm = table.copy(), table.copy()
                tp[l, s, f] += h; tm[l, s, f] -= h
                lp = oracle.oracle_smooth(cfg, n, xyz, t, eps, tp, want_grad=False)[0].astype(np.float64).sum()
                lm = oracle.oracle_smooth(cfg, n, xyz, t, eps, tm, want_grad=False)[0].astype(np.float64).sum()
                np.testing.assert_allclose((lp - lm) / (2 * float(h)), grad[l, s, f], rtol=1e-4, atol=2e-5)


def test_degenerate_perturbations():
    cfg, xyz, t, eps, table = _setup(seed=5, n=100)
    n = len(t)
    loss, grad = oracle.oracle_smooth(cfg, n, xyz, t, np.zeros((n, 4), np.float32), table)
    assert not loss.any() and not grad.any()
    # one perturbation for all queries (eps_stride 0) == the same row repeated
    e1 = np.array([1e-3, -2e-3, 5e-4, 1e-3], np.float32)
    a = oracle.oracle_smooth(cfg, n, xyz, t, e1, table)
    b = oracle.oracle_smooth(cfg, n, xyz, t, np.tile(e1, (n, 1)), table)
    np.testing.assert_array_equal(a[0], b[0]); np.testing.assert_array_equal(a[1], b[1])
    # a perturbation that pushes every coordinate out of range clamps like any query
    big = np.full((n, 4), 5.0, np.float32)
    l1, _ = oracle.oracle_smooth(cfg, n, xyz, t, big, table, want_grad=False)
    y1 = oracle.oracle_fwd(cfg, n, xyz, t, table).astype(np.float64)
    y2 = oracle.oracle_fwd(cfg, n, np.ones((n, 3), np.float32), np.ones(n, np.float32), table).astype(np.float64)
    np.testing.assert_allclose(l1, ((y1 - y2) ** 2).sum(1), rtol=1e-5)


def test_c_oracle_equals_python_bruteforce():
    for (dtype, T, dense) in [("fp32", 1 << 12, True), ("fp16", 5003, False)]:
        L, F = 3, 2
        cfg = oracle.make_config(L, F, T, 4, 40, 2, 9, dtype, dense_coarse=dense)
        rng = np.random.default_rng(5)
        n = 16
        xyz, t = make_queries_uniform(8, n)
        eps = rng.uniform(-0.03, 0.03, (n, 4)).astype(np.float32)
        table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16 if dtype == "fp16" else np.float32)
        loss, grad = oracle.oracle_smooth(cfg, n, xyz, t, eps, table, grad_scale=0.5)
        wl, wg = slow.smooth(np.concatenate([xyz, t[:, None]], 1), eps, table, L, F, T, 4, 40, 2, 9, dense, 0.5)
        np.testing.assert_allclose(loss, wl, rtol=1e-6, atol=1e-12)
        np.testing.assert_allclose(grad, wg, rtol=1e-6, atol=1e-7)
