"""Pins for the oracle's coordinate gradient (Q14/Q24): closed form on
multi-affine tables, exact finite differences of the oracle's own forward on power-of-two grids,
clamp behaviour, and the pure-Python brute force.  CPU only."""
import numpy as np

import oracle
from oracle import slow
from dash_inputs import make_queries_uniform


def test_gradient_of_multi_affine_function_is_reproduced():
    """Table = g on a dense grid, g = prod_d (a_d + b_d x_d): the interpolant IS g, so
    d<dout, out>/dx_d = dout * b_d * prod_{e != d} (a_e + b_e x_e), evaluated at pos/N."""
    ns, nt = 12, 5
    S, St = ns + 1, nt + 1
    cfg = oracle.make_config(1, 1, S ** 3 * St, ns, ns, nt, nt)
    a = np.array([0.3, -1.2, 0.7, 2.0]); b = np.array([1.5, 0.4, -2.2, 0.9])
    gx, gy, gz, gt = np.meshgrid(np.arange(S), np.arange(S), np.arange(S), np.arange(St), indexing="ij")
    vals = ((a[0] + b[0] * gx / ns) * (a[1] + b[1] * gy / ns) * (a[2] + b[2] * gz / ns)
            * (a[3] + b[3] * gt / nt))
    table = np.zeros((1, cfg.T, 1), np.float32)
    table[0, (gx + S * (gy + S * (gz + S * gt))).ravel(), 0] = vals.ravel()
    n = 2000
    xyz, t = make_queries_uniform(4, n)
    dout = np.random.default_rng(1).standard_normal((n, 1)).astype(np.float32)
    dq = oracle.oracle_bwd_input(cfg, n, xyz, t, table, dout)
    p = np.concatenate([(xyz * np.float32(ns)).astype(np.float64) / ns,
                        ((t * np.float32(nt)).astype(np.float64) / nt)[:, None]], 1)
    lin = a[None, :] + b[None, :] * p
    for d in range(4):
        others = np.prod(np.delete(lin, d, axis=1), axis=1)
        want = dout[:, 0].astype(np.float64) * b[d] * others
        scale = np.abs(want).max()
        np.testing.assert_allclose(dq[:, d], want, rtol=0, atol=2e-5 * scale)   # fp32 table entries


def test_finite_differences_of_the_forward_on_pow2_grids():
    """Power-of-two resolutions and coordinates on a 2^-14 lattice: x*N is exact in fp32, the forward is
    exactly linear along one axis inside a cell, so a central difference with h = 2^-13 equals the
    derivative up to the fp32 rounding of the forward's output."""
    L, F, T = 4, 2, 1 << 16
    cfg = oracle.make_config(L, F, T, 16, 128, 8, 64)          # level 0 dense, others hashed
    _, _, dn = oracle.oracle_resolutions(cfg)
    assert dn[0] and not dn[3]
    rng = np.random.default_rng(7)
    n = 400
    # lattice points strictly inside finest-level cells: cell*2^-7 + odd multiple of 2^-12 away from borders
    cells = rng.integers(0, 128, (n, 4)); cells[:, 3] = rng.integers(0, 64, n) * 2
    q = (cells / 128.0 + rng.integers(4, 28, (n, 4)) * 2.0 ** -12).astype(np.float32)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float32)
    dout = rng.standard_normal((n, L * F)).astype(np.float32)
    xyz, t = np.ascontiguousarray(q[:, :3]), np.ascontiguousarray(q[:, 3])
    dq, mag = oracle.oracle_bwd_input(cfg, n, xyz, t, table, dout, want_abs=True)
    h = 2.0 ** -13
    for d in range(4):
        qp, qm = q.copy(), q.copy()
        qp[:, d] += np.float32(h); qm[:, d] -= np.float32(h)
        yp = oracle.oracle_fwd(cfg, n, np.ascontiguousarray(qp[:, :3]), np.ascontiguousarray(qp[:, 3]), table)
        ym = oracle.oracle_fwd(cfg, n, np.ascontiguousarray(qm[:, :3]), np.ascontiguousarray(qm[:, 3]), table)
        fd = ((yp.astype(np.float64) - ym) * dout).sum(1) / (2 * h)
        # forward outputs are fp32-rounded: |y| <= 1 -> 6e-8 * |dout| * L*F / (2h) absolute noise
        noise = 6e-8 * np.abs(dout).sum(1) / (2 * h)
        assert (np.abs(fd - dq[:, d]) <= noise + 1e-6 * mag[:, d]).all()


def test_clamped_coordinates_have_zero_gradient_and_views_work():
    cfg = oracle.make_config(3, 2, 1 << 12, 16, 64, 8, 16)
    rng = np.random.default_rng(2)
    table = rng.uniform(-1, 1, (3, 1 << 12, 2)).astype(np.float32)
    q = rng.random((6, 4), dtype=np.float32)
    q[0, 0] = -0.5; q[1, 1] = 1.0; q[2, 2] = np.nan; q[3, 3] = 7.0
    dout = rng.standard_normal((6, 6)).astype(np.float32)
    xyz, t = np.ascontiguousarray(q[:, :3]), np.ascontiguousarray(q[:, 3])
    dq = oracle.oracle_bwd_input(cfg, 6, xyz, t, table, dout)
    assert dq[0, 0] == 0 and dq[1, 1] == 0 and dq[2, 2] == 0 and dq[3, 3] == 0
    assert np.count_nonzero(dq) == 24 - 4
    # index list + broadcast t
    rows = rng.random((5, 3), dtype=np.float32)
    index = np.array([4, 0, 0, 2], np.int32)
    t0 = np.array([0.3], np.float32)
    d4 = rng.standard_normal((4, 6)).astype(np.float32)
    a = oracle.oracle_bwd_input(cfg, 4, rows, t0, table, d4, index=index, t_stride=0)
    b = oracle.oracle_bwd_input(cfg, 4, np.ascontiguousarray(rows[index]), np.full(4, 0.3, np.float32), table, d4)
    np.testing.assert_array_equal(a, b)


def test_c_oracle_equals_python_bruteforce():
    for (dtype, T, dense) in [("fp32", 1 << 12, True), ("fp16", 5003, False)]:
        L, F = 3, 2
        cfg = oracle.make_config(L, F, T, 4, 40, 2, 9, dtype, dense_coarse=dense)
        rng = np.random.default_rng(5)
        n = 20
        xyz, t = make_queries_uniform(8, n)
        table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16 if dtype == "fp16" else np.float32)
        dout = rng.standard_normal((n, L * F)).astype(np.float32)
        got = oracle.oracle_bwd_input(cfg, n, xyz, t, table, dout)
        want = slow.backward_input(np.concatenate([xyz, t[:, None]], 1), table, dout, L, F, T, 4, 40, 2, 9, dense)
        np.testing.assert_allclose(got, want, rtol=1e-6, atol=1e-6)
