"""Pins for the oracle's forward (quadrilinear interpolation, Eq. 9) and backward
(its transpose).  None of these retype the oracle's formula: they use closed forms, a library
interpolator, linear-algebra identities and brute force.  CPU only."""
import numpy as np
import pytest
from scipy.interpolate import RegularGridInterpolator

import oracle
from oracle import slow
from dash_inputs import CONFIGS, make_queries_uniform, make_workload


def _cfg(L=4, F=2, T=1 << 12, rs=(16, 128), rt=(8, 32), **kw):
    return oracle.make_config(L, F, T, rs[0], rs[1], rt[0], rt[1], **kw)


def _rand_table(cfg, seed=0, dtype=np.float32):
    rng = np.random.default_rng(seed)
    return rng.uniform(-1, 1, size=(cfg.L, cfg.T, cfg.F)).astype(dtype)


# ---------------------------------------------------------------- weights

def test_weights_sum_to_one_nonneg_and_product_form():
    cfg = oracle.config_from_params(CONFIGS["C2"].enc)
    xyz, t = make_queries_uniform(3, 2000)
    idx, w = oracle.oracle_indices(cfg, 2000, xyz, t)
    assert (w >= 0).all() and (w <= 1).all()
    np.testing.assert_allclose(w.sum(-1), 1.0, rtol=0, atol=16 * 2.3e-16)
    # separability: W_k * W_(15-k) is the same for every k (= prod_d w_d (1-w_d))
    prod = w * w[..., ::-1]
    np.testing.assert_allclose(prod, prod[..., :1] * np.ones(16), rtol=1e-12, atol=1e-300)
    # marginal over the three other axes gives the 1-D weight: sum over corners with bit d set = w_d
    rs, rt, _ = oracle.oracle_resolutions(cfg)
    k = np.arange(16)
    for d in range(4):
        res = (rs if d < 3 else rt).astype(np.float32)
        coord = xyz[:, d] if d < 3 else t
        pos = coord[:, None] * res[None, :]                      # fp32 multiply (numpy)
        frac = (pos - np.floor(pos)).astype(np.float64)
        got = w[..., (k >> d) & 1 == 1].sum(-1)
        np.testing.assert_allclose(got, frac, rtol=0, atol=1e-15)


def test_corner_order_bit_d_is_plus_one_along_d():
    """Q6: on a dense level slot differences expose the corner order: +1 in x -> +1, y -> +S, z -> +S^2, t -> +S^3."""
    cfg = oracle.config_from_params(CONFIGS["C2"].enc)
    xyz, t = make_queries_uniform(5, 64)
    idx, _ = oracle.oracle_indices(cfg, 64, xyz, t)
    S = 17
    base = idx[:, 0, 0].astype(np.int64)
    for k in range(16):
        off = (k & 1) + S * ((k >> 1) & 1) + S * S * ((k >> 2) & 1) + S ** 3 * ((k >> 3) & 1)
        assert (idx[:, 0, k].astype(np.int64) - base == off).all()


# ---------------------------------------------------------------- exact at vertices

@pytest.mark.parametrize("dense_coarse", [True, False])
def test_exact_table_value_at_grid_vertices(dense_coarse):
    """All-power-of-two schedule (16->128 spatial, 8->64 temporal, L=4): x = i/N is exact in fp32, so the
    fractional offsets are 0 and the output must equal the table entry of that vertex BIT-exactly."""
    L, F, T = 4, 2, 1 << 17
    cfg = oracle.make_config(L, F, T, 16, 128, 8, 64, dense_coarse=dense_coarse)
    rs, rt, dn = oracle.oracle_resolutions(cfg)
    assert list(rs) == [16, 32, 64, 128] and list(rt) == [8, 16, 32, 64]
    assert dn[0] == dense_coarse
    table = _rand_table(cfg, 1)
    rng = np.random.default_rng(2)
    n = 500
    g = np.stack([rng.integers(0, 16, n), rng.integers(0, 16, n), rng.integers(0, 16, n),
                  rng.integers(0, 8, n)], 1)
    xyz = (g[:, :3] / 16.0).astype(np.float32)     # vertices of level 0 are vertices of every level
    t = (g[:, 3] / 8.0).astype(np.float32)
    out = oracle.oracle_fwd(cfg, n, xyz, t, table)
    for l in range(L):
        mult_s, mult_t = int(rs[l]) // 16, int(rt[l]) // 8
        for i in range(n):
            v = (g[i, 0] * mult_s, g[i, 1] * mult_s, g[i, 2] * mult_s, g[i, 3] * mult_t)
            s = oracle.oracle_vertex_slot(cfg, l, v)
            assert (out[i, l * F:(l + 1) * F] == table[l, s]).all()


def test_constant_table_gives_constant():
    cfg = _cfg()
    table = np.full((cfg.L, cfg.T, cfg.F), 0.37, np.float32)
    xyz, t = make_queries_uniform(9, 1000)
    out = oracle.oracle_fwd(cfg, 1000, xyz, t, table)
    np.testing.assert_allclose(out, np.float32(0.37), rtol=1e-7)


# ---------------------------------------------------------------- multi-affine reproduction + scipy

def _dense_single_level(ns, nt, F=1):
    S, St = ns + 1, nt + 1
    T = S ** 3 * St
    cfg = oracle.make_config(1, F, T, ns, ns, nt, nt)
    _, _, dn = oracle.oracle_resolutions(cfg)
    assert dn[0]
    return cfg, S, St


def test_multi_affine_functions_are_reproduced():
    """Quadrilinear interpolation is exact on g(x) = prod_d (a_d + b_d x_d).  Table filled on the dense
    grid (x fastest); expected value evaluated in double directly from the closed form."""
    ns, nt = 12, 5                                   # non-power-of-two on purpose
    cfg, S, St = _dense_single_level(ns, nt)
    a = np.array([0.3, -1.2, 0.7, 2.0]); b = np.array([1.5, 0.4, -2.2, 0.9])
    gx, gy, gz, gt = np.meshgrid(np.arange(S), np.arange(S), np.arange(S), np.arange(St), indexing="ij")
    vals = ((a[0] + b[0] * gx / ns) * (a[1] + b[1] * gy / ns) * (a[2] + b[2] * gz / ns)
            * (a[3] + b[3] * gt / nt))
    table = np.zeros((1, cfg.T, 1), np.float64)
    table[0, (gx + S * (gy + S * (gz + S * gt))).ravel(), 0] = vals.ravel()
    table32 = table.astype(np.float32)
    xyz, t = make_queries_uniform(4, 3000)
    out = oracle.oracle_fwd(cfg, 3000, xyz, t, table32)[:, 0]
    # the oracle interpolates at pos/N with pos = fl32(x*N): evaluate g there
    px = (xyz * np.float32(ns)).astype(np.float64) / ns
    pt = (t * np.float32(nt)).astype(np.float64) / nt
    want = ((a[0] + b[0] * px[:, 0]) * (a[1] + b[1] * px[:, 1]) * (a[2] + b[2] * px[:, 2])
            * (a[3] + b[3] * pt))
    scale = np.abs(vals).max()
    np.testing.assert_allclose(out, want, rtol=0, atol=4e-7 * scale)   # fp32 table + fp32 output rounding


@pytest.mark.parametrize("ns,nt,F", [(16, 8, 2), (9, 4, 1)])
def test_matches_scipy_regular_grid_interpolator(ns, nt, F):
    cfg, S, St = _dense_single_level(ns, nt, F)
    table = _rand_table(cfg, 5)
    xyz, t = make_queries_uniform(6, 2000)
    out = oracle.oracle_fwd(cfg, 2000, xyz, t, table)
    pts = np.concatenate([(xyz * np.float32(ns)).astype(np.float64),
                          (t * np.float32(nt)).astype(np.float64)[:, None]], 1)
    for f in range(F):
        grid = table[0, :, f].astype(np.float64).reshape(St, S, S, S).transpose(3, 2, 1, 0)  # [x][y][z][t]
        rgi = RegularGridInterpolator((np.arange(S), np.arange(S), np.arange(S), np.arange(St)), grid,
                                      method="linear")
        np.testing.assert_allclose(out[:, f], rgi(pts), rtol=0, atol=2e-7)


def test_t_on_vertex_reduces_to_trilinear():
    """with t on a temporal vertex the 4D interpolation is the 3D (Instant-NGP) trilinear one
    on that time slice — checked against scipy's 3D interpolator."""
    ns, nt = 10, 4
    cfg, S, St = _dense_single_level(ns, nt)
    table = _rand_table(cfg, 8)
    xyz, _ = make_queries_uniform(7, 1000)
    for j in range(nt):
        t = np.full(1000, j / nt, np.float32)        # quarters: exact
        out = oracle.oracle_fwd(cfg, 1000, xyz, t, table)[:, 0]
        vol = table[0, :, 0].astype(np.float64).reshape(St, S, S, S)[j].transpose(2, 1, 0)
        rgi = RegularGridInterpolator((np.arange(S),) * 3, vol, method="linear")
        np.testing.assert_allclose(out, rgi((xyz * np.float32(ns)).astype(np.float64)), rtol=0, atol=2e-7)


# ---------------------------------------------------------------- brute force (second transcription)

@pytest.mark.parametrize("name,kw", [("C1", {}), ("C2", {}), ("C2", {"dense_coarse": False})])
def test_c_oracle_equals_python_bruteforce(name, kw):
    enc = CONFIGS[name].enc
    L, F = enc.L, enc.F
    T = 1 << 12 if name == "C1" else enc.T
    cfg = oracle.make_config(L, F, T, enc.res_s_min, enc.res_s_max, enc.res_t_min, enc.res_t_max, **kw)
    n = 24
    wl = make_workload(name, n_override=n, with_table=False, with_dout=False)
    rng = np.random.default_rng(21)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float32)
    dout = rng.standard_normal((n, L * F)).astype(np.float32)
    q = np.concatenate([wl.xyz, wl.t[:, None]], 1)
    args = (L, F, T, enc.res_s_min, enc.res_s_max, enc.res_t_min, enc.res_t_max, kw.get("dense_coarse", True))
    out = oracle.oracle_fwd(cfg, n, wl.xyz, wl.t, table)
    np.testing.assert_array_equal(out, slow.forward(q, table, *args).astype(np.float32))
    g = oracle.oracle_bwd(cfg, n, wl.xyz, wl.t, dout)
    np.testing.assert_allclose(g, slow.backward(q, dout, *args), rtol=1e-6, atol=1e-7)
    idx, w = oracle.oracle_indices(cfg, n, wl.xyz, wl.t)
    rs, rt, dn = slow.plan(*args[:1], T, *args[3:])
    for i in range(n):
        for l in range(L):
            ref = slow.corners(q[i], rs[l], rt[l], T, dn[l])
            assert [s for s, _ in ref] == list(idx[i, l])
            np.testing.assert_allclose([x for _, x in ref], w[i, l], rtol=1e-15)


def test_non_pow2_table_and_fp16_table_bruteforce():
    L, F, T = 3, 4, 100003
    cfg = oracle.make_config(L, F, T, 16, 200, 8, 40, "fp16")
    xyz, t = make_queries_uniform(31, 16)
    rng = np.random.default_rng(3)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16)
    out = oracle.oracle_fwd(cfg, 16, xyz, t, table)
    q = np.concatenate([xyz, t[:, None]], 1)
    want = slow.forward(q, table, L, F, T, 16, 200, 8, 40)
    np.testing.assert_array_equal(out, want.astype(np.float32))
    idx, _ = oracle.oracle_indices(cfg, 16, xyz, t)
    assert idx.max() < T


# ---------------------------------------------------------------- linear-map identities

def test_linearity_in_the_table_and_level_independence():
    cfg = oracle.config_from_params(CONFIGS["C1"].enc)
    xyz, t = make_queries_uniform(1, 500)
    A, B = _rand_table(cfg, 1), _rand_table(cfg, 2)
    yA, yB = oracle.oracle_fwd(cfg, 500, xyz, t, A), oracle.oracle_fwd(cfg, 500, xyz, t, B)
    comb = (np.float32(2) * A + np.float32(0.5) * B).astype(np.float32)     # exact scalings, one rounding
    yC = oracle.oracle_fwd(cfg, 500, xyz, t, comb)
    np.testing.assert_allclose(yC, 2 * yA.astype(np.float64) + 0.5 * yB, rtol=0, atol=3e-7)
    # columns of level l depend only on table[l]
    A2 = A.copy(); A2[2] = B[2]
    y2 = oracle.oracle_fwd(cfg, 500, xyz, t, A2)
    F = cfg.F
    assert (y2[:, :2 * F] == yA[:, :2 * F]).all() and (y2[:, 3 * F:] == yA[:, 3 * F:]).all()
    assert (y2[:, 2 * F:3 * F] == yB[:, 2 * F:3 * F]).all()


@pytest.mark.parametrize("name", ["C1", "C2"])
def test_adjoint_identity(name):
    """<J theta, g> = <theta, J^T g> in double."""
    n = 3000
    wl = make_workload(name, n_override=n)
    cfg = oracle.config_from_params(wl.spec.enc)
    table = wl.table.astype(np.float32)
    y = oracle.oracle_fwd(cfg, n, wl.xyz, wl.t, table).astype(np.float64)
    g = oracle.oracle_bwd(cfg, n, wl.xyz, wl.t, wl.dout).astype(np.float64)
    lhs = (y * wl.dout).sum()
    rhs = (table.astype(np.float64) * g).sum()
    scale = np.abs(y * wl.dout).sum()
    assert abs(lhs - rhs) <= 2e-6 * scale


def test_finite_difference_equals_jacobian_column():
    """The map is linear in the table: (y(theta + h e_j) - y(theta))/h = J e_j, and J^T g picks the same
    numbers: dtable[j] = sum_n g_n * (J e_j)_n."""
    cfg = oracle.make_config(2, 2, 2048, 4, 8, 2, 4)            # level 0 dense (5^3*3=375), level 1 hashed (3645 > T)
    _, _, dn = oracle.oracle_resolutions(cfg)
    assert dn[0] and not dn[1]
    xyz, t = make_queries_uniform(13, 200)
    rng = np.random.default_rng(5)
    table = rng.uniform(-1, 1, (2, 2048, 2)).astype(np.float32)
    dout = rng.standard_normal((200, 4)).astype(np.float32)
    y0 = oracle.oracle_fwd(cfg, 200, xyz, t, table).astype(np.float64)
    g = oracle.oracle_bwd(cfg, 200, xyz, t, dout).astype(np.float64)
    idx, _ = oracle.oracle_indices(cfg, 200, xyz, t)
    h = 0.25
    for l in range(2):
        touched = np.unique(idx[:, l])
        for s in list(touched[:6]) + list(touched[-3:]):
            for f in range(2):
                tp = table.copy(); tp[l, s, f] += np.float32(h)
                col = (oracle.oracle_fwd(cfg, 200, xyz, t, tp).astype(np.float64) - y0) / h
                assert np.abs(col[:, [c for c in range(4) if c != l * 2 + f]]).max() == 0
                np.testing.assert_allclose((col * dout).sum(), g[l, s, f], rtol=2e-5, atol=2e-6)


def test_backward_checksum_and_unit_gradient():
    """sum over slots of dtable[l][.][f] = sum_n dY[n][lF+f] (weights sum to 1); and a one-hot dY returns
    exactly the 16 (slot, W) pairs of `indices`."""
    name = "C2"
    n = 2000
    wl = make_workload(name, n_override=n)
    cfg = oracle.config_from_params(wl.spec.enc)
    L, F = cfg.L, cfg.F
    g, hits = oracle.oracle_bwd(cfg, n, wl.xyz, wl.t, wl.dout, want_hits=True)
    np.testing.assert_allclose(g.astype(np.float64).sum(1).reshape(-1),
                               wl.dout.astype(np.float64).sum(0), rtol=0, atol=2e-4)
    assert (hits.sum(1) == 16 * n).all()
    idx, w = oracle.oracle_indices(cfg, n, wl.xyz, wl.t)
    for (q, l, f) in [(0, 0, 0), (17, 5, 1), (1999, 15, 0)]:
        d = np.zeros((n, L * F), np.float32); d[q, l * F + f] = 1.0
        gg = oracle.oracle_bwd(cfg, n, wl.xyz, wl.t, d)
        want = np.zeros(cfg.T)
        np.add.at(want, idx[q, l], w[q, l])
        np.testing.assert_array_equal(gg[l, :, f], want.astype(np.float32))
        gg[l, :, f] = 0
        assert not gg.any()


def test_backward_accumulates_into_dtable():
    cfg = oracle.config_from_params(CONFIGS["C1"].enc)
    wl = make_workload("C1", n_override=300)
    g0 = oracle.oracle_bwd(cfg, 300, wl.xyz, wl.t, wl.dout)
    init = np.full((cfg.L, cfg.T, cfg.F), 3.0, np.float32)
    g1 = oracle.oracle_bwd(cfg, 300, wl.xyz, wl.t, wl.dout, dtable=init.copy())
    np.testing.assert_allclose(g1, g0 + 3.0, rtol=0, atol=5e-7)


# ---------------------------------------------------------------- input views

def test_index_list_broadcast_t_and_packed_rows():
    cfg = oracle.config_from_params(CONFIGS["C1"].enc)
    rng = np.random.default_rng(17)
    rows = rng.random((50, 3), dtype=np.float32)
    index = rng.integers(0, 50, 200).astype(np.int32)
    t = rng.random(200, dtype=np.float32)
    table = _rand_table(cfg, 3)
    a = oracle.oracle_fwd(cfg, 200, rows, t, table, index=index)
    b = oracle.oracle_fwd(cfg, 200, np.ascontiguousarray(rows[index]), t, table)
    np.testing.assert_array_equal(a, b)
    # one timestamp for all (t_stride = 0)
    t0 = np.array([0.3125], np.float32)
    c = oracle.oracle_fwd(cfg, 200, rows, t0, table, index=index, t_stride=0)
    d = oracle.oracle_fwd(cfg, 200, rows, np.full(200, 0.3125, np.float32), table, index=index)
    np.testing.assert_array_equal(c, d)
    # packed [N][4] rows: xyz stride 4, t = base+3 stride 4
    packed = np.ascontiguousarray(np.concatenate([rows, rng.random((50, 1), dtype=np.float32)], 1))
    e = oracle.oracle_fwd(cfg, 50, packed, packed.reshape(-1)[3:], table, t_stride=4)
    f = oracle.oracle_fwd(cfg, 50, np.ascontiguousarray(packed[:, :3]), np.ascontiguousarray(packed[:, 3]), table)
    np.testing.assert_array_equal(e, f)


def test_empty_and_invalid():
    cfg = oracle.config_from_params(CONFIGS["C1"].enc)
    xyz, t = make_queries_uniform(0, 4)
    table = _rand_table(cfg, 0)
    out = oracle.oracle_fwd(cfg, 0, xyz, t, table)
    assert out.shape == (0, cfg.L * cfg.F)
    bad = oracle.make_config(4, 3, 64, 16, 128, 8, 32)            # F = 3 unsupported
    with pytest.raises(RuntimeError):
        oracle.oracle_resolutions(bad)
    bad = oracle.make_config(4, 2, 64, 128, 16, 8, 32)            # min > max
    with pytest.raises(RuntimeError):
        oracle.oracle_resolutions(bad)
