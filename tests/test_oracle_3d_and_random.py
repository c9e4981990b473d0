"""(1) The d = 3 encoder of the decomposition stage (G_3D, Eq. 3) is the
4D encoder with temporal resolution 1 and t = 0: the t-vertex is 0, contributes 0 to the XOR of Eq. 8 and the
upper t-corners have weight 0.  Checked against an independent 8-corner trilinear hash-grid written here.
(2) Randomly generated configurations (hypothesis): C oracle vs the pure-Python transcription.  CPU only."""
import numpy as np
from hypothesis import given, settings, strategies as st

import oracle
from oracle import slow
from dash_inputs import make_queries_uniform

P3 = (1, 2654435761, 805459861)


def trilinear_hash_grid(xyz, table, res, T, dense):
    """Instant-NGP style 3D lookup for ONE level, written from its definition: 8 corners, weights
    prod(bit ? w : 1-w), slot = (x*1 ^ y*pi2 ^ z*pi3) mod T or the dense x-fastest index."""
    out = np.zeros((len(xyz), table.shape[1]))
    for n, p in enumerate(xyz):
        pos = (np.float32(p) * np.float32(res)).astype(np.float32)
        c = np.floor(pos).astype(np.int64); w = (pos - np.floor(pos)).astype(np.float64)
        for k in range(8):
            g = [int(c[d]) + ((k >> d) & 1) for d in range(3)]
            wk = np.prod([w[d] if (k >> d) & 1 else 1 - w[d] for d in range(3)])
            if dense:
                S = res + 1
                s = g[0] + S * (g[1] + S * g[2])
            else:
                s = (((g[0] * P3[0]) & 0xFFFFFFFF) ^ ((g[1] * P3[1]) & 0xFFFFFFFF) ^ ((g[2] * P3[2]) & 0xFFFFFFFF)) % T
            out[n] += wk * table[s].astype(np.float64)
    return out


def test_three_d_encoder_is_the_nt1_t0_special_case():
    L, F, T = 5, 2, 1 << 12
    cfg = oracle.make_config(L, F, T, 4, 64, 1, 1)
    rs, rt, dn = oracle.oracle_resolutions(cfg)
    assert list(rt) == [1] * L and dn[0] and dn[1] and not dn[4]    # 5^3*2, 9^3*2 dense; 65^3*2 hashed
    rng = np.random.default_rng(0)
    n = 200
    xyz, _ = make_queries_uniform(5, n)
    t0 = np.zeros(1, np.float32)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float32)
    out = oracle.oracle_fwd(cfg, n, xyz, t0, table, t_stride=0)
    for l in range(L):
        want = trilinear_hash_grid(xyz, table[l], int(rs[l]), T, bool(dn[l]))
        np.testing.assert_allclose(out[:, l * F:(l + 1) * F], want, rtol=0, atol=3e-7)
    # and the backward touches only slots of t-vertex 0 with non-zero values
    dout = rng.standard_normal((n, L * F)).astype(np.float32)
    g = oracle.oracle_bwd(cfg, n, xyz, t0, dout, t_stride=0)
    np.testing.assert_allclose(g.astype(np.float64).sum(1).reshape(-1), dout.astype(np.float64).sum(0), atol=1e-4)


@settings(max_examples=25, deadline=None)
@given(L=st.integers(1, 5), F=st.sampled_from([1, 2, 4, 8]),
       T=st.one_of(st.sampled_from([1, 2, 64, 4096, 1 << 14]), st.integers(3, 20000)),
       rs=st.tuples(st.integers(1, 40), st.integers(0, 300)), rt=st.tuples(st.integers(1, 12), st.integers(0, 60)),
       dense=st.booleans(), half=st.booleans(), seed=st.integers(0, 2 ** 16))
def test_random_configs_c_oracle_equals_bruteforce(L, F, T, rs, rt, dense, half, seed):
    rs_min, rs_max = rs[0], rs[0] + rs[1]
    rt_min, rt_max = rt[0], rt[0] + rt[1]
    cfg = oracle.make_config(L, F, T, rs_min, rs_max, rt_min, rt_max, "fp16" if half else "fp32",
                             dense_coarse=dense)
    rng = np.random.default_rng(seed)
    n = 6
    q = rng.random((n, 4), dtype=np.float32)
    q[0] = [0.0, 1.0, 0.5, np.float32(1) - np.float32(2.0 ** -24)]      # edges in every example
    xyz, t = np.ascontiguousarray(q[:, :3]), np.ascontiguousarray(q[:, 3])
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16 if half else np.float32)
    dout = rng.standard_normal((n, L * F)).astype(np.float32)
    args = (L, F, T, rs_min, rs_max, rt_min, rt_max, dense)
    out = oracle.oracle_fwd(cfg, n, xyz, t, table)
    np.testing.assert_array_equal(out, slow.forward(q, table, *args).astype(np.float32))
    g = oracle.oracle_bwd(cfg, n, xyz, t, dout)
    np.testing.assert_allclose(g, slow.backward(q, dout, *args), rtol=1e-6, atol=1e-6)
    idx, _ = oracle.oracle_indices(cfg, n, xyz, t)
    assert idx.max() < T
    res_s, res_t, dn = oracle.oracle_resolutions(cfg)
    assert list(res_s) == slow.resolutions(rs_min, rs_max, L) and list(res_t) == slow.resolutions(rt_min, rt_max, L)
