"""Pins for the oracle's TOLERANCE TERMS (DESIGN.md §3 Q17, SURVEY.md:381): the conditioning sums
A = sum |W * v| that every elementwise GPU tolerance is a multiple of (`out_abs`, `grad_abs`, `hits`,
`dq_abs`, and the smooth `loss_abs` / `feat_abs` / `grad_abs`), for the 4D and the 3D functions.

A slip in one of those accumulations (`mag += fabs(W[k])`, a dropped fabs, a term counted twice) would pass
every other CPU test and silently loosen the GPU checks.  Two independent pins per term:
  (i)  sign structure: with all terms >= 0 the conditioning sum must EQUAL the value itself;
  (ii) numpy rebuild from the oracle's own (pinned) indices and weights: np.add.at / np.bincount.
Neither retypes the C loops.  CPU only.
"""
import numpy as np
import pytest

import oracle
from dash_inputs import make_queries_uniform


def _setup(seed=0, n=700, L=5, F=2, T=1 << 12, dtype=np.float32, table_dtype="fp32"):
    # levels 0-1 dense ((8+1)^3 (4+1) = 3645 <= 4096), the rest hashed with many collisions
    cfg = oracle.make_config(L, F, T, 8, 96, 4, 24, table_dtype=table_dtype)
    rng = np.random.default_rng(seed)
    xyz, t = make_queries_uniform(seed, n)
    table = rng.uniform(-1, 1, (L, T, F)).astype(dtype)
    dout = rng.standard_normal((n, L * F)).astype(np.float32)
    return cfg, xyz, t, table, dout


# ------------------------------------------------------------------------------------------ forward A

def test_out_abs_equals_out_for_nonnegative_table():
    cfg, xyz, t, table, _ = _setup(1)
    n = len(t)
    out, mag = oracle.oracle_fwd(cfg, n, xyz, t, np.abs(table), want_abs=True)
    assert (mag > 0).all()
    np.testing.assert_array_equal(mag.astype(np.float32), out)          # same double sum, rounded once
    out_n, mag_n = oracle.oracle_fwd(cfg, n, xyz, t, -np.abs(table), want_abs=True)
    np.testing.assert_array_equal(mag_n, mag)                            # |.| removes the sign
    np.testing.assert_array_equal(out_n, -out)


@pytest.mark.parametrize("table_dtype,dtype", [("fp32", np.float32), ("fp16", np.float16)])
def test_out_abs_rebuilt_from_indices(table_dtype, dtype):
    cfg, xyz, t, table, _ = _setup(2, dtype=dtype, table_dtype=table_dtype)
    n, L, F = len(t), cfg.L, cfg.F
    idx, w = oracle.oracle_indices(cfg, n, xyz, t)
    _, mag = oracle.oracle_fwd(cfg, n, xyz, t, table, want_abs=True)
    tab = table.astype(np.float64)
    lev = np.arange(L)[None, :, None]
    want = (w[..., None] * np.abs(tab[lev, idx])).sum(2).reshape(n, L * F)   # [N][L][16][F] -> [N][L*F]
    np.testing.assert_allclose(mag, want, rtol=1e-13, atol=0)
    # and it is strictly tighter than the "weights only" slip  sum_k |W_k| = 1
    assert (mag < 1.0).all() and (mag >= np.abs(oracle.oracle_fwd(cfg, n, xyz, t, table)) * (1 - 1e-6)).all()


# ------------------------------------------------------------------------------------------ backward A, hits

def test_grad_abs_equals_dtable_for_nonnegative_dout():
    cfg, xyz, t, _, dout = _setup(3)
    n = len(t)
    g, mag, hits = oracle.oracle_bwd(cfg, n, xyz, t, np.abs(dout), want_abs=True, want_hits=True)
    np.testing.assert_array_equal(mag.astype(np.float32), g)
    assert ((mag.sum(-1) > 0) == (hits > 0)).all()                       # touched <=> counted


def test_grad_abs_and_hits_rebuilt_from_indices():
    cfg, xyz, t, _, dout = _setup(4)
    n, L, F, T = len(t), cfg.L, cfg.F, cfg.T
    idx, w = oracle.oracle_indices(cfg, n, xyz, t)
    _, mag, hits = oracle.oracle_bwd(cfg, n, xyz, t, dout, want_abs=True, want_hits=True)
    d = np.abs(dout.astype(np.float64)).reshape(n, L, 1, F)
    contrib = w[..., None] * d                                           # [N][L][16][F]
    want = np.zeros((L, T, F))
    cnt = np.zeros((L, T), np.int64)
    for l in range(L):
        np.add.at(want[l], idx[:, l].ravel(), contrib[:, l].reshape(-1, F))
        cnt[l] = np.bincount(idx[:, l].ravel(), minlength=T)
    np.testing.assert_allclose(mag, want, rtol=1e-12, atol=0)
    np.testing.assert_array_equal(hits.astype(np.int64), cnt)
    assert hits.sum() == n * L * 16 and hits.max() > 4                   # collisions are present


def test_grad_abs_is_independent_of_initial_dtable():
    cfg, xyz, t, _, dout = _setup(5)
    n = len(t)
    g0, m0 = oracle.oracle_bwd(cfg, n, xyz, t, dout, want_abs=True)
    start = np.full((cfg.L, cfg.T, cfg.F), 3.0, np.float32)
    g1, m1 = oracle.oracle_bwd(cfg, n, xyz, t, dout, dtable=start.copy(), want_abs=True)
    np.testing.assert_array_equal(m0, m1)                                # A covers the call's own terms only
    np.testing.assert_allclose(g1, g0.astype(np.float64) + 3.0, rtol=0, atol=5e-7)


# ------------------------------------------------------------------------------------------ coordinate gradient A

def test_dq_abs_rebuilt_from_unit_differences():
    """|term| = |dout| N_d |dW_k/dw_d| |v|; the weight derivative magnitude is rebuilt from the oracle's pinned
    weights: |dW_k/dw_d| = W_k / omega_d(k), omega_d(k) = marginal weight of the corner's side along d."""
    cfg, xyz, t, table, dout = _setup(6, n=300)
    n, L, F = len(t), cfg.L, cfg.F
    idx, w = oracle.oracle_indices(cfg, n, xyz, t)
    _, mag = oracle.oracle_bwd_input(cfg, n, xyz, t, table, dout, want_abs=True)
    rs, rt, _ = oracle.oracle_resolutions(cfg)
    k = np.arange(16)
    tab = np.abs(table.astype(np.float64))[np.arange(L)[None, :, None], idx]      # [N][L][16][F]
    s = (tab * np.abs(dout.astype(np.float64)).reshape(n, L, 1, F)).sum(-1)       # [N][L][16]
    want = np.zeros((n, 4))
    for d in range(4):
        bit = ((k >> d) & 1).astype(bool)
        w_hi = w[..., bit].sum(-1, keepdims=True)                                  # = w_d
        omega = np.where(bit[None, None, :], w_hi, 1.0 - w_hi)
        with np.errstate(divide="ignore", invalid="ignore"):
            dw = np.where(omega > 1e-9, w / omega, np.nan)
        ok = ~np.isnan(dw).any(axis=(1, 2))                                        # skip queries sitting on a vertex
        res = (rs if d < 3 else rt).astype(np.float64)[None, :, None]
        want[:, d] = np.where(ok, (np.nan_to_num(dw) * res * s).sum((1, 2)), np.nan)
    sel = ~np.isnan(want)
    assert sel.mean() > 0.9
    np.testing.assert_allclose(mag[sel], want[sel], rtol=1e-7, atol=0)


def test_dq_abs_equals_dq_when_all_terms_share_a_sign():
    """Table increasing in every coordinate direction is impossible under a hash, so use ONE dense level and
    v(vertex) = g_x (monotone along x, constant along the other axes): every x-term is +, so dq_abs[.,0] = dq[.,0],
    and the other axes' terms cancel pairwise: dq = 0 while dq_abs > 0 — the bound is not the value there."""
    ns, nt = 10, 3
    S = ns + 1
    cfg = oracle.make_config(1, 1, S ** 3 * (nt + 1), ns, ns, nt, nt)
    gx = np.arange(S ** 3 * (nt + 1)) % S
    table = (1.0 + gx).astype(np.float32).reshape(1, -1, 1)
    n = 400
    xyz, t = make_queries_uniform(7, n)
    dout = np.ones((n, 1), np.float32)
    dq, mag = oracle.oracle_bwd_input(cfg, n, xyz, t, table, dout, want_abs=True)
    np.testing.assert_allclose(dq[:, 0], ns, rtol=1e-6)                           # d/dx of (1 + ns x) = ns
    np.testing.assert_allclose(dq[:, 1:], 0, atol=1e-4)
    # x axis: |terms| = N * |dW| * v with dW = -/+: sum |.| = ns * (v_lo + v_hi) weighted = ns (2 (1 + c) + 1)
    cell = np.floor(xyz[:, 0] * np.float32(ns)).astype(np.float64)
    np.testing.assert_allclose(mag[:, 0], ns * (2 * (1 + cell) + 1), rtol=1e-12)
    assert (mag[:, 1:] > 1.0).all()


# ------------------------------------------------------------------------------------------ smooth A terms

def test_smooth_abs_terms_rebuilt_from_two_forwards():
    cfg, xyz, t, table, _ = _setup(8, n=400)
    n, L, F, T = len(t), cfg.L, cfg.F, cfg.T
    eps = np.random.default_rng(9).uniform(-2e-2, 2e-2, (n, 4)).astype(np.float32)
    gs = 0.375
    loss, grad, la, fa, ga = oracle.oracle_smooth(cfg, n, xyz, t, eps, table, grad_scale=gs, want_abs=True)
    x2 = (xyz + eps[:, :3]).astype(np.float32)
    t2 = (t + eps[:, 3]).astype(np.float32)
    y1, a1 = oracle.oracle_fwd(cfg, n, xyz, t, table, want_abs=True)
    y2, a2 = oracle.oracle_fwd(cfg, n, x2, t2, table, want_abs=True)
    A = a1 + a2                                                                    # [N][L*F]
    # fp32-rounded forwards give d to ~1e-7 * A; the oracle's own d is in double
    idx1, w1 = oracle.oracle_indices(cfg, n, xyz, t)
    idx2, w2 = oracle.oracle_indices(cfg, n, x2, t2)
    tab = table.astype(np.float64)
    lev = np.arange(L)[None, :, None]
    d = ((w1[..., None] * tab[lev, idx1]).sum(2) - (w2[..., None] * tab[lev, idx2]).sum(2)).reshape(n, L * F)
    np.testing.assert_allclose(fa, A.max(1), rtol=1e-13)
    np.testing.assert_allclose(la, (2 * np.abs(d) * A).sum(1), rtol=1e-9, atol=1e-18)
    want = np.zeros((L, T, F))
    Ar = A.reshape(n, L, 1, F)
    for l in range(L):
        np.add.at(want[l], idx1[:, l].ravel(), (2 * gs * w1[:, l, :, None] * Ar[:, l]).reshape(-1, F))
        np.add.at(want[l], idx2[:, l].ravel(), (2 * gs * w2[:, l, :, None] * Ar[:, l]).reshape(-1, F))
    np.testing.assert_allclose(ga, want, rtol=1e-12, atol=0)
    assert (np.abs(grad) <= ga * (1 + 1e-6) + 1e-30).all()                         # a bound on the value it guards


def test_smooth_abs_terms_scale_with_the_table_not_with_the_weights():
    """Scaling the table by c scales loss_abs by c^2, feat_abs by c, grad_abs by c (it multiplies |W| by A)."""
    cfg, xyz, t, table, _ = _setup(10, n=200)
    n = len(t)
    eps = np.random.default_rng(11).uniform(-1e-2, 1e-2, (n, 4)).astype(np.float32)
    _, _, la, fa, ga = oracle.oracle_smooth(cfg, n, xyz, t, eps, table, want_abs=True)
    _, _, lb, fb, gb = oracle.oracle_smooth(cfg, n, xyz, t, eps, (4 * table).astype(np.float32), want_abs=True)
    np.testing.assert_allclose(lb, 16 * la, rtol=1e-12)
    np.testing.assert_allclose(fb, 4 * fa, rtol=1e-12)
    np.testing.assert_allclose(gb, 4 * ga, rtol=1e-12)


# ------------------------------------------------------------------------------------------ G_3D

def test_3d_abs_terms_and_hits_rebuilt_from_indices():
    L, F, T = 5, 2, 1 << 11
    cfg = oracle.make_config(L, F, T, 8, 128, 1, 1)
    rng = np.random.default_rng(12)
    n = 600
    xyz, _ = make_queries_uniform(12, n)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float32)
    dout = rng.standard_normal((n, L * F)).astype(np.float32)
    idx, w = oracle.oracle3d_indices(cfg, n, xyz)
    out, omag = oracle.oracle3d_fwd(cfg, n, xyz, table, want_abs=True)
    g, gmag, hits = oracle.oracle3d_bwd(cfg, n, xyz, dout, want_abs=True, want_hits=True)
    tab = np.abs(table.astype(np.float64))
    lev = np.arange(L)[None, :, None]
    np.testing.assert_allclose(omag, (w[..., None] * tab[lev, idx]).sum(2).reshape(n, L * F), rtol=1e-13)
    want = np.zeros((L, T, F))
    d = np.abs(dout.astype(np.float64)).reshape(n, L, 1, F)
    for l in range(L):
        np.add.at(want[l], idx[:, l].ravel(), (w[:, l, :, None] * d[:, l]).reshape(-1, F))
        np.testing.assert_array_equal(hits[l], np.bincount(idx[:, l].ravel(), minlength=T))
    np.testing.assert_allclose(gmag, want, rtol=1e-12)
    # sign structure
    o2, m2 = oracle.oracle3d_fwd(cfg, n, xyz, np.abs(table), want_abs=True)
    np.testing.assert_array_equal(m2.astype(np.float32), o2)
    g2, gm2 = oracle.oracle3d_bwd(cfg, n, xyz, np.abs(dout), want_abs=True)
    np.testing.assert_array_equal(gm2.astype(np.float32), g2)


# ------------------------------------------------------------------------------------------ MLP A (Q27)

def _pack(ws, bs):
    return np.concatenate([np.concatenate([w.ravel(), b]) for w, b in zip(ws, bs)]).astype(np.float32)


@pytest.mark.parametrize("quant", [False, True])
def test_mlp_abs_is_the_abs_weight_chain_and_equals_out_when_nonnegative(quant):
    """A_l = |b_l| + |W_l| A_{l-1}, A_0 = |x|, no relu on A (Q27), plus |base|: rebuilt with numpy
    matmuls; with non-negative x, W, b, base every relu is the identity and every term is >= 0, so A == out."""
    rng = np.random.default_rng(13)
    widths = [24, 40, 33, 10]
    ws = [(rng.uniform(-1, 1, (widths[l], widths[l - 1])) / np.sqrt(widths[l - 1])).astype(np.float32)
          for l in range(1, len(widths))]
    bs = [rng.uniform(-0.5, 0.5, widths[l]).astype(np.float32) for l in range(1, len(widths))]
    x = rng.standard_normal((40, widths[0])).astype(np.float32)
    base = rng.standard_normal((40, widths[-1])).astype(np.float32)
    m = oracle.make_mlp_config(widths, quant_bf16=quant)
    _, mag = oracle.oracle_mlp(m, x, _pack(ws, bs), base=base, want_abs=True)
    rnd = (lambda a: np.vectorize(oracle.oracle_to_bf16)(a.astype(np.float64))) if quant else (lambda a: a.astype(np.float64))
    A = np.abs(x.astype(np.float64))
    for w, b in zip(ws, bs):
        A = A @ np.abs(rnd(w)).T + np.abs(b.astype(np.float64))
    np.testing.assert_allclose(mag, A + np.abs(base.astype(np.float64)), rtol=1e-12)
    if not quant:
        pos = _pack([np.abs(w) for w in ws], [np.abs(b) for b in bs])
        out, mag2 = oracle.oracle_mlp(m, np.abs(x), pos, base=np.abs(base), want_abs=True)
        np.testing.assert_array_equal(mag2.astype(np.float32), out)
