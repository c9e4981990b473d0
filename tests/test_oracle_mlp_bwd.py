"""Pins for the oracle's backward through phi_d / the heads (oracle_mlp_bwd; Q30): torch autograd in float64
(a library routine), a hand-worked example with a dead relu, exact finite differences of the pinned forward, sign
structure and numpy rebuilds of the tolerance terms, bf16 operand rounding on representable inputs.  CPU only."""
import numpy as np
import pytest
import torch

import oracle


def pack(ws, bs):
    return np.concatenate([np.concatenate([w.ravel(), b]) for w, b in zip(ws, bs)]).astype(np.float32)


def unpack(vec, widths):
    ws, bs, o = [], [], 0
    for l in range(1, len(widths)):
        J, K = widths[l], widths[l - 1]
        ws.append(vec[o:o + J * K].reshape(J, K)); o += J * K
        bs.append(vec[o:o + J]); o += J
    return ws, bs


def rand_chain(seed, widths, n):
    rng = np.random.default_rng(seed)
    ws = [(rng.uniform(-1, 1, (widths[l], widths[l - 1])) / np.sqrt(widths[l - 1])).astype(np.float32)
          for l in range(1, len(widths))]
    bs = [rng.uniform(-0.3, 0.3, widths[l]).astype(np.float32) for l in range(1, len(widths))]
    x = rng.standard_normal((n, widths[0])).astype(np.float32)
    dout = rng.standard_normal((n, widths[-1])).astype(np.float32)
    return ws, bs, x, dout


@pytest.mark.parametrize("widths", [[7, 5], [12, 9, 4], [32, 48, 40, 10], [16, 24, 24, 24, 6]])
def test_matches_torch_autograd_float64(widths):
    ws, bs, x, dout = rand_chain(sum(widths), widths, 60)
    tw = [torch.tensor(w, dtype=torch.float64, requires_grad=True) for w in ws]
    tb = [torch.tensor(b, dtype=torch.float64, requires_grad=True) for b in bs]
    tx = torch.tensor(x, dtype=torch.float64, requires_grad=True)
    a = tx
    for l, (w, b) in enumerate(zip(tw, tb)):
        a = torch.nn.functional.linear(a, w, b)
        if l < len(tw) - 1:
            a = torch.relu(a)
    (a * torch.tensor(dout, dtype=torch.float64)).sum().backward()
    dfeat, dparams = oracle.oracle_mlp_bwd(oracle.make_mlp_config(widths), x, pack(ws, bs), dout)
    np.testing.assert_allclose(dfeat, tx.grad.numpy().astype(np.float32), rtol=2e-7, atol=1e-30)
    dws, dbs = unpack(dparams, widths)
    for l in range(len(ws)):
        np.testing.assert_allclose(dws[l], tw[l].grad.numpy(), rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(dbs[l], tb[l].grad.numpy(), rtol=1e-12, atol=1e-14)


def test_hand_worked_two_layers_with_a_dead_unit():
    # x = (1, 2); W1 = [[1, 0], [0, -1]], b1 = (0, 1): z1 = (1, -1) -> a1 = (1, 0), unit 1 dead
    # W2 = [[2, 3]], b2 = 0.5: out = 2.5; dout = 4
    x = np.array([[1, 2]], np.float32)
    p = np.array([1, 0, 0, -1, 0, 1, 2, 3, 0.5], np.float32)
    dfeat, dp, fa, pa, mg = oracle.oracle_mlp_bwd(oracle.make_mlp_config([2, 2, 1]), x, p, np.array([[4]], np.float32),
                                                  want_abs=True)
    # delta2 = 4; dW2 = 4 * a1 = (4, 0); db2 = 4; g1 = W2^T 4 = (8, 12); delta1 = (8, 0)
    # dW1 = delta1 x^T = [[8, 16], [0, 0]]; db1 = (8, 0); dfeat = W1^T delta1 = (8, 0)
    np.testing.assert_array_equal(dp, [8, 16, 0, 0, 8, 0, 4, 0, 4])
    np.testing.assert_array_equal(dfeat, [[8, 0]])
    np.testing.assert_array_equal(fa, [[8, 0]])                      # |W1|^T (|W2|^T |dout| * mask) = (8, 0)
    np.testing.assert_array_equal(pa, [8, 16, 0, 0, 8, 0, 4, 0, 4])
    assert mg[0] == pytest.approx(1.0 / 3.0)                         # z1 = (1, -1), S = (1, 3): min(1/1, 1/3)
    # relu'(0) = 0: a unit sitting exactly on the kink passes no gradient
    p0 = p.copy(); p0[5] = 2.0                                       # z1[1] = -2 + 2 = 0
    d0, _ = oracle.oracle_mlp_bwd(oracle.make_mlp_config([2, 2, 1]), x, p0, np.array([[4]], np.float32))
    np.testing.assert_array_equal(d0, [[8, 0]])


def test_central_differences_of_the_pinned_forward_away_from_kinks():
    """The chain is piecewise linear: where no pre-activation changes sign a central difference of oracle_mlp is exact
    up to the forward's fp32 output rounding.  Rows near a kink (margin < 0.05) are left out."""
    widths = [6, 8, 5]
    ws, bs, x, dout = rand_chain(3, widths, 200)
    params = pack(ws, bs)
    m = oracle.make_mlp_config(widths)
    dfeat, dparams, _, _, margin = oracle.oracle_mlp_bwd(m, x, params, dout, want_abs=True)
    keep = margin > 0.05
    assert keep.sum() > 40
    x, dout, dfeat = x[keep], dout[keep], dfeat[keep]
    _, dparams = oracle.oracle_mlp_bwd(m, x, params, dout)
    loss = lambda xx, pp: float((oracle.oracle_mlp(m, xx, pp).astype(np.float64) * dout).sum())
    h = np.float32(2.0 ** -9)                                         # exactly representable steps
    for i in range(0, params.size, 7):
        pp, pm = params.copy(), params.copy()
        pp[i] += h; pm[i] -= h
        fd = (loss(x, pp) - loss(x, pm)) / (float(pp[i]) - float(pm[i]))
        assert abs(fd - dparams[i]) <= 2e-4 * (abs(dparams[i]) + np.abs(dout).sum() * 1e-2), (i, fd, dparams[i])
    for k in range(widths[0]):
        xp, xm = x.copy(), x.copy()
        xp[:, k] += h; xm[:, k] -= h
        step = (xp[:, k].astype(np.float64) - xm[:, k])
        fd = ((oracle.oracle_mlp(m, xp, params).astype(np.float64) - oracle.oracle_mlp(m, xm, params)) * dout).sum(1) / step
        np.testing.assert_allclose(fd, dfeat[:, k], rtol=0, atol=3e-4 * np.abs(dout).sum(1).max())


def test_abs_terms_equal_the_values_when_everything_is_nonnegative_and_rebuild_with_numpy():
    widths = [10, 14, 12, 6]
    ws, bs, x, dout = rand_chain(5, widths, 50)
    ws = [np.abs(w) for w in ws]; bs = [np.abs(b) for b in bs]; x = np.abs(x); dout = np.abs(dout)
    m = oracle.make_mlp_config(widths)
    dfeat, dparams, fa, pa, mg = oracle.oracle_mlp_bwd(m, x, pack(ws, bs), dout, want_abs=True)
    np.testing.assert_array_equal(fa.astype(np.float32), dfeat)      # every mask is 1, every term >= 0
    np.testing.assert_array_equal(pa, dparams)
    assert (mg == 1.0).all()                                         # |z| / sum|terms| = 1 without cancellation
    # random signs: rebuild the bounds with numpy from the forward's own masks
    ws, bs, x, dout = rand_chain(6, widths, 50)
    dfeat, dparams, fa, pa, mg = oracle.oracle_mlp_bwd(m, x, pack(ws, bs), dout, want_abs=True)
    acts, masks, zs, Ss = [x.astype(np.float64)], [], [], []
    for l, (w, b) in enumerate(zip(ws, bs)):
        z = acts[-1] @ w.astype(np.float64).T + b
        S = np.abs(acts[-1])[:, None, :] * np.abs(w.astype(np.float64))[None]
        S = S.sum(-1) + np.abs(b)
        if l < len(ws) - 1:
            zs.append(z); Ss.append(S); masks.append((z > 0).astype(np.float64)); acts.append(np.maximum(z, 0))
    D = np.abs(dout.astype(np.float64))
    want_p = []
    for l in range(len(ws) - 1, -1, -1):
        want_p.insert(0, np.concatenate([(D[:, :, None] * np.abs(acts[l])[:, None, :]).sum(0).ravel(), D.sum(0)]))
        D = D @ np.abs(ws[l].astype(np.float64))
        if l > 0:
            D = D * masks[l - 1]
    np.testing.assert_allclose(fa, D, rtol=1e-12)
    np.testing.assert_allclose(pa, np.concatenate(want_p), rtol=1e-12)
    np.testing.assert_allclose(mg, np.min([(np.abs(z) / S).min(1) for z, S in zip(zs, Ss)], axis=0), rtol=1e-12)
    assert (np.abs(dparams) <= pa * (1 + 1e-12)).all() and (np.abs(dfeat) <= fa * (1 + 1e-6) + 1e-30).all()


def test_bf16_operand_mode_changes_nothing_on_representable_inputs_and_rounds_otherwise():
    widths = [8, 8, 4]
    rng = np.random.default_rng(7)
    rep = lambda a: (np.round(a * 8) / 8).astype(np.float32)          # 3 fractional bits: exact in bf16
    ws = [rep(rng.uniform(-1, 1, (8, 8))), rep(rng.uniform(-1, 1, (4, 8)))]
    bs = [rep(rng.uniform(-1, 1, 8)), rep(rng.uniform(-1, 1, 4))]
    x, dout = rep(rng.uniform(-2, 2, (30, 8))), rep(rng.uniform(-2, 2, (30, 4)))
    plain = oracle.oracle_mlp_bwd(oracle.make_mlp_config(widths), x, pack(ws, bs), dout)
    # hidden activations are sums of <= 9 products of 3-fractional-bit numbers: 6 fractional bits, |a| < 32 -> not all
    # representable in bf16's 8 bits, so only the LAST layer's parameter gradient and nothing upstream is guaranteed equal
    quant = oracle.oracle_mlp_bwd(oracle.make_mlp_config(widths, quant_bf16=True), x, pack(ws, bs), dout)
    one = oracle.make_mlp_config([8, 4])
    p1 = pack(ws[1:], bs[1:])
    a = oracle.oracle_mlp_bwd(one, x, p1, dout)
    b = oracle.oracle_mlp_bwd(oracle.make_mlp_config([8, 4], quant_bf16=True), x, p1, dout)
    np.testing.assert_array_equal(a[0], b[0]); np.testing.assert_array_equal(a[1], b[1])
    assert not np.array_equal(plain[1], quant[1])                    # rounding of the hidden activations shows
    np.testing.assert_allclose(quant[1], plain[1], rtol=0, atol=2.0 ** -7 * np.abs(plain[1]).max() * 4)
    # an input that is NOT representable is rounded to nearest even before it is multiplied
    xx = np.array([[1 + 2.0 ** -8 + 2.0 ** -20]], np.float32)         # just above a tie -> 1 + 2^-7
    _, dp = oracle.oracle_mlp_bwd(oracle.make_mlp_config([1, 1], quant_bf16=True), xx, np.array([1, 0], np.float32),
                                  np.array([[1]], np.float32))
    assert dp[0] == 1 + 2.0 ** -7 and dp[1] == 1.0
