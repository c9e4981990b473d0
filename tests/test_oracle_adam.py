"""Pins of the sparse Adam oracle (oracle/dash_oracle.c `dash_oracle_adam_step`; Q28).
CPU only.  Fixed by: closed forms of Adam (first step, constant gradient), torch.optim.Adam on dense gradients,
torch.optim.SparseAdam for the skip-untouched rule, numpy's float16 conversion for the half rounding."""
import numpy as np
import torch

import oracle


def test_first_step_and_constant_gradient_closed_forms():
    # t = 1: m_hat = g, v_hat = g^2  =>  theta -= lr * g / (|g| + eps); the same holds at every t for a constant g
    g0 = np.array([0.5, -2.0, 1e-3, -7.0], np.float32)
    th = np.array([1.0, 1.0, 1.0, 1.0], np.float32)
    m, v = np.zeros(4, np.float32), np.zeros(4, np.float32)
    lr, eps = 1e-2, 1e-8
    for t in range(1, 6):
        g = g0.copy()
        before = th.astype(np.float64).copy()
        n = oracle.oracle_adam_step(th, g, m, v, lr, 0.9, 0.999, eps, t)
        assert n == 4 and (g == 0).all()
        want = before - lr * g0.astype(np.float64) / (np.abs(g0.astype(np.float64)) + eps)
        np.testing.assert_allclose(th, want, rtol=0, atol=2e-7)
    np.testing.assert_allclose(m, (1 - 0.9 ** 5) * g0, rtol=1e-6)
    np.testing.assert_allclose(v, (1 - 0.999 ** 5) * g0.astype(np.float64) ** 2, rtol=1e-6)


def test_untouched_entries_keep_theta_and_moments():
    rng = np.random.default_rng(0)
    th = rng.standard_normal(100).astype(np.float32)
    m = rng.standard_normal(100).astype(np.float32)
    v = rng.random(100).astype(np.float32)
    g = rng.standard_normal(100).astype(np.float32)
    g[::3] = 0.0
    th0, m0, v0 = th.copy(), m.copy(), v.copy()
    n = oracle.oracle_adam_step(th, g.copy(), m, v, 1e-2, 0.9, 0.99, 1e-15, 7, zero_grad=False)
    assert n == int((g != 0).sum())
    z = g == 0
    np.testing.assert_array_equal(th[z], th0[z]); np.testing.assert_array_equal(m[z], m0[z])
    np.testing.assert_array_equal(v[z], v0[z])
    assert (th[~z] != th0[~z]).all()


def test_matches_torch_adam_on_dense_gradients():
    rng = np.random.default_rng(1)
    n = 5000
    th = rng.standard_normal(n).astype(np.float32)
    p = torch.nn.Parameter(torch.from_numpy(th.copy()).double())
    opt = torch.optim.Adam([p], lr=3e-3, betas=(0.9, 0.99), eps=1e-15)
    m, v = np.zeros(n, np.float32), np.zeros(n, np.float32)
    for t in range(1, 9):
        g = (rng.standard_normal(n) * 10.0 ** rng.uniform(-4, 1, n)).astype(np.float32)
        g[g == 0] = 1.0
        p.grad = torch.from_numpy(g.copy()).double()
        opt.step()
        oracle.oracle_adam_step(th, g, m, v, 3e-3, 0.9, 0.99, 1e-15, t)
        np.testing.assert_allclose(th, p.detach().numpy(), rtol=0, atol=3e-6)   # fp32 state vs double state


def test_matches_torch_sparse_adam_skip_rule():
    rng = np.random.default_rng(2)
    rows, F = 300, 4
    th = rng.standard_normal((rows, F)).astype(np.float32)
    p = torch.nn.Parameter(torch.from_numpy(th.copy()).double())
    opt = torch.optim.SparseAdam([p], lr=1e-2, betas=(0.9, 0.99), eps=1e-15)
    m, v = np.zeros((rows, F), np.float32), np.zeros((rows, F), np.float32)
    for t in range(1, 7):
        idx = np.sort(rng.choice(rows, 40, replace=False))
        vals = rng.standard_normal((40, F))
        vals[vals == 0] = 1.0
        g = np.zeros((rows, F), np.float32)
        g[idx] = vals.astype(np.float32)
        p.grad = torch.sparse_coo_tensor(torch.from_numpy(idx[None, :]), torch.from_numpy(g[idx].astype(np.float64)),
                                         (rows, F))
        opt.step()
        # SparseAdam's bias correction uses the GLOBAL step count, like the oracle's t
        oracle.oracle_adam_step(th.reshape(-1), g.reshape(-1), m.reshape(-1), v.reshape(-1), 1e-2, 0.9, 0.99, 1e-15, t)
        np.testing.assert_allclose(th, p.detach().numpy(), rtol=0, atol=3e-6)


def test_half_rounding_is_numpy_float16():
    rng = np.random.default_rng(3)
    vals = np.concatenate([rng.standard_normal(3000), rng.uniform(-1e-4, 1e-4, 3000), 10.0 ** rng.uniform(-9, 5, 2000),
                           [0.0, 65504.0, 65519.9, 65520.0, 2.0 ** -24, 2.0 ** -25, 1.5 * 2.0 ** -24,
                            1 + 2.0 ** -11, 1 + 3 * 2.0 ** -11]]).astype(np.float32)
    want = vals.astype(np.float16).view(np.uint16)
    got = np.array([oracle.oracle_double_to_half(float(x)) for x in vals], np.uint16)
    np.testing.assert_array_equal(got, want)
    th = vals[:1000].copy(); g = np.ones(1000, np.float32); m = np.zeros(1000, np.float32); v = np.zeros(1000, np.float32)
    h = np.zeros(1000, np.float16)
    oracle.oracle_adam_step(th, g, m, v, 1e-3, 0.9, 0.99, 1e-15, 1, theta16=h)
    np.testing.assert_array_equal(h.view(np.uint16), th.astype(np.float16).view(np.uint16))
