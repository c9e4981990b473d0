"""GPU parity of dash_hash4d_adam_step (sparse Adam over touched entries; Q28) against
the CPU oracle through the C ABI.  Tolerances (fp32 kernel vs double oracle): m, v rel 1e-6; theta within
2.5e-7*|theta| + 4e-6*|update| + 2e-6*lr (m relative to its two terms: they can cancel); untouched entries bit-identical; the fp16 copy equals the IEEE rounding of the
kernel's own master bit for bit; gradients zeroed exactly."""
import numpy as np
import pytest
import torch

import oracle
import paper_2507_19141_b200 as dh
from dash_inputs import CONFIGS, make_workload

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_steps(cfg, shape, grads, half, lr=1e-2, b1=0.9, b2=0.99, eps=1e-15):
    # the ABI carries the hyper-parameters as fp32: the oracle gets exactly those values (1 - beta amplifies the
    # rounding of beta: 1 - fl32(0.99) differs from 0.01 by 1e-6 relative)
    lr, b1, b2, eps = (float(np.float32(x)) for x in (lr, b1, b2, eps))
    rng = np.random.default_rng(5)
    th = rng.uniform(-1e-4, 1e-4, shape).astype(np.float32)
    m, v = np.zeros(shape, np.float32), np.zeros(shape, np.float32)
    h = th.astype(np.float16) if half else None
    th_d, m_d, v_d = dev(th), dev(m), dev(v)
    h_d = dev(h) if half else None
    for t, g in enumerate(grads, start=1):
        th0, m0 = th.copy(), m.copy()
        g_d = dev(g)
        dh.dash_hash4d_adam_step(cfg, th_d, g_d, m_d, v_d, t, lr, b1, b2, eps, table16=h_d)
        torch.cuda.synchronize()
        gg = g.copy()
        n = oracle.oracle_adam_step(th.reshape(-1), gg.reshape(-1), m.reshape(-1), v.reshape(-1), lr, b1, b2, eps, t,
                                    theta16=None if h is None else h.reshape(-1))
        assert n == int((g != 0).sum())
        got_th, got_m, got_v = th_d.cpu().numpy(), m_d.cpu().numpy(), v_d.cpu().numpy()
        assert float(g_d.abs().max()) == 0.0                                   # ZERO_GRAD
        z = g == 0
        # untouched: bit-identical to the previous state (both sides)
        np.testing.assert_array_equal(got_th[z], th0[z])
        upd = np.abs(th.astype(np.float64) - th0)
        err = np.abs(got_th.astype(np.float64) - th)
        # m = beta1 m + (1-beta1) g can cancel: its fp32 error is relative to the terms, not to the result, and
        # reaches theta as lr * err(m_hat) / sqrt(v_hat) <= ~1e-6 * lr
        assert (err <= 2.5e-7 * np.abs(th) + 4e-6 * upd + 2e-6 * lr).all(), f"step {t}: theta worst {err.max():.3e}"
        m_terms = b1 * np.abs(m0.astype(np.float64)) + (1 - b1) * np.abs(g.astype(np.float64))
        assert (np.abs(got_m.astype(np.float64) - m) <= 1e-6 * m_terms + 1e-37).all(), f"step {t}: m"
        np.testing.assert_allclose(got_v, v, rtol=1e-6, atol=1e-37)
        if half:
            got_h = h_d.cpu().numpy()
            np.testing.assert_array_equal(got_h.view(np.uint16)[~z], got_th.astype(np.float16).view(np.uint16)[~z])
            # and close to the oracle's half (the masters may differ in the last fp32 bit)
            assert (np.abs(got_h.astype(np.float64) - h.astype(np.float64)) <= 2.0 ** -10 * np.abs(h) + 2.0 ** -24).all()
        # keep the two sides in lock-step: continue from the oracle's state
        th_d.copy_(dev(th)); m_d.copy_(dev(m)); v_d.copy_(dev(v))
        if half:
            h_d.copy_(dev(h))


@pytest.mark.parametrize("L,T,F,half", [(4, 4096, 2, False), (3, 100003, 1, True), (2, 5001, 1, False),
                                        (16, 1 << 15, 4, True), (1, 3, 1, False)])
def test_adam_random_sparse_gradients(L, T, F, half):
    cfg = dh.make_config(L, F, T, 4, 64, 2, 8, "fp16" if half else "fp32")
    rng = np.random.default_rng(L * T + F)
    grads = []
    for _ in range(4):
        g = (rng.standard_normal((L, T, F)) * 10.0 ** rng.uniform(-6, 1, (L, T, F))).astype(np.float32)
        g[rng.random((L, T, F)) < 0.6] = 0.0                  # 60 % untouched
        grads.append(g)
    run_steps(cfg, (L, T, F), grads, half)


def test_adam_on_real_backward_gradients_c2():
    """Gradients with the sparsity of the workload: dense coarse levels touch 20-47 % of T."""
    wl = make_workload("C2")
    enc = wl.spec.enc
    cfg = dh.config_from_params(enc, flags=dh.FLAG_DENSE_COARSE | dh.FLAG_ZERO_GRAD)
    dt = torch.empty((enc.L, enc.T, enc.F), device="cuda")
    dh.dash_hash4d_bwd(cfg, dev(wl.xyz), dev(wl.t), dev(wl.dout), dt)
    g = dt.cpu().numpy()
    assert 0.15 < (g[0] != 0).mean() < 0.3
    run_steps(cfg, g.shape, [g, g * 0.5], False)


def test_adam_errors():
    cfg = dh.config_from_params(CONFIGS["C1"].enc)
    a = torch.zeros((4, 4096, 2), device="cuda")
    with pytest.raises(dh.Hash4DError):
        dh.dash_hash4d_adam_step(cfg, a, a.clone(), a.clone(), a.clone(), 0)             # step 0
    with pytest.raises(dh.Hash4DError):
        dh.dash_hash4d_adam_step(cfg, a, a.clone(), a.clone(), a.clone(), 1, beta1=1.0)  # beta1 = 1
