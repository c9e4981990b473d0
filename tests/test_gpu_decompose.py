"""GPU parity of dash_decompose (include/dash_decompose.h; Eq. 5; Q31) against the CPU
oracle through the C ABI.  Magnitudes, threshold, counts and the index list are unique results: BIT-EXACT.  L_s is a
double-precision sum in another order (rel 1e-6 after its fp32 rounding); the gradient is three fp32 roundings (rel 1e-6)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2507_19141_b200 as dh

pytestmark = pytest.mark.gpu


def run(dp, k, grad_scale=1.0):
    r = dh.dash_decompose(torch.from_numpy(dp).cuda(), k, grad_scale=grad_scale)
    res = dh.dash_decompose_read(r["result"])
    o = oracle.oracle_decompose(dp, k, grad_scale=grad_scale)
    np.testing.assert_array_equal(r["mag"].cpu().numpy(), o["mag"])
    assert res.tau == np.float32(o["tau"]) and res.n_dynamic == len(o["index"]) and res.n_static == len(dp) - len(o["index"])
    np.testing.assert_array_equal(r["index"].cpu().numpy()[:res.n_dynamic], o["index"])
    assert res.loss == pytest.approx(o["loss"], rel=1e-6, abs=1e-30)
    np.testing.assert_allclose(r["ddp"].cpu().numpy(), o["ddp"], rtol=1e-6, atol=1e-37)
    return res, o


@pytest.mark.parametrize("n", [1, 31, 1024, 1025, 100_003, 1_500_000])
@pytest.mark.parametrize("k", [0.0, 0.01, 30.0, 99.9, 100.0])
def test_decompose_parity_random(n, k):
    rng = np.random.default_rng(n + int(k * 100))
    scale = rng.choice([0.0, 1e-20, 1e-3, 1.0, 1e15], (n, 1)).astype(np.float32)      # zeros, subnormal squares, overflow
    dp = rng.standard_normal((n, 3)).astype(np.float32) * scale
    res, o = run(dp, k, grad_scale=0.25)
    assert res.n_dynamic <= int(np.ceil(n * k / 100.0 - 1e-9) + 0.5)


def test_decompose_ties_nan_and_the_workload_of_config5():
    same = np.tile(np.array([[3, 4, 0]], np.float32), (5000, 1))
    res, _ = run(same, 30.0)
    assert res.n_dynamic == 0 and res.tau == 5.0 and res.loss == 5.0            # nobody is strictly above the tie
    bad = np.array([[np.nan, 0, 0], [1, 2, 2], [np.inf, 0, 0], [0, 0, 0]], np.float32)
    res, _ = run(bad, 50.0)
    assert res.n_dynamic == 2
    # BASELINE.json config 5: 1.5M Gaussians, 30 % dynamic; the index list feeds dash_hash4d_fwd as it is
    rng = np.random.default_rng(4)
    dp = (rng.standard_normal((1_500_000, 3)) * rng.gamma(2.0, 0.01, (1_500_000, 1))).astype(np.float32)
    res, o = run(dp, 30.0)
    assert res.n_dynamic == 450_000
    r = dh.dash_decompose(torch.from_numpy(dp).cuda(), 30.0, want_grad=False)
    assert r["ddp"] is None
    idx = r["index"][:450_000].contiguous()
    assert bool((idx[1:] > idx[:-1]).all())
    enc = dh.make_config(4, 2, 1 << 12, 8, 64, 4, 16)
    xyz = torch.rand((1_500_000, 3), device="cuda"); t = torch.rand(450_000, device="cuda")
    out = dh.dash_hash4d_fwd(enc, xyz, t, torch.zeros((4, 1 << 12, 2), device="cuda"), index=idx)
    assert out.shape == (450_000, 8)


def test_decompose_errors():
    z = torch.zeros((4, 3), device="cuda")
    with pytest.raises(dh.Hash4DError):
        dh.dash_decompose(z, 101.0)
    with pytest.raises(dh.Hash4DError):
        dh.dash_decompose(z, 10.0, workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))
    with pytest.raises(ValueError):
        dh.dash_decompose(torch.zeros((4, 4), device="cuda"), 10.0)
