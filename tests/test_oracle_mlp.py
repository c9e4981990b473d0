"""Pins of the MLP oracle (oracle/dash_oracle.c `dash_oracle_mlp`; Eq. 9-10: tiny MLP phi_d and
the multi-head deformation decoder; Q27).  CPU only.

Fixed by things other than itself: a two-layer example worked by hand, the textbook composition
relu(x W1^T + b1) W2^T + b2 evaluated with numpy's matmul in double, identity / zero special cases, and — for the
bf16 operand rounding the CUDA path applies — torch's own float32 -> bfloat16 conversion plus the tie cases of
round-to-nearest-even written out by hand."""
import numpy as np
import torch

import oracle


def pack(ws, bs):
    return np.concatenate([np.concatenate([w.reshape(-1), b.reshape(-1)]) for w, b in zip(ws, bs)]).astype(np.float32)


def test_hand_worked_two_layer_example():
    # x = (1, -2); W1 = [[1, 2], [3, -1]], b1 = (0.5, -1): z = (1 - 4 + 0.5, 3 + 2 - 1) = (-2.5, 4) -> relu (0, 4)
    # W2 = [[2, -1]], b2 = 0.25: 0*2 - 4 + 0.25 = -3.75; base 1 -> -2.75
    x = np.array([[1.0, -2.0]], np.float32)
    p = pack([np.array([[1, 2], [3, -1]], np.float32), np.array([[2, -1]], np.float32)],
             [np.array([0.5, -1], np.float32), np.array([0.25], np.float32)])
    m = oracle.make_mlp_config([2, 2, 1])
    assert oracle.oracle_mlp(m, x, p)[0, 0] == -3.75
    out, mag = oracle.oracle_mlp(m, x, p, base=np.array([[1.0]], np.float32), want_abs=True)
    assert out[0, 0] == -2.75
    # magnitude bound: A1 = (0.5 + 1 + 4, 1 + 3 + 2) = (5.5, 6); A2 = 0.25 + 2*5.5 + 1*6 = 17.25; + |base| = 18.25
    assert mag[0, 0] == 18.25
    # the LAST layer has no relu: a negative output survives, a hidden negative does not
    m1 = oracle.make_mlp_config([2, 2])
    np.testing.assert_array_equal(oracle.oracle_mlp(m1, x, p[:6]), [[-2.5, 4.0]])


def test_numpy_matmul_composition_random():
    rng = np.random.default_rng(0)
    for widths in ([32, 64, 10], [64, 128, 192, 16], [7, 5], [64, 128, 128, 128, 10]):
        ws = [rng.uniform(-1, 1, (widths[l], widths[l - 1])).astype(np.float32) / np.sqrt(widths[l - 1])
              for l in range(1, len(widths))]
        bs = [rng.uniform(-0.5, 0.5, widths[l]).astype(np.float32) for l in range(1, len(widths))]
        x = rng.standard_normal((50, widths[0])).astype(np.float32)
        base = rng.standard_normal((50, widths[-1])).astype(np.float32)
        a = x.astype(np.float64)
        for l, (w, b) in enumerate(zip(ws, bs)):
            a = a @ w.astype(np.float64).T + b
            if l < len(ws) - 1:
                a = np.maximum(a, 0)
        m = oracle.make_mlp_config(widths)
        assert oracle.mlp_param_count(widths) == pack(ws, bs).size
        out, mag = oracle.oracle_mlp(m, x, pack(ws, bs), base=base, want_abs=True)
        np.testing.assert_allclose(out, (a + base).astype(np.float32), rtol=1e-6, atol=1e-6)
        assert (mag >= np.abs(out) - 1e-5).all()


def test_identity_and_zero_special_cases():
    x = np.random.default_rng(1).standard_normal((9, 16)).astype(np.float32)
    eye = pack([np.eye(16, dtype=np.float32)], [np.zeros(16, np.float32)])
    np.testing.assert_array_equal(oracle.oracle_mlp(oracle.make_mlp_config([16, 16]), x, eye), x)
    # two identity layers = relu(x); zero weights = the bias broadcast
    eye2 = np.concatenate([eye, eye])
    np.testing.assert_array_equal(oracle.oracle_mlp(oracle.make_mlp_config([16, 16, 16]), x, eye2), np.maximum(x, 0))
    zer = pack([np.zeros((3, 16), np.float32)], [np.array([1, 2, 3], np.float32)])
    np.testing.assert_array_equal(oracle.oracle_mlp(oracle.make_mlp_config([16, 3]), x, zer), np.tile([1, 2, 3], (9, 1)))


def test_bf16_rounding_against_torch_and_hand_ties():
    # ties to even on the 8-bit significand: 1 + 2^-8 -> 1 (even), 1 + 3*2^-8 -> 1 + 4*2^-8 (even), just above a tie goes up
    assert oracle.oracle_to_bf16(1 + 2.0 ** -8) == 1.0
    assert oracle.oracle_to_bf16(1 + 3 * 2.0 ** -8) == 1 + 4 * 2.0 ** -8
    assert oracle.oracle_to_bf16(1 + 2.0 ** -8 + 2.0 ** -20) == 1 + 2.0 ** -7
    assert oracle.oracle_to_bf16(-(1 + 2.0 ** -8)) == -1.0
    assert oracle.oracle_to_bf16(0.0) == 0.0 and oracle.oracle_to_bf16(3.0e-5) != 0.0     # no flush of small values
    rng = np.random.default_rng(2)
    v = np.concatenate([rng.standard_normal(2000), rng.uniform(-1e-4, 1e-4, 2000), 10.0 ** rng.uniform(-30, 30, 500)])
    v = v.astype(np.float32)
    want = torch.from_numpy(v).to(torch.bfloat16).to(torch.float32).numpy()
    got = np.array([oracle.oracle_to_bf16(float(x)) for x in v], np.float32)
    np.testing.assert_array_equal(got, want)


def test_quantised_path_is_numpy_composition_of_rounded_operands():
    rng = np.random.default_rng(3)
    widths = [64, 128, 16]
    bf = lambda a: torch.from_numpy(np.asarray(a, np.float32)).to(torch.bfloat16).to(torch.float64).numpy()
    ws = [rng.uniform(-1, 1, (widths[l], widths[l - 1])).astype(np.float32) / 8 for l in (1, 2)]
    bs = [rng.uniform(-0.5, 0.5, widths[l]).astype(np.float32) for l in (1, 2)]
    x = rng.uniform(-1e-3, 1e-3, (40, 64)).astype(np.float32)
    h = np.maximum(bf(x) @ bf(ws[0]).T + bs[0].astype(np.float64), 0)
    want = bf(h) @ bf(ws[1]).T + bs[1].astype(np.float64)       # h rounded via fp32 first, as the oracle does
    got = oracle.oracle_mlp(oracle.make_mlp_config(widths, quant_bf16=True), x, pack(ws, bs))
    np.testing.assert_allclose(got, want.astype(np.float32), rtol=2e-6, atol=1e-7)
    exact = oracle.oracle_mlp(oracle.make_mlp_config(widths), x, pack(ws, bs))
    assert np.abs(got - exact).max() > 0                       # the rounding is really applied ...
    assert np.abs(got - exact).max() < 2e-2                    # ... and is of bf16 size


def test_deform_is_encoder_followed_by_mlp():
    cfg = oracle.make_config(4, 2, 1 << 10, 4, 32, 2, 8)
    rng = np.random.default_rng(4)
    xyz = rng.random((30, 3), dtype=np.float32)
    t = rng.random(30, dtype=np.float32)
    table = rng.uniform(-1, 1, (4, 1 << 10, 2)).astype(np.float32)
    widths = [8, 16, 10]
    params = rng.uniform(-0.3, 0.3, oracle.mlp_param_count(widths)).astype(np.float32)
    m = oracle.make_mlp_config(widths)
    feat = oracle.oracle_fwd(cfg, 30, xyz, t, table)
    np.testing.assert_array_equal(oracle.oracle_deform(cfg, m, 30, xyz, t, table, params),
                                  oracle.oracle_mlp(m, feat, params))
