"""GPU parity of the fused render path (include/dash_deform.h: G_4D -> phi_d -> heads, Eq. 9-10;
DESIGN.md Q27) against the CPU oracle, through the C ABI.

Tolerance (Q27): the kernel feeds its tensor cores bf16 operands.  Against the oracle run with the SAME
operand rounding (QUANT_BF16) what is left is fp32 accumulation order (~K * 2^-24 * A) plus rare one-ulp flips of a
bf16-rounded activation (2^-8 of one term): elementwise |err| <= 4e-3 * A and normwise <= 3e-4, A the magnitude
bound the oracle propagates.  Against the plain double MLP the bf16 rounding itself shows: elementwise 2e-2 * A."""
import numpy as np
import pytest
import torch

import oracle
import paper_2507_19141_b200 as dh
from dash_inputs import CONFIGS, EncoderParams, make_mlp_params, make_queries_uniform, make_workload

pytestmark = pytest.mark.gpu
DC = dh.FLAG_DENSE_COARSE


def dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def check_mlp_out(got, feat, params, widths, base, what):
    ref_q, mag = oracle.oracle_mlp(oracle.make_mlp_config(widths, quant_bf16=True), feat, params, base=base,
                                   want_abs=True)
    ref = oracle.oracle_mlp(oracle.make_mlp_config(widths), feat, params, base=base)
    got = np.asarray(got, np.float64)
    assert np.isfinite(got).all(), what
    err_q = np.abs(got - ref_q)
    assert (err_q <= 4e-3 * mag + 1e-30).all(), f"{what}: worst err/A vs bf16-operand oracle {(err_q / mag).max():.3e}"
    nrm = np.linalg.norm(got - ref_q) / max(np.linalg.norm(ref_q - (0 if base is None else base)), 1e-300)
    assert nrm <= 3e-4, f"{what}: normwise {nrm:.3e}"
    err = np.abs(got - ref)
    assert (err <= 2e-2 * mag + 1e-30).all(), f"{what}: worst err/A vs double oracle {(err / mag).max():.3e}"
    return float((err_q / mag).max()), float(nrm)


MLP_SHAPES = [
    ([64, 128, 10], 1000),
    ([64, 128, 192, 16], 4097),
    ([32, 64, 64, 10], 129),
    ([32, 10], 128),
    ([16, 16], 1),
    ([24, 40, 7], 300),                  # widths that need padding to 16
    ([64, 128, 128, 128, 10], 2000),
    ([256, 64, 10], 513),
    ([64, 128, 10], 0),
]


@pytest.mark.parametrize("widths,N", MLP_SHAPES)
@pytest.mark.parametrize("with_base", [False, True])
def test_mlp_fwd_parity(widths, N, with_base):
    rng = np.random.default_rng(sum(widths) + N)
    feat = rng.standard_normal((N, widths[0])).astype(np.float32)
    params = make_mlp_params(sum(widths), widths)
    base = rng.standard_normal((N, widths[-1])).astype(np.float32) if with_base else None
    m = dh.make_mlp_config(widths)
    assert dh.dash_mlp_param_count(m) == params.size == oracle.mlp_param_count(widths)
    fd = dev(feat) if N else torch.empty((0, widths[0]), device="cuda")
    out = dh.dash_mlp_fwd(m, fd, dev(params), base=dev(base) if N else None)
    torch.cuda.synchronize()
    assert out.shape == (N, widths[-1])
    if N:
        check_mlp_out(out.cpu().numpy(), feat, params, widths, base, f"mlp {widths}")


def test_mlp_identity_is_bf16_rounding_of_the_input():
    """W = I, b = 0, one layer: out must equal the bf16 rounding of feat exactly (products by 1, sums of one term)."""
    K = 64
    feat = np.random.default_rng(0).standard_normal((777, K)).astype(np.float32)
    params = np.concatenate([np.eye(K, dtype=np.float32).reshape(-1), np.zeros(K, np.float32)])
    out = dh.dash_mlp_fwd(dh.make_mlp_config([K, K]), dev(feat), dev(params))
    want = torch.from_numpy(feat).to(torch.bfloat16).to(torch.float32).numpy()
    np.testing.assert_array_equal(out.cpu().numpy(), want)


ENC_CASES = [
    # L, F, T, res_s, res_t, dtype, N, widths (widths[0] = L*F), t_stride
    (16, 2, 1 << 17, (16, 2048), (8, 150), "fp32", 10_000, [32, 64, 10], 1),
    (16, 4, 1 << 15, (16, 1024), (8, 100), "fp16", 5001, [64, 128, 10], 1),
    (16, 4, 1 << 15, (16, 1024), (8, 100), "fp16", 5001, [64, 128, 192, 16], 0),
    (8, 1, 5000, (4, 100), (2, 20), "fp32", 130, [8, 32, 10], 1),
    (6, 8, 1 << 12, (4, 200), (4, 30), "fp16", 1000, [48, 64, 10], 1),
    (12, 2, 1 << 14, (8, 500), (4, 50), "fp32", 127, [24, 48, 48, 10], 0),
]


@pytest.mark.parametrize("L,F,T,rs,rt,dtype,N,widths,t_stride", ENC_CASES)
@pytest.mark.parametrize("fused", [1, 0])
def test_deform_fwd_parity(L, F, T, rs, rt, dtype, N, widths, t_stride, fused, set_debug):
    set_debug(dh.DEBUG_DEFORM_PATH, 1 if fused else 2)
    enc = EncoderParams(L, F, T, rs[0], rs[1], rt[0], rt[1], dtype)
    ocfg, gcfg = oracle.config_from_params(enc), dh.config_from_params(enc)
    rng = np.random.default_rng(L * 7 + F + N)
    xyz, t = make_queries_uniform(L + F + N, N)
    xyz[0] = [0.0, 1.0, np.float32(1) - np.float32(2.0 ** -24)]
    if t_stride == 0:
        t = t[:1].copy()
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16 if dtype == "fp16" else np.float32)
    params = make_mlp_params(N, widths)
    base = rng.standard_normal((N, widths[-1])).astype(np.float32)
    m = dh.make_mlp_config(widths)
    assert (dh.dash_deform_workspace_bytes(gcfg, m, N) == 0) == bool(fused)
    out = dh.dash_deform_fwd(gcfg, m, dev(xyz), dev(t), dev(table), dev(params), base=dev(base), t_stride=t_stride,
                             N=N)
    torch.cuda.synchronize()
    feat = oracle.oracle_fwd(ocfg, N, xyz, t, table, t_stride=t_stride)
    check_mlp_out(out.cpu().numpy(), feat, params, widths, base, f"deform fused={fused}")
    # the fused kernel and the two-pass path see the same fp32 features: the library's own forward
    feat_gpu = dh.dash_hash4d_fwd(gcfg, dev(xyz), dev(t), dev(table), t_stride=t_stride, N=N)
    out2 = dh.dash_mlp_fwd(m, feat_gpu, dev(params), base=dev(base))
    torch.testing.assert_close(out, out2, rtol=0, atol=0)


@pytest.mark.parametrize("name", ["C2", "C3"])
def test_deform_full_size_configs(name):
    """BASELINE.json configs whose table fits L2 (the fused kernel's domain), all queries, index list absent."""
    wl = make_workload(name, with_dout=False)
    enc, N = wl.spec.enc, wl.N
    widths = [enc.L * enc.F, 64, 64, 10]
    params = make_mlp_params(7, widths)
    ocfg, gcfg = oracle.config_from_params(enc), dh.config_from_params(enc)
    table = (wl.table.astype(np.float32) * 1e4).astype(wl.table.dtype)      # features of order 1
    m = dh.make_mlp_config(widths)
    assert dh.dash_deform_workspace_bytes(gcfg, m, N) == 0
    out = dh.dash_deform_fwd(gcfg, m, dev(wl.xyz), dev(wl.t), dev(table), dev(params))
    torch.cuda.synchronize()
    feat = oracle.oracle_fwd(ocfg, N, wl.xyz, wl.t, table)
    check_mlp_out(out.cpu().numpy(), feat, params, widths, None, name)


def test_deform_index_list_c5_sample():
    wl = make_workload("C5", n_override=40_000, with_dout=False)
    enc, N = wl.spec.enc, wl.N
    widths = [enc.L * enc.F, 128, 10]
    params = make_mlp_params(9, widths)
    ocfg, gcfg = oracle.config_from_params(enc), dh.config_from_params(enc)
    table = (wl.table * 1e4).astype(np.float32)
    out = dh.dash_deform_fwd(gcfg, dh.make_mlp_config(widths), dev(wl.xyz), dev(wl.t), dev(table), dev(params),
                             index=dev(wl.index))
    torch.cuda.synchronize()
    feat = oracle.oracle_fwd(ocfg, N, wl.xyz, wl.t, table, index=wl.index)
    check_mlp_out(out.cpu().numpy(), feat, params, widths, None, "C5 sample")


def test_deform_errors():
    enc = CONFIGS["C1"].enc
    cfg = dh.config_from_params(enc)
    x, t = torch.zeros((4, 3), device="cuda"), torch.zeros(4, device="cuda")
    tab = torch.zeros((enc.L, enc.T, enc.F), device="cuda")
    with pytest.raises(dh.Hash4DError) as e:                               # width[0] != L*F
        dh.dash_deform_fwd(cfg, dh.make_mlp_config([16, 10]), x, t, tab, torch.zeros(170, device="cuda"))
    assert e.value.status == 1
    with pytest.raises(dh.Hash4DError) as e:                               # too wide
        dh.dash_mlp_fwd(dh.make_mlp_config([8, 300, 10]), torch.zeros((4, 8), device="cuda"),
                        torch.zeros(10, device="cuda"))
    assert e.value.status == 1
    big = dh.make_mlp_config([256, 256, 256, 256, 16])                     # 3 x 128 KB of weights: over 227 KB
    with pytest.raises(dh.Hash4DError) as e:
        dh.dash_mlp_fwd(big, torch.zeros((4, 256), device="cuda"), torch.zeros(dh.dash_mlp_param_count(big),
                                                                                device="cuda"))
    assert e.value.status == 2


def test_render_and_train_calls_are_cuda_graph_capturable():
    """dash_deform_fwd (fused), dash_hash3d_fwd and dash_hash4d_adam_step only enqueue kernels: a render frame and an
    optimiser step replay from one CUDA graph and give the directly launched results bit for bit."""
    wl = make_workload("C2", n_override=20_000)
    enc, N = wl.spec.enc, wl.N
    gcfg = dh.config_from_params(enc, flags=DC | dh.FLAG_ZERO_GRAD)
    cfg_plain = dh.config_from_params(enc)
    widths = [enc.L * enc.F, 64, 10]
    m = dh.make_mlp_config(widths)
    xyz, t, dout = dev(wl.xyz), dev(wl.t), dev(wl.dout)
    table, prm = dev(wl.table * 1e4), dev(make_mlp_params(1, widths))
    out = torch.empty((N, 10), device="cuda")
    f3 = torch.empty((N, enc.L * enc.F), device="cuda")
    dt = torch.empty((enc.L, enc.T, enc.F), device="cuda")
    theta = table.clone()
    m1, v1 = torch.zeros_like(theta), torch.zeros_like(theta)

    def step():
        dh.dash_deform_fwd(cfg_plain, m, xyz, t, table, prm, out=out)
        dh.dash_hash3d_fwd(cfg_plain, xyz, table, out=f3)
        dh.dash_hash4d_bwd(gcfg, xyz, t, dout, dt)
        dh.dash_hash4d_adam_step(gcfg, theta, dt, m1, v1, 1)

    step()
    torch.cuda.synchronize()
    want = [a.clone() for a in (out, f3, theta, m1, v1)]
    theta.copy_(table); m1.zero_(); v1.zero_(); out.fill_(-1); f3.fill_(-1)
    graph = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step()
    torch.cuda.current_stream().wait_stream(side)
    theta.copy_(table); m1.zero_(); v1.zero_()
    with torch.cuda.graph(graph):
        step()
    theta.copy_(table); m1.zero_(); v1.zero_(); out.fill_(-1); f3.fill_(-1)
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, want[0]) and torch.equal(f3, want[1])
    # the scatter order varies run to run (fp32 reductions): the optimiser state agrees to rounding, not bitwise
    torch.testing.assert_close(theta, want[2], rtol=1e-4, atol=1e-6)
    assert float(dt.abs().max()) == 0.0


def test_deform_two_pass_on_a_table_beyond_l2_c4_sample():
    """C4's 268 MB fp16 table does not fit L2 as one level group: dash_deform_fwd must take the two-pass route
    (level-group-major forward into the caller's workspace, then the MLP kernel) and ask for that workspace."""
    wl = make_workload("C4", n_override=150_000, with_dout=False)
    enc, N = wl.spec.enc, wl.N
    widths = [enc.L * enc.F, 128, 10]
    params = make_mlp_params(5, widths)
    ocfg, gcfg = oracle.config_from_params(enc), dh.config_from_params(enc)
    m = dh.make_mlp_config(widths)
    need = dh.dash_deform_workspace_bytes(gcfg, m, N)
    assert need == N * enc.L * enc.F * 4
    table = (wl.table.astype(np.float32) * 1e4).astype(np.float16)
    with pytest.raises(dh.Hash4DError) as e:                                  # no workspace: status 3
        dh.dash_deform_fwd(gcfg, m, dev(wl.xyz), dev(wl.t), dev(table), dev(params),
                           workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))
    assert e.value.status == 3
    out = dh.dash_deform_fwd(gcfg, m, dev(wl.xyz), dev(wl.t), dev(table), dev(params))
    torch.cuda.synchronize()
    feat = oracle.oracle_fwd(ocfg, N, wl.xyz, wl.t, table)
    check_mlp_out(out.cpu().numpy(), feat, params, widths, None, "C4 sample two-pass")
