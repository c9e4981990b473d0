"""GPU parity of dash_mlp_bwd / dash_deform_bwd (include/dash_deform.h; Q30) against the CPU oracle, through
the C ABI.

Tolerance (derived in DESIGN.md §3b): the kernel feeds its tensor cores bf16 operands; against the oracle run with the
SAME operand rounding what is left is fp32 accumulation order and rare one-ulp flips of a bf16-rounded activation or
delta (2^-8 of ONE term of the next sum): elementwise 4e-3 * A with A the oracle's propagated magnitude bound, normwise
1e-3 (dfeat) / 4e-3 (dparams, which sums every row's flips).  The relu mask is a DECISION taken from a floating-point
value: rows whose closest pre-activation is within 1e-3 of its rounding scale of a kink (oracle `margin`) have no unique
gradient; for them only a validity bound is checked (|err| within twice the unmasked magnitude bound)."""
import ctypes as C

import numpy as np
import pytest
import torch

import oracle
import paper_2507_19141_b200 as dh
from dash_inputs import EncoderParams, make_mlp_params, make_queries_uniform

pytestmark = pytest.mark.gpu


def dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def unmasked_bound(widths, params, dout):
    D, o, mats = np.abs(dout.astype(np.float64)), 0, []
    for l in range(1, len(widths)):
        J, K = widths[l], widths[l - 1]
        mats.append(np.abs(params[o:o + J * K].astype(np.float64)).reshape(J, K)); o += J * K + J
    for w in reversed(mats):
        D = D @ w
    return D


def check_bwd(widths, feat, params, dout, dfeat, dparams, what, p_slack=0.0):
    """p_slack: elementwise absolute allowance on dparams for error that is not the kernel's (the rounding of an fp32
    '+=' into a non-zero start); both dparams checks run on the values as they came back, nothing is clipped."""
    fq, pq, fa, pa, mg = oracle.oracle_mlp_bwd(oracle.make_mlp_config(widths, quant_bf16=True), feat, params, dout,
                                               want_abs=True)
    dfeat, dparams = np.asarray(dfeat, np.float64), np.asarray(dparams, np.float64)
    assert np.isfinite(dfeat).all() and np.isfinite(dparams).all(), what
    ok = mg > 1e-3
    err = np.abs(dfeat - fq)
    assert (err[ok] <= 4e-3 * fa[ok] + 1e-30).all(), f"{what}: dfeat worst err/A {(err[ok] / (fa[ok] + 1e-300)).max():.3e}"
    if ok.any():
        nrm = np.linalg.norm((dfeat - fq)[ok]) / max(np.linalg.norm(fq[ok]), 1e-300)
        assert nrm <= 1e-3, f"{what}: dfeat normwise {nrm:.3e}"
    loose = 2.0 * unmasked_bound(widths, params, dout)
    assert (err[~ok] <= loose[~ok] + 1e-30).all(), f"{what}: dfeat of a near-kink row outside the validity bound"
    errp = np.abs(dparams - pq)
    assert (errp <= 4e-3 * pa + p_slack + 1e-30).all(), f"{what}: dparams worst err/A {(errp / (pa + 1e-300)).max():.3e}"
    slack_norm = float(np.linalg.norm(np.broadcast_to(p_slack, pq.shape)))
    nrmp = (np.linalg.norm(dparams - pq) - slack_norm) / max(np.linalg.norm(pq), 1e-300)
    assert nrmp <= 4e-3, f"{what}: dparams normwise {nrmp:.3e}"
    return float(ok.mean())


SHAPES = [
    ([32, 10], 128), ([32, 10], 1000), ([16, 16], 1), ([32, 64, 10], 300), ([64, 128, 10], 1000),
    ([24, 40, 7], 300),                      # widths that need padding to 16
    ([32, 64, 64, 10], 129), ([32, 128, 128, 10], 20_000), ([32, 64, 48, 32, 10], 777), ([64, 128, 10], 0),
]


@pytest.mark.parametrize("widths,N", SHAPES)
def test_mlp_bwd_parity(widths, N):
    rng = np.random.default_rng(sum(widths) + N)
    feat = rng.standard_normal((N, widths[0])).astype(np.float32)
    params = make_mlp_params(sum(widths), widths)
    dout = rng.standard_normal((N, widths[-1])).astype(np.float32)
    m = dh.make_mlp_config(widths)
    start = rng.standard_normal(params.size).astype(np.float32)           # dparams is ACCUMULATED into
    dp = dev(start)
    fd = dev(feat) if N else torch.empty((0, widths[0]), device="cuda")
    dd = dev(dout) if N else torch.empty((0, widths[-1]), device="cuda")
    dfeat, dp = dh.dash_mlp_bwd(m, fd, dev(params), dd, dp)
    torch.cuda.synchronize()
    assert dfeat.shape == (N, widths[0])
    if N == 0:
        np.testing.assert_array_equal(dp.cpu().numpy(), start)
        return
    got_p = dp.cpu().numpy().astype(np.float64) - start
    # the fp32 '+=' into a random start costs one rounding of the start's magnitude: fold it into the bound
    frac = check_bwd_with_start(widths, feat, params, dout, dfeat.cpu().numpy(), got_p, start, f"mlp_bwd {widths} N={N}")
    assert frac > 0.2


def check_bwd_with_start(widths, feat, params, dout, dfeat, got_p, start, what):
    """dparams was accumulated into a random `start`: the fp32 '+=' rounds at the magnitude of start + gradient, which is
    not the kernel's error.  That rounding is passed on as an absolute slack; the UNCLIPPED difference is what is checked,
    element by element and normwise."""
    _, pq = oracle.oracle_mlp_bwd(oracle.make_mlp_config(widths, quant_bf16=True), feat, params, dout)
    slack = 2.0 ** -22 * (np.abs(start) + np.abs(pq))
    return check_bwd(widths, feat, params, dout, dfeat, got_p, what, p_slack=slack)


def test_mlp_bwd_without_dfeat_and_twice_accumulates():
    widths, N = [32, 64, 10], 500
    rng = np.random.default_rng(1)
    feat = rng.standard_normal((N, 32)).astype(np.float32)
    params = make_mlp_params(2, widths)
    dout = rng.standard_normal((N, 10)).astype(np.float32)
    m = dh.make_mlp_config(widths)
    dp = torch.zeros(params.size, device="cuda")
    none, _ = dh.dash_mlp_bwd(m, dev(feat), dev(params), dev(dout), dp, want_dfeat=False)
    assert none is None
    once = dp.cpu().numpy().copy()
    dh.dash_mlp_bwd(m, dev(feat), dev(params), dev(dout), dp, want_dfeat=False)
    np.testing.assert_allclose(dp.cpu().numpy(), 2 * once, rtol=1e-4, atol=2e-4)
    _, pq = oracle.oracle_mlp_bwd(oracle.make_mlp_config(widths, quant_bf16=True), feat, params, dout)
    assert np.linalg.norm(once - pq) / np.linalg.norm(pq) <= 4e-3


def test_one_layer_is_exact_up_to_fp32_accumulation():
    """No hidden layer: no activation rounding and no mask, so against the bf16-operand oracle only the fp32 summation
    order is left: dfeat to 2e-6 of its magnitude bound, dparams to N * 2^-24."""
    widths, N = [48, 12], 3000
    rng = np.random.default_rng(5)
    feat = rng.standard_normal((N, 48)).astype(np.float32)
    params = make_mlp_params(5, widths)
    dout = rng.standard_normal((N, 12)).astype(np.float32)
    dp = torch.zeros(params.size, device="cuda")
    dfeat, dp = dh.dash_mlp_bwd(dh.make_mlp_config(widths), dev(feat), dev(params), dev(dout), dp)
    fq, pq, fa, pa, _ = oracle.oracle_mlp_bwd(oracle.make_mlp_config(widths, quant_bf16=True), feat, params, dout,
                                              want_abs=True)
    assert (np.abs(dfeat.cpu().numpy() - fq) <= 2e-6 * fa + 1e-30).all()
    assert (np.abs(dp.cpu().numpy() - pq) <= N * 2.0 ** -24 * pa + 1e-30).all()


def test_mlp_bwd_errors():
    big = dh.make_mlp_config([64, 128, 128, 128, 10])                       # tiles + weights beyond 227 KB
    z = lambda *s: torch.zeros(s, device="cuda")
    with pytest.raises(dh.Hash4DError) as e:
        dh.dash_mlp_bwd(big, z(4, 64), z(dh.dash_mlp_param_count(big)), z(4, 10), z(dh.dash_mlp_param_count(big)))
    assert e.value.status == 2
    wide = dh.make_mlp_config([250, 10])
    with pytest.raises(dh.Hash4DError) as e:
        dh.dash_mlp_bwd(wide, z(4, 250), z(dh.dash_mlp_param_count(wide)), z(4, 10), z(dh.dash_mlp_param_count(wide)))
    assert e.value.status == 2
    for widths in ([32, 192, 10], [32, 64, 200]):                           # a layer output wider than one M = 128 tile
        c = dh.make_mlp_config(widths)
        with pytest.raises(dh.Hash4DError) as e:
            dh.dash_mlp_bwd(c, z(4, 32), z(dh.dash_mlp_param_count(c)), z(4, widths[-1]), z(dh.dash_mlp_param_count(c)))
        assert e.value.status == 2 and "128" in str(e.value)
    m = dh.make_mlp_config([32, 10])
    with pytest.raises(ValueError, match="dparams"):
        dh.dash_mlp_bwd(m, z(4, 32), z(330), z(4, 10), z(329))


@pytest.mark.parametrize("dtype,with_index,zero_grad,sort", [("fp32", False, True, False), ("fp16", True, False, False),
                                                             ("fp32", True, True, True), ("fp16", False, False, True)])
def test_deform_bwd_is_the_composition_and_matches_the_oracle(dtype, with_index, zero_grad, sort, set_debug):
    """dash_deform_bwd = hash4d_fwd -> mlp_bwd -> hash4d_bwd (-> bwd_input).  Checked three ways: against the same
    four calls made one by one; dparams against the oracle chain (oracle_fwd -> oracle_mlp_bwd); dtable and dq against
    the oracle's scatter / coordinate gradient fed the GPU's own dfeat (both are linear in it: no mask ambiguity left)."""
    from parity_utils import RTOL_FP32, check_close
    L, F, T = 8, 4, 1 << 12
    enc = EncoderParams(L, F, T, 8, 200, 4, 30, dtype)
    widths = [L * F, 64, 10]
    rng = np.random.default_rng(11)
    rows = 3000
    xyz_rows, _ = make_queries_uniform(3, rows)
    index = rng.integers(0, rows, 4001).astype(np.int32) if with_index else None
    n = len(index) if with_index else rows
    t = rng.random(n, dtype=np.float32)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16 if dtype == "fp16" else np.float32)
    params = make_mlp_params(4, widths)
    dout = rng.standard_normal((n, 10)).astype(np.float32)
    flags = dh.FLAG_DENSE_COARSE | (dh.FLAG_ZERO_GRAD if zero_grad else 0)
    if sort:   # SORT_COARSE: one sort inside the forward serves the table gradient and the coordinate gradient too
        set_debug(dh.DEBUG_BWD_COARSE_LEVELS, 3)
        flags |= dh.FLAG_SORT_COARSE
    gcfg, ocfg = dh.config_from_params(enc, flags=flags), oracle.config_from_params(enc)
    m = dh.make_mlp_config(widths)
    if sort:
        need = dh.binding._load().dash_deform_bwd_workspace_bytes(C.byref(gcfg), C.byref(m), n)
        assert need >= 2 * n * L * F * 4 + 24 * n
    start = 7.0 if zero_grad else 0.0                                       # ZERO_GRAD must overwrite garbage
    dtable = torch.full((L, T, F), start, device="cuda")
    dparams = torch.zeros(params.size, device="cuda")
    dq = torch.empty((n, 4), device="cuda")
    xd, td, idx, tabd, pd, dd = dev(xyz_rows), dev(t), dev(index), dev(table), dev(params), dev(dout)
    dh.dash_deform_bwd(gcfg, m, xd, td, tabd, pd, dd, dtable, dparams, dq=dq, index=idx)
    torch.cuda.synchronize()
    # (1) the same calls, one by one
    plain = dh.config_from_params(enc)
    feat = dh.dash_hash4d_fwd(plain, xd, td, tabd, index=idx)
    dp2 = torch.zeros_like(dparams)
    dfeat, _ = dh.dash_mlp_bwd(m, feat, pd, dd, dp2)
    dt2 = torch.zeros((L, T, F), device="cuda")
    dh.dash_hash4d_bwd(plain, xd, td, dfeat, dt2, index=idx)
    dq2 = dh.dash_hash4d_bwd_input(plain, xd, td, tabd, dfeat, index=idx)
    torch.testing.assert_close(dparams, dp2, rtol=1e-4, atol=2e-4)          # fp32 reductions in a different order
    torch.testing.assert_close(dtable, dt2, rtol=1e-4, atol=1e-5)
    torch.testing.assert_close(dq, dq2, rtol=1e-4, atol=1e-4)
    # (2) dparams against the oracle chain
    feat_o = oracle.oracle_fwd(ocfg, n, xyz_rows, t, table, index=index)
    fq, pq, fa, pa, mg = oracle.oracle_mlp_bwd(oracle.make_mlp_config(widths, quant_bf16=True), feat_o, params, dout,
                                               want_abs=True)
    assert (np.abs(dparams.cpu().numpy() - pq) <= 4e-3 * pa + 1e-30).all()
    # (3) scatter and coordinate gradient of the GPU's dfeat, by the oracle
    dfeat_h = dfeat.cpu().numpy()
    ref_t, mag_t, hits = oracle.oracle_bwd(ocfg, n, xyz_rows, t, dfeat_h, index=index, want_abs=True, want_hits=True)
    check_close(dtable.cpu().numpy(), ref_t, mag_t, RTOL_FP32, L, hits=hits, what="deform_bwd dtable")
    ref_q, mag_q = oracle.oracle_bwd_input(ocfg, n, xyz_rows, t, table, dfeat_h, index=index, want_abs=True)
    assert (np.abs(dq.cpu().numpy() - ref_q) <= (2e-3 if dtype == "fp16" else 1e-5) * mag_q + 1e-30).all()


def test_deform_bwd_errors():
    enc = EncoderParams(4, 2, 1 << 10, 8, 64, 4, 16)
    z = lambda *s: torch.zeros(s, device="cuda")
    m = dh.make_mlp_config([8, 10])
    det = dh.config_from_params(enc, flags=dh.FLAG_DENSE_COARSE | dh.FLAG_DETERMINISTIC_BWD)
    with pytest.raises(dh.Hash4DError) as e:
        dh.dash_deform_bwd(det, m, z(5, 3), z(5), z(4, 1 << 10, 2), z(90), z(5, 10), z(4, 1 << 10, 2), z(90))
    assert e.value.status == 1
    cfg = dh.config_from_params(enc)
    with pytest.raises(dh.Hash4DError) as e:                               # width[0] != L*F
        dh.dash_deform_bwd(cfg, dh.make_mlp_config([16, 10]), z(5, 3), z(5), z(4, 1 << 10, 2), z(170), z(5, 10),
                           z(4, 1 << 10, 2), z(170))
    assert e.value.status == 1


def test_training_calls_are_cuda_graph_capturable():
    """dash_deform_bwd (four composed launches), dash_mlp_bwd and the C ABI of dash_decompose only enqueue kernels on the
    current stream: a captured training step replays and gives the directly launched results (the index list, counts
    and dfeat bit for bit; the reductions to their rounding)."""
    import ctypes as C
    L, F, T, n = 8, 2, 1 << 12, 6000
    enc = EncoderParams(L, F, T, 8, 200, 4, 30)
    cfg = dh.config_from_params(enc, flags=dh.FLAG_DENSE_COARSE | dh.FLAG_ZERO_GRAD)
    widths = [L * F, 64, 10]
    m = dh.make_mlp_config(widths)
    rng = np.random.default_rng(3)
    xyz, t = make_queries_uniform(5, n)
    xd, td = dev(xyz), dev(t)
    table = dev(rng.uniform(-1, 1, (L, T, F)).astype(np.float32))
    prm = dev(make_mlp_params(2, widths)); dout = dev(rng.standard_normal((n, 10)).astype(np.float32))
    feat = dev(rng.standard_normal((n, L * F)).astype(np.float32))
    dtable = torch.empty((L, T, F), device="cuda"); dparams = torch.zeros(prm.numel(), device="cuda")
    dq = torch.empty((n, 4), device="cuda"); dfeat = torch.empty((n, L * F), device="cuda")
    dp2 = torch.zeros_like(dparams)
    ws = torch.empty(dh.binding._load().dash_deform_bwd_workspace_bytes(C.byref(cfg), C.byref(m), n) + 16,
                     dtype=torch.uint8, device="cuda")
    mot = dev(rng.standard_normal((n, 3)).astype(np.float32))
    lib = dh.binding._load()
    mag = torch.empty(n, device="cuda"); idx = torch.empty(n, dtype=torch.int32, device="cuda")
    res = torch.zeros(16, dtype=torch.uint8, device="cuda"); ddp = torch.empty((n, 3), device="cuda")
    wsd = torch.empty(lib.dash_decompose_workspace_bytes(n) + 16, dtype=torch.uint8, device="cuda")

    def step():
        dparams.zero_(); dp2.zero_()
        dh.dash_deform_bwd(cfg, m, xd, td, table, prm, dout, dtable, dparams, dq=dq, workspace=ws)
        dh.dash_mlp_bwd(m, feat, prm, dout, dp2, dfeat=dfeat)
        rc = lib.dash_decompose(n, C.c_void_p(mot.data_ptr()), 30.0, 1.0, C.c_void_p(mag.data_ptr()),
                                C.c_void_p(idx.data_ptr()), C.c_void_p(res.data_ptr()), C.c_void_p(ddp.data_ptr()),
                                C.c_void_p(wsd.data_ptr()), wsd.numel(), C.c_void_p(torch.cuda.current_stream().cuda_stream))
        assert rc == 0

    step()
    torch.cuda.synchronize()
    want = [a.clone() for a in (dtable, dparams, dq, dfeat, dp2, idx, res, ddp)]
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step()
    torch.cuda.current_stream().wait_stream(side)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        step()
    for a in (dtable, dq, dfeat, ddp):
        a.fill_(-1)
    idx.fill_(-1); res.zero_()
    graph.replay()
    torch.cuda.synchronize()
    nd = dh.dash_decompose_read(res).n_dynamic
    assert nd == dh.dash_decompose_read(want[6]).n_dynamic == 1800
    assert torch.equal(idx[:nd], want[5][:nd]) and torch.equal(res, want[6]) and torch.equal(ddp, want[7])
    assert torch.equal(dfeat, want[3])                       # no reductions on this path: bit for bit
    # fp32 reductions across CTAs land in another order: entries are sums of 6,000 O(1) terms that partly cancel
    torch.testing.assert_close(dp2, want[4], rtol=1e-4, atol=2e-4)
    torch.testing.assert_close(dparams, want[1], rtol=1e-4, atol=2e-4)
    torch.testing.assert_close(dtable, want[0], rtol=1e-4, atol=1e-5)
    torch.testing.assert_close(dq, want[2], rtol=1e-4, atol=1e-4)


def test_one_layer_without_dfeat_issues_no_dgrad_at_all():
    """n_layers = 1 and dfeat = NULL: the kernel's only MMAs are the wgrad; its per-step commit then tracks nothing."""
    widths, N = [32, 10], 2000
    rng = np.random.default_rng(8)
    feat = rng.standard_normal((N, 32)).astype(np.float32)
    params = make_mlp_params(8, widths)
    dout = rng.standard_normal((N, 10)).astype(np.float32)
    dp = torch.zeros(params.size, device="cuda")
    none, dp = dh.dash_mlp_bwd(dh.make_mlp_config(widths), dev(feat), dev(params), dev(dout), dp, want_dfeat=False)
    torch.cuda.synchronize()
    _, pq, _, pa, _ = oracle.oracle_mlp_bwd(oracle.make_mlp_config(widths, quant_bf16=True), feat, params, dout,
                                            want_abs=True)
    assert none is None and (np.abs(dp.cpu().numpy() - pq) <= N * 2.0 ** -24 * pa + 1e-30).all()
