"""GPU parity of the time-slice render path (dash_hash4d_slice_t / _slice_fwd / dash_deform_slice_fwd; Q29)
against the 4D oracle evaluated at one timestamp.  Same tolerance as the forward (the blend adds two fp32 roundings)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2507_19141_b200 as dh
from dash_inputs import EncoderParams, make_mlp_params, make_queries_uniform, make_workload
from parity_utils import RTOL_FP16, RTOL_FP32, check_close
from test_gpu_deform import check_mlp_out

pytestmark = pytest.mark.gpu
DC = dh.FLAG_DENSE_COARSE


def dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


CASES = [
    # L, F, T, res_s, res_t, dtype, N, flags
    (16, 2, 1 << 17, (16, 2048), (8, 150), "fp32", 20_001, DC),
    (16, 4, 1 << 15, (16, 1024), (8, 100), "fp16", 5001, DC),
    (6, 1, 1 << 12, (4, 200), (2, 40), "fp32", 777, 0),
    (5, 8, 1 << 12, (4, 100), (2, 20), "fp16", 300, DC),
    (3, 2, 5000, (2, 6), (2, 6), "fp32", 200, DC),          # T not a power of two, every level dense: allowed
]


@pytest.mark.parametrize("L,F,T,rs,rt,dtype,N,flags", CASES)
@pytest.mark.parametrize("tval", [0.0, 0.4321, 1.0])
def test_slice_fwd_parity(L, F, T, rs, rt, dtype, N, flags, tval):
    enc = EncoderParams(L, F, T, rs[0], rs[1], rt[0], rt[1], dtype)
    ocfg = oracle.config_from_params(enc, dense_coarse=bool(flags & DC))
    gcfg = dh.config_from_params(enc, flags=flags)
    if T & (T - 1):
        assert oracle.oracle_resolutions(ocfg)[2].all()
    xyz, _ = make_queries_uniform(L + N, N)
    xyz[0] = [0.0, 1.0, np.float32(1) - np.float32(2.0 ** -24)]
    t = np.array([tval], np.float32)
    rng = np.random.default_rng(N)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16 if dtype == "fp16" else np.float32)
    sl = dh.dash_hash4d_slice_t(gcfg, dev(t), dev(table))
    out = dh.dash_hash4d_slice_fwd(gcfg, dev(xyz), sl)
    torch.cuda.synchronize()
    ref, mag = oracle.oracle_fwd(ocfg, N, xyz, t, table, t_stride=0, want_abs=True)
    tr = lambda a: np.asarray(a).reshape(N, L, F).transpose(1, 0, 2)
    check_close(tr(out.cpu().numpy()), tr(ref), tr(mag), RTOL_FP16 if dtype == "fp16" else RTOL_FP32, L,
                what="slice fwd")
    # and it agrees with the library's own 16-corner forward at the same timestamp
    out16 = dh.dash_hash4d_fwd(gcfg, dev(xyz), dev(t), dev(table), t_stride=0)
    torch.testing.assert_close(out, out16, rtol=1e-5, atol=1e-6)


def test_slice_full_size_c3_and_index_list():
    wl = make_workload("C3", with_dout=False)
    enc, N = wl.spec.enc, wl.N
    ocfg, gcfg = oracle.config_from_params(enc), dh.config_from_params(enc)
    t = np.array([wl.t[7]], np.float32)                                   # a frame-aligned timestamp j/300
    sl = dh.dash_hash4d_slice_t(gcfg, dev(t), dev(wl.table))
    out = dh.dash_hash4d_slice_fwd(gcfg, dev(wl.xyz), sl)
    torch.cuda.synchronize()
    ref, mag = oracle.oracle_fwd(ocfg, N, wl.xyz, t, wl.table, t_stride=0, want_abs=True)
    L, F = enc.L, enc.F
    tr = lambda a: np.asarray(a).reshape(N, L, F).transpose(1, 0, 2)
    check_close(tr(out.cpu().numpy()), tr(ref), tr(mag), RTOL_FP32, L, what="C3 slice")
    index = np.random.default_rng(0).integers(0, N, 10_000).astype(np.int32)
    out_i = dh.dash_hash4d_slice_fwd(gcfg, dev(wl.xyz), sl, index=dev(index))
    torch.testing.assert_close(out_i, out[torch.from_numpy(index).long().cuda()], rtol=0, atol=0)


@pytest.mark.parametrize("path", [0, 2])       # 0: the library decides (fused here); 2: two-pass, as for a slice beyond L2
@pytest.mark.parametrize("name,widths_tail", [("C2", [64, 64, 10]), ("C2", [128, 10])])
def test_deform_slice_fwd_parity(name, widths_tail, path, set_debug):
    set_debug(dh.DEBUG_DEFORM_PATH, path)
    wl = make_workload(name, n_override=30_000, with_dout=False)
    enc, N = wl.spec.enc, wl.N
    widths = [enc.L * enc.F] + widths_tail
    ocfg, gcfg = oracle.config_from_params(enc), dh.config_from_params(enc)
    table = (wl.table * 1e4).astype(np.float32)
    params = make_mlp_params(3, widths)
    base = np.random.default_rng(1).standard_normal((N, 10)).astype(np.float32)
    t = np.array([0.6180339], np.float32)
    m = dh.make_mlp_config(widths)
    sl = dh.dash_hash4d_slice_t(gcfg, dev(t), dev(table))
    need = dh.dash_deform_slice_workspace_bytes(gcfg, m, N)
    assert (need == 0) == (path == 0) and (path == 0 or need == N * enc.L * enc.F * 4)
    out = dh.dash_deform_slice_fwd(gcfg, m, dev(wl.xyz), sl, dev(params), base=dev(base))
    torch.cuda.synchronize()
    feat = oracle.oracle_fwd(ocfg, N, wl.xyz, t, table, t_stride=0)
    check_mlp_out(out.cpu().numpy(), feat, params, widths, base, "deform slice")


def test_slice_errors():
    cfg = dh.make_config(4, 2, 100003, 16, 512, 8, 64)                     # hashed levels, T not a power of two
    t = torch.zeros(1, device="cuda")
    with pytest.raises(dh.Hash4DError) as e:
        dh.dash_hash4d_slice_t(cfg, t, torch.zeros((4, 100003, 2), device="cuda"))
    assert e.value.status == 2
