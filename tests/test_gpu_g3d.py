"""GPU parity of the 3D hash encoder G_3D (dash_hash3d_*; Eq. 3; Q26) against the CPU
oracle through the C ABI: indices bit-exact, features / gradients within tests/parity_utils.py tolerances.
Run on the B200 box:  python -m pytest tests -m gpu"""
import numpy as np
import pytest
import torch

import oracle
import paper_2507_19141_b200 as dh
from dash_inputs import make_g3d_workload, make_points_clustered, make_queries_uniform
from parity_utils import RTOL_FP16, RTOL_FP32, check_close, fixed_point_quantum

pytestmark = pytest.mark.gpu
DC = dh.FLAG_DENSE_COARSE


def dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def configs(L, F, T, rs, dtype="fp32", flags=DC, primes=(0, 0, 0, 0)):
    # temporal fields deliberately invalid (0): the 3D calls must ignore them
    o = oracle.make_config(L, F, T, rs[0], rs[1], 0, 0, dtype, primes=primes, dense_coarse=bool(flags & DC))
    g = dh.make_config(L, F, T, rs[0], rs[1], 0, 0, dtype, primes=primes, flags=flags)
    return o, g


VARIANTS = [
    # L, F, T, res_s, dtype, N
    (1, 1, 4096, (16, 16), "fp32", 1000),
    (4, 1, 100003, (16, 200), "fp16", 3001),
    (5, 2, 1 << 14, (8, 300), "fp16", 2049),
    (16, 2, 1 << 19, (16, 2048), "fp32", 50_001),       # Instant-NGP-like: dense l = 0..3
    (16, 4, 1 << 17, (16, 4096), "fp16", 20_000),
    (7, 8, 1 << 12, (4, 512), "fp32", 5000),
    (3, 8, 5000, (4, 64), "fp16", 777),
    (16, 2, 1 << 19, (16, 2048), "fp32", 0),
]


@pytest.mark.parametrize("L,F,T,rs,dtype,N", VARIANTS)
@pytest.mark.parametrize("flags", [DC, 0, DC | dh.FLAG_ZERO_GRAD, DC | dh.FLAG_DETERMINISTIC_BWD])
def test_g3d_parity(L, F, T, rs, dtype, N, flags):
    ocfg, gcfg = configs(L, F, T, rs, dtype, flags)
    rs_o, dn_o = oracle.oracle3d_resolutions(ocfg)
    rs_g, dn_g = dh.dash_hash3d_resolutions(gcfg)
    assert list(rs_o) == rs_g and list(dn_o) == dn_g
    rng = np.random.default_rng(L * 131 + F * 7 + N)
    if N >= 20_000:
        xyz = make_points_clustered(L + F, N, 64, 0.05)
    else:
        xyz, _ = make_queries_uniform(L * 17 + F, max(N, 1))
        xyz = xyz[:N]
    if N > 3:
        xyz[0] = [0.0, 1.0, np.float32(1) - np.float32(2.0 ** -24)]
        xyz[1] = [np.nan, -0.5, 1.5]
        xyz[2] = [0.5, 0.25, 0.125]                      # on vertices of power-of-two levels
    table = rng.uniform(-1e-4, 1e-4, (L, T, F)).astype(np.float16 if dtype == "fp16" else np.float32)
    dout = rng.standard_normal((N, L * F)).astype(np.float32)
    xd = dev(xyz) if N else torch.empty((0, 3), device="cuda")
    tr = lambda a: np.asarray(a).reshape(N, L, F).transpose(1, 0, 2)

    if not (flags & ~DC):            # indices + forward once per dense/hashed setting
        ref_idx, ref_w = oracle.oracle3d_indices(ocfg, N, xyz)
        idx, w = dh.dash_hash3d_indices(gcfg, xd, N=N)
        torch.cuda.synchronize()
        assert np.array_equal(idx.cpu().numpy().view(np.uint32), ref_idx)
        if N:
            np.testing.assert_allclose(w.cpu().numpy(), ref_w, rtol=1e-6, atol=1e-9)
            assert ref_idx.max() < T
        ref, mag = oracle.oracle3d_fwd(ocfg, N, xyz, table, want_abs=True)
        out = dh.dash_hash3d_fwd(gcfg, xd, dev(table), N=N)
        torch.cuda.synchronize()
        if N:
            check_close(tr(out.cpu().numpy()), tr(ref), tr(mag), RTOL_FP16 if dtype == "fp16" else RTOL_FP32, L,
                        what="g3d fwd")

    start = np.zeros((L, T, F), np.float32)
    ref, mag, hits = oracle.oracle3d_bwd(ocfg, N, xyz, dout, dtable=start.copy(), want_abs=True, want_hits=True)
    dt = dev(start)
    dt.fill_(7.0)
    if not (flags & dh.FLAG_ZERO_GRAD):
        dh.dash_hash4d_zero(gcfg, dt)
    dh.dash_hash3d_bwd(gcfg, xd, dev(dout), dt, N=N)
    torch.cuda.synchronize()
    got = dt.cpu().numpy()
    q = fixed_point_quantum(N, float(np.abs(dout).max())) if (flags & dh.FLAG_DETERMINISTIC_BWD and N) else 0.0
    check_close(got, ref, mag, RTOL_FP32, L, hits=hits, what="g3d bwd", quantum=q)


def test_g3d_index_list_and_packed_rows():
    L, F, T = 8, 2, 1 << 15
    ocfg, gcfg = configs(L, F, T, (16, 512))
    rng = np.random.default_rng(4)
    rows = rng.random((5000, 4), dtype=np.float32)                      # packed [rows][4]; 4th column unused
    index = rng.integers(0, 5000, 12_345).astype(np.int32)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float32)
    ref, mag = oracle.oracle3d_fwd(ocfg, len(index), rows, table, index=index, want_abs=True)
    out = dh.dash_hash3d_fwd(gcfg, dev(rows), dev(table), index=dev(index))
    torch.cuda.synchronize()
    tr = lambda a: np.asarray(a).reshape(len(index), L, F).transpose(1, 0, 2)
    check_close(tr(out.cpu().numpy()), tr(ref), tr(mag), RTOL_FP32, L, what="g3d indexed fwd")


def test_g3d_equals_4d_kernels_at_nt1_t0():
    """The 8-corner kernels against the library's own 16-corner kernels in the special case where they must agree."""
    L, F, T, N = 6, 4, 1 << 14, 9000
    g3 = dh.make_config(L, F, T, 8, 400, 1, 1, "fp16", flags=0)
    xyz, _ = make_queries_uniform(3, N)
    rng = np.random.default_rng(8)
    table = dev(rng.uniform(-1, 1, (L, T, F)).astype(np.float16))
    xd, t0 = dev(xyz), torch.zeros(1, device="cuda")
    a = dh.dash_hash3d_fwd(g3, xd, table)
    b = dh.dash_hash4d_fwd(g3, xd, t0, table, t_stride=0)
    i3, _ = dh.dash_hash3d_indices(g3, xd)
    i4, _ = dh.dash_hash4d_indices(g3, xd, t0, t_stride=0)
    torch.cuda.synchronize()
    assert torch.equal(i3, i4[:, :, :8])
    torch.testing.assert_close(a, b, rtol=1e-6, atol=1e-7)


def test_g3d_errors():
    cfg = dh.make_config(4, 2, 4096, 16, 8, 0, 0)                       # res_s_min > res_s_max
    x = torch.zeros((4, 3), device="cuda")
    with pytest.raises(dh.Hash4DError) as e:
        dh.dash_hash3d_fwd(cfg, x, torch.zeros((4, 4096, 2), device="cuda"))
    assert e.value.status == 1
    cfg = dh.make_config(4, 2, 4096, 16, 64, 0, 0)
    with pytest.raises(dh.Hash4DError):                                  # the 4D call does need a temporal range
        dh.dash_hash4d_fwd(cfg, x, torch.zeros(4, device="cuda"), torch.zeros((4, 4096, 2), device="cuda"))


def test_g3d_full_size_workload():
    """1.5M points, L=16 F=2 T=2^19 (dash_inputs.G3D_SPEC), the launch configuration bench.py times."""
    wl = make_g3d_workload()
    enc, N = wl.spec.enc, wl.N
    ocfg, gcfg = configs(enc.L, enc.F, enc.T, (enc.res_s_min, enc.res_s_max))
    L, F = enc.L, enc.F
    tr = lambda a: np.asarray(a).reshape(N, L, F).transpose(1, 0, 2)
    xd = dev(wl.xyz)
    ref, mag = oracle.oracle3d_fwd(ocfg, N, wl.xyz, wl.table, want_abs=True)
    out = dh.dash_hash3d_fwd(gcfg, xd, dev(wl.table))
    torch.cuda.synchronize()
    check_close(tr(out.cpu().numpy()), tr(ref), tr(mag), RTOL_FP32, L, what="G3D fwd")
    del ref, mag, out
    ref, mag, hits = oracle.oracle3d_bwd(ocfg, N, wl.xyz, wl.dout, want_abs=True, want_hits=True)
    dt = torch.full((L, enc.T, F), 7.0, device="cuda")
    dh.dash_hash3d_bwd(dh.with_flags(gcfg, DC | dh.FLAG_ZERO_GRAD), xd, dev(wl.dout), dt)
    torch.cuda.synchronize()
    check_close(dt.cpu().numpy(), ref, mag, RTOL_FP32, L, hits=hits, what="G3D bwd")
    sel = np.arange(0, N, N // 65536)[:65536]
    ref_idx, _ = oracle.oracle3d_indices(ocfg, len(sel), np.ascontiguousarray(wl.xyz[sel]), want_weights=False)
    idx, _ = dh.dash_hash3d_indices(gcfg, dev(wl.xyz[sel]), want_weights=False)
    assert np.array_equal(idx.cpu().numpy().view(np.uint32), ref_idx)


@pytest.mark.parametrize("L,F,T,rs,dtype,N", [v for v in VARIANTS if v[5] > 0])
@pytest.mark.parametrize("group", [0, 1, 4])
def test_g3d_coordinate_gradient_parity(L, F, T, rs, dtype, N, group, set_debug):
    """dash_hash3d_bwd_input against oracle3d_bwd_input: |err| <= rtol * sum|terms| (rtol as the 4D call: 1e-5 fp32,
    2e-3 fp16 tables), with edge points (vertices, clamped and NaN coordinates) and an index list."""
    set_debug(dh.DEBUG_FWD_GROUP, group)
    ocfg, gcfg = configs(L, F, T, rs, dtype)
    rng = np.random.default_rng(L * 31 + F + N)
    pts = make_points_clustered(L + F, N)
    pts[:6] = [[0, 0, 0], [1, 1, 1], [0.5, 0.25, 0.75], [-1, 0.3, 2], [np.nan, 0.5, 0.5], [np.float32(1) - np.float32(2.0 ** -24)] * 3]
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16 if dtype == "fp16" else np.float32)
    dout = rng.standard_normal((N, L * F)).astype(np.float32)
    ref, mag = oracle.oracle3d_bwd_input(ocfg, N, pts, table, dout, want_abs=True)
    dq = torch.full((N, 3), 7.0, device="cuda")                                # overwritten, not accumulated
    dh.dash_hash3d_bwd_input(gcfg, dev(pts), dev(table), dev(dout), dq=dq)
    torch.cuda.synchronize()
    rtol = RTOL_FP16 if dtype == "fp16" else RTOL_FP32
    err = np.abs(dq.cpu().numpy().astype(np.float64) - ref)
    assert (err <= rtol * mag + 1e-30).all(), f"worst err/A {(err / (mag + 1e-300)).max():.3e}"
    assert dq[3, 0] == 0 and dq[3, 2] == 0 and dq[4, 0] == 0                    # clamped / NaN coordinates
    index = rng.integers(0, N, 500).astype(np.int32)
    got = dh.dash_hash3d_bwd_input(gcfg, dev(pts), dev(table), dev(dout[:500].copy()), index=dev(index)).cpu().numpy()
    ref_i, mag_i = oracle.oracle3d_bwd_input(ocfg, 500, pts, table, dout[:500].copy(), index=index, want_abs=True)
    assert (np.abs(got - ref_i) <= rtol * mag_i + 1e-30).all()
