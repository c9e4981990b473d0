"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Indices bit-exact; features / gradients within the tolerances of tests/parity_utils.py.
Run on the B200 box:  python -m pytest tests -m gpu
"""
import os

import numpy as np
import pytest
import torch

import oracle
import paper_2507_19141_b200 as dh
from dash_inputs import CONFIGS, EncoderParams, make_queries_uniform, make_workload
from parity_utils import RTOL_FP16, RTOL_FP32, check_close, fixed_point_quantum

pytestmark = pytest.mark.gpu

DC = dh.FLAG_DENSE_COARSE


def dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def both_configs(enc: EncoderParams, flags=DC, primes=(0, 0, 0, 0)):
    ocfg = oracle.config_from_params(enc, primes=primes, dense_coarse=bool(flags & DC))
    gcfg = dh.config_from_params(enc, primes=primes, flags=flags)
    return ocfg, gcfg


def u32(t: torch.Tensor) -> np.ndarray:
    return t.cpu().numpy().view(np.uint32)


def run_fwd_parity(enc, xyz, t, table, index=None, t_stride=1, flags=DC, primes=(0, 0, 0, 0), rtol=None,
                   what=""):
    ocfg, gcfg = both_configs(enc, flags, primes)
    N = len(index) if index is not None else (len(t) if t_stride else len(xyz))
    ref, mag = oracle.oracle_fwd(ocfg, N, xyz, t, table, index=index, t_stride=t_stride, want_abs=True)
    out = dh.dash_hash4d_fwd(gcfg, dev(xyz), dev(t), dev(table), index=dev(index), t_stride=t_stride, N=N)
    torch.cuda.synchronize()
    rtol = rtol or (RTOL_FP16 if enc.table_dtype == "fp16" else RTOL_FP32)
    L, F = enc.L, enc.F
    tr = lambda a: np.asarray(a).reshape(N, L, F).transpose(1, 0, 2)
    return check_close(tr(out.cpu().numpy()), tr(ref), tr(mag), rtol, L, what=what + " fwd")


def run_bwd_parity(enc, xyz, t, dout, index=None, t_stride=1, flags=DC, primes=(0, 0, 0, 0), what="",
                   init=None):
    ocfg, gcfg = both_configs(enc, flags, primes)
    N = len(index) if index is not None else (len(t) if t_stride else len(xyz))
    L, F, T = enc.L, enc.F, enc.T
    start = np.zeros((L, T, F), np.float32) if init is None else init.copy()
    ref, mag, hits = oracle.oracle_bwd(ocfg, N, xyz, t, dout, index=index, t_stride=t_stride,
                                       dtable=start.copy(), want_abs=True, want_hits=True)
    if init is not None:
        mag = mag + np.abs(init)
    dt = dev(start)
    if init is None and not (flags & dh.FLAG_ZERO_GRAD):
        dt.fill_(7.0)                      # garbage: dash_hash4d_zero must clear it
        dh.dash_hash4d_zero(gcfg, dt)
    elif flags & dh.FLAG_ZERO_GRAD:
        dt.fill_(7.0)                      # garbage: ZERO_GRAD must overwrite it
    dh.dash_hash4d_bwd(gcfg, dev(xyz), dev(t), dev(dout), dt, index=dev(index), t_stride=t_stride, N=N)
    torch.cuda.synchronize()
    got = dt.cpu().numpy()
    quantum = fixed_point_quantum(N, float(np.abs(dout).max())) if flags & dh.FLAG_DETERMINISTIC_BWD else 0.0
    worst = check_close(got, ref, mag, RTOL_FP32, L, hits=hits, what=what + " bwd", quantum=quantum)
    # whole-buffer checksum, valid at any size: weights sum to 1
    np.testing.assert_allclose(got.astype(np.float64).sum(1).reshape(-1)
                               - (0 if init is None else init.astype(np.float64).sum(1).reshape(-1)),
                               dout.astype(np.float64).sum(0), rtol=0,
                               atol=1e-5 * np.abs(dout).astype(np.float64).sum(0).max() + 1e-6)
    return got, worst


# ----------------------------------------------------------------------------------------------------
# BASELINE.json configs: indices bit-exact, fwd + bwd parity at FULL size, bench launch configuration
# ----------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C5"])
def test_config_full_size_parity(name):
    wl = make_workload(name)
    enc = wl.spec.enc
    ocfg, gcfg = both_configs(enc)
    N = wl.N
    # indices: bit-exact.  Full for C1-C3; a strided 64k-query sample for C4/C5 (1 GB dumps otherwise)
    if N <= 300_000:
        sel = None
        xyz_s, t_s, idx_s, Ns = wl.xyz, wl.t, wl.index, N
    else:
        sel = np.arange(0, N, N // 65536)[:65536]
        t_s, Ns = np.ascontiguousarray(wl.t[sel]), len(sel)
        if wl.index is not None:
            xyz_s, idx_s = wl.xyz, np.ascontiguousarray(wl.index[sel])
        else:
            xyz_s, idx_s = np.ascontiguousarray(wl.xyz[sel]), None
    ref_idx, ref_w = oracle.oracle_indices(ocfg, Ns, xyz_s, t_s, index=idx_s)
    idx, w = dh.dash_hash4d_indices(gcfg, dev(xyz_s), dev(t_s), index=dev(idx_s), N=Ns)
    torch.cuda.synchronize()
    assert np.array_equal(u32(idx), ref_idx), f"{name}: corner indices differ"
    np.testing.assert_allclose(w.cpu().numpy(), ref_w, rtol=1e-6, atol=1e-9)
    assert u32(idx).max() < enc.T
    del ref_idx, ref_w, idx, w
    run_fwd_parity(enc, wl.xyz, wl.t, wl.table, index=wl.index, what=name)
    run_bwd_parity(enc, wl.xyz, wl.t, wl.dout, index=wl.index, what=name)
    run_bwd_parity(enc, wl.xyz, wl.t, wl.dout, index=wl.index, flags=DC | dh.FLAG_ZERO_GRAD,
                   what=name + " zero_grad")


# ----------------------------------------------------------------------------------------------------
# Variants: F x dtype x L x T (incl. non-power-of-two T, ragged tiles, L not a multiple of the group)
# ----------------------------------------------------------------------------------------------------

VARIANTS = [
    # L, F, T, res_s, res_t, dtype, N
    (1, 1, 4096, (16, 16), (8, 8), "fp32", 1000),
    (4, 1, 100003, (16, 200), (8, 40), "fp16", 3001),
    (5, 2, 1 << 14, (8, 300), (4, 60), "fp16", 2049),
    (12, 2, 1 << 15, (16, 1024), (8, 100), "fp32", 4097),
    (16, 4, 1 << 15, (16, 2048), (8, 150), "fp32", 3333),
    (7, 4, 50021, (16, 512), (8, 64), "fp16", 2500),
    (3, 8, 1 << 13, (16, 64), (8, 16), "fp32", 777),
    (16, 8, 1 << 14, (16, 4096), (8, 300), "fp16", 1500),
    (32, 2, 1 << 12, (4, 4096), (2, 300), "fp32", 1025),
    (17, 2, 1 << 12, (4, 999), (2, 77), "fp32", 513),
]


@pytest.mark.parametrize("L,F,T,rs,rt,dtype,N", VARIANTS)
@pytest.mark.parametrize("flags", [DC, 0])
def test_variants(L, F, T, rs, rt, dtype, N, flags):
    enc = EncoderParams(L, F, T, rs[0], rs[1], rt[0], rt[1], dtype)
    rng = np.random.default_rng(L * 1000 + F)
    xyz, t = make_queries_uniform(L * 7 + F, N)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16 if dtype == "fp16" else np.float32)
    dout = rng.standard_normal((N, L * F)).astype(np.float32)
    ocfg, gcfg = both_configs(enc, flags)
    ref_idx, _ = oracle.oracle_indices(ocfg, N, xyz, t)
    idx, _ = dh.dash_hash4d_indices(gcfg, dev(xyz), dev(t))
    assert np.array_equal(u32(idx), ref_idx)
    # fp16 tables: the conversion is exact, so the fp32 bar holds too (stricter than the stated 2e-3)
    run_fwd_parity(enc, xyz, t, table, flags=flags, rtol=RTOL_FP32)
    run_bwd_parity(enc, xyz, t, dout, flags=flags)
    run_bwd_parity(enc, xyz, t, dout, flags=flags | dh.FLAG_ZERO_GRAD)


@pytest.mark.parametrize("group", [1, 2, 4, 8, 16])
def test_every_level_group_size(group, set_debug):
    """The scheduler's level-group size only changes the launch shape, never the result."""
    set_debug(dh.DEBUG_FWD_GROUP, group)
    set_debug(dh.DEBUG_BWD_GROUP, group)
    for (L, F, dtype) in [(16, 2, "fp32"), (16, 4, "fp16"), (6, 2, "fp32")]:
        enc = EncoderParams(L, F, 1 << 14, 16, 1024, 8, 100, dtype)
        rng = np.random.default_rng(group)
        N = 1237
        xyz, t = make_queries_uniform(group, N)
        table = rng.uniform(-1, 1, (L, enc.T, F)).astype(np.float16 if dtype == "fp16" else np.float32)
        dout = rng.standard_normal((N, L * F)).astype(np.float32)
        run_fwd_parity(enc, xyz, t, table, rtol=RTOL_FP32)
        run_bwd_parity(enc, xyz, t, dout)
        run_bwd_parity(enc, xyz, t, dout, flags=DC | dh.FLAG_ZERO_GRAD)


def test_custom_primes():
    enc = EncoderParams(6, 2, 1 << 13, 16, 512, 8, 64)
    primes = (7, 19349663, 83492791, 2971215073)
    rng = np.random.default_rng(1)
    xyz, t = make_queries_uniform(2, 2000)
    table = rng.uniform(-1, 1, (6, enc.T, 2)).astype(np.float32)
    ocfg, gcfg = both_configs(enc, primes=primes)
    ref_idx, _ = oracle.oracle_indices(ocfg, 2000, xyz, t)
    idx, _ = dh.dash_hash4d_indices(gcfg, dev(xyz), dev(t))
    assert np.array_equal(u32(idx), ref_idx)
    run_fwd_parity(enc, xyz, t, table, primes=primes)


# ----------------------------------------------------------------------------------------------------
# Input views: index list, broadcast t, packed [N][4] rows
# ----------------------------------------------------------------------------------------------------

def test_index_list_broadcast_t_and_packed_rows():
    enc = CONFIGS["C2"].enc
    rng = np.random.default_rng(5)
    rows = rng.random((500, 3), dtype=np.float32)
    index = rng.integers(0, 500, 3000).astype(np.int32)
    t = rng.random(3000, dtype=np.float32)
    table = rng.uniform(-1, 1, (enc.L, enc.T, enc.F)).astype(np.float32)
    dout = rng.standard_normal((3000, enc.L * enc.F)).astype(np.float32)
    run_fwd_parity(enc, rows, t, table, index=index)
    run_bwd_parity(enc, rows, t, dout, index=index)
    # one timestamp per call (render-frame shape)
    t0 = np.array([0.40625], np.float32)
    run_fwd_parity(enc, rows, t0, table, index=index, t_stride=0)
    run_bwd_parity(enc, rows, t0, dout, index=index, t_stride=0)
    # packed rows: xyz stride 4, t = base + 3, stride 4
    packed = np.ascontiguousarray(rng.random((700, 4), dtype=np.float32))
    ocfg, gcfg = both_configs(enc)
    ref = oracle.oracle_fwd(ocfg, 700, packed, packed.reshape(-1)[3:], table, t_stride=4)
    pd = dev(packed)
    out = dh.dash_hash4d_fwd(gcfg, pd, pd.view(-1)[3:], dev(table), t_stride=4, N=700)
    ref2 = oracle.oracle_fwd(ocfg, 700, np.ascontiguousarray(packed[:, :3]),
                             np.ascontiguousarray(packed[:, 3]), table)
    assert np.array_equal(ref, ref2)
    np.testing.assert_allclose(out.cpu().numpy(), ref, rtol=1e-5, atol=1e-6)


# ----------------------------------------------------------------------------------------------------
# Edge inputs (reading Q12, Q4, Q5)
# ----------------------------------------------------------------------------------------------------

def test_edge_inputs_indices_bit_exact():
    enc = CONFIGS["C3"].enc
    one_m = np.nextafter(np.float32(1), np.float32(0))
    special = np.array([0.0, one_m, 1.0, 2.5, -0.0, -1.0, np.nan, np.inf, -np.inf, 0.5, 0.25, 1e-30,
                        np.float32(1) / 3, 1 - 2.0 ** -12], np.float32)
    frames = (np.arange(300) / 300.0).astype(np.float32)          # frame-aligned timestamps (Q4 hazard)
    verts = (np.arange(0, 4097) / 4096.0).astype(np.float32)      # exact grid vertices of the finest level
    coords = np.concatenate([special, frames, verts])
    rng = np.random.default_rng(0)
    N = 20000
    q = coords[rng.integers(0, len(coords), (N, 4))]
    q[:len(coords)] = coords[:, None]                              # every special value on all 4 axes at once
    xyz, t = np.ascontiguousarray(q[:, :3]), np.ascontiguousarray(q[:, 3])
    ocfg, gcfg = both_configs(enc)
    ref_idx, ref_w = oracle.oracle_indices(ocfg, N, xyz, t)
    idx, w = dh.dash_hash4d_indices(gcfg, dev(xyz), dev(t))
    assert np.array_equal(u32(idx), ref_idx)
    np.testing.assert_allclose(w.cpu().numpy(), ref_w, rtol=1e-6, atol=1e-9)
    table = rng.uniform(-1, 1, (enc.L, enc.T, enc.F)).astype(np.float32)
    run_fwd_parity(enc, xyz, t, table, what="edge")
    dout = rng.standard_normal((N, enc.L * enc.F)).astype(np.float32)
    run_bwd_parity(enc, xyz, t, dout, what="edge")


def test_exact_table_value_at_vertices_bitwise():
    """Power-of-two schedule, x = i/N: weights are exactly 0/1 so the GPU must return the table entry
    bit for bit (the sum has one non-zero term)."""
    enc = EncoderParams(4, 2, 1 << 17, 16, 128, 8, 64)
    rng = np.random.default_rng(2)
    n = 4096
    g = np.stack([rng.integers(0, 16, n), rng.integers(0, 16, n), rng.integers(0, 16, n),
                  rng.integers(0, 8, n)], 1)
    xyz = (g[:, :3] / 16.0).astype(np.float32)
    t = (g[:, 3] / 8.0).astype(np.float32)
    table = rng.uniform(-1, 1, (4, enc.T, 2)).astype(np.float32)
    ocfg, gcfg = both_configs(enc)
    ref = oracle.oracle_fwd(ocfg, n, xyz, t, table)
    out = dh.dash_hash4d_fwd(gcfg, dev(xyz), dev(t), dev(table))
    assert np.array_equal(out.cpu().numpy(), ref)


def test_empty_and_single_query():
    enc = CONFIGS["C1"].enc
    ocfg, gcfg = both_configs(enc)
    table = dev(np.zeros((enc.L, enc.T, enc.F), np.float32))
    xyz = torch.empty((0, 3), device="cuda"); t = torch.empty((0,), device="cuda")
    out = dh.dash_hash4d_fwd(gcfg, xyz, t, table, N=0, t_stride=1)
    assert out.shape == (0, enc.L * enc.F)
    dt = torch.full((enc.L, enc.T, enc.F), 3.0, device="cuda")
    dh.dash_hash4d_bwd(gcfg, xyz, t, torch.empty((0, enc.L * enc.F), device="cuda"), dt, N=0, t_stride=1)
    assert (dt == 3.0).all()
    dh.dash_hash4d_bwd(dh.with_flags(gcfg, DC | dh.FLAG_ZERO_GRAD), xyz, t,
                       torch.empty((0, enc.L * enc.F), device="cuda"), dt, N=0, t_stride=1)
    assert (dt == 0.0).all()
    xyz1, t1 = make_queries_uniform(3, 1)
    rng = np.random.default_rng(3)
    tab = rng.uniform(-1, 1, (enc.L, enc.T, enc.F)).astype(np.float32)
    run_fwd_parity(enc, xyz1, t1, tab)
    run_bwd_parity(enc, xyz1, t1, rng.standard_normal((1, enc.L * enc.F)).astype(np.float32))


def test_bwd_accumulates_into_existing_gradient():
    enc = CONFIGS["C1"].enc
    wl = make_workload("C1")
    rng = np.random.default_rng(9)
    init = rng.standard_normal((enc.L, enc.T, enc.F)).astype(np.float32)
    run_bwd_parity(enc, wl.xyz, wl.t, wl.dout, init=init)


def test_unit_gradient_returns_the_16_corner_weights():
    enc = CONFIGS["C2"].enc
    ocfg, gcfg = both_configs(enc)
    n = 512
    xyz, t = make_queries_uniform(4, n)
    ref_idx, ref_w = oracle.oracle_indices(ocfg, n, xyz, t)
    for (q, l, f) in [(0, 0, 0), (100, 7, 1), (511, 15, 0)]:
        d = np.zeros((n, enc.L * enc.F), np.float32); d[q, l * enc.F + f] = 1.0
        dt = torch.zeros((enc.L, enc.T, enc.F), device="cuda")
        dh.dash_hash4d_bwd(gcfg, dev(xyz), dev(t), dev(d), dt)
        got = dt.cpu().numpy()
        want = np.zeros(enc.T); np.add.at(want, ref_idx[q, l], ref_w[q, l])
        np.testing.assert_allclose(got[l, :, f], want, rtol=1e-6, atol=1e-9)
        got[l, :, f] = 0
        assert not got.any()


# ----------------------------------------------------------------------------------------------------
# Adjoint identity with device results, determinism, validation flag
# ----------------------------------------------------------------------------------------------------

def test_adjoint_identity_on_device():
    wl = make_workload("C2")
    enc = wl.spec.enc
    _, gcfg = both_configs(enc)
    xyz, t, tab, dout = dev(wl.xyz), dev(wl.t), dev(wl.table), dev(wl.dout)
    y = dh.dash_hash4d_fwd(gcfg, xyz, t, tab)
    g = torch.zeros((enc.L, enc.T, enc.F), device="cuda")
    dh.dash_hash4d_bwd(gcfg, xyz, t, dout, g)
    lhs = (y.double() * dout.double()).sum().item()
    rhs = (tab.double() * g.double()).sum().item()
    scale = (y.double() * dout.double()).abs().sum().item()
    assert abs(lhs - rhs) <= 1e-6 * scale


@pytest.mark.parametrize("name", ["C1", "C2", "C5"])
def test_deterministic_bwd_is_bitwise_reproducible_and_accurate(name):
    n_over = 200_000 if name == "C5" else None
    wl = make_workload(name, n_override=n_over, with_table=False)
    enc = wl.spec.enc
    flags = DC | dh.FLAG_DETERMINISTIC_BWD
    runs = []
    for _ in range(3):
        got, _ = run_bwd_parity(enc, wl.xyz, wl.t, wl.dout, index=wl.index, flags=flags, what=name + " det")
        runs.append(got)
    assert np.array_equal(runs[0], runs[1]) and np.array_equal(runs[0], runs[2])
    got_z, _ = run_bwd_parity(enc, wl.xyz, wl.t, wl.dout, index=wl.index,
                              flags=flags | dh.FLAG_ZERO_GRAD, what=name + " det zero")
    assert np.array_equal(runs[0], got_z)
    # workspace too small is reported, not ignored
    _, gcfg = both_configs(enc, flags)
    with pytest.raises(dh.Hash4DError) as ei:
        dh.dash_hash4d_bwd(gcfg, dev(wl.xyz), dev(wl.t), dev(wl.dout),
                           torch.zeros((enc.L, enc.T, enc.F), device="cuda"), index=dev(wl.index),
                           workspace=torch.empty(1024, dtype=torch.uint8, device="cuda"))
    assert ei.value.status == 3


def test_nondeterministic_bwd_stays_within_tolerance_across_runs():
    wl = make_workload("C5", n_override=400_000, with_table=False)
    for _ in range(3):
        run_bwd_parity(wl.spec.enc, wl.xyz, wl.t, wl.dout, index=wl.index)


def test_validate_inputs_flag():
    enc = CONFIGS["C1"].enc
    _, gcfg = both_configs(enc, DC | dh.FLAG_VALIDATE_INPUTS)
    xyz, t = make_queries_uniform(1, 1000)
    table = dev(np.zeros((enc.L, enc.T, enc.F), np.float32))
    dh.dash_hash4d_fwd(gcfg, dev(xyz), dev(t), table)          # clean inputs pass
    bad = xyz.copy(); bad[17, 1] = np.nan; bad[400, 2] = 1.5
    with pytest.raises(dh.Hash4DError) as ei:
        dh.dash_hash4d_fwd(gcfg, dev(bad), dev(t), table)
    assert ei.value.status == 1 and "2 coordinates" in str(ei.value)


def test_host_buffer_entry_points_match():
    wl = make_workload("C1")
    enc = wl.spec.enc
    ocfg, gcfg = both_configs(enc)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    out_h = torch.empty((wl.N, enc.L * enc.F)).pin_memory()
    dt_h = torch.empty((enc.L, enc.T, enc.F)).pin_memory()
    st = {}
    dh.dash_hash4d_fwd_host(gcfg, pin(wl.xyz), pin(wl.t), dev(wl.table), out_h, staging=st)
    dh.dash_hash4d_bwd_host(gcfg, pin(wl.xyz), pin(wl.t), pin(wl.dout), dt_h, staging=st, reuse_queries=True)
    torch.cuda.synchronize()
    np.testing.assert_allclose(out_h.numpy(), oracle.oracle_fwd(ocfg, wl.N, wl.xyz, wl.t, wl.table),
                               rtol=1e-5, atol=1e-9)
    np.testing.assert_allclose(dt_h.numpy(), oracle.oracle_bwd(ocfg, wl.N, wl.xyz, wl.t, wl.dout),
                               rtol=1e-4, atol=1e-5)


def test_launch_counter_counts_kernels():
    enc = CONFIGS["C1"].enc
    _, gcfg = both_configs(enc)
    wl = make_workload("C1")
    xyz, t, tab = dev(wl.xyz), dev(wl.t), dev(wl.table)
    dh.dash_hash4d_launch_count(reset=True)
    dh.dash_hash4d_fwd(gcfg, xyz, t, tab)
    assert dh.dash_hash4d_launch_count() == 1


# ----------------------------------------------------------------------------------------------------
# NEXT #1: coordinate gradient  dq[n][d] = d<dout[n], G_4D(x_n)>/dx_d   (Q24)
# ----------------------------------------------------------------------------------------------------

def run_bwd_input_parity(enc, xyz, t, table, dout, index=None, t_stride=1, flags=DC, what=""):
    ocfg, gcfg = both_configs(enc, flags)
    N = len(index) if index is not None else (len(t) if t_stride else len(xyz))
    ref, mag = oracle.oracle_bwd_input(ocfg, N, xyz, t, table, dout, index=index, t_stride=t_stride,
                                       want_abs=True)
    dq = torch.full((N, 4), 9.0, device="cuda")          # garbage: the call must overwrite
    dh.dash_hash4d_bwd_input(gcfg, dev(xyz), dev(t), dev(table), dev(dout), dq=dq, index=dev(index),
                             t_stride=t_stride, N=N)
    torch.cuda.synchronize()
    got = dq.cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all()
    err = np.abs(got - ref)
    assert (err <= RTOL_FP32 * mag + 1e-30).all(), \
        f"{what} bwd_input: worst err/A {(err / (mag + 1e-300)).max():.3e}"
    for d in range(4):                                     # normwise per axis
        assert np.linalg.norm(got[:, d] - ref[:, d]) <= RTOL_FP32 * np.linalg.norm(ref[:, d]) + 1e-30
    return got


@pytest.mark.parametrize("name", ["C1", "C2", "C4", "C5"])
def test_bwd_input_configs(name):
    n_over = {"C4": 200_000, "C5": 200_000}.get(name)
    wl = make_workload(name, n_override=n_over)
    run_bwd_input_parity(wl.spec.enc, wl.xyz, wl.t, wl.table, wl.dout, index=wl.index, what=name)


@pytest.mark.parametrize("L,F,T,rs,rt,dtype,N", VARIANTS)
def test_bwd_input_variants(L, F, T, rs, rt, dtype, N):
    enc = EncoderParams(L, F, T, rs[0], rs[1], rt[0], rt[1], dtype)
    rng = np.random.default_rng(L * 100 + F)
    xyz, t = make_queries_uniform(L + F, N)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16 if dtype == "fp16" else np.float32)
    dout = rng.standard_normal((N, L * F)).astype(np.float32)
    run_bwd_input_parity(enc, xyz, t, table, dout)
    run_bwd_input_parity(enc, xyz, t, table, dout, flags=0)


@pytest.mark.parametrize("group", [1, 2, 4, 8, 16])
def test_bwd_input_every_group_size_and_views(group, set_debug):
    set_debug(dh.DEBUG_FWD_GROUP, group)
    enc = EncoderParams(12, 2, 1 << 14, 16, 1024, 8, 100)
    rng = np.random.default_rng(group)
    rows = rng.random((300, 3), dtype=np.float32)
    index = rng.integers(0, 300, 1111).astype(np.int32)
    table = rng.uniform(-1, 1, (12, enc.T, 2)).astype(np.float32)
    dout = rng.standard_normal((1111, 24)).astype(np.float32)
    run_bwd_input_parity(enc, rows, rng.random(1111, dtype=np.float32), table, dout, index=index)
    run_bwd_input_parity(enc, rows, np.array([0.7], np.float32), table, dout, index=index, t_stride=0)


def test_bwd_input_clamped_coordinates_get_zero():
    enc = CONFIGS["C1"].enc
    rng = np.random.default_rng(3)
    q = rng.random((64, 4), dtype=np.float32)
    q[0, 0] = -0.5; q[1, 1] = 1.0; q[2, 2] = np.nan; q[3, 3] = 7.0; q[4] = [np.nan, -1, 2, np.inf]
    table = rng.uniform(-1, 1, (enc.L, enc.T, enc.F)).astype(np.float32)
    dout = rng.standard_normal((64, enc.L * enc.F)).astype(np.float32)
    got = run_bwd_input_parity(enc, np.ascontiguousarray(q[:, :3]), np.ascontiguousarray(q[:, 3]), table, dout)
    assert got[0, 0] == 0 and got[1, 1] == 0 and got[2, 2] == 0 and got[3, 3] == 0 and not got[4].any()


def test_three_d_special_case_nt1_t0():
    """G_3D = the 4D kernels with temporal resolution 1 and one timestamp t = 0."""
    enc = EncoderParams(5, 2, 1 << 12, 4, 64, 1, 1)
    rng = np.random.default_rng(0)
    n = 3000
    xyz, _ = make_queries_uniform(5, n)
    t0 = np.zeros(1, np.float32)
    table = rng.uniform(-1, 1, (5, enc.T, 2)).astype(np.float32)
    dout = rng.standard_normal((n, 10)).astype(np.float32)
    run_fwd_parity(enc, xyz, t0, table, t_stride=0, what="3d")
    run_bwd_parity(enc, xyz, t0, dout, t_stride=0, what="3d")
    run_bwd_input_parity(enc, xyz, t0, table, dout, t_stride=0, what="3d")


def test_host_step_overlapped_copies_match():
    wl = make_workload("C2", n_override=20000)
    enc = wl.spec.enc
    ocfg, gcfg = both_configs(enc, DC | dh.FLAG_ZERO_GRAD)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    out_h = torch.empty((wl.N, enc.L * enc.F)).pin_memory()
    dt_h = torch.empty((enc.L, enc.T, enc.F)).pin_memory()
    step = dh.HostStep(gcfg)
    ref_o = oracle.oracle_fwd(ocfg, wl.N, wl.xyz, wl.t, wl.table)
    ref_g = oracle.oracle_bwd(ocfg, wl.N, wl.xyz, wl.t, wl.dout)
    for _ in range(3):                                   # repeated steps reuse the staging buffers
        out_h.fill_(-1); dt_h.fill_(-1)
        step(pin(wl.xyz), pin(wl.t), dev(wl.table), pin(wl.dout), out_h, dt_h)
        torch.cuda.synchronize()
        np.testing.assert_allclose(out_h.numpy(), ref_o, rtol=1e-5, atol=1e-9)
        np.testing.assert_allclose(dt_h.numpy(), ref_g, rtol=1e-4, atol=1e-5)


# ----------------------------------------------------------------------------------------------------
# NEXT #2: smoothness regulariser, Eq. 11 (Q25)
# ----------------------------------------------------------------------------------------------------

def run_smooth_parity(enc, xyz, t, eps, table, index=None, t_stride=1, flags=DC, grad_scale=0.7, what="",
                      with_grad=True, use_init=True, max_hits=0):
    ocfg, gcfg = both_configs(enc, flags)
    N = len(index) if index is not None else (len(t) if t_stride else len(xyz))
    L, F, T = enc.L, enc.F, enc.T
    # accumulate semantics: start from a non-zero gradient.  (Not in the degenerate case where ~1000 tiny
    # terms are added to one slot: each fp32 add then rounds at the ulp of the large start value, an error
    # of hits * 2^-24 * |init| that has nothing to do with the regulariser.)
    init = np.random.default_rng(1).standard_normal((L, T, F)).astype(np.float32) * (1e-3 if use_init else 0)
    ref_l, ref_g, la, fa, ga = oracle.oracle_smooth(ocfg, N, xyz, t, eps, table, grad_scale=grad_scale,
                                                   index=index, t_stride=t_stride, dtable=init.copy(),
                                                   want_grad=True, want_abs=True)
    loss = torch.full((N,), 5.0, device="cuda")                       # garbage: must be overwritten
    dt = dev(init) if with_grad else None
    dh.dash_hash4d_smooth(gcfg, dev(xyz), dev(t), dev(eps), dev(table), grad_scale=grad_scale, loss=loss,
                          dtable=dt, index=dev(index), t_stride=t_stride, N=N)
    torch.cuda.synchronize()
    got_l = loss.cpu().numpy().astype(np.float64)
    assert np.isfinite(got_l).all()
    # |d| is a difference of two interpolants: its fp32 error is relative to A + A' (oracle's feat_abs),
    # so the loss tolerance has the first-order term 2|d| err(d) (loss_abs) and the second-order err(d)^2
    allow = RTOL_FP32 * la + L * F * (RTOL_FP32 * fa) ** 2 + 1e-30
    err = np.abs(got_l - ref_l)
    assert (err <= allow).all(), f"{what} smooth loss: worst {np.max(err / allow):.2f} x tolerance"
    assert abs(got_l.sum() - ref_l.astype(np.float64).sum()) <= RTOL_FP32 * la.sum() + 1e-30
    if with_grad:
        got_g = dt.cpu().numpy().astype(np.float64)
        errg = np.abs(got_g - ref_g)
        # max_hits: worst-case recursive-summation term (n-1) * 2^-24 * sum|terms| for slots that receive
        # ~max_hits same-sign fp32 reductions (degenerate inputs only; 0 elsewhere)
        allow_g = (RTOL_FP32 + max_hits * 2.0 ** -24) * (ga + np.abs(init)) + 1e-30
        worst = np.unravel_index(np.argmax(errg / allow_g), errg.shape)
        assert (errg <= allow_g).all(), (f"{what} smooth grad: worst {np.max(errg / allow_g):.2f} x tolerance at "
                                         f"{worst}: got {got_g[worst]:.6e} ref {ref_g[worst]:.6e} A {ga[worst]:.3e}")
        for l in range(L):
            num = np.linalg.norm(got_g[l] - ref_g[l]); den = np.linalg.norm(ref_g[l] - init[l])
            assert num <= (1e-4 + max_hits * 2.0 ** -24) * den + 1e-12, f"{what} smooth grad level {l}: {num / max(den, 1e-300):.2e}"
    return got_l


@pytest.mark.parametrize("name,scale", [("C1", 1e-3), ("C2", 1e-3), ("C2", 3e-2), ("C4", 5e-4), ("C5", 2e-3)])
def test_smooth_configs(name, scale):
    n_over = {"C2": 30_000, "C4": 100_000, "C5": 100_000}.get(name)
    wl = make_workload(name, n_override=n_over, with_dout=False)
    eps = np.random.default_rng(9).uniform(-scale, scale, (wl.N, 4)).astype(np.float32)
    run_smooth_parity(wl.spec.enc, wl.xyz, wl.t, eps, (wl.table.astype(np.float32) * 1e4).astype(wl.table.dtype),
                      index=wl.index, what=f"{name} eps={scale}")


@pytest.mark.parametrize("L,F,T,rs,rt,dtype,N", VARIANTS)
def test_smooth_variants(L, F, T, rs, rt, dtype, N):
    enc = EncoderParams(L, F, T, rs[0], rs[1], rt[0], rt[1], dtype)
    rng = np.random.default_rng(L * 10 + F)
    xyz, t = make_queries_uniform(L + 3 * F, N)
    eps = rng.uniform(-4e-3, 4e-3, (N, 4)).astype(np.float32)
    table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16 if dtype == "fp16" else np.float32)
    run_smooth_parity(enc, xyz, t, eps, table)
    run_smooth_parity(enc, xyz, t, eps, table, flags=0, with_grad=False)


@pytest.mark.parametrize("group", [1, 2, 4, 8, 16])
def test_smooth_group_sizes_shared_eps_and_degenerate(group, set_debug):
    set_debug(dh.DEBUG_SMOOTH_GROUP, group)
    enc = EncoderParams(12, 2, 1 << 14, 16, 1024, 8, 100)
    rng = np.random.default_rng(group)
    rows = rng.random((300, 3), dtype=np.float32)
    index = rng.integers(0, 300, 999).astype(np.int32)
    t = rng.random(999, dtype=np.float32)
    table = rng.uniform(-1, 1, (12, enc.T, 2)).astype(np.float32)
    run_smooth_parity(enc, rows, t, rng.uniform(-2e-3, 2e-3, (999, 4)).astype(np.float32), table, index=index,
                      what="per-query eps")
    run_smooth_parity(enc, rows, t, np.array([1e-3, -2e-3, 5e-4, 1e-3], np.float32), table, index=index,
                      what="shared eps")
    got = run_smooth_parity(enc, rows, t, np.zeros((999, 4), np.float32), table, index=index, what="eps=0")
    assert not got.any()                                            # eps = 0: loss exactly 0
    run_smooth_parity(enc, rows, t, np.full((999, 4), 5.0, np.float32), table, index=index, what="clamped",
                      use_init=False, max_hits=999)
    run_smooth_parity(enc, rows, np.array([0.3], np.float32), np.array([1e-3, 0, 0, 2e-3], np.float32), table,
                      index=index, t_stride=0, what="broadcast t")


def test_smooth_rejects_deterministic_flag():
    enc = CONFIGS["C1"].enc
    _, gcfg = both_configs(enc, DC | dh.FLAG_DETERMINISTIC_BWD)
    xyz, t = make_queries_uniform(0, 16)
    with pytest.raises(dh.Hash4DError) as ei:
        dh.dash_hash4d_smooth(gcfg, dev(xyz), dev(t), dev(np.zeros(4, np.float32)),
                              dev(np.zeros((enc.L, enc.T, enc.F), np.float32)),
                              dtable=torch.zeros((enc.L, enc.T, enc.F), device="cuda"))
    assert ei.value.status == 2


def test_calls_are_cuda_graph_capturable():
    """The library only enqueues kernels on the caller's stream (no allocation, no sync), so a whole
    step can be captured once and replayed — the launch-bound small configs (C1/C2) are run that way."""
    wl = make_workload("C2", n_override=20000)
    enc = wl.spec.enc
    ocfg, gcfg = both_configs(enc, DC | dh.FLAG_ZERO_GRAD)
    xyz, t, table, dout = dev(wl.xyz), dev(wl.t), dev(wl.table), dev(wl.dout)
    out = torch.empty((wl.N, enc.L * enc.F), device="cuda")
    dt = torch.empty((enc.L, enc.T, enc.F), device="cuda")
    dq = torch.empty((wl.N, 4), device="cuda")

    def step():
        dh.dash_hash4d_fwd(gcfg, xyz, t, table, out=out)
        dh.dash_hash4d_bwd(gcfg, xyz, t, dout, dt)
        dh.dash_hash4d_bwd_input(gcfg, xyz, t, table, dout, dq=dq)

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step()                                           # warm-up outside capture
    torch.cuda.current_stream().wait_stream(side)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        step()
    out.fill_(-1); dt.fill_(-1); dq.fill_(-1)
    for _ in range(2):
        graph.replay()
    torch.cuda.synchronize()
    np.testing.assert_allclose(out.cpu().numpy(), oracle.oracle_fwd(ocfg, wl.N, wl.xyz, wl.t, wl.table),
                               rtol=1e-5, atol=1e-9)
    np.testing.assert_allclose(dt.cpu().numpy(), oracle.oracle_bwd(ocfg, wl.N, wl.xyz, wl.t, wl.dout),
                               rtol=1e-4, atol=1e-5)
    np.testing.assert_allclose(dq.cpu().numpy(),
                               oracle.oracle_bwd_input(ocfg, wl.N, wl.xyz, wl.t, wl.table, wl.dout),
                               rtol=1e-3, atol=1e-5)


def test_binding_rejects_buffers_that_do_not_match_the_config():
    """The C ABI takes raw pointers; the binding is where allocation sizes are known: a short table /
    out / dout / dtable / t / index, rows < N, or an out-of-range index under VALIDATE_INPUTS must raise, not corrupt."""
    enc = EncoderParams(4, 2, 1 << 10, 8, 64, 4, 16)
    cfg = dh.config_from_params(enc)
    n = 100
    xyz, t = torch.rand((n, 3), device="cuda"), torch.rand(n, device="cuda")
    table = torch.zeros((enc.L, enc.T, enc.F), device="cuda")
    dout = torch.zeros((n, enc.L * enc.F), device="cuda")
    dtable = torch.zeros_like(table)
    dh.dash_hash4d_fwd(cfg, xyz, t, table)                                        # the well-formed call passes
    with pytest.raises(ValueError, match="table"):
        dh.dash_hash4d_fwd(cfg, xyz, t, table[:-1].contiguous())
    with pytest.raises(ValueError, match="out"):
        dh.dash_hash4d_fwd(cfg, xyz, t, table, out=torch.empty((n - 1, enc.L * enc.F), device="cuda"))
    with pytest.raises(ValueError, match="t holds"):
        dh.dash_hash4d_fwd(cfg, xyz, t[:50].contiguous(), table, t_stride=1)
    with pytest.raises(ValueError, match="rows"):
        dh.dash_hash4d_fwd(cfg, xyz, t, table, N=n + 1)
    with pytest.raises(ValueError, match="dout"):
        dh.dash_hash4d_bwd(cfg, xyz, t, dout[:-1].contiguous(), dtable)
    with pytest.raises(ValueError, match="dtable"):
        dh.dash_hash4d_bwd(cfg, xyz, t, dout, dtable[:, :-1].contiguous())
    index = torch.arange(n, device="cuda", dtype=torch.int32)
    with pytest.raises(ValueError, match="index"):
        dh.dash_hash4d_fwd(cfg, xyz, t, table, index=index[:10].contiguous(), N=n)
    bad = index.clone(); bad[7] = n + 5
    cfg_v = dh.config_from_params(enc, flags=DC | dh.FLAG_VALIDATE_INPUTS)
    with pytest.raises(ValueError, match="index values"):
        dh.dash_hash4d_fwd(cfg_v, xyz, t, table, index=bad)
    with pytest.raises(ValueError, match="dq"):
        dh.dash_hash4d_bwd_input(cfg, xyz, t, table, dout, dq=torch.empty((n, 3), device="cuda"))
    with pytest.raises(ValueError, match="slice"):
        dh.dash_hash4d_slice_fwd(cfg, xyz, torch.zeros((enc.L, enc.T - 1, enc.F), device="cuda"))
    with pytest.raises(ValueError, match="m holds"):
        dh.dash_hash4d_adam_step(cfg, table, dtable, torch.zeros(5, device="cuda"), torch.zeros_like(table), 1)


@pytest.mark.parametrize("group", [0, 1, 2, 4])
def test_zero_grad_overwrites_garbage_for_every_group_size(group, set_debug):
    """ZERO_GRAD zeroes each level group's slice (possibly only 4-byte aligned) right before scattering into it:
    N spans many tiles with a ragged tail, L is not a multiple of G, T*F*4 is not always a multiple of 16."""
    variant = 0
    set_debug(dh.DEBUG_BWD_GROUP, group)
    for (L, F, T, n) in [(7, 4, 1 << 13, 40_003), (5, 2, 1 << 12, 3_001), (3, 1, 1003, 777)]:
        enc = EncoderParams(L, F, T, 8, 300, 4, 40)
        rng = np.random.default_rng(L + n)
        xyz, t = make_queries_uniform(L + n, n)
        dout = rng.standard_normal((n, L * F)).astype(np.float32)
        run_bwd_parity(enc, xyz, t, dout, flags=DC | dh.FLAG_ZERO_GRAD, what=f"zero-grad v{variant} G{group} L{L}")


def test_zero_grad_through_the_raw_abi_without_workspace():
    enc = EncoderParams(6, 4, 1 << 12, 8, 200, 4, 30)
    ocfg, gcfg = both_configs(enc, DC | dh.FLAG_ZERO_GRAD)
    n = 5000
    xyz, t = make_queries_uniform(9, n)
    dout = np.random.default_rng(9).standard_normal((n, 24)).astype(np.float32)
    ref, mag = oracle.oracle_bwd(ocfg, n, xyz, t, dout, want_abs=True)
    dt = torch.full((6, 1 << 12, 4), 7.0, device="cuda")
    lib = dh.binding._load()
    import ctypes as C
    xd, td, dd = dev(xyz), dev(t), dev(dout)                                      # keep the device copies alive
    rc = lib.dash_hash4d_bwd(C.byref(gcfg), n, C.c_void_p(xd.data_ptr()), 3, C.c_void_p(td.data_ptr()), 1,
                             None, C.c_void_p(dd.data_ptr()), C.c_void_p(dt.data_ptr()), None, 0,
                             C.c_void_p(torch.cuda.current_stream().cuda_stream))
    torch.cuda.synchronize()
    assert rc == 0
    check_close(dt.cpu().numpy(), ref, mag, RTOL_FP32, 6, what="zero-grad, no workspace")


@pytest.mark.parametrize("bits", [1, 4, 6, 7])
@pytest.mark.parametrize("with_index", [False, True])
def test_sort_queries_is_a_permutation_in_key_order(bits, with_index):
    """dash_hash4d_sort_queries: `order` is a permutation of 0..N-1 and the Morton keys of the coarse spatial cells
    (rebuilt here with numpy: one exact power-of-two fp32 product, floor, bit interleave) are non-decreasing along it.
    Ties may come in any order, so only what is unique is compared."""
    rng = np.random.default_rng(bits)
    rows = 5000
    xyz = rng.random((rows, 3), dtype=np.float32)
    xyz[:5] = [[0, 0, 0], [1, 1, 1], [np.nan, 0.5, -3], [np.float32(1) - np.float32(2.0 ** -24)] * 3, [0.5, 0.25, 0.75]]
    index = rng.integers(0, rows, 7001).astype(np.int32) if with_index else None
    order = dh.dash_hash4d_sort_queries(dev(xyz), index=dev(index), bits=bits).cpu().numpy()
    n = len(index) if with_index else rows
    assert order.shape == (n,) and np.array_equal(np.sort(order), np.arange(n))
    pts = xyz[index] if with_index else xyz
    c = np.clip(np.nan_to_num(pts, nan=0.0), 0, np.float32(1) - np.float32(2.0 ** -24)).astype(np.float32)
    cell = np.minimum((c * np.float32(2 ** bits)).astype(np.uint32), 2 ** bits - 1)
    key = np.zeros(n, np.uint64)
    for b in range(bits):
        for d in range(3):
            key |= ((cell[:, d].astype(np.uint64) >> b) & 1) << (3 * b + d)
    assert (np.diff(key[order].astype(np.int64)) >= 0).all()
    # the sorted order is a valid index list: the forward in that order is the forward, permuted
    enc = EncoderParams(4, 2, 1 << 10, 8, 64, 4, 16)
    cfg = dh.config_from_params(enc)
    t = rng.random(n, dtype=np.float32)
    table = dev(rng.uniform(-1, 1, (4, 1 << 10, 2)).astype(np.float32))
    base = dh.dash_hash4d_fwd(cfg, dev(xyz), dev(t), table, index=dev(index)).cpu().numpy()
    idx_s = (index[order] if with_index else order.astype(np.int32))
    got = dh.dash_hash4d_fwd(cfg, dev(xyz), dev(t[order]), table, index=dev(idx_s)).cpu().numpy()
    np.testing.assert_array_equal(got, base[order])
