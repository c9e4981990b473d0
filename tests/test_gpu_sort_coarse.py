"""GPU parity of the collision-aware path (DASH_HASH4D_FLAG_SORT_COARSE): counting sort of the queries by the 4D cell
of the finest coarse level; backward: run-merged reductions on the coarse levels; forward: the coarse levels walked in
that order; the other levels unchanged.  The results are those of the plain calls (forward: same values; backward: same
sums in another order), so every check is the plain call's check against the oracle (tests/parity_utils.py): element by
element with the hits-aware tolerance, normwise per level, and the whole-buffer checksum.  BASELINE.json config 5 is the
workload the flag exists for.
"""
import ctypes as C

import numpy as np
import pytest
import torch

import oracle
import paper_2507_19141_b200 as dh
from dash_inputs import EncoderParams, make_queries_uniform, make_workload
from parity_utils import RTOL_FP32, check_close
from test_gpu_parity import DC, both_configs, dev, run_bwd_input_parity, run_bwd_parity, run_fwd_parity

pytestmark = pytest.mark.gpu

SC = dh.FLAG_SORT_COARSE
ZG = dh.FLAG_ZERO_GRAD
READY = dh.FLAG_ORDER_READY


@pytest.mark.parametrize("name", ["C3", "C4", "C5"])
def test_full_size_configs(name):
    """The bench's launch configuration (ZERO_GRAD + SORT_COARSE, the library's own choice of coarse levels; the forward
    sorts, the backward of the same step reuses the order).  C3 (N F < 2^21) takes the plain path and needs no workspace."""
    wl = make_workload(name)
    enc, N = wl.spec.enc, wl.N
    cfg = dh.config_from_params(enc, flags=DC | ZG | SC)
    need = dh.dash_hash4d_workspace_bytes(cfg, N, dh.OP_BWD)
    assert need == dh.dash_hash4d_workspace_bytes(cfg, N, dh.OP_FWD)
    assert (need >= 24 * N) if N * enc.F >= (1 << 21) else (need == 0)
    run_fwd_parity(enc, wl.xyz, wl.t, wl.table, index=wl.index, flags=DC | SC, what=name + " sort_coarse")
    run_bwd_parity(enc, wl.xyz, wl.t, wl.dout, index=wl.index, flags=DC | ZG | SC, what=name + " sort_coarse")
    if need:
        # one step as bench.py runs it: fwd sorts into the workspace, bwd (ORDER_READY) reuses it
        ocfg, _ = both_configs(enc, DC)
        ws = torch.empty(need, dtype=torch.uint8, device="cuda")
        xd, td, idd = dev(wl.xyz), dev(wl.t), dev(wl.index)
        out = dh.dash_hash4d_fwd(cfg, xd, td, dev(wl.table), index=idd, workspace=ws)
        dt = torch.full((enc.L, enc.T, enc.F), 7.0, device="cuda")
        dh.dash_hash4d_bwd(dh.with_flags(cfg, DC | ZG | SC | READY), xd, td, dev(wl.dout), dt, index=idd, workspace=ws)
        torch.cuda.synchronize()
        ref, mag, hits = oracle.oracle_bwd(ocfg, N, wl.xyz, wl.t, wl.dout, index=wl.index, want_abs=True, want_hits=True)
        check_close(dt.cpu().numpy(), ref, mag, RTOL_FP32, enc.L, hits=hits, what=name + " bwd on the forward's order")
        plain = dh.dash_hash4d_fwd(dh.config_from_params(enc, flags=DC), xd, td, dev(wl.table), index=idd)
        assert torch.equal(out, plain), "the sorted forward computes the same fp32 values, in another thread order"


@pytest.mark.parametrize("levels", [1, 2, 3, 5, 16])
@pytest.mark.parametrize("chunk", [1, 7, 64])
def test_forced_coarse_levels_and_chunks(levels, chunk, set_debug):
    """Any number of leading levels (hashed ones included, up to all of them) and any chunk length give the plain result;
    N is ragged against the chunk and against the 128-pair blocks."""
    set_debug(dh.DEBUG_BWD_COARSE_LEVELS, levels)
    set_debug(dh.DEBUG_BWD_RUN_CHUNK, chunk)
    for (L, F, T, n, flags) in [(5, 2, 1 << 12, 3001, DC | SC), (16, 4, 1 << 14, 2500, DC | ZG | SC),
                                (7, 1, 100003, 1237, SC), (3, 8, 1 << 13, 777, DC | ZG | SC)]:
        enc = EncoderParams(L, F, T, 4, 300, 2, 40)
        rng = np.random.default_rng(L * 100 + levels + chunk)
        xyz, t = make_queries_uniform(L + levels, n)
        dout = rng.standard_normal((n, L * F)).astype(np.float32)
        run_bwd_parity(enc, xyz, t, dout, flags=flags, what=f"sort_coarse L{L} F{F} levels{levels} chunk{chunk}")
        if chunk == 7:   # the forward does not depend on the chunk length
            table = rng.uniform(-1, 1, (L, T, F)).astype(np.float32)
            run_fwd_parity(enc, xyz, t, table, flags=flags & ~ZG, what=f"sort_coarse fwd L{L} F{F} levels{levels}")


def test_long_runs_index_list_broadcast_t_and_existing_gradient(set_debug):
    """Clustered queries (long runs on every coarse level), an index list with repeats, one timestamp for the whole call,
    and accumulation into a gradient buffer that already holds values."""
    set_debug(dh.DEBUG_BWD_COARSE_LEVELS, 4)
    enc = EncoderParams(8, 2, 1 << 13, 8, 512, 4, 64)
    rng = np.random.default_rng(5)
    rows = 4000
    xyz = np.clip(0.4 + 0.01 * rng.standard_normal((rows, 3)), 0, 0.999).astype(np.float32)
    index = np.repeat(np.sort(rng.choice(rows, 1500, replace=False)).astype(np.int32), 4)
    n = len(index)
    t = rng.random(n, dtype=np.float32)
    dout = rng.standard_normal((n, 16)).astype(np.float32)
    run_bwd_parity(enc, xyz, t, dout, index=index, flags=DC | ZG | SC, what="clustered, indexed")
    init = rng.standard_normal((8, 1 << 13, 2)).astype(np.float32)
    run_bwd_parity(enc, xyz, t, dout, index=index, flags=DC | SC, init=init, what="clustered, accumulate")
    t1 = np.array([0.37], np.float32)
    run_bwd_parity(enc, xyz, t1, dout[:rows], t_stride=0, flags=DC | ZG | SC, what="one timestamp")
    table = rng.uniform(-1, 1, (8, 1 << 13, 2)).astype(np.float16)
    enc16 = EncoderParams(8, 2, 1 << 13, 8, 512, 4, 64, "fp16")
    run_fwd_parity(enc16, xyz, t, table, index=index, flags=DC | SC, rtol=RTOL_FP32, what="clustered, indexed, fp16")
    run_fwd_parity(enc16, xyz, t1, table, t_stride=0, flags=DC | SC, rtol=RTOL_FP32, what="one timestamp, fp16")


def test_tiny_and_edge_inputs(set_debug):
    """N = 1, N below one chunk, every query in one cell, clamped / NaN coordinates."""
    set_debug(dh.DEBUG_BWD_COARSE_LEVELS, 2)
    enc = EncoderParams(4, 2, 1 << 10, 8, 64, 4, 16)
    rng = np.random.default_rng(11)
    for n in (1, 2, 63):
        xyz, t = make_queries_uniform(n, n)
        dout = rng.standard_normal((n, 8)).astype(np.float32)
        run_bwd_parity(enc, xyz, t, dout, flags=DC | ZG | SC, what=f"N={n}")
    n = 300
    xyz = np.full((n, 3), 0.51, np.float32)
    t = np.full(n, 0.26, np.float32)
    dout = rng.standard_normal((n, 8)).astype(np.float32)
    run_bwd_parity(enc, xyz, t, dout, flags=DC | ZG | SC, what="one cell")
    xyz, t = make_queries_uniform(3, n)
    xyz[:6] = [[0, 0, 0], [1, 1, 1], [np.nan, 0.5, -3], [2, 0.1, 0.2], [-1, -1, -1], [0.5, np.inf, 0.5]]
    t[:4] = [1.0, np.nan, -0.5, 7.0]
    run_bwd_parity(enc, xyz, t, dout, flags=DC | ZG | SC, what="edge coordinates")


def test_workspace_is_required_and_sized_by_the_library(set_debug):
    set_debug(dh.DEBUG_BWD_COARSE_LEVELS, 2)
    enc = EncoderParams(4, 2, 1 << 10, 8, 64, 4, 16)
    cfg = dh.config_from_params(enc, flags=DC | SC)
    n = 1000
    need = dh.dash_hash4d_workspace_bytes(cfg, n, dh.OP_BWD)
    assert need >= 24 * n
    assert dh.dash_hash4d_workspace_bytes(cfg, n, dh.OP_FWD) == need       # one buffer serves fwd and bwd of a step
    assert dh.dash_hash4d_workspace_bytes(cfg, n, dh.OP_BWD_INPUT) == need
    assert dh.dash_hash4d_workspace_bytes(cfg, n, dh.OP_SMOOTH) == 0       # the other calls ignore the flag
    assert dh.dash_hash4d_workspace_bytes(dh.with_flags(cfg, DC | SC | dh.FLAG_DETERMINISTIC_BWD), n, dh.OP_BWD) == \
        dh.dash_hash4d_workspace_bytes(dh.with_flags(cfg, DC | dh.FLAG_DETERMINISTIC_BWD), n, dh.OP_BWD)
    xyz, t = make_queries_uniform(1, n)
    dout = np.zeros((n, 8), np.float32)
    xd, td, dd = dev(xyz), dev(t), dev(dout)
    dt = torch.zeros((4, 1 << 10, 2), device="cuda")
    small = torch.empty(need - 16, dtype=torch.uint8, device="cuda")
    lib = dh.binding._load()
    rc = lib.dash_hash4d_bwd(C.byref(cfg), n, C.c_void_p(xd.data_ptr()), 3, C.c_void_p(td.data_ptr()), 1, None,
                             C.c_void_p(dd.data_ptr()), C.c_void_p(dt.data_ptr()), C.c_void_p(small.data_ptr()),
                             small.numel(), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == 3 and "workspace" in dh.dash_hash4d_last_error()          # DASH_HASH4D_WORKSPACE_TOO_SMALL
    rc = lib.dash_hash4d_bwd(C.byref(cfg), n, C.c_void_p(xd.data_ptr()), 3, C.c_void_p(td.data_ptr()), 1, None,
                             C.c_void_p(dd.data_ptr()), C.c_void_p(dt.data_ptr()), None, 0,
                             C.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == 3


def test_flag_is_ignored_by_the_deterministic_mode(set_debug):
    set_debug(dh.DEBUG_BWD_COARSE_LEVELS, 2)
    enc = EncoderParams(4, 2, 1 << 10, 8, 64, 4, 16)
    n = 2000
    rng = np.random.default_rng(2)
    xyz, t = make_queries_uniform(2, n)
    dout = rng.standard_normal((n, 8)).astype(np.float32)
    got = []
    for flags in (DC | ZG | dh.FLAG_DETERMINISTIC_BWD, DC | ZG | dh.FLAG_DETERMINISTIC_BWD | SC):
        cfg = dh.config_from_params(enc, flags=flags)
        dt = torch.empty((4, 1 << 10, 2), device="cuda")
        dh.dash_hash4d_bwd(cfg, dev(xyz), dev(t), dev(dout), dt)
        got.append(dt.cpu().numpy())
    assert np.array_equal(got[0], got[1])                      # bitwise equal with and without the flag


def _g3d_parity(o3, g3, xyz, table, dout, index=None, what=""):
    n = len(index) if index is not None else len(xyz)
    L = g3.L
    ref, mag = oracle.oracle3d_fwd(o3, n, xyz, table, index=index, want_abs=True)
    out = dh.dash_hash3d_fwd(g3, dev(xyz), dev(table), index=dev(index))
    tr = lambda a: np.asarray(a).reshape(n, L, g3.F).transpose(1, 0, 2)
    check_close(tr(out.cpu().numpy()), tr(ref), tr(mag), RTOL_FP32, L, what=what + " g3d fwd")
    plain = dh.dash_hash3d_fwd(dh.with_flags(g3, DC), dev(xyz), dev(table), index=dev(index))
    assert torch.equal(out, plain)
    refg, magg, hits = oracle.oracle3d_bwd(o3, n, xyz, dout, index=index, want_abs=True, want_hits=True)
    dt = torch.full((L, g3.T, g3.F), 7.0, device="cuda")
    dh.dash_hash3d_bwd(g3, dev(xyz), dev(dout), dt, index=dev(index))
    check_close(dt.cpu().numpy(), refg, magg, RTOL_FP32, L, hits=hits, what=what + " g3d bwd")


@pytest.mark.parametrize("levels", [1, 3, 6])
def test_g3d_forced_levels(levels, set_debug):
    """dash_hash3d_fwd / _bwd honour the flag: 3D cells, no t in the key, 4 corners per lane in the run kernel."""
    set_debug(dh.DEBUG_BWD_COARSE_LEVELS, levels)
    rng = np.random.default_rng(levels)
    for (L, F, T, n) in [(6, 2, 1 << 12, 3001), (5, 4, 30011, 1237), (3, 1, 1 << 10, 600)]:
        o3 = oracle.make_config(L, F, T, 4, 200, 1, 1)
        g3 = dh.make_config(L, F, T, 4, 200, 1, 1, flags=DC | ZG | SC)
        assert dh.dash_hash3d_workspace_bytes(g3, n, dh.OP_BWD) >= 24 * n
        xyz = np.clip(0.5 + 0.2 * rng.standard_normal((n, 3)), 0, 0.999).astype(np.float32)
        table = rng.uniform(-1, 1, (L, T, F)).astype(np.float32)
        dout = rng.standard_normal((n, L * F)).astype(np.float32)
        _g3d_parity(o3, g3, xyz, table, dout, what=f"L{L} F{F} levels{levels}")
        index = rng.integers(0, n, 2 * n).astype(np.int32)
        _g3d_parity(o3, g3, xyz, table, rng.standard_normal((2 * n, L * F)).astype(np.float32), index=index,
                    what=f"indexed L{L} F{F} levels{levels}")


def test_g3d_full_size_workload():
    """The bench's G_3D workload (1.5M Gaussians, L = 16, F = 2, T = 2^19) with the library's own choice of levels."""
    from dash_inputs import make_g3d_workload
    wl = make_g3d_workload()
    enc = wl.spec.enc
    o3 = oracle.make_config(enc.L, enc.F, enc.T, enc.res_s_min, enc.res_s_max, 1, 1)
    g3 = dh.make_config(enc.L, enc.F, enc.T, enc.res_s_min, enc.res_s_max, 1, 1, flags=DC | ZG | SC)
    assert dh.dash_hash3d_workspace_bytes(g3, wl.N, dh.OP_FWD) >= 24 * wl.N
    _g3d_parity(o3, g3, wl.xyz, wl.table, wl.dout, what="G3D workload")


def test_sorted_step_is_cuda_graph_capturable(set_debug):
    """A whole step — forward with its sort, backward on the forward's order — captured once and replayed."""
    set_debug(dh.DEBUG_BWD_COARSE_LEVELS, 3)
    enc = EncoderParams(6, 2, 1 << 12, 8, 256, 4, 32)
    n = 5000
    rng = np.random.default_rng(4)
    xyz, t = make_queries_uniform(4, n)
    table = rng.uniform(-1, 1, (6, 1 << 12, 2)).astype(np.float32)
    dout = rng.standard_normal((n, 12)).astype(np.float32)
    ocfg, gcfg = both_configs(enc, DC | ZG | SC)
    bcfg = dh.with_flags(gcfg, DC | ZG | SC | READY)
    ref_f, mag_f = oracle.oracle_fwd(ocfg, n, xyz, t, table, want_abs=True)
    ref, mag, hits = oracle.oracle_bwd(ocfg, n, xyz, t, dout, want_abs=True, want_hits=True)
    xd, td, tabd, dd = dev(xyz), dev(t), dev(table), dev(dout)
    out = torch.empty((n, 12), device="cuda")
    dt = torch.full((6, 1 << 12, 2), 7.0, device="cuda")
    ws = torch.empty(dh.dash_hash4d_workspace_bytes(gcfg, n, dh.OP_BWD), dtype=torch.uint8, device="cuda")
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        dh.dash_hash4d_fwd(gcfg, xd, td, tabd, out=out, workspace=ws)         # warm-up outside the capture
        dh.dash_hash4d_bwd(bcfg, xd, td, dd, dt, workspace=ws)
        stream.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            dh.dash_hash4d_fwd(gcfg, xd, td, tabd, out=out, workspace=ws)
            dh.dash_hash4d_bwd(bcfg, xd, td, dd, dt, workspace=ws)
    for _ in range(2):
        dt.fill_(3.0); out.fill_(5.0); ws.zero_()                              # the replay rebuilds the order itself
        graph.replay()
        torch.cuda.synchronize()
        check_close(dt.cpu().numpy(), ref, mag, RTOL_FP32, 6, hits=hits, what="graph replay bwd")
        tr = lambda a: np.asarray(a).reshape(n, 6, 2).transpose(1, 0, 2)
        check_close(tr(out.cpu().numpy()), tr(ref_f), tr(mag_f), RTOL_FP32, 6, what="graph replay fwd")


def test_packed_rows_custom_primes_non_power_of_two_table_and_validate_flag(set_debug):
    """The sorted path under the other options of the ABI: packed [N][4] rows (xyz stride 4, t = base + 3, stride 4),
    custom primes with Eq. 8 on every level (no dense levels), a table size that is not a power of two, a single level,
    and VALIDATE_INPUTS sharing the workspace header with the sort."""
    set_debug(dh.DEBUG_BWD_COARSE_LEVELS, 3)
    rng = np.random.default_rng(21)
    n = 2500
    packed = np.ascontiguousarray(rng.random((n, 4), dtype=np.float32))
    xyz, t = np.ascontiguousarray(packed[:, :3]), np.ascontiguousarray(packed[:, 3])
    primes = (1, 2246822519, 3266489917, 668265263)
    enc = EncoderParams(6, 2, 50021, 8, 256, 4, 32)
    table = rng.uniform(-1, 1, (6, 50021, 2)).astype(np.float32)
    dout = rng.standard_normal((n, 12)).astype(np.float32)
    run_fwd_parity(enc, xyz, t, table, flags=SC, primes=primes, what="hashed everywhere, custom primes, T = 50021")
    run_bwd_parity(enc, xyz, t, dout, flags=SC | ZG, primes=primes, what="hashed everywhere, custom primes, T = 50021")
    ocfg, gcfg = both_configs(enc, DC | SC | ZG)
    pd = dev(packed)
    out = dh.dash_hash4d_fwd(gcfg, pd, pd.view(-1)[3:], dev(table), t_stride=4, N=n)
    assert torch.equal(out, dh.dash_hash4d_fwd(dh.with_flags(gcfg, DC), dev(xyz), dev(t), dev(table)))
    dt = torch.full((6, 50021, 2), 7.0, device="cuda")
    dh.dash_hash4d_bwd(gcfg, pd, pd.view(-1)[3:], dev(dout), dt, t_stride=4, N=n)
    ref, mag, hits = oracle.oracle_bwd(ocfg, n, xyz, t, dout, want_abs=True, want_hits=True)
    check_close(dt.cpu().numpy(), ref, mag, RTOL_FP32, 6, hits=hits, what="packed rows")
    # one level only
    enc1 = EncoderParams(1, 4, 1 << 12, 16, 16, 8, 8)
    run_bwd_parity(enc1, xyz, t, rng.standard_normal((n, 4)).astype(np.float32), flags=DC | SC | ZG, what="L = 1")
    run_fwd_parity(enc1, xyz, t, rng.uniform(-1, 1, (1, 1 << 12, 4)).astype(np.float32), flags=DC | SC, what="L = 1")
    # VALIDATE_INPUTS: the scan uses the workspace header, the sort the bytes behind it
    vcfg = dh.config_from_params(enc, flags=DC | SC | ZG | dh.FLAG_VALIDATE_INPUTS)
    dh.dash_hash4d_bwd(vcfg, dev(xyz), dev(t), dev(dout), dt)
    check_close(dt.cpu().numpy(), ref, mag, RTOL_FP32, 6, hits=hits, what="validate + sort")
    bad = xyz.copy(); bad[5, 0] = np.nan
    with pytest.raises(dh.Hash4DError):
        dh.dash_hash4d_bwd(vcfg, dev(bad), dev(t), dev(dout), dt)


def test_bwd_input_walks_the_sorted_order(set_debug):
    """dash_hash4d_bwd_input / dash_hash3d_bwd_input under SORT_COARSE: the forward's gathers in the forward's order; the
    coordinate gradient of every query is unchanged (compared with the oracle and, bitwise, with the plain call)."""
    set_debug(dh.DEBUG_BWD_COARSE_LEVELS, 3)
    rng = np.random.default_rng(8)
    n = 3001
    enc = EncoderParams(6, 2, 1 << 12, 8, 256, 4, 32)
    xyz, t = make_queries_uniform(8, n)
    table = rng.uniform(-1, 1, (6, 1 << 12, 2)).astype(np.float32)
    dout = rng.standard_normal((n, 12)).astype(np.float32)
    run_bwd_input_parity(enc, xyz, t, table, dout, flags=DC | SC, what="sort_coarse")
    index = rng.integers(0, n, 2 * n).astype(np.int32)
    t2 = rng.random(2 * n, dtype=np.float32)
    d2 = rng.standard_normal((2 * n, 12)).astype(np.float32)
    run_bwd_input_parity(enc, xyz, t2, table, d2, index=index, flags=DC | SC, what="sort_coarse, indexed")
    gs, gp = dh.config_from_params(enc, flags=DC | SC), dh.config_from_params(enc, flags=DC)
    a = dh.dash_hash4d_bwd_input(gs, dev(xyz), dev(t), dev(table), dev(dout))
    b = dh.dash_hash4d_bwd_input(gp, dev(xyz), dev(t), dev(table), dev(dout))
    assert torch.equal(a, b)
    # the order of the step's forward serves it
    ws = torch.empty(dh.dash_hash4d_workspace_bytes(gs, n, dh.OP_FWD), dtype=torch.uint8, device="cuda")
    dh.dash_hash4d_fwd(gs, dev(xyz), dev(t), dev(table), workspace=ws)
    c = dh.dash_hash4d_bwd_input(dh.with_flags(gs, DC | SC | READY), dev(xyz), dev(t), dev(table), dev(dout), workspace=ws)
    assert torch.equal(c, b)
    g3s = dh.make_config(6, 2, 1 << 12, 8, 256, 1, 1, flags=DC | SC)
    g3p = dh.make_config(6, 2, 1 << 12, 8, 256, 1, 1, flags=DC)
    assert torch.equal(dh.dash_hash3d_bwd_input(g3s, dev(xyz), dev(table), dev(dout)),
                       dh.dash_hash3d_bwd_input(g3p, dev(xyz), dev(table), dev(dout)))


def test_the_order_in_the_workspace_is_a_permutation_sorted_by_the_morton_key_of_the_cell(set_debug):
    """What the speed of the path rests on (never its results): after a call with SORT_COARSE the workspace holds, behind
    its 128-byte header, `order` [N] int32 — a permutation of the queries along which the Morton code of the 4D cell on the
    key level (the last coarse level) never decreases — then the keys, then `sorted_q` [N] float4 = the coordinates of
    query order[i].  The key is rebuilt here with numpy: one binary32 product and a floor per axis (the library's own cell
    location), bit b of x, y, z (while b < bits_s) and of t (while b < bits_t) interleaved from bit 0 up."""
    levels = 3
    set_debug(dh.DEBUG_BWD_COARSE_LEVELS, levels)
    enc = EncoderParams(6, 2, 1 << 12, 8, 256, 4, 32)
    rng = np.random.default_rng(17)
    rows = 3000
    xyz = np.clip(0.5 + 0.25 * rng.standard_normal((rows, 3)), 0, 0.999).astype(np.float32)
    index = rng.integers(0, rows, 5003).astype(np.int32)
    n = len(index)
    t = rng.random(n, dtype=np.float32)
    cfg = dh.config_from_params(enc, flags=DC | SC)
    ws = torch.zeros(dh.dash_hash4d_workspace_bytes(cfg, n, dh.OP_FWD), dtype=torch.uint8, device="cuda")
    table = dev(rng.uniform(-1, 1, (6, 1 << 12, 2)).astype(np.float32))
    dh.dash_hash4d_fwd(cfg, dev(xyz), dev(t), table, index=dev(index), workspace=ws)
    torch.cuda.synchronize()
    raw = ws.cpu().numpy()
    r16 = lambda v: (v + 15) // 16 * 16
    order = raw[128:128 + 4 * n].view(np.int32)
    sq_at = 128 + 2 * r16(4 * n)
    sorted_q = raw[sq_at:sq_at + 16 * n].view(np.float32).reshape(n, 4)
    assert np.array_equal(np.sort(order), np.arange(n))
    pts = np.concatenate([xyz[index], t[:, None]], axis=1)
    assert np.array_equal(sorted_q, pts[order])
    res_s, res_t, _ = dh.dash_hash4d_resolutions(cfg)
    ns, nt = res_s[levels - 1], res_t[levels - 1]
    bits_s, bits_t = int(np.ceil(np.log2(ns))), int(np.ceil(np.log2(nt)))
    assert 3 * bits_s + bits_t <= 22 and max(bits_s, bits_t) <= 7      # no coarsening of the key at this size
    cell = np.empty((n, 4), np.uint64)
    for d in range(4):
        cell[:, d] = np.floor(pts[:, d] * np.float32(nt if d == 3 else ns)).astype(np.uint64)
    key = np.zeros(n, np.uint64)
    pos = 0
    for b in range(8):
        if b < bits_s:
            for d in range(3):
                key |= ((cell[:, d] >> np.uint64(b)) & np.uint64(1)) << np.uint64(pos + d)
            pos += 3
        if b < bits_t:
            key |= ((cell[:, 3] >> np.uint64(b)) & np.uint64(1)) << np.uint64(pos)
            pos += 1
    assert (np.diff(key[order].astype(np.int64)) >= 0).all()
    assert len(np.unique(key)) > 50                                      # the check is not vacuous


def test_host_step_runs_the_default_path_with_one_workspace():
    """HostStep (the host-buffer call bench.py's e2e leg times) runs the same launches as the device-resident step: one
    workspace owned by the object, the forward sorts into it, the backward reuses the order (ORDER_READY) and does not
    sort a second time.  C4's encoder at N = 2^19 (N F = 2^21) takes the sorted path by the library's own rule.  The
    results are those of the direct device calls: forward bitwise, gradient sums in another order."""
    wl = make_workload("C4", n_override=1 << 19)
    enc, N = wl.spec.enc, wl.N
    cfg = dh.config_from_params(enc, flags=DC | ZG | SC)
    need = dh.dash_hash4d_workspace_bytes(cfg, N, dh.OP_BWD)
    assert need > 0, "the workload must take the sorted path"
    xd, td, tab, dd = dev(wl.xyz), dev(wl.t), dev(wl.table), dev(wl.dout)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    out_d = torch.empty((N, enc.L * enc.F), device="cuda")
    dt_d = torch.full((enc.L, enc.T, enc.F), 7.0, device="cuda")
    dh.dash_hash4d_launch_count(reset=True)
    dh.dash_hash4d_fwd(cfg, xd, td, tab, out=out_d, workspace=ws)
    dh.dash_hash4d_bwd(dh.with_flags(cfg, DC | ZG | SC | READY), xd, td, dd, dt_d, workspace=ws)
    device_step_launches = dh.dash_hash4d_launch_count(reset=True)
    scratch = torch.empty_like(dt_d)
    dh.dash_hash4d_bwd(cfg, xd, td, dd, scratch, workspace=ws)         # a backward that sorts again: more launches
    bwd_resorting = dh.dash_hash4d_launch_count(reset=True)
    dh.dash_hash4d_bwd(dh.with_flags(cfg, DC | ZG | SC | READY), xd, td, dd, scratch, workspace=ws)
    assert bwd_resorting > dh.dash_hash4d_launch_count(reset=True), "ORDER_READY must save the sort's launches"
    torch.cuda.synchronize()

    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    out_h = torch.empty((N, enc.L * enc.F)).pin_memory()
    dt_h = torch.empty((enc.L, enc.T, enc.F)).pin_memory()
    step = dh.HostStep(cfg)
    xyz_h, t_h, dout_h = pin(wl.xyz), pin(wl.t), pin(wl.dout)
    for it in range(2):                                                 # the second step reuses buffers and workspace
        out_h.fill_(-1); dt_h.fill_(-1)
        dh.dash_hash4d_launch_count(reset=True)
        step(xyz_h, t_h, tab, dout_h, out_h, dt_h)
        assert dh.dash_hash4d_launch_count(reset=True) == device_step_launches
        torch.cuda.synchronize()
        assert torch.equal(out_h, out_d.cpu())
        np.testing.assert_allclose(dt_h.numpy(), dt_d.cpu().numpy(), rtol=1e-4, atol=1e-5)
        ws_ptr = step.buf["workspace"].data_ptr()
        if it:
            assert ws_ptr == first_ptr, "the workspace is allocated once"
        first_ptr = ws_ptr


def test_order_ready_claim_is_checked_under_validate_inputs():
    """ORDER_READY is a promise about the workspace.  The sort stamps what it sorted (N, strides, key, the query pointers);
    with VALIDATE_INPUTS (which synchronises anyway) a call that claims ORDER_READY for other queries, or on a workspace no
    sort has written, is refused with INVALID_ARG instead of silently computing with a foreign order."""
    wl = make_workload("C4", n_override=(1 << 19) + 64)   # N - 1 still takes the sorted path (N F >= 2^21)
    enc, N = wl.spec.enc, wl.N
    V = dh.FLAG_VALIDATE_INPUTS
    cfg = dh.config_from_params(enc, flags=DC | ZG | SC)
    ready = dh.with_flags(cfg, DC | ZG | SC | READY | V)
    need = dh.dash_hash4d_workspace_bytes(ready, N, dh.OP_BWD)
    assert need > 0
    xd, td, tab, dd = dev(wl.xyz), dev(wl.t), dev(wl.table), dev(wl.dout)
    dt = torch.empty((enc.L, enc.T, enc.F), device="cuda")
    fresh = torch.zeros(need, dtype=torch.uint8, device="cuda")
    with pytest.raises(dh.Hash4DError) as e:                            # nothing has sorted into this workspace
        dh.dash_hash4d_bwd(ready, xd, td, dd, dt, workspace=fresh)
    assert e.value.status == 1 and "ORDER_READY" in str(e.value)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    out = dh.dash_hash4d_fwd(cfg, xd, td, tab, workspace=ws)            # sorts and stamps
    dh.dash_hash4d_bwd(ready, xd, td, dd, dt, workspace=ws)             # the honest claim passes, validation included
    want = dh.dash_hash4d_bwd(dh.with_flags(cfg, DC | ZG | SC | READY), xd, td, dd, torch.empty_like(dt), workspace=ws)
    torch.cuda.synchronize()
    np.testing.assert_allclose(dt.cpu().numpy(), want.cpu().numpy(), rtol=1e-4, atol=1e-5)
    assert torch.equal(dh.dash_hash4d_fwd(ready, xd, td, tab, workspace=ws), out)
    with pytest.raises(dh.Hash4DError) as e:                            # fewer queries than the order was built for
        dh.dash_hash4d_bwd(ready, xd, td, dd, dt, N=N - 1, workspace=ws)
    assert e.value.status == 1 and "different N" in str(e.value)
    with pytest.raises(dh.Hash4DError) as e:                            # other coordinates (a copy at another address)
        dh.dash_hash4d_bwd(ready, xd.clone(), td, dd, dt, workspace=ws)
    assert e.value.status == 1 and "pointer" in str(e.value)
    with pytest.raises(dh.Hash4DError):                                 # an index list appears
        dh.dash_hash4d_bwd_input(ready, xd, td, tab, dd, index=torch.arange(N, dtype=torch.int32, device="cuda"),
                                 workspace=ws)
    dh.dash_hash4d_bwd(ready, xd, td, dd, dt, workspace=ws)             # the refused calls left the stamp intact
