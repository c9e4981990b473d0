"""ctypes front of the CPU oracle (oracle/dash_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_2507_19141_b200 and shares no code with the CUDA path.

All arrays are host numpy arrays.  Function names mirror the C ABI of the product
(include/dash_hash4d.h) with the prefix `oracle_`; semantics: DESIGN.md §2-§3.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np

from . import build as _build

FLAG_DENSE_COARSE = 1


class OracleConfig(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("L", C.c_uint32), ("F", C.c_uint32), ("T", C.c_uint32),
                ("res_s_min", C.c_uint32), ("res_s_max", C.c_uint32),
                ("res_t_min", C.c_uint32), ("res_t_max", C.c_uint32),
                ("primes", C.c_uint32 * 4), ("table_dtype", C.c_uint32), ("flags", C.c_uint32)]


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.dash_oracle_threads.restype = C.c_int
    return _lib


def make_config(L, F, T, res_s_min, res_s_max, res_t_min, res_t_max, table_dtype="fp32",
                primes=(0, 0, 0, 0), dense_coarse=True) -> OracleConfig:
    c = OracleConfig()
    c.struct_size = C.sizeof(OracleConfig)
    c.L, c.F, c.T = L, F, T
    c.res_s_min, c.res_s_max, c.res_t_min, c.res_t_max = res_s_min, res_s_max, res_t_min, res_t_max
    c.primes = (C.c_uint32 * 4)(*primes)
    c.table_dtype = {"fp32": 0, "fp16": 1}[table_dtype]
    c.flags = FLAG_DENSE_COARSE if dense_coarse else 0
    return c


def config_from_params(enc, **kw) -> OracleConfig:
    """enc: dash_inputs.EncoderParams (plain numbers only)."""
    return make_config(enc.L, enc.F, enc.T, enc.res_s_min, enc.res_s_max, enc.res_t_min,
                       enc.res_t_max, enc.table_dtype, **kw)


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError(f"{what} failed with oracle status {rc}")


def _query_args(xyz, t, index, t_stride):
    assert xyz.dtype == np.float32 and xyz.ndim == 2 and xyz.shape[1] in (3, 4) and xyz.flags.c_contiguous
    assert t.dtype == np.float32 and t.flags.c_contiguous
    if index is not None:
        assert index.dtype == np.int32 and index.flags.c_contiguous
    return C.c_uint32(xyz.shape[1]), C.c_uint32(t_stride)


def threads() -> int:
    return int(lib().dash_oracle_threads())


def set_threads(n: int) -> None:
    lib().dash_oracle_set_threads(C.c_int(n))


def oracle_resolutions(cfg: OracleConfig):
    L = cfg.L
    rs, rt, dn = np.zeros(L, np.uint32), np.zeros(L, np.uint32), np.zeros(L, np.uint8)
    _check(lib().dash_oracle_resolutions(C.byref(cfg), _p(rs), _p(rt), _p(dn)), "resolutions")
    return rs, rt, dn.astype(bool)


def oracle_indices(cfg, N, xyz, t, index=None, t_stride=1, want_weights=True):
    xs, ts = _query_args(xyz, t, index, t_stride)
    idx = np.zeros((N, cfg.L, 16), np.uint32)
    w = np.zeros((N, cfg.L, 16), np.float64) if want_weights else None
    _check(lib().dash_oracle_indices(C.byref(cfg), C.c_uint64(N), _p(xyz), xs, _p(t), ts, _p(index),
                                     _p(idx), _p(w)), "indices")
    return idx, w


def oracle_fwd(cfg, N, xyz, t, table, index=None, t_stride=1, want_abs=False):
    xs, ts = _query_args(xyz, t, index, t_stride)
    want = np.float16 if cfg.table_dtype == 1 else np.float32
    assert table.dtype == want and table.flags.c_contiguous and table.size == cfg.L * cfg.T * cfg.F
    out = np.zeros((N, cfg.L * cfg.F), np.float32)
    mag = np.zeros((N, cfg.L * cfg.F), np.float64) if want_abs else None
    _check(lib().dash_oracle_fwd(C.byref(cfg), C.c_uint64(N), _p(xyz), xs, _p(t), ts, _p(index),
                                 _p(table), _p(out), _p(mag)), "fwd")
    return (out, mag) if want_abs else out


def oracle_bwd(cfg, N, xyz, t, dout, index=None, t_stride=1, dtable=None, want_abs=False,
               want_hits=False):
    """Returns dtable [L][T][F] fp32 (accumulated into `dtable` if given), and optionally
    sum|W*dY| per entry (double) and contributions per slot (uint32)."""
    xs, ts = _query_args(xyz, t, index, t_stride)
    assert dout.dtype == np.float32 and dout.flags.c_contiguous and dout.size == N * cfg.L * cfg.F
    if dtable is None:
        dtable = np.zeros((cfg.L, cfg.T, cfg.F), np.float32)
    assert dtable.dtype == np.float32 and dtable.flags.c_contiguous
    mag = np.zeros((cfg.L, cfg.T, cfg.F), np.float64) if want_abs else None
    hits = np.zeros((cfg.L, cfg.T), np.uint32) if want_hits else None
    _check(lib().dash_oracle_bwd(C.byref(cfg), C.c_uint64(N), _p(xyz), xs, _p(t), ts, _p(index),
                                 _p(dout), _p(dtable), _p(mag), _p(hits)), "bwd")
    res = [dtable]
    if want_abs:
        res.append(mag)
    if want_hits:
        res.append(hits)
    return res[0] if len(res) == 1 else tuple(res)


# ---- debug exports used only by the pin tests ----

def oracle_vertex_slot(cfg, level: int, g) -> int:
    garr = (C.c_uint32 * 4)(*[int(v) for v in g])
    out = C.c_uint32(0)
    _check(lib().dash_oracle_vertex_slot(C.byref(cfg), C.c_uint32(level), garr, C.byref(out)), "vertex_slot")
    return int(out.value)


def oracle_locate(x: float, n: int):
    cell, frac = C.c_uint32(0), C.c_float(0)
    lib().dash_oracle_locate(C.c_float(x), C.c_uint32(n), C.byref(cell), C.byref(frac))
    return int(cell.value), float(frac.value)


def oracle_half_to_double(h: int) -> float:
    f = lib().dash_oracle_half_to_double
    f.restype = C.c_double
    return float(f(C.c_uint16(h)))


def oracle_bwd_input(cfg, N, xyz, t, table, dout, index=None, t_stride=1, want_abs=False):
    """dq[n] = d<dout[n], G_4D(x_n)>/d(x,y,z,t): [N][4] fp32 (Q14/Q24)."""
    xs, ts = _query_args(xyz, t, index, t_stride)
    dq = np.zeros((N, 4), np.float32)
    mag = np.zeros((N, 4), np.float64) if want_abs else None
    _check(lib().dash_oracle_bwd_input(C.byref(cfg), C.c_uint64(N), _p(xyz), xs, _p(t), ts, _p(index),
                                       _p(table), _p(dout), _p(dq), _p(mag)), "bwd_input")
    return (dq, mag) if want_abs else dq


def oracle_smooth(cfg, N, xyz, t, eps, table, grad_scale=1.0, index=None, t_stride=1, dtable=None,
                  want_grad=True, want_abs=False):
    """Eq. 11: loss[n] = ||G(x_n) - G(x_n + eps_n)||^2 and, if want_grad, dtable +=
    grad_scale * d(sum_n loss[n])/d table.  eps: [N][4] or [1][4]/[4] (one perturbation for all).
    -> (loss, dtable[, loss_abs, feat_abs, grad_abs])."""
    xs, ts = _query_args(xyz, t, index, t_stride)
    eps = np.ascontiguousarray(eps, np.float32)
    eps_stride = 0 if eps.size == 4 else 4
    assert eps_stride == 0 or eps.size == 4 * N
    loss = np.zeros(N, np.float32)
    if want_grad and dtable is None:
        dtable = np.zeros((cfg.L, cfg.T, cfg.F), np.float32)
    la = np.zeros(N, np.float64) if want_abs else None
    fa = np.zeros(N, np.float64) if want_abs else None
    ga = np.zeros((cfg.L, cfg.T, cfg.F), np.float64) if (want_abs and want_grad) else None
    _check(lib().dash_oracle_smooth(C.byref(cfg), C.c_uint64(N), _p(xyz), xs, _p(t), ts, _p(index), _p(eps),
                                    C.c_uint32(eps_stride), _p(table), C.c_double(grad_scale), _p(loss),
                                    _p(dtable if want_grad else None), _p(la), _p(fa), _p(ga)), "smooth")
    return (loss, dtable, la, fa, ga) if want_abs else (loss, dtable)


# ---- G_3D (Eq. 3; Q26) ----

def _point_args(xyz, index):
    assert xyz.dtype == np.float32 and xyz.ndim == 2 and xyz.shape[1] in (3, 4) and xyz.flags.c_contiguous
    if index is not None:
        assert index.dtype == np.int32 and index.flags.c_contiguous
    return C.c_uint32(xyz.shape[1])


def oracle3d_resolutions(cfg: OracleConfig):
    rs, dn = np.zeros(cfg.L, np.uint32), np.zeros(cfg.L, np.uint8)
    _check(lib().dash_oracle3d_resolutions(C.byref(cfg), _p(rs), _p(dn)), "3d resolutions")
    return rs, dn.astype(bool)


def oracle3d_indices(cfg, N, xyz, index=None, want_weights=True):
    xs = _point_args(xyz, index)
    idx = np.zeros((N, cfg.L, 8), np.uint32)
    w = np.zeros((N, cfg.L, 8), np.float64) if want_weights else None
    _check(lib().dash_oracle3d_indices(C.byref(cfg), C.c_uint64(N), _p(xyz), xs, _p(index), _p(idx), _p(w)),
           "3d indices")
    return idx, w


def oracle3d_fwd(cfg, N, xyz, table, index=None, want_abs=False):
    xs = _point_args(xyz, index)
    want = np.float16 if cfg.table_dtype == 1 else np.float32
    assert table.dtype == want and table.flags.c_contiguous and table.size == cfg.L * cfg.T * cfg.F
    out = np.zeros((N, cfg.L * cfg.F), np.float32)
    mag = np.zeros((N, cfg.L * cfg.F), np.float64) if want_abs else None
    _check(lib().dash_oracle3d_fwd(C.byref(cfg), C.c_uint64(N), _p(xyz), xs, _p(index), _p(table), _p(out),
                                   _p(mag)), "3d fwd")
    return (out, mag) if want_abs else out


def oracle3d_bwd(cfg, N, xyz, dout, index=None, dtable=None, want_abs=False, want_hits=False):
    xs = _point_args(xyz, index)
    assert dout.dtype == np.float32 and dout.flags.c_contiguous and dout.size == N * cfg.L * cfg.F
    if dtable is None:
        dtable = np.zeros((cfg.L, cfg.T, cfg.F), np.float32)
    assert dtable.dtype == np.float32 and dtable.flags.c_contiguous
    mag = np.zeros((cfg.L, cfg.T, cfg.F), np.float64) if want_abs else None
    hits = np.zeros((cfg.L, cfg.T), np.uint32) if want_hits else None
    _check(lib().dash_oracle3d_bwd(C.byref(cfg), C.c_uint64(N), _p(xyz), xs, _p(index), _p(dout), _p(dtable),
                                   _p(mag), _p(hits)), "3d bwd")
    res = [dtable]
    if want_abs:
        res.append(mag)
    if want_hits:
        res.append(hits)
    return res[0] if len(res) == 1 else tuple(res)


def oracle3d_bwd_input(cfg, N, xyz, table, dout, index=None, want_abs=False):
    """dq[n] = d<dout[n], G_3D(p_n)>/d(x,y,z): [N][3] fp32 (DESIGN.md §9 item 2)."""
    xs = _point_args(xyz, index)
    dq = np.zeros((N, 3), np.float32)
    mag = np.zeros((N, 3), np.float64) if want_abs else None
    _check(lib().dash_oracle3d_bwd_input(C.byref(cfg), C.c_uint64(N), _p(xyz), xs, _p(index), _p(table), _p(dout),
                                         _p(dq), _p(mag)), "3d bwd_input")
    return (dq, mag) if want_abs else dq


# ---- phi_d + multi-head deformation decoder (Eq. 9-10; Q27) ----

MLP_QUANT_BF16 = 1


class OracleMlpConfig(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_layers", C.c_uint32), ("width", C.c_uint32 * 5),
                ("flags", C.c_uint32)]


def make_mlp_config(widths, quant_bf16=False) -> OracleMlpConfig:
    """widths = [inputs, out_1, ..., out_n], 1 <= n <= 4."""
    assert 2 <= len(widths) <= 5
    m = OracleMlpConfig()
    m.struct_size = C.sizeof(OracleMlpConfig)
    m.n_layers = len(widths) - 1
    m.width = (C.c_uint32 * 5)(*(list(widths) + [0] * (5 - len(widths))))
    m.flags = MLP_QUANT_BF16 if quant_bf16 else 0
    return m


def mlp_param_count(widths) -> int:
    return sum(widths[l] * widths[l - 1] + widths[l] for l in range(1, len(widths)))


def oracle_to_bf16(v: float) -> float:
    f = lib().dash_oracle_to_bf16
    f.restype = C.c_double
    return float(f(C.c_double(v)))


def oracle_mlp(mcfg: OracleMlpConfig, feat, params, base=None, want_abs=False):
    """out = base + MLP(feat): [N][width_n] fp32 (+ the propagated magnitude bound, double)."""
    widths = list(mcfg.width)[:mcfg.n_layers + 1]
    assert feat.dtype == np.float32 and feat.flags.c_contiguous and feat.ndim == 2 and feat.shape[1] == widths[0]
    assert params.dtype == np.float32 and params.flags.c_contiguous and params.size == mlp_param_count(widths)
    N = feat.shape[0]
    if base is not None:
        assert base.dtype == np.float32 and base.flags.c_contiguous and base.shape == (N, widths[-1])
    out = np.zeros((N, widths[-1]), np.float32)
    mag = np.zeros((N, widths[-1]), np.float64) if want_abs else None
    _check(lib().dash_oracle_mlp(C.byref(mcfg), C.c_uint64(N), _p(feat), _p(params), _p(base), _p(out), _p(mag)),
           "mlp")
    return (out, mag) if want_abs else out


def oracle_mlp_bwd(mcfg: OracleMlpConfig, feat, params, dout, want_dfeat=True, want_abs=False):
    """Backward of oracle_mlp by the chain rule (forward recomputed): -> (dfeat [N][width_0] fp32 or None,
    dparams [P] float64, packed like params[, dfeat_abs, dparams_abs, margin])."""
    widths = list(mcfg.width)[:mcfg.n_layers + 1]
    assert feat.dtype == np.float32 and feat.flags.c_contiguous and feat.ndim == 2 and feat.shape[1] == widths[0]
    assert params.dtype == np.float32 and params.flags.c_contiguous and params.size == mlp_param_count(widths)
    N = feat.shape[0]
    assert dout.dtype == np.float32 and dout.flags.c_contiguous and dout.shape == (N, widths[-1])
    dfeat = np.zeros((N, widths[0]), np.float32) if want_dfeat else None
    dparams = np.zeros(params.size, np.float64)
    fa = np.zeros((N, widths[0]), np.float64) if want_abs else None
    pa = np.zeros(params.size, np.float64) if want_abs else None
    mg = np.zeros(N, np.float64) if want_abs else None
    _check(lib().dash_oracle_mlp_bwd(C.byref(mcfg), C.c_uint64(N), _p(feat), _p(params), _p(dout), _p(dfeat),
                                     _p(dparams), _p(fa), _p(pa), _p(mg)), "mlp_bwd")
    return (dfeat, dparams, fa, pa, mg) if want_abs else (dfeat, dparams)


def oracle_deform(cfg, mcfg, N, xyz, t, table, params, base=None, index=None, t_stride=1, want_abs=False):
    """Eq. 9-10: out = base + MLP(G_4D(x)); the features are the fp32 outputs of oracle_fwd."""
    feat = oracle_fwd(cfg, N, xyz, t, table, index=index, t_stride=t_stride)
    return oracle_mlp(mcfg, feat, params, base=base, want_abs=want_abs)


# ---- self-supervised decomposition (Eq. 5; Q31) ----

def oracle_decompose(dp, k_percent, grad_scale=1.0, want_grad=True):
    """dp [N][3] fp32 -> dict(mag [N] fp32, tau fp32, index (ascending int32 list of the dynamic Gaussians), loss (L_s,
    float), ddp [N][3] fp32 or None)."""
    assert dp.dtype == np.float32 and dp.flags.c_contiguous and dp.ndim == 2 and dp.shape[1] == 3
    N = dp.shape[0]
    mag = np.zeros(N, np.float32)
    idx = np.zeros(max(N, 1), np.int32)
    tau, nd, loss = C.c_float(0), C.c_uint64(0), C.c_double(0)
    ddp = np.zeros((N, 3), np.float32) if want_grad else None
    _check(lib().dash_oracle_decompose(C.c_uint64(N), _p(dp), C.c_double(k_percent), C.c_double(grad_scale), _p(mag),
                                       C.byref(tau), _p(idx), C.byref(nd), C.byref(loss), _p(ddp)), "decompose")
    return {"mag": mag, "tau": float(tau.value), "index": idx[:nd.value].copy(), "loss": float(loss.value), "ddp": ddp}


# ---- sparse Adam over the touched table entries (Q28) ----

def oracle_double_to_half(d: float) -> int:
    f = lib().dash_oracle_double_to_half
    f.restype = C.c_uint16
    return int(f(C.c_double(d)))


def oracle_adam_step(theta, grad, m, v, lr, beta1, beta2, eps, t, theta16=None, zero_grad=True):
    """In place on fp32 arrays theta, grad, m, v (and uint16-viewed theta16).  -> number of touched entries."""
    for a in (theta, grad, m, v):
        assert a.dtype == np.float32 and a.flags.c_contiguous and a.size == theta.size
    if theta16 is not None:
        assert theta16.dtype == np.float16 and theta16.flags.c_contiguous and theta16.size == theta.size
    touched = C.c_uint64(0)
    _check(lib().dash_oracle_adam_step(C.c_uint64(theta.size), C.c_double(lr), C.c_double(beta1), C.c_double(beta2),
                                       C.c_double(eps), C.c_uint32(t), _p(theta), _p(theta16), _p(grad), _p(m), _p(v),
                                       C.c_int(1 if zero_grad else 0), C.byref(touched)), "adam_step")
    return int(touched.value)
