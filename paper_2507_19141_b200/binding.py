"""ctypes binding of libdash_hash4d.so — same names as include/dash_hash4d.h.

Marshalling only: torch tensors give device pointers and the current CUDA stream; nothing of the
method is computed here.  PyTorch is used for device memory and streams, nothing else.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import torch

from . import build as _build

FLAG_DENSE_COARSE = 1
FLAG_DETERMINISTIC_BWD = 2
FLAG_VALIDATE_INPUTS = 4
FLAG_ZERO_GRAD = 8
FLAG_SORT_COARSE = 16
FLAG_ORDER_READY = 32
OP_FWD, OP_BWD, OP_INDICES, OP_BWD_INPUT, OP_SMOOTH = 0, 1, 2, 3, 4

_STATUS = {1: "INVALID_ARG", 2: "UNSUPPORTED", 3: "WORKSPACE_TOO_SMALL", 4: "CUDA_ERROR"}

EXPORTS = ["dash_hash4d_resolutions", "dash_hash4d_workspace_bytes", "dash_hash3d_workspace_bytes", "dash_hash4d_fwd",
           "dash_hash4d_bwd", "dash_hash4d_bwd_input", "dash_hash4d_smooth", "dash_hash4d_indices", "dash_hash4d_zero", "dash_hash4d_last_error",
           "dash_hash4d_launch_count", "dash_hash4d_set_debug", "dash_hash4d_build_id",
           "dash_hash3d_resolutions", "dash_hash3d_fwd", "dash_hash3d_bwd", "dash_hash3d_indices", "dash_hash3d_bwd_input",
           "dash_hash4d_adam_step", "dash_mlp_param_count", "dash_mlp_fwd", "dash_mlp_bwd", "dash_deform_bwd", "dash_deform_bwd_workspace_bytes", "dash_deform_workspace_bytes", "dash_deform_fwd",
           "dash_hash4d_slice_t", "dash_hash4d_slice_fwd", "dash_deform_slice_fwd",
           "dash_hash4d_sort_workspace_bytes", "dash_hash4d_sort_queries", "dash_hash4d_sort_queries_static",
           "dash_deform_slice_workspace_bytes",
           "dash_decompose_workspace_bytes", "dash_decompose"]


CEIL_EXPORTS = ["dash_ceiling_launch"]   # include/dash_ceilings.h, in libdash_ceilings.so (measurement tools, not the method)


class Hash4DError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"dash_hash4d status {status} ({_STATUS.get(status, '?')}): {message}")
        self.status = status


class Hash4DConfig(C.Structure):
    """Mirror of `struct dash_hash4d_config` (include/dash_hash4d.h)."""
    _fields_ = [("struct_size", C.c_uint32), ("L", C.c_uint32), ("F", C.c_uint32), ("T", C.c_uint32),
                ("res_s_min", C.c_uint32), ("res_s_max", C.c_uint32),
                ("res_t_min", C.c_uint32), ("res_t_max", C.c_uint32),
                ("primes", C.c_uint32 * 4), ("table_dtype", C.c_uint32), ("flags", C.c_uint32)]


class AdamConfig(C.Structure):
    """Mirror of `struct dash_adam_config` (include/dash_hash4d.h)."""
    _fields_ = [("struct_size", C.c_uint32), ("step", C.c_uint32), ("lr", C.c_float), ("beta1", C.c_float),
                ("beta2", C.c_float), ("eps", C.c_float), ("flags", C.c_uint32)]


ADAM_ZERO_GRAD = 1


class MlpConfig(C.Structure):
    """Mirror of `struct dash_mlp_config` (include/dash_deform.h)."""
    _fields_ = [("struct_size", C.c_uint32), ("n_layers", C.c_uint32), ("width", C.c_uint32 * 5),
                ("flags", C.c_uint32)]


class CeilingParams(C.Structure):
    """Mirror of `struct dash_ceiling_params` (include/dash_ceilings.h)."""
    _fields_ = [("struct_size", C.c_uint32), ("kind", C.c_uint32), ("width", C.c_uint32), ("pattern", C.c_uint32),
                ("footprint_bytes", C.c_uint64), ("grid", C.c_uint32), ("block", C.c_uint32),
                ("dyn_smem", C.c_uint32), ("iters", C.c_uint32), ("seed", C.c_uint32), ("reserved", C.c_uint32)]


class DecomposeResult(C.Structure):
    """Mirror of `struct dash_decompose_result` (include/dash_decompose.h)."""
    _fields_ = [("n_dynamic", C.c_uint32), ("n_static", C.c_uint32), ("tau", C.c_float), ("loss", C.c_float)]


CEIL_COPY, CEIL_GATHER, CEIL_RED, CEIL_SMEM_ATOMIC, CEIL_TMA_GATHER, CEIL_SMEM_ATOMIC_U64 = range(6)
CEIL_INDEPENDENT, CEIL_PAIR_ALIGNED, CEIL_PAIR_XCORNER = range(3)

_lib: Optional[C.CDLL] = None


def library_path() -> str:
    return _build.LIB


def _load() -> C.CDLL:
    """Load the in-tree library; build it if the sources are newer and nvcc is present.  Fails loudly:
    there is no fallback implementation."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.is_stale():
        # never run old kernels against new sources: a stale library that cannot be rebuilt is an error
        try:
            _build.build()
        except Exception as exc:  # noqa: BLE001
            raise ImportError(f"libdash_hash4d.so is missing or older than its sources and the nvcc build "
                              f"failed: {exc}") from exc
    return _bind(C.CDLL(path))


def _bind(lib: C.CDLL) -> C.CDLL:
    global _lib
    vp, u32, u64, sz = C.c_void_p, C.c_uint32, C.c_uint64, C.c_size_t
    cfgp = C.POINTER(Hash4DConfig)
    lib.dash_hash4d_resolutions.argtypes = [cfgp, vp, vp, vp]
    lib.dash_hash4d_resolutions.restype = C.c_int
    lib.dash_hash4d_workspace_bytes.argtypes = [cfgp, u64, C.c_int]
    lib.dash_hash4d_workspace_bytes.restype = sz
    lib.dash_hash3d_workspace_bytes.argtypes = [cfgp, u64, C.c_int]
    lib.dash_hash3d_workspace_bytes.restype = sz
    lib.dash_hash4d_fwd.argtypes = [cfgp, u64, vp, u32, vp, u32, vp, vp, vp, vp, sz, vp]
    lib.dash_hash4d_fwd.restype = C.c_int
    lib.dash_hash4d_bwd.argtypes = [cfgp, u64, vp, u32, vp, u32, vp, vp, vp, vp, sz, vp]
    lib.dash_hash4d_bwd.restype = C.c_int
    lib.dash_hash4d_bwd_input.argtypes = [cfgp, u64, vp, u32, vp, u32, vp, vp, vp, vp, vp, sz, vp]
    lib.dash_hash4d_bwd_input.restype = C.c_int
    lib.dash_hash4d_smooth.argtypes = [cfgp, u64, vp, u32, vp, u32, vp, vp, u32, vp, C.c_float, vp, vp, vp, sz, vp]
    lib.dash_hash4d_smooth.restype = C.c_int
    lib.dash_hash4d_indices.argtypes = [cfgp, u64, vp, u32, vp, u32, vp, vp, vp, vp]
    lib.dash_hash4d_indices.restype = C.c_int
    lib.dash_hash4d_zero.argtypes = [cfgp, vp, vp]
    lib.dash_hash4d_zero.restype = C.c_int
    lib.dash_hash4d_last_error.argtypes = []
    lib.dash_hash4d_last_error.restype = C.c_char_p
    lib.dash_hash3d_resolutions.argtypes = [cfgp, vp, vp]
    lib.dash_hash3d_resolutions.restype = C.c_int
    lib.dash_hash3d_fwd.argtypes = [cfgp, u64, vp, u32, vp, vp, vp, vp, sz, vp]
    lib.dash_hash3d_fwd.restype = C.c_int
    lib.dash_hash3d_bwd.argtypes = [cfgp, u64, vp, u32, vp, vp, vp, vp, sz, vp]
    lib.dash_hash3d_bwd.restype = C.c_int
    lib.dash_hash3d_bwd_input.argtypes = [cfgp, u64, vp, u32, vp, vp, vp, vp, vp, sz, vp]
    lib.dash_hash3d_bwd_input.restype = C.c_int
    lib.dash_hash3d_indices.argtypes = [cfgp, u64, vp, u32, vp, vp, vp, vp]
    lib.dash_hash3d_indices.restype = C.c_int
    lib.dash_hash4d_adam_step.argtypes = [cfgp, C.POINTER(AdamConfig), vp, vp, vp, vp, vp, vp]
    lib.dash_hash4d_adam_step.restype = C.c_int
    mlpp = C.POINTER(MlpConfig)
    lib.dash_mlp_param_count.argtypes = [mlpp]
    lib.dash_mlp_param_count.restype = sz
    lib.dash_mlp_fwd.argtypes = [mlpp, u64, vp, vp, vp, vp, vp]
    lib.dash_mlp_fwd.restype = C.c_int
    lib.dash_mlp_bwd.argtypes = [mlpp, u64, vp, vp, vp, vp, vp, vp]
    lib.dash_mlp_bwd.restype = C.c_int
    lib.dash_deform_bwd_workspace_bytes.argtypes = [cfgp, mlpp, u64]
    lib.dash_deform_bwd_workspace_bytes.restype = sz
    lib.dash_deform_bwd.argtypes = [cfgp, mlpp, u64, vp, u32, vp, u32, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.dash_deform_bwd.restype = C.c_int
    lib.dash_deform_workspace_bytes.argtypes = [cfgp, mlpp, u64]
    lib.dash_deform_workspace_bytes.restype = sz
    lib.dash_deform_fwd.argtypes = [cfgp, mlpp, u64, vp, u32, vp, u32, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.dash_deform_fwd.restype = C.c_int
    lib.dash_hash4d_slice_t.argtypes = [cfgp, vp, vp, vp, vp]
    lib.dash_hash4d_slice_t.restype = C.c_int
    lib.dash_hash4d_slice_fwd.argtypes = [cfgp, u64, vp, u32, vp, vp, vp, vp]
    lib.dash_hash4d_slice_fwd.restype = C.c_int
    lib.dash_deform_slice_fwd.argtypes = [cfgp, mlpp, u64, vp, u32, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.dash_deform_slice_workspace_bytes.argtypes = [cfgp, mlpp, u64]
    lib.dash_deform_slice_workspace_bytes.restype = sz
    lib.dash_deform_slice_fwd.restype = C.c_int
    lib.dash_hash4d_launch_count.argtypes = [C.c_int]
    lib.dash_hash4d_launch_count.restype = u64
    lib.dash_hash4d_sort_workspace_bytes.argtypes = [u64, u32]
    lib.dash_hash4d_sort_workspace_bytes.restype = sz
    lib.dash_hash4d_sort_queries.argtypes = [u64, vp, u32, vp, u32, vp, vp, sz, vp]
    lib.dash_hash4d_sort_queries.restype = C.c_int
    lib.dash_hash4d_sort_queries_static.argtypes = [u64, vp, u32, vp, u32, vp, vp]
    lib.dash_hash4d_sort_queries_static.restype = C.c_int
    lib.dash_decompose_workspace_bytes.argtypes = [u64]
    lib.dash_decompose_workspace_bytes.restype = sz
    lib.dash_decompose.argtypes = [u64, vp, C.c_double, C.c_float, vp, vp, vp, vp, vp, sz, vp]
    lib.dash_decompose.restype = C.c_int
    lib.dash_hash4d_build_id.argtypes = []
    lib.dash_hash4d_build_id.restype = C.c_char_p
    lib.dash_hash4d_set_debug.argtypes = [C.c_int, C.c_int64]
    lib.dash_hash4d_set_debug.restype = C.c_int
    _lib = lib
    return lib


_ceil_lib: Optional[C.CDLL] = None


def ceilings_library_path() -> str:
    return _build.CEIL_LIB


def _load_ceilings() -> C.CDLL:
    """The microbenchmark library (include/dash_ceilings.h), separate from the product library."""
    global _ceil_lib
    if _ceil_lib is None:
        if _build.ceilings_is_stale():
            try:
                _build.build_ceilings()
            except Exception as exc:  # noqa: BLE001
                raise ImportError(f"libdash_ceilings.so is missing or older than its sources and the nvcc build "
                                  f"failed: {exc}") from exc
        lib = C.CDLL(_build.CEIL_LIB)
        lib.dash_ceiling_launch.argtypes = [C.POINTER(CeilingParams), C.c_void_p, C.c_void_p, C.POINTER(C.c_uint64),
                                            C.c_void_p]
        lib.dash_ceiling_launch.restype = C.c_int
        _ceil_lib = lib
    return _ceil_lib


def exported_symbols() -> list[str]:
    """Names the product headers declare that resolve in the product library."""
    lib = _load()
    return [n for n in EXPORTS if hasattr(lib, n)]


def make_config(L, F, T, res_s_min, res_s_max, res_t_min, res_t_max, table_dtype="fp32",
                primes=(0, 0, 0, 0), flags=FLAG_DENSE_COARSE) -> Hash4DConfig:
    c = Hash4DConfig()
    c.struct_size = C.sizeof(Hash4DConfig)
    c.L, c.F, c.T = L, F, T
    c.res_s_min, c.res_s_max, c.res_t_min, c.res_t_max = res_s_min, res_s_max, res_t_min, res_t_max
    c.primes = (C.c_uint32 * 4)(*primes)
    c.table_dtype = {"fp32": 0, "fp16": 1}[table_dtype]
    c.flags = flags
    return c


def config_from_params(enc, **kw) -> Hash4DConfig:
    """enc: dash_inputs.EncoderParams (plain numbers)."""
    return make_config(enc.L, enc.F, enc.T, enc.res_s_min, enc.res_s_max, enc.res_t_min,
                       enc.res_t_max, enc.table_dtype, **kw)


def with_flags(cfg: Hash4DConfig, flags: int) -> Hash4DConfig:
    c = Hash4DConfig.from_buffer_copy(bytes(cfg))
    c.flags = flags
    return c


def _check(rc: int):
    if rc != 0:
        raise Hash4DError(rc, dash_hash4d_last_error())


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t: Optional[torch.Tensor], dtype, what: str):
    if t is None:
        return
    if not t.is_cuda:
        raise ValueError(f"{what} must be a CUDA tensor (no CPU fallback exists)")
    if t.dtype != dtype or not t.is_contiguous():
        raise ValueError(f"{what} must be contiguous {dtype}")


def _at_least(t: Optional[torch.Tensor], count: int, what: str):
    """The C ABI takes raw pointers and cannot know the allocation sizes: check them here."""
    if t is not None and t.numel() < count:
        raise ValueError(f"{what} holds {t.numel()} elements, the call needs {count}")


def _exactly(t: Optional[torch.Tensor], count: int, what: str):
    """count == 0 means the config itself is invalid: let the C ABI report that with its own status code."""
    if t is not None and count and t.numel() != count:
        raise ValueError(f"{what} holds {t.numel()} elements, the config says {count}")


def _one_device(*tensors):
    devs = {t.device for t in tensors if t is not None}
    if len(devs) > 1:
        raise ValueError(f"all tensors of a call must live on one device, got {sorted(map(str, devs))}")
    dev = next(iter(devs))
    if dev != torch.device("cuda", torch.cuda.current_device()):
        raise ValueError(f"tensors live on {dev} but the current device is cuda:{torch.cuda.current_device()} "
                         "(the call enqueues on the current stream)")


def _check_queries(cfg, xyz, t, index, ts: int, N: int):
    """Sizes of the query arrays for N queries; under VALIDATE_INPUTS also the range of the index list."""
    if N < 0:
        raise ValueError("N < 0")
    if index is not None:
        _at_least(index, N, "index")
        if (cfg.flags & FLAG_VALIDATE_INPUTS) and N:
            lo, hi = int(index[:N].min()), int(index[:N].max())
            if lo < 0 or hi >= xyz.shape[0]:
                raise ValueError(f"index values span [{lo}, {hi}] but xyz has {xyz.shape[0]} rows")
    elif xyz.shape[0] < N:
        raise ValueError(f"xyz has {xyz.shape[0]} rows, the call needs {N}")
    if t is not None and N:
        _at_least(t, (N - 1) * ts + 1, "t")


def _table_elems(cfg) -> int:
    return int(cfg.L) * int(cfg.T) * int(cfg.F)


def _strides(xyz: torch.Tensor, t: torch.Tensor, t_stride: Optional[int]):
    if xyz.dim() != 2 or xyz.shape[1] not in (3, 4):
        raise ValueError("xyz must be [rows][3] or [rows][4]")
    if t_stride is None:
        t_stride = 0 if t.numel() == 1 else 1
    return int(xyz.shape[1]), int(t_stride)


def dash_hash4d_last_error() -> str:
    return _load().dash_hash4d_last_error().decode()


def dash_hash4d_launch_count(reset: bool = False) -> int:
    return int(_load().dash_hash4d_launch_count(1 if reset else 0))


(DEBUG_FWD_GROUP, DEBUG_BWD_GROUP, DEBUG_SMOOTH_GROUP, DEBUG_DEFORM_PATH, DEBUG_BWD_VARIANT,
 DEBUG_BWD_COARSE_LEVELS, DEBUG_BWD_RUN_CHUNK, DEBUG_FWD_ORDERED_LEVELS, DEBUG_SORT_KEY_BITS) = range(9)   # include/dash_debug.h


def dash_hash4d_set_debug(key: int, value: int) -> None:
    """Tuning override for sweeps (include/dash_debug.h `dash_debug_key`); 0 restores the library's choice."""
    _check(_load().dash_hash4d_set_debug(int(key), int(value)))


def dash_hash4d_resolutions(cfg: Hash4DConfig):
    """-> (res_s, res_t, is_dense) as Python lists (host only; needs no GPU)."""
    L = max(int(cfg.L), 1)
    rs, rt, dn = (C.c_uint32 * L)(), (C.c_uint32 * L)(), (C.c_uint8 * L)()
    _check(_load().dash_hash4d_resolutions(C.byref(cfg), rs, rt, dn))
    return list(rs), list(rt), [bool(v) for v in dn]


def dash_hash4d_workspace_bytes(cfg: Hash4DConfig, N: int, op: int) -> int:
    return int(_load().dash_hash4d_workspace_bytes(C.byref(cfg), N, op))


def dash_hash3d_workspace_bytes(cfg: Hash4DConfig, N: int, op: int) -> int:
    return int(_load().dash_hash3d_workspace_bytes(C.byref(cfg), N, op))


def _workspace(cfg, N, op, workspace, device, dims=4):
    need = dash_hash4d_workspace_bytes(cfg, N, op) if dims == 4 else dash_hash3d_workspace_bytes(cfg, N, op)
    if need and workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=device)
    if workspace is not None and not workspace.is_cuda:
        raise ValueError("workspace must be a CUDA tensor")
    return workspace, (0 if workspace is None else workspace.numel() * workspace.element_size())


def dash_hash4d_fwd(cfg, xyz, t, table, out=None, index=None, t_stride=None, N=None, workspace=None):
    """out[n][l*F+f] = sum_k W_k table[l][slot_k][f]; returns `out` ([N][L*F] fp32, CUDA)."""
    _dev(xyz, torch.float32, "xyz"); _dev(t, torch.float32, "t"); _dev(index, torch.int32, "index")
    _dev(table, torch.float16 if cfg.table_dtype == 1 else torch.float32, "table")
    xs, ts = _strides(xyz, t, t_stride)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    if out is None:
        out = torch.empty((N, cfg.L * cfg.F), dtype=torch.float32, device=xyz.device)
    _dev(out, torch.float32, "out")
    _check_queries(cfg, xyz, t, index, ts, N)
    _exactly(table, _table_elems(cfg), "table"); _at_least(out, N * cfg.L * cfg.F, "out")
    _one_device(xyz, t, index, table, out, workspace)
    workspace, wbytes = _workspace(cfg, N, OP_FWD, workspace, xyz.device)
    _check(_load().dash_hash4d_fwd(C.byref(cfg), N, _ptr(xyz), xs, _ptr(t), ts, _ptr(index),
                                   _ptr(table), _ptr(out), _ptr(workspace), wbytes, _stream()))
    return out


def dash_hash4d_bwd(cfg, xyz, t, dout, dtable, index=None, t_stride=None, N=None, workspace=None):
    """dtable[l][slot_k][f] += W_k dout[n][l*F+f]; returns `dtable` ([L][T][F] fp32, CUDA)."""
    _dev(xyz, torch.float32, "xyz"); _dev(t, torch.float32, "t"); _dev(index, torch.int32, "index")
    _dev(dout, torch.float32, "dout"); _dev(dtable, torch.float32, "dtable")
    xs, ts = _strides(xyz, t, t_stride)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    _check_queries(cfg, xyz, t, index, ts, N)
    _at_least(dout, N * cfg.L * cfg.F, "dout"); _exactly(dtable, _table_elems(cfg), "dtable")
    _one_device(xyz, t, index, dout, dtable, workspace)
    workspace, wbytes = _workspace(cfg, N, OP_BWD, workspace, xyz.device)
    _check(_load().dash_hash4d_bwd(C.byref(cfg), N, _ptr(xyz), xs, _ptr(t), ts, _ptr(index),
                                   _ptr(dout), _ptr(dtable), _ptr(workspace), wbytes, _stream()))
    return dtable


def dash_hash4d_bwd_input(cfg, xyz, t, table, dout, dq=None, index=None, t_stride=None, N=None,
                          workspace=None):
    """dq[n] = d<dout[n], G_4D(x_n)>/d(x,y,z,t); returns `dq` ([N][4] fp32, CUDA, overwritten)."""
    _dev(xyz, torch.float32, "xyz"); _dev(t, torch.float32, "t"); _dev(index, torch.int32, "index")
    _dev(table, torch.float16 if cfg.table_dtype == 1 else torch.float32, "table")
    _dev(dout, torch.float32, "dout")
    xs, ts = _strides(xyz, t, t_stride)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    if dq is None:
        dq = torch.empty((N, 4), dtype=torch.float32, device=xyz.device)
    _dev(dq, torch.float32, "dq")
    _check_queries(cfg, xyz, t, index, ts, N)
    _exactly(table, _table_elems(cfg), "table"); _at_least(dout, N * cfg.L * cfg.F, "dout")
    _at_least(dq, 4 * N, "dq"); _one_device(xyz, t, index, table, dout, dq, workspace)
    workspace, wbytes = _workspace(cfg, N, OP_BWD_INPUT, workspace, xyz.device)
    _check(_load().dash_hash4d_bwd_input(C.byref(cfg), N, _ptr(xyz), xs, _ptr(t), ts, _ptr(index),
                                         _ptr(table), _ptr(dout), _ptr(dq), _ptr(workspace), wbytes,
                                         _stream()))
    return dq


def dash_hash4d_smooth(cfg, xyz, t, eps, table, grad_scale=1.0, loss=None, dtable=None, index=None,
                       t_stride=None, N=None, workspace=None):
    """Eq. 11: loss[n] = ||G(x_n) - G(x_n + eps_n)||^2 ([N] fp32, overwritten) and, if `dtable` is given,
    dtable += grad_scale * d(sum loss)/d table.  eps: [N][4] CUDA fp32, or 4 values for all queries."""
    _dev(xyz, torch.float32, "xyz"); _dev(t, torch.float32, "t"); _dev(index, torch.int32, "index")
    _dev(table, torch.float16 if cfg.table_dtype == 1 else torch.float32, "table")
    _dev(eps, torch.float32, "eps"); _dev(dtable, torch.float32, "dtable")
    xs, ts = _strides(xyz, t, t_stride)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    eps_stride = 0 if eps.numel() == 4 else 4
    if eps_stride and eps.numel() != 4 * N:
        raise ValueError("eps must hold 4 values, or 4 per query")
    if loss is None:
        loss = torch.empty((N,), dtype=torch.float32, device=xyz.device)
    _dev(loss, torch.float32, "loss")
    _check_queries(cfg, xyz, t, index, ts, N)
    _exactly(table, _table_elems(cfg), "table"); _exactly(dtable, _table_elems(cfg), "dtable")
    _at_least(loss, N, "loss"); _one_device(xyz, t, index, eps, table, loss, dtable, workspace)
    workspace, wbytes = _workspace(cfg, N, OP_SMOOTH, workspace, xyz.device)
    _check(_load().dash_hash4d_smooth(C.byref(cfg), N, _ptr(xyz), xs, _ptr(t), ts, _ptr(index), _ptr(eps),
                                      eps_stride, _ptr(table), float(grad_scale), _ptr(loss), _ptr(dtable),
                                      _ptr(workspace), wbytes, _stream()))
    return loss, dtable


def dash_hash4d_indices(cfg, xyz, t, index=None, t_stride=None, N=None, want_weights=True):
    """-> (idx [N][L][16] int32-viewed uint32, w [N][L][16] fp32 or None)."""
    _dev(xyz, torch.float32, "xyz"); _dev(t, torch.float32, "t"); _dev(index, torch.int32, "index")
    xs, ts = _strides(xyz, t, t_stride)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    _check_queries(cfg, xyz, t, index, ts, N); _one_device(xyz, t, index)
    idx = torch.empty((N, cfg.L, 16), dtype=torch.int32, device=xyz.device)   # bits are uint32
    w = torch.empty((N, cfg.L, 16), dtype=torch.float32, device=xyz.device) if want_weights else None
    _check(_load().dash_hash4d_indices(C.byref(cfg), N, _ptr(xyz), xs, _ptr(t), ts, _ptr(index),
                                       _ptr(idx), _ptr(w), _stream()))
    return idx, w


def dash_hash4d_zero(cfg, dtable):
    _dev(dtable, torch.float32, "dtable")
    _exactly(dtable, _table_elems(cfg), "dtable"); _one_device(dtable)
    _check(_load().dash_hash4d_zero(C.byref(cfg), _ptr(dtable), _stream()))
    return dtable


def dash_hash4d_sort_queries(xyz, index=None, bits=6, N=None, order=None, workspace=None):
    """-> order [N] int32: query numbers sorted by the Morton code of their coarse spatial cell (2^bits per axis)."""
    _dev(xyz, torch.float32, "xyz"); _dev(index, torch.int32, "index")
    xs = int(xyz.shape[1])
    if xyz.dim() != 2 or xs not in (3, 4):
        raise ValueError("xyz must be [rows][3] or [rows][4]")
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    if index is not None:
        _at_least(index, N, "index")
    elif xyz.shape[0] < N:
        raise ValueError(f"xyz has {xyz.shape[0]} rows, the call needs {N}")
    if order is None:
        order = torch.empty((N,), dtype=torch.int32, device=xyz.device)
    _dev(order, torch.int32, "order"); _at_least(order, N, "order")
    need = int(_load().dash_hash4d_sort_workspace_bytes(N, int(bits)))
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=xyz.device)
    _one_device(xyz, index, order, workspace)
    _check(_load().dash_hash4d_sort_queries(N, _ptr(xyz), xs, _ptr(index), int(bits), _ptr(order), _ptr(workspace),
                                            workspace.numel(), _stream()))
    return order


SORT_STATIC_MAX_N = 1 << 20   # DASH_HASH4D_SORT_STATIC_MAX_N
SORT_STATIC_MAX_BITS = 6       # DASH_HASH4D_SORT_STATIC_MAX_BITS


def dash_hash4d_sort_queries_static(xyz, order, index=None, bits=6, N=None):
    """dash_hash4d_sort_queries without any device allocation, for callers that cannot make one: a plug-in whose host
    application owns the GPU memory pool, a per-frame loop that must not stall the device in cudaMalloc / cudaFree, a
    process whose HBM is already full.  The sort's scratch is a fixed ~5 MB array inside the library (held by every GPU
    that loads it), so N <= SORT_STATIC_MAX_N and bits <= SORT_STATIC_MAX_BITS; beyond that the library refuses
    (Hash4DError, UNSUPPORTED) and dash_hash4d_sort_queries with a workspace is the call to use.  `order` ([N] int32) is
    the caller's buffer and is required: this wrapper, too, creates no tensor.  Calls share the scratch: do not let two of
    them overlap on the GPU.  The first call on a device does a one-time address look-up; make it outside stream capture."""
    _dev(xyz, torch.float32, "xyz"); _dev(index, torch.int32, "index"); _dev(order, torch.int32, "order")
    if order is None:
        raise ValueError("order is required: the no-allocation call writes into the caller's buffer")
    if xyz.dim() != 2 or int(xyz.shape[1]) not in (3, 4):
        raise ValueError("xyz must be [rows][3] or [rows][4]")
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    if index is not None:
        _at_least(index, N, "index")
    elif xyz.shape[0] < N:
        raise ValueError(f"xyz has {xyz.shape[0]} rows, the call needs {N}")
    _at_least(order, N, "order")
    _one_device(xyz, index, order)
    _check(_load().dash_hash4d_sort_queries_static(N, _ptr(xyz), int(xyz.shape[1]), _ptr(index), int(bits),
                                                   _ptr(order), _stream()))
    return order


# ---- G_3D (Eq. 3): the same encoder with d = 3; temporal config fields ignored -------

def _xyz_stride(xyz: torch.Tensor) -> int:
    if xyz.dim() != 2 or xyz.shape[1] not in (3, 4):
        raise ValueError("xyz must be [rows][3] or [rows][4]")
    return int(xyz.shape[1])


def dash_hash3d_resolutions(cfg: Hash4DConfig):
    """-> (res_s, is_dense) as Python lists (host only; needs no GPU)."""
    L = max(int(cfg.L), 1)
    rs, dn = (C.c_uint32 * L)(), (C.c_uint8 * L)()
    _check(_load().dash_hash3d_resolutions(C.byref(cfg), rs, dn))
    return list(rs), [bool(v) for v in dn]


def dash_hash3d_fwd(cfg, xyz, table, out=None, index=None, N=None, workspace=None):
    """out[n][l*F+f] = sum_{k<8} W_k table[l][slot_k][f]; returns `out` ([N][L*F] fp32, CUDA)."""
    _dev(xyz, torch.float32, "xyz"); _dev(index, torch.int32, "index")
    _dev(table, torch.float16 if cfg.table_dtype == 1 else torch.float32, "table")
    xs = _xyz_stride(xyz)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    if out is None:
        out = torch.empty((N, cfg.L * cfg.F), dtype=torch.float32, device=xyz.device)
    _dev(out, torch.float32, "out")
    _check_queries(cfg, xyz, None, index, 0, N)
    _exactly(table, _table_elems(cfg), "table"); _at_least(out, N * cfg.L * cfg.F, "out")
    _one_device(xyz, index, table, out, workspace)
    workspace, wbytes = _workspace(cfg, N, OP_FWD, workspace, xyz.device, dims=3)
    _check(_load().dash_hash3d_fwd(C.byref(cfg), N, _ptr(xyz), xs, _ptr(index), _ptr(table), _ptr(out),
                                   _ptr(workspace), wbytes, _stream()))
    return out


def dash_hash3d_bwd(cfg, xyz, dout, dtable, index=None, N=None, workspace=None):
    """dtable[l][slot_k][f] += W_k dout[n][l*F+f] over the 8 corners; returns `dtable`."""
    _dev(xyz, torch.float32, "xyz"); _dev(index, torch.int32, "index")
    _dev(dout, torch.float32, "dout"); _dev(dtable, torch.float32, "dtable")
    xs = _xyz_stride(xyz)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    _check_queries(cfg, xyz, None, index, 0, N)
    _at_least(dout, N * cfg.L * cfg.F, "dout"); _exactly(dtable, _table_elems(cfg), "dtable")
    _one_device(xyz, index, dout, dtable, workspace)
    workspace, wbytes = _workspace(cfg, N, OP_BWD, workspace, xyz.device, dims=3)
    _check(_load().dash_hash3d_bwd(C.byref(cfg), N, _ptr(xyz), xs, _ptr(index), _ptr(dout), _ptr(dtable),
                                   _ptr(workspace), wbytes, _stream()))
    return dtable


def dash_hash3d_bwd_input(cfg, xyz, table, dout, dq=None, index=None, N=None, workspace=None):
    """dq[n] = d<dout[n], G_3D(p_n)>/d(x,y,z); returns `dq` ([N][3] fp32, CUDA, overwritten)."""
    _dev(xyz, torch.float32, "xyz"); _dev(index, torch.int32, "index"); _dev(dout, torch.float32, "dout")
    _dev(table, torch.float16 if cfg.table_dtype == 1 else torch.float32, "table")
    xs = _xyz_stride(xyz)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    if dq is None:
        dq = torch.empty((N, 3), dtype=torch.float32, device=xyz.device)
    _dev(dq, torch.float32, "dq")
    _check_queries(cfg, xyz, None, index, 0, N)
    _exactly(table, _table_elems(cfg), "table"); _at_least(dout, N * cfg.L * cfg.F, "dout"); _at_least(dq, 3 * N, "dq")
    _one_device(xyz, index, table, dout, dq, workspace)
    workspace, wbytes = _workspace(cfg, N, OP_BWD_INPUT, workspace, xyz.device, dims=3)
    _check(_load().dash_hash3d_bwd_input(C.byref(cfg), N, _ptr(xyz), xs, _ptr(index), _ptr(table), _ptr(dout),
                                         _ptr(dq), _ptr(workspace), wbytes, _stream()))
    return dq


def dash_hash3d_indices(cfg, xyz, index=None, N=None, want_weights=True):
    """-> (idx [N][L][8] int32-viewed uint32, w [N][L][8] fp32 or None)."""
    _dev(xyz, torch.float32, "xyz"); _dev(index, torch.int32, "index")
    xs = _xyz_stride(xyz)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    _check_queries(cfg, xyz, None, index, 0, N); _one_device(xyz, index)
    idx = torch.empty((N, cfg.L, 8), dtype=torch.int32, device=xyz.device)
    w = torch.empty((N, cfg.L, 8), dtype=torch.float32, device=xyz.device) if want_weights else None
    _check(_load().dash_hash3d_indices(C.byref(cfg), N, _ptr(xyz), xs, _ptr(index), _ptr(idx), _ptr(w),
                                       _stream()))
    return idx, w


def dash_hash4d_adam_step(cfg, theta, dtable, m, v, step, lr=1e-2, beta1=0.9, beta2=0.99, eps=1e-15, table16=None,
                          zero_grad=True):
    """Sparse Adam over the entries with a non-zero gradient (in place on theta, m, v[, table16], dtable)."""
    for name, a in (("theta", theta), ("dtable", dtable), ("m", m), ("v", v)):
        _dev(a, torch.float32, name)
    _dev(table16, torch.float16, "table16")
    for name, a in (("theta", theta), ("dtable", dtable), ("m", m), ("v", v), ("table16", table16)):
        _exactly(a, _table_elems(cfg), name)
    _one_device(theta, dtable, m, v, table16)
    opt = AdamConfig()
    opt.struct_size = C.sizeof(AdamConfig)
    opt.step, opt.lr, opt.beta1, opt.beta2, opt.eps = int(step), lr, beta1, beta2, eps
    opt.flags = ADAM_ZERO_GRAD if zero_grad else 0
    _check(_load().dash_hash4d_adam_step(C.byref(cfg), C.byref(opt), _ptr(theta), _ptr(table16), _ptr(dtable),
                                         _ptr(m), _ptr(v), _stream()))
    return theta


# ---- render path: G_4D -> phi_d -> heads (include/dash_deform.h; Eq. 9-10) -------------

def make_mlp_config(widths) -> MlpConfig:
    """widths = [inputs, out_1, ..., out_n], 1 <= n <= 4."""
    if not 2 <= len(widths) <= 5:
        raise ValueError("an MLP chain has 1..4 layers")
    m = MlpConfig()
    m.struct_size = C.sizeof(MlpConfig)
    m.n_layers = len(widths) - 1
    m.width = (C.c_uint32 * 5)(*(list(widths) + [0] * (5 - len(widths))))
    m.flags = 0
    return m


def dash_mlp_param_count(mlp: MlpConfig) -> int:
    return int(_load().dash_mlp_param_count(C.byref(mlp)))


def dash_mlp_fwd(mlp, feat, params, base=None, out=None):
    """out = base + MLP(feat): [N][width_n] fp32 (tcgen05 bf16 x bf16 -> fp32)."""
    _dev(feat, torch.float32, "feat"); _dev(params, torch.float32, "params"); _dev(base, torch.float32, "base")
    N = int(feat.shape[0])
    n_out = int(mlp.width[mlp.n_layers])
    if out is None:
        out = torch.empty((N, n_out), dtype=torch.float32, device=feat.device)
    _dev(out, torch.float32, "out")
    _exactly(feat, N * int(mlp.width[0]), "feat"); _exactly(params, dash_mlp_param_count(mlp), "params")
    _at_least(base, N * n_out, "base"); _at_least(out, N * n_out, "out"); _one_device(feat, params, base, out)
    _check(_load().dash_mlp_fwd(C.byref(mlp), N, _ptr(feat), _ptr(params), _ptr(base), _ptr(out), _stream()))
    return out


def dash_mlp_bwd(mlp, feat, params, dout, dparams, dfeat=None, want_dfeat=True):
    """Backward of dash_mlp_fwd: dparams += dL/d params (packed like params); returns (dfeat or None, dparams)."""
    for name, a in (("feat", feat), ("params", params), ("dout", dout), ("dparams", dparams), ("dfeat", dfeat)):
        _dev(a, torch.float32, name)
    N = int(feat.shape[0])
    n_out = int(mlp.width[mlp.n_layers])
    if want_dfeat and dfeat is None:
        dfeat = torch.empty((N, int(mlp.width[0])), dtype=torch.float32, device=feat.device)
    _exactly(feat, N * int(mlp.width[0]), "feat"); _exactly(params, dash_mlp_param_count(mlp), "params")
    _exactly(dparams, dash_mlp_param_count(mlp), "dparams"); _at_least(dout, N * n_out, "dout")
    _at_least(dfeat, N * int(mlp.width[0]), "dfeat"); _one_device(feat, params, dout, dparams, dfeat)
    _check(_load().dash_mlp_bwd(C.byref(mlp), N, _ptr(feat), _ptr(params), _ptr(dout), _ptr(dfeat), _ptr(dparams),
                                _stream()))
    return dfeat, dparams


def dash_deform_bwd(cfg, mlp, xyz, t, table, params, dout, dtable, dparams, dq=None, index=None, t_stride=None, N=None,
                    workspace=None):
    """Backward of dash_deform_fwd: dtable (+)= table gradient, dparams += MLP parameter gradient, dq (optional,
    [N][4]) = coordinate gradient.  Returns (dtable, dparams, dq)."""
    _dev(xyz, torch.float32, "xyz"); _dev(t, torch.float32, "t"); _dev(index, torch.int32, "index")
    _dev(table, torch.float16 if cfg.table_dtype == 1 else torch.float32, "table")
    for name, a in (("params", params), ("dout", dout), ("dtable", dtable), ("dparams", dparams), ("dq", dq)):
        _dev(a, torch.float32, name)
    xs, ts = _strides(xyz, t, t_stride)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    n_out = int(mlp.width[mlp.n_layers])
    _check_queries(cfg, xyz, t, index, ts, N)
    _exactly(table, _table_elems(cfg), "table"); _exactly(dtable, _table_elems(cfg), "dtable")
    _exactly(params, dash_mlp_param_count(mlp), "params"); _exactly(dparams, dash_mlp_param_count(mlp), "dparams")
    _at_least(dout, N * n_out, "dout"); _at_least(dq, 4 * N, "dq")
    need = int(_load().dash_deform_bwd_workspace_bytes(C.byref(cfg), C.byref(mlp), N))
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=xyz.device)
    _one_device(xyz, t, index, table, params, dout, dtable, dparams, dq, workspace)
    _check(_load().dash_deform_bwd(C.byref(cfg), C.byref(mlp), N, _ptr(xyz), xs, _ptr(t), ts, _ptr(index), _ptr(table),
                                   _ptr(params), _ptr(dout), _ptr(dtable), _ptr(dparams), _ptr(dq), _ptr(workspace),
                                   workspace.numel(), _stream()))
    return dtable, dparams, dq


def dash_deform_workspace_bytes(cfg, mlp, N: int) -> int:
    return int(_load().dash_deform_workspace_bytes(C.byref(cfg), C.byref(mlp), N))


def dash_deform_fwd(cfg, mlp, xyz, t, table, params, base=None, out=None, index=None, t_stride=None, N=None,
                    workspace=None):
    """out[n] = base[n] + MLP(G_4D(x_n)) (Eq. 9-10) in one call; returns `out` ([N][width_n] fp32, CUDA)."""
    _dev(xyz, torch.float32, "xyz"); _dev(t, torch.float32, "t"); _dev(index, torch.int32, "index")
    _dev(table, torch.float16 if cfg.table_dtype == 1 else torch.float32, "table")
    _dev(params, torch.float32, "params"); _dev(base, torch.float32, "base")
    xs, ts = _strides(xyz, t, t_stride)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    n_out = int(mlp.width[mlp.n_layers])
    if out is None:
        out = torch.empty((N, n_out), dtype=torch.float32, device=xyz.device)
    _dev(out, torch.float32, "out")
    _check_queries(cfg, xyz, t, index, ts, N)
    _exactly(table, _table_elems(cfg), "table"); _exactly(params, dash_mlp_param_count(mlp), "params")
    _at_least(base, N * n_out, "base"); _at_least(out, N * n_out, "out")
    _one_device(xyz, t, index, table, params, base, out, workspace)
    need = dash_deform_workspace_bytes(cfg, mlp, N)
    if need and workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=xyz.device)
    wbytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    _check(_load().dash_deform_fwd(C.byref(cfg), C.byref(mlp), N, _ptr(xyz), xs, _ptr(t), ts, _ptr(index),
                                   _ptr(table), _ptr(params), _ptr(base), _ptr(out), _ptr(workspace), wbytes,
                                   _stream()))
    return out


# ---- time slice: the render path at one timestamp (include/dash_deform.h; Q29) -----------------

def dash_hash4d_slice_t(cfg, t, table, slice_out=None):
    """slice[l][u] = blend of the two t-layers of level l at the one timestamp t ([L][T][F] fp32, CUDA)."""
    _dev(t, torch.float32, "t")
    _dev(table, torch.float16 if cfg.table_dtype == 1 else torch.float32, "table")
    if slice_out is None:
        slice_out = torch.empty((cfg.L, cfg.T, cfg.F), dtype=torch.float32, device=table.device)
    _dev(slice_out, torch.float32, "slice")
    _at_least(t, 1, "t"); _exactly(table, _table_elems(cfg), "table"); _exactly(slice_out, _table_elems(cfg), "slice")
    _one_device(t, table, slice_out)
    _check(_load().dash_hash4d_slice_t(C.byref(cfg), _ptr(t), _ptr(table), _ptr(slice_out), _stream()))
    return slice_out


def dash_hash4d_slice_fwd(cfg, xyz, slice_t, out=None, index=None, N=None):
    """G_4D(xyz_n, t) from a slice: 8-corner lookups; returns `out` ([N][L*F] fp32)."""
    _dev(xyz, torch.float32, "xyz"); _dev(index, torch.int32, "index"); _dev(slice_t, torch.float32, "slice")
    xs = _xyz_stride(xyz)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    if out is None:
        out = torch.empty((N, cfg.L * cfg.F), dtype=torch.float32, device=xyz.device)
    _dev(out, torch.float32, "out")
    _check_queries(cfg, xyz, None, index, 0, N)
    _exactly(slice_t, _table_elems(cfg), "slice"); _at_least(out, N * cfg.L * cfg.F, "out")
    _one_device(xyz, index, slice_t, out)
    _check(_load().dash_hash4d_slice_fwd(C.byref(cfg), N, _ptr(xyz), xs, _ptr(index), _ptr(slice_t), _ptr(out),
                                         _stream()))
    return out


def dash_deform_slice_workspace_bytes(cfg, mlp, N: int) -> int:
    return int(_load().dash_deform_slice_workspace_bytes(C.byref(cfg), C.byref(mlp), N))


def dash_deform_slice_fwd(cfg, mlp, xyz, slice_t, params, base=None, out=None, index=None, N=None, workspace=None):
    """out[n] = base[n] + MLP(G_4D(xyz_n, t)) from a slice, fused kernel with 8-corner gathers."""
    _dev(xyz, torch.float32, "xyz"); _dev(index, torch.int32, "index"); _dev(slice_t, torch.float32, "slice")
    _dev(params, torch.float32, "params"); _dev(base, torch.float32, "base")
    xs = _xyz_stride(xyz)
    if N is None:
        N = int(index.numel()) if index is not None else int(xyz.shape[0])
    if out is None:
        out = torch.empty((N, int(mlp.width[mlp.n_layers])), dtype=torch.float32, device=xyz.device)
    _dev(out, torch.float32, "out")
    n_out = int(mlp.width[mlp.n_layers])
    _check_queries(cfg, xyz, None, index, 0, N)
    _exactly(slice_t, _table_elems(cfg), "slice"); _exactly(params, dash_mlp_param_count(mlp), "params")
    _at_least(base, N * n_out, "base"); _at_least(out, N * n_out, "out")
    _one_device(xyz, index, slice_t, params, base, out, workspace)
    need = dash_deform_slice_workspace_bytes(cfg, mlp, N)
    if need and workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=xyz.device)
    wbytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    _check(_load().dash_deform_slice_fwd(C.byref(cfg), C.byref(mlp), N, _ptr(xyz), xs, _ptr(index), _ptr(slice_t),
                                         _ptr(params), _ptr(base), _ptr(out), _ptr(workspace), wbytes, _stream()))
    return out


# ---- host-buffer entry points (bench.py "e2e"): copies in, C-ABI calls, copies out -----------------

def dash_hash4d_fwd_host(cfg, xyz_h, t_h, table_d, out_h, index_h=None, t_stride=None, staging=None):
    """Forward with HOST (pinned) query and output buffers; the table stays resident on the device
    (it is the model's parameter).  Copies are async on the current stream; caller synchronises."""
    st = staging if staging is not None else {}
    xyz_d = _stage(st, "xyz", xyz_h); t_d = _stage(st, "t", t_h)
    index_d = _stage(st, "index", index_h) if index_h is not None else None
    out_d = st.get("out")
    if out_d is None or out_d.shape != out_h.shape:
        out_d = st["out"] = torch.empty(out_h.shape, dtype=torch.float32, device=torch.device("cuda", torch.cuda.current_device()))
    dash_hash4d_fwd(cfg, xyz_d, t_d, table_d, out=out_d, index=index_d, t_stride=t_stride)
    out_h.copy_(out_d, non_blocking=True)
    return out_h


def dash_hash4d_bwd_host(cfg, xyz_h, t_h, dout_h, dtable_h, index_h=None, t_stride=None, staging=None,
                         reuse_queries=False):
    """Backward with HOST (pinned) buffers: dout in, dtable out (zeroed on the device first)."""
    st = staging if staging is not None else {}
    if reuse_queries and "xyz" in st:
        xyz_d, t_d, index_d = st["xyz"], st["t"], st.get("index")
    else:
        xyz_d = _stage(st, "xyz", xyz_h); t_d = _stage(st, "t", t_h)
        index_d = _stage(st, "index", index_h) if index_h is not None else None
    dout_d = _stage(st, "dout", dout_h)
    dt_d = st.get("dtable")
    if dt_d is None or dt_d.shape != dtable_h.shape:
        dt_d = st["dtable"] = torch.empty(dtable_h.shape, dtype=torch.float32, device=torch.device("cuda", torch.cuda.current_device()))
    if not (cfg.flags & FLAG_ZERO_GRAD):
        dash_hash4d_zero(cfg, dt_d)
    dash_hash4d_bwd(cfg, xyz_d, t_d, dout_d, dt_d, index=index_d, t_stride=t_stride)
    dtable_h.copy_(dt_d, non_blocking=True)
    return dtable_h


def _stage(st: dict, key: str, host: torch.Tensor) -> torch.Tensor:
    dev = st.get(key)
    if dev is None or dev.shape != host.shape or dev.dtype != host.dtype:
        dev = st[key] = torch.empty(host.shape, dtype=host.dtype, device=torch.device("cuda", torch.cuda.current_device()))
    dev.copy_(host, non_blocking=True)
    return dev


class HostStep:
    """One training-shaped step with HOST (pinned) buffers: queries and dY in, features and table gradient
    out, the table resident on the device.  Copies run on two side streams so that the D2H of `out`
    overlaps the H2D of `dout` and the backward (PCIe is full duplex); every arithmetic step is still a
    C-ABI call on the compute stream.  Device staging buffers are owned by this object and reused."""

    def __init__(self, cfg: Hash4DConfig):
        self.cfg = cfg
        self.h2d = torch.cuda.Stream()
        self.d2h = torch.cuda.Stream()
        self.buf: dict = {}
        self.out_copied = None        # event: previous step's D2H finished (buffers reusable)

    def _dev_like(self, key, host):
        cur = self.buf.get(key)
        if cur is None or cur.shape != host.shape or cur.dtype != host.dtype:
            cur = self.buf[key] = torch.empty(host.shape, dtype=host.dtype, device=torch.device("cuda", torch.cuda.current_device()))
        return cur

    def __call__(self, xyz_h, t_h, table_d, dout_h, out_h, dtable_h, index_h=None, t_stride=None):
        cfg, main = self.cfg, torch.cuda.current_stream()
        if self.out_copied is not None:                 # do not overwrite buffers still being read back
            self.h2d.wait_event(self.out_copied)
            main.wait_event(self.out_copied)
        self.h2d.wait_stream(main)
        with torch.cuda.stream(self.h2d):
            xyz_d = self._dev_like("xyz", xyz_h); xyz_d.copy_(xyz_h, non_blocking=True)
            t_d = self._dev_like("t", t_h); t_d.copy_(t_h, non_blocking=True)
            index_d = None
            if index_h is not None:
                index_d = self._dev_like("index", index_h); index_d.copy_(index_h, non_blocking=True)
            q_ready = torch.cuda.Event(); q_ready.record(self.h2d)
            dout_d = self._dev_like("dout", dout_h); dout_d.copy_(dout_h, non_blocking=True)
            d_ready = torch.cuda.Event(); d_ready.record(self.h2d)
        out_d = self._dev_like("out", out_h)
        dt_d = self._dev_like("dtable", dtable_h)
        # ONE workspace, owned by this object, serves both calls of the step: under SORT_COARSE the forward leaves the
        # cell-sorted order in it and the backward reuses it (ORDER_READY) instead of sorting again.
        N = int(index_h.numel()) if index_h is not None else int(xyz_h.shape[0])   # as dash_hash4d_fwd counts them
        need = max(dash_hash4d_workspace_bytes(cfg, N, OP_FWD), dash_hash4d_workspace_bytes(cfg, N, OP_BWD))
        ws = self.buf.get("workspace")
        if need and (ws is None or ws.numel() < need):
            ws = self.buf["workspace"] = torch.empty(need, dtype=torch.uint8,
                                                     device=torch.device("cuda", torch.cuda.current_device()))
        ws = ws if need else None
        cfg_bwd = cfg
        if (cfg.flags & FLAG_SORT_COARSE) and not (cfg.flags & FLAG_DETERMINISTIC_BWD):
            cfg_bwd = with_flags(cfg, cfg.flags | FLAG_ORDER_READY)
        main.wait_event(q_ready)
        dash_hash4d_fwd(cfg, xyz_d, t_d, table_d, out=out_d, index=index_d, t_stride=t_stride, workspace=ws)
        f_done = torch.cuda.Event(); f_done.record(main)
        with torch.cuda.stream(self.d2h):
            self.d2h.wait_event(f_done)
            out_h.copy_(out_d, non_blocking=True)
        main.wait_event(d_ready)
        if not (cfg.flags & FLAG_ZERO_GRAD):
            dash_hash4d_zero(cfg, dt_d)
        dash_hash4d_bwd(cfg_bwd, xyz_d, t_d, dout_d, dt_d, index=index_d, t_stride=t_stride, workspace=ws)
        b_done = torch.cuda.Event(); b_done.record(main)
        with torch.cuda.stream(self.d2h):
            self.d2h.wait_event(b_done)
            dtable_h.copy_(dt_d, non_blocking=True)
            self.out_copied = torch.cuda.Event(); self.out_copied.record(self.d2h)
        main.wait_event(self.out_copied)               # results are complete when the caller's stream is
        return out_h, dtable_h


# ---- chip-ceiling microbenchmarks (include/dash_ceilings.h; bench.py --ceilings) --------------------------

def dash_ceiling_launch(kind, buf, sink, width=8, pattern=CEIL_INDEPENDENT, footprint_bytes=None, grid=0, block=0,
                        dyn_smem=0, iters=16, seed=1) -> int:
    """One launch of a microbenchmark kernel on the current stream; returns its number of lane accesses."""
    _dev(buf, torch.uint8, "buf"); _dev(sink, torch.uint8, "sink"); _one_device(buf, sink)
    p = CeilingParams()
    p.struct_size = C.sizeof(CeilingParams)
    p.kind, p.width, p.pattern = int(kind), int(width), int(pattern)
    p.footprint_bytes = int(buf.numel() if footprint_bytes is None else footprint_bytes)
    if p.footprint_bytes > buf.numel() or sink.numel() < (p.footprint_bytes if kind == CEIL_COPY else 16):
        raise ValueError("buf / sink smaller than the footprint")
    p.grid, p.block, p.dyn_smem, p.iters, p.seed = int(grid), int(block), int(dyn_smem), int(iters), int(seed)
    ops = C.c_uint64(0)
    rc = _load_ceilings().dash_ceiling_launch(C.byref(p), _ptr(buf), _ptr(sink), C.byref(ops), _stream())
    if rc != 0:
        raise Hash4DError(rc, "dash_ceiling_launch: bad parameters or launch failure")
    return int(ops.value)


# ---- self-supervised decomposition (include/dash_decompose.h; Eq. 5) -------------------------

def dash_decompose(dp, k_percent, grad_scale=1.0, want_grad=True, workspace=None):
    """dp [N][3] CUDA fp32 -> dict(mag [N], index (the whole [N] int32 buffer; the first n_dynamic entries are valid),
    result (4 x 32-bit CUDA tensor viewed as uint8: n_dynamic, n_static, tau, loss), ddp [N][3] or None).  Nothing is
    synchronised: read `result` with `dash_decompose_read(result)` when the counts are needed on the host."""
    _dev(dp, torch.float32, "dp")
    if dp.dim() != 2 or dp.shape[1] != 3:
        raise ValueError("dp must be [N][3]")
    N = int(dp.shape[0])
    dev = dp.device
    mag = torch.empty((N,), dtype=torch.float32, device=dev)
    index = torch.empty((max(N, 1),), dtype=torch.int32, device=dev)
    result = torch.zeros(C.sizeof(DecomposeResult), dtype=torch.uint8, device=dev)
    ddp = torch.empty((N, 3), dtype=torch.float32, device=dev) if want_grad else None
    need = int(_load().dash_decompose_workspace_bytes(N))
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=dev)
    _one_device(dp, workspace)
    rc = _load().dash_decompose(N, _ptr(dp), float(k_percent), float(grad_scale), _ptr(mag), _ptr(index), _ptr(result),
                                _ptr(ddp), _ptr(workspace), workspace.numel(), _stream())
    if rc != 0:
        raise Hash4DError(rc, "dash_decompose: bad arguments, workspace too small or launch failure")
    return {"mag": mag, "index": index, "result": result, "ddp": ddp}


def dash_decompose_read(result: torch.Tensor) -> DecomposeResult:
    """Copy the 16-byte result to the host (synchronises)."""
    return DecomposeResult.from_buffer_copy(bytes(result.cpu().numpy().tobytes()))
