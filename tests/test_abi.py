"""CPU-side checks of the product's C-ABI library: it loads, exports every symbol include/dash_hash4d.h
declares, validates arguments, and evaluates Eq. 7 (host-only call).  No compute call is made."""
import ctypes as C
import os
import re

import pytest

import paper_2507_19141_b200 as dh
from dash_inputs import CONFIGS

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared(only=None, skip=()):
    names = []
    inc = os.path.join(ROOT, "include")
    for fn in sorted(os.listdir(inc)):
        if fn.endswith(".h") and fn not in skip and (only is None or fn in only):
            text = open(os.path.join(inc, fn)).read()
            names += re.findall(r"DASH_API\s+[\w\s\*]+?\b(dash_\w+)\s*\(", text)
    return names


def test_library_exports_every_declared_symbol():
    names = _declared(skip=("dash_ceilings.h",))
    assert len(names) >= 8 and "dash_hash4d_fwd" in names and "dash_hash4d_bwd" in names \
        and "dash_hash4d_indices" in names and "dash_hash3d_fwd" in names and "dash_hash4d_set_debug" in names
    lib = C.CDLL(dh.library_path())
    for n in names:
        assert hasattr(lib, n), n
    assert set(dh.exported_symbols()) == set(names)


def test_microbenchmarks_live_in_their_own_library():
    """include/dash_ceilings.h is served by libdash_ceilings.so; the product library exports only the method."""
    names = _declared(only=("dash_ceilings.h",))
    assert names == ["dash_ceiling_launch"] == dh.binding.CEIL_EXPORTS
    from paper_2507_19141_b200 import build as b
    b.build_ceilings()
    assert not b.ceilings_is_stale()
    ceil = C.CDLL(dh.binding.ceilings_library_path())
    assert hasattr(ceil, "dash_ceiling_launch")
    assert not hasattr(C.CDLL(dh.library_path()), "dash_ceiling_launch")
    product_header = open(os.path.join(ROOT, "include", "dash_hash4d.h")).read()
    assert "dash_debug_key" not in product_header and "dash_debug.h" not in product_header


def test_struct_layout_matches_header():
    assert C.sizeof(dh.Hash4DConfig) == 14 * 4


def _rows(path):
    for line in open(path):
        line = line.split("#")[0].strip()
        if line:
            yield line


def test_resolutions_match_printed_lists(golden_dir):
    for row in _rows(os.path.join(golden_dir, "resolutions.txt")):
        head, vals = row.split(":")
        _, n_min, n_max, L = head.split()
        want = [int(v) for v in vals.split()]
        cfg = dh.make_config(int(L), 2, 1 << 12, int(n_min), int(n_max), int(n_min), int(n_max))
        rs, rt, _ = dh.dash_hash4d_resolutions(cfg)
        assert rs == want and rt == want


def test_dense_levels_per_config():
    want = {"C1": [], "C2": [0, 1], "C3": [0, 1, 2], "C4": [0, 1, 2, 3], "C5": [0, 1, 2]}
    for name, levels in want.items():
        cfg = dh.config_from_params(CONFIGS[name].enc)
        _, _, dn = dh.dash_hash4d_resolutions(cfg)
        assert [l for l, d in enumerate(dn) if d] == levels
        cfg = dh.config_from_params(CONFIGS[name].enc, flags=0)
        assert not any(dh.dash_hash4d_resolutions(cfg)[2])


@pytest.mark.parametrize("kw,status", [
    (dict(L=0), 1), (dict(L=33), 1), (dict(F=3), 2), (dict(F=16), 1), (dict(T=0), 1),
    (dict(res_s_min=0), 1), (dict(res_s_min=200, res_s_max=100), 1), (dict(res_t_min=9, res_t_max=8), 1),
    (dict(res_s_max=(1 << 22) + 1), 1), (dict(table_dtype=2), 1), (dict(flags=64), 1), (dict(struct_size=8), 1),
])
def test_bad_configs_are_rejected(kw, status):
    cfg = dh.make_config(4, 2, 4096, 16, 128, 8, 32)
    for k, v in kw.items():
        setattr(cfg, k, v)
    with pytest.raises(dh.Hash4DError) as ei:
        dh.dash_hash4d_resolutions(cfg)
    assert ei.value.status == status
    assert dh.dash_hash4d_last_error() != ""
    assert dh.dash_hash4d_workspace_bytes(cfg, 10, dh.OP_BWD) == 0


def test_workspace_sizes():
    enc = CONFIGS["C2"].enc
    cfg = dh.config_from_params(enc)
    for op in (dh.OP_FWD, dh.OP_BWD, dh.OP_INDICES):
        assert dh.dash_hash4d_workspace_bytes(cfg, 1000, op) == 0
    det = dh.config_from_params(enc, flags=dh.FLAG_DENSE_COARSE | dh.FLAG_DETERMINISTIC_BWD)
    assert dh.dash_hash4d_workspace_bytes(det, 1000, dh.OP_BWD) == 128 + enc.L * enc.T * enc.F * 8
    assert dh.dash_hash4d_workspace_bytes(det, 1000, dh.OP_FWD) == 0
    val = dh.config_from_params(enc, flags=dh.FLAG_DENSE_COARSE | dh.FLAG_VALIDATE_INPUTS)
    assert dh.dash_hash4d_workspace_bytes(val, 1000, dh.OP_FWD) == 128


def test_sort_coarse_workspace_and_flag_rules():
    """DASH_HASH4D_FLAG_SORT_COARSE (include/dash_hash4d.h): needs a workspace only where the library takes the sorted
    path (N*F >= 2^21, at least one level with Ns^3 Nt <= 2N), the same size for fwd and bwd, none for the other calls,
    none under DETERMINISTIC_BWD; ORDER_READY changes no size; bit 64 is still an unknown flag."""
    sc = dh.FLAG_DENSE_COARSE | dh.FLAG_SORT_COARSE
    for name, n in (("C4", 1_000_000), ("C5", 1_800_000)):
        cfg = dh.config_from_params(CONFIGS[name].enc, flags=sc)
        need = dh.dash_hash4d_workspace_bytes(cfg, n, dh.OP_BWD)
        bins = 1 << 22                                        # level 3: 48^3 x 16 cells -> 6 + 6 + 6 + 4 key bits
        assert need == 128 + 2 * 4 * n + 16 * n + 4 * bins + 4 * (bins // 1024)
        assert dh.dash_hash4d_workspace_bytes(cfg, n, dh.OP_FWD) == need
        assert dh.dash_hash4d_workspace_bytes(dh.with_flags(cfg, sc | dh.FLAG_ORDER_READY), n, dh.OP_BWD) == need
        assert dh.dash_hash4d_workspace_bytes(cfg, n, dh.OP_BWD_INPUT) == need
        for op in (dh.OP_INDICES, dh.OP_SMOOTH):
            assert dh.dash_hash4d_workspace_bytes(cfg, n, op) == 0
        below = (1 << 21) // CONFIGS[name].enc.F - 1
        assert dh.dash_hash4d_workspace_bytes(cfg, below, dh.OP_BWD) == 0              # below the threshold: plain path
        assert dh.dash_hash4d_workspace_bytes(cfg, below + 1, dh.OP_BWD) > 24 * below
        det = dh.with_flags(cfg, sc | dh.FLAG_DETERMINISTIC_BWD)
        assert dh.dash_hash4d_workspace_bytes(det, n, dh.OP_FWD) == 0
    c3 = dh.config_from_params(CONFIGS["C3"].enc, flags=sc)
    assert dh.dash_hash4d_workspace_bytes(c3, CONFIGS["C3"].N, dh.OP_BWD) == 0
    # a very fine coarsest level: no level qualifies, no workspace, the flag does nothing
    fine = dh.make_config(4, 2, 1 << 19, 1024, 4096, 64, 300, flags=sc)
    assert dh.dash_hash4d_workspace_bytes(fine, 1 << 20, dh.OP_BWD) == 0
    bad = dh.config_from_params(CONFIGS["C4"].enc, flags=64)
    res = (C.c_uint32 * 16)()
    assert dh.binding._load().dash_hash4d_resolutions(C.byref(bad), res, res, None) == 1


def test_null_and_stride_validation_happens_before_any_cuda_call():
    lib = C.CDLL(dh.library_path())
    lib.dash_hash4d_fwd.restype = C.c_int
    cfg = dh.make_config(4, 2, 4096, 16, 128, 8, 32)
    u64, u32, vp = C.c_uint64, C.c_uint32, C.c_void_p
    # N = 0 is OK and a no-op, whatever the pointers
    assert lib.dash_hash4d_fwd(C.byref(cfg), u64(0), vp(0), u32(3), vp(0), u32(1), vp(0), vp(0), vp(0),
                               vp(0), C.c_size_t(0), vp(0)) == 0
    # null xyz
    assert lib.dash_hash4d_fwd(C.byref(cfg), u64(4), vp(0), u32(3), vp(0), u32(1), vp(0), vp(0), vp(0),
                               vp(0), C.c_size_t(0), vp(0)) == 1
    # bad stride (fake non-null, never dereferenced: validation fails first)
    fake = vp(4096)
    assert lib.dash_hash4d_fwd(C.byref(cfg), u64(4), fake, u32(5), fake, u32(1), vp(0), fake, fake,
                               vp(0), C.c_size_t(0), vp(0)) == 1
    assert lib.dash_hash4d_fwd(C.byref(cfg), u64(4), fake, u32(3), fake, u32(2), vp(0), fake, fake,
                               vp(0), C.c_size_t(0), vp(0)) == 1
    # misaligned table
    assert lib.dash_hash4d_fwd(C.byref(cfg), u64(4), fake, u32(3), fake, u32(1), vp(0), vp(4100), fake,
                               vp(0), C.c_size_t(0), vp(0)) == 1


def test_binding_refuses_cpu_tensors():
    import torch
    cfg = dh.make_config(4, 2, 4096, 16, 128, 8, 32)
    x = torch.zeros(4, 3); t = torch.zeros(4); tab = torch.zeros(4, 4096, 2)
    with pytest.raises(ValueError):
        dh.dash_hash4d_fwd(cfg, x, t, tab)


def test_build_id_is_the_hash_of_the_sources_beside_the_library():
    from paper_2507_19141_b200 import build as b
    lib = C.CDLL(dh.library_path())
    lib.dash_hash4d_build_id.restype = C.c_char_p
    assert lib.dash_hash4d_build_id().decode() == b.source_hash() == b.built_id()
    assert not b.is_stale()


def test_set_debug_validates_and_reads_no_environment(monkeypatch):
    """Overrides go through dash_hash4d_set_debug only; the old environment knobs are dead."""
    assert dh.dash_hash4d_set_debug(dh.DEBUG_FWD_GROUP, 4) is None
    dh.dash_hash4d_set_debug(dh.DEBUG_FWD_GROUP, 0)
    with pytest.raises(dh.Hash4DError):
        dh.dash_hash4d_set_debug(99, 1)
    with pytest.raises(dh.Hash4DError):
        dh.dash_hash4d_set_debug(dh.DEBUG_BWD_GROUP, -1)
    src = "".join(open(os.path.join(ROOT, "paper_2507_19141_b200", "csrc", f)).read()
                  for f in os.listdir(os.path.join(ROOT, "paper_2507_19141_b200", "csrc")))
    assert "getenv" not in src


def test_mlp_bwd_refuses_layer_outputs_wider_than_one_tile():
    """dash_mlp_bwd issues one M = 128 weight-gradient tile per layer: an output width above 128 is UNSUPPORTED (decided
    on the host before any pointer is looked at), widths up to 128 pass the plan (NULL buffers then give INVALID_ARG)."""
    lib = dh.binding._load()
    call = lambda widths: lib.dash_mlp_bwd(C.byref(dh.make_mlp_config(widths)), 4, None, None, None, None, None, None)
    for widths in ([32, 192, 10], [32, 64, 200], [32, 129]):
        assert call(widths) == 2, widths
        assert "128" in dh.dash_hash4d_last_error()
    for widths in ([32, 128, 10], [32, 128, 128, 10], [240, 16]):
        assert call(widths) == 1, widths


def test_decompose_failures_set_the_last_error_message():
    """dash_decompose reports through the library's one error channel: each refusal (decided on the host, no GPU needed)
    leaves its own message in dash_hash4d_last_error() rather than whatever an earlier call left there."""
    lib = dh.binding._load()
    call = lambda n, k, result, ws, ws_bytes: lib.dash_decompose(n, None, k, 1.0, None, None, result, None, ws, ws_bytes, None)
    dh.dash_hash4d_set_debug(dh.DEBUG_FWD_GROUP, 0)                       # a successful call: message cleared
    assert dh.dash_hash4d_last_error() == ""
    assert call(4, 101.0, C.c_void_p(16), None, 0) == 1
    assert "k_percent" in dh.dash_hash4d_last_error()
    assert call(4, 10.0, None, None, 0) == 1
    assert "result" in dh.dash_hash4d_last_error()
    assert call(1 << 31, 10.0, C.c_void_p(16), None, 0) == 2
    assert "int32" in dh.dash_hash4d_last_error()
    assert call(0, 10.0, C.c_void_p(16), None, 0) == 3
    assert "workspace bytes" in dh.dash_hash4d_last_error()
    assert call(0, 10.0, C.c_void_p(16), C.c_void_p(8), 1 << 20) == 1
    assert "aligned" in dh.dash_hash4d_last_error()
