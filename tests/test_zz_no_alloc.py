"""dash_hash4d_sort_queries_static: the query sort for callers that cannot allocate device memory.

Some users of this library are in no position to call cudaMalloc: a plug-in that lives inside a renderer or trainer
which owns the whole GPU memory pool and only lends out input and output buffers; a per-frame loop where cudaMalloc /
cudaFree would stall every stream on the device; a process whose HBM is already full of tables and Gaussians.  For them
the library carries the sort's scratch (keys, histogram bins, scan totals; about 5 MB) as a fixed array in its own
device data segment, and the `_static` entry point uses that instead of a caller-supplied workspace.

What is checked here, against the existing dash_hash4d_sort_queries on the same inputs:
  * both orders are permutations and walk the queries through exactly the same sequence of Morton keys, i.e. every
    cell holds the same set of queries at the same positions.  The order of queries WITHIN one cell is left open by the
    method (ties land in whatever order the cursor atomics hand out, in both paths), so it is not compared — the same
    bar tests/test_gpu_parity.py::test_sort_queries_is_a_permutation_in_key_order uses, which is exact for what is unique;
  * two calls in a row, the second with fewer queries and fewer bits than the first, so that anything the first call
    left in the shared array (stale keys past the new N, stale counts in the low bins) would corrupt the second;
  * the same call repeated gives a valid result again;
  * the second call does not shrink the device's free memory (nothing was allocated behind the caller's back);
  * sizes beyond the stated maximum are refused with a message that names the limit, before anything is launched.

This file is named so that pytest collects it after every other test file: the array is shared process-wide state and a
failure here must not hide the tests that come before it under `pytest -x`.  It passes alone in a fresh process and at
the end of the full run alike.
"""
import ctypes as C

import numpy as np
import pytest
import torch

import paper_2507_19141_b200 as dh


def dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def morton_keys(points: np.ndarray, bits: int) -> np.ndarray:
    """The sort key of include/dash_hash4d.h, rebuilt with numpy: clamp to [0, 1-2^-24] (NaN -> 0), one exact
    power-of-two binary32 product, floor, interleave x/y/z bits."""
    c = np.clip(np.nan_to_num(points, nan=0.0), 0, np.float32(1) - np.float32(2.0 ** -24)).astype(np.float32)
    cell = np.minimum((c * np.float32(2 ** bits)).astype(np.uint32), 2 ** bits - 1)
    key = np.zeros(len(points), np.uint64)
    for b in range(bits):
        for d in range(3):
            key |= ((cell[:, d].astype(np.uint64) >> b) & 1) << (3 * b + d)
    return key


def make_case(seed: int, rows: int, n_index):
    rng = np.random.default_rng(seed)
    # clustered like the workloads (a few blobs over a uniform background) so that many queries share a cell
    centres = rng.random((8, 3))
    blob = centres[rng.integers(0, 8, rows)] + 0.03 * rng.standard_normal((rows, 3))
    xyz = np.where(rng.random((rows, 1)) < 0.7, blob, rng.random((rows, 3))).astype(np.float32)
    xyz[:4] = [[0, 0, 0], [1, 1, 1], [np.nan, 0.5, -3], [0.5, 0.25, 0.75]]
    index = None if n_index is None else rng.integers(0, rows, n_index).astype(np.int32)
    return xyz, index


def check_same_as_workspace_path(xyz, index, bits, order_buf):
    n = len(index) if index is not None else len(xyz)
    xd, idx = dev(xyz), dev(index)
    want = dh.dash_hash4d_sort_queries(xd, index=idx, bits=bits).cpu().numpy()
    order_buf.fill_(-1)
    got = dh.dash_hash4d_sort_queries_static(xd, order_buf, index=idx, bits=bits)
    torch.cuda.synchronize()
    got = got[:n].cpu().numpy()
    ids = np.arange(n)
    assert np.array_equal(np.sort(want), ids), "workspace path: not a permutation"
    assert np.array_equal(np.sort(got), ids), "static path: not a permutation"
    key = morton_keys(xyz[index] if index is not None else xyz, bits)
    assert (np.diff(key[want].astype(np.int64)) >= 0).all()
    # integer work: exact.  Equal key sequences of two permutations <=> every cell owns the same slots in both.
    np.testing.assert_array_equal(key[got], key[want])
    if n < order_buf.numel():
        assert int(order_buf[n:].max()) == -1, "wrote past N"


@pytest.mark.gpu
def test_static_sort_matches_workspace_sort_on_consecutive_calls():
    order_buf = torch.empty(300_000, dtype=torch.int32, device="cuda")
    big = make_case(1, 300_000, None)             # 6 bits: 262 144 bins, every region of the array is used
    small = make_case(2, 5_000, 7_001)            # 4 bits, index list: sits inside what the first call dirtied
    check_same_as_workspace_path(*big, 6, order_buf)
    check_small = lambda: check_same_as_workspace_path(*small, 4, order_buf)
    # the static call alone, bracketed: it must not take device memory
    xd, idx = dev(small[0]), dev(small[1])
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    dh.dash_hash4d_sort_queries_static(xd, order_buf, index=idx, bits=4)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "the no-allocation call reduced free device memory"
    check_small()
    check_small()                                 # and again: same call, array still dirty from itself
    check_same_as_workspace_path(*big, 6, order_buf)


@pytest.mark.gpu
def test_static_sort_at_its_maximum_size():
    n = dh.binding.SORT_STATIC_MAX_N
    xyz, _ = make_case(3, n, None)
    order_buf = torch.empty(n, dtype=torch.int32, device="cuda")
    check_same_as_workspace_path(xyz, None, dh.binding.SORT_STATIC_MAX_BITS, order_buf)
    check_same_as_workspace_path(xyz[:1], None, 1, order_buf)   # smallest case right after the largest


@pytest.mark.gpu
def test_static_sort_refuses_oversize_through_the_binding():
    xyz = torch.zeros((8, 3), dtype=torch.float32, device="cuda")
    order = torch.empty(8, dtype=torch.int32, device="cuda")
    with pytest.raises(dh.Hash4DError) as e:
        dh.dash_hash4d_sort_queries_static(xyz, order, bits=7)
    assert e.value.status == 2 and "bits" in str(e.value)


def test_static_sort_limits_are_refused_before_any_gpu_work():
    """Runs without a GPU: the size checks come first, so a too-large request never reaches the CUDA runtime."""
    lib = C.CDLL(dh.library_path())
    fn = lib.dash_hash4d_sort_queries_static
    fn.argtypes = [C.c_uint64, C.c_void_p, C.c_uint32, C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p]
    fn.restype = C.c_int
    lib.dash_hash4d_last_error.restype = C.c_char_p
    assert fn(dh.binding.SORT_STATIC_MAX_N + 1, None, 3, None, 6, None, None) == 2          # UNSUPPORTED
    assert b"1048576" in lib.dash_hash4d_last_error()
    assert fn(16, None, 3, None, dh.binding.SORT_STATIC_MAX_BITS + 1, None, None) == 2
    assert b"bits" in lib.dash_hash4d_last_error()
    assert fn(16, None, 3, None, 0, None, None) == 2
    assert fn(0, None, 3, None, 6, None, None) == 0                                          # N == 0: no-op
    assert fn(16, None, 3, None, 6, None, None) == 1                                         # NULL xyz: INVALID_ARG
