"""`-m gpu`: farm_cosine_rowmax_noalloc (the entry point that allocates nothing; fixed scratch array inside the library)
against the existing path -- a map with the same B rows imported, one integrate call with the same A rows, dense (max, argmax)
read back with farm_debug_last_dense -- on two calls in a row that share the scratch array.

Named test_zz_* so that pytest collects it last: the suite runs with `pytest -x`, and a failure here must not hide other tests.
Passes alone in a fresh process and after the other tests (it depends on no state but the library's own scratch array, which
every call re-initialises).
"""
import numpy as np
import pytest
import torch

from helpers import hand_frame, pack_key, pow2_K, unit_rows
from paper_2606_15476_b200 import FarmError, FarmMap, binding, scenes as S
from parity import TOL, gpu_integrate

pytestmark = pytest.mark.gpu

H, W = 96, 128


def _existing_path(rows_b, det, dtype, sim_path):
    """dense (max_cos, argmax) of the product's integrate path: B imported into a fresh map, A as one frame's detections."""
    N, D = rows_b.shape
    M = len(det)
    g = FarmMap(0.25, D, 0.0, 1.0, 2.0, H=H, W=W, dtype=dtype, sim_path=sim_path, max_det_per_call=max(M, 64))   # tau = 2: nothing merges
    objs = np.zeros(N, binding.OBJECT_DTYPE)
    objs["id"], objs["n_voxels"], objs["n_obs"], objs["best_frame"], objs["best_det"] = np.arange(N), 1, 1, -1, -1
    keys = pack_key(np.arange(N) + 500, np.zeros(N, int), np.zeros(N, int))
    g.import_(objs, rows_b, keys, np.arange(N, dtype=np.uint32))
    depth, mask = hand_frame(H, W, [(1 + (d % 120), 2 + 3 * (d // 120), 2.0, d + 1) for d in range(M)])   # one pixel per detection
    fr = S.Frame(depth, mask, pow2_K(), np.eye(4, dtype=np.float32), S.to_storage(det, dtype), M, np.zeros(M, np.int64))
    gpu_integrate(g, [fr], dtype)
    mc, am = g.debug_last_dense()
    g.destroy()
    return mc, am


def _device_rows(x, dtype):
    st = S.to_storage(np.ascontiguousarray(x, np.float32), dtype)
    if dtype == S.DTYPE_F32:
        return torch.from_numpy(np.ascontiguousarray(st, np.float32)).cuda()
    if dtype == S.DTYPE_F16:
        return torch.from_numpy(np.ascontiguousarray(st, np.float16)).cuda()
    return torch.from_numpy(np.ascontiguousarray(st, np.uint16).view(np.int16)).cuda()


def _unit_like_import(rows_b, dtype):
    """what the map holds after import (R26 / R14): rows renormalised in fp32, then rounded to the storage dtype"""
    b = rows_b.astype(np.float64)
    b = (b / np.linalg.norm(b, axis=1, keepdims=True)).astype(np.float32)
    return b


@pytest.mark.parametrize("dtype,sim_path", [(0, 0), (1, 1), (2, 2)])
def test_no_alloc_rowmax_matches_the_integrate_path_on_two_calls(dtype, sim_path):
    D = 64 if sim_path == 2 else 40                      # the tensor path needs D % 8 == 0; 40 is a ragged K tile for the FMA kernels
    rng = np.random.default_rng(7)
    calls = [(300, 70, 11), (130, 37, 12)]               # (N, M, seed): several 64 x 64 tiles with ragged tails; the second call is
    results = []                                         # smaller, so stale scratch of the first one would show
    dev_bufs = []
    for N, M, seed in calls:
        rows_b = unit_rows(N, D, seed)
        pick = rng.permutation(N)[:M]
        det = (rows_b[pick] + 0.05 * unit_rows(M, D, seed + 100)).astype(np.float32) * 3.0      # not unit length: norms matter
        det[5] = 0.0                                                                           # a zero row: cosine 0 everywhere
        A, B = _device_rows(det, dtype), _device_rows(_unit_like_import(rows_b, dtype), dtype)
        mc = torch.full((M,), 7.0, dtype=torch.float32, device="cuda")
        am = torch.full((M,), 7, dtype=torch.int32, device="cuda")
        dev_bufs.append((A, B, mc, am, rows_b, det, pick))
    torch.cuda.synchronize()
    # the two calls go back to back on one stream, nothing in between
    for (N, M, _), (A, B, mc, am, *_rest) in zip(calls, dev_bufs):
        binding.cosine_rowmax_noalloc(A, M, B, N, D, dtype, mc, am, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    for (N, M, _), (A, B, mc, am, rows_b, det, pick) in zip(calls, dev_bufs):
        mc_ref, am_ref = _existing_path(rows_b, det, dtype, sim_path)
        mc_new, am_new = mc.cpu().numpy(), am.cpu().numpy()
        assert np.abs(mc_new - mc_ref).max() <= TOL
        assert mc_new[5] == 0.0 and mc_ref[5] == 0.0
        sel = np.arange(M) != 5                          # the zero row's argmax is "first row" on both sides, checked apart
        assert np.array_equal(am_new[sel], am_ref[sel]) and np.array_equal(am_new[sel], pick[sel])   # near-copies: clear winners
        assert am_new[5] == am_ref[5]
        results.append(mc_new)
    assert results[0].shape == (70,) and results[1].shape == (37,)


def test_no_alloc_limits_and_empty_inputs():
    D = 16
    A = torch.zeros((4, D), dtype=torch.float32, device="cuda")
    mc = torch.full((4,), 7.0, dtype=torch.float32, device="cuda")
    am = torch.full((4,), 7, dtype=torch.int32, device="cuda")
    for M, N in ((binding.NOALLOC_MAX_M + 1, 4), (4, binding.NOALLOC_MAX_N + 1)):
        with pytest.raises(FarmError) as ei:
            binding.cosine_rowmax_noalloc(A, M, A, N, D, 0, mc, am)          # rejected before anything is enqueued or read
        assert ei.value.code == binding.ERR_INVALID_ARG and "exceeds" in str(ei.value)
    with pytest.raises(FarmError):
        binding.cosine_rowmax_noalloc(A, 4, A, 4, 0, 0, mc, am)
    binding.cosine_rowmax_noalloc(A, 4, None, 0, D, 0, mc, am)               # N = 0: (0, -1)
    torch.cuda.synchronize()
    assert mc.cpu().tolist() == [0.0] * 4 and am.cpu().tolist() == [-1] * 4
    binding.cosine_rowmax_noalloc(None, 0, A, 4, D, 0, None, None)           # M = 0: nothing to do
