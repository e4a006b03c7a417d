"""`-m gpu`: FARM_OPT_INPUTS_READY = 1, the split similarity schedule: from the third call on the similarity
kernel of a call starts when the previous call's similarity kernel ends -- before that call's decision scan and merge -- computes
the rows that merge does not write with the rows it does write masked, and those rows afterwards from the delta buffer.  Results
must be identical to the stream-ordered schedule and to the oracle.

In a file of its own, collected after the other parity files: these tests run kernels of consecutive calls concurrently, and the
suite runs with `pytest -x`.
"""
import numpy as np
import pytest
import torch

from helpers import generate_frames, integrate_frames, margin_filter
from paper_2606_15476_b200 import scenes as S
from parity import compare_call, compare_dense, compare_maps, make_pair, upload
from test_gpu_parity import _stress_pair

pytestmark = pytest.mark.gpu


def _integrate_ready(g, frames, dtype):
    """the option's contract: the inputs are complete in device memory when the call is made"""
    d = upload(frames, dtype)
    torch.cuda.synchronize()
    g.integrate_batch(len(frames), d["depth"], d["mask"], d["K"], d["T"], d["desc"], d["n_det"])
    return d


@pytest.mark.parametrize("cfg_id,n,sim_path", [(1, 40, 2), (2, 60, 0)])
def test_inputs_ready_split_similarity_every_call_matches_oracle(oracle, cfg_id, n, sim_path):
    """FARM_OPT_INPUTS_READY = 1: from the third call on the similarity kernel runs the split schedule (old rows minus the rows
    the previous call merges into, then those rows from the delta buffer).  Every call's decisions, scores and dense
    (max, argmax) and the final map against the oracle -- fp16 and bf16, maps of 1 to 3 column tiles."""
    cfg = S.get_config(cfg_id)
    pre = generate_frames(cfg_id, range(20, 20 + n) if cfg_id == 1 else range(n))
    o, g = make_pair(oracle, cfg, sim_path=sim_path, inputs_ready=1)
    keep = []
    n_dense = 0
    for fr in pre:
        frames = margin_filter(o.clone, [fr], cfg.tau)
        integrate_frames(o, frames)
        keep.append(_integrate_ready(g, frames, cfg.dtype))
        compare_call(g, o)
        n_dense += compare_dense(g, o)
    compare_maps(g, o)
    assert n_dense > n and len(o.read(voxels=False)[0]) > 30


def test_inputs_ready_back_to_back_calls_equal_the_stream_ordered_run(oracle):
    """The same with nothing between the calls (no read, no sync: the kernels of consecutive calls really overlap), on the
    configs[4] structure (bf16 tensor path, several row and column tiles, 800 detections per call, half of them merged): the map
    after 6 calls equals the oracle's and is byte-equal to the run without the option."""
    sc = S.StressScene(n_batches=6, frames_per_batch=8, n_objects=700)
    calls = []
    o = None
    maps = []
    for ready in (1, 0):
        oo, g = _stress_pair(oracle, sc, inputs_ready=ready, max_voxels=1 << 24)
        if o is None:
            o = oo
            for b in range(6):
                frames = margin_filter(o.clone, sc.batch(b), sc.cfg.tau)
                integrate_frames(o, frames)
                calls.append(frames)
        staged = [upload(fr, sc.cfg.dtype) for fr in calls]
        torch.cuda.synchronize()
        for d, fr in zip(staged, calls):
            g.integrate_batch(len(fr), d["depth"], d["mask"], d["K"], d["T"], d["desc"], d["n_det"])
        compare_call(g, o)
        compare_maps(g, o)
        maps.append(g.read(voxels=False))
        g.destroy()
    assert np.array_equal(maps[0][0], maps[1][0]) and np.array_equal(maps[0][1], maps[1][1])     # objects, descriptors


@pytest.mark.parametrize("cfg_id,n", [(1, 60), (2, 50)])
def test_inputs_ready_single_frame_series_back_to_back(oracle, cfg_id, n):
    """The bench's single-frame series: n single-frame calls with nothing between them (prep, lift and the similarity kernel of a
    call run beside the previous call's probe -> scoring -> scan -> merge chain; the probe kernel reads its small queue along the
    diagonal and waits for its lift kernel on the device).  Last call and final map against the oracle."""
    cfg = S.get_config(cfg_id)
    o, g = make_pair(oracle, cfg, inputs_ready=1)
    calls = []
    for fr in generate_frames(cfg_id, range(20, 20 + n) if cfg_id == 1 else range(n)):
        frames = margin_filter(o.clone, [fr], cfg.tau)
        integrate_frames(o, frames)
        calls.append(frames)
    staged = [upload(fr, cfg.dtype) for fr in calls]
    torch.cuda.synchronize()
    for d, fr in zip(staged, calls):
        g.integrate_batch(len(fr), d["depth"], d["mask"], d["K"], d["T"], d["desc"], d["n_det"])
    compare_call(g, o)
    compare_maps(g, o)
    assert len(o.read(voxels=False)[0]) > 30


def test_inputs_ready_with_host_buffers_back_to_back(oracle):
    """farm_map_integrate_batch_host with the option: the library stages the inputs itself (two staging sets), the early and side
    streams wait for the copy; 40 single-frame calls with nothing between them, final map against the oracle."""
    from helpers import stack_frames
    cfg = S.get_config(1)
    o, g = make_pair(oracle, cfg, inputs_ready=1)
    keep = []
    for fr in generate_frames(1, range(20, 60)):
        frames = margin_filter(o.clone, [fr], cfg.tau)
        integrate_frames(o, frames)
        depth, mask, K, T, desc, n_det = stack_frames(frames)
        keep.append((depth, mask, K, T, np.ascontiguousarray(desc), n_det))     # host buffers stay alive until the sync
        g.integrate_batch_host(1, *keep[-1])
    compare_call(g, o)
    compare_maps(g, o)


@pytest.mark.parametrize("ready", [0, 1])
def test_skinny_calls_on_a_map_with_more_column_tiles_than_sms(oracle, ready):
    """One row tile of detections (M = 70) against N = 40,000 objects: more 256-column tiles than SMs, so the tensor-core
    similarity kernel runs the grid it sizes for skinny calls (the same number of rounds for every CTA) and, with the split
    schedule, ends without its early programmatic trigger.  Five calls (the last three split when ready = 1); matches rewrite
    rows that later calls match again.  Every call and the final map against the oracle."""
    from helpers import hand_frame, pack_key, pow2_K, unit_rows
    from paper_2606_15476_b200 import FarmMap, binding
    N, D, M, Hh, Ww, dtype = 40000, 64, 70, 96, 128, S.DTYPE_BF16
    rows = unit_rows(N, D, 3)
    objs = np.zeros(N, binding.OBJECT_DTYPE)
    objs["id"], objs["n_voxels"], objs["n_obs"], objs["best_frame"], objs["best_det"] = np.arange(N), 1, 1, -1, -1
    keys = pack_key(np.arange(N) + 500, np.zeros(N, int), np.zeros(N, int))
    owner = np.arange(N, dtype=np.uint32)
    o = oracle.OracleMap(0.25, D, 0.0, 1.0, 0.9, dtype, Hh, Ww)
    g = FarmMap(0.25, D, 0.0, 1.0, 0.9, H=Hh, W=Ww, dtype=dtype, max_objects=N + 1024, max_det_per_call=128, inputs_ready=ready)
    assert o.import_(objs, rows, keys, owner) == 0
    g.import_(objs, rows, keys, owner)
    rng = np.random.default_rng(11)
    pool = rng.permutation(N)[:120]                      # the calls pick from one pool: rows rewritten by a call are matched again
    n_dense = 0
    for call in range(5):
        pick = rng.permutation(pool)[:50]
        near = rows[pick] + 0.02 * unit_rows(50, D, 100 + call)                   # cosine ~ 0.9998 with its row, ~ 0.5 at most elsewhere
        det = np.concatenate([near, unit_rows(M - 50, D, 200 + call)]).astype(np.float32) * 2.0   # the last 20 match nothing: spawns
        depth, mask = hand_frame(Hh, Ww, [(1 + (d % 120), 2 + 3 * (d // 120) + 9 * call, 2.0, d + 1) for d in range(M)])
        fr = S.Frame(depth, mask, pow2_K(), np.eye(4, dtype=np.float32), S.to_storage(det, dtype), M, np.zeros(M, np.int64))
        frames = margin_filter(o.clone, [fr], 0.9)
        integrate_frames(o, frames)
        keep = _integrate_ready(g, frames, dtype)
        compare_call(g, o)
        n_dense += compare_dense(g, o)
        st = g.last_assoc()[3]
        assert int(st["matches"]) >= 45 and int(st["spawns"]) >= 15
    compare_maps(g, o)
    assert n_dense >= 5 * 45


@pytest.mark.parametrize("dtype", [1, 2])
def test_inputs_ready_exact_ties_among_rewritten_rows_go_to_the_lowest_id(oracle, dtype):
    """R18 inside phase 2.  Two pairs of objects with bit-identical rows, (7, 200) and (250, 30); call 2 merges the same
    descriptor into both members of a pair (voxel overlap steers one detection to each), so the rewritten rows are again
    bit-identical and sit in the delta buffer in whatever order the merge warps reached it.  Call 3 -- the first split call --
    asks for them with detections that overlap nothing: the dense argmax decides, the cosines tie exactly, and the lower id of
    each pair must win although its delta column may come second."""
    from helpers import hand_frame, pack_key, pow2_K, unit_rows
    from paper_2606_15476_b200.binding import OBJECT_DTYPE
    D, N, H, W = 64, 300, 96, 128
    rows = unit_rows(N, D, 51)
    rows[200] = rows[7]
    rows[30] = rows[250]

    class Cfg:
        voxel, w_geo, w_sem, tau = 0.25, 0.5, 0.5, 0.3
    Cfg.D, Cfg.dtype = D, dtype
    I4 = np.eye(4, dtype=np.float32)
    for rep in range(3):
        o, g = make_pair(oracle, Cfg, H=H, W=W, sim_path=2, inputs_ready=1)
        objs = np.zeros(N, OBJECT_DTYPE)
        objs["id"], objs["n_voxels"], objs["n_obs"], objs["best_frame"], objs["best_det"] = np.arange(N), 1, 1, -1, -1
        ix = np.arange(N) + 1000
        ix[7], ix[200], ix[250], ix[30] = 0, 2, 4, 6          # one voxel (ix, 0, 8) each; everything else far away
        keys = pack_key(ix, np.zeros(N, int), np.full(N, 8))
        assert o.import_(objs, rows, keys, np.arange(N, dtype=np.uint32)) == 0
        g.import_(objs, rows, keys, np.arange(N, dtype=np.uint32))
        near = lambda i, s: (rows[i] + 0.1 * unit_rows(1, D, s)[0]).astype(np.float32)
        a1, a2 = near(7, 61 + rep), near(250, 71 + rep)
        K2 = pow2_K(128.0, 0.0, 48.0)                         # cx = 0: pixel (u, 48) at z = 2 is the point (u / 64, 0, 2)
        calls = [
            # call 1: a stray detection far from everything (spawns); calls 1 and 2 run the stream-ordered schedule
            ([(10, 10, 3.0, 1)], unit_rows(1, D, 81 + rep)),
            # call 2: u = 0, 32, 64, 96 -> voxels 0, 2, 4, 6 = objects 7, 200, 250, 30; the same descriptor for both members of a pair
            ([(0, 48, 2.0, 1), (32, 48, 2.0, 2), (64, 48, 2.0, 3), (96, 48, 2.0, 4)], np.stack([a1, a1, a2, a2])),
            # call 3: the two queries; they overlap nothing
            ([(10, 20, 3.0, 1), (20, 20, 3.0, 2)], np.stack([rows[7], rows[250]]).astype(np.float32)),
        ]
        for k, (px, desc) in enumerate(calls):
            depth, mask = hand_frame(H, W, px)
            fr = S.Frame(depth, mask, K2 if k == 1 else pow2_K(), I4, S.to_storage(desc, dtype), len(desc), np.zeros(len(desc), np.int64))
            integrate_frames(o, [fr])
            _integrate_ready(g, [fr], dtype)
            compare_call(g, o)
            if k == 1:                                        # the pairs really were rewritten, identically, by call 2
                assert list(o.last_assoc()[0]) == [7, 200, 250, 30]
                d = g.read(voxels=False)[1]
                assert np.array_equal(d[7], d[200]) and np.array_equal(d[250], d[30]) and not np.array_equal(d[7], rows[7])
        ao = o.last_assoc()[0]
        ag = g.last_assoc()[0]
        assert list(ao) == [7, 30] and list(ag) == [7, 30]
        mc_g, am_g = g.debug_last_dense()
        mc_o, am_o = o.last_dense()
        assert list(am_g) == [7, 30] and list(am_o) == [7, 30]
        compare_maps(g, o, voxels=False)
        g.destroy()


def test_inputs_ready_with_every_optional_structure(oracle):
    """The optional structures ride on the state the split schedule double-buffers (per-detection boxes and moments written by
    the lift kernel on its own stream, statistics, the list of the call's entities built by the merge): Gaussians, covisibility
    bitset, views and weighted edges on the mini stress scene, five calls back to back, against the oracle."""
    from test_gpu_parity import _compare_gaussians
    from test_gpu_parity_r2 import _compare_views
    sc = S.StressScene(n_batches=5, frames_per_batch=8, n_objects=700)
    o, g = _stress_pair(oracle, sc, inputs_ready=1, max_voxels=1 << 24, gaussian=1, covisibility=1, views=2, edges=3)
    o.set_option(o.OPT_VIEWS_K, 2)
    o.set_option(o.OPT_EDGES_K, 3)
    calls = []
    for b in range(5):
        frames = margin_filter(o.clone, sc.batch(b), sc.cfg.tau)
        integrate_frames(o, frames)
        calls.append(frames)
    staged = [upload(fr, sc.cfg.dtype) for fr in calls]
    torch.cuda.synchronize()
    for d, fr in zip(staged, calls):
        g.integrate_batch(len(fr), d["depth"], d["mask"], d["K"], d["T"], d["desc"], d["n_det"])
    compare_call(g, o, check_sets=False)
    _compare_gaussians(g, o)
    compare_maps(g, o, voxels=False)
    assert np.array_equal(g.read_covisibility(), o.read_covisibility())
    assert _compare_views(g, o) > 700
    ao, bo, wo = o.read_edges()
    ag, bg, wg = g.read_edges()
    assert np.array_equal(ag, ao) and np.array_equal(bg, bo) and np.abs(wg - wo).max() <= 1e-9 * float(wo.max())
    w_o, mu_o, cov_o = o.read_gaussians()
    w_g, mu_g, cov_g = g.read_gaussians()
    assert np.array_equal(w_g, w_o) and np.abs(mu_g - mu_o).max() <= 1e-4 and np.abs(cov_g - cov_o).max() <= 1e-4
