"""`-m gpu`: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs."""
import numpy as np
import pytest
import torch

from helpers import (KEY_EMPTY, hand_frame, integrate_frames, margin_filter, pack_key, pow2_K, unit_rows)
from paper_2606_15476_b200 import FarmMap, scenes as S
from parity import TOL, compare_call, compare_maps, gpu_integrate, make_pair, upload

pytestmark = pytest.mark.gpu


def _run_sequence(oracle, cfg, frames_per_call, n_calls, start=0, filter_margins=True, **kw):
    sc = S.BoxScene(cfg)
    o, g = make_pair(oracle, cfg, **kw)
    k = start
    for _ in range(n_calls):
        frames = [sc.frame(k + i) for i in range(frames_per_call)]
        k += frames_per_call
        if filter_margins:
            frames = margin_filter(o.clone, frames, cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o)
    compare_maps(g, o)
    return o, g


def test_debug_backproject_bit_exact(oracle):
    """R5/R6: per-pixel world points and keys; fp32 op order identical, no FMA contraction."""
    cfg = S.get_config(1)
    sc = S.BoxScene(cfg)
    o, g = make_pair(oracle, cfg)
    for k in (30, 200):
        fr = sc.frame(k)
        d = upload([fr], cfg.dtype)
        xyz = torch.empty((cfg.H, cfg.W, 3), dtype=torch.float32, device="cuda")
        keys = torch.empty((cfg.H, cfg.W), dtype=torch.int64, device="cuda")
        g.debug_backproject(d["depth"], d["mask"], d["K"], d["T"], fr.n_det, xyz, keys)
        torch.cuda.synchronize()
        xo, ko = o.backproject(fr.depth, fr.mask, fr.K, fr.T, fr.n_det)
        xg = xyz.cpu().numpy()
        kg = keys.cpu().numpy().view(np.uint64)
        assert np.array_equal(kg, ko)
        assert np.array_equal(np.isnan(xg), np.isnan(xo))
        assert np.array_equal(xg[~np.isnan(xg)], xo[~np.isnan(xo)])       # bit-exact, stronger than 1e-4
        assert (ko != KEY_EMPTY).sum() > 10000


def test_config0_full_sequence(oracle):
    """BASELINE.json configs[0]: all 20 frames, every intermediate and the final map."""
    cfg = S.get_config(0)
    o, g = _run_sequence(oracle, cfg, 1, cfg.n_frames)
    objs, _, _, _ = g.read()
    assert 5 <= len(objs) <= 40


def test_config1_prefix_f16(oracle):
    """configs[1] (room, D=512 fp16, misses and false positives): a prefix spanning many tiles."""
    cfg = S.get_config(1)
    o, g = _run_sequence(oracle, cfg, 1, 36, start=20)
    objs, _, _, _ = g.read(voxels=False)
    assert len(objs) > 40 and objs["n_obs"].max() > 5          # the map grows and objects are re-observed


def test_config2_prefix_bf16(oracle):
    """configs[2] (house, D=1024 bf16, 0.9-cosine distractor clusters)."""
    cfg = S.get_config(2)
    _run_sequence(oracle, cfg, 1, 14, start=0)


def test_config3_prefix_outdoor_bf16(oracle):
    """configs[3] (outdoor, 1280x720, 10 cm voxels, range 30 m, far surfaces smeared by sigma = 0.002 z^2)."""
    cfg = S.get_config(3)
    _run_sequence(oracle, cfg, 1, 4, start=0)


def test_batched_frames_one_snapshot(oracle):
    """F > 1: frames of one call share the entry snapshot (R2); ragged F."""
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    o, g = make_pair(oracle, cfg)
    k = 0
    for F in (3, 1, 5, 4):
        frames = margin_filter(o.clone, [sc.frame(k + i) for i in range(F)], cfg.tau)
        k += F
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o)
    compare_maps(g, o)


def test_hand_cases(oracle):
    """The oracle's hand pins run through the CUDA path: strict threshold, R12 lowest index, R8, R3, R23."""
    H, W = 96, 128
    I4 = np.eye(4, dtype=np.float32)
    e = np.eye(4, dtype=np.float32)

    class Cfg:
        voxel, D, w_geo, w_sem, tau, dtype = 0.25, 4, 0.5, 0.5, 0.5, 0

    def frame(px, desc, T=I4):
        depth, mask = hand_frame(H, W, px)
        return S.Frame(depth, mask, pow2_K(), T, np.ascontiguousarray(desc, np.float32), len(desc), np.zeros(len(desc), np.int64))

    o, g = make_pair(oracle, Cfg, H=H, W=W)
    seq = [
        frame([(64, 40, 2.0, 2), (66, 41, 2.0, 1), (96, 48, 2.0, 1)], e[:2]),           # R2/R12/R13/R20
        frame([(64, 40, 2.0, 2), (66, 41, 2.0, 1), (96, 48, 2.0, 1)], e[:2]),
        frame([(64, 48, 2.0, 1), (70, 48, 2.0, 3)], e[:3]),                              # R8: label 2 empty
        frame([(10, 10, 0.0, 1), (12, 10, np.nan, 1), (13, 10, np.inf, 1), (17, 10, 1.0, 3), (18, 10, 1.0, 2)], e[:2]),
        frame([], e[:0]),                                                                # no detections at all
        frame([(64, 48, 2.0, 1), (80, 48, 2.0, 1), (96, 48, 2.0, 1), (112, 48, 2.0, 1)], e[:1]),
    ]
    for fr in seq:
        integrate_frames(o, [fr])
        gpu_integrate(g, [fr], 0)
        compare_call(g, o)
    compare_maps(g, o)


def test_score_hand_case_via_import(oracle):
    """P6 through import + integrate: 0.875 match, and 0.5 is NOT > 0.5."""
    H, W = 96, 128
    I4 = np.eye(4, dtype=np.float32)
    e1 = np.array([[1, 0, 0, 0]], np.float32)
    depth, mask = hand_frame(H, W, [(64, 48, 2.0, 1), (80, 48, 2.0, 1), (96, 48, 2.0, 1), (112, 48, 2.0, 1)])
    fr = S.Frame(depth, mask, pow2_K(), I4, e1, 1, np.zeros(1, np.int64))
    from paper_2606_15476_b200.binding import OBJECT_DTYPE
    for own, expect, new in (([(0, 0, 8), (1, 0, 8), (2, 0, 8)] + [(50 + i, 0, 0) for i in range(5)], 0.875, 0),
                             ([(50 + i, 0, 0) for i in range(8)], 0.5, 1)):
        keys = np.array([pack_key(*k) for k in own], np.uint64)
        obj = np.zeros(1, OBJECT_DTYPE)
        obj["n_voxels"], obj["n_obs"], obj["best_frame"], obj["best_det"] = 8, 1, -1, -1
        g = FarmMap(0.25, 4, 0.5, 0.5, 0.5, H=H, W=W)
        g.import_(obj, e1, keys, np.zeros(8, np.uint32))
        gpu_integrate(g, [fr], 0)
        a, n, b, st = g.last_assoc()
        assert b[0] == np.float32(expect) and n[0] == new and a[0] == (1 if new else 0)


def test_import_round_trip_and_continue(oracle):
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    o, g = make_pair(oracle, cfg)
    for k in range(6):
        fr = sc.frame(k)
        integrate_frames(o, [fr])
        gpu_integrate(g, [fr], cfg.dtype)
    objs, desc, keys, owners = g.read()
    g2 = FarmMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, H=cfg.H, W=cfg.W, dtype=cfg.dtype)
    g2.import_(objs, desc, keys, owners)
    compare_maps(g2, o)
    frames = margin_filter(o.clone, [sc.frame(6)], cfg.tau)
    integrate_frames(o, frames)
    gpu_integrate(g2, frames, cfg.dtype)
    compare_call(g2, o, check_sets=True)
    compare_maps(g2, o)
    # duplicate key is rejected
    g3 = FarmMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, H=cfg.H, W=cfg.W, dtype=cfg.dtype)
    from paper_2606_15476_b200 import FarmError
    with pytest.raises(FarmError):
        g3.import_(objs, desc, np.concatenate([keys, keys[:1]]), np.concatenate([owners, owners[:1]]))


def test_determinism_two_runs_byte_equal(oracle):
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    outs = []
    for _ in range(2):
        g = FarmMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, H=cfg.H, W=cfg.W, dtype=cfg.dtype)
        for k in range(10):
            gpu_integrate(g, [sc.frame(k)], cfg.dtype)
        objs, desc, keys, owners = g.read()
        order = np.argsort(keys)
        outs.append((objs.tobytes(), desc.tobytes(), keys[order].tobytes(), owners[order].tobytes()))
    assert outs[0] == outs[1]


def test_odd_width_scalar_path(oracle):
    """W not a multiple of 8 takes the scalar-load variant of the lift kernel; ragged tiles on both axes."""
    class Cfg:
        voxel, D, w_geo, w_sem, tau, dtype = 0.05, 8, 0.5, 0.5, 0.5, 0
    H, W = 37, 203
    g0 = np.random.default_rng(3)
    o, g = make_pair(oracle, Cfg, H=H, W=W)
    K = np.array([[150, 0, 100], [0, 150, 18], [0, 0, 1]], np.float32)
    for it in range(3):
        depth = (1.5 + 0.5 * g0.random((H, W))).astype(np.float32)
        mask = np.zeros((H, W), np.uint16)
        mask[5:30, 10:90] = 1
        mask[8:36, 100:203] = 2
        mask[0:4, :] = 3
        T = S.pose_from_yaw(np.array([0.1 * it, 0.0, 1.0]), 0.3)
        fr = S.Frame(depth, mask, K, T, unit_rows(3, 8, 5), 3, np.zeros(3, np.int64))
        integrate_frames(o, [fr])
        gpu_integrate(g, [fr], 0)
        compare_call(g, o)
    compare_maps(g, o)


def test_capacity_error_is_sticky(oracle):
    from paper_2606_15476_b200 import FarmError
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    g = FarmMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, H=cfg.H, W=cfg.W, dtype=cfg.dtype, max_objects=2)
    gpu_integrate(g, [sc.frame(0)], cfg.dtype)
    with pytest.raises(FarmError) as ei:
        g.last_assoc()
    assert ei.value.code == -3


def _stress_pair(oracle, sc, **kw):
    from paper_2606_15476_b200.binding import OBJECT_DTYPE
    cfg = sc.cfg
    ijk, owner, n_vox, desc = sc.build_map()
    keys = pack_key(ijk[:, 0], ijk[:, 1], ijk[:, 2])
    objs = np.zeros(len(n_vox), OBJECT_DTYPE)
    objs["id"], objs["n_voxels"], objs["n_obs"], objs["best_frame"], objs["best_det"] = np.arange(len(n_vox)), n_vox, 1, -1, -1
    o, g = make_pair(oracle, cfg, max_det_per_call=1600, max_objects=len(n_vox) + 8000, **kw)
    assert o.import_(objs, desc, keys, owner) == 0
    g.import_(objs, desc, keys, owner)
    return o, g


def test_config4_mini_stress_batches(oracle):
    """configs[4] structure at reduced size: imported blob map, batches of 4 frames x 100 detections, half of
    them overlapping existing objects; whole pipeline and final map against the oracle."""
    sc = S.StressScene(n_batches=2, frames_per_batch=4, n_objects=700)
    o, g = _stress_pair(oracle, sc)
    compare_maps(g, o)
    for b in range(2):
        frames = margin_filter(o.clone, sc.batch(b), sc.cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, sc.cfg.dtype)
        compare_call(g, o)
        a, n, _, st = g.last_assoc()
        assert 0.4 < st["matches"] / st["n_det"] < 0.6
    compare_maps(g, o)


def test_config4_full_size_sampled_against_oracle(oracle):
    """configs[4] at the size and in the launch configuration bench.py times: 50,000 imported objects (~1e8
    voxels), 16-frame batches of 1,600 detections.  The oracle cannot hold the whole map in a std::map within
    the test budget, so (R2: every detection is scored against the entry snapshot, independently of the other
    detections of the call) sampled frames are integrated one by one into clones of an oracle map that holds
    every descriptor and the voxels of the objects those frames can touch; per detection the decision, score,
    voxel set, pixel count, box and overlap histogram must agree.  Whole-map invariants (P9, P12) are then
    checked on the GPU state after two batches."""
    from paper_2606_15476_b200.binding import OBJECT_DTYPE
    F, DET, N0, WITH_VOX = 16, 100, 50000, 2000
    sc = S.StressScene(n_batches=2, frames_per_batch=F, n_objects=N0)
    cfg = sc.cfg
    ijk, owner, n_vox, desc = sc.build_map()
    keys = pack_key(ijk[:, 0], ijk[:, 1], ijk[:, 2])
    del ijk
    objs = np.zeros(len(n_vox), OBJECT_DTYPE)
    objs["id"], objs["n_voxels"], objs["n_obs"], objs["best_frame"], objs["best_det"] = np.arange(len(n_vox)), n_vox, 1, -1, -1
    g = FarmMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, H=cfg.H, W=cfg.W, dtype=cfg.dtype,
                max_objects=N0 + 3 * F * DET, max_voxels=int(len(keys) * 1.05) + 2000000,
                max_blocks=len(keys) // 16 + 100000, max_det_per_call=F * DET, max_frames_per_call=F,
                max_pairs_per_call=1 << 21)
    g.import_(objs, desc, keys, owner)
    # oracle: all descriptors, voxels of the first WITH_VOX objects (the targets of batches 0 and 1 are 0..1599)
    o = oracle.OracleMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, cfg.dtype, cfg.H, cfg.W)
    sel = owner < WITH_VOX
    objs_o = objs.copy()
    objs_o["n_voxels"] = np.where(np.arange(len(n_vox)) < WITH_VOX, n_vox, 0)
    assert o.import_(objs_o, desc, keys[sel], owner[sel]) == 0
    n_keys = len(keys)
    del keys, owner, sel

    frames = sc.batch(0)
    gpu_integrate(g, frames, cfg.dtype)
    ag, ng, bg, stg = g.last_assoc()
    offg, keyg, npxg, boxg = g.debug_last_voxels()
    og, objg, cntg = g.debug_last_overlaps()
    assert int(stg["n_det"]) == F * DET and int(stg["matches"]) == F * DET // 2 and int(stg["spawns"]) == F * DET // 2
    assert int(stg["unique_voxels"]) == int(offg[-1])
    checked = 0
    for f in (0, 3, 7, 10, 12, 15):
        oc = o.clone()
        integrate_frames(oc, [frames[f]])
        ao, no, bo, so, sto = oc.last_assoc()
        offo, keyo, npxo, boxo = oc.last_voxels()
        oo, objo, cnto = oc.last_overlaps()
        for d in range(DET):
            j = f * DET + d
            assert npxg[j] == npxo[d]
            assert np.array_equal(np.sort(keyg[offg[j]:offg[j + 1]]), keyo[offo[d]:offo[d + 1]])      # bit-exact V_d
            assert np.array_equal(boxg[j], boxo[d])
            order = np.argsort(objg[og[j]:og[j + 1]])
            assert np.array_equal(objg[og[j]:og[j + 1]][order], objo[oo[d]:oo[d + 1]])
            assert np.array_equal(cntg[og[j]:og[j + 1]][order], cnto[oo[d]:oo[d + 1]])
            assert abs(float(bg[j]) - float(bo[d])) <= TOL
            near = abs(float(bo[d]) - cfg.tau) <= 1e-3 or (not no[d] and float(bo[d]) - float(so[d]) <= 1e-3)
            if near:
                continue                                   # BASELINE.json: decisions are compared at margins > 1e-3
            assert ng[j] == no[d]
            if not no[d]:
                assert ag[j] == ao[d]                      # matched: same object; spawned ids depend on the whole call
            checked += 1
    assert checked > 500
    # new ids in detection index order (R20)
    new_ids = ag[ng.astype(bool)]
    assert np.array_equal(new_ids, N0 + np.arange(len(new_ids)))

    gpu_integrate(g, sc.batch(1), cfg.dtype)
    _, _, _, st1 = g.last_assoc()
    assert int(st1["matches"]) == F * DET // 2 and int(st1["spawns"]) == F * DET // 2
    objs_g, _, _, _ = g.read(voxels=False, descriptors=False)
    n_obj, n_voxels_now = g.counts()
    assert n_obj == len(objs_g) == N0 + 2 * (F * DET // 2)                                   # P12
    assert int(objs_g["n_obs"].astype(np.int64).sum()) == N0 + 2 * F * DET                   # P12
    assert int(objs_g["n_voxels"].astype(np.int64).sum()) == n_voxels_now                    # P9
    assert n_voxels_now > n_keys
    assert np.array_equal(objs_g["n_voxels"][5000:N0], n_vox[5000:N0])                       # untouched fillers
    tot = g.sync()
    assert int(tot["frames"]) == 2 * F and int(tot["matches"]) == F * DET


def _compare_gaussians(g, o):
    mu_o, cov_o, hell_o = o.last_gaussians()
    mu_g, cov_g, hell_g = g.last_gaussians()
    assert np.abs(mu_g - mu_o).max(initial=0) <= TOL
    assert np.abs(cov_g - cov_o).max(initial=0) <= TOL
    assert np.array_equal(hell_g < 0, hell_o < 0)
    assert np.abs(hell_g - hell_o).max(initial=0) <= TOL
    return hell_o


@pytest.mark.parametrize("cfg_id,n_calls,per_call", [(0, 20, 1), (1, 4, 1), (0, 4, 3)])
def test_gaussian_geometry_matches_oracle(oracle, cfg_id, n_calls, per_call):
    """Rules G1-G4: per-detection Gaussians, Hellinger distance of every match and the
    sufficient-statistics entity Gaussians, carried beside the unchanged voxel rule."""
    cfg = S.get_config(cfg_id)
    sc = S.BoxScene(cfg)
    o, g = make_pair(oracle, cfg, gaussian=1)
    k, n_match = 0, 0
    for _ in range(n_calls):
        frames = margin_filter(o.clone, [sc.frame(k + i) for i in range(per_call)], cfg.tau)
        k += per_call
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o, check_sets=False)
        hell = _compare_gaussians(g, o)
        n_match += int((hell >= 0).sum())
        assert ((hell < 0) | (hell <= 1.0)).all()
    assert n_match > 3
    compare_maps(g, o, voxels=False)
    w_o, mu_o, cov_o = o.read_gaussians()
    w_g, mu_g, cov_g = g.read_gaussians()
    assert np.array_equal(w_g, w_o)                                # point counts: exact
    assert np.abs(mu_g - mu_o).max(initial=0) <= TOL and np.abs(cov_g - cov_o).max(initial=0) <= TOL


def test_gaussian_mini_stress_and_off_by_default(oracle):
    sc = S.StressScene(n_batches=2, frames_per_batch=4, n_objects=700)
    o, g = _stress_pair(oracle, sc, gaussian=1)
    for b in range(2):
        frames = margin_filter(o.clone, sc.batch(b), sc.cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, sc.cfg.dtype)
        compare_call(g, o, check_sets=False)
        hell = _compare_gaussians(g, o)
        assert (hell < 0).all()                                     # imported objects carry no Gaussian (weight 0)
    w_o, mu_o, cov_o = o.read_gaussians()
    w_g, mu_g, cov_g = g.read_gaussians()
    assert np.array_equal(w_g, w_o) and np.abs(mu_g - mu_o).max() <= TOL and np.abs(cov_g - cov_o).max() <= TOL
    from paper_2606_15476_b200.binding import FarmError
    _, g2 = make_pair(oracle, S.get_config(0))
    with pytest.raises(FarmError):
        g2.read_gaussians()


def test_covisibility_bitset_matches_oracle(oracle):
    """Rule C1 (PAPER.md:354 step 7): the N x ceil(N/64) bitset of co-observed entity pairs, bit-exact, on batched
    config-0 calls and on the mini stress scene (imported map, 400 detections per call)."""
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    o, g = make_pair(oracle, cfg, covisibility=1)
    for k in range(0, 18, 3):
        frames = margin_filter(o.clone, [sc.frame(k + i) for i in range(3)], cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o, check_sets=False)
        assert np.array_equal(g.read_covisibility(), o.read_covisibility())
    assert int(np.unpackbits(o.read_covisibility().view(np.uint8)).sum()) > 20
    sc4 = S.StressScene(n_batches=2, frames_per_batch=4, n_objects=700)
    o4, g4 = _stress_pair(oracle, sc4, covisibility=1)
    for b in range(2):
        frames = margin_filter(o4.clone, sc4.batch(b), sc4.cfg.tau)
        integrate_frames(o4, frames)
        gpu_integrate(g4, frames, sc4.cfg.dtype)
        compare_call(g4, o4, check_sets=False)
    ro, rg = o4.read_covisibility(), g4.read_covisibility()
    assert np.array_equal(rg, ro)


def test_host_buffer_entry_point_matches_device_path(oracle):
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    o, g = make_pair(oracle, cfg)
    from helpers import stack_frames
    for k in range(5):
        fr = sc.frame(k)
        integrate_frames(o, [fr])
        depth, mask, K, T, desc, n_det = stack_frames([fr])
        g.integrate_batch_host(1, depth, mask, K, T, np.ascontiguousarray(desc), n_det)
        compare_call(g, o)
    compare_maps(g, o)


def test_pipelined_host_calls_with_async_result_reads(oracle):
    """Back-to-back host-buffer calls (copy of call t+1 overlaps the kernels of call t, two staging sets) with
    non-blocking result reads: every call's results and the final map equal the oracle's."""
    import torch
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    o, g = make_pair(oracle, cfg)
    from helpers import stack_frames
    n_calls, expected, got, keep = 7, [], [], []
    for k in range(n_calls):
        fr = sc.frame(k)
        integrate_frames(o, [fr])
        ao, no, bo, so, sto = o.last_assoc()
        expected.append((ao.copy(), no.copy(), bo.copy()))
        depth, mask, K, T, desc, n_det = stack_frames([fr])
        pins = [torch.from_numpy(np.ascontiguousarray(x)).pin_memory() for x in (depth, mask.view(np.int16), K, T, desc)]
        keep.append(pins)                                   # host buffers stay alive until the sync
        g.integrate_batch_host(1, pins[0], pins[1], pins[2], pins[3], pins[4], n_det)
        M = int(n_det.sum())
        res = (torch.empty(M, dtype=torch.int32).pin_memory(), torch.empty(M, dtype=torch.uint8).pin_memory(),
               torch.empty(M, dtype=torch.float32).pin_memory())
        g.last_assoc_async(res[0], res[1], res[2], None)
        got.append(res)
    g.sync()
    for (ao, no, bo), (ag, ng, bg) in zip(expected, got):
        assert np.array_equal(ag.numpy(), ao)
        assert np.array_equal(ng.numpy(), no)
        assert np.abs(bg.numpy() - bo).max(initial=0) <= 1e-4
    compare_maps(g, o)


def test_tile_queue_overflow_every_pixel_its_own_voxel(oracle):
    """Degenerate case: (almost) every pixel of a tile lands in its own voxel, more distinct pairs per tile
    than the lift kernel's shared-memory queue holds (overflow goes straight to the global queue)."""
    class Cfg:
        voxel, D, w_geo, w_sem, tau, dtype = 0.01, 8, 0.5, 0.5, 0.5, 0
    H, W = 24, 256
    g0 = np.random.default_rng(11)
    o, g = make_pair(oracle, Cfg, H=H, W=W)
    K = np.array([[100, 0, 128], [0, 100, 12], [0, 0, 1]], np.float32)
    for it in range(2):
        depth = (1.0 + 4.0 * g0.random((H, W))).astype(np.float32)
        mask = np.ones((H, W), np.uint16)
        mask[:, 128:] = 2
        fr = S.Frame(depth, mask, K, np.eye(4, dtype=np.float32), unit_rows(2, 8, 5), 2, np.zeros(2, np.int64))
        integrate_frames(o, [fr])
        gpu_integrate(g, [fr], 0)
        compare_call(g, o)
        _, _, _, st = g.last_assoc()
        assert st["unique_voxels"] > 0.9 * H * W
    compare_maps(g, o)


def test_many_detections_in_one_tile_label_slots_overflow(oracle):
    """Every pixel of a 64x16 tile carries its own detection (hundreds of labels per tile): more than the lift
    kernel's 32 per-tile label slots, threads whose 8 pixels straddle 8 detections (stray-pixel path), and
    records that bypass the tile table."""
    class Cfg:
        voxel, D, w_geo, w_sem, tau, dtype = 0.05, 8, 0.5, 0.5, 0.5, 0
    H, W = 32, 128
    n_det = 300
    g0 = np.random.default_rng(3)
    o, g = make_pair(oracle, Cfg, H=H, W=W, max_det_per_call=512)
    K = np.array([[100, 0, 64], [0, 100, 16], [0, 0, 1]], np.float32)
    for it in range(2):
        depth = (1.0 + 2.0 * g0.random((H, W))).astype(np.float32)
        mask = (g0.integers(0, n_det + 40, size=(H, W))).astype(np.uint16)      # also labels > n_det (ignored, R3) and 0
        mask[4:8, 16:48] = 7                                                      # one block of a single label as well
        fr = S.Frame(depth, mask, K, np.eye(4, dtype=np.float32), unit_rows(n_det, 8, 9 + it), n_det, np.zeros(n_det, np.int64))
        integrate_frames(o, [fr])
        gpu_integrate(g, [fr], 0)
        compare_call(g, o)
        _, _, _, st = g.last_assoc()
        assert st["ignored_pixels"] > 0
    compare_maps(g, o)


@pytest.mark.parametrize("n_same", [5, 90])
def test_many_detections_fuse_into_one_entity(oracle, n_same):
    """several detections may claim one entity and all fuse into it.  n_same detections of one call
    match the same object: member lists that fit the merge kernel's shared-memory list (5) and that do not (90)."""
    class Cfg:
        voxel, D, w_geo, w_sem, tau, dtype = 0.25, 16, 0.5, 0.5, 0.5, 0
    H, W = 96, 128
    I4 = np.eye(4, dtype=np.float32)
    base = unit_rows(1, 16, 2)
    o, g = make_pair(oracle, Cfg, H=H, W=W, max_det_per_call=128)
    # call 1: one detection creates the object; call 2: n_same detections over the same voxels with nearby descriptors
    px = [(u, v, 2.0, 1) for v in range(40, 48) for u in range(60, 76)]
    d1, m1 = hand_frame(H, W, px)
    fr1 = S.Frame(d1, m1, pow2_K(), I4, base, 1, np.zeros(1, np.int64))
    rng = np.random.default_rng(4)
    desc = base + 0.02 * rng.standard_normal((n_same, 16)).astype(np.float32)
    desc /= np.linalg.norm(desc, axis=1, keepdims=True)
    px2 = [(60 + (k % 16), 40 + k // 16, 2.0, k + 1) for k in range(n_same)]         # one pixel per detection
    d2, m2 = hand_frame(H, W, px2)
    fr2 = S.Frame(d2, m2, pow2_K(), I4, desc.astype(np.float32), n_same, np.zeros(n_same, np.int64))
    for fr in (fr1, fr2, fr2):
        integrate_frames(o, [fr])
        gpu_integrate(g, [fr], 0)
        compare_call(g, o)
    a, n, _, _ = g.last_assoc()
    assert (a == 0).all() and not n.any()
    objs, _, _, _ = g.read()
    assert len(objs) == 1 and objs["n_obs"][0] == 1 + 2 * n_same
    compare_maps(g, o)


@pytest.mark.parametrize("dtype,D", [(1, 20), (2, 36), (0, 7)])
def test_descriptor_lengths_off_the_vector_paths(oracle, dtype, D):
    """D not a multiple of 8 (no 128-bit row loads, no TMA: CUDA-core similarity) for f16 / bf16 / f32."""
    cfg = S.get_config(0)

    class Cfg:
        voxel, w_geo, w_sem, tau = cfg.voxel, cfg.w_geo, cfg.w_sem, cfg.tau
    Cfg.D, Cfg.dtype = D, dtype
    sc = S.BoxScene(cfg)
    o, g = make_pair(oracle, Cfg, H=cfg.H, W=cfg.W)
    rng = np.random.default_rng(8)
    basis = unit_rows(64, D, 1)
    for k in range(6):
        fr = sc.frame(k)
        # re-describe the frame's detections with D-long descriptors tied to the underlying box id
        ids = np.asarray(fr.box_ids) % 64
        d = basis[ids[:fr.n_det]] + 0.01 * rng.standard_normal((fr.n_det, D)).astype(np.float32)
        d /= np.linalg.norm(d, axis=1, keepdims=True)
        fr2 = S.Frame(fr.depth, fr.mask, fr.K, fr.T, S.to_storage(d.astype(np.float32), dtype), fr.n_det, np.zeros(fr.n_det, np.int64))
        frames = margin_filter(o.clone, [fr2], cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, dtype)
        compare_call(g, o)
    compare_maps(g, o)


def test_epoch_tag_wraparound_after_65534_calls(oracle):
    """The per-call scratch tables are never cleared: their keys carry a 16-bit call epoch, and the tables are
    wiped once when it wraps.  65,700 calls that keep re-observing the same two objects must leave exactly the
    oracle's map, and the calls right after the wrap must still report exact voxel sets and overlaps."""
    class Cfg:
        voxel, D, w_geo, w_sem, tau, dtype = 0.25, 4, 0.5, 0.5, 0.5, 0
    H, W = 16, 32
    I4 = np.eye(4, dtype=np.float32)
    e = np.eye(4, dtype=np.float32)
    o, g = make_pair(oracle, Cfg, H=H, W=W)
    px = [(u, v, 2.0, 1) for v in range(4, 8) for u in range(4, 12)] + [(u, v, 3.0, 2) for v in range(9, 13) for u in range(16, 28)]
    depth, mask = hand_frame(H, W, px)
    K = np.array([[16, 0, 16], [0, 16, 8], [0, 0, 1]], np.float32)
    fr = S.Frame(depth, mask, K, I4, np.ascontiguousarray(e[:2]), 2, np.zeros(2, np.int64))
    d = upload([fr], 0)
    n_calls, o_calls = 65700, 0
    for k in range(n_calls):
        g.integrate_batch(1, d["depth"], d["mask"], d["K"], d["T"], d["desc"], d["n_det"])
        if k in (0, 1, 65532, 65533, 65534, 65535, 65536, n_calls - 1):
            while o_calls <= k:                                      # bring the oracle to the same call
                integrate_frames(o, [fr])
                o_calls += 1
            compare_call(g, o)
    compare_maps(g, o)
    objs, _, _, _ = g.read()
    assert len(objs) == 2 and objs["n_obs"][0] == n_calls



def test_block_table_and_scratch_overflow_are_loud(oracle):
    """Data-dependent capacity failures never truncate silently: too few voxel blocks, or too few per-call pair
    slots, set the sticky device error that the next sync / read / last_assoc returns as FARM_ERR_CAPACITY."""
    from paper_2606_15476_b200 import FarmError
    H, W = 24, 256
    g0 = np.random.default_rng(11)
    depth = (1.0 + 4.0 * g0.random((H, W))).astype(np.float32)       # ~ every pixel in its own voxel block
    mask = np.ones((H, W), np.uint16)
    K = np.array([[100, 0, 128], [0, 100, 12], [0, 0, 1]], np.float32)
    fr = S.Frame(depth, mask, K, np.eye(4, dtype=np.float32), unit_rows(1, 8, 5), 1, np.zeros(1, np.int64))
    g = FarmMap(0.01, 8, 0.5, 0.5, 0.5, H=H, W=W, max_blocks=64)      # 1024 block slots for ~6000 blocks
    gpu_integrate(g, [fr], 0)
    with pytest.raises(FarmError) as ei:
        g.sync()
    assert ei.value.code == -3 and "voxel table full" in str(ei.value)
    with pytest.raises(FarmError):                                   # sticky
        g.read()
    g2 = FarmMap(0.01, 8, 0.5, 0.5, 0.5, H=H, W=W, max_pairs_per_call=1024)
    gpu_integrate(g2, [fr], 0)
    with pytest.raises(FarmError) as ei:
        g2.last_assoc()
    assert ei.value.code == -3


@pytest.mark.parametrize("overlap,sim_path", [(0, 0), (2, 0), (3, 0), (1, 1), (1, 2)])
def test_stream_orders_and_similarity_paths_give_the_same_map(oracle, overlap, sim_path):
    """The launch orders (FARM_OPT_OVERLAP 0 / 2 / 3 beside the default 1) and the forced similarity paths
    (CUDA-core FMA, tcgen05) are different schedules of the same rules: every one must reproduce the oracle."""
    cfg = S.get_config(1)
    sc = S.BoxScene(cfg)
    o, g = make_pair(oracle, cfg, overlap=overlap, sim_path=sim_path)
    for k in range(20, 28):
        frames = margin_filter(o.clone, [sc.frame(k)], cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o)
    compare_maps(g, o)
