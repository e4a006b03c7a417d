"""Pins of the CPU oracle against what the paper, BASELINE.json and the mathematics fix (P1-P12).

The paper prints no worked numeric example for the mapping path, so the pins are closed
forms on hand-placed points, brute force on tiny inputs, library routines for the special cases that
reduce to one, and invariants.  None of the expected values below comes from the oracle or the CUDA path.
"""
import numpy as np
import pytest
import torch

from helpers import (KEY_EMPTY, hand_frame, integrate_frames, pack_key, pow2_K, unit_rows, unpack_key)
from paper_2606_15476_b200 import scenes as S

H, W = 96, 128
I4 = np.eye(4, dtype=np.float32)


def new_map(oracle, vs=0.25, D=4, w_geo=0.5, w_sem=0.5, tau=0.5, dtype=0, H_=H, W_=W, **kw):
    return oracle.OracleMap(vs, D, w_geo, w_sem, tau, dtype, H_, W_, **kw)


def translate(x, y, z):
    T = I4.copy()
    T[:3, 3] = [x, y, z]
    return T


# ------------------------------------------------------------------------------------------------ P1
def test_P1_backprojection_closed_form(oracle):
    """R5.  fx=fy=128, cx=64, cy=48: pixel (96,48), z=2 -> (0.5, 0, 2) exactly (power-of-two intrinsics)."""
    m = new_map(oracle)
    depth, mask = hand_frame(H, W, [(96, 48, 2.0, 1), (64, 48, 3.0, 1), (32, 16, 4.0, 1)])
    xyz, _ = m.backproject(depth, mask, pow2_K(), I4, 1)
    assert tuple(xyz[48, 96]) == (0.5, 0.0, 2.0)
    assert tuple(xyz[48, 64]) == (0.0, 0.0, 3.0)            # principal point -> (0,0,z)
    assert tuple(xyz[16, 32]) == (-1.0, -1.0, 4.0)          # (32-64)/128*4, (16-48)/128*4
    assert np.isnan(xyz[0, 0]).all()                        # unmasked pixel -> NaN
    xyz, _ = m.backproject(depth, mask, pow2_K(), translate(1, 2, 3), 1)
    assert tuple(xyz[48, 96]) == (1.5, 2.0, 5.0)
    # 90 degrees about the camera z axis: (x,y,z) -> (-y, x, z)
    Rz = I4.copy()
    Rz[:3, :3] = [[0, -1, 0], [1, 0, 0], [0, 0, 1]]
    xyz, _ = m.backproject(depth, mask, pow2_K(), Rz, 1)
    assert tuple(xyz[16, 32]) == (1.0, -1.0, 4.0)
    assert tuple(xyz[48, 96]) == (0.0, 0.5, 2.0)


def test_P1_depth_is_camera_z_not_ray_length(oracle):
    """A transposed rotation or a ray-length reading of depth fails here: camera looking along world +x."""
    m = new_map(oracle)
    T = S.pose_from_yaw(np.array([1.0, 2.0, 1.5]), 0.0)     # right=(0,-1,0) down=(0,0,-1) fwd=(1,0,0)
    depth, mask = hand_frame(H, W, [(96, 16, 2.0, 1)])
    xyz, _ = m.backproject(depth, mask, pow2_K(), T, 1)
    # camera point (0.5,-0.5,2) -> world = pos + 0.5*right - 0.5*down + 2*fwd = (3, 1.5, 2.0)
    assert tuple(xyz[16, 96]) == (3.0, 1.5, 2.0)


def test_P2_project_backproject_round_trip(oracle):
    """R5.  World points on an exactly representable lattice project to integer pixels and come back equal."""
    m = new_map(oracle)
    T = translate(0.5, -0.25, 1.0)
    pts = []
    for z in (1.0, 2.0, 4.0):
        for u in (0, 17, 64, 127):
            for v in (0, 48, 95):
                pts.append((u, v, z))
    depth, mask = hand_frame(H, W, [(u, v, z, 1) for u, v, z in pts if z == 2.0])
    xyz, _ = m.backproject(depth, mask, pow2_K(), T, 1)
    for u, v, z in pts:
        if z != 2.0:
            continue
        Xc = np.array([(u - 64) / 128 * z, (v - 48) / 128 * z, z])   # exact in binary
        Xw = Xc + np.array([0.5, -0.25, 1.0])
        # forward projection of the world point lands on the integer pixel
        pc = Xw - np.array([0.5, -0.25, 1.0])
        assert 128 * pc[0] / pc[2] + 64 == u and 128 * pc[1] / pc[2] + 48 == v
        assert np.array_equal(xyz[v, u], Xw.astype(np.float32))


# ------------------------------------------------------------------------------------------------ P3
def test_P3_voxel_keys(oracle):
    """R6.  floor (not truncation), boundaries, packing, range."""
    m = new_map(oracle, vs=0.25)
    depth, mask = hand_frame(H, W, [(96, 48, 2.0, 1)])
    _, keys = m.backproject(depth, mask, pow2_K(), I4, 1)
    assert keys[48, 96] == pack_key(2, 0, 8)                # (0.5,0,2)/0.25
    _, keys = m.backproject(depth, mask, pow2_K(), translate(1, 2, 3), 1)
    assert keys[48, 96] == pack_key(6, 8, 20)               # (1.5,2,5)/0.25
    assert keys[0, 0] == KEY_EMPTY
    # negative coordinate: X = -0.0078125 with voxel 0.05 -> index -1 (floor), truncation would give 0
    m2 = new_map(oracle, vs=0.05)
    depth, mask = hand_frame(H, W, [(63, 48, 1.0, 1)])
    xyz, keys = m2.backproject(depth, mask, pow2_K(), I4, 1)
    assert xyz[48, 63, 0] == np.float32(-1 / 128)
    ix, iy, iz = unpack_key(keys[48, 63])
    # the index is floor(fp32(X * fp32(1/0.05))) -- evaluated here in the same precision the rule states
    inv = np.float32(1.0) / np.float32(0.05)
    assert (ix, iy) == (-1, 0) and iz == int(np.floor(np.float32(1.0) * inv))
    # a point exactly on a voxel boundary k*vs belongs to voxel k (vs = 0.25 is exact)
    m3 = new_map(oracle, vs=0.25)
    depth, mask = hand_frame(H, W, [(80, 48, 2.0, 1), (48, 48, 2.0, 1)])    # X = +0.25, -0.25
    _, keys = m3.backproject(depth, mask, pow2_K(), I4, 1)
    assert keys[48, 80] == pack_key(1, 0, 8) and keys[48, 48] == pack_key(-1, 0, 8)


def test_P3_key_range_and_pack_round_trip(oracle):
    """R6: indices in [-2^20, 2^20) are kept, outside dropped and counted; pack/unpack round trip at the edge."""
    lim = 1 << 20
    for idx in (-lim, lim - 1, 0, -1):
        k = pack_key(idx, -idx - 1 if idx >= 0 else -idx - 1, idx)
        assert unpack_key(k)[0] == idx and unpack_key(k)[2] == idx
    m = new_map(oracle, vs=1.0)
    # X = z * (u-64)/128 with T translating to just inside / outside the range
    depth, mask = hand_frame(H, W, [(64, 48, 1.0, 1), (65, 48, 1.0, 2)])
    T_in = translate(float(lim - 1), 0, 0)       # X = 2^20-1 -> valid (index 2^20-1)
    _, keys = m.backproject(depth, mask, pow2_K(), T_in, 2)
    assert keys[48, 64] == pack_key(lim - 1, 0, 1)
    T_out = translate(float(lim), 0, 0)          # X = 2^20 -> out of range
    _, keys = m.backproject(depth, mask, pow2_K(), T_out, 2)
    assert keys[48, 64] == KEY_EMPTY
    T_neg = translate(float(-lim), 0, 0)         # X = -2^20 exactly -> index -2^20 valid
    _, keys = m.backproject(depth, mask, pow2_K(), T_neg, 2)
    assert keys[48, 64] == pack_key(-lim, 0, 1)
    # integrate: the out-of-range detection is dropped and counted, and it is skipped (R8)
    desc = unit_rows(2, 4)
    m.integrate(depth, mask, pow2_K(), T_out, desc, 2)
    assoc, is_new, _, _, st = m.last_assoc()
    assert st["dropped_points"] == 2 and st["valid_points"] == 0
    assert list(assoc) == [-1, -1] and st["skipped"] == 2


def test_R4_depth_validity_and_R3_labels(oracle):
    m = new_map(oracle, z_min=0.5, z_max=3.0)
    px = [(10, 10, 0.0, 1), (11, 10, -1.0, 1), (12, 10, np.nan, 1), (13, 10, np.inf, 1), (14, 10, 0.5, 1),
          (15, 10, 3.0, 1), (16, 10, 3.0001, 1), (17, 10, 1.0, 3), (18, 10, 1.0, 2)]
    depth, mask = hand_frame(H, W, px)
    xyz, keys = m.backproject(depth, mask, pow2_K(), I4, 2)
    valid = ~np.isnan(xyz[10, :, 0])
    assert list(np.nonzero(valid)[0]) == [15, 18]           # z in (z_min, z_max], label <= n_det
    m.integrate(depth, mask, pow2_K(), I4, unit_rows(2, 4), 2)
    _, _, _, _, st = m.last_assoc()
    assert st["ignored_pixels"] == 1 and st["valid_points"] == 2


# ------------------------------------------------------------------------------------------------ P4/P5
def _scene_run(oracle, n_frames=6):
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    m = oracle.OracleMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, cfg.dtype, cfg.H, cfg.W)
    return cfg, sc, m


def test_P4_detection_sets_independent_loop(oracle):
    """R7: |V_d| equals the size of a set built by a second loop over the debug per-pixel keys; the pixel
    counts per key add up to n_px_d."""
    cfg, sc, m = _scene_run(oracle)
    for k in range(3):
        fr = sc.frame(k)
        m.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
        off, keys, n_px, box = m.last_voxels()
        xyz, pk = m.backproject(fr.depth, fr.mask, fr.K, fr.T, fr.n_det)
        for d in range(fr.n_det):
            sel = (fr.mask == d + 1) & (pk != KEY_EMPTY)
            uniq, cnt = np.unique(pk[sel], return_counts=True)
            assert np.array_equal(uniq, keys[off[d]:off[d + 1]])
            assert cnt.sum() == n_px[d]
            pts = xyz[sel]
            assert np.array_equal(box[d, :3], pts.min(0)) and np.array_equal(box[d, 3:], pts.max(0))


def test_P5_overlap_brute_force(oracle):
    """R9: c[d][o] against explicit python set intersection over all (d, o) pairs."""
    cfg, sc, m = _scene_run(oracle)
    for k in range(8):
        fr = sc.frame(k)
        _, _, keys_before, owners_before = m.read()
        m.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
        off, keys, _, _ = m.last_voxels()
        ooff, oobj, ocnt = m.last_overlaps()
        N = int(owners_before.max()) + 1 if len(owners_before) else 0
        sets = [set(keys_before[owners_before == o].tolist()) for o in range(N)]
        for d in range(fr.n_det):
            Vd = set(keys[off[d]:off[d + 1]].tolist())
            expect = {o: len(Vd & sets[o]) for o in range(N) if len(Vd & sets[o])}
            got = dict(zip(oobj[ooff[d]:ooff[d + 1]].tolist(), ocnt[ooff[d]:ooff[d + 1]].tolist()))
            assert got == expect
    assert N > 0


# ------------------------------------------------------------------------------------------------ P6
def _obj(n_voxels, n_obs=1):
    o = np.zeros(1, dtype=[("id", "<i4"), ("n_voxels", "<u4"), ("n_obs", "<u4"), ("aabb_min", "<f4", 3),
                           ("aabb_max", "<f4", 3), ("best_frame", "<i4"), ("best_det", "<i4"),
                           ("best_pixels", "<u4"), ("best_cam_pos", "<f4", 3), ("n_points", "<u8")])
    o["n_voxels"], o["n_obs"] = n_voxels, n_obs
    return o


def _four_voxel_detection():
    # z=2, v=48: u=64,80,96,112 -> X = 0, .25, .5, .75 -> voxels (0..3, 0, 8) at voxel 0.25
    return hand_frame(H, W, [(64, 48, 2.0, 1), (80, 48, 2.0, 1), (96, 48, 2.0, 1), (112, 48, 2.0, 1)])


def test_P6_score_hand_case_and_strict_threshold(oracle):
    """R10/R17/R18: |V_d|=4, |V_o|=8, c=3, cos=1, w=.5/.5 -> 0.875 > 0.5 match;  c=0, cos=1 -> 0.5, NOT > 0.5."""
    e1 = np.array([[1, 0, 0, 0]], np.float32)
    own = [(0, 0, 8), (1, 0, 8), (2, 0, 8)] + [(50 + i, 0, 0) for i in range(5)]
    keys = np.array([pack_key(*k) for k in own], np.uint64)
    m = new_map(oracle)
    assert m.import_(np.asarray(_obj(8), oracle.OBJECT_DTYPE), e1, keys, np.zeros(8, np.uint32)) == 0
    depth, mask = _four_voxel_detection()
    m.integrate(depth, mask, pow2_K(), I4, e1, 1)
    assoc, is_new, best, _, _ = m.last_assoc()
    assert assoc[0] == 0 and is_new[0] == 0 and best[0] == np.float32(0.875)
    # no overlap, identical descriptor: score = 0.5 exactly, strict '>' -> spawn
    m = new_map(oracle)
    far = np.array([pack_key(50 + i, 0, 0) for i in range(8)], np.uint64)
    m.import_(np.asarray(_obj(8), oracle.OBJECT_DTYPE), e1, far, np.zeros(8, np.uint32))
    m.integrate(depth, mask, pow2_K(), I4, e1, 1)
    assoc, is_new, best, _, _ = m.last_assoc()
    assert best[0] == np.float32(0.5) and is_new[0] == 1 and assoc[0] == 1
    # min(|V_d|,|V_o|) picks the object side when it is smaller: |V_o|=2, c=2 -> g=1
    m = new_map(oracle)
    m.import_(np.asarray(_obj(2), oracle.OBJECT_DTYPE), e1, keys[:2], np.zeros(2, np.uint32))
    m.integrate(depth, mask, pow2_K(), I4, np.array([[0, 1, 0, 0]], np.float32), 1)
    assoc, is_new, best, _, _ = m.last_assoc()
    assert best[0] == np.float32(0.5) and is_new[0] == 1          # g=1, cos=0 -> 0.5, spawn


def test_R18_argmax_ties_go_to_lowest_id(oracle):
    e1 = np.array([[1, 0, 0, 0]], np.float32)
    objs = np.concatenate([_obj(1), _obj(1)])
    keys = np.array([pack_key(0, 0, 8), pack_key(1, 0, 8)], np.uint64)
    m = new_map(oracle, w_geo=1.0, w_sem=0.0, tau=0.1)
    m.import_(np.asarray(objs, oracle.OBJECT_DTYPE), np.repeat(e1, 2, 0), keys, np.array([0, 1], np.uint32))
    depth, mask = _four_voxel_detection()
    m.integrate(depth, mask, pow2_K(), I4, e1, 1)          # c=1/min(4,1)=1 for both objects -> tie
    assoc, _, best, second, _ = m.last_assoc()
    assert assoc[0] == 0 and best[0] == 1.0 and second[0] == 1.0


# ------------------------------------------------------------------------------------------------ P7
def test_P7_cosine(oracle):
    """R15: closed forms by hand and the oracle's similarity values against a library GEMM."""
    f = unit_rows(1, 16, 3)[0]
    assert abs(oracle.cosine(f, f) - 1.0) < 1e-7
    e = np.eye(4, dtype=np.float32)
    assert oracle.cosine(e[0], e[1]) == 0.0
    assert abs(oracle.cosine(np.array([3, 4], np.float32), np.array([4, 3], np.float32)) - 24 / 25) < 1e-7
    assert oracle.cosine(np.array([1, 2], np.float32), np.array([-2, -4], np.float32)) == -1.0   # clamp side
    assert oracle.cosine(np.zeros(4, np.float32), e[0]) == 0.0                                   # zero norm
    g = np.random.default_rng(5)
    A = g.standard_normal((7, 96)).astype(np.float32)
    B = g.standard_normal((11, 96)).astype(np.float32)
    ref = (A.astype(np.float64) @ B.astype(np.float64).T) / np.outer(np.linalg.norm(A.astype(np.float64), axis=1),
                                                                     np.linalg.norm(B.astype(np.float64), axis=1))
    got = np.array([[oracle.cosine(a, b) for b in B] for a in A])
    assert np.abs(got - ref).max() <= 1e-6


@pytest.mark.parametrize("dtype", [0, 1, 2])
def test_P7_dense_similarity_in_situ_vs_library_gemm(oracle, dtype):
    """R14-R16, R19: with no voxel overlap best_score = w_sem * max_o cos(a_d, shadow_o); operands are the
    storage-dtype values.  Checked against torch matmul on the same converted operands."""
    D, N, Mdet = 32, 9, 3
    g = np.random.default_rng(11)
    objdesc = unit_rows(N, D, 21)
    objs = np.concatenate([_obj(1) for _ in range(N)])
    keys = np.array([pack_key(500 + i, 0, 0) for i in range(N)], np.uint64)
    m = new_map(oracle, D=D, dtype=dtype)
    m.import_(np.asarray(objs, oracle.OBJECT_DTYPE), objdesc, keys, np.arange(N, dtype=np.uint32))
    det = unit_rows(Mdet, D, 22)
    det_st = S.to_storage(det, dtype)
    depth, mask = hand_frame(H, W, [(64 + 16 * d, 48, 2.0, d + 1) for d in range(Mdet)])
    m.integrate(depth, mask, pow2_K(), I4, det_st, Mdet)
    _, is_new, best, _, _ = m.last_assoc()
    tdt = {0: torch.float32, 1: torch.float16, 2: torch.bfloat16}[dtype]
    A = torch.from_numpy(det).to(tdt).to(torch.float64)                   # library conversion, RNE
    Bm = torch.from_numpy(objdesc).to(tdt).to(torch.float64)
    cos = (A @ Bm.T) / torch.outer(A.norm(dim=1), Bm.norm(dim=1))
    ref = 0.5 * cos.max(dim=1).values.numpy()
    assert np.abs(best - ref).max() <= 1e-6
    assert is_new.all()


@pytest.mark.parametrize("dtype,tdt", [(1, torch.float16), (2, torch.bfloat16)])
def test_storage_rounding_matches_library(oracle, dtype, tdt):
    g = np.random.default_rng(2)
    x = np.concatenate([g.standard_normal(2000).astype(np.float32) * 0.1,
                        np.array([0.0, -0.0, 1.0, 65504.0, 1e-8, 3.0e-5, 1.00390625, 1.01171875], np.float32)])
    got = oracle.round_to_storage(x, dtype)
    ref = torch.from_numpy(x).to(tdt).to(torch.float32).numpy()
    assert np.array_equal(got, ref)
    if dtype == 2:                                          # the generator's own bf16 packer agrees too
        assert np.array_equal(S.bf16_bits_to_f32(S.f32_to_bf16_bits(x)), ref)


# ------------------------------------------------------------------------------------------------ P8
def _geo_only_map(oracle, desc0, n_obs):
    keys = np.array([pack_key(i, 0, 8) for i in range(4)], np.uint64)
    m = new_map(oracle, w_geo=1.0, w_sem=0.0, tau=0.5)
    m.import_(np.asarray(_obj(4, n_obs), oracle.OBJECT_DTYPE), desc0, keys, np.zeros(4, np.uint32))
    return m


def test_P8_running_mean_closed_forms(oracle):
    """R21 (PAPER.md:352 'detection-count weighted average'): e1 then e2 -> (1,1)/sqrt2;
    n_obs=3 of e1 plus one e2 -> (3,1)/sqrt10;  k identical vectors leave f unchanged; unit norm always."""
    e = np.eye(4, dtype=np.float32)
    depth, mask = _four_voxel_detection()
    m = _geo_only_map(oracle, e[:1], 1)
    m.integrate(depth, mask, pow2_K(), I4, e[1:2], 1)
    objs, desc, _, _ = m.read()
    assert len(objs) == 1 and objs["n_obs"][0] == 2
    assert np.allclose(desc[0], np.array([1, 1, 0, 0]) / np.sqrt(2), atol=1e-7)
    m = _geo_only_map(oracle, e[:1], 3)
    m.integrate(depth, mask, pow2_K(), I4, 5.0 * e[1:2], 1)     # detection rows are normalised first
    objs, desc, _, _ = m.read()
    assert objs["n_obs"][0] == 4
    assert np.allclose(desc[0], np.array([3, 1, 0, 0]) / np.sqrt(10), atol=1e-7)
    f = unit_rows(1, 4, 9)
    m = _geo_only_map(oracle, f, 2)
    for _ in range(3):
        m.integrate(depth, mask, pow2_K(), I4, f, 1)
    objs, desc, _, _ = m.read()
    assert objs["n_obs"][0] == 5 and np.allclose(desc[0], f[0], atol=1e-6)
    assert abs(np.linalg.norm(desc[0].astype(np.float64)) - 1) < 1e-6


def test_P8_several_detections_fuse_into_one_entity(oracle):
    """several detections of one batch may claim one entity and all fuse into it."""
    e = np.eye(4, dtype=np.float32)
    m = _geo_only_map(oracle, e[:1], 1)
    d1, m1 = hand_frame(H, W, [(64, 48, 2.0, 1), (80, 48, 2.0, 2)])     # two detections, one voxel each, both owned
    m.integrate(d1, m1, pow2_K(), I4, np.stack([e[1], e[2]]), 2)
    assoc, is_new, _, _, _ = m.last_assoc()
    assert list(assoc) == [0, 0] and not is_new.any()
    objs, desc, _, _ = m.read()
    assert objs["n_obs"][0] == 3 and np.allclose(desc[0], np.array([1, 1, 1, 0]) / np.sqrt(3), atol=1e-7)


# ------------------------------------------------------------------------------------------------ R2 / R12 / R13 / R20 / R23
def test_R2_snapshot_and_R12_lowest_index_wins(oracle):
    """Two detections of one call that see the same new voxel: both spawn (snapshot, R2), ids in index
    order (R20), the shared voxel goes to the lower index (R12), the other may own nothing (R13)."""
    e = np.eye(4, dtype=np.float32)
    m = new_map(oracle)
    # det 2 (label 2) sits at lower pixel index than det 1 to make sure 'lowest j' is not 'first pixel seen'
    depth, mask = hand_frame(H, W, [(64, 40, 2.0, 2), (66, 41, 2.0, 1), (96, 48, 2.0, 1)])
    # (64,40): X=0,Y=-.125 -> (0,-1,8); (66,41): X=.03125,Y=-.109 -> (0,-1,8) as well; (96,48) -> (2,0,8)
    m.integrate(depth, mask, pow2_K(), I4, e[:2], 2)
    assoc, is_new, _, _, st = m.last_assoc()
    assert list(assoc) == [0, 1] and is_new.all() and st["spawns"] == 2
    objs, _, keys, owners = m.read()
    assert dict(zip(keys.tolist(), owners.tolist())) == {int(pack_key(0, -1, 8)): 0, int(pack_key(2, 0, 8)): 0}
    assert list(objs["n_voxels"]) == [2, 0]
    # keys owned at entry never change owner
    m.integrate(depth, mask, pow2_K(), I4, e[:2], 2)
    _, _, keys2, owners2 = m.read()
    assert np.array_equal(keys, keys2) and np.array_equal(owners, owners2)


def test_R8_empty_detection_is_skipped(oracle):
    e = np.eye(4, dtype=np.float32)
    m = new_map(oracle)
    depth, mask = hand_frame(H, W, [(64, 48, 2.0, 1), (70, 48, 2.0, 3)])      # label 2 has no pixel
    m.integrate(depth, mask, pow2_K(), I4, e[:3], 3)
    assoc, is_new, best, _, st = m.last_assoc()
    assert list(assoc) == [0, -1, 1] and list(is_new) == [1, 0, 1] and st["skipped"] == 1
    objs, _, _, _ = m.read()
    assert len(objs) == 2 and objs["n_obs"].sum() == 2


def test_R23_best_view(oracle):
    """Largest n_px wins; ties keep the earliest (frame_seq, det index); camera position recorded."""
    e = np.eye(4, dtype=np.float32)
    m = new_map(oracle, w_geo=1.0, w_sem=0.0, tau=0.5)
    two = [(64, 48, 2.0, 1), (65, 48, 2.0, 1)]
    three = two + [(66, 48, 2.0, 1)]
    for k, (px, t) in enumerate([(two, 0.0), (three, 0.0), (three, 0.0), (two, 0.0)]):
        depth, mask = hand_frame(H, W, px)
        T = translate(t, 0, 0)
        T[2, 3] = k * 1e-3                                   # camera z differs per frame, same voxel
        m.integrate(depth, mask, pow2_K(), T, e[:1], 1)
    objs, _, _, _ = m.read()
    assert len(objs) == 1
    assert objs["best_pixels"][0] == 3 and objs["best_frame"][0] == 1 and objs["best_det"][0] == 0
    assert objs["best_cam_pos"][0][2] == np.float32(1e-3)
    assert objs["n_points"][0] == 2 + 3 + 3 + 2 and objs["n_obs"][0] == 4


def test_batch_frames_share_one_snapshot(oracle):
    """R2 with F>1 (PAPER.md:65 frames of all cameras stacked): global index j runs over frames in order;
    frame_seq advances by F."""
    e = np.eye(4, dtype=np.float32)
    m = new_map(oracle)
    fa = hand_frame(H, W, [(64, 48, 2.0, 1)])
    fb = hand_frame(H, W, [(64, 48, 2.0, 1), (96, 48, 2.0, 2)])
    depth = np.stack([fa[0], fb[0]])
    mask = np.stack([fa[1], fb[1]])
    K = np.stack([pow2_K(), pow2_K()])
    T = np.stack([I4, I4])
    m.integrate_batch(depth, mask, K, T, e[:3], [1, 2])
    assoc, is_new, _, _, _ = m.last_assoc()
    assert list(assoc) == [0, 1, 2] and is_new.all()         # same voxel seen from two frames: two objects
    objs, _, keys, owners = m.read()
    assert list(objs["n_voxels"]) == [1, 0, 1]
    assert list(objs["best_frame"]) == [0, 1, 1] and list(objs["best_det"]) == [0, 0, 1]
    m.integrate_batch(depth, mask, K, T, e[:3], [1, 2])
    assoc, is_new, best, _, _ = m.last_assoc()
    objs, _, _, _ = m.read()
    # det 1 (frame 1) sees a voxel owned by object 0 (g=1, cos=0 -> 0.5) and its own object 1 owns nothing
    # (R13: g=0, cos=1 -> 0.5): neither passes the strict threshold, so it spawns again (frame_seq 3)
    assert list(assoc) == [0, 3, 2] and list(is_new) == [0, 1, 0] and best[1] == np.float32(0.5)
    assert list(objs["best_frame"]) == [0, 1, 1, 3]          # ties keep the earliest view; seq advanced by F


# ------------------------------------------------------------------------------------------------ P9-P12
def test_P9_P10_P12_invariants_on_generated_scene(oracle):
    cfg, sc, m = _scene_run(oracle)
    union = set()
    non_skipped = 0
    spawns = 0
    prev_boxes = None
    for k in range(12):
        fr = sc.frame(k)
        m.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
        assoc, is_new, best, _, st = m.last_assoc()
        off, keys, n_px, box = m.last_voxels()
        for d in range(fr.n_det):
            if assoc[d] >= 0:
                union |= set(keys[off[d]:off[d + 1]].tolist())
        non_skipped += int((assoc >= 0).sum())
        spawns += int(is_new.sum())
        objs, desc, vk, vo = m.read()
        # P9 voxel conservation: independent of every association decision
        assert objs["n_voxels"].sum() == len(vk) == len(union) and set(vk.tolist()) == union
        assert np.array_equal(np.bincount(vo, minlength=len(objs)), objs["n_voxels"])
        # P12
        assert objs["n_obs"].sum() == non_skipped and len(objs) == spawns
        # unit-norm descriptors (BASELINE.json invariant)
        assert np.abs(np.linalg.norm(desc.astype(np.float64), axis=1) - 1).max() < 1e-6
        # P10: AABB contains every merged point; only grows
        xyz, pk = m.backproject(fr.depth, fr.mask, fr.K, fr.T, fr.n_det)
        for d in range(fr.n_det):
            if assoc[d] < 0:
                continue
            pts = xyz[(fr.mask == d + 1) & (pk != KEY_EMPTY)]
            o = objs[assoc[d]]
            assert (pts >= o["aabb_min"]).all() and (pts <= o["aabb_max"]).all()
        if prev_boxes is not None:
            n = len(prev_boxes)
            assert (objs["aabb_min"][:n] <= prev_boxes["aabb_min"]).all()
            assert (objs["aabb_max"][:n] >= prev_boxes["aabb_max"]).all()
        prev_boxes = objs.copy()
        # P10b: every voxel an object owns that was inserted by one of its own detections touches its AABB
    # empty map + M non-empty detections -> ids in index order
    _, _, m2 = _scene_run(oracle)
    fr = sc.frame(0)
    m2.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
    assoc, is_new, best, _, _ = m2.last_assoc()
    assert list(assoc) == list(range(fr.n_det)) and is_new.all() and (best == 0).all()


def test_P11_idempotence(oracle):
    """Same frame twice: second pass g = 1 exactly, cos = 1, score = w_geo + w_sem, no spawns, voxel sets
    and AABBs unchanged, n_obs doubled, descriptors unchanged."""
    cfg, sc, m = _scene_run(oracle)
    fr = sc.frame(3)
    m.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
    o1, d1, k1, w1 = m.read()
    assert (o1["n_voxels"] > 0).all()                        # the exception of P11 does not arise here
    m.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
    assoc, is_new, best, _, st = m.last_assoc()
    o2, d2, k2, w2 = m.read()
    assert not is_new.any() and list(assoc) == list(range(fr.n_det))
    assert np.abs(best - 1.0).max() <= 1e-6
    assert np.array_equal(k1, k2) and np.array_equal(w1, w2)
    assert np.array_equal(o1["aabb_min"], o2["aabb_min"]) and np.array_equal(o1["aabb_max"], o2["aabb_max"])
    assert np.array_equal(o2["n_obs"], 2 * o1["n_obs"]) and np.abs(d1 - d2).max() <= 1e-6


def test_constant_footprint_per_entity(oracle):
    """per-entity footprint constant in observation count (descriptor, AABB, view state)."""
    e = np.eye(4, dtype=np.float32)
    m = new_map(oracle, w_geo=1.0, w_sem=0.0, tau=0.5)
    depth, mask = _four_voxel_detection()
    for _ in range(5):
        m.integrate(depth, mask, pow2_K(), I4, e[:1], 1)
    objs, desc, keys, _ = m.read()
    assert len(objs) == 1 and desc.shape == (1, 4) and len(keys) == 4 and objs["n_obs"][0] == 5


def test_R26_import_round_trip(oracle):
    cfg, sc, m = _scene_run(oracle)
    for k in range(5):
        fr = sc.frame(k)
        m.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
    objs, desc, keys, owners = m.read()
    m2 = oracle.OracleMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, cfg.dtype, cfg.H, cfg.W)
    perm = np.random.default_rng(0).permutation(len(keys))
    assert m2.import_(objs, desc, keys[perm], owners[perm]) == 0
    o2, d2, k2, w2 = m2.read()
    assert np.array_equal(objs, o2) and np.array_equal(keys, k2) and np.array_equal(owners, w2)
    assert np.abs(desc - d2).max() <= 1e-7
    # both continue identically
    fr = sc.frame(5)
    for mm in (m, m2):
        mm.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
    a1, a2 = m.last_assoc(), m2.last_assoc()
    assert np.array_equal(a1[0], a2[0]) and np.abs(a1[2] - a2[2]).max() <= 1e-6
    # duplicate key -> rejected
    m3 = oracle.OracleMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, cfg.dtype, cfg.H, cfg.W)
    assert m3.import_(objs, desc, np.concatenate([keys, keys[:1]]), np.concatenate([owners, owners[:1]])) != 0
