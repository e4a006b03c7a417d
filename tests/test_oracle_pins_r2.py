"""Round-2 pins of the CPU oracle (additions to tests/test_oracle_pins.py, which is left untouched).

R22 object AABB tightness, `stats.unique_voxels`, and the dense row max / argmax of R16 / R18 (the value the
association takes its matched object from when w_sem > tau).  Expected values come from independent numpy
loops over the oracle's debug per-pixel output, from a library GEMM + numpy.argmax, or from hand cases;
none comes from the oracle function under test or from the CUDA path.
"""
import numpy as np
import pytest
import torch

from helpers import KEY_EMPTY, hand_frame, pack_key, pow2_K, unit_rows
from paper_2606_15476_b200 import scenes as S

H, W = 96, 128
I4 = np.eye(4, dtype=np.float32)


def _obj(oracle, n, n_voxels=1):
    o = np.zeros(n, oracle.OBJECT_DTYPE)
    o["id"], o["n_voxels"], o["n_obs"], o["best_frame"], o["best_det"] = np.arange(n), n_voxels, 1, -1, -1
    return o


# ------------------------------------------------------------------------------------------ R22 tightness
def test_R22_object_aabb_is_exactly_the_min_max_of_its_merged_points(oracle):
    """A freshly spawned object's AABB == box_d of its detection; after k merges it == the exact fp32 min / max
    over the debug back-projection's points of every detection merged into it (not merely a superset)."""
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    m = oracle.OracleMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, cfg.dtype, cfg.H, cfg.W)
    lo, hi = {}, {}                                          # independent bookkeeping per object id
    merges = 0
    for k in range(10):
        fr = sc.frame(k)
        m.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
        assoc, is_new, _, _, _ = m.last_assoc()
        _, _, n_px, box = m.last_voxels()
        xyz, pk = m.backproject(fr.depth, fr.mask, fr.K, fr.T, fr.n_det)
        objs, _, _, _ = m.read(voxels=False)
        for d in range(fr.n_det):
            if assoc[d] < 0:
                continue
            pts = xyz[(fr.mask == d + 1) & (pk != KEY_EMPTY)]
            o = int(assoc[d])
            if is_new[d]:
                assert o not in lo
                assert np.array_equal(objs["aabb_min"][o], box[d, :3]) or (assoc == o).sum() > 1
                lo[o], hi[o] = pts.min(0), pts.max(0)
            else:
                merges += 1
                lo[o], hi[o] = np.minimum(lo[o], pts.min(0)), np.maximum(hi[o], pts.max(0))
        for o in lo:
            assert np.array_equal(objs["aabb_min"][o], lo[o]), (k, o)
            assert np.array_equal(objs["aabb_max"][o], hi[o]), (k, o)
    assert merges > 10 and len(lo) == len(objs)


def test_R22_new_object_box_equals_box_d_hand_case(oracle):
    """Two pixels at (96,48,z=2) and (64,40,z=2): box_d = [(0,-.125,2), (.5,0,2)] exactly; the spawned object has it."""
    e = np.eye(4, dtype=np.float32)
    m = oracle.OracleMap(0.25, 4, 0.5, 0.5, 0.5, 0, H, W)
    depth, mask = hand_frame(H, W, [(96, 48, 2.0, 1), (64, 40, 2.0, 1)])
    m.integrate(depth, mask, pow2_K(), I4, e[:1], 1)
    objs, _, _, _ = m.read()
    assert list(objs["aabb_min"][0]) == [0.0, -0.125, 2.0] and list(objs["aabb_max"][0]) == [0.5, 0.0, 2.0]
    # a second, disjoint detection of another object does not touch it (a box merged into one object too many would)
    depth2, mask2 = hand_frame(H, W, [(10, 10, 3.0, 1)])
    m.integrate(depth2, mask2, pow2_K(), I4, e[1:2], 1)
    objs, _, _, _ = m.read()
    assert len(objs) == 2
    assert list(objs["aabb_min"][0]) == [0.0, -0.125, 2.0] and list(objs["aabb_max"][0]) == [0.5, 0.0, 2.0]
    assert np.array_equal(objs["aabb_min"][1], objs["aabb_max"][1])            # a single point


def test_stats_unique_voxels_is_the_sum_of_set_sizes(oracle):
    """stats.unique_voxels == sum_d |V_d| with V_d rebuilt by np.unique over the debug per-pixel keys (P4's loop);
    valid_points == number of valid masked pixels with an in-range key."""
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    m = oracle.OracleMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, cfg.dtype, cfg.H, cfg.W)
    for k in range(4):
        fr = sc.frame(k)
        m.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
        _, _, _, _, st = m.last_assoc()
        _, pk = m.backproject(fr.depth, fr.mask, fr.K, fr.T, fr.n_det)
        tot, pts = 0, 0
        for d in range(fr.n_det):
            sel = (fr.mask == d + 1) & (pk != KEY_EMPTY)
            tot += len(np.unique(pk[sel]))
            pts += int(sel.sum())
        assert int(st["unique_voxels"]) == tot and tot > 100
        assert int(st["valid_points"]) == pts


# ------------------------------------------------------------------------------------------ R16/R18 dense argmax
@pytest.mark.parametrize("dtype", [0, 1, 2])
def test_dense_row_max_and_argmax_vs_library_gemm(oracle, dtype):
    """R16: the oracle's dense (max, argmax) per detection against numpy.argmax of a float64 library GEMM on the
    library-converted storage operands; includes an exact tie (two bit-identical map rows): lowest id wins (R18)."""
    D, N, Mdet = 48, 37, 5
    objdesc = unit_rows(N, D, 31)
    det = unit_rows(Mdet, D, 32)
    det[1] = objdesc[20] + 0.01 * unit_rows(1, D, 33)[0]        # close to object 20
    det[3] = objdesc[11]                                        # identical to objects 11 and (below) 29: tie
    objdesc[29] = objdesc[11]
    m = oracle.OracleMap(0.25, D, 0.3, 0.7, 0.5, dtype, H, W)
    keys = np.array([pack_key(500 + i, 0, 0) for i in range(N)], np.uint64)
    assert m.import_(_obj(oracle, N), objdesc, keys, np.arange(N, dtype=np.uint32)) == 0
    depth, mask = hand_frame(H, W, [(8 + 16 * d, 48, 2.0, d + 1) for d in range(Mdet)])
    m.integrate(depth, mask, pow2_K(), I4, S.to_storage(det, dtype), Mdet)
    mc, am = m.last_dense()
    tdt = {0: torch.float32, 1: torch.float16, 2: torch.bfloat16}[dtype]
    A = torch.from_numpy(det).to(tdt).to(torch.float64).numpy()
    # R26/R14: imported rows are renormalised in fp32-or-better, then shadowed in the storage dtype
    Bn = objdesc.astype(np.float64)
    Bn = (Bn / np.linalg.norm(Bn, axis=1, keepdims=True)).astype(np.float32)
    B = torch.from_numpy(Bn).to(tdt).to(torch.float64).numpy()
    cos = np.clip((A @ B.T) / np.outer(np.linalg.norm(A, axis=1), np.linalg.norm(B, axis=1)), -1, 1)
    ref_arg = cos.argmax(axis=1)                                # numpy: first maximum = lowest id
    assert np.abs(mc - cos.max(axis=1)).max() <= 1e-6
    assert np.abs(m.last_dense_second() - np.sort(cos, axis=1)[:, -2]).max() <= 1e-6
    far = np.sort(cos, axis=1)[:, -1] - np.sort(cos, axis=1)[:, -2] > 1e-5
    far[3] = True                                               # the exact tie is decided by the id rule
    assert np.array_equal(am[far], ref_arg[far])
    assert am[3] == 11 and am[1] == 20
    # with w_sem = 0.7 > tau = 0.5 and no voxel overlap the dense argmax IS the decision (R19)
    assoc, is_new, best, _, _ = m.last_assoc()
    for d in range(Mdet):
        s = np.float32(0.7) * np.float32(cos[d].max())
        if abs(float(s) - 0.5) < 1e-4:
            continue
        if s > 0.5:
            assert not is_new[d] and assoc[d] == am[d]
        else:
            assert is_new[d]
        assert abs(float(best[d]) - float(s)) <= 1e-6
    assert not is_new[1] and not is_new[3] and assoc[3] == 11


def test_dense_of_skipped_detection_and_empty_map(oracle):
    e = np.eye(4, dtype=np.float32)
    m = oracle.OracleMap(0.25, 4, 0.5, 0.5, 0.5, 0, H, W)
    depth, mask = hand_frame(H, W, [(64, 48, 2.0, 1)])
    m.integrate(depth, mask, pow2_K(), I4, e[:2], 2)            # empty map; detection 1 has no pixels (R8)
    mc, am = m.last_dense()
    assert list(am) == [-1, -1] and list(mc) == [0.0, 0.0]
    m.integrate(depth, mask, pow2_K(), I4, e[:2], 2)
    mc, am = m.last_dense()
    assert list(am) == [0, -1] and mc[0] == 1.0
