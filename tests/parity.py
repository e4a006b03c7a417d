"""GPU-vs-oracle comparison helpers used by the `-m gpu` tests and by __graft_entry__.smoke().

Bar (BASELINE.json north_star): voxel sets, overlap counts, association decisions, object counts and all
integer state bit-exact; points, AABBs, descriptors and scores within 1e-4 absolute.
"""
import numpy as np
import torch

from helpers import stack_frames
from paper_2606_15476_b200 import FarmMap, scenes as S

TOL = 1e-4


def upload(frames, dtype):
    depth, mask, K, T, desc, n_det = stack_frames(frames)
    dev = torch.device("cuda:0")
    d = {
        "depth": torch.from_numpy(depth).to(dev),
        "mask": torch.from_numpy(mask.view(np.int16)).to(dev),
        "K": torch.from_numpy(K).to(dev).contiguous(),
        "T": torch.from_numpy(T).to(dev).contiguous(),
        "n_det": n_det,
    }
    if desc is None or desc.size == 0:
        d["desc"] = None
    elif dtype == S.DTYPE_F32:
        d["desc"] = torch.from_numpy(np.ascontiguousarray(desc, np.float32)).to(dev)
    elif dtype == S.DTYPE_F16:
        d["desc"] = torch.from_numpy(np.ascontiguousarray(desc, np.float16)).to(dev)
    else:
        d["desc"] = torch.from_numpy(np.ascontiguousarray(desc, np.uint16).view(np.int16)).to(dev)
    return d


def gpu_integrate(g: FarmMap, frames, dtype):
    d = upload(frames, dtype)
    g.integrate_batch(len(frames), d["depth"], d["mask"], d["K"], d["T"], d["desc"], d["n_det"])
    return d


def make_pair(oracle, cfg, H=None, W=None, **kw):
    H = cfg.H if H is None else H
    W = cfg.W if W is None else W
    o = oracle.OracleMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, cfg.dtype, H, W)
    g = FarmMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, H=H, W=W, dtype=cfg.dtype, **kw)
    return o, g


def compare_call(g: FarmMap, o, check_sets=True):
    """Compare the results of the last integrate call of both sides."""
    ao, no, bo, so, sto = o.last_assoc()
    ag, ng, bg, stg = g.last_assoc()
    assert np.array_equal(ag, ao), (ag, ao)
    assert np.array_equal(ng, no)
    assert np.abs(bg - bo).max(initial=0) <= TOL, np.abs(bg - bo).max()
    for k in ("valid_points", "dropped_points", "ignored_pixels", "unique_voxels", "matches", "spawns", "skipped", "n_det"):
        assert int(stg[k]) == int(sto[k]), (k, stg[k], sto[k])
    if check_sets:
        offo, keyo, npxo, boxo = o.last_voxels()
        offg, keyg, npxg, boxg = g.debug_last_voxels()
        assert np.array_equal(offg, offo)
        assert np.array_equal(npxg, npxo)
        M = len(npxo)
        for d in range(M):
            assert np.array_equal(np.sort(keyg[offg[d]:offg[d + 1]]), keyo[offo[d]:offo[d + 1]])   # bit-exact voxel sets
        has = npxo > 0
        assert np.array_equal(boxg[has], boxo[has])                # exact fp32 min/max of identical points
        oo, objo, cnto = o.last_overlaps()
        og, objg, cntg = g.debug_last_overlaps()
        assert np.array_equal(og, oo)
        for d in range(M):
            order = np.argsort(objg[og[d]:og[d + 1]])
            assert np.array_equal(objg[og[d]:og[d + 1]][order], objo[oo[d]:oo[d + 1]])
            assert np.array_equal(cntg[og[d]:og[d + 1]][order], cnto[oo[d]:oo[d + 1]])


def compare_maps(g: FarmMap, o, voxels=True):
    objo, desco, keyo, owno = o.read(voxels=voxels)
    objg, descg, keyg, owng = g.read(voxels=voxels)
    assert len(objg) == len(objo)
    for f in ("id", "n_voxels", "n_obs", "best_frame", "best_det", "best_pixels", "n_points"):
        assert np.array_equal(objg[f], objo[f]), f
    for f in ("aabb_min", "aabb_max", "best_cam_pos"):
        assert np.array_equal(objg[f], objo[f]), f
    assert np.abs(descg - desco).max(initial=0) <= TOL
    if voxels:
        order = np.argsort(keyg)
        assert np.array_equal(keyg[order], keyo)
        assert np.array_equal(owng[order], owno)


def compare_dense(g: FarmMap, o):
    """R16/R18: dense row maximum of the clamped cosine and its argmax (lowest id on ties) of the last call.  The argmax
    is compared wherever the oracle's runner-up is more than 1e-4 away, and on exact ties (bit-identical map rows),
    which the id rule decides on both sides.  Returns the number of rows whose argmax was compared."""
    mc_o, am_o = o.last_dense()
    sec = o.last_dense_second()
    mc_g, am_g = g.debug_last_dense()
    ok = o.last_assoc()[0] >= 0                                   # skipped detections have no dense row in the oracle
    assert np.abs(mc_g - mc_o)[ok].max(initial=0) <= TOL
    clear = ok & (am_o >= 0) & ((mc_o - sec > 1e-4) | (mc_o == sec))
    assert np.array_equal(am_g[clear], am_o[clear]), (am_g[clear], am_o[clear])
    return int(clear.sum())


def dense_decided(o):
    """number of detections of the oracle's last call matched to an object they share NO voxel with: the dense
    argmax supplied the matched object (R19)"""
    assoc, is_new, _, _, _ = o.last_assoc()
    off, obj, _ = o.last_overlaps()
    n = 0
    for d in range(len(assoc)):
        if assoc[d] >= 0 and not is_new[d] and assoc[d] not in set(obj[off[d]:off[d + 1]].tolist()):
            n += 1
    return n
