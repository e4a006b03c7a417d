"""Pins of the round-2 oracle rules (SURVEY.md §8(f) NEXT-1..4), `-m "not gpu"`.

U1-U4 union-find correspondence with entity merges, H1-H3 Hellinger distance as the geometric term
(PAPER.md:350, 358), V1-V2 view selection, Q1-Q5 retrieval scoring.
Expected values: hand cases, closed forms, conservation laws, a brute-force Python restatement of the match graph and
its connected components from independently pinned quantities, numpy argsort for ranks.  None comes from the function
under test or from the CUDA path.
"""
import numpy as np
import pytest

from helpers import hand_frame, pack_key, pow2_K, unit_rows
from paper_2606_15476_b200 import scenes as S

H, W = 96, 128
I4 = np.eye(4, dtype=np.float32)
E = np.eye(8, dtype=np.float32)


def _objs(oracle, n_voxels):
    o = np.zeros(len(n_voxels), oracle.OBJECT_DTYPE)
    o["id"], o["n_voxels"], o["n_obs"], o["best_frame"], o["best_det"] = np.arange(len(n_voxels)), n_voxels, 1, -1, -1
    return o


def _four_px(label=1, u0=64):
    # z = 2, v = 48: u = 64, 80, 96, 112 -> X = 0, .25, .5, .75 -> voxels (0..3, 0, 8) at voxel 0.25
    return [(u0 + 16 * i, 48, 2.0, label) for i in range(4)]


# ================================================================================================ U: union-find
def test_U_detection_bridges_two_entities(oracle):
    """P:350 "a detection retaining two or more entities is what later bridges previously separate entities":
    objects 0 and 1 each own two of the detection's four voxels and both look like it -> both retained -> merged;
    winner = lowest id; voxels re-owned, counts summed, descriptor count-weighted, loser dead with alias."""
    m = oracle.OracleMap(0.25, 8, 0.5, 0.5, 0.5, 0, H, W)
    m.set_option(m.OPT_CORRESPONDENCE, 1)
    keys = np.array([pack_key(0, 0, 8), pack_key(1, 0, 8), pack_key(2, 0, 8), pack_key(3, 0, 8), pack_key(90, 0, 0)], np.uint64)
    owners = np.array([0, 0, 1, 1, 2], np.uint32)
    objs = _objs(oracle, [2, 2, 1])
    objs["n_obs"] = [3, 1, 1]
    desc = np.stack([E[0], E[1], E[5]])
    assert m.import_(objs, desc, keys, owners) == 0
    d = (E[0] + E[1]) / np.sqrt(2)                                  # cos = 0.707 with both; g = 2/min(4,2) = 1
    depth, mask = hand_frame(H, W, _four_px())
    m.integrate(depth, mask, pow2_K(), I4, d[None].astype(np.float32), 1)
    assoc, is_new, best, _, st = m.last_assoc()
    assert assoc[0] == 0 and is_new[0] == 0 and st["matches"] == 1 and st["spawns"] == 0
    assert abs(best[0] - (0.5 + 0.5 / np.sqrt(2))) < 1e-6
    frm, into = m.last_merges()
    assert list(frm) == [1] and list(into) == [0]
    assert list(m.read_alias()) == [0, 0, 2]
    o, dsc, k, own = m.read()
    assert list(o["n_voxels"]) == [4, 0, 1] and list(o["n_obs"]) == [5, 0, 1]
    assert sorted(own[np.isin(k, keys[:4])]) == [0, 0, 0, 0]        # the loser's voxels are the winner's now
    # count-weighted mean: 3 e0 + 1 e1 + (e0 + e1)/sqrt2, normalised
    v = 3 * E[0] + E[1] + d
    assert np.abs(dsc[0] - v / np.linalg.norm(v)).max() < 1e-6
    assert np.abs(dsc[1]).max() == 0.0 and np.abs(dsc[2] - E[5]).max() < 1e-7
    # the dead id never matches again; the same detection now matches the winner alone
    m.integrate(depth, mask, pow2_K(), I4, d[None].astype(np.float32), 1)
    assoc, is_new, _, _, _ = m.last_assoc()
    assert assoc[0] == 0 and len(m.last_merges()[0]) == 0


def test_U_no_bridge_without_the_option_and_chain_of_three(oracle):
    """Off by default: the same scene leaves both objects alone.  With it, two detections that each bridge a pair
    (0-1, 1-2) put all three entities into one component: winner 0."""
    keys = np.array([pack_key(i, 0, 8) for i in range(4)] + [pack_key(i, 4, 8) for i in range(4)], np.uint64)
    #   det A sees voxels x=0..3 (y=0): objects 0 owns x=0,1; object 1 owns x=2,3
    #   det B sees voxels x=0..3 (y=4): object 1 owns x=0,1 there; object 2 owns x=2,3
    owners = np.array([0, 0, 1, 1, 1, 1, 2, 2], np.uint32)
    desc = np.stack([E[0], E[0], E[0]])
    px = _four_px(1) + [(64 + 16 * i, 112, 2.0, 2) for i in range(4)]      # v = 112 -> Y = (112-48)/128*2 = 1.0 -> iy = 4
    depth, mask = hand_frame(H + 32, W, px)
    for opt, expect_alias in ((0, [0, 1, 2]), (1, [0, 0, 0])):
        m = oracle.OracleMap(0.25, 8, 0.5, 0.5, 0.5, 0, H + 32, W)
        m.set_option(m.OPT_CORRESPONDENCE, opt)
        assert m.import_(_objs(oracle, [2, 4, 2]), desc, keys, owners) == 0
        m.integrate(depth, mask, pow2_K(), I4, np.stack([E[0], E[0]]), 2)
        assoc, is_new, _, _, _ = m.last_assoc()
        assert list(m.read_alias()) == expect_alias and not is_new.any()
        o, _, k, own = m.read()
        if opt:
            assert list(assoc) == [0, 0] and list(o["n_voxels"]) == [8, 0, 0] and list(o["n_obs"]) == [5, 0, 0]
            assert (own == 0).all()
        else:
            assert list(o["n_voxels"]) == [2, 4, 2] and o["n_obs"].sum() == 5


def test_U_same_call_duplicate_spawn_is_repaired(oracle):
    """The R2 consequence pinned in test_batch_frames_share_one_snapshot (two frames of one call see the same new
    voxel -> two objects, the second owning nothing and never matched again) is repaired by the detection-detection
    edge (U2): c_dd = 1, g = 1, cos = 1 -> one entity."""
    m = oracle.OracleMap(0.25, 4, 0.5, 0.5, 0.5, 0, H, W)
    m.set_option(m.OPT_CORRESPONDENCE, 1)
    e = np.eye(4, dtype=np.float32)
    fa = hand_frame(H, W, [(64, 48, 2.0, 1)])
    fb = hand_frame(H, W, [(64, 48, 2.0, 1), (96, 48, 2.0, 2)])
    depth, mask = np.stack([fa[0], fb[0]]), np.stack([fa[1], fb[1]])
    K, T = np.stack([pow2_K(), pow2_K()]), np.stack([I4, I4])
    m.integrate_batch(depth, mask, K, T, np.stack([e[0], e[0], e[2]]), [1, 2])
    assoc, is_new, _, _, st = m.last_assoc()
    assert list(assoc) == [0, 0, 1] and list(is_new) == [1, 0, 1] and st["spawns"] == 2 and st["matches"] == 1
    o, _, _, _ = m.read()
    assert list(o["n_voxels"]) == [1, 1] and list(o["n_obs"]) == [2, 1]
    assert list(o["best_frame"]) == [0, 1]                          # R23 tie keeps the earliest view
    # a different-looking detection of the same voxel is NOT linked (cos = 0 -> 0.5, strict)
    m2 = oracle.OracleMap(0.25, 4, 0.5, 0.5, 0.5, 0, H, W)
    m2.set_option(m2.OPT_CORRESPONDENCE, 1)
    m2.integrate_batch(depth, mask, K, T, np.stack([e[0], e[1], e[2]]), [1, 2])
    assert list(m2.last_assoc()[0]) == [0, 1, 2]


def split_map_arrays(objs, desc, keys, owners):
    """every object of an exported map cut into two entities (voxels alternate between them in key order; same
    descriptor, counts split): a later detection of the object overlaps both halves and bridges them"""
    N = len(objs)
    order = np.argsort(keys)
    keys, owners = keys[order], owners[order]
    rank = np.zeros(len(keys), np.int64)
    for o in range(N):
        sel = np.nonzero(owners == o)[0]
        rank[sel] = np.arange(len(sel))
    own2 = (2 * owners.astype(np.int64) + (rank & 1)).astype(np.uint32)
    objs2 = np.repeat(objs, 2)
    objs2["id"] = np.arange(2 * N)
    objs2["n_voxels"] = np.bincount(own2, minlength=2 * N)
    objs2["n_obs"] = np.maximum(objs2["n_obs"] // 2, 1)
    objs2["n_points"] //= 2
    return objs2, np.repeat(desc, 2, axis=0), keys, own2


def split_map_scene(oracle, cfg, sc, w_geo, w_sem, tau, n_build=9):
    """an oracle map with the correspondence option on, imported from the split export of a plain run over the first
    n_build frames"""
    plain = oracle.OracleMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, cfg.dtype, cfg.H, cfg.W)
    for k in range(n_build):
        fr = sc.frame(k)
        plain.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
    m = oracle.OracleMap(cfg.voxel, cfg.D, w_geo, w_sem, tau, cfg.dtype, cfg.H, cfg.W)
    m.set_option(m.OPT_CORRESPONDENCE, 1)
    assert m.import_(*split_map_arrays(*plain.read())) == 0
    return m


def _brute_components(n_nodes, edges):
    adj = {i: set() for i in range(n_nodes)}
    for a, b in edges:
        adj[a].add(b)
        adj[b].add(a)
    comp, seen = {}, set()
    for s in range(n_nodes):
        if s in seen:
            continue
        stack, members = [s], []
        while stack:
            x = stack.pop()
            if x in seen:
                continue
            seen.add(x)
            members.append(x)
            stack.extend(adj[x] - seen)
        for x in members:
            comp[x] = min(members)
    return comp


def test_U_components_against_brute_force_on_generated_scene(oracle):
    """configs[0] in batches of 3 frames with loosened weights (w_geo = 0.7, w_sem = 0.3, tau = 0.25: several entities
    pass per detection).  The match graph is rebuilt in Python from independently pinned quantities -- overlap counts
    (P5), set sizes (P4), numpy cosines (P7) -- its components by a graph search, and assignments, new ids, merges,
    conservation of observations and voxels are checked against it."""
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    wg, ws, tau = np.float32(0.7), np.float32(0.3), np.float32(0.25)
    m = split_map_scene(oracle, cfg, sc, float(wg), float(ws), float(tau))
    objs_i, _, keys_i, _ = m.read()
    total_dets, total_merges, union_keys = int(objs_i["n_obs"].sum()), 0, set(keys_i.tolist())
    for call in range(3, 6):
        frames = [sc.frame(3 * call + i) for i in range(3)]
        objs0, desc0, keys0, own0 = m.read()
        alias0 = m.read_alias()
        N = len(objs0)
        depth = np.stack([f.depth for f in frames]); mask = np.stack([f.mask for f in frames])
        K = np.stack([f.K for f in frames]); T = np.stack([f.T for f in frames])
        desc = np.concatenate([f.desc for f in frames]); n_det = [f.n_det for f in frames]
        m.integrate_batch(depth, mask, K, T, desc, n_det)
        assoc, is_new, best, _, st = m.last_assoc()
        off, vkeys, n_px, _ = m.last_voxels()
        ooff, oobj, ocnt = m.last_overlaps()
        M = len(assoc)
        owner0 = dict(zip(keys0.tolist(), own0.tolist()))
        A = desc.astype(np.float64); A /= np.linalg.norm(A, axis=1, keepdims=True)
        B = desc0.astype(np.float64)
        nb = np.linalg.norm(B, axis=1, keepdims=True); B = np.divide(B, nb, out=np.zeros_like(B), where=nb > 0)
        cos = np.clip(A @ B.T, -1, 1) if N else np.zeros((M, 0))
        edges, close = [], False
        claim = {}
        for d in range(M):
            if n_px[d] == 0:
                continue
            for k in vkeys[off[d]:off[d + 1]].tolist():
                if k not in owner0:
                    claim.setdefault(k, d)
        retained = {}
        for d in range(M):
            if n_px[d] == 0:
                continue
            ov = dict(zip(oobj[ooff[d]:ooff[d + 1]].tolist(), ocnt[ooff[d]:ooff[d + 1]].tolist()))
            nv = off[d + 1] - off[d]
            retained[d] = []
            for o in range(N):
                mn = min(nv, int(objs0["n_voxels"][o]))
                g = np.float32(ov.get(o, 0)) / np.float32(mn) if mn else np.float32(0)
                s = wg * g + ws * np.float32(cos[d, o])
                close |= abs(float(s) - float(tau)) < 1e-4
                if s > tau:
                    retained[d].append(o)
                    edges.append((N + d, o))
        for d in range(M):
            if n_px[d] == 0 or retained[d]:
                continue
            cdd = {}
            for k in vkeys[off[d]:off[d + 1]].tolist():
                e = claim.get(k, d)
                if e != d:
                    cdd[e] = cdd.get(e, 0) + 1
            for e, c in cdd.items():
                mn = min(off[d + 1] - off[d], off[e + 1] - off[e])
                s = wg * (np.float32(c) / np.float32(mn)) + ws * np.float32(np.clip(A[d] @ A[e], -1, 1))
                close |= abs(float(s) - float(tau)) < 1e-4
                if s > tau:
                    edges.append((N + d, N + e))
        assert not close, "a score sits on the threshold; change the seed of this pin"
        comp = _brute_components(N + M, edges)
        new_ids, nxt = {}, N
        for d in range(M):
            if n_px[d] == 0:
                assert assoc[d] == -1
                continue
            r = comp[N + d]
            if r < N:
                assert assoc[d] == r and not is_new[d]
            else:
                if r not in new_ids:
                    new_ids[r] = nxt
                    nxt += 1
                    assert is_new[d]
                else:
                    assert not is_new[d]
                assert assoc[d] == new_ids[r]
        frm, into = m.last_merges()
        expect_merges = sorted((o, comp[o]) for o in range(N) if comp[o] != o)
        assert sorted(zip(frm.tolist(), into.tolist())) == expect_merges
        total_merges += len(frm)
        total_dets += int((assoc >= 0).sum())
        for d in range(M):
            if assoc[d] >= 0:
                union_keys |= set(vkeys[off[d]:off[d + 1]].tolist())
        objs1, desc1, keys1, own1 = m.read()
        alias1 = m.read_alias()
        live = alias1 == np.arange(len(alias1))
        assert objs1["n_obs"].sum() == total_dets and (objs1["n_obs"][~live] == 0).all()           # observations conserved
        assert objs1["n_voxels"].sum() == len(keys1) == len(union_keys)                              # voxels conserved
        assert np.array_equal(np.bincount(own1, minlength=len(objs1)), objs1["n_voxels"]) and live[own1].all()
        assert np.abs(np.linalg.norm(desc1[live].astype(np.float64), axis=1) - 1).max() < 1e-6
        assert (alias1[:N][alias0 != np.arange(N)] != np.arange(N)[alias0 != np.arange(N)]).all()   # dead stays dead
    assert total_merges >= 2, total_merges


def test_U_idempotent_when_nothing_bridges(oracle):
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    a = oracle.OracleMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, cfg.dtype, cfg.H, cfg.W)
    b = oracle.OracleMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, cfg.dtype, cfg.H, cfg.W)
    b.set_option(b.OPT_CORRESPONDENCE, 1)
    n_merge = 0
    for k in range(8):
        fr = sc.frame(k)
        for mm in (a, b):
            mm.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
        n_merge += len(b.last_merges()[0])
        if n_merge == 0:                                        # until the first bridge both readings agree exactly
            assert np.array_equal(a.last_assoc()[0], b.last_assoc()[0])
    assert (b.read_alias() == np.arange(len(b.read_alias()))).sum() <= len(a.read()[0])


# ================================================================================================ H: Hellinger geometry
def _hellinger_np(mu1, S1, mu2, S2):
    Sb = 0.5 * (S1 + S2)
    d = mu1 - mu2
    bc = (np.linalg.det(S1) ** 0.25) * (np.linalg.det(S2) ** 0.25) / np.sqrt(np.linalg.det(Sb)) * np.exp(-0.125 * d @ np.linalg.solve(Sb, d))
    return np.sqrt(max(0.0, 1.0 - bc))


def _unpack(c):
    return np.array([[c[0], c[1], c[2]], [c[1], c[3], c[4]], [c[2], c[4], c[5]]], np.float64)


def test_H_same_frame_twice_gives_g_one_and_far_objects_g_zero(oracle):
    """H3: g = 1 - H.  The same frame twice: H(p, p) = 0 -> g = 1, cos = 1 -> score = w_geo + w_sem, everything matches.
    The voxel overlap plays no part: with a coarser voxel grid the decision is the same."""
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    m = oracle.OracleMap(cfg.voxel, cfg.D, 0.5, 0.5, 0.5, cfg.dtype, cfg.H, cfg.W)
    m.set_option(m.OPT_GEOMETRY, 1)
    fr = sc.frame(2)
    m.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
    assert m.last_assoc()[1].all()
    m.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
    assoc, is_new, best, _, _ = m.last_assoc()
    assert list(assoc) == list(range(fr.n_det)) and not is_new.any() and np.abs(best - 1.0).max() < 1e-6


def test_H_decisions_against_numpy_hellinger_and_prefilter(oracle):
    """H1-H3 on configs[0]: candidates are exactly the entities with cos > prefilter; g = 1 - H with H from
    numpy.linalg on the (independently pinned, G-P1/G-P2) Gaussians read before the call; the budget drops candidates."""
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    for budget, pre in ((1.0, 0.3), (0.9, -1.0)):
        m = oracle.OracleMap(cfg.voxel, cfg.D, 0.5, 0.5, 0.5, cfg.dtype, cfg.H, cfg.W)
        m.set_option(m.OPT_GEOMETRY, 1)
        m.set_option(m.OPT_PREFILTER_COS, pre)
        m.set_option(m.OPT_HELLINGER_BUDGET, budget)
        n_checked = n_match = n_gated = 0
        for k in range(12):
            fr = sc.frame(k)
            objs0, desc0, _, _ = m.read(voxels=False)
            w0, mu0, cov0 = m.read_gaussians()
            N = len(objs0)
            m.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
            assoc, is_new, best, _, _ = m.last_assoc()
            mu_d, cov_d, _ = m.last_gaussians()
            A = fr.desc.astype(np.float64); A /= np.linalg.norm(A, axis=1, keepdims=True)
            eps2 = float(np.float32(cfg.voxel)) ** 2
            for d in range(fr.n_det):
                if assoc[d] < 0:
                    continue
                scores = {}
                for o in range(N):
                    c = float(np.clip(A[d] @ (desc0[o].astype(np.float64) / np.linalg.norm(desc0[o].astype(np.float64))), -1, 1))
                    if not c > pre:
                        continue
                    g = 0.0
                    if w0[o] > 0:
                        h = _hellinger_np(mu_d[d].astype(np.float64), _unpack(cov_d[d]) + eps2 * np.eye(3),
                                          mu0[o].astype(np.float64), _unpack(cov0[o]) + eps2 * np.eye(3))
                        if h > budget:
                            n_gated += 1
                            continue
                        g = 1.0 - h
                    scores[o] = 0.5 * g + 0.5 * c
                exp_best = max(scores.values()) if scores else 0.0
                # exported Gaussians are fp32: the recomputed H carries ~1e-4
                assert abs(float(best[d]) - exp_best) < 2e-3, (k, d, best[d], exp_best)
                if abs(exp_best - 0.5) > 5e-3:
                    assert bool(is_new[d]) == (not exp_best > 0.5)
                    if exp_best > 0.5:
                        top = sorted(scores.items(), key=lambda kv: (-kv[1], kv[0]))
                        if len(top) < 2 or top[0][1] - top[1][1] > 5e-3:
                            assert assoc[d] == top[0][0]
                        n_match += 1
                    n_checked += 1
        assert n_checked > 30 and n_match > 10
    assert n_gated > 0                                              # the 0.9 budget did drop candidates


# ================================================================================================ V: view selection
def _view_scene(oracle, k, poses, **opts):
    """one object (8x8 pixel patch, voxel 0.25) seen from camera positions `poses` = (x, y, z) looking along +z"""
    HV = WV = 512                                                   # fx = 128, cx = cy = 256: +-63 degrees
    m = oracle.OracleMap(0.25, 4, 1.0, 0.0, 0.2, 0, HV, WV)         # geometry alone decides: everything matches
    m.set_option(m.OPT_VIEWS_K, k)
    for key, v in opts.items():
        m.set_option(key, v)
    e = np.eye(4, dtype=np.float32)
    for (x, y, z) in poses:
        # the object sits around world (0, 0, 4): pixel (u, v) at depth zc back-projects to (x + (u-64)/128*zc, ...)
        zc = 4.0 - z
        px = [(int(round(256 - x / zc * 128)) + du, int(round(256 - y / zc * 128)) + dv, zc, 1) for du in range(-2, 3) for dv in range(-2, 3)]
        depth, mask = hand_frame(HV, WV, px)
        T = I4.copy(); T[:3, 3] = [x, y, z]
        m.integrate(depth, mask, pow2_K(128.0, 256.0, 256.0), T, e[:1], 1)
    return m


def test_V_direction_and_distance_rules(oracle):
    """V2 with the default 30 degree threshold (cos = 0.866) and closer ratio 0.8, object at (0, 0, 4):
    (0,0,0) first view, always kept;  (0.35,0,0): 5 degrees off, same distance -> dropped;  (3,0,0): 36.9 degrees
    -> kept;  (0,0,1.5): same direction as the first but distance 2.5 < 0.8 * 4 -> kept (sufficiently closer)."""
    m = _view_scene(oracle, 4, [(0, 0, 0), (0.35, 0, 0), (3.0, 0, 0), (0, 0, 1.5)])
    views, counts = m.read_views()
    assert counts[0] == 3 and len(m.read()[0]) == 1
    assert list(views[0]["frame"][:3]) == [0, 2, 3]
    assert np.allclose(views[0]["dist"][:3], [4.0, 5.0, 2.5], atol=0.05)
    assert np.allclose(views[0]["dir"][0], [0, 0, 1], atol=0.02) and np.allclose(views[0]["dir"][1], [-0.6, 0, 0.8], atol=0.02)
    assert np.allclose(np.linalg.norm(views[0]["dir"][:3], axis=1), 1.0, atol=1e-6)
    assert np.array_equal(views[0]["cam"][1], [3.0, 0, 0])


def test_V_full_set_replaces_the_farthest_view_only_if_closer(oracle):
    """k = 2: views at distance 4 (dir 0 deg) and 5 (36.9 deg) fill the set; a third direction at distance 5.66 is
    dropped (not closer than the farthest kept), a fourth (45 degrees, distance 4.24) replaces the farthest (the 5.0 one)."""
    m = _view_scene(oracle, 2, [(0, 0, 0), (3.0, 0, 0), (-4.0, 0, 0), (-3.0, 0, 1.0)])
    views, counts = m.read_views()
    assert counts[0] == 2
    assert list(views[0]["frame"]) == [0, 3]                        # slot of the replaced view is reused
    assert np.allclose(views[0]["dist"], [4.0, np.sqrt(18.0)], atol=0.05)
    # k = 0: off, nothing is stored
    m0 = _view_scene(oracle, 0, [(0, 0, 0)])
    assert m0.read_views()[1].sum() == 0


# ================================================================================================ Q: retrieval scoring
def _query_inputs(N=40, dims=(16, 12, 20), seed=3):
    g = np.random.default_rng(seed)
    emb = [unit_rows(N, d, seed + i) for i, d in enumerate(dims)]
    cls = g.integers(0, 4, N).astype(np.int32)
    cen = g.uniform(-3, 3, (N, 3)).astype(np.float32)
    alive = np.ones(N, np.uint8)
    qt = [unit_rows(1, dims[0], 50)[0], unit_rows(1, dims[0], 51)[0], unit_rows(1, dims[1], 52)[0], unit_rows(1, dims[2], 53)[0]]
    return alive, emb, cls, cen, qt


def test_Q_rrf_by_hand_on_five_entities(oracle):
    """Q1-Q2 by hand: five entities, one-hot-like embeddings so that each channel's order is known.
    s_sem = sum_c w_c / (5 + rank_c), w = 1.0, 0.5, 0.75, 1.0."""
    N = 5
    e = np.eye(5, dtype=np.float32)
    # space 0: similarity to q = e0 decreases with index;  space 1: reversed;  space 2: order 2, 0, 1, 3, 4
    emb0 = np.stack([e[0] * (1 - 0.1 * i) + e[1] * (0.1 * i + 1e-3) for i in range(5)])
    emb1 = emb0[::-1].copy()
    emb2 = np.stack([e[0] * x + e[1] * (1 - x) for x in (0.8, 0.7, 0.9, 0.4, 0.2)])
    q = [e[0], e[0], e[0], e[0]]
    r = oracle.query(np.ones(N, np.uint8), [emb0, emb1, emb2], np.zeros(N, np.int32), np.zeros((N, 3), np.float32), q, -1, [], [], 3)
    ranks = [np.array([1, 2, 3, 4, 5]), np.array([1, 2, 3, 4, 5]), np.array([5, 4, 3, 2, 1]), np.array([2, 3, 1, 4, 5])]
    w = [1.0, 0.5, 0.75, 1.0]
    expect = sum(wc / (5.0 + rk) for wc, rk in zip(w, ranks))
    assert np.abs(r["s_sem"] - expect).max() < 1e-6
    assert np.abs(r["s"] - expect).max() < 1e-6 and (r["gbar"] == 1).all()                 # no predicate: gbar = 1
    assert list(r["top"]) == list(np.argsort(-expect, kind="stable")[:3])


def test_Q_ranks_against_numpy_argsort_and_class_factor(oracle):
    alive, emb, cls, cen, qt = _query_inputs()
    alive[[7, 19]] = 0
    r = oracle.query(alive, emb, cls, cen, qt, 2, [], [], 10, want_cos=True)
    live = np.nonzero(alive)[0]
    s = np.zeros(len(alive))
    for ch, (sp, wc) in enumerate(zip((0, 0, 1, 2), (1.0, 0.5, 0.75, 1.0))):
        c = (emb[sp].astype(np.float64) @ qt[ch].astype(np.float64)) / (np.linalg.norm(emb[sp], axis=1) * np.linalg.norm(qt[ch]))
        assert np.abs(r["cos"][ch][live] - c[live]).max() < 1e-6
        order = live[np.argsort(-c[live], kind="stable")]
        rank = np.empty(len(alive)); rank[order] = np.arange(1, len(live) + 1)
        s[live] += wc / (5.0 + rank[live])
    s[cls != 2] *= 0.3                                                                       # soft class factor
    s[alive == 0] = 0
    assert np.abs(r["s_sem"] - s).max() < 1e-6
    top = live[np.argsort(-s[live], kind="stable")][:10]
    assert list(r["top"]) == list(top) and (r["s"][alive == 0] == 0).all()


def test_Q_predicates_closed_forms_and_composite(oracle):
    """Q4-Q5: Near(d) = exp(-d^2 / (2 * 0.5^2)): Near(0) = 1, Near(0.5) = e^-1/2; NextTo with sigma = 1: NextTo(1) = e^-1/2;
    Closest / Farthest = 1 / (|rank - r*| + 1); s = s_sem * (0.5 + 0.5 * gbar), gbar = geometric mean."""
    alive, emb, cls, cen, qt = _query_inputs(N=12)
    # the landmark query equals entity 4's embeddings in every space -> rank 1 in all channels -> bound to 4
    ql = [emb[0][4], emb[0][4], emb[1][4], emb[2][4]]
    cen[:] = 0
    cen[:, 0] = np.arange(12) * 0.25                                 # entity o sits |o - 4| * 0.25 m from the landmark
    d = np.abs(np.arange(12) - 4) * 0.25
    base = oracle.query(alive, emb, cls, cen, qt, -1, [], [], 12)
    for ptype, g in ((oracle.PRED_NEAR, np.exp(-d * d / 0.5)), (oracle.PRED_NEXTTO, np.exp(-d * d / 2.0))):
        r = oracle.query(alive, emb, cls, cen, qt, -1, [ptype], [ql], 12)
        assert list(r["landmarks"]) == [4]
        assert np.abs(r["gbar"] - g).max() < 1e-6 and r["gbar"][4] == 1.0
        assert np.abs(r["s"] - base["s_sem"] * (0.5 + 0.5 * g)).max() < 1e-6
    assert abs(np.exp(-0.5) - oracle.query(alive, emb, cls, cen, qt, -1, [oracle.PRED_NEAR], [ql], 1)["gbar"][6]) < 1e-6   # d = 0.5 = sigma
    assert abs(np.exp(-0.5) - oracle.query(alive, emb, cls, cen, qt, -1, [oracle.PRED_NEXTTO], [ql], 1)["gbar"][8]) < 1e-6  # d = 1.0 = sigma
    # ranks by distance to the landmark (ties -> lower id): 4 | 3 5 | 2 6 | 1 7 | 0 8 | 9 10 11
    rank = np.array([8, 6, 4, 2, 1, 3, 5, 7, 9, 10, 11, 12])
    r = oracle.query(alive, emb, cls, cen, qt, -1, [oracle.PRED_CLOSEST], [ql], 12)
    assert np.abs(r["gbar"] - 1.0 / (np.abs(rank - 1) + 1)).max() < 1e-6
    r = oracle.query(alive, emb, cls, cen, qt, -1, [oracle.PRED_FARTHEST], [ql], 12)
    assert np.abs(r["gbar"] - 1.0 / (np.abs(rank - 12) + 1)).max() < 1e-6
    # two predicates: geometric mean
    r = oracle.query(alive, emb, cls, cen, qt, -1, [oracle.PRED_NEAR, oracle.PRED_CLOSEST], [ql, ql], 12)
    gm = np.sqrt(np.exp(-d * d / 0.5) * (1.0 / (np.abs(rank - 1) + 1)))
    assert np.abs(r["gbar"] - gm).max() < 1e-6
    s = base["s_sem"] * (0.5 + 0.5 * gm)
    assert np.abs(r["s"] - s).max() < 1e-6 and list(r["top"]) == list(np.argsort(-r["s"], kind="stable"))


# ================================================================================================ W: weighted covisibility edges
def _bhatt_np(mu1, S1, mu2, S2):
    Sb = 0.5 * (S1 + S2)
    d = mu1 - mu2
    return 0.125 * d @ np.linalg.solve(Sb, d) + 0.5 * np.log(np.linalg.det(Sb) / np.sqrt(np.linalg.det(S1) * np.linalg.det(S2)))


def test_W_bhattacharyya_closed_forms(oracle):
    """W2's distance: equal isotropic covariances -> DB = |dmu|^2 / (8 sigma^2); equal means -> the log term alone;
    H = sqrt(1 - exp(-DB)) against the pinned Hellinger routine; the general formula through numpy.linalg."""
    iso = lambda v: np.array([v, 0, 0, v, 0, v], np.float64)
    z = np.zeros(3)
    assert abs(oracle.bhattacharyya(z, iso(0.04), np.array([1.0, 0, 0]), iso(0.04), 0.0) - 1.0 / (8 * 0.04)) < 1e-12
    assert abs(oracle.bhattacharyya(z, iso(1.0), z, iso(4.0), 0.0) - 1.5 * np.log(2.5 / 2.0)) < 1e-12
    g = np.random.default_rng(4)
    pk = lambda M_: np.array([M_[0, 0], M_[0, 1], M_[0, 2], M_[1, 1], M_[1, 2], M_[2, 2]])
    for _ in range(30):
        A, B = g.standard_normal((3, 3)), g.standard_normal((3, 3))
        S1, S2 = A @ A.T + 0.1 * np.eye(3), B @ B.T + 0.1 * np.eye(3)
        mu1, mu2 = g.standard_normal(3), g.standard_normal(3) * 2
        db = oracle.bhattacharyya(mu1, pk(S1), mu2, pk(S2), 0.01)
        assert abs(db - _bhatt_np(mu1, S1 + 0.01 * np.eye(3), mu2, S2 + 0.01 * np.eye(3))) < 1e-9
        assert abs(np.sqrt(1 - np.exp(-db)) - oracle.hellinger(mu1, pk(S1), mu2, pk(S2), 0.01)) < 1e-9
    # far apart: H has saturated, DB still orders the pairs
    far1 = oracle.bhattacharyya(z, iso(0.01), np.array([5.0, 0, 0]), iso(0.01), 0.0)
    far2 = oracle.bhattacharyya(z, iso(0.01), np.array([6.0, 0, 0]), iso(0.01), 0.0)
    assert far2 > far1 > 100 and oracle.hellinger(z, iso(0.01), np.array([5.0, 0, 0]), iso(0.01), 0.0) == 1.0


def _two_patches(labels=(1, 2)):
    px = [(40 + du, 40 + dv, 2.0, labels[0]) for du in range(4) for dv in range(4)]
    if len(labels) > 1:
        px += [(90 + du, 40 + dv, 2.0, labels[1]) for du in range(4) for dv in range(4)]
    return hand_frame(H, W, px)


def test_W_decay_closed_form(oracle):
    """W4 with decay 0.5 and k = 1: the pair {0, 1} is co-observed in calls 1, 2 and 4 (call 3 sees object 0 alone):
    w = ((1 * 0.5 + 1) * 0.25) + 1 = 1.375 at call 4, 0.6875 one call later without an observation."""
    e = np.eye(4, dtype=np.float32)
    m = oracle.OracleMap(0.25, 4, 0.5, 0.5, 0.5, 0, H, W)
    m.set_option(m.OPT_EDGES_K, 1)
    m.set_option(m.OPT_EDGE_DECAY, 0.5)
    both, one = _two_patches(), _two_patches((1,))
    for call, (fr, n) in enumerate([(both, 2), (both, 2), (one, 1), (both, 2)]):
        m.integrate(fr[0], fr[1], pow2_K(), I4, e[:n], n)
    a, b, w = m.read_edges()
    assert list(a) == [0] and list(b) == [1] and abs(w[0] - 1.375) < 1e-6
    m.integrate(one[0], one[1], pow2_K(), I4, e[:1], 1)
    assert abs(m.read_edges()[2][0] - 0.6875) < 1e-6
    assert len(m.read()[0]) == 2


@pytest.mark.parametrize("k,cut", [(2, 2.0), (3, 1.05)])
def test_W_knn_graph_against_brute_force(oracle, k, cut):
    """W1-W4 on configs[0] in batches of 3 frames: the kNN graph in Hellinger order (through the Bhattacharyya distance,
    W2), the median cutoff and the decayed weights rebuilt in Python from the exported (pinned: G-P1, G-P2) entity
    Gaussians with a numpy.linalg Bhattacharyya distance."""
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    m = oracle.OracleMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, cfg.dtype, cfg.H, cfg.W)
    m.set_option(m.OPT_EDGES_K, k)
    m.set_option(m.OPT_EDGE_CUTOFF, cut)
    decay, eps2 = 0.9, float(np.float32(cfg.voxel)) ** 2
    edges, n_dropped = {}, 0
    for call in range(1, 7):
        frames = [sc.frame(3 * (call - 1) + i) for i in range(3)]
        depth = np.stack([f.depth for f in frames]); mask = np.stack([f.mask for f in frames])
        K = np.stack([f.K for f in frames]); T = np.stack([f.T for f in frames])
        m.integrate_batch(depth, mask, K, T, np.concatenate([f.desc for f in frames]), [f.n_det for f in frames])
        assoc = m.last_assoc()[0]
        wgt, mu, cov = m.read_gaussians()
        Sset = sorted({int(t) for t in assoc if t >= 0 and wgt[t] > 0})
        touched = set()
        for a in Sset:
            d = sorted((np.float32(_bhatt_np(mu[a].astype(np.float64), _unpack(cov[a]) + eps2 * np.eye(3),
                                             mu[b].astype(np.float64), _unpack(cov[b]) + eps2 * np.eye(3))), b) for b in Sset if b != a)
            kk = min(k, len(d))
            if kk == 0:
                continue
            med = d[(kk - 1) // 2][0]
            if kk < len(d):
                assert d[kk][0] - d[kk - 1][0] > 1e-5 * d[kk][0], "kNN boundary too close: change the seed"
            for dist, b in d[:kk]:
                assert abs(float(dist) - cut * float(med)) > 1e-5 * float(dist) or dist == med, "cutoff too close"
                if dist <= np.float32(cut) * med:
                    touched.add((min(a, b), max(a, b)))
                else:
                    n_dropped += 1
        for e in touched:
            w, t = edges.get(e, (0.0, call))
            edges[e] = (w * decay ** (call - t) + 1.0, call)
        a_, b_, w_ = m.read_edges()
        exp = sorted(edges.items())
        assert list(zip(a_.tolist(), b_.tolist())) == [e for e, _ in exp]
        assert np.abs(w_ - np.array([w * decay ** (call - t) for _, (w, t) in exp])).max() < 1e-5
    assert len(edges) > 5 and (cut > 1.5 or n_dropped > 0)
