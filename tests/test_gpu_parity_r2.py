"""`-m gpu`, round 2: the decision paths and sizes round 1 left without evidence.

* w_sem > tau: a non-overlapping object can pass the threshold, so the matched object's id comes from the dense
  similarity epilogue (row argmax, lowest id on ties, R16/R18/R19) -- on the tcgen05 path (several tiles on both
  axes), the CUDA-core FMA path, and with exact ties (bit-identical map rows).
* `farm_debug_last_dense` against the oracle's dense (max, argmax).
"""
import dataclasses

import numpy as np
import pytest

from helpers import generate_frames, hand_frame, integrate_frames, margin_filter, pack_key, pow2_K, unit_rows
from paper_2606_15476_b200 import FarmMap, scenes as S
from parity import TOL, compare_call, compare_dense, compare_maps, dense_decided, gpu_integrate, make_pair

pytestmark = pytest.mark.gpu

WEIGHTS = [(0.3, 0.7, 0.5), (0.0, 1.0, 0.6)]


def _with_weights(cfg, w):
    return dataclasses.replace(cfg, w_geo=w[0], w_sem=w[1], tau=w[2])


@pytest.mark.parametrize("w", WEIGHTS)
def test_dense_argmax_decides_on_config2_distractor_clusters(oracle, w):
    """configs[2] (0.9-cosine distractor clusters, D=1024 bf16, tcgen05 path) with w_sem > tau: cluster members match
    one another without sharing a voxel, so the dense argmax decides."""
    cfg = _with_weights(S.get_config(2), w)
    frames_all = generate_frames(2, range(0, 40))
    o, g = make_pair(oracle, cfg)
    n_dense, n_rows = 0, 0
    for fr in frames_all:
        frames = margin_filter(o.clone, [fr], cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o)
        n_rows += compare_dense(g, o)
        n_dense += dense_decided(o)
    compare_maps(g, o)
    assert n_dense >= 5 and n_rows > 500, (n_dense, n_rows)


def _stress_frames_with_far_matches(sc, b, desc_map, rng):
    """batch b of the mini stress scene; the detections that look at empty space get the descriptor of a random FILLER
    object (+ view noise) instead of a fresh one: with w_sem > tau they match that object without any voxel overlap"""
    out = []
    n_t = len(sc._blob_ijk)
    for fr in sc.batch(b):
        desc = S.storage_to_f32(fr.desc, sc.cfg.dtype).copy()
        for d in np.nonzero(fr.box_ids < 0)[0]:
            tgt = int(rng.integers(n_t, len(desc_map)))
            v = desc_map[tgt] + (0.1 / np.sqrt(desc.shape[1])) * rng.standard_normal(desc.shape[1])
            desc[d] = v / np.linalg.norm(v)
        out.append(S.Frame(fr.depth, fr.mask, fr.K, fr.T, S.to_storage(desc.astype(np.float32), sc.cfg.dtype), fr.n_det, fr.box_ids))
    return out


@pytest.mark.parametrize("sim_path", [2, 3])
@pytest.mark.parametrize("w", WEIGHTS)
def test_dense_argmax_decides_multi_tile_tensor_path(oracle, w, sim_path):
    """M = 400 detections x N >= 700 objects, D = 1024 bf16: more than one tile on both axes of similarity_tc_kernel
    (128 x 256); half of the detections can only match through the dense argmax."""
    from paper_2606_15476_b200.binding import OBJECT_DTYPE
    sc = S.StressScene(n_batches=2, frames_per_batch=4, n_objects=700)
    cfg = _with_weights(sc.cfg, w)
    ijk, owner, n_vox, desc = sc.build_map()
    keys = pack_key(ijk[:, 0], ijk[:, 1], ijk[:, 2])
    objs = np.zeros(len(n_vox), OBJECT_DTYPE)
    objs["id"], objs["n_voxels"], objs["n_obs"], objs["best_frame"], objs["best_det"] = np.arange(len(n_vox)), n_vox, 1, -1, -1
    o, g = make_pair(oracle, cfg, max_det_per_call=1600, max_objects=len(n_vox) + 8000, sim_path=sim_path)
    assert o.import_(objs, desc, keys, owner) == 0
    g.import_(objs, desc, keys, owner)
    rng = np.random.default_rng(17)
    n_dense = 0
    for b in range(2):
        frames = margin_filter(o.clone, _stress_frames_with_far_matches(sc, b, desc, rng), cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o)
        assert compare_dense(g, o) > 300
        n_dense += dense_decided(o)
    compare_maps(g, o)
    assert n_dense > 250, n_dense


@pytest.mark.parametrize("cfg_id,sim_path,n", [(0, 0, 20), (1, 1, 30), (1, 2, 30)])
@pytest.mark.parametrize("w", WEIGHTS)
def test_dense_argmax_decides_fma_and_small_tensor_paths(oracle, w, cfg_id, sim_path, n):
    """fp32 (configs[0], CUDA-core FMA), and configs[1] (f16) forced through the FMA path and the tcgen05 path."""
    cfg = _with_weights(S.get_config(cfg_id), w)
    frames_all = generate_frames(cfg_id, range(20, 20 + n) if cfg_id == 1 else range(n))
    o, g = make_pair(oracle, cfg, sim_path=sim_path)
    rows = 0
    for fr in frames_all:
        frames = margin_filter(o.clone, [fr], cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o)
        rows += compare_dense(g, o)
    compare_maps(g, o)
    assert rows > 50


@pytest.mark.parametrize("dtype,sim_path", [(0, 0), (1, 1), (1, 2), (2, 1), (2, 2), (1, 3), (2, 3)])
def test_exact_ties_go_to_the_lowest_id(oracle, dtype, sim_path):
    """R18 with bit-identical map rows (same tile, neighbouring tiles, far tiles of the 128 x 256 tensor tiling) and
    detections equal to them: cosine clamps to exactly 1 for all of them and the lowest id must win -- in the dense
    argmax and in the decision (w_geo = 0, w_sem = 1, tau = 0.6: the dense argmax IS the decision)."""
    from paper_2606_15476_b200.binding import OBJECT_DTYPE
    D, N = 64, 900
    H, W = 96, 128
    rows = unit_rows(N, D, 41)
    groups = [[5, 300, 301], [310, 400], [255, 256], [700, 12, 899]]
    for grp in groups:
        for i in grp[1:]:
            rows[i] = rows[grp[0]]
    det = np.stack([rows[g[0]] for g in groups] + [rows[77]]).astype(np.float32)
    Mdet = len(det)

    class Cfg:
        voxel, w_geo, w_sem, tau = 0.25, 0.0, 1.0, 0.6
    Cfg.D, Cfg.dtype = D, dtype
    o, g = make_pair(oracle, Cfg, H=H, W=W, sim_path=sim_path)
    objs = np.zeros(N, OBJECT_DTYPE)
    objs["id"], objs["n_voxels"], objs["n_obs"], objs["best_frame"], objs["best_det"] = np.arange(N), 1, 1, -1, -1
    keys = pack_key(np.arange(N) + 500, np.zeros(N, int), np.zeros(N, int))
    assert o.import_(objs, rows, keys, np.arange(N, dtype=np.uint32)) == 0
    g.import_(objs, rows, keys, np.arange(N, dtype=np.uint32))
    depth, mask = hand_frame(H, W, [(8 + 16 * d, 48, 2.0, d + 1) for d in range(Mdet)])
    fr = S.Frame(depth, mask, pow2_K(), np.eye(4, dtype=np.float32), S.to_storage(det, dtype), Mdet, np.zeros(Mdet, np.int64))
    integrate_frames(o, [fr])
    gpu_integrate(g, [fr], dtype)
    ao, no, bo, _, _ = o.last_assoc()
    ag, ng, bg, _ = g.last_assoc()
    assert np.array_equal(ag, ao) and np.array_equal(ng, no) and np.abs(bg - bo).max() <= TOL
    mc_o, am_o = o.last_dense()
    mc_g, am_g = g.debug_last_dense()
    assert np.array_equal(am_g, am_o) and np.abs(mc_g - mc_o).max() <= TOL
    assert list(ao) == [5, 310, 255, 12, 77] and not no.any()
    compare_maps(g, o)


def test_resume_continues_frame_numbering_and_import_checks_counts(oracle):
    """Scene-state resume: export, import into a new map, set the frame counter, continue -- best-view
    records keep global frame numbers.  An object whose n_voxels disagrees with its voxel list is rejected."""
    from paper_2606_15476_b200 import FarmError
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    o, g = make_pair(oracle, cfg)
    for k in range(6):
        fr = sc.frame(k)
        integrate_frames(o, [fr])
        gpu_integrate(g, [fr], cfg.dtype)
    assert g.get_frame_seq() == 6
    objs, desc, keys, owners = g.read()
    g2 = FarmMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, H=cfg.H, W=cfg.W, dtype=cfg.dtype)
    g2.import_(objs, desc, keys, owners)
    g2.set_frame_seq(6)
    with pytest.raises(FarmError):
        g2.set_frame_seq(3)                                        # only forward
    for k in range(6, 12):
        frames = margin_filter(o.clone, [sc.frame(k)], cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g2, frames, cfg.dtype)
        compare_call(g2, o)
    compare_maps(g2, o)                                            # includes best_frame of views taken after the resume
    assert g2.get_frame_seq() == 12
    bad = objs.copy()
    bad["n_voxels"][0] += 1
    g3 = FarmMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, H=cfg.H, W=cfg.W, dtype=cfg.dtype)
    with pytest.raises(FarmError) as ei:
        g3.import_(bad, desc, keys, owners)
    assert ei.value.code == -1 and "n_voxels" in str(ei.value)


def test_misaligned_descriptors_fail_before_anything_is_enqueued(oracle):
    """A 16-bit descriptor pointer that TMA cannot address is refused with FARM_ERR_INVALID_ARG and the map, the frame
    counter and the per-call results are untouched; the next (aligned) call is exact."""
    import torch
    from paper_2606_15476_b200 import FarmError
    from parity import upload
    cfg = S.get_config(1)
    frames = generate_frames(1, range(20, 24))
    o, g = make_pair(oracle, cfg, sim_path=2)
    for fr in frames[:2]:
        integrate_frames(o, [fr])
        gpu_integrate(g, [fr], cfg.dtype)
    def snapshot():
        objs, desc, keys, owners = g.read()
        order = np.argsort(keys)                                # the export order of voxels is arbitrary
        return objs, desc, keys[order], owners[order]
    before = snapshot()
    d = upload([frames[2]], cfg.dtype)
    raw = torch.empty(d["desc"].numel() + 8, dtype=d["desc"].dtype, device="cuda")
    off = raw[1:1 + d["desc"].numel()].view(d["desc"].shape)        # 2 bytes off a 16-byte boundary
    off.copy_(d["desc"])
    assert off.data_ptr() % 16 != 0
    with pytest.raises(FarmError) as ei:
        g.integrate_batch(1, d["depth"], d["mask"], d["K"], d["T"], off.data_ptr(), d["n_det"])
    assert ei.value.code == -1
    assert g.get_frame_seq() == 2
    after = snapshot()
    assert all(np.array_equal(a, b) for a, b in zip(before, after))
    for fr in frames[2:]:
        fl = margin_filter(o.clone, [fr], cfg.tau)
        integrate_frames(o, fl)
        gpu_integrate(g, fl, cfg.dtype)
        compare_call(g, o)
    compare_maps(g, o)


def test_launch_blocking_environment_selects_the_single_stream_order(oracle, monkeypatch):
    """CUDA_LAUNCH_BLOCKING serialises kernels, which the device-side waits of the default order cannot survive: the
    library then uses the single-stream order (no waits) and still reproduces the oracle."""
    monkeypatch.setenv("CUDA_LAUNCH_BLOCKING", "1")
    cfg = S.get_config(1)
    frames_all = generate_frames(1, range(20, 26))
    o, g = make_pair(oracle, cfg)
    for fr in frames_all:
        frames = margin_filter(o.clone, [fr], cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o)
    compare_maps(g, o)


def _compare_views(g, o):
    vo, co = o.read_views()
    vg, cg = g.read_views()
    assert np.array_equal(cg, co)
    for i in range(len(co)):
        k = int(co[i])
        for fld in ("frame", "det", "n_px"):
            assert np.array_equal(vg[i][fld][:k], vo[i][fld][:k]), (i, fld)
        for fld in ("cam", "dir", "dist"):
            assert np.array_equal(vg[i][fld][:k], vo[i][fld][:k]), (i, fld)      # fp32 on both sides, same operation order
    return int(co.sum())


@pytest.mark.parametrize("cfg_id,n,per_call,k,vcos", [(0, 20, 1, 3, None), (0, 18, 3, 2, None), (1, 40, 1, 2, 0.97)])
def test_view_diversity_sets_match_oracle(oracle, cfg_id, n, per_call, k, vcos):
    """V1-V2 (PAPER.md:353 step 6, "up to k representative views"): which views every object keeps, and their
    records, bit-exact -- single-frame and batched calls, set sizes 2..4 so that replacement of the farthest view occurs."""
    cfg = S.get_config(cfg_id)
    frames_all = generate_frames(cfg_id, range(20, 20 + n) if cfg_id == 1 else range(n))
    o, g = make_pair(oracle, cfg, views=k, view_cos=vcos)
    o.set_option(o.OPT_VIEWS_K, k)
    if vcos is not None:
        o.set_option(o.OPT_VIEW_COS, vcos)
    for c in range(0, n, per_call):
        frames = margin_filter(o.clone, frames_all[c:c + per_call], cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o, check_sets=False)
        total = _compare_views(g, o)
    compare_maps(g, o, voxels=False)
    _, counts = o.read_views()
    assert total > len(counts) and counts.max() == k           # some objects hold several views, some sets are full


# ------------------------------------------------------------------------------------------------ retrieval scoring (Q1-Q5)
def _ternary_rows(n, d, nnz, rng):
    """rows with exactly nnz entries of +-1: all norms equal and every dot product is an exact small integer, so the
    cosine ORDER (hence every rank) is the same in any accumulation order and precision"""
    out = np.zeros((n, d), np.float32)
    for i in range(n):
        idx = rng.choice(d, nnz, replace=False)
        out[i, idx] = rng.choice([-1.0, 1.0], nnz)
    return out


def _query_scene(oracle, gaussian):
    """mini stress scene, imported with random object boxes, one batch integrated (new objects carry Gaussians)"""
    from paper_2606_15476_b200.binding import OBJECT_DTYPE
    sc = S.StressScene(n_batches=1, frames_per_batch=4, n_objects=700)
    cfg = sc.cfg
    ijk, owner, n_vox, desc = sc.build_map()
    keys = pack_key(ijk[:, 0], ijk[:, 1], ijk[:, 2])
    rng = np.random.default_rng(5)
    objs = np.zeros(len(n_vox), OBJECT_DTYPE)
    objs["id"], objs["n_voxels"], objs["n_obs"], objs["best_frame"], objs["best_det"] = np.arange(len(n_vox)), n_vox, 1, -1, -1
    c = rng.uniform(-4, 4, (len(n_vox), 3)).astype(np.float32)
    objs["aabb_min"], objs["aabb_max"] = c - 0.25, c + 0.25
    o, g = make_pair(oracle, cfg, max_det_per_call=1600, max_objects=len(n_vox) + 8000, gaussian=gaussian)
    assert o.import_(objs, desc, keys, owner) == 0
    g.import_(objs, desc, keys, owner)
    frames = margin_filter(o.clone, sc.batch(0), cfg.tau)
    integrate_frames(o, frames)
    gpu_integrate(g, frames, cfg.dtype)
    compare_call(g, o, check_sets=False)
    objs_o, _, _, _ = o.read(voxels=False)
    alive = (objs_o["n_obs"] > 0).astype(np.uint8)
    cen = (0.5 * (objs_o["aabb_min"].astype(np.float64) + objs_o["aabb_max"].astype(np.float64))).astype(np.float32)
    if gaussian:
        w, mu, _ = o.read_gaussians()
        cen[w > 0] = mu[w > 0]
    return o, g, alive, cen


@pytest.mark.parametrize("emb_dtype,gaussian", [(0, 1), (2, 0)])
def test_retrieval_scoring_exact_ranks(oracle, emb_dtype, gaussian):
    """Q1-Q5 against the oracle on ~1,100 entities: reciprocal-rank fusion over four channels in three
    embedding spaces, landmark binding, Near / NextTo / Closest / Farthest, composite score, class factor, top-K.
    Embeddings are +-1/0 rows of equal norm, so every rank is decided by exact integer dot products on both sides."""
    import torch
    o, g, alive, cen = _query_scene(oracle, gaussian)
    N = len(alive)
    rng = np.random.default_rng(23)
    dims, nnz = (64, 48, 96), (24, 16, 32)
    emb = [_ternary_rows(N, d, z, rng) for d, z in zip(dims, nnz)]
    cls = rng.integers(0, 5, N).astype(np.int32)
    tdt = {0: torch.float32, 1: torch.float16, 2: torch.bfloat16}[emb_dtype]
    emb_dev = [torch.from_numpy(e).to("cuda").to(tdt).contiguous() for e in emb]
    cls_dev = torch.from_numpy(cls).to("cuda")
    qv = lambda sp: _ternary_rows(1, dims[sp], nnz[sp], rng)[0]
    qt = [qv(0), qv(0), qv(1), qv(2)]
    lm_ids = [int(rng.integers(0, N)), int(rng.integers(0, N)), int(rng.integers(0, N))]
    # each landmark variable asks for one particular entity: its own embeddings, rank 1 in every channel
    qls = [[emb[0][i], emb[0][i], emb[1][i], emb[2][i]] for i in lm_ids]
    cases = [([], [], -1), ([oracle.PRED_NEAR], qls[:1], 3), ([oracle.PRED_NEXTTO, oracle.PRED_CLOSEST], qls[:2], -1),
             ([oracle.PRED_FARTHEST, oracle.PRED_NEAR, oracle.PRED_CLOSEST], qls, 1)]
    for ptypes, ql, tcls in cases:
        ro = oracle.query(alive, emb, cls, cen, qt, tcls, ptypes, ql, 20)
        rg = g.query(emb_dev, emb_dtype, cls_dev, qt, tcls, ptypes, ql, 20)
        assert np.array_equal(rg["landmarks"], ro["landmarks"])
        assert np.abs(rg["s_sem"] - ro["s_sem"]).max() <= 1e-6
        assert np.abs(rg["gbar"] - ro["gbar"]).max() <= 1e-5
        assert np.abs(rg["s"] - ro["s"]).max() <= 1e-6
        so = np.sort(ro["s"])[::-1]
        k_ok = 20
        for k in range(20):                                        # compare the prefix whose scores are clearly separated
            if so[k] - so[k + 1] <= 1e-6:
                k_ok = k
                break
        assert np.array_equal(rg["top"][:k_ok], ro["top"][:k_ok]) and k_ok >= 3
        assert np.abs(rg["top_scores"][:k_ok] - ro["s"][ro["top"][:k_ok]]).max() <= 1e-6
    assert list(ro["landmarks"]) == [min(np.nonzero((emb[0] == emb[0][i]).all(1))[0]) for i in lm_ids]


def test_retrieval_scoring_float_embeddings_robust_entities(oracle):
    """random unit float embeddings (bf16): cosines within 1e-3 of the oracle's; s_sem equal for every entity whose cosine is
    separated from both of its rank neighbours by more than 1e-5 in every channel (a swap of two near-tied entities
    changes only those two)."""
    import torch
    o, g, alive, cen = _query_scene(oracle, 0)
    N = len(alive)
    dims = (128, 64, 256)
    emb = [S.bf16_bits_to_f32(S.f32_to_bf16_bits(unit_rows(N, d, 70 + i))) for i, d in enumerate(dims)]
    emb_dev = [torch.from_numpy(e).to("cuda").to(torch.bfloat16).contiguous() for e in emb]
    qt = [unit_rows(1, dims[0], 80)[0], unit_rows(1, dims[0], 81)[0], unit_rows(1, dims[1], 82)[0], unit_rows(1, dims[2], 83)[0]]
    ro = oracle.query(alive, emb, np.zeros(N, np.int32), cen, qt, -1, [], [], 10, want_cos=True)
    rg = g.query(emb_dev, 2, None, qt, -1, [], [], 10)
    robust = np.ones(N, bool)
    for ch in range(4):
        c = ro["cos"][ch].astype(np.float64)
        order = np.argsort(-c, kind="stable")
        gap = np.full(N, np.inf)
        d = np.abs(np.diff(c[order]))
        gap[order[1:]] = np.minimum(gap[order[1:]], d)
        gap[order[:-1]] = np.minimum(gap[order[:-1]], d)
        robust &= gap > 1e-5
    assert robust.sum() > 0.5 * N
    assert np.abs(rg["s_sem"] - ro["s_sem"])[robust].max() <= 1e-6
    assert np.abs(rg["s_sem"] - ro["s_sem"]).max() <= 0.02


# ------------------------------------------------------------------------------------------------ correspondence (U1-U4)
def _compare_corr(g, o):
    assert np.array_equal(g.read_alias(), o.read_alias())
    lg, wg = g.last_merges()
    lo, wo = o.last_merges()
    order = np.argsort(lo)
    assert np.array_equal(lg, lo[order]) and np.array_equal(wg, wo[order])
    return len(lo)


def test_correspondence_hand_cases(oracle):
    """The oracle's U pins through the CUDA path: a detection bridging two entities (winner = lowest id, voxels re-owned,
    count-weighted descriptor), a chain of three entities joined by two detections, and a same-call duplicate spawn."""
    from paper_2606_15476_b200.binding import OBJECT_DTYPE
    H, W = 128, 128
    I4 = np.eye(4, dtype=np.float32)
    E = np.eye(8, dtype=np.float32)

    class Cfg:
        voxel, D, w_geo, w_sem, tau, dtype = 0.25, 8, 0.5, 0.5, 0.5, 0

    def pair():
        o, g = make_pair(oracle, Cfg, H=H, W=W, correspondence=1)
        o.set_option(o.OPT_CORRESPONDENCE, 1)
        return o, g

    def objs(nv, nobs=None):
        ob = np.zeros(len(nv), OBJECT_DTYPE)
        ob["id"], ob["n_voxels"], ob["n_obs"], ob["best_frame"], ob["best_det"] = np.arange(len(nv)), nv, nobs or 1, -1, -1
        return ob

    def frame(px, desc):
        depth, mask = hand_frame(H, W, px)
        return S.Frame(depth, mask, pow2_K(), I4, np.ascontiguousarray(desc, np.float32), len(desc), np.zeros(len(desc), np.int64))

    four = lambda lab, v: [(64 + 16 * i, v, 2.0, lab) for i in range(4)]
    # (1) bridge
    o, g = pair()
    keys = np.array([pack_key(0, 0, 8), pack_key(1, 0, 8), pack_key(2, 0, 8), pack_key(3, 0, 8), pack_key(90, 0, 0)], np.uint64)
    owners = np.array([0, 0, 1, 1, 2], np.uint32)
    ob, desc = objs([2, 2, 1], [3, 1, 1]), np.stack([E[0], E[1], E[5]])
    assert o.import_(ob, desc, keys, owners) == 0
    g.import_(ob, desc, keys, owners)
    fr = frame(four(1, 48), [(E[0] + E[1]) / np.sqrt(2)])
    for _ in range(2):
        integrate_frames(o, [fr])
        gpu_integrate(g, [fr], 0)
        compare_call(g, o)
        _compare_corr(g, o)
    assert list(g.read_alias()) == [0, 0, 2]
    compare_maps(g, o)
    # (2) chain of three
    o, g = pair()
    keys = np.array([pack_key(i, 0, 8) for i in range(4)] + [pack_key(i, 4, 8) for i in range(4)], np.uint64)
    owners = np.array([0, 0, 1, 1, 1, 1, 2, 2], np.uint32)
    ob, desc = objs([2, 4, 2]), np.stack([E[0], E[0], E[0]])
    assert o.import_(ob, desc, keys, owners) == 0
    g.import_(ob, desc, keys, owners)
    fr = frame(four(1, 48) + four(2, 112), [E[0], E[0]])
    integrate_frames(o, [fr])
    gpu_integrate(g, [fr], 0)
    compare_call(g, o)
    assert _compare_corr(g, o) == 2 and list(g.read_alias()) == [0, 0, 0]
    compare_maps(g, o)
    # (3) two frames of one call see the same new voxel with the same descriptor: one entity, not two
    o, g = pair()
    fa, fb = frame([(64, 48, 2.0, 1)], [E[0]]), frame([(64, 48, 2.0, 1), (96, 48, 2.0, 2)], [E[0], E[2]])
    integrate_frames(o, [fa, fb])
    gpu_integrate(g, [fa, fb], 0)
    compare_call(g, o)
    a, n, _, st = g.last_assoc()
    assert list(a) == [0, 0, 1] and list(n) == [1, 0, 1] and st["spawns"] == 2 and st["matches"] == 1
    integrate_frames(o, [fa, fb])
    gpu_integrate(g, [fa, fb], 0)
    compare_call(g, o)
    compare_maps(g, o)


@pytest.mark.parametrize("w", [(0.7, 0.3, 0.25), (0.5, 0.5, 0.5)])
def test_correspondence_split_map_scene(oracle, w):
    """A generated scene that forces bridges: the map of a plain configs[0] run with every object cut into two entities;
    later detections of an object overlap both halves and merge them.  Per call: decisions, merges, alias; at the end
    the whole map (voxel owners resolved through the merges, count-weighted descriptors, dead ids)."""
    from test_oracle_next import split_map_arrays
    cfg = _with_weights(S.get_config(0), w)
    sc = S.BoxScene(cfg)
    plain = oracle.OracleMap(cfg.voxel, cfg.D, 0.5, 0.5, 0.5, cfg.dtype, cfg.H, cfg.W)
    for k in range(9):
        fr = sc.frame(k)
        plain.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
    arrays = split_map_arrays(*plain.read())
    o, g = make_pair(oracle, cfg, correspondence=1, gaussian=1, covisibility=1, views=2)
    o.set_option(o.OPT_CORRESPONDENCE, 1)
    o.set_option(o.OPT_VIEWS_K, 2)
    assert o.import_(*arrays) == 0
    g.import_(*arrays)
    merges = 0
    for call in range(3, 6):
        frames = margin_filter(o.clone, [sc.frame(3 * call + i) for i in range(3)], cfg.tau, all_pairs=True)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o)
        merges += _compare_corr(g, o)
        assert np.array_equal(g.read_covisibility(), o.read_covisibility())     # C1 + U4: the losers' rows and columns absorbed
        _compare_views(g, o)                                                     # V + U4: the losers' views offered to the winner
    compare_maps(g, o)
    w_o, mu_o, cov_o = o.read_gaussians()
    w_g, mu_g, cov_g = g.read_gaussians()
    assert np.array_equal(w_g, w_o) and np.abs(mu_g - mu_o).max() <= TOL and np.abs(cov_g - cov_o).max() <= TOL
    assert merges >= 3, merges


def test_correspondence_dense_edges_on_the_tensor_path(oracle):
    """w_sem > tau (0, 1, 0.6), mini stress scene, tcgen05 similarity with the emitting epilogue: half of the detections
    that look at an existing object carry a descriptor half-way between that object's and a filler object's, so they
    retain BOTH (the filler without any voxel overlap: a dense edge) and bridge them."""
    from paper_2606_15476_b200.binding import OBJECT_DTYPE
    sc = S.StressScene(n_batches=1, frames_per_batch=4, n_objects=700)
    cfg = _with_weights(sc.cfg, (0.0, 1.0, 0.6))
    ijk, owner, n_vox, desc = sc.build_map()
    keys = pack_key(ijk[:, 0], ijk[:, 1], ijk[:, 2])
    objs = np.zeros(len(n_vox), OBJECT_DTYPE)
    objs["id"], objs["n_voxels"], objs["n_obs"], objs["best_frame"], objs["best_det"] = np.arange(len(n_vox)), n_vox, 1, -1, -1
    o, g = make_pair(oracle, cfg, max_det_per_call=1600, max_objects=len(n_vox) + 8000, sim_path=2, correspondence=1)
    o.set_option(o.OPT_CORRESPONDENCE, 1)
    assert o.import_(objs, desc, keys, owner) == 0
    g.import_(objs, desc, keys, owner)
    rng = np.random.default_rng(3)
    n_t = len(sc._blob_ijk)
    frames = []
    for fr in sc.batch(0):
        d = S.storage_to_f32(fr.desc, cfg.dtype).copy()
        for k in np.nonzero(fr.box_ids > 0)[0][::2]:
            v = d[k] + desc[int(rng.integers(n_t, len(desc)))]
            d[k] = v / np.linalg.norm(v)
        frames.append(S.Frame(fr.depth, fr.mask, fr.K, fr.T, S.to_storage(d.astype(np.float32), cfg.dtype), fr.n_det, fr.box_ids))
    frames = margin_filter(o.clone, frames, cfg.tau, all_pairs=True)
    integrate_frames(o, frames)
    gpu_integrate(g, frames, cfg.dtype)
    compare_call(g, o)
    assert _compare_corr(g, o) > 50
    compare_maps(g, o)


# ------------------------------------------------------------------------------------------------ Hellinger geometry (H1-H3)
@pytest.mark.parametrize("cfg_id,n,per_call,corr", [(0, 20, 1, 0), (0, 18, 3, 1), (1, 30, 1, 0)])
def test_hellinger_geometry_decisions(oracle, cfg_id, n, per_call, corr):
    """FARM_OPT_GEOMETRY = 1: the paper's own association: similarity prefilter from the similarity
    epilogue, g = 1 - Hellinger distance between Gaussians, same score / threshold / spawn rule; with and without the
    union-find correspondence."""
    cfg = S.get_config(cfg_id)
    frames_all = generate_frames(cfg_id, range(20, 20 + n) if cfg_id == 1 else range(n))
    o, g = make_pair(oracle, cfg, gaussian=1, geometry=1, prefilter_cos=0.3, correspondence=corr)
    o.set_option(o.OPT_GEOMETRY, 1)
    o.set_option(o.OPT_PREFILTER_COS, 0.3)
    o.set_option(o.OPT_CORRESPONDENCE, corr)
    matched = 0
    for c in range(0, n, per_call):
        frames = margin_filter(o.clone, frames_all[c:c + per_call], cfg.tau, all_pairs=bool(corr))
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o)
        matched += int(o.last_assoc()[4]["matches"])
        if corr:
            _compare_corr(g, o)
    compare_maps(g, o)
    assert matched > 10


def test_retrieval_skips_absorbed_entities(oracle):
    """Q1: only live entities are ranked.  On the split-map scene (correspondence on, several merges) the dead ids get
    rank / score 0 on both sides and the ranks of the live ones close up."""
    import torch
    from test_oracle_next import split_map_arrays
    cfg = _with_weights(S.get_config(0), (0.7, 0.3, 0.25))
    sc = S.BoxScene(cfg)
    plain = oracle.OracleMap(cfg.voxel, cfg.D, 0.5, 0.5, 0.5, cfg.dtype, cfg.H, cfg.W)
    for k in range(9):
        fr = sc.frame(k)
        plain.integrate(fr.depth, fr.mask, fr.K, fr.T, fr.desc, fr.n_det)
    arrays = split_map_arrays(*plain.read())
    o, g = make_pair(oracle, cfg, correspondence=1)
    o.set_option(o.OPT_CORRESPONDENCE, 1)
    assert o.import_(*arrays) == 0
    g.import_(*arrays)
    for call in range(3, 6):
        frames = margin_filter(o.clone, [sc.frame(3 * call + i) for i in range(3)], cfg.tau, all_pairs=True)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
    objs_o, _, _, _ = o.read(voxels=False)
    alive = (objs_o["n_obs"] > 0).astype(np.uint8)
    N = len(alive)
    assert 0 < alive.sum() < N                                     # some entities were absorbed
    cen = (0.5 * (objs_o["aabb_min"].astype(np.float64) + objs_o["aabb_max"].astype(np.float64))).astype(np.float32)
    cen[alive == 0] = 0
    rng = np.random.default_rng(2)
    dims, nnz = (32, 32, 32), (12, 12, 12)
    emb = [_ternary_rows(N, d, z, rng) for d, z in zip(dims, nnz)]
    emb_dev = [torch.from_numpy(e).to("cuda").contiguous() for e in emb]
    live_ids = np.nonzero(alive)[0]
    lm = int(live_ids[len(live_ids) // 2])
    qt = [_ternary_rows(1, 32, 12, rng)[0] for _ in range(4)]
    ql = [[emb[0][lm], emb[0][lm], emb[1][lm], emb[2][lm]]]
    ro = oracle.query(alive, emb, np.zeros(N, np.int32), cen, qt, -1, [oracle.PRED_NEXTTO], ql, 5)
    rg = g.query(emb_dev, 0, None, qt, -1, [oracle.PRED_NEXTTO], ql, 5)
    assert np.array_equal(rg["landmarks"], ro["landmarks"])
    assert np.abs(rg["s_sem"] - ro["s_sem"]).max() <= 1e-6 and np.abs(rg["s"] - ro["s"]).max() <= 1e-6
    assert (rg["s"][alive == 0] == 0).all() and (rg["top"] >= 0).all() and alive[rg["top"]].all()


# ------------------------------------------------------------------------------------------ W1-W4 weighted edges
@pytest.mark.parametrize("cfg_id,n,per_call,k,cut,decay", [(0, 20, 1, 2, 2.0, None), (0, 18, 3, 3, 1.05, 0.5), (1, 30, 1, 8, 1.5, None),
                                                           (1, 24, 4, 4, 2.0, 0.75)])
def test_weighted_covisibility_edges_match_oracle(oracle, cfg_id, n, per_call, k, cut, decay):
    """W1-W4: the kNN graph in Hellinger order with the median cutoff decides WHICH pairs are counted (fp32
    distance of an fp64 evaluation on both sides), the decayed weights are fp64: same edge list after every call, weights
    to 1e-9.  k = 2..8 covers both register-resident top-k widths of the kernel; batched calls put 10-40 entities in S."""
    cfg = S.get_config(cfg_id)
    frames_all = generate_frames(cfg_id, range(20, 20 + n) if cfg_id == 1 else range(n))
    o, g = make_pair(oracle, cfg, gaussian=1, edges=k, edge_cutoff=cut, edge_decay=decay)
    o.set_option(o.OPT_EDGES_K, k)
    o.set_option(o.OPT_EDGE_CUTOFF, cut)
    if decay is not None:
        o.set_option(o.OPT_EDGE_DECAY, decay)
    sizes = []
    for c in range(0, n, per_call):
        frames = margin_filter(o.clone, frames_all[c:c + per_call], cfg.tau)
        integrate_frames(o, frames)
        gpu_integrate(g, frames, cfg.dtype)
        compare_call(g, o, check_sets=False)
        ao, bo, wo = o.read_edges()
        ag, bg, wg = g.read_edges()
        assert np.array_equal(ag, ao) and np.array_equal(bg, bo), (c, len(ao), len(ag))
        assert np.abs(wg - wo).max(initial=0.0) <= 1e-9 * max(1.0, float(wo.max(initial=0.0)))
        sizes.append(len(ao))
    compare_maps(g, o, voxels=False)
    assert sizes[-1] > 10 and wo.max() > 1.5 and (wo < 0.999).any()     # repeated pairs accumulate, stale ones decay


def test_weighted_edges_option_checks(oracle):
    cfg = S.get_config(0)
    fr = generate_frames(0, range(1))[0]
    for kw in (dict(edges=2), dict(edges=2, gaussian=1, correspondence=1)):      # needs the Gaussians; not with entity merges
        g = FarmMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, H=cfg.H, W=cfg.W, dtype=cfg.dtype, **kw)
        with pytest.raises(Exception):
            gpu_integrate(g, [fr], cfg.dtype)
        g.destroy()
    g = FarmMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, H=cfg.H, W=cfg.W, dtype=cfg.dtype, gaussian=1)
    gpu_integrate(g, [fr], cfg.dtype)
    with pytest.raises(Exception):
        g.read_edges()                                                          # FARM_OPT_EDGES is off
    g.destroy()
