"""Seeded synthetic inputs for the FARM mapping hot path (BASELINE.json `configs`).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: no voxel keys, no overlap, no cosine, no association.  It only knows scene geometry
(axis-aligned boxes, a room shell, a pinhole camera) and how to ray-cast depth / instance masks and draw
descriptors.  It imports neither `oracle/` nor the CUDA binding.

Stand-in statement: the paper measures on ScanNet / HM3D / FARM-Scenes RGB-D streams with detector masks
and descriptors.  None of that data exists here; these generators reproduce
the shapes, sizes, value distributions and structure of those workloads as BASELINE.json prescribes.

Conventions
  world: z up.  camera: OpenCV axes (x right, y down, z forward), depth = camera-frame z (not ray length).
  T_world_cam: 4x4 row-major, camera -> world.  K: fx=K[0,0], fy=K[1,1], cx=K[0,2], cy=K[1,2].
  mask: uint16, 0 = background, k in 1..n_det = detection k-1 (descriptor row k-1).
  descriptors: storage dtype of the config; bf16 is carried as raw uint16 bit patterns.
Random numbers: numpy Philox (counter based) keyed by (seed, stream) so every frame generates
independently of the others.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

DTYPE_F32, DTYPE_F16, DTYPE_BF16 = 0, 1, 2
SEED_BASE = 15476000  # seed_i = SEED_BASE + i (fill-in)


def rng_for(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed), int(stream)]))


# --------------------------------------------------------------------------------------- dtype helpers
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bfloat16 bit pattern (uint16), round-to-nearest-even.  Storage format conversion only."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def to_storage(x: np.ndarray, dtype: int) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float32)
    if dtype == DTYPE_F32:
        return x
    if dtype == DTYPE_F16:
        return x.astype(np.float16)
    if dtype == DTYPE_BF16:
        return f32_to_bf16_bits(x)
    raise ValueError(dtype)


def storage_to_f32(x: np.ndarray, dtype: int) -> np.ndarray:
    if dtype == DTYPE_F32:
        return np.asarray(x, dtype=np.float32)
    if dtype == DTYPE_F16:
        return np.asarray(x, dtype=np.float16).astype(np.float32)
    return bf16_bits_to_f32(x)


def storage_itemsize(dtype: int) -> int:
    return 4 if dtype == DTYPE_F32 else 2


# --------------------------------------------------------------------------------------------- configs
@dataclass
class SceneConfig:
    index: int
    name: str
    extent: Tuple[float, float, float]        # Lx, Ly, Lz of one floor (metres)
    floors: int
    outdoor: bool
    n_boxes: int
    side: Tuple[float, float]
    H: int
    W: int
    fx: float
    cx: float
    cy: float
    n_frames: int
    n_det: int
    D: int
    dtype: int
    voxel: float
    traj: str                                  # 'circle' | 'walk'
    walk_step: float = 0.05
    walk_yaw_deg: float = 5.0
    miss_prob: float = 0.0
    fp_prob: float = 0.0
    z_max: float = 0.0                         # 0 = unlimited
    n_clusters: int = 0
    cluster_size: int = 0
    w_geo: float = 0.5
    w_sem: float = 0.5
    tau: float = 0.5
    frames_per_call: int = 1

    @property
    def seed(self) -> int:
        return SEED_BASE + self.index


def get_config(i: int) -> SceneConfig:
    """BASELINE.json configs[i] made concrete (fill-ins A14-A17)."""
    if i == 0:
        return SceneConfig(0, "tiny_room", (5.0, 5.0, 3.0), 1, False, 30, (0.2, 1.0), 120, 160, 120.0, 80.0, 60.0,
                           20, 4, 64, DTYPE_F32, 0.05, "circle")
    if i == 1:
        return SceneConfig(1, "room", (8.0, 6.0, 3.0), 1, False, 100, (0.2, 1.0), 480, 640, 525.0, 320.0, 240.0,
                           300, 20, 512, DTYPE_F16, 0.025, "walk", miss_prob=0.10, fp_prob=0.05)
    if i == 2:
        return SceneConfig(2, "house", (40.0, 20.0, 3.0), 2, False, 2000, (0.2, 1.0), 480, 640, 525.0, 320.0, 240.0,
                           1000, 40, 1024, DTYPE_BF16, 0.025, "walk", walk_step=0.15, n_clusters=40, cluster_size=6)
    if i == 3:
        return SceneConfig(3, "outdoor", (125.0, 120.0, 40.0), 1, True, 10000, (0.3, 6.0), 720, 1280, 1050.0, 640.0,
                           360.0, 2000, 60, 1024, DTYPE_BF16, 0.10, "walk", walk_step=0.6, z_max=30.0)
    if i == 4:
        # frames come from StressScene, not BoxScene; listed here for the map parameters
        return SceneConfig(4, "stress", (0.0, 0.0, 0.0), 1, False, 50000, (0.0, 0.0), 480, 640, 525.0, 320.0, 240.0,
                           16 * 36, 100, 1024, DTYPE_BF16, 0.025, "grid", frames_per_call=16)
    raise ValueError(i)


@dataclass
class Frame:
    depth: np.ndarray            # f32 [H,W]
    mask: np.ndarray             # u16 [H,W]
    K: np.ndarray                # f32 [3,3]
    T: np.ndarray                # f32 [4,4]
    desc: np.ndarray             # [n_det, D] storage dtype
    n_det: int
    box_ids: np.ndarray          # int64 [n_det] ground-truth box per detection (-1 = false positive)


def intrinsics(cfg: SceneConfig) -> np.ndarray:
    return np.array([[cfg.fx, 0.0, cfg.cx], [0.0, cfg.fx, cfg.cy], [0.0, 0.0, 1.0]], dtype=np.float32)


def pose_from_yaw(pos: np.ndarray, yaw: float) -> np.ndarray:
    """Camera at `pos`, looking along (cos yaw, sin yaw, 0), zero pitch/roll, z-up world."""
    c, s = np.cos(yaw), np.sin(yaw)
    right = np.array([s, -c, 0.0])
    down = np.array([0.0, 0.0, -1.0])
    fwd = np.array([c, s, 0.0])
    T = np.eye(4, dtype=np.float64)
    T[:3, 0], T[:3, 1], T[:3, 2], T[:3, 3] = right, down, fwd, pos
    return T.astype(np.float32)


def drop_detections(frame: Frame, drop: List[int]) -> Frame:
    """Remove detections (0-based rows) from a frame: label -> 0, remaining rows compacted, labels renumbered.
    Used by the tests' margin filter (score margins > 1e-3 are enforced by removal)."""
    if not drop:
        return frame
    keep = [d for d in range(frame.n_det) if d not in set(drop)]
    lut = np.zeros(frame.n_det + 1, dtype=np.uint16)
    for new, old in enumerate(keep):
        lut[old + 1] = new + 1
    m = frame.mask.copy()
    inside = m <= frame.n_det
    m[inside] = lut[m[inside]]
    return Frame(frame.depth, m, frame.K, frame.T, np.ascontiguousarray(frame.desc[keep]), len(keep),
                 frame.box_ids[keep])


# ------------------------------------------------------------------------------------------ box scenes
class BoxScene:
    """Configs 0-3: axis-aligned boxes inside a room shell (or on a ground plane), ray-cast per frame."""

    def __init__(self, cfg: SceneConfig, n_frames: Optional[int] = None):
        self.cfg = cfg
        self.n_frames = cfg.n_frames if n_frames is None else int(n_frames)
        self._build_trajectory()
        self._build_boxes()
        self._build_descriptors()

    # ---- trajectory (built first: boxes keep clear of it)
    def _build_trajectory(self):
        cfg = self.cfg
        Lx, Ly, Lz = cfg.extent
        n = cfg.n_frames  # always the full trajectory so that a prefix is a prefix
        pos = np.zeros((n, 3))
        yaw = np.zeros(n)
        if cfg.traj == "circle":
            c = np.array([Lx / 2, Ly / 2])
            for k in range(n):
                a = 2 * np.pi * k / n
                p = c + 2.0 * np.array([np.cos(a), np.sin(a)])
                pos[k] = [p[0], p[1], 1.5]
                yaw[k] = a + np.pi  # look at the centre
        else:
            g = rng_for(cfg.seed, 1)
            per_floor = n // cfg.floors
            m = 0.4
            for fl in range(cfg.floors):
                p = np.array([g.uniform(m, Lx - m), g.uniform(m, Ly - m)])
                y = g.uniform(0, 2 * np.pi)
                k0 = fl * per_floor
                k1 = n if fl == cfg.floors - 1 else k0 + per_floor
                for k in range(k0, k1):
                    pos[k] = [p[0], p[1], fl * Lz + 1.5]
                    yaw[k] = y
                    y = y + np.deg2rad(cfg.walk_yaw_deg) * g.standard_normal()
                    # walk mostly forward so that the trajectory covers ground (outdoor: ~1.2 km)
                    step = cfg.walk_step * (np.array([np.cos(y), np.sin(y)]) + 0.3 * g.standard_normal(2))
                    q = p + step
                    for ax, L in ((0, Lx), (1, Ly)):
                        if q[ax] < m:
                            q[ax] = 2 * m - q[ax]
                            y = g.uniform(0, 2 * np.pi)
                        if q[ax] > L - m:
                            q[ax] = 2 * (L - m) - q[ax]
                            y = g.uniform(0, 2 * np.pi)
                    p = q
        self.cam_pos, self.cam_yaw = pos, yaw

    # ---- boxes
    def _build_boxes(self):
        cfg = self.cfg
        g = rng_for(cfg.seed, 2)
        Lx, Ly, Lz = cfg.extent
        n = cfg.n_boxes
        lo = np.zeros((n, 3))
        hi = np.zeros((n, 3))
        floor_of = np.zeros(n, dtype=np.int64)
        cam = self.cam_pos
        clear = 0.35
        # coarse 2-D occupancy grid of the camera path for a fast keep-out test
        cell = 0.5
        gx, gy = int(np.ceil(Lx / cell)) + 1, int(np.ceil(Ly / cell)) + 1
        path = np.zeros((cfg.floors, gx, gy), dtype=bool)
        fl_of_cam = np.minimum((cam[:, 2] // Lz).astype(int), cfg.floors - 1)
        path[fl_of_cam, (cam[:, 0] / cell).astype(int), (cam[:, 1] / cell).astype(int)] = True
        placed = 0
        tries = 0
        # spatial hash of placed boxes for the non-intersection test (indoor scenes)
        bins: dict = {}
        bcell = max(cfg.side[1], 1.0)
        # cluster members are placed near their cluster centre (config 2)
        n_cl = cfg.n_clusters * cfg.cluster_size
        cl_centre = None
        while placed < n:
            tries += 1
            if tries > 400 * n:
                raise RuntimeError("box placement failed")
            fl = int(g.integers(cfg.floors))
            if cfg.outdoor:
                u = g.uniform()
                s = np.full(3, cfg.side[0] + (cfg.side[1] - cfg.side[0]) * u ** 6)  # cubes; most are small
            else:
                s = g.uniform(cfg.side[0], cfg.side[1], size=3)
            if placed < n_cl:
                j = placed % cfg.cluster_size
                if j == 0:
                    cl_centre = np.array([g.uniform(2, Lx - 2), g.uniform(2, Ly - 2)])
                    cl_floor = fl
                fl = cl_floor
                cxy = cl_centre + g.uniform(-1.5, 1.5, size=2)     # members within 3 m of each other
            else:
                cxy = np.array([g.uniform(s[0] / 2, Lx - s[0] / 2), g.uniform(s[1] / 2, Ly - s[1] / 2)])
            if cfg.outdoor:
                z0 = 0.0                                           # resting on the ground
            else:
                z0 = g.uniform(0.0, Lz - s[2]) if g.uniform() < 0.5 else 0.0
            b_lo = np.array([cxy[0] - s[0] / 2, cxy[1] - s[1] / 2, fl * Lz + z0])
            b_hi = b_lo + s
            if b_lo[0] < 0 or b_lo[1] < 0 or b_hi[0] > Lx or b_hi[1] > Ly:
                continue
            # keep clear of the camera path (only boxes that span camera height matter)
            if b_lo[2] - clear < fl * Lz + 1.5 < b_hi[2] + clear:
                i0, i1 = int(max(b_lo[0] - clear, 0) / cell), int(min(b_hi[0] + clear, Lx) / cell)
                j0, j1 = int(max(b_lo[1] - clear, 0) / cell), int(min(b_hi[1] + clear, Ly) / cell)
                if path[fl, i0:i1 + 1, j0:j1 + 1].any():
                    continue
            if not cfg.outdoor:  # non-intersecting by rejection
                ok = True
                kx0, kx1 = int(b_lo[0] // bcell), int(b_hi[0] // bcell)
                ky0, ky1 = int(b_lo[1] // bcell), int(b_hi[1] // bcell)
                for kx in range(kx0 - 1, kx1 + 2):
                    for ky in range(ky0 - 1, ky1 + 2):
                        for q in bins.get((fl, kx, ky), ()):
                            if np.all(b_lo < hi[q] + 0.02) and np.all(lo[q] < b_hi + 0.02):
                                ok = False
                                break
                        if not ok:
                            break
                    if not ok:
                        break
                if not ok:
                    continue
                for kx in range(kx0, kx1 + 1):
                    for ky in range(ky0, ky1 + 1):
                        bins.setdefault((fl, kx, ky), []).append(placed)
            lo[placed], hi[placed], floor_of[placed] = b_lo, b_hi, fl
            placed += 1
        self.box_lo, self.box_hi, self.box_floor = lo, hi, floor_of

    # ---- descriptors
    def _build_descriptors(self):
        cfg = self.cfg
        g = rng_for(cfg.seed, 3)
        base = g.standard_normal((cfg.n_boxes, cfg.D))
        base /= np.linalg.norm(base, axis=1, keepdims=True)
        # same-class distractor clusters: b_i = sqrt(.9) c + sqrt(.1) e_i, e_i orthonormal and orthogonal to c
        for c in range(cfg.n_clusters):
            m = cfg.cluster_size
            q, _ = np.linalg.qr(g.standard_normal((cfg.D, m + 1)))
            for j in range(m):
                base[c * m + j] = np.sqrt(0.9) * q[:, 0] + np.sqrt(0.1) * q[:, j + 1]
        self.base_desc = base

    def view_descriptor(self, g: np.random.Generator, base: np.ndarray) -> np.ndarray:
        """base + noise vector of expected length 0.1 (reading A15), renormalised."""
        D = base.shape[-1]
        v = base + (0.1 / np.sqrt(D)) * g.standard_normal(base.shape)
        return v / np.linalg.norm(v, axis=-1, keepdims=True)

    # ---- ray casting
    def _raycast(self, T: np.ndarray, fl: int):
        cfg = self.cfg
        H, W = cfg.H, cfg.W
        R = T[:3, :3].astype(np.float64)
        o = T[:3, 3].astype(np.float64)
        Lx, Ly, Lz = cfg.extent
        u = (np.arange(W) - cfg.cx) / cfg.fx
        v = (np.arange(H) - cfg.cy) / cfg.fx
        # direction in world per pixel: R @ (u, v, 1); parameter along it equals camera-frame z
        dirs = (R[:, 0][None, None, :] * u[None, :, None] + R[:, 1][None, None, :] * v[:, None, None]
                + R[:, 2][None, None, :])                                     # [H,W,3]
        with np.errstate(divide="ignore", invalid="ignore"):
            if cfg.outdoor:
                tz = (0.0 - o[2]) / dirs[..., 2]
                depth = np.where((dirs[..., 2] < 0) & (tz > 0), tz, np.inf)
            else:
                z_lo, z_hi = fl * Lz, (fl + 1) * Lz
                lo3 = np.array([0.0, 0.0, z_lo])
                hi3 = np.array([Lx, Ly, z_hi])
                t1 = (lo3 - o) / dirs
                t2 = (hi3 - o) / dirs
                depth = np.min(np.where(dirs > 0, t2, np.where(dirs < 0, t1, np.inf)), axis=-1)
        label = np.zeros((H, W), dtype=np.int64)
        # candidate boxes: same floor, in front of the camera, within range
        far = cfg.z_max if cfg.z_max > 0 else np.inf
        cand = np.nonzero(self.box_floor == fl)[0]
        centre = 0.5 * (self.box_lo[cand] + self.box_hi[cand])
        rad = 0.5 * np.linalg.norm(self.box_hi[cand] - self.box_lo[cand], axis=1)
        zc = (centre - o) @ R[:, 2]
        cand = cand[(zc + rad > 0.05) & (zc - rad < far)]
        corners_sel = np.array([[i, j, k] for i in (0, 1) for j in (0, 1) for k in (0, 1)], dtype=bool)
        for b in cand:
            lo, hi = self.box_lo[b], self.box_hi[b]
            cs = np.where(corners_sel, hi[None, :], lo[None, :])              # [8,3]
            pc = (cs - o) @ R                                                 # camera frame
            if np.all(pc[:, 2] <= 0.05):
                continue
            if np.any(pc[:, 2] <= 0.05):
                u0, u1, v0, v1 = 0, W - 1, 0, H - 1
            else:
                pu = cfg.fx * pc[:, 0] / pc[:, 2] + cfg.cx
                pv = cfg.fx * pc[:, 1] / pc[:, 2] + cfg.cy
                u0, u1 = int(np.floor(pu.min())) - 1, int(np.ceil(pu.max())) + 1
                v0, v1 = int(np.floor(pv.min())) - 1, int(np.ceil(pv.max())) + 1
                if u1 < 0 or v1 < 0 or u0 >= W or v0 >= H:
                    continue
                u0, v0, u1, v1 = max(u0, 0), max(v0, 0), min(u1, W - 1), min(v1, H - 1)
            d = dirs[v0:v1 + 1, u0:u1 + 1]
            with np.errstate(divide="ignore", invalid="ignore"):
                t1 = (lo - o) / d
                t2 = (hi - o) / d
            tn = np.nanmax(np.minimum(t1, t2), axis=-1)
            tf = np.nanmin(np.maximum(t1, t2), axis=-1)
            sub_depth = depth[v0:v1 + 1, u0:u1 + 1]
            hit = (tn <= tf) & (tn > 1e-6) & (tn < sub_depth)
            sub_depth[hit] = tn[hit]
            label[v0:v1 + 1, u0:u1 + 1][hit] = b + 1
        depth = np.where(np.isfinite(depth), depth, 0.0)
        return depth, label

    @staticmethod
    def _erode(label: np.ndarray) -> np.ndarray:
        """A pixel keeps its label only if all 8 neighbours carry the same label; border pixels -> 0 (A18)."""
        out = np.zeros_like(label)
        c = label[1:-1, 1:-1]
        same = np.ones_like(c, dtype=bool)
        H, W = label.shape
        for dv in (-1, 0, 1):
            for du in (-1, 0, 1):
                if dv == 0 and du == 0:
                    continue
                same &= label[1 + dv:H - 1 + dv, 1 + du:W - 1 + du] == c
        out[1:-1, 1:-1] = np.where(same, c, 0)
        return out

    def frame(self, k: int) -> Frame:
        cfg = self.cfg
        g = rng_for(cfg.seed, 1000 + k)
        fl = min(int(self.cam_pos[k, 2] // cfg.extent[2]), cfg.floors - 1)
        T = pose_from_yaw(self.cam_pos[k], self.cam_yaw[k])
        depth, label = self._raycast(T, fl)
        # sensor noise: sigma = 0.002 z^2
        depth = depth + 0.002 * depth * depth * g.standard_normal(depth.shape)
        if cfg.z_max > 0:
            depth = np.where(depth > cfg.z_max, 0.0, depth)
        depth = np.where(depth > 0, depth, 0.0).astype(np.float32)
        label = self._erode(label)
        label[depth <= 0] = 0
        ids, counts = np.unique(label[label > 0], return_counts=True)
        order = np.lexsort((ids, -counts))[: cfg.n_det]
        chosen = [(int(ids[i]) - 1, int(counts[i])) for i in order]
        # missed detections
        if cfg.miss_prob > 0:
            keep = g.uniform(size=len(chosen)) >= cfg.miss_prob
            chosen = [c for c, kf in zip(chosen, keep) if kf]
        work = np.zeros(label.shape, dtype=np.int64)           # provisional ids 1..len
        descs = []
        boxes = []
        for i, (b, _) in enumerate(chosen):
            work[label == b + 1] = i + 1
            descs.append(self.view_descriptor(g, self.base_desc[b]))
            boxes.append(b)
        # false positives: random filled ellipses painted over whatever is there
        if cfg.fp_prob > 0:
            n_fp = int(g.binomial(cfg.n_det, cfg.fp_prob))
            vv, uu = np.mgrid[0:cfg.H, 0:cfg.W]
            for _ in range(n_fp):
                cu, cv = g.uniform(0, cfg.W), g.uniform(0, cfg.H)
                a, b2 = g.uniform(10, 60), g.uniform(10, 60)
                inside = ((uu - cu) / a) ** 2 + ((vv - cv) / b2) ** 2 <= 1.0
                inside &= depth > 0
                if not inside.any():
                    continue
                work[inside] = len(descs) + 1
                r = g.standard_normal(cfg.D)
                descs.append(r / np.linalg.norm(r))
                boxes.append(-1)
        # final labels 1..n in descending pixel count (ties -> lower provisional id)
        ids, counts = np.unique(work[work > 0], return_counts=True)
        order = np.lexsort((ids, -counts))
        mask = np.zeros(label.shape, dtype=np.uint16)
        rows, bids = [], []
        for new, i in enumerate(order):
            mask[work == ids[i]] = new + 1
            rows.append(descs[int(ids[i]) - 1])
            bids.append(boxes[int(ids[i]) - 1])
        n_det = len(rows)
        desc = to_storage(np.array(rows, dtype=np.float32).reshape(n_det, cfg.D), cfg.dtype)
        return Frame(depth, mask, intrinsics(cfg), T, desc, n_det, np.array(bids, dtype=np.int64))

    def frames(self, k0: int = 0, k1: Optional[int] = None) -> List[Frame]:
        k1 = self.n_frames if k1 is None else k1
        return [self.frame(k) for k in range(k0, k1)]


# ---- parallel frame generation: the ray caster is single-threaded numpy and frames are independent by construction
# (every frame draws from its own Philox stream).  spawn context: the parent may hold a CUDA context.
_GEN_SCENE: dict = {}


def _gen_one(args):
    ci, k = args
    if ci not in _GEN_SCENE:
        _GEN_SCENE[ci] = BoxScene(get_config(ci))
    return k, _GEN_SCENE[ci].frame(k)


def generate_frames(cfg_index: int, ks, procs: Optional[int] = None) -> List[Frame]:
    """[BoxScene(get_config(cfg_index)).frame(k) for k in ks], generated by a pool of worker processes."""
    import multiprocessing as mp
    import os
    ks = list(ks)
    procs = min(procs or max(1, (os.cpu_count() or 2) - 2), 14, max(len(ks), 1))
    if procs <= 1 or len(ks) < 4:
        return [_gen_one((cfg_index, k))[1] for k in ks]
    with mp.get_context("spawn").Pool(procs) as pool:
        out = dict(pool.imap_unordered(_gen_one, [(cfg_index, k) for k in ks], chunksize=max(1, len(ks) // (procs * 4))))
    return [out[k] for k in ks]


# --------------------------------------------------------------------------------------- config 4: stress
class StressScene:
    """Config 4 (batched throughput stress): a pre-populated map of `n_objects` voxel blobs plus batches of
    `frames_per_batch` frames with 100 detections each on a 10x10 grid of 64x48 tiles; 50 % of the detections
    look at an existing object.

    Geometry only: the blob of a looked-at object is the set of voxels its depth patch passes through
    (every pixel ray at its depth), extruded along the same pixel rays to the requested size.  The voxel
    index of a scene point is floor(point / voxel) in float64 -- the scene's own bookkeeping of where its
    surfaces are, independent of the method's fp32 arithmetic (the two agree except for points within an
    ulp of a voxel face, which merely become new voxels of the matched object).
    All cameras look along world +x; frames are placed on a y-z lattice wide enough that their frusta and
    blobs never meet.  Filler objects are random stacks of overlapping rectangles (6-connected) far away.
    """

    GRID = 10
    TILE_W, TILE_H = 64, 48

    def __init__(self, n_batches: int, frames_per_batch: int = 16, n_objects: int = 50000,
                 mean_blob: int = 2000, seed: Optional[int] = None, cfg: Optional[SceneConfig] = None):
        self.cfg = cfg or get_config(4)
        self.n_batches, self.F = n_batches, frames_per_batch
        self.seed = self.cfg.seed if seed is None else seed
        self.n_objects, self.mean_blob = n_objects, mean_blob
        self.n_frames = n_batches * frames_per_batch
        self._frames: List[Frame] = []
        self._blob_ijk: List[np.ndarray] = []      # per target object: int32 [n,3]
        self._blob_desc: List[np.ndarray] = []
        side = int(np.ceil(np.sqrt(self.n_frames)))
        self._lattice = side
        for g in range(self.n_frames):
            self._make_frame(g)

    # ---- frames
    MASK_W, MASK_H = 48, 36      # labelled region, centred in each 64x48 tile (56 % of the image is masked)

    def _make_frame(self, g: int):
        cfg = self.cfg
        rng = rng_for(self.seed, 100 + g)
        H, W, fx, cx, cy, vs = cfg.H, cfg.W, cfg.fx, cfg.cx, cfg.cy, cfg.voxel
        pos = np.array([0.0, 10.0 * (g % self._lattice), 8.0 * (g // self._lattice) + 2.0])
        T = pose_from_yaw(pos, 0.0)                       # right=(0,-1,0) down=(0,0,-1) fwd=(1,0,0)
        depth = np.full((H, W), 4.5, dtype=np.float64)    # far wall behind everything, unlabelled
        mask = np.zeros((H, W), dtype=np.uint16)
        n_det = self.GRID * self.GRID
        z0_frame = rng.uniform(0.9, 3.2)
        uu, vv = np.meshgrid(np.arange(self.TILE_W), np.arange(self.TILE_H))
        base = rng.standard_normal((n_det, cfg.D))
        base /= np.linalg.norm(base, axis=1, keepdims=True)
        is_target = np.zeros(n_det, dtype=bool)
        is_target[rng.permutation(n_det)[: n_det // 2]] = True
        mu0, mv0 = (self.TILE_W - self.MASK_W) // 2, (self.TILE_H - self.MASK_H) // 2
        for d in range(n_det):
            ty, tx = divmod(d, self.GRID)
            u0, v0 = tx * self.TILE_W, ty * self.TILE_H
            z0 = z0_frame * rng.uniform(0.9, 1.1)
            a, b = rng.uniform(-0.0015, 0.0015, size=2) * z0
            c, ph = rng.uniform(0.0, 0.02) * z0, rng.uniform(0, 2 * np.pi)
            z = z0 + a * (uu - 32) + b * (vv - 24) + c * np.sin(uu / 9.0 + ph) * np.cos(vv / 7.0)
            z = z + 0.002 * z * z * rng.standard_normal(z.shape)          # sensor noise sigma = 0.002 z^2
            depth[v0:v0 + self.TILE_H, u0:u0 + self.TILE_W] = np.clip(z, 0.5, 4.0)
            mask[v0 + mv0:v0 + mv0 + self.MASK_H, u0 + mu0:u0 + mu0 + self.MASK_W] = d + 1
        depth32 = depth.astype(np.float32)

        def pack(P):  # scene bookkeeping: voxel cell of a float64 point, three 21-bit fields in one int64
            q = np.floor(P / vs).astype(np.int64) + (1 << 20)
            return (q[..., 0] << 42) | (q[..., 1] << 21) | q[..., 2]

        # blobs of the looked-at objects, from the depth actually stored in the frame
        keys_l, owner_l = [], []
        targets = np.nonzero(is_target)[0]
        for slot, d in enumerate(targets):
            ty, tx = divmod(int(d), self.GRID)
            u = np.arange(tx * self.TILE_W + mu0, tx * self.TILE_W + mu0 + self.MASK_W)
            v = np.arange(ty * self.TILE_H + mv0, ty * self.TILE_H + mv0 + self.MASK_H)
            U, V = np.meshgrid(u, v)
            zz = depth32[V, U].astype(np.float64)
            xn, yn = (U - cx) / fx, (V - cy) / fx
            surf = np.unique(pack(np.stack([pos[0] + zz, pos[1] - xn * zz, pos[2] - yn * zz], -1)).ravel())
            target_size = rng.uniform(0.5, 1.5) * self.mean_blob
            # extrude along the pixel rays; layer k lies 0.8*k voxels behind the surface and is wider by (z_k/z)^2
            zm = float(zz.mean())
            k = np.arange(1, int(2.0 / (0.8 * vs)) + 1)
            grow = np.cumsum(0.8 * len(surf) * ((zm + k * 0.8 * vs) / zm) ** 2 / 3.0)
            L = int(np.searchsorted(grow, max(target_size - len(surf), 0.0))) + 1
            stride = int(max(1, np.floor(0.5 * vs * fx / zz.max())))
            zs = zz[::stride, ::stride][None] + (k[:L, None, None] * (0.8 * vs))
            xs, ys = xn[::stride, ::stride][None], yn[::stride, ::stride][None]
            deep = np.unique(pack(np.stack([pos[0] + zs, pos[1] - xs * zs, pos[2] - ys * zs], -1)).ravel())
            kk = np.union1d(surf, deep)
            keys_l.append(kk)
            owner_l.append(np.full(len(kk), slot, dtype=np.int64))
        # exclusive ownership inside the frame: the lowest slot keeps a voxel two blobs share
        if keys_l:
            allk, allo = np.concatenate(keys_l), np.concatenate(owner_l)
            order = np.lexsort((allo, allk))
            allk, allo = allk[order], allo[order]
            first = np.ones(len(allk), dtype=bool)
            first[1:] = allk[1:] != allk[:-1]
            allk, allo = allk[first], allo[first]
            m21 = (1 << 21) - 1
            ijk = np.stack([(allk >> 42) & m21, (allk >> 21) & m21, allk & m21], 1) - (1 << 20)
            for slot, d in enumerate(targets):
                self._blob_ijk.append(ijk[allo == slot].astype(np.int32))
                self._blob_desc.append(base[d])
        descs = self._view_desc(rng, base)
        frame = Frame(depth32, mask, intrinsics(cfg), T, to_storage(descs.astype(np.float32), cfg.dtype), n_det,
                      np.where(is_target, 1, -1).astype(np.int64))
        self._frames.append(frame)

    @staticmethod
    def _view_desc(rng, base):
        D = base.shape[-1]
        v = base + (0.1 / np.sqrt(D)) * rng.standard_normal(base.shape)
        return v / np.linalg.norm(v, axis=-1, keepdims=True)

    def batch(self, b: int) -> List[Frame]:
        return self._frames[b * self.F:(b + 1) * self.F]

    # ---- the pre-populated map
    def build_map(self):
        """Returns (ijk int32 [nv,3], owner uint32 [nv], n_voxels uint32 [N], desc float32 [N,D], aabb [N,6])."""
        cfg = self.cfg
        rng = rng_for(self.seed, 7)
        n_t = len(self._blob_ijk)
        n_fill = max(self.n_objects - n_t, 0)
        N = n_t + n_fill
        # filler objects: L layers, each an axis-aligned rectangle overlapping the previous one
        L = 12
        side = max(int(round(np.sqrt(self.mean_blob / L))), 2)
        w = rng.integers(max(side - 3, 1), side + 4, size=(n_fill, L))
        h = rng.integers(max(side - 3, 1), side + 4, size=(n_fill, L))
        x0 = 20 + np.cumsum(rng.integers(-2, 3, size=(n_fill, L)), axis=1)
        y0 = 20 + np.cumsum(rng.integers(-2, 3, size=(n_fill, L)), axis=1)
        cells = int(np.ceil(np.sqrt(max(n_fill, 1))))
        cell_i = np.arange(n_fill) % cells
        cell_j = np.arange(n_fill) // cells
        area = (w * h).reshape(-1)
        tot = int(area.sum())
        rect = np.repeat(np.arange(n_fill * L), area)                       # rectangle id per voxel
        within = np.arange(tot) - np.repeat(np.cumsum(area) - area, area)   # index inside the rectangle
        wf = w.reshape(-1)[rect]
        dx, dy = within % wf, within // wf
        obj = rect // L
        lay = rect % L
        fill_ijk = np.stack([-4000 + x0.reshape(-1)[rect] + dx - 64 * cell_i[obj],
                             y0.reshape(-1)[rect] + dy + 64 * cell_j[obj],
                             lay + 40], axis=1).astype(np.int32)
        fill_owner = (n_t + obj).astype(np.uint32)
        t_owner = np.concatenate([np.full(len(b), i, dtype=np.uint32) for i, b in enumerate(self._blob_ijk)]) \
            if n_t else np.zeros(0, np.uint32)
        ijk = np.concatenate(self._blob_ijk + [fill_ijk]) if n_t else fill_ijk
        owner = np.concatenate([t_owner, fill_owner])
        n_vox = np.bincount(owner, minlength=N).astype(np.uint32)
        fd = rng.standard_normal((n_fill, cfg.D)).astype(np.float32)
        fd /= np.linalg.norm(fd, axis=1, keepdims=True)
        desc = np.concatenate([np.array(self._blob_desc, dtype=np.float32).reshape(n_t, cfg.D), fd])
        return ijk, owner, n_vox, desc
