"""Thin ctypes binding of libfarm_map.so (include/farm.h).  Argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; this module owns no arithmetic and has
no CPU fallback: if the library is missing, or no CUDA device is present, calls fail loudly.
PyTorch appears only as the owner of device memory and streams (tensors in, `.data_ptr()` out).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libfarm_map.so")

FARM_OK, ERR_INVALID_ARG, ERR_CUDA, ERR_CAPACITY, ERR_STATE, ERR_RANGE = 0, -1, -2, -3, -4, -5
DTYPE_F32, DTYPE_F16, DTYPE_BF16 = 0, 1, 2
OPT_DESC_DTYPE, OPT_MAX_OBJECTS, OPT_MAX_VOXELS, OPT_IMG_W, OPT_IMG_H = 1, 2, 3, 4, 5
OPT_MAX_DET_PER_CALL, OPT_STREAM, OPT_MAX_PAIRS_PER_CALL, OPT_MAX_FRAMES_PER_CALL, OPT_SIM_PATH = 6, 7, 8, 9, 10
OPT_TIMING = 11
OPT_OVERLAP = 12
OPT_MAX_BLOCKS = 13
OPT_GAUSSIAN = 14
OPT_COVISIBILITY = 15
OPT_VIEWS = 16
OPT_CORRESPONDENCE = 17
OPT_GEOMETRY = 18
OPT_EDGES = 19
OPT_INPUTS_READY = 20
OPTF_EDGE_DECAY, OPTF_EDGE_CUTOFF = 107, 108
N_STAGES = 6
STAGE_NAMES = ["prep", "lift", "similarity", "probe", "associate", "merge"]
OPTF_Z_MIN, OPTF_Z_MAX, OPTF_VIEW_COS, OPTF_VIEW_CLOSER, OPTF_PREFILTER_COS, OPTF_HELLINGER_BUDGET = 101, 102, 103, 104, 105, 106
VIEW_DTYPE = np.dtype([("frame", "<i4"), ("det", "<i4"), ("n_px", "<u4"), ("cam", "<f4", 3), ("dir", "<f4", 3), ("dist", "<f4")])
KEY_EMPTY = 0xFFFFFFFFFFFFFFFF

OBJECT_DTYPE = np.dtype(
    [("id", "<i4"), ("n_voxels", "<u4"), ("n_obs", "<u4"), ("aabb_min", "<f4", 3), ("aabb_max", "<f4", 3),
     ("best_frame", "<i4"), ("best_det", "<i4"), ("best_pixels", "<u4"), ("best_cam_pos", "<f4", 3),
     ("n_points", "<u8")], align=True)
STATS_DTYPE = np.dtype(
    [("valid_points", "<u8"), ("dropped_points", "<u8"), ("ignored_pixels", "<u8"), ("unique_voxels", "<u8"),
     ("matches", "<u4"), ("spawns", "<u4"), ("skipped", "<u4"), ("n_det", "<u4")], align=True)
TOTALS_DTYPE = np.dtype([("frames", "<u8"), ("calls", "<u8"), ("valid_points", "<u8"), ("unique_voxels", "<u8"),
                         ("matches", "<u8"), ("spawns", "<u8")])

EXPORTS = ["farm_map_create", "farm_map_destroy", "farm_map_set_option_i", "farm_map_set_option_f",
           "farm_map_integrate", "farm_map_integrate_batch", "farm_map_integrate_batch_host", "farm_map_stage_times", "farm_map_last_assoc", "farm_map_last_assoc_async", "farm_map_last_gaussians", "farm_map_read_gaussians", "farm_map_read_covisibility",
           "farm_map_read",
           "farm_map_import", "farm_map_sync", "farm_map_kernel_launches", "farm_last_error",
           "farm_map_get_frame_seq", "farm_map_set_frame_seq", "farm_map_read_views", "farm_map_query", "farm_map_read_alias",
           "farm_map_last_merges", "farm_map_read_edges", "farm_cosine_rowmax_noalloc",
           "farm_debug_backproject", "farm_debug_last_voxels", "farm_debug_last_overlaps", "farm_debug_last_dense"]


class FarmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"farm error {code}: {msg}")
        self.code = code


_lib = None


def load_library():
    """dlopen libfarm_map.so.  Raises if it has not been built (python -m paper_2606_15476_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} missing: build it with `python -m paper_2606_15476_b200.build` "
                                    "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        vp, ci, cf, ll = C.c_void_p, C.c_int, C.c_float, C.c_longlong
        lib.farm_map_create.argtypes = [cf, ci, cf, cf, cf, C.POINTER(vp)]
        lib.farm_map_destroy.argtypes = [vp]
        lib.farm_map_set_option_i.argtypes = [vp, ci, ll]
        lib.farm_map_set_option_f.argtypes = [vp, ci, cf]
        lib.farm_map_integrate.argtypes = [vp, vp, vp, vp, vp, vp, ci]
        lib.farm_map_integrate_batch.argtypes = [vp, ci, vp, vp, vp, vp, vp, vp]
        lib.farm_map_integrate_batch_host.argtypes = [vp, ci, vp, vp, vp, vp, vp, vp]
        lib.farm_map_stage_times.argtypes = [vp, vp, vp, ci]
        lib.farm_map_last_assoc.argtypes = [vp, vp, vp, vp, vp]
        lib.farm_map_last_assoc_async.argtypes = [vp, vp, vp, vp, vp]
        lib.farm_map_last_gaussians.argtypes = [vp, vp, vp, vp]
        lib.farm_map_read_gaussians.argtypes = [vp, vp, vp, vp]
        lib.farm_map_read_covisibility.argtypes = [vp, vp, vp]
        lib.farm_map_read_views.argtypes = [vp, vp, vp]
        lib.farm_map_read_alias.argtypes = [vp, vp]
        lib.farm_map_read_edges.argtypes = [vp, vp, vp, vp, C.c_uint64, vp]
        lib.farm_cosine_rowmax_noalloc.argtypes = [vp, ci, vp, ci, ci, ci, vp, vp, vp]
        lib.farm_map_last_merges.argtypes = [vp, vp, vp, vp]
        lib.farm_map_query.argtypes = [vp, vp, vp, vp, ci, ci, ci, ci, vp, vp, ci, ci, vp, vp, ci, vp, vp, vp, vp, vp, vp]
        lib.farm_map_read.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        lib.farm_map_import.argtypes = [vp, vp, ci, vp, vp, vp, ll]
        lib.farm_map_sync.argtypes = [vp, vp]
        lib.farm_map_kernel_launches.argtypes = [vp]
        lib.farm_map_kernel_launches.restype = ll
        lib.farm_map_get_frame_seq.argtypes = [vp, C.POINTER(ll)]
        lib.farm_map_set_frame_seq.argtypes = [vp, ll]
        lib.farm_last_error.restype = C.c_char_p
        lib.farm_debug_backproject.argtypes = [vp, vp, vp, vp, vp, ci, vp, vp]
        lib.farm_debug_last_voxels.argtypes = [vp, vp, vp, vp, vp]
        lib.farm_debug_last_overlaps.argtypes = [vp, vp, vp, vp]
        lib.farm_debug_last_dense.argtypes = [vp, vp, vp]
        _lib = lib
    return _lib


def _check(rc):
    if rc != FARM_OK:
        raise FarmError(rc, load_library().farm_last_error().decode())


def _hp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _dp(t):
    """device pointer of a CUDA torch tensor (or a raw int)"""
    if t is None:
        return None
    if isinstance(t, int):
        return C.c_void_p(t)
    assert t.is_cuda and t.is_contiguous(), "device tensors must be contiguous CUDA tensors"
    return C.c_void_p(t.data_ptr())


NOALLOC_MAX_M, NOALLOC_MAX_N = 4096, 65536


def cosine_rowmax_noalloc(A, M, B, N, D, dtype, max_cos, argmax, stream=None):
    """farm_cosine_rowmax_noalloc: dense cosine of A [M, D] against B [N, D] (DEVICE, `dtype`) with fused row max / argmax into
    max_cos f32 [M] / argmax i32 [M] (DEVICE); allocates nothing (fixed scratch array in the library, M <= 4096, N <= 65536);
    enqueued on `stream` (a cudaStream_t as int, default stream if None), not synchronised."""
    _check(load_library().farm_cosine_rowmax_noalloc(_dp(A), int(M), _dp(B), int(N), int(D), int(dtype), _dp(max_cos), _dp(argmax),
                                                     C.c_void_p(stream) if stream else None))


class FarmMap:
    """farm_map_* with the same names and argument order as the C ABI."""

    def __init__(self, voxel_size, D, w_geo, w_sem, tau, *, H, W, dtype=DTYPE_F32, max_objects=None,
                 max_voxels=None, max_blocks=None, max_det_per_call=None, max_pairs_per_call=None, max_frames_per_call=None,
                 stream=None, z_min=None, z_max=None, sim_path=None, timing=None, overlap=None, gaussian=None, covisibility=None,
                 views=None, view_cos=None, view_closer=None, correspondence=None, geometry=None, prefilter_cos=None,
                 hellinger_budget=None, edges=None, edge_decay=None, edge_cutoff=None, inputs_ready=None):
        lib = load_library()
        self.D, self.dtype, self.H, self.W = D, dtype, H, W
        self._last_M = 0
        self._h = C.c_void_p()
        _check(lib.farm_map_create(voxel_size, D, w_geo, w_sem, tau, C.byref(self._h)))
        self.set_option_i(OPT_IMG_H, H)
        self.set_option_i(OPT_IMG_W, W)
        self.set_option_i(OPT_DESC_DTYPE, dtype)
        for key, v in ((OPT_MAX_OBJECTS, max_objects), (OPT_MAX_VOXELS, max_voxels), (OPT_MAX_BLOCKS, max_blocks),
                       (OPT_MAX_DET_PER_CALL, max_det_per_call), (OPT_MAX_PAIRS_PER_CALL, max_pairs_per_call),
                       (OPT_MAX_FRAMES_PER_CALL, max_frames_per_call), (OPT_STREAM, stream), (OPT_SIM_PATH, sim_path),
                       (OPT_TIMING, timing), (OPT_OVERLAP, overlap), (OPT_GAUSSIAN, gaussian), (OPT_COVISIBILITY, covisibility),
                       (OPT_VIEWS, views), (OPT_CORRESPONDENCE, correspondence), (OPT_GEOMETRY, geometry),
                       (OPT_EDGES, edges), (OPT_INPUTS_READY, inputs_ready)):
            if v is not None:
                self.set_option_i(key, int(v))
        if z_min is not None:
            self.set_option_f(OPTF_Z_MIN, z_min)
        if z_max is not None:
            self.set_option_f(OPTF_Z_MAX, z_max)
        if view_cos is not None:
            self.set_option_f(OPTF_VIEW_COS, view_cos)
        if view_closer is not None:
            self.set_option_f(OPTF_VIEW_CLOSER, view_closer)
        if prefilter_cos is not None:
            self.set_option_f(OPTF_PREFILTER_COS, prefilter_cos)
        if hellinger_budget is not None:
            self.set_option_f(OPTF_HELLINGER_BUDGET, hellinger_budget)
        if edge_decay is not None:
            self.set_option_f(OPTF_EDGE_DECAY, edge_decay)
        if edge_cutoff is not None:
            self.set_option_f(OPTF_EDGE_CUTOFF, edge_cutoff)
        self.views_k = int(views or 0)

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load_library().farm_map_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = destroy

    def set_option_i(self, key, value):
        _check(load_library().farm_map_set_option_i(self._h, key, int(value)))

    def set_option_f(self, key, value):
        _check(load_library().farm_map_set_option_f(self._h, key, float(value)))

    # ---- the hot path (device tensors)
    def integrate(self, depth, instance_mask, K, T_world_cam, det_descriptors, n_det):
        _check(load_library().farm_map_integrate(self._h, _dp(depth), _dp(instance_mask), _dp(K), _dp(T_world_cam),
                                                 _dp(det_descriptors), int(n_det)))
        self._last_M = int(n_det)

    def integrate_batch(self, n_frames, depth, instance_mask, K, T_world_cam, det_descriptors, n_det):
        n_det = np.ascontiguousarray(n_det, np.int32)
        assert n_det.size == n_frames
        _check(load_library().farm_map_integrate_batch(self._h, int(n_frames), _dp(depth), _dp(instance_mask), _dp(K),
                                                       _dp(T_world_cam), _dp(det_descriptors), _hp(n_det)))
        self._last_M = int(n_det.sum())

    def integrate_batch_host(self, n_frames, depth, instance_mask, K, T_world_cam, det_descriptors, n_det):
        """Host (numpy or pinned torch CPU) buffers; the library stages them itself."""
        n_det = np.ascontiguousarray(n_det, np.int32)

        def hp(x):
            if x is None:
                return None
            return C.c_void_p(x.data_ptr()) if hasattr(x, "data_ptr") else _hp(x)
        _check(load_library().farm_map_integrate_batch_host(self._h, int(n_frames), hp(depth), hp(instance_mask), hp(K),
                                                            hp(T_world_cam), hp(det_descriptors), _hp(n_det)))
        self._last_M = int(n_det.sum())

    def stage_times(self, reset=False):
        ms = np.zeros(N_STAGES, np.float32)
        ln = np.zeros(N_STAGES, np.int64)
        _check(load_library().farm_map_stage_times(self._h, _hp(ms), _hp(ln), int(bool(reset))))
        return ms, ln

    # ---- results (host arrays)
    def last_assoc(self, M=None):
        M = self._last_M if M is None else M
        obj = np.empty(M, np.int32)
        is_new = np.empty(M, np.uint8)
        best = np.empty(M, np.float32)
        st = np.zeros(1, STATS_DTYPE)
        _check(load_library().farm_map_last_assoc(self._h, _hp(obj), _hp(is_new), _hp(best), _hp(st)))
        return obj, is_new, best, st[0]

    def last_assoc_async(self, obj_id, is_new, best_score, stats):
        """Enqueue the D2H copies of the last call's results into pinned torch CPU tensors / numpy arrays (any may be
        None); valid after the next sync()."""
        def hp(x):
            if x is None:
                return None
            return C.c_void_p(x.data_ptr()) if hasattr(x, "data_ptr") else _hp(x)
        _check(load_library().farm_map_last_assoc_async(self._h, hp(obj_id), hp(is_new), hp(best_score), hp(stats)))

    def read(self, voxels=True, descriptors=True):
        lib = load_library()
        n = C.c_int(0)
        nv = C.c_longlong(0)
        _check(lib.farm_map_read(self._h, None, C.byref(n), None, None, None, C.byref(nv) if voxels else None))
        objs = np.zeros(n.value, OBJECT_DTYPE)
        desc = np.empty((n.value, self.D), np.float32) if descriptors else None
        keys = np.empty(nv.value, np.uint64) if voxels else None
        owners = np.empty(nv.value, np.uint32) if voxels else None
        _check(lib.farm_map_read(self._h, _hp(objs), C.byref(n), _hp(desc), _hp(keys), _hp(owners),
                                 C.byref(nv) if voxels else None))
        return objs, desc, keys, owners

    def last_gaussians(self):
        """(mu [M,3], cov [M,6], hellinger [M]) of the last call's detections (FARM_OPT_GAUSSIAN)."""
        M = self._last_M
        mu, cov, hell = np.zeros((M, 3), np.float32), np.zeros((M, 6), np.float32), np.zeros(M, np.float32)
        _check(load_library().farm_map_last_gaussians(self._h, _hp(mu), _hp(cov), _hp(hell)))
        return mu, cov, hell

    def read_gaussians(self):
        """(weight [N] f64, mu [N,3], cov [N,6]) of the map's objects (FARM_OPT_GAUSSIAN)."""
        n = C.c_int(0)
        _check(load_library().farm_map_read(self._h, None, C.byref(n), None, None, None, None))
        N = n.value
        w, mu, cov = np.zeros(N, np.float64), np.zeros((N, 3), np.float32), np.zeros((N, 6), np.float32)
        _check(load_library().farm_map_read_gaussians(self._h, _hp(w), _hp(mu), _hp(cov)))
        return w, mu, cov

    def query(self, emb, emb_dtype, cls, q_target, target_class, pred_types, q_landmarks, topk):
        """farm_map_query.  emb: three CUDA tensors [N, d_s]; cls: CUDA int32 tensor [N] or None; q_target: four host
        vectors (d0, d0, d1, d2); q_landmarks: one such list of four per predicate.  Returns dict(top, top_scores,
        landmarks, s_sem, gbar, s)."""
        n = C.c_int(0)
        _check(load_library().farm_map_read(self._h, None, C.byref(n), None, None, None, None))
        N, P = n.value, len(pred_types)
        dims = [int(e.shape[1]) for e in emb]
        qt = np.ascontiguousarray(np.concatenate([np.asarray(x, np.float32).ravel() for x in q_target]), np.float32)
        ql = np.ascontiguousarray(np.concatenate([np.asarray(x, np.float32).ravel() for lm in q_landmarks for x in lm])
                                  if P else np.zeros(1), np.float32)
        pt = np.ascontiguousarray(pred_types if P else [0], np.int32)
        top, tsc = np.full(topk, -1, np.int32), np.zeros(topk, np.float32)
        lms = np.full(max(P, 1), -1, np.int32)
        s_sem, gbar, s = np.zeros(N, np.float32), np.zeros(N, np.float32), np.zeros(N, np.float32)
        _check(load_library().farm_map_query(self._h, _dp(emb[0]), _dp(emb[1]), _dp(emb[2]), dims[0], dims[1], dims[2],
                                             int(emb_dtype), _dp(cls), _hp(qt), int(target_class), P, _hp(pt), _hp(ql), int(topk),
                                             _hp(top), _hp(tsc), _hp(lms), _hp(s_sem), _hp(gbar), _hp(s)))
        return {"top": top, "top_scores": tsc, "landmarks": lms[:P], "s_sem": s_sem, "gbar": gbar, "s": s}

    def read_alias(self):
        """alias [N]: the live entity every id stands for (FARM_OPT_CORRESPONDENCE)."""
        n = C.c_int(0)
        _check(load_library().farm_map_read(self._h, None, C.byref(n), None, None, None, None))
        al = np.zeros(n.value, np.int32)
        _check(load_library().farm_map_read_alias(self._h, _hp(al)))
        return al

    def last_merges(self):
        """(loser [n], winner [n]) entity merges of the last call, sorted by loser (FARM_OPT_CORRESPONDENCE)."""
        n = C.c_int(0)
        _check(load_library().farm_map_last_merges(self._h, None, None, C.byref(n)))
        a, b = np.zeros(n.value, np.int32), np.zeros(n.value, np.int32)
        if n.value:
            _check(load_library().farm_map_last_merges(self._h, _hp(a), _hp(b), C.byref(n)))
        order = np.argsort(a)
        return a[order], b[order]

    def read_views(self):
        """(views [N, k] VIEW_DTYPE, counts [N]) retained views per object (FARM_OPT_VIEWS = k)."""
        n = C.c_int(0)
        _check(load_library().farm_map_read(self._h, None, C.byref(n), None, None, None, None))
        views = np.zeros((n.value, max(self.views_k, 1)), VIEW_DTYPE)
        counts = np.zeros(n.value, np.int32)
        _check(load_library().farm_map_read_views(self._h, _hp(views), _hp(counts)))
        return views[:, :self.views_k], counts

    def read_edges(self):
        """(a [n] uint32, b [n] uint32, w [n] float64): weighted covisibility edges a < b sorted by (a, b), weights
        discounted to the last integrate call (FARM_OPT_EDGES = k)."""
        lib = load_library()
        n = C.c_uint64(0)
        _check(lib.farm_map_read_edges(self._h, None, None, None, 0, C.byref(n)))
        a, b, w = np.zeros(n.value, np.uint32), np.zeros(n.value, np.uint32), np.zeros(n.value, np.float64)
        _check(lib.farm_map_read_edges(self._h, _hp(a), _hp(b), _hp(w), n.value, C.byref(n)))
        return a, b, w

    def read_covisibility(self):
        """uint64 [N, ceil(N/64)] covisibility bitset (FARM_OPT_COVISIBILITY)."""
        lib = load_library()
        w = C.c_int(0)
        _check(lib.farm_map_read_covisibility(self._h, None, C.byref(w)))
        n = C.c_int(0)
        _check(lib.farm_map_read(self._h, None, C.byref(n), None, None, None, None))
        rows = np.zeros((n.value, w.value), np.uint64)
        _check(lib.farm_map_read_covisibility(self._h, _hp(rows), C.byref(w)))
        return rows

    def counts(self):
        """(number of objects, number of owned voxels) without copying the map out."""
        n = C.c_int(0)
        nv = C.c_longlong(0)
        _check(load_library().farm_map_read(self._h, None, C.byref(n), None, None, None, C.byref(nv)))
        return n.value, nv.value

    def import_(self, objects, descriptors, voxel_keys, voxel_owner):
        objects = np.ascontiguousarray(objects, OBJECT_DTYPE)
        descriptors = np.ascontiguousarray(descriptors, np.float32)
        voxel_keys = np.ascontiguousarray(voxel_keys, np.uint64)
        voxel_owner = np.ascontiguousarray(voxel_owner, np.uint32)
        _check(load_library().farm_map_import(self._h, _hp(objects), len(objects), _hp(descriptors), _hp(voxel_keys),
                                              _hp(voxel_owner), len(voxel_keys)))

    def sync(self):
        t = np.zeros(1, TOTALS_DTYPE)
        _check(load_library().farm_map_sync(self._h, _hp(t)))
        return t[0]

    def kernel_launches(self):
        return int(load_library().farm_map_kernel_launches(self._h))

    def get_frame_seq(self):
        v = C.c_longlong(0)
        _check(load_library().farm_map_get_frame_seq(self._h, C.byref(v)))
        return v.value

    def set_frame_seq(self, frame_seq):
        _check(load_library().farm_map_set_frame_seq(self._h, int(frame_seq)))

    # ---- parity / debug
    def debug_backproject(self, depth, instance_mask, K, T_world_cam, n_det, xyz, keys):
        _check(load_library().farm_debug_backproject(self._h, _dp(depth), _dp(instance_mask), _dp(K), _dp(T_world_cam),
                                                     int(n_det), _dp(xyz), _dp(keys)))

    def debug_last_voxels(self):
        lib = load_library()
        M = self._last_M
        off = np.zeros(M + 1, np.int64)
        _check(lib.farm_debug_last_voxels(self._h, _hp(off), None, None, None))
        keys = np.empty(int(off[M]), np.uint64)
        n_px = np.empty(M, np.uint32)
        box = np.empty((M, 6), np.float32)
        _check(lib.farm_debug_last_voxels(self._h, _hp(off), _hp(keys), _hp(n_px), _hp(box)))
        return off, keys, n_px, box

    def debug_last_overlaps(self):
        lib = load_library()
        M = self._last_M
        off = np.zeros(M + 1, np.int64)
        _check(lib.farm_debug_last_overlaps(self._h, _hp(off), None, None))
        obj = np.empty(int(off[M]), np.int32)
        cnt = np.empty(int(off[M]), np.uint32)
        _check(lib.farm_debug_last_overlaps(self._h, _hp(off), _hp(obj), _hp(cnt)))
        return off, obj, cnt

    def debug_last_dense(self):
        M = self._last_M
        mc = np.empty(M, np.float32)
        am = np.empty(M, np.int32)
        _check(load_library().farm_debug_last_dense(self._h, _hp(mc), _hp(am)))
        return mc, am
