"""ctypes wrapper of the CPU oracle (oracle/farm_oracle.cpp).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
Argument marshalling only; every rule lives in the C++ file.
"""
import ctypes as C
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import build as _build  # noqa: E402  (oracle/build.py)

sys.path.pop(0)

OBJECT_DTYPE = np.dtype(
    [("id", "<i4"), ("n_voxels", "<u4"), ("n_obs", "<u4"), ("aabb_min", "<f4", 3), ("aabb_max", "<f4", 3),
     ("best_frame", "<i4"), ("best_det", "<i4"), ("best_pixels", "<u4"), ("best_cam_pos", "<f4", 3),
     ("n_points", "<u8")], align=True)
STATS_DTYPE = np.dtype(
    [("valid_points", "<u8"), ("dropped_points", "<u8"), ("ignored_pixels", "<u8"), ("unique_voxels", "<u8"),
     ("matches", "<u4"), ("spawns", "<u4"), ("skipped", "<u4"), ("n_det", "<u4")], align=True)
assert OBJECT_DTYPE.itemsize == 72
VIEW_DTYPE = np.dtype([("frame", "<i4"), ("det", "<i4"), ("n_px", "<u4"), ("cam", "<f4", 3), ("dir", "<f4", 3), ("dist", "<f4")])
assert VIEW_DTYPE.itemsize == 40
PRED_NEAR, PRED_NEXTTO, PRED_CLOSEST, PRED_FARTHEST = 0, 1, 2, 3

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_create.restype = C.c_void_p
        _lib.oracle_create.argtypes = [C.c_float, C.c_int, C.c_float, C.c_float, C.c_float, C.c_int, C.c_int,
                                       C.c_int, C.c_float, C.c_float]
        _lib.oracle_clone.restype = C.c_void_p
        _lib.oracle_clone.argtypes = [C.c_void_p]
        _lib.oracle_n_voxels.restype = C.c_longlong
        _lib.oracle_round_to_storage.restype = C.c_float
        _lib.oracle_round_to_storage.argtypes = [C.c_float, C.c_int]
        _lib.oracle_cosine.restype = C.c_float
        _lib.oracle_set_option.argtypes = [C.c_void_p, C.c_int, C.c_double]
        _lib.oracle_hellinger.restype = C.c_double
        _lib.oracle_hellinger.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double]
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class OracleMap:
    def __init__(self, voxel_size, D, w_geo, w_sem, tau, dtype, H, W, z_min=0.0, z_max=float("inf")):
        self.D, self.dtype, self.H, self.W = D, dtype, H, W
        self.h = C.c_void_p(lib().oracle_create(voxel_size, D, w_geo, w_sem, tau, dtype, H, W, z_min, z_max))

    def __del__(self):
        if getattr(self, "h", None):
            lib().oracle_destroy(self.h)
            self.h = None

    # ---- round-2 options (all off by default): U correspondence, H geometry, V views
    OPT_CORRESPONDENCE, OPT_GEOMETRY, OPT_PREFILTER_COS, OPT_HELLINGER_BUDGET, OPT_VIEWS_K, OPT_VIEW_COS, OPT_VIEW_CLOSER = 1, 2, 3, 4, 5, 6, 7
    OPT_EDGES_K, OPT_EDGE_DECAY, OPT_EDGE_CUTOFF = 8, 9, 10

    def set_option(self, key, value):
        rc = lib().oracle_set_option(self.h, C.c_int(key), C.c_double(value))
        assert rc == 0, f"oracle option {key} = {value} rejected"
        if key == self.OPT_VIEWS_K:
            self.views_k = int(value)

    def last_tau_gap(self):
        """per detection the smallest |score - tau| over every scored pair (tests: margin filter with correspondence)"""
        M = lib().oracle_last_M(self.h)
        gap = np.zeros(M, np.float32)
        lib().oracle_last_tau_gap(self.h, _p(gap))
        return gap

    def read_edges(self):
        """W: (a [n], b [n], w [n]) weighted covisibility edges, a < b, ascending, weights decayed to now."""
        lib().oracle_read_edges.restype = C.c_longlong
        n = lib().oracle_read_edges(self.h, None, None, None)
        a, b, w = np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros(n, np.float64)
        lib().oracle_read_edges(self.h, _p(a), _p(b), _p(w))
        return a, b, w

    def read_alias(self):
        """U4: alias [N]: the live entity every id now stands for (itself while alive)."""
        N = lib().oracle_n_objects(self.h)
        al = np.zeros(N, np.int32)
        lib().oracle_read_alias(self.h, _p(al))
        return al

    def last_merges(self):
        """U4: (loser [n], winner [n]) entity merges executed by the last call."""
        n = lib().oracle_last_merges(self.h, None, None)
        a, b = np.zeros(n, np.int32), np.zeros(n, np.int32)
        lib().oracle_last_merges(self.h, _p(a), _p(b))
        return a, b

    def read_views(self):
        """V: (views [N, k] VIEW_DTYPE, counts [N])"""
        N = lib().oracle_n_objects(self.h)
        k = getattr(self, "views_k", 0)
        views = np.zeros((N, max(k, 1)), VIEW_DTYPE)
        counts = np.zeros(N, np.int32)
        if k:
            lib().oracle_read_views(self.h, _p(views), _p(counts), C.c_int(k))
        return views[:, :k], counts

    def clone(self):
        c = OracleMap.__new__(OracleMap)
        c.D, c.dtype, c.H, c.W = self.D, self.dtype, self.H, self.W
        c.views_k = getattr(self, "views_k", 0)
        c.h = C.c_void_p(lib().oracle_clone(self.h))
        return c

    def backproject(self, depth, mask, K, T, n_det):
        depth = np.ascontiguousarray(depth, np.float32)
        mask = np.ascontiguousarray(mask, np.uint16)
        K = np.ascontiguousarray(K, np.float32)
        T = np.ascontiguousarray(T, np.float32)
        xyz = np.empty((self.H, self.W, 3), np.float32)
        keys = np.empty((self.H, self.W), np.uint64)
        lib().oracle_backproject(self.h, _p(depth), _p(mask), _p(K), _p(T), C.c_int(n_det), _p(xyz), _p(keys))
        return xyz, keys

    def integrate_batch(self, depth, mask, K, T, desc, n_det):
        n_det = np.ascontiguousarray(n_det, np.int32).reshape(-1)
        F = n_det.shape[0]
        depth = np.ascontiguousarray(depth, np.float32).reshape(F, self.H, self.W)
        mask = np.ascontiguousarray(mask, np.uint16).reshape(F, self.H, self.W)
        K = np.ascontiguousarray(K, np.float32).reshape(F, 3, 3)
        T = np.ascontiguousarray(T, np.float32).reshape(F, 4, 4)
        desc = np.ascontiguousarray(desc)
        assert desc.dtype.itemsize == (4 if self.dtype == 0 else 2)
        assert desc.size == int(n_det.sum()) * self.D
        return lib().oracle_integrate_batch(self.h, C.c_int(F), _p(depth), _p(mask), _p(K), _p(T), _p(desc),
                                            _p(n_det))

    def integrate(self, depth, mask, K, T, desc, n_det):
        return self.integrate_batch(depth, mask, K, T, desc, [n_det])

    def last_assoc(self):
        M = lib().oracle_last_M(self.h)
        assoc = np.empty(M, np.int32)
        is_new = np.empty(M, np.uint8)
        best = np.empty(M, np.float32)
        second = np.empty(M, np.float32)
        st = np.zeros(1, STATS_DTYPE)
        lib().oracle_last_assoc(self.h, _p(assoc), _p(is_new), _p(best), _p(second), _p(st))
        return assoc, is_new, best, second, st[0]

    def last_dense(self):
        """R16: (max_o clamp(cos) [M], argmax [M], lowest id on ties; (0, -1) for skipped detections / empty map)."""
        M = lib().oracle_last_M(self.h)
        mc = np.zeros(M, np.float32)
        am = np.zeros(M, np.int32)
        lib().oracle_last_dense(self.h, _p(mc), _p(am), None)
        return mc, am

    def last_dense_second(self):
        """runner-up of the dense row maximum (-inf when N < 2); tests use it to skip near-ties"""
        M = lib().oracle_last_M(self.h)
        sec = np.zeros(M, np.float32)
        lib().oracle_last_dense(self.h, None, None, _p(sec))
        return sec

    def last_voxels(self):
        M = lib().oracle_last_M(self.h)
        off = np.empty(M + 1, np.int64)
        lib().oracle_last_voxels(self.h, _p(off), None, None, None)
        keys = np.empty(int(off[M]), np.uint64)
        n_px = np.empty(M, np.uint32)
        box = np.empty((M, 6), np.float32)
        lib().oracle_last_voxels(self.h, _p(off), _p(keys), _p(n_px), _p(box))
        return off, keys, n_px, box

    def last_overlaps(self):
        M = lib().oracle_last_M(self.h)
        off = np.empty(M + 1, np.int64)
        lib().oracle_last_overlaps(self.h, _p(off), None, None)
        obj = np.empty(int(off[M]), np.int32)
        cnt = np.empty(int(off[M]), np.uint32)
        lib().oracle_last_overlaps(self.h, _p(off), _p(obj), _p(cnt))
        return off, obj, cnt

    def last_gaussians(self):
        """G1 / G4: (mu [M,3], cov [M,6] packed xx xy xz yy yz zz, hellinger [M]) of the last call's detections."""
        M = lib().oracle_last_M(self.h)
        mu = np.zeros((M, 3), np.float32)
        cov = np.zeros((M, 6), np.float32)
        hell = np.zeros(M, np.float32)
        lib().oracle_last_gaussians(self.h, _p(mu), _p(cov), _p(hell))
        return mu, cov, hell

    def read_gaussians(self):
        """G2: (weight [N] float64, mu [N,3], cov [N,6]) of the map's entities."""
        N = lib().oracle_n_objects(self.h)
        w = np.zeros(N, np.float64)
        mu = np.zeros((N, 3), np.float32)
        cov = np.zeros((N, 6), np.float32)
        lib().oracle_read_gaussians(self.h, _p(w), _p(mu), _p(cov))
        return w, mu, cov

    def read_covisibility(self):
        """C1: uint64 [N, ceil(N/64)]; bit b of row a = entities a and b were observed in one call."""
        N = lib().oracle_n_objects(self.h)
        words = lib().oracle_covis_words(self.h)
        rows = np.zeros((N, words), np.uint64)
        lib().oracle_read_covis(self.h, _p(rows))
        return rows

    def read(self, voxels=True):
        N = lib().oracle_n_objects(self.h)
        nv = lib().oracle_n_voxels(self.h)
        objs = np.zeros(N, OBJECT_DTYPE)
        desc = np.empty((N, self.D), np.float32)
        keys = np.empty(nv if voxels else 0, np.uint64)
        owners = np.empty(nv if voxels else 0, np.uint32)
        lib().oracle_read(self.h, _p(objs), _p(desc), _p(keys) if voxels else None, _p(owners) if voxels else None)
        return objs, desc, keys, owners

    def import_(self, objs, desc, keys, owners):
        objs = np.ascontiguousarray(objs, OBJECT_DTYPE)
        desc = np.ascontiguousarray(desc, np.float32)
        keys = np.ascontiguousarray(keys, np.uint64)
        owners = np.ascontiguousarray(owners, np.uint32)
        return lib().oracle_import(self.h, _p(objs), C.c_int(len(objs)), _p(desc), _p(keys), _p(owners),
                                   C.c_longlong(len(keys)))


def round_to_storage(x, dtype):
    x = np.asarray(x, np.float32)
    out = np.empty_like(x)
    flat_in, flat_out = x.reshape(-1), out.reshape(-1)
    for i in range(flat_in.size):
        flat_out[i] = lib().oracle_round_to_storage(float(flat_in[i]), dtype)
    return out


def hellinger(mu1, cov1, mu2, cov2, eps2):
    """G3: Hellinger distance of two 3-D Gaussians; cov packed xx xy xz yy yz zz; eps2 added to the diagonals."""
    a = [np.ascontiguousarray(x, np.float64) for x in (mu1, cov1, mu2, cov2)]
    return float(lib().oracle_hellinger(_p(a[0]), _p(a[1]), _p(a[2]), _p(a[3]), C.c_double(eps2)))


def bhattacharyya(mu1, cov1, mu2, cov2, eps2):
    """W2: Bhattacharyya distance of two 3-D Gaussians (H = sqrt(1 - exp(-DB))); cov packed xx xy xz yy yz zz."""
    lib().oracle_bhattacharyya.restype = C.c_double
    lib().oracle_bhattacharyya.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double]
    a = [np.ascontiguousarray(x, np.float64) for x in (mu1, cov1, mu2, cov2)]
    return float(lib().oracle_bhattacharyya(_p(a[0]), _p(a[1]), _p(a[2]), _p(a[3]), C.c_double(eps2)))


def cosine(a, b):
    a = np.ascontiguousarray(a, np.float32)
    b = np.ascontiguousarray(b, np.float32)
    return float(lib().oracle_cosine(_p(a), _p(b), C.c_int(a.size)))


def query(alive, emb, cls, centroid, q_target, target_class, pred_types, q_landmarks, topk, want_cos=False):
    """Q1-Q5 retrieval scoring.  emb: three [N, d_s] float32 arrays; q_target: four channel vectors (d0, d0, d1, d2);
    q_landmarks: one such list of four per predicate.  Returns dict(s_sem, gbar, s, landmarks, top[, cos])."""
    N = len(alive)
    alive = np.ascontiguousarray(alive, np.uint8)
    emb = [np.ascontiguousarray(e, np.float32) for e in emb]
    dims = [e.shape[1] for e in emb]
    cls = np.ascontiguousarray(cls, np.int32)
    centroid = np.ascontiguousarray(centroid, np.float32)
    qt = np.ascontiguousarray(np.concatenate([np.asarray(x, np.float32).ravel() for x in q_target]), np.float32)
    P = len(pred_types)
    pt = np.ascontiguousarray(pred_types, np.int32)
    ql = np.ascontiguousarray(np.concatenate([np.asarray(x, np.float32).ravel() for lm in q_landmarks for x in lm]) if P else np.zeros(1), np.float32)
    s_sem, gbar, sc = np.zeros(N, np.float32), np.zeros(N, np.float32), np.zeros(N, np.float32)
    lms = np.zeros(max(P, 1), np.int32)
    top = np.zeros(topk, np.int32)
    cos = np.zeros((4, N), np.float32) if want_cos else None
    rc = lib().oracle_query(C.c_int(N), _p(alive), _p(emb[0]), _p(emb[1]), _p(emb[2]), C.c_int(dims[0]), C.c_int(dims[1]),
                            C.c_int(dims[2]), _p(cls), _p(centroid), _p(qt), C.c_int(target_class), C.c_int(P), _p(pt), _p(ql),
                            C.c_int(topk), _p(s_sem), _p(gbar), _p(sc), _p(lms), _p(top), _p(cos))
    assert rc == 0
    out = {"s_sem": s_sem, "gbar": gbar, "s": sc, "landmarks": lms[:P], "top": top}
    if want_cos:
        out["cos"] = cos
    return out
