"""Shared test helpers: hand-made frames, key packing as include/farm.h defines it, margin filter."""
import numpy as np

KEY_BIAS = 1 << 20
KEY_EMPTY = np.uint64(0xFFFFFFFFFFFFFFFF)


def pack_key(ix, iy, iz):
    """Voxel key layout of include/farm.h: three biased 21-bit indices, x highest."""
    ix = np.asarray(ix, np.int64) + KEY_BIAS
    iy = np.asarray(iy, np.int64) + KEY_BIAS
    iz = np.asarray(iz, np.int64) + KEY_BIAS
    return ((ix.astype(np.uint64) << np.uint64(42)) | (iy.astype(np.uint64) << np.uint64(21)) | iz.astype(np.uint64))


def unpack_key(k):
    k = np.asarray(k, np.uint64)
    m = np.uint64((1 << 21) - 1)
    return (((k >> np.uint64(42)) & m).astype(np.int64) - KEY_BIAS,
            ((k >> np.uint64(21)) & m).astype(np.int64) - KEY_BIAS,
            (k & m).astype(np.int64) - KEY_BIAS)


def pow2_K(f=128.0, cx=64.0, cy=48.0):
    return np.array([[f, 0, cx], [0, f, cy], [0, 0, 1]], np.float32)


def hand_frame(H, W, pixels):
    """pixels: iterable of (u, v, z, label).  Returns depth f32[H,W], mask u16[H,W]."""
    depth = np.zeros((H, W), np.float32)
    mask = np.zeros((H, W), np.uint16)
    for u, v, z, lab in pixels:
        depth[v, u] = z
        mask[v, u] = lab
    return depth, mask


def unit_rows(n, D, seed=0):
    g = np.random.default_rng(seed)
    x = g.standard_normal((n, D)).astype(np.float32)
    return x / np.linalg.norm(x, axis=1, keepdims=True)


def margin_filter(make_oracle_clone, frames, tau, margin=1e-3, max_rounds=8):
    """detections whose oracle score is within `margin` of tau or of the runner-up are
    removed from the batch (label -> 0, rows compacted).  `make_oracle_clone()` must return an oracle map in
    the state before this batch (we re-run the batch on a fresh clone each round)."""
    from paper_2606_15476_b200 import scenes as S
    for _ in range(max_rounds):
        m = make_oracle_clone()
        integrate_frames(m, frames)
        assoc, is_new, best, second, _ = m.last_assoc()
        bad = []
        for j in range(len(assoc)):
            if assoc[j] < 0:
                continue
            close_tau = abs(float(best[j]) - tau) <= margin
            close_second = (not is_new[j]) and (float(best[j]) - float(second[j]) <= margin)
            if close_tau or close_second:
                bad.append(j)
        if not bad:
            return frames
        out, base = [], 0
        for fr in frames:
            drop = [j - base for j in bad if base <= j < base + fr.n_det]
            out.append(S.drop_detections(fr, drop))
            base += fr.n_det
        frames = out
    return frames


def stack_frames(frames):
    depth = np.stack([f.depth for f in frames])
    mask = np.stack([f.mask for f in frames])
    K = np.stack([f.K for f in frames])
    T = np.stack([f.T for f in frames])
    desc = np.concatenate([f.desc for f in frames], axis=0) if frames else None
    n_det = np.array([f.n_det for f in frames], np.int32)
    return depth, mask, K, T, desc, n_det


def integrate_frames(m, frames):
    depth, mask, K, T, desc, n_det = stack_frames(frames)
    return m.integrate_batch(depth, mask, K, T, desc, n_det)
