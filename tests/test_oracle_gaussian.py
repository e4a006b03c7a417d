"""Pins of the oracle's paper-faithful geometry (rules G1-G4).

None of these re-types the oracle's formulas: the detection and entity Gaussians are checked against
numpy's mean / cov of explicitly collected point sets, the Hellinger distance against its textbook special
cases and against the general formula evaluated with numpy.linalg.
"""
import numpy as np

from helpers import hand_frame, pow2_K, unit_rows

H, W = 96, 128
PACK = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]


def unpack(c):
    S = np.zeros((3, 3))
    for k, (a, b) in enumerate(PACK):
        S[a, b] = S[b, a] = c[k]
    return S


def new_map(oracle, vs=0.25, D=4):
    return oracle.OracleMap(vs, D, 0.5, 0.5, 0.5, 0, H, W)


def patch_frame(u0, v0, w, h, z_of, label=1):
    px = [(u, v, float(z_of(u, v)), label) for v in range(v0, v0 + h) for u in range(u0, u0 + w)]
    return hand_frame(H, W, px)


def test_GP1_detection_gaussian_is_numpy_mean_and_population_cov(oracle):
    """G1 ("lifted into a 3D Gaussian over the masked depth points"): mean and 1/n covariance of
    exactly the points the debug back-projection returns."""
    m = new_map(oracle)
    depth, mask = patch_frame(40, 30, 17, 9, lambda u, v: 2.0 + 0.01 * (u - 40) - 0.02 * (v - 30) + 0.003 * ((u * v) % 5))
    K, T = pow2_K(), np.eye(4, dtype=np.float32)
    xyz, keys = m.backproject(depth, mask, K, T, 1)
    pts = xyz[mask == 1].astype(np.float64)
    m.integrate(depth, mask, K, T, unit_rows(1, 4), 1)
    mu, cov, hell = m.last_gaussians()
    assert np.allclose(mu[0], pts.mean(0), atol=1e-6)
    assert np.allclose(unpack(cov[0]), np.cov(pts.T, bias=True), atol=1e-7)
    assert hell[0] == -1.0                                    # spawned: no entity to compare with (G4)
    w, mu_o, cov_o = m.read_gaussians()
    assert w[0] == len(pts) and np.allclose(mu_o[0], mu[0]) and np.allclose(cov_o[0], cov[0])


def test_GP2_sufficient_statistics_merge_of_two_halves_is_the_whole(oracle):
    """G2 (PAPER.md:352 M1 = w mu, M2 = w (Sigma + mu mu^T)): two detections of one entity in two calls give the
    Gaussian of the union of their points; weights are point counts."""
    m = new_map(oracle, vs=0.25)
    K, T = pow2_K(), np.eye(4, dtype=np.float32)
    zf = lambda u, v: 2.0 + 0.004 * (u - 40)
    dA, mA = patch_frame(40, 30, 12, 8, zf)
    dB, mB = patch_frame(46, 30, 14, 8, zf)                    # overlaps A in space: same voxels -> matched
    f = unit_rows(1, 4)
    m.integrate(dA, mA, K, T, f, 1)
    m.integrate(dB, mB, K, T, f, 1)
    assoc, is_new, _, _, _ = m.last_assoc()
    assert assoc[0] == 0 and not is_new[0]
    ptsA = m.backproject(dA, mA, K, T, 1)[0][mA == 1].astype(np.float64)
    ptsB = m.backproject(dB, mB, K, T, 1)[0][mB == 1].astype(np.float64)
    allp = np.concatenate([ptsA, ptsB])
    w, mu, cov = m.read_gaussians()
    assert w[0] == len(allp)
    assert np.allclose(mu[0], allp.mean(0), atol=1e-6)
    assert np.allclose(unpack(cov[0]), np.cov(allp.T, bias=True), atol=1e-7)


def test_GP3_hellinger_closed_forms(oracle):
    """G3 ("unitless and bounded in [0,1]"): textbook special cases of the Gaussian Hellinger distance."""
    I6 = np.array([1, 0, 0, 1, 0, 1], float)
    mu = np.array([0.3, -1.0, 2.0])
    assert oracle.hellinger(mu, 0.04 * I6, mu, 0.04 * I6, 0.0) == 0.0                      # H(p, p) = 0
    # equal isotropic covariances: H^2 = 1 - exp(-|dmu|^2 / (8 sigma^2))
    s2, d = 0.09, np.array([0.2, -0.1, 0.4])
    h = oracle.hellinger(mu, s2 * I6, mu + d, s2 * I6, 0.0)
    assert abs(h * h - (1 - np.exp(-(d @ d) / (8 * s2)))) < 1e-12
    # equal means, isotropic a^2 I and b^2 I in 3-D: BC = (2ab / (a^2 + b^2))^(3/2)
    a, b = 0.2, 0.5
    h = oracle.hellinger(mu, a * a * I6, mu, b * b * I6, 0.0)
    assert abs(h * h - (1 - (2 * a * b / (a * a + b * b)) ** 1.5)) < 1e-12
    # far apart -> 1, symmetric, in [0, 1]
    assert abs(oracle.hellinger(mu, 0.01 * I6, mu + 100.0, 0.01 * I6, 0.0) - 1.0) < 1e-12
    g = np.random.default_rng(5)
    for _ in range(50):
        A, B = g.standard_normal((3, 3)), g.standard_normal((3, 3))
        S1, S2 = A @ A.T + 0.05 * np.eye(3), B @ B.T + 0.05 * np.eye(3)
        c1, c2 = np.array([S1[a_, b_] for a_, b_ in PACK]), np.array([S2[a_, b_] for a_, b_ in PACK])
        m1, m2 = g.standard_normal(3), g.standard_normal(3)
        h12, h21 = oracle.hellinger(m1, c1, m2, c2, 0.0), oracle.hellinger(m2, c2, m1, c1, 0.0)
        assert 0.0 <= h12 <= 1.0 and abs(h12 - h21) < 1e-12
        # general formula through numpy.linalg (library determinant and solve)
        Sb = 0.5 * (S1 + S2)
        bc = (np.linalg.det(S1) ** 0.25 * np.linalg.det(S2) ** 0.25 / np.sqrt(np.linalg.det(Sb))
              * np.exp(-0.125 * (m1 - m2) @ np.linalg.solve(Sb, m1 - m2)))
        assert abs(h12 - np.sqrt(max(1 - bc, 0.0))) < 1e-9
    # the eps2 regulariser is an addition to both diagonals
    c = np.array([0.04, 0.01, 0.0, 0.02, 0.0, 1e-9])
    assert abs(oracle.hellinger(mu, c, mu + d, 2 * c, 0.01) - oracle.hellinger(mu, c + 0.01 * I6, mu + d, 2 * c + 0.01 * I6, 0.0)) < 1e-12


def test_GP4_hellinger_of_a_match_uses_the_entry_snapshot(oracle):
    """G4: the reported distance is between the detection's Gaussian and the matched entity's Gaussian as it was
    at entry (R2), regularised with eps = voxel_size; re-observing the same patch gives 0."""
    vs = 0.25
    m = new_map(oracle, vs=vs)
    K, T = pow2_K(), np.eye(4, dtype=np.float32)
    zf = lambda u, v: 2.0 + 0.004 * (u - 40)
    dA, mA = patch_frame(40, 30, 12, 8, zf)
    dB, mB = patch_frame(44, 30, 12, 8, zf)
    f = unit_rows(1, 4)
    m.integrate(dA, mA, K, T, f, 1)
    _, muA, covA = m.read_gaussians()
    m.integrate(dA, mA, K, T, f, 1)
    assert 0.0 <= m.last_gaussians()[2][0] < 1e-6                # identical Gaussians (up to the merge rounding)
    _, mu1, cov1 = m.read_gaussians()
    m.integrate(dB, mB, K, T, f, 1)
    muB, covB, hell = m.last_gaussians()
    assert m.last_assoc()[0][0] == 0
    expect = oracle.hellinger(muB[0], covB[0], mu1[0], cov1[0], vs * vs)
    assert abs(hell[0] - expect) < 1e-6 and 0.0 < hell[0] < 1.0


def test_CP1_covisibility_bitset_is_the_set_of_co_observed_pairs(oracle):
    """C1 ("A bitset adjacency (N x ceil(N/64) blocks) marks all pairs of entities that were jointly
    visible in the current batch"): brute-force pair enumeration over the per-call association lists; symmetric, no
    diagonal, bits only accumulate."""
    from paper_2606_15476_b200 import scenes as S
    from helpers import integrate_frames
    cfg = S.get_config(0)
    sc = S.BoxScene(cfg)
    m = oracle.OracleMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, cfg.dtype, cfg.H, cfg.W)
    pairs, prev = set(), None
    for k in range(0, 12, 2):
        integrate_frames(m, [sc.frame(k), sc.frame(k + 1)])        # one call = one batch of two frames
        assoc = m.last_assoc()[0]
        seen = sorted(set(int(a) for a in assoc if a >= 0))
        pairs |= {(a, b) for a in seen for b in seen if a != b}
        rows = m.read_covisibility()
        N = rows.shape[0]
        assert rows.shape[1] == (N + 63) // 64
        got = {(a, b) for a in range(N) for b in range(N) if (int(rows[a, b >> 6]) >> (b & 63)) & 1}
        assert got == pairs
        assert all((b, a) in got for a, b in got) and all(a != b for a, b in got)
        if prev is not None:
            assert prev <= got
        prev = got
    assert len(pairs) > 10
