"""Pins for the enclosing balls of the pseudo i-particle (App. B): GEO and Ritter's EBS.  Independent facts:
every member is inside; special cases with known answers; the smallest enclosing ball (found here by an independent
iteration in double) bounds both from below, and EBS stays within the ~10 % Ritter claims and the paper repeats."""
import numpy as np

import oracle


def _pts(k, rng, scale=1.0):
    p = np.zeros((k, 4), np.float32)
    p[:, :3] = rng.normal(size=(k, 3)) * scale + rng.normal(size=3)
    p[:, 3] = 1.0
    return p


def _seb_radius(x, iters=4000):
    """Badoiu-Clarkson: move the centre 1/(i+1) of the way to the farthest point; converges to the smallest enclosing ball."""
    c = x[0].copy()
    for i in range(1, iters):
        far = x[np.argmax(((x - c) ** 2).sum(1))]
        c += (far - c) / (i + 1)
    return np.sqrt(((x - c) ** 2).sum(1).max())


def test_members_are_enclosed_and_radius_is_the_exact_maximum():
    rng = np.random.default_rng(1)
    for k in (1, 2, 3, 5, 17, 32):
        for kind in (0, 1, 2, 3, 4):
            p = _pts(k, rng, scale=10.0 ** rng.uniform(-3, 1))
            ball = oracle.group_ball(p, np.arange(k), kind)
            d = np.sqrt(((p[:, :3].astype(np.float64) - ball[:3].astype(np.float64)) ** 2).sum(1))
            assert np.all(d <= ball[3] * (1 + 2e-7) + 1e-30)
            assert np.isclose(d.max(), ball[3], rtol=3e-7, atol=1e-30)


def test_special_cases():
    one = np.array([[1.5, -2.0, 3.0, 1.0]], np.float32)
    two = np.array([[0, 0, 0, 1], [2, 4, 4, 1]], np.float32)                       # distance 6
    line = np.zeros((9, 4), np.float32)
    line[:, 0] = np.arange(9)                                                      # collinear: diameter 8
    for kind in (0, 1, 2, 3, 4):
        b = oracle.group_ball(one, [0], kind)
        assert np.array_equal(b[:3], one[0, :3]) and b[3] == 0
        b = oracle.group_ball(two, [0, 1], kind)
        assert np.allclose(b, [1, 2, 2, 3], atol=1e-6)
        b = oracle.group_ball(line, np.arange(9), kind)
        assert np.allclose(b, [4, 0, 0, 4], atol=1e-6)
    # members are a SUBSET of the array: only they count
    rng = np.random.default_rng(2)
    p = _pts(40, rng)
    mem = np.array([3, 7, 8, 20, 31], np.uint32)
    for kind in (0, 1, 2, 3, 4):
        assert np.array_equal(oracle.group_ball(p, mem, kind), oracle.group_ball(p[mem], np.arange(5), kind))


def test_radii_against_the_smallest_enclosing_ball():
    """EBS "overestimation is 5% in most cases and ~10% in the worst case"; GEO "smaller than 1.15 r_SEB in most cases"."""
    rng = np.random.default_rng(3)
    ratios = {0: [], 1: []}
    for _ in range(300):
        k = int(rng.integers(4, 33))
        p = _pts(k, rng)
        seb = _seb_radius(p[:, :3].astype(np.float64))
        for kind in (0, 1):
            ratios[kind].append(oracle.group_ball(p, np.arange(k), kind)[3] / seb)
    geo, ebs = np.array(ratios[0]), np.array(ratios[1])
    assert geo.min() > 1 - 2e-3 and ebs.min() > 1 - 2e-3               # nothing beats the smallest ball (iteration tolerance)
    assert np.median(ebs) < 1.08 and ebs.max() < 1.25
    assert np.median(geo) < 1.15 and np.median(ebs) < np.median(geo)   # EBS is the tighter of the two (Fig. B.10)


def test_com_and_cmp_balls():
    """App. B items 4 and 5: COM is centred on the mass-weighted mean of the members; CMP is the smaller of GEO and COM; COM is the
    loosest of the generators ("r_ball in the COM is much bigger")."""
    rng = np.random.default_rng(7)
    r = {0: [], 2: [], 3: []}
    for _ in range(200):
        k = int(rng.integers(2, 33))
        p = _pts(k, rng)
        p[:, 3] = rng.uniform(0.1, 3.0, k).astype(np.float32)
        com = (p[:, 3:4].astype(np.float64) * p[:, :3]).sum(0) / p[:, 3].astype(np.float64).sum()
        b = {kind: oracle.group_ball(p, np.arange(k), kind) for kind in (0, 2, 3)}
        assert np.allclose(b[2][:3], com, atol=2e-6 * np.abs(p[:, :3]).max())
        assert b[3][3] == min(b[0][3], b[2][3])
        assert np.array_equal(b[3], b[0]) or np.array_equal(b[3], b[2])
        for kind in r:
            r[kind].append(b[kind][3])
    assert np.mean(r[2]) > np.mean(r[0]) >= np.mean(r[3])
    # massless members: COM is undefined, the ball falls back to GEO
    p = _pts(6, rng)
    p[:, 3] = 0.0
    assert np.array_equal(oracle.group_ball(p, np.arange(6), 2), oracle.group_ball(p, np.arange(6), 0))


def _seb_by_definition(x):
    """The smallest enclosing ball written out (double): it is fixed by 2, 3 or 4 of the points on its boundary, so the smallest ball
    among the circumscribed balls of all such subsets that contain every point is it.  O(k^4): tiny sets only."""
    from itertools import combinations
    k = x.shape[0]
    best = (np.inf, None)
    for m in (2, 3, 4):
        for sub in combinations(range(k), m):
            q = x[list(sub)]
            a = q[1:] - q[0]                                   # centre = q0 + sum l_j a_j, 2 a_i . (c - q0) = |a_i|^2
            g = 2.0 * a @ a.T
            if abs(np.linalg.det(g)) < 1e-14 * np.prod(np.diag(g)):
                continue
            lam = np.linalg.solve(g, (a * a).sum(1))
            c = q[0] + lam @ a
            r = np.sqrt(((q[0] - c) ** 2).sum())
            if r < best[0] and np.all(np.sqrt(((x - c) ** 2).sum(1)) <= r * (1 + 1e-9)):
                best = (r, c)
    return best


def test_seb_is_the_smallest_enclosing_ball():
    """App. B item 1: the oracle's SEB (Welzl's recursion in single precision, reading R19) against the definition in double on
    random sets of 2 .. 12 points, on points of a sphere's surface (many near-cospherical supports) and on flat and collinear sets."""
    rng = np.random.default_rng(11)
    cases = [_pts(int(rng.integers(2, 13)), rng, scale=10.0 ** rng.uniform(-2, 1)) for _ in range(60)]
    sph = rng.normal(size=(10, 3)); sph /= np.linalg.norm(sph, axis=1)[:, None]
    p = np.zeros((10, 4), np.float32); p[:, :3] = 3.0 * sph + 1.0; cases.append(p)
    flat = _pts(9, rng); flat[:, 2] = 0.5; cases.append(flat)
    for p in cases:
        k = p.shape[0]
        r_def, c_def = _seb_by_definition(p[:, :3].astype(np.float64))
        b = oracle.group_ball(p, np.arange(k), 4)
        assert r_def * (1 - 1e-6) <= b[3] <= r_def * (1 + 2e-5), (k, b[3], r_def)
        assert np.linalg.norm(b[:3] - c_def) <= 3e-3 * r_def
    # and it is never larger than the other generators' balls (Fig. B.10 plots r_ball / r_SEB >= 1)
    for _ in range(200):
        k = int(rng.integers(2, 33))
        p = _pts(k, rng)
        r = [oracle.group_ball(p, np.arange(k), kind)[3] for kind in (0, 1, 2, 3, 4)]
        assert r[4] <= min(r[:4]) * (1 + 1e-5)
        assert r[4] >= _seb_radius(p[:, :3].astype(np.float64)) * (1 - 2e-3)
