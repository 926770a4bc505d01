"""Pins for the oracle's direct sum (eq. 1) and group tree walk (O7: eq. 5-7)."""
import numpy as np
import pytest

from paper_1610_07279_b200 import workloads as W


def _brute_numpy(pos, eps):
    p = pos.astype(np.float64)
    d = p[None, :, :3] - p[:, None, :3]
    r2 = (d ** 2).sum(-1) + eps * eps
    np.fill_diagonal(r2, np.inf)
    u = 1.0 / np.sqrt(r2)
    acc = (p[None, :, 3:4] * u[..., None] ** 3 * d).sum(1)
    pot = -(p[None, :, 3] * u).sum(1)
    return np.concatenate([acc, pot[:, None]], axis=1)


def test_direct_matches_numpy_bruteforce(oracle):
    rng = np.random.default_rng(1)
    pos = W.plummer(300, seed=3)
    pos[:, 3] = rng.uniform(0.1, 2.0, 300).astype(np.float32)
    ref = _brute_numpy(pos, 0.05)
    out = oracle.direct(pos, 0.05)
    assert np.allclose(out, ref, rtol=1e-12, atol=1e-13)
    sub = np.array([5, 17, 299], np.uint32)
    assert np.allclose(oracle.direct(pos, 0.05, sub), ref[sub], rtol=1e-12, atol=1e-13)


def test_two_body_closed_form(oracle):
    """Textbook: two softened point masses on the x axis."""
    m1, m2, d, eps = 2.0, 3.0, 1.5, 0.25
    pos = np.array([[0, 0, 0, m1], [d, 0, 0, m2]], np.float32)
    out = oracle.direct(pos, eps)
    s = (d * d + eps * eps)
    assert out[0] == pytest.approx([m2 * d / s ** 1.5, 0, 0, -m2 / s ** 0.5], rel=1e-12)
    assert out[1] == pytest.approx([-m1 * d / s ** 1.5, 0, 0, -m1 / s ** 0.5], rel=1e-12)


def test_cube_corner_symmetry(oracle):
    """8 equal masses on cube corners: |a| equal, pointing at the centre; a test mass at the centre feels 0."""
    c = np.array([[x, y, z] for x in (-1, 1) for y in (-1, 1) for z in (-1, 1)], np.float32)
    pos = np.concatenate([np.c_[c, np.ones(8, np.float32)], [[0, 0, 0, 1e-3]]]).astype(np.float32)
    out = oracle.direct(pos, 0.1)
    assert np.allclose(out[8, :3], 0, atol=1e-14)
    a = out[:8, :3]
    mag = np.linalg.norm(a, axis=1)
    assert np.allclose(mag, mag[0], rtol=1e-12)
    assert np.allclose(a / mag[:, None], -c / np.sqrt(3), atol=1e-12)


@pytest.mark.parametrize("n,active_frac,G", [(1500, 1.0, 32), (1500, 0.2, 32), (777, 1.0, 16), (40, 1.0, 32)])
def test_walk_with_nothing_accepted_equals_direct(oracle, n, active_frac, G):
    """Delta_acc = 0 / theta = 0: no cell is ever accepted, the list is all particles => eq. 1."""
    pos = W.hernquist(n, seed=5)
    t = oracle.build_tree(pos, n_leaf=8)
    eps = float(np.float32(0.01))  # the walk takes eps as fp32: give eq. 1 the same value
    ref = oracle.direct(t.pos_sorted, eps)
    active = None if active_frac == 1.0 else W.random_active_subset(n, active_frac)
    rows = np.arange(n) if active is None else active
    for kind, aold in ((1, None), (0, np.ones(n, np.float32))):
        out, cnt = oracle.walk_tree(t, eps=eps, mac_kind=kind, mac_param=0.0, aold=aold, active=active, group_size=G)
        assert np.allclose(out[rows], ref[rows], rtol=1e-11, atol=1e-13)
        assert cnt["interactions"] == len(rows) * n
        if active is not None:
            mask = np.ones(n, bool)
            mask[active] = False
            assert np.all(out[mask] == 0)  # only active entries written


def test_pseudo_i_distance_is_conservative(oracle):
    """the ball-surface distance never exceeds the true distance of any member to the pseudo-j."""
    pos = W.plummer(4096, seed=8)
    t = oracle.build_tree(pos)
    rng = np.random.default_rng(0)
    p = t.pos_sorted.astype(np.float64)
    for g in range(0, 128, 3):
        members = np.arange(32 * g, 32 * g + 32, dtype=np.uint32)
        members = members[rng.random(32) < 0.6]
        if members.size == 0:
            continue
        ball = oracle.group_ball(t.pos_sorted, members).astype(np.float64)
        rk = np.linalg.norm(p[members, :3] - ball[:3], axis=1)
        assert np.all(rk <= ball[3] * (1 + 1e-6))
        for J in rng.integers(0, t.n_nodes, 50):
            rJ = t.com[J, :3].astype(np.float64)
            d = max(np.linalg.norm(rJ - ball[:3]) - ball[3], 0.0)
            assert d <= np.linalg.norm(p[members, :3] - rJ, axis=1).min() * (1 + 1e-6) + 1e-7


@pytest.fixture(scope="module")
def plummer_case(oracle):
    pos, cfg = W.make_config("plummer_2p13", seed=1)
    t = oracle.build_tree(pos)
    ref = oracle.direct(t.pos_sorted, cfg["eps"])
    boot, _ = oracle.walk_tree(t, eps=cfg["eps"], mac_kind=1, mac_param=0.5)
    aold = np.linalg.norm(boot[:, :3], axis=1).astype(np.float32)
    return t, cfg, ref, aold


def _rel_err(out, ref):
    return np.linalg.norm(out[:, :3] - ref[:, :3], axis=1) / np.linalg.norm(ref[:, :3], axis=1)


def test_error_shrinks_as_accuracy_parameter_tightens(oracle, plummer_case):
    """tighter Delta_acc => smaller error; ~1e-3 median for Delta_acc 2^-8..2^-6."""
    t, cfg, ref, aold = plummer_case
    med, p99, work, mom = [], [], [], []
    for ld in (1, 3, 5, 7, 9, 11, 14, 17, 20):
        out, cnt = oracle.walk_tree(t, eps=cfg["eps"], mac_kind=0, mac_param=2.0 ** -ld, aold=aold)
        e = _rel_err(out, ref)
        med.append(np.median(e)); p99.append(np.percentile(e, 99)); work.append(cnt["interactions"])
        m = t.pos_sorted[:, 3:4].astype(np.float64)
        mom.append(np.linalg.norm((m * out[:, :3]).sum(0)) / (m[:, 0] * np.linalg.norm(out[:, :3], axis=1)).sum())
    assert all(a > b for a, b in zip(med, med[1:])) and all(a > b for a, b in zip(p99, p99[1:]))
    assert all(a < b for a, b in zip(work, work[1:]))
    assert 3e-4 < med[3] < 3e-3            # Delta_acc = 2^-7
    assert med[-1] < 1e-5
    assert mom[-1] < mom[0] and mom[3] < 3 * med[3]   # momentum near-conservation tracks the force error
    # opening angle eq. 2 as well: theta 0.9 -> 0.3 monotone
    e_t = [np.median(_rel_err(oracle.walk_tree(t, eps=cfg["eps"], mac_kind=1, mac_param=th)[0], ref)) for th in (0.9, 0.6, 0.3)]
    assert e_t[0] > e_t[1] > e_t[2]


def test_potential_matches_direct(oracle, plummer_case):
    t, cfg, ref, aold = plummer_case
    out, _ = oracle.walk_tree(t, eps=cfg["eps"], mac_kind=0, mac_param=2.0 ** -9, aold=aold)
    assert np.median(np.abs(out[:, 3] - ref[:, 3]) / np.abs(ref[:, 3])) < 2e-4
    assert np.all(out[:, 3] < 0)


def test_plummer_closed_form_large_n(oracle):
    """Exact Plummer sphere (a = 1, truncated at R = 20, mass renormalised to 1):
    M(<r) = r^3/(1+r^2)^{3/2} / M_R,  a_r = -M(<r)/r^2,  Phi(r) = -[(1+r^2)^{-1/2} - (1+R^2)^{-3/2} ... ]
    Here the potential is checked through Phi(r) = -M(<r)/r - int_r^R dM/r' computed by quadrature of the
    closed-form density, the radial acceleration through M(<r)."""
    n = 1 << 15
    pos = W.plummer(n, seed=2)
    eps = 1.0 / 64
    t = oracle.build_tree(pos)
    boot, _ = oracle.walk_tree(t, eps=eps, mac_kind=1, mac_param=0.5)
    aold = np.linalg.norm(boot[:, :3], axis=1).astype(np.float32)
    out, _ = oracle.walk_tree(t, eps=eps, mac_kind=0, mac_param=2.0 ** -9, aold=aold)
    p = t.pos_sorted.astype(np.float64)
    r = np.linalg.norm(p[:, :3], axis=1)
    a_r = (out[:, :3] * p[:, :3]).sum(1) / r
    R = 20.0
    MR = R ** 3 / (1 + R * R) ** 1.5
    mass = lambda x: x ** 3 / (1 + x * x) ** 1.5 / MR
    # Phi(r) = -M(<r)/r - int_r^R (dM/dr')/r' dr' ; dM/dr = 3 r^2 (1+r^2)^{-5/2}/MR ; integral closed form:
    # int 3 r (1+r^2)^{-5/2} dr = -(1+r^2)^{-3/2}
    phi = lambda x: -mass(x) / x - ((1 + x * x) ** -1.5 - (1 + R * R) ** -1.5) / MR
    edges = np.geomspace(0.2, 8.0, 13)
    for lo, hi in zip(edges[:-1], edges[1:]):
        sel = (r >= lo) & (r < hi)
        k = sel.sum()
        assert k > 300
        assert np.mean(a_r[sel]) == pytest.approx(np.mean(-mass(r[sel]) / r[sel] ** 2), rel=6.0 / np.sqrt(k))
        assert np.mean(out[sel, 3]) == pytest.approx(np.mean(phi(r[sel])), rel=0.02)


# ---- group splitting by the critical separation r_crit (reading R13) ---------------------------------------
def _pieces_numpy(pos_sorted, members, r_crit):
    """Independent restatement of R13 in numpy float32: halve the member list while its GEO ball is wider than r_crit."""
    p = pos_sorted[members, :3].astype(np.float32)
    c = np.float32(0.5) * (p.min(0) + p.max(0))
    d = p - c
    b = np.sqrt(np.max(np.float32(d[:, 2] * d[:, 2]) + (np.float32(d[:, 1] * d[:, 1]) + np.float32(d[:, 0] * d[:, 0]))))
    if len(members) > 1 and b > r_crit:
        mid = (len(members) + 1) // 2
        return _pieces_numpy(pos_sorted, members[:mid], r_crit) + _pieces_numpy(pos_sorted, members[mid:], r_crit)
    return [members]


@pytest.mark.parametrize("r_crit", [0.0, 0.05, 0.3, 1.0])
def test_rcrit_split_equals_walking_each_piece_as_its_own_active_set(oracle, r_crit):
    """A chunk walked with r_crit must give exactly what walking each piece of the R13 recursion separately gives
    (pieces found by an independent numpy restatement), and as many traversals as there are pieces."""
    n = 4000
    pos = W.hernquist(n, seed=8)
    t = oracle.build_tree(pos)
    eps = 0.01
    active = W.random_active_subset(n, 0.6, seed=2)
    kw = dict(eps=eps, mac_kind=1, mac_param=0.7)
    out, c = oracle.walk_tree(t, active=active, r_crit=r_crit, **kw)
    n_pieces, inter = 0, 0
    ref = np.zeros_like(out)
    for g in range((n + 31) // 32):
        members = active[(active >= 32 * g) & (active < 32 * g + 32)]
        if members.size == 0:
            continue
        for piece in _pieces_numpy(t.pos_sorted, members, np.float32(r_crit)):
            o, cc = oracle.walk_tree(t, active=piece, group_range=(g, g + 1), **kw)
            ref[piece] = o[piece]
            n_pieces += 1
            inter += cc["interactions"]
            ball = oracle.group_ball(t.pos_sorted, piece)
            assert piece.size == 1 or ball[3] <= r_crit
    assert c["groups"] == n_pieces and c["interactions"] == inter
    assert np.array_equal(out, ref)
    if r_crit == 0.0:
        assert c["groups"] == active.size     # every member on its own: b_I = 0


def test_rcrit_infinite_is_the_unsplit_walk_and_small_rcrit_shortens_lists(oracle):
    pos = W.nfw(6000, seed=3)
    t = oracle.build_tree(pos)
    eps = 2.0 ** -8
    boot, _ = oracle.walk_tree(t, eps=eps, mac_kind=1, mac_param=0.5)
    aold = np.linalg.norm(boot[:, :3], axis=1).astype(np.float32)
    kw = dict(eps=eps, mac_kind=0, mac_param=2.0 ** -9, aold=aold)
    a, ca = oracle.walk_tree(t, **kw)
    b, cb = oracle.walk_tree(t, r_crit=float("inf"), **kw)
    assert np.array_equal(a, b) and ca == cb
    s, cs = oracle.walk_tree(t, r_crit=0.25, **kw)
    assert cs["groups"] > ca["groups"] and cs["interactions"] < ca["interactions"]   # tighter balls => shorter lists
    direct = oracle.direct(t.pos_sorted, eps)
    err = lambda o: np.median(np.linalg.norm(o[:, :3] - direct[:, :3], axis=1) / np.linalg.norm(direct[:, :3], axis=1))
    # a tight ball accepts cells right at the eq. 5 threshold, a wide one opens more than it must: the error moves towards
    # (never far beyond) the per-particle criterion's Delta_acc-sized error
    assert err(a) <= err(s) < 2.0 * 2.0 ** -9


def test_rcrit_zero_is_the_textbook_per_particle_tree_walk(oracle):
    """r_crit = 0: every particle walks alone with b_I = 0, i.e. the classic Barnes-Hut walk with the point MAC of eq. 5
    (d = |r_J - r_i|).  Pure-Python recursive restatement on a tiny case, fp32 MAC arithmetic, double sums."""
    n = 400
    pos = W.plummer(n, seed=12)
    t = oracle.build_tree(pos, n_leaf=4)
    eps, dacc = 0.02, 2.0 ** -6
    boot = oracle.direct(t.pos_sorted, eps)
    aold = np.linalg.norm(boot[:, :3], axis=1).astype(np.float32)
    out, c = oracle.walk_tree(t, eps=eps, mac_kind=0, mac_param=dacc, aold=aold, r_crit=0.0)
    f32, P = np.float32, t.pos_sorted
    eps2 = float(f32(eps)) ** 2
    ref = np.zeros((n, 4))
    n_int = 0
    for i in range(n):
        thr = f32(dacc) * aold[i]
        stack = [0]
        while stack:
            J = stack.pop()
            d3 = (t.com[J, :3] - P[i, :3]).astype(f32)
            r2 = f32(np.float64(d3[2]) ** 2 + f32(np.float64(d3[1]) ** 2 + f32(d3[0] * d3[0])))   # fmaf = one rounding of the exact product-sum
            d = f32(np.sqrt(r2))
            mb2 = f32(f32(t.com[J, 3] * t.b[J]) * t.b[J])
            if d > 0 and f32(thr * f32(f32(d * d) * f32(d * d))) >= mb2:
                src = [(t.com[J].astype(np.float64))]
            elif t.child[J] == 0xFFFFFFFF:
                src = [P[s].astype(np.float64) for s in range(t.head[J], t.head[J] + t.num[J]) if s != i]
                n_int += 1 if t.head[J] <= i < t.head[J] + t.num[J] else 0   # the walk counts the self entry (P:331 convention)
            else:
                stack.extend(range(t.child[J], t.child[J] + t.nchild[J]))
                continue
            for q in src:
                dx = q[:3] - P[i, :3].astype(np.float64)
                u = 1.0 / np.sqrt(dx @ dx + eps2)
                ref[i, :3] += q[3] * u ** 3 * dx
                ref[i, 3] -= q[3] * u
                n_int += 1
    assert c["groups"] == n and c["interactions"] == n_int
    assert np.allclose(out, ref, rtol=1e-11, atol=1e-13)


# ---- pins for the group's a_min (reading R4) and for the opening-angle criterion (eq. 2) -------------------
def _fma32(a, b, c):
    """fmaf on float32 values: the product of two float32 is exact in double; one rounding to float32 of the sum."""
    return np.float32(np.float64(a) * np.float64(b) + np.float64(c))


def _python_group_walk(t, members, ball, thr, accept_fn, eps):
    """O7 for one piece, written out: pending stack from the root, eq. 6-7 distance to the ball surface in fp32, the caller's
    acceptance test, monopole sums in double.  Returns (accepted cells, particle entries, out[k,4], MAC tests)."""
    f32, P = np.float32, t.pos_sorted
    eps2 = float(f32(eps)) ** 2
    cells, parts, tests = [], [], 0
    stack = [0]
    while stack:
        J = stack.pop()
        tests += 1
        d3 = (t.com[J, :3] - ball[:3]).astype(f32)
        r2 = _fma32(d3[2], d3[2], _fma32(d3[1], d3[1], f32(d3[0] * d3[0])))
        d = max(f32(f32(np.sqrt(r2)) - ball[3]), f32(0.0))          # eq. 6-7: distance to the nearest point of the ball
        if d > 0 and accept_fn(J, d):
            cells.append(J)
        elif t.child[J] == 0xFFFFFFFF:
            parts.extend(range(t.head[J], t.head[J] + t.num[J]))
        else:
            stack.extend(range(t.child[J], t.child[J] + t.nchild[J]))
    out = np.zeros((len(members), 4))
    for q, i in enumerate(members):
        src = [t.com[J].astype(np.float64) for J in cells] + [P[s].astype(np.float64) for s in parts if s != i]
        for e in src:
            dx = e[:3] - P[i, :3].astype(np.float64)
            u = 1.0 / np.sqrt(dx @ dx + eps2)
            out[q, :3] += e[3] * u ** 3 * dx
            out[q, 3] -= e[3] * u
    return cells, parts, out, tests


@pytest.mark.parametrize("G", [8, 32])
def test_group_amin_is_the_minimum_over_members(oracle, G):
    """Reading R4 + P:118 ("conservative"): a group tests eq. 5 with Delta_acc * min_k |a_old,k| and the distance from the ball
    surface, so that a cell accepted for the group is accepted by eq. 5 for EVERY member with that member's own
    |a_old| and own distance.  |a_old| is spread over four decades inside every group, so a max, a mean or 'first member'
    reading changes the lists.  Value pin: a pure-Python group walk with thr = Delta * min(aold[K]) reproduces the oracle's
    counts and sums; property pin: group acceptance => per-particle acceptance, evaluated in double."""
    n = 400
    pos = W.plummer(n, seed=21)
    t = oracle.build_tree(pos, n_leaf=4)
    eps, dacc = 0.02, 2.0 ** -5
    rng = np.random.default_rng(5)
    aold = (10.0 ** rng.uniform(-2.0, 2.0, n)).astype(np.float32)          # four decades, uncorrelated with position
    out, c = oracle.walk_tree(t, eps=eps, mac_kind=0, mac_param=dacc, aold=aold, group_size=G)
    f32 = np.float32
    n_int = n_tests = n_list = n_checked = 0
    p64 = t.pos_sorted.astype(np.float64)
    for g in range((n + G - 1) // G):
        K = np.arange(g * G, min(n, (g + 1) * G), dtype=np.uint32)
        ball = oracle.group_ball(t.pos_sorted, K)
        thr = f32(f32(dacc) * aold[K].min())
        mb2 = lambda J: f32(f32(t.com[J, 3] * t.b[J]) * t.b[J])
        cells, parts, ref, tests = _python_group_walk(
            t, K, ball, thr, lambda J, d: f32(thr * f32(f32(d * d) * f32(d * d))) >= mb2(J), eps)
        assert np.allclose(out[K], ref, rtol=1e-11, atol=1e-13)
        n_int += len(K) * (len(cells) + len(parts)); n_tests += tests; n_list += len(cells) + len(parts)
        for J in cells:                 # eq. 5 per member: Delta |a_i| d_i^4 >= m_J b_J^2, all in double
            di = np.linalg.norm(p64[K, :3] - t.com[J, :3].astype(np.float64), axis=1)
            lhs = dacc * aold[K].astype(np.float64) * di ** 4
            assert np.all(lhs >= float(t.com[J, 3]) * float(t.b[J]) ** 2 * (1 - 1e-5))
            n_checked += 1
    assert c["interactions"] == n_int and c["mac_tests"] == n_tests and c["list_entries"] == n_list
    assert n_checked > 10 * (n // G)        # the pin is not vacuous: cells are accepted


def test_opening_angle_is_b_over_d(oracle):
    """eq. 2: a cell is accepted when b_J / d <= theta, b_J the RADIUS of the cell's sphere and d the distance
    to it.  r_crit = 0 makes every particle its own group (b_I = 0, d = |r_J - r_i|): the textbook per-particle walk, the
    criterion written literally in double.  Counts and sums must equal the oracle's (a diameter-for-radius slip, or d^2 for
    d, changes the lists)."""
    n = 400
    pos = W.hernquist(n, seed=14)
    t = oracle.build_tree(pos, n_leaf=4)
    eps, theta = 0.02, 0.6
    out, c = oracle.walk_tree(t, eps=eps, mac_kind=1, mac_param=theta, r_crit=0.0)
    n_int = n_tests = n_cells = 0
    theta32 = float(np.float32(theta))
    for i in range(n):
        K = np.array([i], np.uint32)
        ball = np.append(t.pos_sorted[i, :3], np.float32(0.0)).astype(np.float32)
        cells, parts, ref, tests = _python_group_walk(t, K, ball, None, lambda J, d: float(t.b[J]) / float(d) <= theta32, eps)
        assert np.allclose(out[i], ref[0], rtol=1e-11, atol=1e-13)
        n_int += len(cells) + len(parts); n_tests += tests; n_cells += len(cells)
    assert c["groups"] == n and c["interactions"] == n_int and c["mac_tests"] == n_tests
    assert n_cells > 20 * n         # cells are accepted: the criterion is exercised
