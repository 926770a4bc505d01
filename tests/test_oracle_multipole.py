"""Pins for the oracle's multipole MAC (NEXT row f3; eq. 3-4): B_2 against the parallel-axis theorem and
its bounds, the fp32 square-root-free form of eq. 3 (R16) against eq. 3 written literally in double on a
pure-Python per-particle Barnes-Hut walk, and the error falling with Delta_mul against the double direct sum."""
import numpy as np

import oracle
from paper_1610_07279_b200 import workloads as W


def test_b2_definition_parallel_axis_and_bounds():
    pos = W.hernquist(6000, seed=2)
    t = oracle.build_tree(pos, n_leaf=8)
    B2 = oracle.b2(t.pos_sorted, t.head, t.num, t.com)
    m, com, P = t.com[:, 3].astype(np.float64), t.com[:, :3].astype(np.float64), t.pos_sorted.astype(np.float64)
    one = t.num == 1
    assert np.all(B2[one] == 0)                                              # a single particle is its own centre
    assert np.all(B2 <= m * t.b.astype(np.float64) ** 2 * (1 + 1e-5) + 1e-12)  # every |r_j - r_J| <= b_J
    # parallel-axis theorem: B2_J = sum over children (B2_c + m_c |r_c - r_J|^2), up to the fp32 rounding of the stored centres
    internal = np.nonzero(t.child != 0xFFFFFFFF)[0]
    for J in internal[:: max(1, internal.size // 300)]:
        cs = np.arange(t.child[J], t.child[J] + t.nchild[J])
        rhs = (B2[cs].astype(np.float64) + m[cs] * ((com[cs] - com[J]) ** 2).sum(1)).sum()
        assert abs(B2[J] - rhs) <= 2e-4 * rhs + 1e-12
    # root against numpy
    d2 = ((P[:, :3] - com[0]) ** 2).sum(1)
    assert np.isclose(B2[0], (P[:, 3] * d2).sum(), rtol=1e-6)


def test_multipole_mac_is_eq3_on_a_textbook_walk():
    """r_crit = 0: every particle walks alone (b_I = 0, d = |r_J - r_i|).  The reference decides with eq. 3 LITERALLY, in
    double; no decision of this case lies within 1e-5 of the threshold, so the fp32 rearrangement must agree everywhere."""
    n = 400
    pos = W.plummer(n, seed=12)
    t = oracle.build_tree(pos, n_leaf=4)
    eps, dmul = 0.02, 2.0 ** -4
    B2 = oracle.b2(t.pos_sorted, t.head, t.num, t.com)
    out, c = oracle.walk_tree(t, eps=eps, mac_kind=2, mac_param=dmul, r_crit=0.0, B2=B2)
    P = t.pos_sorted
    eps2 = float(np.float32(eps)) ** 2
    ref = np.zeros((n, 4))
    n_int = near = 0
    for i in range(n):
        stack = [0]
        while stack:
            J = stack.pop()
            d3 = (t.com[J, :3] - P[i, :3]).astype(np.float32).astype(np.float64)
            d = np.sqrt(d3 @ d3)
            b = float(t.b[J])
            rhs = 0.5 * b + np.sqrt(0.25 * b * b + np.sqrt(3.0 * float(B2[J]) / dmul))      # eq. 3
            near += abs(d - rhs) <= 1e-5 * rhs and d > 0
            if d > 0 and d >= rhs:
                src = [t.com[J].astype(np.float64)]
            elif t.child[J] == 0xFFFFFFFF:
                src = [P[s].astype(np.float64) for s in range(t.head[J], t.head[J] + t.num[J]) if s != i]
                n_int += 1 if t.head[J] <= i < t.head[J] + t.num[J] else 0
            else:
                stack.extend(range(t.child[J], t.child[J] + t.nchild[J]))
                continue
            for q in src:
                dx = q[:3] - P[i, :3].astype(np.float64)
                u = 1.0 / np.sqrt(dx @ dx + eps2)
                ref[i, :3] += q[3] * u ** 3 * dx
                ref[i, 3] -= q[3] * u
                n_int += 1
    assert near == 0
    assert c["groups"] == n and c["interactions"] == n_int
    assert np.allclose(out, ref, rtol=1e-11, atol=1e-13)


def test_multipole_error_shrinks_with_delta_mul_and_zero_is_direct():
    n = 3000
    pos = W.plummer(n, seed=4)
    t = oracle.build_tree(pos)
    eps = 1.0 / 64
    direct = oracle.direct(t.pos_sorted, eps)
    med, inter = [], []
    for e in (-2, 2, 6, 10, 14):
        out, c = oracle.walk_tree(t, eps=eps, mac_kind=2, mac_param=2.0 ** -e)
        err = np.linalg.norm(out[:, :3] - direct[:, :3], axis=1) / np.linalg.norm(direct[:, :3], axis=1)
        med.append(np.median(err))
        inter.append(c["interactions"])
    assert all(b < a for a, b in zip(med, med[1:])) and all(b > a for a, b in zip(inter, inter[1:])), (med, inter)
    assert med[0] > 1e-3 and med[-1] < 2e-4
    out, c = oracle.walk_tree(t, eps=eps, mac_kind=2, mac_param=0.0)         # Delta = 0: nothing with extent is accepted
    assert np.allclose(out, direct, rtol=1e-9, atol=1e-12)
