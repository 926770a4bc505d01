"""Pins for the oracle's sort (O3), canonical tree (O4) and pseudo-j moments (O5)."""
import numpy as np
import pytest

from paper_1610_07279_b200 import workloads as W


def test_sort_is_stable_permutation(oracle):
    rng = np.random.default_rng(0)
    key = rng.integers(0, 50, size=4000).astype(np.uint64)  # many ties
    ks, perm = oracle.sort(key)
    assert sorted(perm.tolist()) == list(range(4000))
    assert np.all(ks[1:] >= ks[:-1]) and np.all(ks == key[perm])
    ties = ks[1:] == ks[:-1]
    assert np.all(perm[1:][ties] > perm[:-1][ties])
    assert np.array_equal(perm, np.argsort(key, kind="stable"))


def _recursive_tree(keys, n_leaf):
    """Independent top-down reference: recursive descent grouping by octal digit, then BFS numbering."""
    n = len(keys)
    root = dict(head=0, num=n, level=0, kids=[])

    def split(nd):
        if nd["num"] <= n_leaf or nd["level"] >= 21:
            return
        sh = 3 * (21 - nd["level"] - 1)
        buckets = {}
        for s in range(nd["head"], nd["head"] + nd["num"]):
            buckets.setdefault((int(keys[s]) >> sh) & 7, []).append(s)
        for d in sorted(buckets):
            rng_ = buckets[d]
            assert rng_ == list(range(rng_[0], rng_[-1] + 1))
            kid = dict(head=rng_[0], num=len(rng_), level=nd["level"] + 1, kids=[])
            nd["kids"].append(kid)
            split(kid)

    split(root)
    order, frontier = [], [root]
    while frontier:
        order += frontier
        frontier = [k for nd in frontier for k in nd["kids"]]
    ids = {id(nd): i for i, nd in enumerate(order)}
    head = [nd["head"] for nd in order]
    num = [nd["num"] for nd in order]
    level = [nd["level"] for nd in order]
    child = [ids[id(nd["kids"][0])] if nd["kids"] else 0xFFFFFFFF for nd in order]
    nchild = [len(nd["kids"]) for nd in order]
    return head, num, level, child, nchild


@pytest.mark.parametrize("n,n_leaf,kind", [(1, 16, 0), (7, 16, 0), (300, 4, 0), (2500, 16, 0), (2500, 8, 1), (1000, 1, 0)])
def test_tree_matches_recursive_reference(oracle, n, n_leaf, kind):
    pos = W.plummer(n, seed=n + n_leaf)
    if n >= 300:
        pos[10:40, :3] = pos[5, :3]  # > n_leaf coincident particles: a level-21 leaf and a single-child chain
    t = oracle.build_tree(pos, key_kind=kind, n_leaf=n_leaf)
    head, num, level, child, nchild = _recursive_tree(t.key, n_leaf)
    assert t.n_nodes == len(head)
    assert t.head.tolist() == head and t.num.tolist() == num and t.level.tolist() == level
    assert t.child.tolist() == child and t.nchild.tolist() == nchild
    for L in range(22):
        assert t.level_ofs[L] == int(np.searchsorted(t.level, L))


def test_tree_invariants(oracle):
    pos = W.hernquist(20000, seed=2)
    t = oracle.build_tree(pos, n_leaf=16)
    leaf = t.child == 0xFFFFFFFF
    assert np.all((t.num[leaf] <= 16) | (t.level[leaf] == 21))
    assert int(t.num[leaf].sum()) == t.n  # leaves tile the particles
    assert np.all(np.diff(t.level.astype(int)) >= 0)  # breadth-first ids
    for J in np.nonzero(~leaf)[0][:2000]:
        c0, nc = int(t.child[J]), int(t.nchild[J])
        assert 1 <= nc <= 8
        assert t.head[c0] == t.head[J] and int(t.num[c0:c0 + nc].sum()) == int(t.num[J])
        assert np.all(t.head[c0 + 1:c0 + nc] == t.head[c0:c0 + nc - 1] + t.num[c0:c0 + nc - 1])
        assert np.all(t.level[c0:c0 + nc] == t.level[J] + 1)
    # every key of a node shares the node's 3*level-bit prefix, and neighbours outside do not
    for J in range(0, t.n_nodes, 37):
        h, c, L = int(t.head[J]), int(t.num[J]), int(t.level[J])
        sh = np.uint64(63 - 3 * L)
        pre = t.key[h:h + c] >> sh if L else np.zeros(c, np.uint64)
        assert np.all(pre == pre[0])
        if L and h > 0:
            assert (t.key[h - 1] >> sh) != pre[0]
        if L and h + c < t.n:
            assert (t.key[h + c] >> sh) != pre[0]


def test_moments_match_definitions(oracle):
    """m_J total mass, r_J centre of mass, b_J radius about r_J containing all the cell's particles."""
    rng = np.random.default_rng(4)
    pos = W.plummer(3000, seed=9)
    pos[:, 3] = rng.uniform(0.5, 1.5, 3000).astype(np.float32) / 3000  # unequal masses: catches a dropped weight
    t = oracle.build_tree(pos, n_leaf=8)
    p = t.pos_sorted.astype(np.float64)
    assert abs(t.com[0, 3] - p[:, 3].sum()) < 1e-6 * p[:, 3].sum()
    assert np.allclose(t.com[0, :3], (p[:, :3] * p[:, 3:4]).sum(0) / p[:, 3].sum(), rtol=0, atol=1e-6)
    for J in range(0, t.n_nodes, 5):
        h, c = int(t.head[J]), int(t.num[J])
        q = p[h:h + c]
        m = q[:, 3].sum()
        com = (q[:, :3] * q[:, 3:4]).sum(0) / m
        assert abs(t.com[J, 3] - m) <= 2e-7 * m
        assert np.all(np.abs(t.com[J, :3] - com) <= 1.2e-7 * np.maximum(1e-3, np.abs(com)))
        dist = np.linalg.norm(q[:, :3] - t.com[J, :3].astype(np.float64), axis=1)
        assert np.all(dist <= t.b[J] * (1 + 1e-6) + 1e-30)          # containment
        assert abs(dist.max() - t.b[J]) <= 1e-6 * max(dist.max(), 1e-30)  # attained
        if c == 1:
            assert np.array_equal(t.com[J], t.pos_sorted[h]) and t.b[J] == 0.0
