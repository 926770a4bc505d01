"""-m gpu parity: tree build (B1-B6) through the C ABI vs the CPU oracle.  Keys, permutation and node arrays are
bit-exact; moments within a tolerance derived from fp32 accumulation."""
import numpy as np
import pytest

from paper_1610_07279_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _check_build(oracle, pos, key_kind, n_leaf):
    from gpu_util import gpu_build
    g, v = gpu_build(pos, key_kind=key_kind, n_leaf=n_leaf)
    t = oracle.build_tree(pos, key_kind=key_kind, n_leaf=n_leaf)
    assert np.array_equal(np.array(v["box"], np.float32), t.box)
    assert np.array_equal(v["key"], t.key)
    assert np.array_equal(v["perm"], t.perm)
    assert np.array_equal(v["pos_m_sorted"], t.pos_sorted)
    assert v["n_nodes"] == t.n_nodes
    assert np.array_equal(v["node_head"], t.head) and np.array_equal(v["node_num"], t.num)
    assert np.array_equal(v["node_child"], t.child) and np.array_equal(v["node_nchild"], t.nchild)
    assert np.array_equal(v["node_level"], t.level)
    assert np.array_equal(v["level_ofs"], t.level_ofs)
    assert v["n_levels_tree"] == t.n_levels
    # moments: mass and centre vs the oracle's double sums; fp32 tree summation => a few ulp of the coordinate scale
    # (sequential fp32 sum of <= n_leaf particles per leaf, then <= 8 children per level: error grows with n_leaf)
    scale = np.abs(t.pos_sorted[:, :3]).max()
    tol = 2e-7 * (2 + n_leaf / 8)
    assert np.all(np.abs(v["node_com"][:, 3] - t.com[:, 3]) <= tol * t.com[:, 3])
    assert np.abs(v["node_com"][:, :3] - t.com[:, :3]).max() <= tol * scale
    one = t.num == 1
    assert np.array_equal(v["node_com"][one], t.com[one]) and np.all(v["node_b"][one] == 0)
    # radius: exactly the definition, applied to the centre the CUDA build stored
    b_def = oracle.radius(t.pos_sorted, t.head, t.num, v["node_com"])
    assert np.all(np.abs(v["node_b"] - b_def) <= 1e-6 * b_def + 1e-7 * scale * 1e-3)
    # and close to the oracle's own radius (centres differ by rounding)
    assert np.all(np.abs(v["node_b"] - t.b) <= 1e-6 * t.b + 2 * tol * scale)
    g.close()
    return v, t


@pytest.mark.parametrize("model,n,n_leaf,kind", [
    ("plummer", 1 << 13, 16, 0), ("plummer", 1 << 13, 16, 1), ("hernquist", 100003, 16, 0),
    ("nfw", 50000, 8, 0), ("m31_like", 70001, 32, 0), ("plummer", 3000, 1, 0), ("hernquist", 5000, 64, 1),
])
def test_build_matches_oracle(oracle, model, n, n_leaf, kind):
    pos = getattr(W, model)(n, seed=3)
    _check_build(oracle, pos, kind, n_leaf)


@pytest.mark.parametrize("n", [1, 2, 17, 31, 32, 33, 255, 256, 257])
def test_build_tiny_and_ragged(oracle, n):
    _check_build(oracle, W.plummer(n, seed=n), 0, 16)
    _check_build(oracle, W.plummer(n, seed=n), 0, 4)


@pytest.mark.parametrize("n_clump,spread,kind", [(40, 1e-4, 0), (600, 3e-4, 0), (1500, 3e-4, 1), (5000, 2e-4, 0), (20000, 1e-5, 0)])
def test_sort_runs_of_equal_upper_bits(oracle, n_clump, spread, kind):
    """B3's five-pass sort leaves the low 23 key bits to fix-up kernels (sort_pairs.cu): a tight clump of DISTINCT particles inside one
    cell of 2^-13 of a wide root cube gives runs of equal upper bits that are short (insertion sort), medium (rank sort in shared
    memory) or too long for either (the build then repeats itself with all eight passes): perm must be the oracle's in every case."""
    rng = np.random.default_rng(n_clump)
    n_far = 3000
    pos = np.zeros((n_far + 3 * n_clump, 4), np.float32)
    pos[:n_far, :3] = rng.uniform(-16.0, 16.0, (n_far, 3))
    for c, ctr in enumerate(((0.123, 0.456, -0.789), (5.0, -3.0, 2.0), (-7.77, 7.77, 0.01))):
        sl = slice(n_far + c * n_clump, n_far + (c + 1) * n_clump)
        pos[sl, :3] = np.asarray(ctr, np.float32) + rng.uniform(-spread, spread, (n_clump, 3)).astype(np.float32)
    pos[:, 3] = 1.0 / pos.shape[0]
    pos = pos[rng.permutation(pos.shape[0])]
    from gpu_util import gpu_build
    g, v = gpu_build(pos, key_kind=kind)
    t = oracle.build_tree(pos, key_kind=kind)
    assert np.array_equal(v["key"], t.key) and np.array_equal(v["perm"], t.perm) and np.array_equal(v["pos_m_sorted"], t.pos_sorted)
    assert v["n_nodes"] == t.n_nodes and np.array_equal(v["node_head"], t.head) and np.array_equal(v["node_num"], t.num)
    assert np.array_equal(v["node_child"], t.child) and np.array_equal(v["node_level"], t.level)
    g.close()
    top = t.key >> np.uint64(23)
    runs = np.diff(np.flatnonzero(np.concatenate([[True], top[1:] != top[:-1], [True]])))
    assert runs.max() >= min(n_clump // 8, 33) or n_clump < 100       # the case really has long runs of equal upper bits


def test_sort_long_ordered_run_of_coincident_particles(oracle):
    """A run of equal upper key bits far longer than the fix-up kernels take, but already in order (50 000 coincident particles: equal keys,
    ascending original index), next to a too-long run of distinct particles in a second build: the run head stops measuring at the limit and
    the ordered / unordered decision is taken in parallel by the entries of the run; perm is the oracle's in both."""
    rng = np.random.default_rng(77)
    n_far, n_same = 3000, 50000
    pos = np.zeros((n_far + n_same + 600, 4), np.float32)
    pos[:n_far, :3] = rng.uniform(-16.0, 16.0, (n_far, 3))
    pos[n_far:n_far + n_same, :3] = np.asarray((1.25, -2.5, 0.375), np.float32)
    pos[n_far + n_same:, :3] = np.asarray((5.0, -3.0, 2.0), np.float32) + rng.uniform(-3e-4, 3e-4, (600, 3)).astype(np.float32)
    pos[:, 3] = 1.0 / pos.shape[0]
    order = rng.permutation(pos.shape[0])
    from gpu_util import gpu_build

    def check(p, kind):       # index work only (one leaf of 50 000 particles is outside the moment tolerances of _check_build)
        g, v = gpu_build(p, key_kind=kind)
        t = oracle.build_tree(p, key_kind=kind)
        assert np.array_equal(v["key"], t.key) and np.array_equal(v["perm"], t.perm) and np.array_equal(v["pos_m_sorted"], t.pos_sorted)
        assert v["n_nodes"] == t.n_nodes and np.array_equal(v["node_head"], t.head) and np.array_equal(v["node_num"], t.num)
        assert np.array_equal(v["node_child"], t.child) and np.array_equal(v["node_level"], t.level)
        g.close()
        top = t.key >> np.uint64(23)
        return np.diff(np.flatnonzero(np.concatenate([[True], top[1:] != top[:-1], [True]]))).max()

    assert check(pos[order], 0) >= n_same
    pos[n_far:n_far + n_same, :3] += rng.uniform(-1e-5, 1e-5, (n_same, 3)).astype(np.float32)      # now distinct: the eight-pass repeat
    assert check(pos[order], 1) > 2048


def test_build_degenerate_inputs(oracle):
    # all particles at one point: root cube side 1, one level-21 leaf chain
    pos = np.tile(np.array([[0.25, -1.0, 3.0, 0.01]], np.float32), (100, 1))
    _check_build(oracle, pos, 0, 16)
    # clusters of coincident particles inside a normal distribution: level-21 leaves with num > n_leaf, single-child chains
    pos = W.plummer(5000, seed=4)
    pos[100:160, :3] = pos[7, :3]
    pos[900:920, :3] = pos[901, :3]
    _check_build(oracle, pos, 0, 16)
    _check_build(oracle, pos, 1, 8)
    # unequal masses
    pos = W.hernquist(20000, seed=6)
    pos[:, 3] *= np.random.default_rng(0).uniform(0.2, 3.0, 20000).astype(np.float32)
    _check_build(oracle, pos, 0, 16)


def test_build_full_size_hernquist(oracle):
    """BASELINE.json configs[1]: Hernquist N = 2^20, full-size bit-exact tree."""
    pos, cfg = W.make_config("hernquist_2p20", seed=1)
    v, t = _check_build(oracle, pos, 0, 16)
    assert 0.15 * t.n < t.n_nodes < 0.4 * t.n


def test_update_moments_with_moved_particles(oracle):
    import torch
    from gpu_util import gpu_build, dev, view_to_numpy
    pos = W.plummer(20000, seed=5)
    g, v = gpu_build(pos)
    rng = np.random.default_rng(1)
    moved = v["pos_m_sorted"].copy()
    moved[:, :3] += rng.normal(scale=1e-3, size=(20000, 3)).astype(np.float32)
    g.update_moments(dev(moved))
    v2 = view_to_numpy(g.get_tree_view())
    assert np.array_equal(v2["node_head"], v["node_head"]) and np.array_equal(v2["pos_m_sorted"], moved)
    com, b = oracle.moments(moved, v["node_head"], v["node_num"])
    scale = np.abs(moved[:, :3]).max()
    assert np.abs(v2["node_com"][:, :3] - com[:, :3]).max() <= 4e-7 * scale
    assert np.all(np.abs(v2["node_b"] - b) <= 1e-6 * b + 8e-7 * scale)
    g.close()


def test_errors(oracle):
    import torch
    from gpu_util import dev
    from paper_1610_07279_b200.binding import Gothic, GothicError
    pos = W.plummer(4096, seed=1)
    g = Gothic(4096, node_max=64)
    with pytest.raises(GothicError, match="capacity"):
        g.build_tree(dev(pos), n_leaf=4)
    acc = torch.zeros(4096, 4, device="cuda")
    with pytest.raises(GothicError, match="not built"):
        g.walk_tree(acc, eps=0.1, mac_kind=1, mac_param=0.5)
    g.close()
    g = Gothic(1000)
    with pytest.raises(GothicError, match="argument"):
        g.build_tree(dev(pos))  # n > n_max
    with pytest.raises(GothicError):
        Gothic(1000, group_size=5)
    g.close()
