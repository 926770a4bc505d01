"""Pins for the oracle's space-filling-curve keys (App. A) and root box (R1).
None of these re-types the oracle's formula: they are curve invariants, a hand-evaluated table and a
naive bit interleave."""
import itertools
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_level1_digits_match_paper_formula(oracle):
    rows = [tuple(int(v) for v in ln.split()) for ln in open(os.path.join(GOLD, "ph_level1_order.txt"))
            if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 8
    for x, y, z, d in rows:
        assert oracle.encode_peano3d(1, x, y, z) == d


@pytest.mark.parametrize("nlev", [1, 2, 3, 4])
def test_peano_is_bijective_and_one_stroke(oracle, nlev):
    """the PH curve is a 'one-stroke sketch': consecutive keys are face-adjacent cells."""
    m = 1 << nlev
    cells = {}
    for x, y, z in itertools.product(range(m), repeat=3):
        k = oracle.encode_peano3d(nlev, x, y, z)
        assert k not in cells
        cells[k] = (x, y, z)
    assert sorted(cells) == list(range(m ** 3))
    for k in range(m ** 3 - 1):
        a, b = cells[k], cells[k + 1]
        assert sum(abs(p - q) for p, q in zip(a, b)) == 1


@pytest.mark.parametrize("nlev", [2, 3, 4, 5])
def test_peano_prefix_hierarchy(oracle, nlev):
    """dividing a cube into eight sub-cubes = dividing the key into eight equal parts, i.e. the
    key of the parent cell is the key with its last octal digit dropped."""
    rng = np.random.default_rng(nlev)
    for x, y, z in rng.integers(0, 1 << nlev, size=(300, 3)):
        assert oracle.encode_peano3d(nlev, int(x), int(y), int(z)) >> 3 == \
            oracle.encode_peano3d(nlev - 1, int(x) >> 1, int(y) >> 1, int(z) >> 1)


def test_peano_decoder_inverts_encoder(oracle):
    """Listing 2 is the decoder of Listing 1."""
    rng = np.random.default_rng(3)
    for x, y, z in rng.integers(0, 1 << 21, size=(2000, 3)):
        k = oracle.encode_peano3d(21, int(x), int(y), int(z))
        assert k < (1 << 63)
        assert oracle.decode_peano3d(21, k) == (int(x), int(y), int(z))
    for nlev in (1, 2, 3):
        for k in range(8 ** nlev):
            x, y, z = oracle.decode_peano3d(nlev, k)
            assert oracle.encode_peano3d(nlev, x, y, z) == k


def test_peano_extremes(oracle):
    # the curve starts in the corner cell (0,0,0); by the hierarchy + level-1 table it ends at (max,0,0)
    assert oracle.encode_peano3d(21, 0, 0, 0) == 0
    assert oracle.encode_peano3d(21, (1 << 21) - 1, 0, 0) == (1 << 63) - 1


def _naive_interleave(x, y, z):
    k = 0
    for b in range(21):
        k |= ((x >> b) & 1) << (3 * b + 2) | ((y >> b) & 1) << (3 * b + 1) | ((z >> b) & 1) << (3 * b)
    return k


def test_morton_is_plain_bit_interleave(oracle):
    """Listing 3 extends the Raman & Wise dilation to 63 bits = textbook interleave."""
    rng = np.random.default_rng(5)
    pts = rng.integers(0, 1 << 21, size=(5000, 3)).tolist() + [[0, 0, 0], [(1 << 21) - 1] * 3, [1, 0, 0], [0, 1, 0], [0, 0, 1]]
    for x, y, z in pts:
        assert oracle.morton3d(x, y, z) == _naive_interleave(x, y, z)


def test_root_box_and_key_quantisation(oracle):
    """R1: anchor at minima, power-of-two side strictly greater than the extent, 21 bits, clamp."""
    rng = np.random.default_rng(11)
    pos = np.zeros((1000, 4), np.float32)
    pos[:, :3] = rng.normal(size=(1000, 3)) * 3
    pos[:, 3] = 1e-3
    box = oracle.root_box(pos)
    assert np.all(box[:3] == pos[:, :3].min(axis=0))
    ext = (pos[:, :3].max(axis=0) - pos[:, :3].min(axis=0)).max()
    side = float(box[3])
    assert side > ext >= side / 2 and np.log2(side) == int(np.log2(side))
    for kind, enc in ((0, lambda a, b, c: oracle.encode_peano3d(21, a, b, c)), (1, oracle.morton3d)):
        k = oracle.keys(pos, box, kind)
        g = np.floor((pos[:, :3].astype(np.float64) - box[:3].astype(np.float64)) * (2.0 ** 21 / side)).astype(np.int64)
        # float64 floor can differ from the fp32 subtract only where the fp32 difference rounds across a cell
        # boundary; recompute exactly as specified for those (fp32 subtract, exact scale)
        g32 = np.floor((pos[:, :3] - box[:3]) * np.float32(2.0 ** 21 / side)).astype(np.int64)
        g32 = np.clip(g32, 0, (1 << 21) - 1)
        assert np.abs(g - g32).max() <= 1 and np.mean(np.all(g == g32, axis=1)) > 0.85
        for i in range(0, 1000, 7):
            assert int(k[i]) == enc(int(g32[i, 0]), int(g32[i, 1]), int(g32[i, 2]))
    # degenerate: all particles at one point -> side 1, all keys 0
    one = np.tile(np.array([[1.5, -2.0, 3.0, 1.0]], np.float32), (5, 1))
    b1 = oracle.root_box(one)
    assert b1[3] == 1.0 and np.all(oracle.keys(one, b1, 0) == 0)
