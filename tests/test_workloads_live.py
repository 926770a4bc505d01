"""Input recipes of the live block-stepping workloads (paper_1610_07279_b200/workloads.py): seeded, finite, near virial equilibrium.  No GPU."""
import numpy as np
import pytest

from paper_1610_07279_b200 import workloads as W


def _virial_ratio(pos, vel):
    """2K / |W| with W from the spherically averaged enclosed mass (G = 1)."""
    r = np.linalg.norm(pos[:, :3].astype(np.float64), axis=1)
    m = pos[:, 3].astype(np.float64)
    k = 0.5 * (m * (vel[:, :3].astype(np.float64) ** 2).sum(axis=1)).sum()
    o = np.argsort(r)
    return 2.0 * k / (m[o] * np.cumsum(m[o]) / r[o]).sum()


@pytest.mark.parametrize("name", sorted(W.LIVE_CONFIGS))
def test_live_configs_are_seeded_and_near_equilibrium(name):
    pos, vel, cfg = W.make_live_config(name, seed=5, n=1 << 16)
    pos2, vel2, _ = W.make_live_config(name, seed=5, n=1 << 16)
    assert np.array_equal(pos, pos2) and np.array_equal(vel, vel2)
    assert pos.shape == vel.shape == (1 << 16, 4) and pos.dtype == vel.dtype == np.float32
    assert np.isfinite(vel).all() and np.all(vel[:, 3] == 0)
    assert 0.8 < _virial_ratio(pos, vel) < 1.2


def test_m31_positions_do_not_depend_on_asking_for_components():
    """m31_like(components=True) returns the same particles as the BASELINE.json configs[3] generator plus their component; the disk
    (11 % by count) rotates about z in m31_velocities' stand-in, halo and bulge do not."""
    pos = W.m31_like(50000, seed=2)
    pos_c, comp = W.m31_like(50000, seed=2, components=True)
    assert np.array_equal(pos, pos_c)
    assert np.bincount(comp).tolist() == [40500, 4000, 5500]
    vel = W.m31_velocities(pos, comp, seed=3)
    lz = pos[:, 0].astype(np.float64) * vel[:, 1] - pos[:, 1].astype(np.float64) * vel[:, 0]
    disk = comp == 2
    assert np.mean(lz[disk] > 0) > 0.99 and abs(np.mean(np.sign(lz[~disk]))) < 0.05
    assert np.abs(pos[disk, 2]).mean() < 0.2 * np.abs(pos[~disk, 2]).mean()
