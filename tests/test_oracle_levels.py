"""Pins for block time-step levels and active sets (O6; reading R6 from BASELINE.json configs[2])."""
import numpy as np

from paper_1610_07279_b200 import workloads as W


def test_levels_are_floor_log2_of_timestep(oracle):
    """dt = eta sqrt(eps/|a|) floored to a power of two: compare with float64 log2 away from boundaries."""
    rng = np.random.default_rng(0)
    n = 20000
    acc = np.zeros((n, 4), np.float32)
    acc[:, :3] = rng.normal(size=(n, 3)) * np.exp(rng.uniform(-6, 6, (n, 1)))
    eps, eta = 2.0 ** -8, 0.5
    lev, emin, nlev = oracle.levels(acc, eps, eta, max_levels=64)
    a = np.linalg.norm(acc[:, :3].astype(np.float64), axis=1)
    ex = np.log2(eta * np.sqrt(eps / a))
    safe = np.abs(ex - np.round(ex)) > 1e-5
    assert emin == int(np.floor(ex).min()) or not safe[np.argmin(ex)]
    assert np.all(lev[safe] == (np.floor(ex[safe]) - emin).astype(int))
    assert nlev == int(lev.max()) + 1
    # clamp: coarser-wanting particles are clamped down
    lev4, emin4, nlev4 = oracle.levels(acc, eps, eta, max_levels=4)
    assert emin4 == emin and nlev4 == 4 and np.all(lev4 == np.minimum(lev, 3))
    # |a| = 0 -> coarsest level
    acc[7, :3] = 0
    assert oracle.levels(acc, eps, eta, max_levels=8)[0][7] == 7


def test_active_sets_nest_and_cover_cycle(oracle):
    rng = np.random.default_rng(1)
    lev = rng.integers(0, 4, 5000).astype(np.uint8)
    nlev = 4
    times = np.zeros(5000, int)
    prev = None
    for s in range(1, 2 ** (nlev - 1) + 1):
        act = oracle.active_set(lev, s)
        assert np.all(np.diff(act.astype(np.int64)) > 0)
        ctz = (s & -s).bit_length() - 1
        assert np.array_equal(act, np.nonzero(lev <= ctz)[0])
        times[act] += 1
    assert np.all(times == 2 ** (nlev - 1 - lev.astype(int)))  # a level-l particle is active 2^(nlev-1-l) times
    assert oracle.active_set(lev, 2 ** (nlev - 1)).shape[0] == 5000  # last substep: everyone
    assert set(oracle.active_set(lev, 1)) <= set(oracle.active_set(lev, 2)) <= set(oracle.active_set(lev, 4))


def test_nfw_level_histogram_closed_form(oracle):
    """NFW (r_s = 1, R = 10, M = 1): |a|(r) = mu(r)/(mu_R r^2) is monotone decreasing, so the radius at
    which dt = 0.5 sqrt(eps/|a|) crosses a power of two gives the level mass fractions in closed form;
    eps = 2^-8 gives exponents -5..-2 => 4 levels (the paper's NFW runs had 4)."""
    n = 1 << 18
    pos = W.nfw(n, seed=1)
    p = pos.astype(np.float64)
    r = np.linalg.norm(p[:, :3], axis=1)
    mu = lambda x: np.log1p(x) - x / (1 + x)
    a_mag = mu(r) / (mu(10.0) * r * r)
    acc = np.zeros((n, 4), np.float32)
    acc[:, :3] = (-(a_mag / r)[:, None] * p[:, :3]).astype(np.float32)
    lev, emin, nlev = oracle.levels(acc, 2.0 ** -8, 0.5, 8)
    # analytic: level boundaries at radii where 0.25*eps/|a| = 4^e
    assert nlev == 4 and emin == -5
    rr = np.geomspace(1e-4, 10, 200001)
    ex = np.floor(np.log2(0.5 * np.sqrt(2.0 ** -8 / (mu(rr) / (mu(10.0) * rr * rr)))))
    frac = [(mu(rr[ex <= e].max()) - (mu(rr[ex < e].max()) if np.any(ex < e) else 0)) / mu(10.0) for e in range(-5, -1)]
    hist = np.bincount(lev, minlength=4) / n
    assert np.allclose(hist, frac, atol=0.01)
    # over the 8-substep cycle the work is sum_l frac_l * 2^(3-l) particle-walks per particle
    cyc = sum(oracle.active_set(lev, s).shape[0] for s in range(1, 9)) / n
    assert abs(cyc - sum(f * 2 ** (3 - l) for l, f in enumerate(frac))) < 0.05
