"""Pins for the oracle's predictor-corrector (O8; eq. 15-17) against what the mathematics fixes:
closed-form kinematics under a constant acceleration, the leap-frog it must reduce to for shared fixed steps,
second-order convergence on the harmonic oscillator, and the block-alignment invariant of the level migration (R15)."""
import math

import numpy as np

import oracle


def _wanted_level(a_vec, eps, eta, e_min, max_levels):
    """R6 written out in double with math.log2 (not through oracle.levels): the level the criterion dt = eta sqrt(eps/|a|), floored
    to a power of two, asks for, and whether |a| sits so close to a power-of-two boundary of dt that single precision may round
    to the other side."""
    a = math.sqrt(sum(float(x) ** 2 for x in a_vec))
    lg = math.log2(eta * math.sqrt(eps / a))
    near = abs(lg - round(lg)) < 1e-3
    return min(max(math.floor(lg) - e_min, 0), max_levels - 1), near


def _state(n, rng):
    pos = np.zeros((n, 4), np.float32)
    pos[:, :3] = rng.normal(size=(n, 3))
    pos[:, 3] = rng.uniform(0.5, 2.0, n)
    vel = np.zeros((n, 4), np.float32)
    vel[:, :3] = rng.normal(size=(n, 3))
    return pos, vel


def test_constant_acceleration_closed_form():
    """a = g for ever: r(t) = r0 + v0 dt + g dt^2/2 and v(t) = v0 + g dt exactly; every particle has its own t_last."""
    rng = np.random.default_rng(1)
    n = 1000
    pos, vel = _state(n, rng)
    acc = np.zeros((n, 4), np.float32)
    acc[:, :3] = rng.normal(size=(n, 3))
    t_last = rng.integers(0, 40, n).astype(np.uint32)
    t_now, unit = 64, 2.0 ** -7
    pred = oracle.predict(pos, vel, acc, t_last, t_now, unit)
    dt = (t_now - t_last.astype(np.float64)) * unit
    r_exact = pos[:, :3].astype(np.float64) + vel[:, :3].astype(np.float64) * dt[:, None] + 0.5 * acc[:, :3].astype(np.float64) * dt[:, None] ** 2
    assert np.allclose(pred[:, :3], r_exact, rtol=0, atol=4e-7 * np.abs(r_exact).max())
    assert np.array_equal(pred[:, 3], pos[:, 3])                      # mass carried along
    active = np.arange(0, n, 3, dtype=np.uint32)
    p2, v2, a2, t2 = pos.copy(), vel.copy(), acc.copy(), t_last.copy()
    oracle.correct(active, pred, acc, t_now, unit, p2, v2, a2, t2)
    v_exact = vel[:, :3].astype(np.float64) + acc[:, :3].astype(np.float64) * dt[:, None]
    assert np.allclose(v2[active, :3], v_exact[active], rtol=0, atol=4e-7 * np.abs(v_exact).max())
    assert np.array_equal(p2[active], pred[active]) and np.all(t2[active] == t_now)
    rest = np.setdiff1d(np.arange(n), active)
    assert np.array_equal(p2[rest], pos[rest]) and np.array_equal(v2[rest], vel[rest]) and np.array_equal(t2[rest], t_last[rest])


def _oscillate(n_steps, dt_unit):
    """x'' = -x from (1, 0) for n_steps shared steps through oracle.predict / oracle.correct (force evaluated here in fp32)."""
    pos = np.array([[1.0, 0.0, 0.0, 1.0]], np.float32)
    vel = np.zeros((1, 4), np.float32)
    acc = np.array([[-1.0, 0.0, 0.0, 0.0]], np.float32)
    t_last = np.zeros(1, np.uint32)
    act = np.zeros(1, np.uint32)
    for s in range(1, n_steps + 1):
        pred = oracle.predict(pos, vel, acc, t_last, s, dt_unit)
        acc_new = np.zeros((1, 4), np.float32)
        acc_new[0, 0] = -pred[0, 0]
        oracle.correct(act, pred, acc_new, s, dt_unit, pos, vel, acc, t_last)
    return float(pos[0, 0]), float(vel[0, 0])


def test_shared_step_is_leapfrog_and_second_order():
    """"For fixed shared timesteps, the Runge-Kutta integrator reduces to the leap-frog method" -- compared with a
    kick-drift-kick leap-frog written here in float64; and the error at t = 1 falls 4x when the step halves."""
    errs = []
    for k in (4, 5, 6):
        n_steps, dt = 2 ** k, 2.0 ** -k
        x, v = 1.0, 0.0
        for _ in range(n_steps):                       # textbook KDK
            v += 0.5 * dt * (-x)
            x += dt * v
            v += 0.5 * dt * (-x)
        xo, vo = _oscillate(n_steps, dt)
        assert abs(xo - x) < 2e-6 and abs(vo - v) < 2e-6
        errs.append(np.hypot(xo - np.cos(1.0), vo + np.sin(1.0)))
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5, errs


def test_prediction_is_from_the_last_corrected_state():
    """An inactive particle predicted at two successive substeps is extrapolated from the SAME state (not chained)."""
    rng = np.random.default_rng(3)
    pos, vel = _state(50, rng)
    acc = np.zeros((50, 4), np.float32)
    acc[:, :3] = rng.normal(size=(50, 3))
    t_last = np.full(50, 8, np.uint32)
    unit = 2.0 ** -6
    p1 = oracle.predict(pos, vel, acc, t_last, 9, unit)
    p2 = oracle.predict(pos, vel, acc, t_last, 10, unit)
    d1 = (p1[:, :3] - pos[:, :3]).astype(np.float64)
    d2 = (p2[:, :3] - pos[:, :3]).astype(np.float64)
    exact2 = 2 * unit * vel[:, :3].astype(np.float64) + 0.5 * (2 * unit) ** 2 * acc[:, :3].astype(np.float64)
    assert np.allclose(d2, exact2, atol=3e-7 * np.abs(pos[:, :3]).max()) and not np.allclose(d2, 2 * d1, atol=1e-9)
    assert np.array_equal(oracle.predict(pos, vel, acc, t_last, 8, unit)[:, :3], pos[:, :3])     # dt = 0: unchanged


def test_level_migration_keeps_blocks_aligned():
    """R15 over a whole cycle with random accelerations: a particle is only ever corrected at multiples of its step, never
    jumps more than one level coarser, and goes finer as far as the new acceleration asks."""
    rng = np.random.default_rng(5)
    n, eps, eta, max_levels = 4000, 2.0 ** -8, 0.5, 6
    acc = np.zeros((n, 4), np.float32)
    acc[:, :3] = rng.normal(size=(n, 3)) * np.exp(rng.uniform(-3, 3, (n, 1)))
    level, e_min, nlev = oracle.levels(acc, eps, eta, max_levels)
    assert nlev == max_levels
    pos, vel = _state(n, rng)
    t_last = np.zeros(n, np.uint32)
    unit = 2.0 ** e_min
    saw_far_jump = False
    for t in range(1, 2 ** (max_levels - 1) + 1):
        active = oracle.active_set(level, t)
        assert np.all(t % (1 << level[active].astype(np.int64)) == 0)
        assert np.all((t - t_last[active]) == (1 << level[active].astype(np.int64)))         # exactly one own step since last time
        acc_new = np.zeros((n, 4), np.float32)
        acc_new[:, :3] = acc[:, :3] * np.exp(rng.uniform(-1.5, 1.5, (n, 1))).astype(np.float32)
        before = level.copy()
        pred = oracle.predict(pos, vel, acc, t_last, t, unit)
        oracle.correct(active, pred, acc_new, t, unit, pos, vel, acc, t_last, level, eps=eps, eta=eta, e_min=e_min, max_levels=max_levels)
        moved = level.astype(int) - before.astype(int)
        inactive = np.setdiff1d(np.arange(n), active)
        assert np.all(moved[inactive] == 0) and np.all(moved[active] <= 1)
        coarser = active[moved[active] == 1]
        assert np.all(t % (1 << level[coarser].astype(np.int64)) == 0)
        assert np.all(level < max_levels)
        # no corrected particle keeps a step longer than the criterion allows for its NEW acceleration (R6):
        # finer is taken at once and in full, whatever the distance; coarser at most one level
        jumps = 0
        for i in active:
            want, near = _wanted_level(acc_new[i, :3], eps, eta, e_min, max_levels)
            if near:
                continue
            assert level[i] <= want, (t, i, before[i], level[i], want)
            if want < before[i]:
                assert level[i] == want, (t, i, before[i], level[i], want)
                jumps += before[i] - want >= 2
        saw_far_jump = saw_far_jump or jumps > 0
    assert saw_far_jump                                   # the run did contain moves of two or more levels finer
    assert np.all(t_last[oracle.active_set(level, 2 ** (max_levels - 1))] <= 2 ** (max_levels - 1))


def test_finer_migration_takes_the_whole_jump_at_once():
    """Hand case for R15's "any FINER level at once": eps = 2^-8, eta = 1/2, |a| = 2^-8 / s^2 gives dt = s/2; with s = 1.5 * 2^j
    that is 0.75 * 2^j, exponent j - 1, far from any boundary.  e_min = -10.  Particles on level 5 (j = -4) and level 3 (j = -6)
    whose new |a| is 16x / 256x the old one (dt 4x / 16x shorter) must land exactly two / four levels finer in ONE correction,
    clamped at level 0; one whose |a| falls 4x (dt 2x longer) goes one level coarser because t_now = 32 is a multiple of it."""
    eps, eta, e_min, max_levels = 2.0 ** -8, 0.5, -10, 8
    amag = lambda j: 2.0 ** -8 / (1.5 * 2.0 ** j) ** 2
    cur = np.array([5, 5, 3, 3, 3], np.uint8)
    scale = np.array([16.0, 256.0, 16.0, 256.0, 0.25])
    expect = np.array([3, 1, 1, 0, 4], np.uint8)
    n = cur.shape[0]
    acc = np.zeros((n, 4), np.float32)
    acc_new = np.zeros((n, 4), np.float32)
    for i in range(n):
        acc[i, i % 3] = amag(int(cur[i]) + e_min + 1)
        acc_new[i, (i + 1) % 3] = -acc[i, i % 3] * scale[i]
        assert _wanted_level(acc[i, :3], eps, eta, e_min, max_levels) == (cur[i], False)
    t_now = 32
    t_last = (t_now - (1 << cur.astype(np.int64))).astype(np.uint32)
    rng = np.random.default_rng(9)
    pos, vel = _state(n, rng)
    level = cur.copy()
    pred = oracle.predict(pos, vel, acc, t_last, t_now, 2.0 ** e_min)
    oracle.correct(np.arange(n, dtype=np.uint32), pred, acc_new, t_now, 2.0 ** e_min, pos, vel, acc, t_last, level,
                   eps=eps, eta=eta, e_min=e_min, max_levels=max_levels)
    assert level.tolist() == expect.tolist()
