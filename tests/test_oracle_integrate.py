"""Pins for the oracle's predictor-corrector (O8; eq. 15-17) against what the mathematics fixes:
closed-form kinematics under a constant acceleration, the leap-frog it must reduce to for shared fixed steps,
second-order convergence on the harmonic oscillator, and the block-alignment invariant of the level migration (R15)."""
import numpy as np

import oracle


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
    assert np.all(t_last[oracle.active_set(level, 2 ** (max_levels - 1))] <= 2 ** (max_levels - 1))
