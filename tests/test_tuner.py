"""Host logic of the rebuild-interval tuner (paper_1610_07279_b200/tuner.py; eq. 8-12) on synthetic timings: no GPU."""
import pytest

from paper_1610_07279_b200.tuner import RebuildTuner


class Machine:
    """A stand-in for the live loop: the walk costs w0[class] * (1 + growth * age) per active particle, a rebuild t_make more than a refresh."""

    def __init__(self, n_sub, n_active, w0, growth, t_make, t_refresh=0.4):
        self.n_sub, self.n_active, self.w0, self.growth, self.t_make, self.t_refresh = n_sub, n_active, w0, growth, t_make, t_refresh

    def run(self, decide, n_steps):
        """decide(step index, substep) -> rebuild?  Returns the mean time per step over the second half of the run."""
        age, total = 0, 0.0
        for s in range(n_steps):
            substep = s % self.n_sub + 1
            cls = RebuildTuner.step_class(substep)
            rebuild = decide(s, substep)
            age = 0 if rebuild else age + 1
            tree = self.t_refresh + (self.t_make if rebuild else 0.0)
            walk = self.w0[cls] * (1.0 + self.growth * age) * self.n_active[cls]
            self.feed(substep, rebuild, tree, walk, self.n_active[cls])
            if s >= n_steps // 2:
                total += tree + walk
        return total / (n_steps - n_steps // 2)

    feed = staticmethod(lambda *a: None)


def _tuned(machine, n_steps, **kw):
    tuner = RebuildTuner(**kw)
    machine.feed = tuner.observe
    mean = machine.run(lambda s, substep: tuner.want_rebuild(substep), n_steps)
    machine.feed = lambda *a: None
    return tuner, mean


def _best_fixed(machine, n_steps, ks=range(1, 200)):
    return min((machine.run(lambda s, substep, k=k: s % k == 0, n_steps), k) for k in ks)


@pytest.mark.parametrize("t_make,growth", [(2.0, 0.05), (2.7, 0.01), (1.0, 0.2), (8.0, 0.002), (0.3, 0.5)])
def test_linear_growth_reproduces_eq_12(t_make, growth):
    """Equal steps whose walk time grows linearly with the tree's age (eq. 9, t_1 = 5 ms, dt = 5 ms * growth): the interval settles at the
    whole-number optimum of eq. 8-12, the smallest n with dt n (n + 1) / 2 >= t_make, which is within one step of n^2 = 2 t_make / dt."""
    m = Machine(1, {0: 1000}, {0: 5e-3}, growth, t_make)
    tuner, mean = _tuned(m, 4000, max_age=10 ** 6, ref_refresh=10 ** 9)
    dt = 5.0 * growth
    n_opt = next(n for n in range(1, 10 ** 6) if dt * n * (n + 1) / 2 >= t_make)
    iv = tuner.intervals()
    assert len(iv) >= 4 and iv[-1] == iv[-2] == n_opt, (iv[-6:], n_opt)
    assert abs(n_opt - (2.0 * t_make / dt) ** 0.5) <= 1.0
    best_mean, best_k = _best_fixed(m, 4000)
    assert abs(best_k - n_opt) <= 1 and mean <= 1.002 * best_mean           # (a finite run: the brute-force optimum may sit one step off)


def test_block_steps_rebuild_where_it_pays():
    """A block cycle of 4 substeps (sparse, populous, sparse, all active) with per-class costs and a tree that ages 30 % per step: the tuner
    must do at least as well as the best fixed interval, and it does so by rebuilding before the populous steps, not before the sparse ones."""
    m = Machine(4, {0: 50_000, 1: 1_000_000, 2: 4_000_000}, {0: 3e-6, 1: 1e-6, 2: 1.2e-6}, 0.3, 1.0)
    tuner, mean = _tuned(m, 4000, max_age=10 ** 6, ref_refresh=10 ** 9)
    best_mean, best_k = _best_fixed(m, 4000, ks=range(1, 33))
    assert mean <= 1.01 * best_mean, (mean, best_mean, best_k)
    late = tuner.history[-400:]
    rebuilt_by_class = {c: sum(1 for h in late if h[0] and h[2] == c) for c in (0, 1, 2)}
    assert rebuilt_by_class[2] == 100 and rebuilt_by_class[0] <= 4, rebuilt_by_class


def test_a_tree_that_does_not_age_is_left_alone():
    """Active counts that differ 80-fold between the steps of a cycle, per-particle costs that differ by class, no ageing: after one
    fresh-tree reference per class the tuner never rebuilds again (until a reference is due for renewal)."""
    m = Machine(8, {0: 50_000, 1: 1_000_000, 2: 2_000_000, 3: 4_000_000}, {0: 3e-6, 1: 1e-6, 2: 1.2e-6, 3: 1.5e-6}, 0.0, 2.5)
    tuner, _ = _tuned(m, 400, max_age=10 ** 6, ref_refresh=10 ** 9)
    assert sum(1 for h in tuner.history if h[0]) == 4 and tuner.loss == 0.0
    assert not any(h[0] for h in tuner.history[16:])
    tuner, _ = _tuned(m, 400, max_age=10 ** 6, ref_refresh=100)
    assert 8 <= sum(1 for h in tuner.history if h[0]) <= 20            # renewed references only


def test_bootstrap_empty_steps_and_the_age_cap():
    tuner = RebuildTuner(max_age=5)
    assert tuner.want_rebuild(1) and tuner.t_make is None             # the first step builds
    tuner.observe(1, True, 3.0, 1.0, 100)
    assert not tuner.want_rebuild(1)                                  # then one refresh step, to time it
    tuner.observe(1, False, 0.5, 0.0, 0)                              # an empty active list adds nothing
    assert tuner.t_make == 2.5 and tuner.loss == 0.0
    for _ in range(3):
        assert not tuner.want_rebuild(1)
        tuner.observe(1, False, 0.5, 1.0, 100)
    assert tuner.want_rebuild(1)                                      # age cap
