"""Host-side choice of the tree rebuild interval from timings (section 2.6, eq. 8-12), on top of gothic_live_step.

The paper minimises the mean time per step t_tot / n with t_tot = t_make + sum_i t_walk^(i) (eq. 8).  For walk times that grow linearly
with the age of the tree, t_walk^(i) = t_1 + (i - 1) dt (eq. 9, fitted by least squares), the minimum is at n^2 = 2 t_make / dt (eq. 12);
for whole numbers of steps it is the smallest n with dt n (n + 1) / 2 >= t_make.  Read step by step, that is: rebuild before a step
if the walk time LOST to the old tree since the last rebuild, plus what this step would lose on the old tree, reaches the price of a
rebuild.  The rule below is this form, because it carries over to block time steps, where the number of active particles changes from
step to step and a raw t_walk^(i) is not a function of the tree's age alone:

  * steps are sorted into classes by ctz(substep) (all steps of a class have the same levels active) and the walk cost is taken per
    active particle, w = t_walk / n_active;
  * w0[class] is w on a FRESH tree, i.e. observed on a rebuild step of that class.  A class without such a reference (or with one older
    than `ref_refresh` steps) gets a rebuild at its next step, so that the references do not depend on how the rebuilds happen to fall
    within the cycle;
  * eq. 9 per class, in relative form: w / w0[class] - 1 = slope[class] * age, the slope fitted by least squares through the origin over
    the observations on aged trees (exponentially forgotten);
  * every step on an aged tree adds (w - w0[class]) * n_active to the loss (never less than zero); a rebuild resets the loss;
  * t_make is the tree stage of a rebuild step minus the tree stage of a refresh step (moments only), both as last measured;
  * the step about to be taken, of class c at age a, rebuilds when loss + slope[c] * a * w0[c] * n_active[c] >= t_make.

For equal steps and linear growth this is the whole-number optimum of eq. 8-12 (tests/test_tuner.py).  The paper's other two growth models
(App. C) and its chi^2 choice between them (eq. 14) are not implemented.  Everything here is host arithmetic on three numbers per step
(Gothic.live_timing()); the method's own arithmetic stays in the kernels."""
from __future__ import annotations


class RebuildTuner:
    def __init__(self, max_age: int = 64, ref_refresh: int = 512, forget: float = 0.9):
        self.max_age = max_age          # rebuild at the latest after this many steps on one tree
        self.ref_refresh = ref_refresh  # a fresh-tree reference older than this many steps is taken again
        self.forget = forget            # weight of the older observations in the slope fit, per new observation
        self.t_rebuild = None           # tree stage of the last rebuild step [ms]
        self.t_refresh = None           # tree stage of the last refresh step [ms]
        self.w0 = {}                    # class -> (w on a fresh tree, step at which it was seen)
        self.fit = {}                   # class -> [sum age * e, sum age^2] with e = w / w0 - 1
        self.n_last = {}                # class -> n_active last seen
        self.loss = 0.0                 # walk time lost to the tree's age since the last rebuild [ms]
        self.age = 0                    # steps since the last rebuild (0 = the rebuild step itself)
        self.steps = 0
        self.history = []               # (rebuilt, age, class, tree_ms, walk_ms, n_active, loss)

    @staticmethod
    def step_class(substep: int) -> int:
        return (substep & -substep).bit_length() - 1

    @property
    def t_make(self):
        """What a rebuild costs over a refresh, or None before both have been seen."""
        if self.t_rebuild is None or self.t_refresh is None:
            return None
        return max(self.t_rebuild - self.t_refresh, 0.0)

    def slope(self, cls: int) -> float:
        sxy, sxx = self.fit.get(cls, (0.0, 0.0))
        return max(sxy / sxx, 0.0) if sxx > 0.0 else 0.0

    def want_rebuild(self, substep: int) -> bool:
        """Should the step about to be taken (1-based index `substep` within the cycle) rebuild the tree?"""
        if self.t_make is None:         # until both kinds of step have been timed: one of each
            return self.t_rebuild is None or self.t_refresh is not None
        cls = self.step_class(substep)
        ref = self.w0.get(cls)
        if ref is None or self.steps - ref[1] > self.ref_refresh:
            return True
        age = self.age + 1
        if age >= self.max_age:
            return True
        predicted = self.slope(cls) * age * ref[0] * self.n_last.get(cls, 0)
        return self.loss + predicted >= self.t_make

    def observe(self, substep: int, rebuilt: bool, tree_ms: float, walk_ms: float, n_active: int) -> None:
        """One finished step: `substep` is its 1-based index within the cycle, the rest is Gothic.live_timing()'s."""
        cls = self.step_class(substep)
        self.steps += 1
        if rebuilt:
            self.t_rebuild, self.age, self.loss = tree_ms, 0, 0.0
        else:
            self.t_refresh = tree_ms
            self.age += 1
        self.n_last[cls] = n_active
        if n_active > 0:
            w = walk_ms / n_active
            if rebuilt:
                self.w0[cls] = (w, self.steps)
            elif cls in self.w0 and self.w0[cls][0] > 0.0:
                w0 = self.w0[cls][0]
                e = w / w0 - 1.0
                self.loss += max(0.0, e) * w0 * n_active
                f = self.fit.setdefault(cls, [0.0, 0.0])
                f[0] = self.forget * f[0] + self.age * e
                f[1] = self.forget * f[1] + self.age * self.age
        self.history.append((rebuilt, self.age, cls, tree_ms, walk_ms, n_active, self.loss))

    def intervals(self) -> list[int]:
        """Lengths of the finished rebuild intervals so far (steps per tree)."""
        out, run = [], None
        for rebuilt, *_ in self.history:
            if rebuilt:
                if run is not None:
                    out.append(run)
                run = 1
            elif run is not None:
                run += 1
        return out
