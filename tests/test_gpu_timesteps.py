"""-m gpu parity: block time-step levels (T1) and active-set compaction (T2): bit-exact vs the oracle."""
import numpy as np
import pytest
import torch

from paper_1610_07279_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _run(oracle, acc, eps, eta, max_levels):
    from gpu_util import dev
    from paper_1610_07279_b200.binding import Gothic
    n = acc.shape[0]
    g = Gothic(n)
    level = torch.zeros(n, dtype=torch.uint8, device="cuda")
    active = torch.zeros(n, dtype=torch.int32, device="cuda")
    n_act = torch.zeros(1, dtype=torch.int32, device="cuda")
    en = torch.zeros(2, dtype=torch.int32, device="cuda")
    g.set_timesteps(level, acc_pot=dev(acc), eps=eps, eta=eta, max_levels=max_levels, substep=1, active=active,
                    n_active_dev=n_act, emin_nlev_dev=en)
    lev_o, emin, nlev = oracle.levels(acc, eps, eta, max_levels)
    assert np.array_equal(level.cpu().numpy(), lev_o)
    assert en.cpu().tolist() == [emin, nlev]
    for s in range(1, 2 ** (nlev - 1) + 1):
        if s > 1:
            g.set_timesteps(level, acc_pot=None, eps=eps, substep=s, active=active, n_active_dev=n_act)
        a_o = oracle.active_set(lev_o, s)
        k = int(n_act.item())
        assert k == a_o.shape[0]
        assert np.array_equal(active[:k].cpu().numpy().view(np.uint32), a_o)
    g.close()


@pytest.mark.parametrize("n", [1, 7, 2047, 2048, 2049, 100000, (1 << 20) + 3])
def test_levels_and_active_sets_random(oracle, n):
    rng = np.random.default_rng(n)
    acc = np.zeros((n, 4), np.float32)
    acc[:, :3] = rng.normal(size=(n, 3)) * np.exp(rng.uniform(-4, 4, (n, 1)))
    if n > 10:
        acc[3, :3] = 0          # |a| = 0 -> coarsest
        acc[5, :3] = 1e30       # overflow of |a|^2 -> q = 0
        acc[6, :3] = 1e-30      # underflow of |a|^2 -> coarsest
    _run(oracle, acc, 2.0 ** -8, 0.5, 8)
    _run(oracle, acc, 0.013, 0.3, 5)


def test_levels_on_model_accelerations(oracle):
    """NFW analytic accelerations: 4 levels as in the paper's NFW runs."""
    n = 1 << 18
    pos = W.nfw(n, seed=1)
    p = pos.astype(np.float64)
    r = np.linalg.norm(p[:, :3], axis=1)
    mu = lambda x: np.log1p(x) - x / (1 + x)
    acc = np.zeros((n, 4), np.float32)
    acc[:, :3] = (-(mu(r) / (mu(10.0) * r ** 3))[:, None] * p[:, :3]).astype(np.float32)
    _run(oracle, acc, 2.0 ** -8, 0.5, 8)
