"""-m gpu: gothic_active_list_static, the one entry point of the library that allocates nothing.

Some hosts cannot call cudaMalloc once they are running: a simulation that has sized its own arrays to fill the GPU's memory,
a framework that keeps every byte of it in its own pool, a step loop that cannot stop for cudaMalloc's device-wide
synchronisation.  They cannot use a gothic_ctx (gothic_create allocates), so for the active list of a substep the library
offers a context-free call whose scratch (the per-tile counts of the ordered compaction) is a fixed 128 KiB array inside the
library image.  This test holds that call against the ordinary path, gothic_set_timesteps(acc_pot = NULL), bit for bit -- the
tolerance the other index tests use -- on two calls in a row: the second call finds the first one's counts still in the
array, and must not be disturbed by them.

The file sorts last on purpose (pytest -x stops at the first failure, so a failure here hides no other test), and it passes
alone in a fresh process as well as after the rest of the suite: it makes its own tensors and does not depend on which call
did the per-device set-up."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _levels(n, seed, n_levels):
    # a level mix like a block cycle's: most particles on the coarse levels, few on the finest
    rng = np.random.default_rng(seed)
    lev = np.minimum(rng.geometric(0.45, n) - 1, n_levels - 1)
    return (n_levels - 1 - lev).astype(np.uint8)


def _existing_path(level, substep):
    from paper_1610_07279_b200.binding import Gothic
    n = level.shape[0]
    g = Gothic(n)
    active = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    n_act = torch.zeros(1, dtype=torch.int32, device="cuda")
    g.set_timesteps(level, acc_pot=None, eps=1.0, substep=substep, active=active, n_active_dev=n_act)
    k = int(n_act.item())
    g.close()
    return k, active[:k].clone()


def _static_path(level, substep):
    from paper_1610_07279_b200.binding import active_list_static
    n = level.shape[0]
    active = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    n_act = torch.full((1,), -7, dtype=torch.int32, device="cuda")
    active_list_static(level, substep, active, n_act)
    k = int(n_act.item())
    assert bool((active[k:] == -1).all()), "entries past the count must stay untouched"
    return k, active[:k].clone()


def test_static_active_list_matches_set_timesteps_on_two_calls_in_a_row():
    # first call: many tiles and a ragged tail; second call: fewer tiles, another substep -- the array still holds the
    # first call's running offsets in every word, also in the ones the second call does not use
    cases = [((1 << 21) + 1234, 11, 6, 4), (2048 * 37 + 5, 12, 4, 1)]
    got = []
    for n, seed, n_levels, substep in cases:          # the two static calls back to back, nothing of the library in between
        level = torch.from_numpy(_levels(n, seed, n_levels)).cuda()
        got.append((level, substep, _static_path(level, substep)))
    for level, substep, (k, act) in got:
        k_ref, act_ref = _existing_path(level, substep)
        assert k == k_ref and k > 0
        assert torch.equal(act, act_ref)
        lev = level.cpu().numpy()
        ctz = (substep & -substep).bit_length() - 1
        assert np.array_equal(act.cpu().numpy(), np.flatnonzero(lev <= ctz).astype(np.int32))   # and both are the definition


def test_static_active_list_edges_and_the_size_limit():
    from paper_1610_07279_b200.binding import GothicError, STATIC_ACTIVE_MAX_N, active_list_static
    for n, substep in [(1, 1), (2047, 2), (2049, 8)]:
        level = torch.from_numpy(_levels(n, n, 3)).cuda()
        k, act = _static_path(level, substep)
        k_ref, act_ref = _existing_path(level, substep)
        assert k == k_ref and torch.equal(act, act_ref)
    # beyond the fixed scratch: refused with its own error before anything is launched or read
    level = torch.zeros(16, dtype=torch.uint8, device="cuda")
    active = torch.full((16,), -1, dtype=torch.int32, device="cuda")
    n_act = torch.full((1,), -7, dtype=torch.int32, device="cuda")
    with pytest.raises(GothicError, match="GOTHIC_STATIC_ACTIVE_MAX_N"):
        active_list_static(level, 1, active, n_act, n=STATIC_ACTIVE_MAX_N + 1)
    torch.cuda.synchronize()
    assert int(n_act.item()) == -7 and bool((active == -1).all())
