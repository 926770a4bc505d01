"""-m gpu: one compact scenario that touches every kernel of the library, small enough to run under compute-sanitizer
(racecheck / memcheck / synccheck on the small configurations).

    compute-sanitizer --tool memcheck  python -m pytest tests/test_gpu_sanitizer_scenario.py -q -m gpu
    compute-sanitizer --tool racecheck python -m pytest tests/test_gpu_sanitizer_scenario.py -q -m gpu
    compute-sanitizer --tool synccheck python -m pytest tests/test_gpu_sanitizer_scenario.py -q -m gpu

(one tool per run; the summaries are kept in profiles/r02_sanitizer.md).  Without the sanitizer it is an ordinary parity
test: interaction counts equal the oracle's for every (G, MAC, ball, r_crit) it walks, levels / active list bit-exact, the
predictor / corrector bit-exact, and the spill path of the traversal stack is taken without overflow."""
import numpy as np
import pytest
import torch

from paper_1610_07279_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _oracle_on_gpu_tree(oracle, v, **kw):
    return oracle.walk(v["pos_m_sorted"], v["node_head"], v["node_num"], v["node_child"], v["node_nchild"],
                       v["node_com"], v["node_b"], **kw)


@pytest.mark.parametrize("G", [8, 32])
def test_scenario_all_kernels(oracle, G):
    from gpu_util import gpu_build, gpu_walk, dev
    n, eps = 6001, 2.0 ** -6
    pos = W.hernquist(n, seed=9)
    for key_kind in (0, 1):                                        # Peano-Hilbert and Morton keys, sort, nodes, moments
        g, v = gpu_build(pos, key_kind=key_kind, n_leaf=8, group_size=G)
        t = oracle.build_tree(pos, key_kind=key_kind, n_leaf=8)
        assert np.array_equal(v["key"], t.key) and np.array_equal(v["perm"], t.perm) and np.array_equal(v["node_head"], t.head)
        if key_kind == 0:
            g.close()
    out, _, aold = gpu_walk(g, n, eps=eps, mac_kind=1, mac_param=0.5, amag=True, count=False)
    # levels + active list (T1, T2)
    acc = dev(out.astype(np.float32))
    level = torch.zeros(n, dtype=torch.uint8, device="cuda")
    active = torch.zeros(n, dtype=torch.int32, device="cuda")
    n_act = torch.zeros(1, dtype=torch.int32, device="cuda")
    info = torch.zeros(2, dtype=torch.int32, device="cuda")
    g.set_timesteps(level, acc_pot=acc, eps=eps, substep=2, active=active, n_active_dev=n_act, emin_nlev_dev=info)
    lev_ref, emin, nlev = oracle.levels(out.astype(np.float32), eps)
    assert np.array_equal(level.cpu().numpy(), lev_ref) and info.tolist() == [emin, nlev]
    act_ref = oracle.active_set(lev_ref, 2)
    na = int(n_act.item())
    assert na == act_ref.shape[0] and np.array_equal(active[:na].cpu().numpy().view(np.uint32), act_ref)
    sparse = W.random_active_subset(n, 0.07, seed=3)
    # every MAC x every ball, full and sparse active sets, with and without group splitting
    for mac_kind, param in ((0, 2.0 ** -8), (1, 0.55), (2, 2.0 ** -6)):
        for ball in (0, 1, 2, 3, 4):
            g.set_ball(ball)
            for act, r_crit in ((None, float("inf")), (sparse, 0.2), (act_ref, 0.0)):
                _, cnt, _ = gpu_walk(g, n, eps=eps, mac_kind=mac_kind, mac_param=param, aold=aold, active=act, r_crit=r_crit)
                _, c = _oracle_on_gpu_tree(oracle, v, eps=eps, mac_kind=mac_kind, mac_param=param, aold=aold, active=act, group_size=G,
                                           r_crit=r_crit, ball_kind=ball, B2=v["node_b2"])
                assert cnt == c["interactions"], (G, mac_kind, ball, r_crit)
    g.set_ball(0)
    # moments refresh on moved particles, predictor / corrector with level migration (row f1)
    rng = np.random.default_rng(5)
    ps = v["pos_m_sorted"].copy()
    vel = (0.3 * rng.standard_normal((n, 4))).astype(np.float32)
    acc_s = out.astype(np.float32)                       # the walk writes rows in sorted order
    t_last = np.zeros(n, np.uint32)
    dt_unit = float(2.0 ** emin)
    pred = torch.zeros(n, 4, device="cuda")
    d_ps, d_vel, d_acc, d_tl, d_lev = dev(ps), dev(vel), dev(acc_s), dev(t_last.view(np.int32)), dev(lev_ref)
    g.predict(d_ps, d_vel, d_acc, d_tl, pred, t_now=2, dt_unit=dt_unit)
    ref_pred = oracle.predict(ps, vel, acc_s, t_last, 2, dt_unit)
    assert np.array_equal(pred.cpu().numpy(), ref_pred)
    acc_new = acc_s.copy()
    acc_new[:, :3] *= np.exp(rng.uniform(-2, 2, (n, 1))).astype(np.float32)
    p2, v2, a2, t2, l2 = ps.copy(), vel.copy(), acc_s.copy(), t_last.copy(), lev_ref.copy()
    oracle.correct(act_ref, ref_pred, acc_new, 2, dt_unit, p2, v2, a2, t2, l2, eps=eps, eta=0.5, e_min=emin, max_levels=8)
    g.correct(pred, dev(acc_new), d_ps, d_vel, d_acc, d_tl, t_now=2, dt_unit=dt_unit, active=dev(act_ref.view(np.int32)), level=d_lev,
              eps=eps, eta=0.5, e_min=emin, max_levels=8)
    assert np.array_equal(d_ps.cpu().numpy(), p2) and np.array_equal(d_vel.cpu().numpy(), v2) and np.array_equal(d_lev.cpu().numpy(), l2)
    g.update_moments(pred)
    g.check()
    g.close()


def test_scenario_stack_spill(oracle):
    """theta = 0 with one particle per leaf: the pending families outgrow the 256 shared-memory slots of a warp and travel
    through the global spill area (default size: no overflow); the result is the direct sum (eq. 1)."""
    from gpu_util import dev
    from paper_1610_07279_b200.binding import Gothic
    n = 1 << 15
    pos = W.plummer(n, seed=4)
    g = Gothic(n)
    g.build_tree(dev(pos), n_leaf=1)
    acc = torch.zeros(n, 4, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    act = torch.arange(0, 64, dtype=torch.int32, device="cuda")
    g.walk_tree(acc, eps=0.01, mac_kind=1, mac_param=0.0, active=act, n_interactions=cnt)
    g.check()
    assert int(cnt.item()) == 64 * n
    v = g.get_tree_view()
    ps = v["pos_m_sorted"].cpu().numpy()
    ref = oracle.direct(ps, 0.01, targets=np.arange(64, dtype=np.uint32))
    out = acc[:64].cpu().numpy().astype(np.float64)
    e = np.linalg.norm(out[:, :3] - ref[:64, :3], axis=1) / np.linalg.norm(ref[:64, :3], axis=1)
    assert e.max() < 1e-4
    g.close()
