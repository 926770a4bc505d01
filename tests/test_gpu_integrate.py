"""-m gpu parity: predictor / corrector under block time steps (eq. 15-17, row f1) through the C ABI.
Positions, velocities, times and levels are compared BIT-EXACTLY with the oracle (same fused multiply-adds, R15);
one end-to-end run integrates a small Plummer sphere over block cycles and checks energy conservation."""
import numpy as np
import pytest
import torch

from paper_1610_07279_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _rand_state(n, seed):
    rng = np.random.default_rng(seed)
    pos = np.zeros((n, 4), np.float32)
    pos[:, :3] = rng.normal(size=(n, 3))
    pos[:, 3] = rng.uniform(0.5, 2, n)
    vel = np.zeros((n, 4), np.float32)
    vel[:, :3] = rng.normal(size=(n, 3))
    acc = np.zeros((n, 4), np.float32)
    acc[:, :3] = rng.normal(size=(n, 3)) * np.exp(rng.uniform(-3, 3, (n, 1)))
    acc[:, 3] = -rng.uniform(1, 2, n)
    return rng, pos, vel, acc


@pytest.mark.parametrize("n", [1, 33, 4097, 100003])
def test_predict_and_correct_bit_exact(oracle, n):
    from gpu_util import dev
    from paper_1610_07279_b200.binding import Gothic
    rng, pos, vel, acc = _rand_state(n, n)
    eps, eta, max_levels = 2.0 ** -8, 0.5, 6
    level, e_min, nlev = oracle.levels(acc, eps, eta, max_levels)
    unit = 2.0 ** e_min
    t_now = 16
    t_last = (t_now - (1 << level.astype(np.int64))).clip(0).astype(np.uint32)
    t_last[rng.random(n) < 0.3] = t_now - 1
    g = Gothic(n)
    d = dict(pos=dev(pos), vel=dev(vel), acc=dev(acc), t=dev(t_last.view(np.int32)), lev=dev(level))
    pred = torch.zeros(n, 4, device="cuda")
    g.predict(d["pos"], d["vel"], d["acc"], d["t"], pred, t_now=t_now, dt_unit=unit)
    pred_ref = oracle.predict(pos, vel, acc, t_last, t_now, unit)
    assert np.array_equal(pred.cpu().numpy(), pred_ref)
    acc_new = acc.copy()
    acc_new[:, :3] *= np.exp(rng.uniform(-2, 2, (n, 1))).astype(np.float32)
    for mode in ("list", "device_count", "all"):
        active = oracle.active_set(level, t_now) if mode != "all" else np.arange(n, dtype=np.uint32)
        p2, v2, a2, t2, l2 = pos.copy(), vel.copy(), acc.copy(), t_last.copy(), level.copy()
        oracle.correct(active, pred_ref, acc_new, t_now, unit, p2, v2, a2, t2, l2, eps=eps, eta=eta, e_min=e_min, max_levels=max_levels)
        dd = {k: v.clone() for k, v in d.items()}
        kw = dict(t_now=t_now, dt_unit=unit, level=dd["lev"], eps=eps, eta=eta, e_min=e_min, max_levels=max_levels)
        if mode == "list":
            kw.update(active=dev(active.view(np.int32)))
        elif mode == "device_count":
            padded = np.concatenate([active, np.zeros(7, np.uint32)])
            kw.update(active=dev(padded.view(np.int32)), n_active_dev=torch.tensor([active.shape[0]], dtype=torch.int32, device="cuda"))
        g.correct(pred, dev(acc_new), dd["pos"], dd["vel"], dd["acc"], dd["t"], **kw)
        g.check()
        assert np.array_equal(dd["pos"].cpu().numpy(), p2) and np.array_equal(dd["vel"].cpu().numpy(), v2)
        assert np.array_equal(dd["acc"].cpu().numpy(), a2) and np.array_equal(dd["t"].cpu().numpy().view(np.uint32), t2)
        assert np.array_equal(dd["lev"].cpu().numpy(), l2)
    g.close()


def test_integrate_rejects_bad_arguments():
    from paper_1610_07279_b200.binding import Gothic, GothicError
    g = Gothic(64)
    z4 = torch.zeros(64, 4, device="cuda")
    t = torch.zeros(64, dtype=torch.int32, device="cuda")
    with pytest.raises(GothicError):
        g.predict(z4, z4, z4, t, z4.clone(), t_now=1, dt_unit=0.0)
    with pytest.raises(GothicError):
        g.correct(z4, z4, z4.clone(), z4.clone(), z4, t, t_now=1, dt_unit=1.0)        # acc_new aliases acc_pot
    g.close()


def test_block_step_integration_conserves_energy(oracle):
    """Plummer sphere in virial equilibrium, N = 4096, integrated for 4 block cycles on the GPU (predict -> build -> walk ->
    correct with level migration).  Energy from the double-precision direct sum (oracle.direct) must be conserved to 1e-3."""
    from paper_1610_07279_b200.binding import Gothic, MAC_ACCELERATION, MAC_OPENING_ANGLE
    n, eps, dacc, eta, max_levels = 4096, 1.0 / 64, 2.0 ** -9, 0.25, 6
    pos_np = W.plummer(n, seed=3)
    rng = np.random.default_rng(4)
    r = np.linalg.norm(pos_np[:, :3].astype(np.float64), axis=1)
    sigma = np.sqrt(1.0 / (6.0 * np.sqrt(1.0 + r * r)))                  # isotropic Plummer: sigma^2 = -Phi/6
    vel_np = np.zeros((n, 4), np.float32)
    vel_np[:, :3] = (rng.normal(size=(n, 3)) * sigma[:, None]).astype(np.float32)

    def energy(p, v):
        d = oracle.direct(p, eps)
        m = p[:, 3].astype(np.float64)
        return 0.5 * (m * (v[:, :3].astype(np.float64) ** 2).sum(1)).sum() + 0.5 * (m * d[:, 3]).sum()

    g = Gothic(n)
    # the state lives in the sorted order of the FIRST build; later builds re-sort predicted copies
    g.build_tree(torch.from_numpy(pos_np).cuda())
    v0 = g.get_tree_view()
    perm = v0["perm"].long()
    pos = v0["pos_m_sorted"].clone()
    vel = torch.from_numpy(vel_np).cuda()[perm].contiguous()
    acc = torch.zeros(n, 4, device="cuda")
    amag = torch.zeros(n, device="cuda")
    g.walk_tree(acc, eps=eps, mac_kind=MAC_OPENING_ANGLE, mac_param=0.3, amag_out=amag)
    e0 = energy(pos.cpu().numpy(), vel.cpu().numpy())
    level = torch.zeros(n, dtype=torch.uint8, device="cuda")
    active = torch.zeros(n, dtype=torch.int32, device="cuda")
    n_act = torch.zeros(1, dtype=torch.int32, device="cuda")
    info = torch.zeros(2, dtype=torch.int32, device="cuda")
    pred = torch.zeros(n, 4, device="cuda")
    acc_new = torch.zeros(n, 4, device="cuda")
    for cycle in range(4):
        g.set_timesteps(level, acc_pot=acc, eps=eps, eta=eta, max_levels=max_levels, emin_nlev_dev=info)
        e_min, nlev = info.tolist()
        unit = 2.0 ** e_min
        t_last = torch.zeros(n, dtype=torch.int32, device="cuda")
        for t in range(1, 2 ** (max_levels - 1) + 1):
            g.set_timesteps(level, acc_pot=None, eps=eps, substep=t, active=active, n_active_dev=n_act)
            g.predict(pos, vel, acc, t_last, pred, t_now=t, dt_unit=unit)
            # gravity from the predicted j-particles on the active i-particles: fresh tree in the predicted positions,
            # active indices mapped into its sorted order
            g.build_tree(pred)
            p2 = g.get_tree_view()["perm"].long()
            inv = torch.empty_like(p2)
            inv[p2] = torch.arange(n, device="cuda")
            na = int(n_act.item())
            act_sorted = torch.sort(inv[active[:na].long()]).values.int().contiguous()
            acc_s = torch.zeros(n, 4, device="cuda")
            g.walk_tree(acc_s, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=dacc, aold=amag[p2].contiguous(), active=act_sorted)
            acc_new[p2] = acc_s
            g.correct(pred, acc_new, pos, vel, acc, t_last, t_now=t, dt_unit=unit, active=active, n_active_dev=n_act,
                      level=level, eps=eps, eta=eta, e_min=e_min, max_levels=max_levels)
            amag = torch.linalg.norm(acc[:, :3], dim=1).contiguous()
        g.check()
        assert int(t_last.min().item()) == 2 ** (max_levels - 1)          # everybody synchronised at the end of the cycle
    e1 = energy(pos.cpu().numpy(), vel.cpu().numpy())
    assert abs(e1 - e0) / abs(e0) < 1e-3, (e0, e1)
    assert -0.4 < e0 < -0.05                                               # bound, near virial (E ~ -3 pi / 64 = -0.147 for a = M = 1)
    g.close()
