"""-m gpu: the host-buffer conveniences (bench.py's e2e leg) give exactly what the device-pointer calls give: same kernels, same
order, deterministic => bit-identical; the device-pointer path is itself held against the oracle in the other -m gpu tests."""
import numpy as np
import pytest
import torch

from paper_1610_07279_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("model,n", [("plummer", 1 << 13), ("nfw", 50001)])
def test_block_cycle_host_equals_device_calls(oracle, model, n):
    from paper_1610_07279_b200.binding import Gothic, MAC_ACCELERATION, MAC_OPENING_ANGLE
    pos_np = getattr(W, model)(n, seed=3)
    eps, dacc, eta, max_levels, r_crit = 2.0 ** -7, 2.0 ** -8, 0.5, 8, 0.5
    g = Gothic(n)
    pos = torch.from_numpy(pos_np).cuda()
    # previous accelerations (ORIGINAL order) from a bootstrap walk
    g.build_tree(pos)
    perm = g.get_tree_view()["perm"].long()
    acc_s = torch.zeros(n, 4, device="cuda")
    g.walk_tree(acc_s, eps=eps, mac_kind=MAC_OPENING_ANGLE, mac_param=0.5)
    acc_prev = torch.empty_like(acc_s)
    acc_prev[perm] = acc_s
    # ---- host call ----
    h_pos, h_prev = torch.from_numpy(pos_np).pin_memory(), acc_prev.cpu().pin_memory()
    h_out, h_lev = torch.empty(n, 4).pin_memory(), torch.empty(n, dtype=torch.uint8).pin_memory()
    info = g.block_cycle_host(h_pos, h_prev, h_out, eps=eps, delta_acc=dacc, eta=eta, max_levels=max_levels, level_host=h_lev, count=True, r_crit=r_crit)
    # ---- the same cycle through the device-pointer calls ----
    g.build_tree(pos)
    perm = g.get_tree_view()["perm"].long()
    acc = acc_prev[perm].contiguous()
    a64 = acc.cpu().numpy()      # |a| as k_gather_acc forms it: sqrt(fma(az, az, fma(ay, ay, ax * ax))) in fp32
    amag = torch.from_numpy(np.sqrt(np.float32(np.float64(a64[:, 2]) ** 2 + np.float32(np.float64(a64[:, 1]) ** 2 + np.float32(a64[:, 0] * a64[:, 0]))).astype(np.float32))).cuda()
    level = torch.zeros(n, dtype=torch.uint8, device="cuda")
    active = torch.zeros(n, dtype=torch.int32, device="cuda")
    n_act = torch.zeros(1, dtype=torch.int32, device="cuda")
    en = torch.zeros(2, dtype=torch.int32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    g.set_timesteps(level, acc_pot=acc, eps=eps, eta=eta, max_levels=max_levels, emin_nlev_dev=en)
    e_min, nlev = en.tolist()
    assert (info["e_min"], info["n_levels"], info["n_substeps"]) == (e_min, nlev, 2 ** (nlev - 1))
    for s in range(1, 2 ** (nlev - 1) + 1):
        g.set_timesteps(level, acc_pot=None, eps=eps, substep=s, active=active, n_active_dev=n_act)
        g.update_moments()
        g.walk_tree(acc, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=dacc, aold=amag, active=active, n_active_dev=n_act, amag_out=amag,
                    n_interactions=cnt, r_crit=r_crit)
    g.check()
    out = torch.empty_like(acc)
    out[perm] = acc
    lev = torch.empty_like(level)
    lev[perm] = level
    assert torch.equal(h_out.cuda(), out) and torch.equal(h_lev.cuda(), lev)
    assert info["interactions"] == int(cnt.item())
    # levels against the oracle (original order)
    lev_ref, emin_ref, nlev_ref = oracle.levels(acc_prev.cpu().numpy(), eps, eta, max_levels)
    assert np.array_equal(h_lev.numpy(), lev_ref) and (emin_ref, nlev_ref) == (e_min, nlev)
    g.close()


@pytest.mark.parametrize("model,n", [("plummer", 20000), ("hernquist", 30011)])
def test_block_cycle_host_vs_oracle(oracle, model, n):
    """The e2e call itself against the oracle, nothing of the CUDA path on the reference side: the oracle builds its own tree and moments,
    takes the levels from the same previous accelerations and walks every substep's active set with its own running |a_old|.  Levels and
    the substep count are bit-exact; accelerations within the north_star tolerances (MAC flips at threshold allowed), counts to 1e-3."""
    from paper_1610_07279_b200.binding import Gothic
    pos = getattr(W, model)(n, seed=6)
    eps, dacc, eta, max_levels, r_crit = 2.0 ** -6, 2.0 ** -8, 0.5, 6, 0.5
    t = oracle.build_tree(pos)
    boot, _ = oracle.walk_tree(t, eps=eps, mac_kind=1, mac_param=0.5)
    acc_prev = np.zeros((n, 4), np.float32)
    acc_prev[t.perm] = boot.astype(np.float32)                 # ORIGINAL order
    # ---- the cycle in the oracle (sorted order) ----
    acc_s = acc_prev[t.perm]
    lev_s, e_min, nlev = oracle.levels(acc_s, eps, eta, max_levels)
    amag = np.sqrt(np.float32(np.float64(acc_s[:, 2]) ** 2 + np.float32(np.float64(acc_s[:, 1]) ** 2 + np.float32(acc_s[:, 0] * acc_s[:, 0]))).astype(np.float32))
    ref = acc_s.astype(np.float64)
    total = 0
    for s in range(1, 2 ** (nlev - 1) + 1):
        act = oracle.active_set(lev_s, s)
        o, c = oracle.walk_tree(t, eps=eps, mac_kind=0, mac_param=dacc, aold=amag, active=act, r_crit=r_crit)
        ref[act] = o[act]
        amag[act] = np.linalg.norm(o[act, :3], axis=1).astype(np.float32)
        total += c["interactions"]
    # ---- the host call ----
    g = Gothic(n)
    h_out, h_lev = torch.empty(n, 4).pin_memory(), torch.empty(n, dtype=torch.uint8).pin_memory()
    info = g.block_cycle_host(torch.from_numpy(pos).pin_memory(), torch.from_numpy(acc_prev).pin_memory(), h_out, eps=eps, delta_acc=dacc, eta=eta,
                              max_levels=max_levels, level_host=h_lev, count=True, r_crit=r_crit)
    g.check()
    assert (info["e_min"], info["n_levels"], info["n_substeps"]) == (e_min, nlev, 2 ** (nlev - 1))
    assert np.array_equal(h_lev.numpy()[t.perm], lev_s)
    out = h_out.numpy().astype(np.float64)[t.perm]
    e = np.linalg.norm(out[:, :3] - ref[:, :3], axis=1) / np.linalg.norm(ref[:, :3], axis=1)
    pe = np.abs(out[:, 3] - ref[:, 3]) / np.abs(ref[:, 3])
    assert np.percentile(e, 99.9) <= 1e-4 and e.max() <= 1e-2 and np.median(pe) <= 1e-4, (np.percentile(e, 99.9), e.max(), np.median(pe))
    assert abs(info["interactions"] - total) <= 1e-3 * total, (info["interactions"], total)
    g.close()


def test_gravity_host_equals_device_calls():
    from paper_1610_07279_b200.binding import Gothic, MAC_ACCELERATION, MAC_OPENING_ANGLE
    n = 30000
    pos_np = W.hernquist(n, seed=5)
    eps = 2.0 ** -7
    g = Gothic(n)
    h_pos = torch.from_numpy(pos_np).pin_memory()
    h_acc, h_perm = torch.empty(n, 4).pin_memory(), torch.empty(n, dtype=torch.int32).pin_memory()
    g.gravity_host(h_pos, h_acc, eps=eps, mac_kind=MAC_OPENING_ANGLE, mac_param=0.6, perm_host=h_perm)
    pos = torch.from_numpy(pos_np).cuda()
    g.build_tree(pos)
    acc = torch.zeros(n, 4, device="cuda")
    g.walk_tree(acc, eps=eps, mac_kind=MAC_OPENING_ANGLE, mac_param=0.6)
    assert torch.equal(h_acc.cuda(), acc) and torch.equal(h_perm.cuda(), g.get_tree_view()["perm"])
    # acceleration MAC with |a_old| given in ORIGINAL order
    aold_orig = torch.empty(n, device="cuda")
    perm = h_perm.cuda().long()
    aold_sorted = torch.linalg.norm(acc[:, :3], dim=1).contiguous()
    aold_orig[perm] = aold_sorted
    g.gravity_host(h_pos, h_acc, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=2.0 ** -8, aold_host=aold_orig.cpu().pin_memory(), r_crit=0.5)
    g.walk_tree(acc, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=2.0 ** -8, aold=aold_sorted, r_crit=0.5)
    assert torch.equal(h_acc.cuda(), acc)
    g.close()
