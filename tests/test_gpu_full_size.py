"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

configs[2] / configs[3] (NFW and M31-like, N = 2^24, one block-step cycle): keys, permutation, node arrays, levels and
every substep's active list are compared bit-exactly over all N; accelerations and potentials on samples of i-groups the
oracle walks one by one (on the GPU-built tree and moments).
configs[4] (NFW, N = 2^22): accuracy-parameter and active-fraction sweep; sampled parity, and the error against the
double-precision direct sum (eq. 1) on a 4096-particle sample must shrink as Delta_acc tightens (Fig. 3)."""
import numpy as np
import pytest
import torch

from paper_1610_07279_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_999, TOL_MAX, TOL_POT_MEDIAN = 1e-4, 1e-2, 1e-4   # BASELINE.json north_star
G = 32


def _parity(out, ref, rows):
    from gpu_util import acc_rel_err
    e = acc_rel_err(out[rows], ref[rows])
    pe = np.abs(out[rows, 3] - ref[rows, 3]) / np.abs(ref[rows, 3])
    assert np.percentile(e, 99.9) <= TOL_999 and e.max() <= TOL_MAX, (np.percentile(e, 99.9), e.max())
    assert np.median(pe) <= TOL_POT_MEDIAN and pe.max() <= 1e-3, (np.median(pe), pe.max())


def _group_samples(n, per=64, pieces=4):
    n_groups = n // G
    return [(lo, lo + per) for lo in np.linspace(0, n_groups - per, pieces).astype(int)]


def _seeded_group_ids(pos_sorted, seed, places=16, run=8, widest=8):
    """Group ids for the count-equality checks: `places` seeded random runs of `run` consecutive groups plus the `widest` groups
    with the largest GEO ball (the ones r_crit splits the deepest)."""
    n = pos_sorted.shape[0]
    n_groups = n // G
    rng = np.random.default_rng(seed)
    starts = rng.choice(n_groups - run, places, replace=False)
    ids = np.concatenate([np.arange(s0, s0 + run) for s0 in starts])
    xyz = pos_sorted[: n_groups * G, :3].reshape(n_groups, G, 3)
    ctr = 0.5 * (xyz.min(axis=1) + xyz.max(axis=1))
    r2 = ((xyz - ctr[:, None, :]) ** 2).sum(axis=2).max(axis=1)
    ids = np.concatenate([ids, np.argsort(r2)[-widest:]])
    return np.unique(ids).astype(np.int64)


def _count_equality(g, oracle_walk, gids, members, n, *, eps, dacc, aold, r_crit, out_full, active=None):
    """Walks ONLY `members` (the active particles of the groups `gids`) on the GPU with its own device counter and holds the count
    against the oracle's sum over the same groups: EQUAL, the sharpest check of the suite, here at full size.  The rows of that
    restricted walk are also bit-identical to the full walk's (a group's arithmetic does not depend on which other groups walk)."""
    from gpu_util import dev
    from paper_1610_07279_b200.binding import MAC_ACCELERATION
    acc2 = torch.zeros(n, 4, device="cuda")
    cnt2 = torch.zeros(1, dtype=torch.int64, device="cuda")
    g.walk_tree(acc2, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=dacc, aold=dev(aold), active=dev(members.astype(np.uint32), torch.int32),
                r_crit=r_crit, n_interactions=cnt2)
    g.check()
    total = 0
    for gid in gids:
        _, c = oracle_walk(eps=eps, mac_kind=0, mac_param=dacc, aold=aold, active=active, group_range=(int(gid), int(gid) + 1), r_crit=r_crit)
        total += c["interactions"]
    assert int(cnt2.item()) == total, (int(cnt2.item()), total)
    assert np.array_equal(acc2.cpu().numpy()[members], out_full[members].astype(np.float32))


def _rows_of(ranges, active=None):
    rows = np.concatenate([np.arange(lo * G, hi * G) for lo, hi in ranges])
    if active is not None:
        rows = rows[np.isin(rows, active)]
    return rows


@pytest.mark.parametrize("name", ["nfw_2p24_block", "m31_2p24_block"])
def test_block_cycle_full_size(oracle, name):
    from gpu_util import view_to_numpy
    from paper_1610_07279_b200.binding import Gothic, MAC_ACCELERATION, MAC_OPENING_ANGLE
    pos, cfg = W.make_config(name, seed=1)
    n, eps, dacc, r_crit = cfg["n"], cfg["eps"], cfg["delta_acc"], cfg["r_crit"]
    g = Gothic(n)
    d_pos = torch.from_numpy(pos).cuda()
    g.build_tree(d_pos)
    v = view_to_numpy(g.get_tree_view())
    # ---- B1-B5 bit-exact over all N; B6 on the oracle's own arithmetic ----
    t = oracle.build_tree(pos)
    assert np.array_equal(np.asarray(v["box"], np.float32), t.box)
    assert np.array_equal(v["key"], t.key) and np.array_equal(v["perm"], t.perm)
    assert v["n_nodes"] == t.n_nodes
    for a, b in (("node_head", t.head), ("node_num", t.num), ("node_child", t.child), ("node_level", t.level), ("node_nchild", t.nchild)):
        assert np.array_equal(v[a], b), a
    assert np.array_equal(v["pos_m_sorted"], t.pos_sorted)
    assert np.allclose(v["node_com"], t.com, rtol=2e-5, atol=1e-6)
    b_def = oracle.radius(t.pos_sorted, t.head, t.num, v["node_com"])      # the definition (double) about the stored centres
    assert np.all(np.abs(v["node_b"] - b_def) <= 1e-6 * b_def + 1e-9 * float(t.box[3]))
    del t

    def oracle_walk(**kw):
        return oracle.walk(v["pos_m_sorted"], v["node_head"], v["node_num"], v["node_child"], v["node_nchild"], v["node_com"], v["node_b"], **kw)

    acc = torch.zeros(n, 4, device="cuda")
    amag = torch.zeros(n, device="cuda")
    g.walk_tree(acc, eps=eps, mac_kind=MAC_OPENING_ANGLE, mac_param=0.5, amag_out=amag, r_crit=r_crit)
    aold = amag.cpu().numpy()
    ranges = _group_samples(n)
    # ---- all-active acceleration-MAC walk (the "shared step") ----
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    g.walk_tree(acc, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=dacc, aold=amag, amag_out=amag, r_crit=r_crit, n_interactions=cnt)
    g.check()
    out = acc.cpu().numpy().astype(np.float64)
    for lo, hi in ranges:
        ref, _ = oracle_walk(eps=eps, mac_kind=0, mac_param=dacc, aold=aold, group_range=(lo, hi), r_crit=r_crit)
        _parity(out, ref, _rows_of([(lo, hi)]))
    assert np.all(np.isfinite(out)) and np.all(out[:, 3] < 0)
    m = v["pos_m_sorted"][:, 3].astype(np.float64)
    mom = np.linalg.norm((m[:, None] * out[:, :3]).sum(0)) / (m * np.linalg.norm(out[:, :3], axis=1)).sum()
    assert mom < 2e-3, mom                       # momentum near-conservation (north_star)
    assert 800 < int(cnt.item()) / n < 4000      # interactions per particle at Delta_acc = 2^-9
    gids = _seeded_group_ids(v["pos_m_sorted"], seed=20261105)
    members = np.concatenate([np.arange(gid * G, (gid + 1) * G) for gid in gids])
    _count_equality(g, oracle_walk, gids, members, n, eps=eps, dacc=dacc, aold=aold, r_crit=r_crit, out_full=out)
    # ---- T1: levels bit-exact over all N ----
    level = torch.zeros(n, dtype=torch.uint8, device="cuda")
    active = torch.zeros(n, dtype=torch.int32, device="cuda")
    n_act = torch.zeros(1, dtype=torch.int32, device="cuda")
    info = torch.zeros(2, dtype=torch.int32, device="cuda")
    g.set_timesteps(level, acc_pot=acc, eps=eps, eta=0.5, max_levels=8, emin_nlev_dev=info)
    lev_ref, emin, nlev = oracle.levels(acc.cpu().numpy(), eps, 0.5, 8)
    assert np.array_equal(level.cpu().numpy(), lev_ref) and info.tolist() == [emin, nlev]
    assert 3 <= nlev <= 8
    # ---- T2 + W for every substep of the cycle ----
    aold = amag.cpu().numpy()
    for s in range(1, 2 ** (nlev - 1) + 1):
        g.set_timesteps(level, acc_pot=None, eps=eps, substep=s, active=active, n_active_dev=n_act)
        act_ref = oracle.active_set(lev_ref, s)
        na = int(n_act.item())
        assert na == act_ref.shape[0] and np.array_equal(active[:na].cpu().numpy().view(np.uint32), act_ref)
        if s > 8 and s % 8:
            continue                             # M31-like cycles have up to 128 substeps: walk the first 8 and every 8th
        g.update_moments()
        before = acc.clone()
        g.walk_tree(acc, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=dacc, aold=amag, active=active, n_active_dev=n_act, r_crit=r_crit)
        g.check()
        out = acc.cpu().numpy().astype(np.float64)
        for lo, hi in ranges[:2] + ranges[-1:]:
            ref, _ = oracle_walk(eps=eps, mac_kind=0, mac_param=dacc, aold=aold, active=act_ref, group_range=(lo, hi), r_crit=r_crit)
            rows = _rows_of([(lo, hi)], act_ref)
            if rows.size:
                _parity(out, ref, rows)
        if s in (1, 2, 2 ** (nlev - 1)):          # count equality on seeded groups, incl. the sparsest member masks of this substep
            per_group = np.bincount(act_ref // G, minlength=n // G)
            lonely = np.flatnonzero(per_group == 1)
            rng = np.random.default_rng(100 + s)
            gs = np.unique(np.concatenate([gids, rng.choice(lonely, min(8, lonely.size), replace=False) if lonely.size else gids[:0]]))
            gs = gs[per_group[gs] > 0]
            members = act_ref[np.isin(act_ref // G, gs)]
            if members.size:
                _count_equality(g, oracle_walk, gs, members, n, eps=eps, dacc=dacc, aold=aold, r_crit=r_crit, out_full=out, active=act_ref)
        inactive = torch.ones(n, dtype=torch.bool, device="cuda")
        inactive[active[:na].long()] = False
        assert torch.equal(acc[inactive], before[inactive])     # only active rows are written
    g.close()


def test_sweep_full_size(oracle):
    from gpu_util import gpu_build, gpu_walk, acc_rel_err
    pos, cfg = W.make_config("nfw_2p22_sweep", seed=1)
    n, eps, r_crit = cfg["n"], cfg["eps"], cfg["r_crit"]
    g, v = gpu_build(pos)
    boot, _, aold = gpu_walk(g, n, eps=eps, mac_kind=1, mac_param=0.5, amag=True, count=False, r_crit=r_crit)
    ranges = _group_samples(n, per=32, pieces=4)            # 4 x 32 groups = 4096 particles
    rows = _rows_of(ranges)
    direct = oracle.direct(v["pos_m_sorted"], eps, targets=rows.astype(np.uint32))

    def oracle_walk(**kw):
        return oracle.walk(v["pos_m_sorted"], v["node_head"], v["node_num"], v["node_child"], v["node_nchild"], v["node_com"], v["node_b"], **kw)

    med, inter = [], []
    for e in (1, 5, 9, 13, 17, 20):
        dacc = 2.0 ** -e
        out, cnt, _ = gpu_walk(g, n, eps=eps, mac_kind=0, mac_param=dacc, aold=aold, r_crit=r_crit)
        for lo, hi in ranges:
            ref, _ = oracle_walk(eps=eps, mac_kind=0, mac_param=dacc, aold=aold, group_range=(lo, hi), r_crit=r_crit)
            _parity(out, ref, _rows_of([(lo, hi)]))
        med.append(float(np.median(acc_rel_err(out[rows], direct))))
        inter.append(cnt)
    assert all(b > a for a, b in zip(inter, inter[1:])), inter                 # tighter accuracy opens more cells
    assert all(b < a for a, b in zip(med, med[1:])), med                       # error falls with Delta_acc (Fig. 3)
    assert med[0] > 3e-3 and med[2] < 3e-3 and med[-1] < 1e-4, med             # ~1e-3 at 2^-9, still falling at 2^-20
    # active-fraction sweep at the configured accuracy: random subsets, fixed seed
    for frac in (0.01, 0.1, 0.5):
        active = W.random_active_subset(n, frac, seed=7)
        out, cnt, _ = gpu_walk(g, n, eps=eps, mac_kind=0, mac_param=cfg["delta_acc"], aold=aold, active=active, r_crit=r_crit)
        for lo, hi in ranges:
            ref, _ = oracle_walk(eps=eps, mac_kind=0, mac_param=cfg["delta_acc"], aold=aold, active=active, group_range=(lo, hi), r_crit=r_crit)
            rr = _rows_of([(lo, hi)], active)
            if rr.size:
                _parity(out, ref, rr)
    g.close()
