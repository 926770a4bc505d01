"""-m gpu parity of the LIVE block-stepping path (gothic_live_*; PAPER.md:179-187 with moving particles, level migration and a
rebuild interval; R15): two full block cycles on the GPU against the oracle.

Stage-wise (every step, identical inputs): the oracle is fed the GPU's state BEFORE the step and must reproduce the step's
prediction, tree (on rebuild steps), active list, interaction count, corrected rows, migrated levels and clock bit for bit; only the
walk's accelerations carry the north_star tolerance (fp32 sums, rsqrt.approx).  Free-running: an oracle-only replay from the same
initial conditions (own trees, own moments, fp64 sums) ends within rounding of the GPU's positions and velocities."""
import numpy as np
import pytest
import torch

from paper_1610_07279_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _amag32(a):
    a = a.astype(np.float32)
    return np.sqrt(np.float32(np.float64(a[:, 2]) ** 2 + np.float32(np.float64(a[:, 1]) ** 2 + np.float32(a[:, 0] * a[:, 0]))).astype(np.float32))


def _state(g):
    st = g.live_get()
    out = {k: (v.cpu().numpy() if isinstance(v, torch.Tensor) else v) for k, v in st.items()}
    for k in ("t_last", "orig", "active"):
        out[k] = out[k].view(np.uint32)
    out["active"] = out["active"][: int(out["n_active"][0])]
    return out


# the 2^20 case runs one cycle: the rebuild from predicted positions (nearly sorted input, k_permute_state) at a size where the sort's
# fix-up kernels and full 2048-key event tiles see moved particles
@pytest.mark.parametrize("model,n,every", [("plummer", 6000, 3), ("hernquist", 9001, 1), ("nfw", 8192, 1000), ("nfw", 1 << 20, 2)])
def test_live_steps_stagewise_vs_oracle(oracle, model, n, every):
    from gpu_util import dev, view_to_numpy
    from paper_1610_07279_b200.binding import Gothic
    eps, eta, max_levels, dacc, r_crit = 1.0 / 64, 0.25, 5, 2.0 ** -8, 0.5
    pos = getattr(W, model)(n, seed=3)
    vel = W.isotropic_velocities(pos, model, seed=4)
    g = Gothic(n)
    g.live_init(dev(pos), dev(vel), eps=eps, eta=eta, max_levels=max_levels, theta_boot=0.4)
    st = _state(g)
    t0 = oracle.build_tree(pos)
    assert np.array_equal(st["orig"], t0.perm) and np.array_equal(st["pos_m"], pos[t0.perm]) and np.array_equal(st["vel"], vel[t0.perm])
    boot, _ = oracle.walk_tree(t0, eps=eps, mac_kind=1, mac_param=0.4)
    e = np.linalg.norm(st["acc_pot"][:, :3] - boot[:, :3], axis=1) / np.linalg.norm(boot[:, :3], axis=1)
    assert np.percentile(e, 99.9) < 1e-4 and e.max() < 1e-2
    lev, e_min, nlev = oracle.levels(st["acc_pot"], eps, eta, max_levels)
    assert np.array_equal(st["level"], lev) and (st["e_min"], st["n_levels"], st["n_substeps"], st["t_now"]) == (e_min, nlev, 2 ** (nlev - 1), 0)
    assert np.all(st["t_last"] == 0) and np.array_equal(st["amag"], _amag32(st["acc_pot"]))
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    seen_migration = False
    steps = 0
    for cycle in range(2 if n < (1 << 18) else 1):
        for _ in range(st["n_substeps"]):
            prev, t, unit = st, st["t_now"] + 1, 2.0 ** st["e_min"]
            rebuild = steps % every == every - 1
            before = int(cnt.item())
            g.live_step(delta_acc=dacc, r_crit=r_crit, rebuild=rebuild, n_interactions=cnt)
            g.check()
            st = _state(g)
            steps += 1
            # prediction (eq. 15-16) of all particles, and the tree it went into
            pred = oracle.predict(prev["pos_m"], prev["vel"], prev["acc_pot"], prev["t_last"], t, unit)
            rows = {k: prev[k].copy() for k in ("pos_m", "vel", "acc_pot", "amag", "t_last", "level", "orig")}
            v = view_to_numpy(g.get_tree_view())
            if rebuild:
                tr = oracle.build_tree(pred)
                for k in rows:
                    rows[k] = rows[k][tr.perm]
                pred = pred[tr.perm]
                assert np.array_equal(st["orig"], rows["orig"])
                assert np.array_equal(v["node_head"], tr.head) and np.array_equal(v["node_child"], tr.child) and np.array_equal(v["key"], tr.key)
                assert st["steps_since_rebuild"] == 0
            assert np.array_equal(v["pos_m_sorted"], pred)
            # active list of the substep from the (re-ordered) levels
            act = oracle.active_set(rows["level"], t)
            assert np.array_equal(st["active"], act)
            # the walk: counts equal on the GPU's moments, accelerations within tolerance
            ref, c = oracle.walk(v["pos_m_sorted"], v["node_head"], v["node_num"], v["node_child"], v["node_nchild"], v["node_com"], v["node_b"],
                                 eps=eps, mac_kind=0, mac_param=dacc, aold=rows["amag"], active=act, r_crit=r_crit)
            assert int(cnt.item()) - before == c["interactions"]
            acc_new = st["acc_pot"]
            e = np.linalg.norm(acc_new[act, :3] - ref[act, :3], axis=1) / np.linalg.norm(ref[act, :3], axis=1)
            assert np.percentile(e, 99.9) < 1e-4 and e.max() < 1e-2
            # the corrector (eq. 17) and the level migration (R15) on the GPU's own new accelerations: bit-exact
            oracle.correct(act, pred, acc_new, t, unit, rows["pos_m"], rows["vel"], rows["acc_pot"], rows["t_last"], rows["level"],
                           eps=eps, eta=eta, e_min=prev["e_min"], max_levels=max_levels)
            seen_migration |= bool(np.any(rows["level"] != (prev["level"][tr.perm] if rebuild else prev["level"])))
            rows["amag"][act] = _amag32(acc_new[act])
            if t == prev["n_substeps"]:        # end of the cycle: everybody synchronised, fresh levels, clock back to zero
                assert np.all(rows["t_last"] == t)
                rows["level"], e_min, nlev = oracle.levels(rows["acc_pot"], eps, eta, max_levels)
                rows["t_last"][:] = 0
                assert (st["e_min"], st["n_levels"], st["t_now"]) == (e_min, nlev, 0)
            else:
                assert (st["e_min"], st["n_levels"], st["t_now"]) == (prev["e_min"], prev["n_levels"], t)
            for k in rows:
                assert np.array_equal(st[k], rows[k]), (k, steps)
    assert seen_migration and steps >= 4
    g.close()


def test_live_step_refuses_a_tree_that_is_not_its_own():
    """Another build on the same context between two live steps -- same n, other particles -- ends the live run: the rows no longer belong
    to the tree.  The step returns GOTHIC_ERR_STATE and leaves the clock where it was; gothic_live_init starts a new run."""
    from gpu_util import dev
    from paper_1610_07279_b200.binding import Gothic, GothicError
    n, eps = 4000, 1.0 / 64
    pos = W.plummer(n, seed=21)
    vel = W.isotropic_velocities(pos, "plummer", seed=22)
    g = Gothic(n)
    with pytest.raises(GothicError, match="-2"):
        g.live_step(delta_acc=2.0 ** -8)                     # before gothic_live_init
    g.live_init(dev(pos), dev(vel), eps=eps, eta=0.25, max_levels=4, theta_boot=0.5)
    g.live_step(delta_acc=2.0 ** -8, r_crit=0.5, rebuild=True)       # the run's own rebuild is fine
    g.live_step(delta_acc=2.0 ** -8, r_crit=0.5)
    before = g.live_get(arrays=False)
    assert before["steps"] == 2
    g.build_tree(dev(W.plummer(n, seed=23)))                 # somebody else's tree, same n
    with pytest.raises(GothicError, match="-2"):
        g.live_step(delta_acc=2.0 ** -8, r_crit=0.5)
    after = g.live_get(arrays=False)
    assert (after["t_now"], after["steps"]) == (before["t_now"], before["steps"])
    g.live_init(dev(pos), dev(vel), eps=eps, eta=0.25, max_levels=4, theta_boot=0.5)
    g.live_step(delta_acc=2.0 ** -8, r_crit=0.5)
    g.check()
    assert g.live_get(arrays=False)["steps"] == 1
    g.close()


def test_live_timing_feeds_the_rebuild_tuner():
    """gothic_live_timing returns the last step's stage times and active count; the host-side tuner (eq. 8-12) drives the rebuild flag
    from them.  The rebuild flag changes no result a tree-independent check can see: the active counts of the cycle are those of a run
    with a fixed interval, since levels depend on accelerations only to within the MAC's error -- so only sanity is asserted here."""
    from gpu_util import dev
    from paper_1610_07279_b200.binding import Gothic, GothicError
    from paper_1610_07279_b200.tuner import RebuildTuner
    n, eps = 50000, 1.0 / 64
    pos = W.plummer(n, seed=31)
    vel = W.isotropic_velocities(pos, "plummer", seed=32)
    g = Gothic(n)
    g.live_init(dev(pos), dev(vel), eps=eps, eta=0.25, max_levels=5, theta_boot=0.5)
    with pytest.raises(GothicError, match="-2"):
        g.live_timing()                                       # no step yet
    tuner = RebuildTuner(max_age=6)
    for cycle in range(3):
        st = g.live_get(arrays=False)
        for s in range(st["n_substeps"]):
            rebuild = tuner.want_rebuild(s + 1)
            g.live_step(delta_acc=2.0 ** -8, r_crit=0.5, rebuild=rebuild)
            tree_ms, walk_ms, n_active = g.live_timing()
            assert 0.0 < tree_ms < 1e3 and 0.0 <= walk_ms < 1e3
            assert n_active == int(g.live_get(arrays="n_active")["n_active"].item()) and 0 <= n_active <= n
            assert g.live_get(arrays=False)["steps_since_rebuild"] == (0 if rebuild else tuner.age + 1)
            tuner.observe(s + 1, rebuild, tree_ms, walk_ms, n_active)
        assert n_active == n                                  # the last substep of a cycle has everybody active
    g.check()
    assert tuner.t_make is not None and tuner.t_make >= 0.0
    iv = tuner.intervals()
    assert len(iv) >= 2 and max(iv) <= 6
    g.close()


def test_live_free_running_vs_oracle_only(oracle):
    """Nothing of the CUDA path on the reference side: the oracle integrates the same initial conditions with its own trees, its own
    moments and double-precision sums (tree rebuilt every second step on both sides).  After one full cycle positions and velocities
    agree to rounding growth (1e-5 of the system scale) and the levels of all but a handful of threshold particles are equal."""
    from gpu_util import dev
    from paper_1610_07279_b200.binding import Gothic
    n, eps, eta, max_levels, dacc, r_crit = 5000, 1.0 / 64, 0.25, 5, 2.0 ** -9, 0.5
    pos = W.plummer(n, seed=8)
    vel = W.isotropic_velocities(pos, "plummer", seed=9)
    g = Gothic(n)
    g.live_init(dev(pos), dev(vel), eps=eps, eta=eta, max_levels=max_levels, theta_boot=0.4)
    n_sub = g.live_get()["n_substeps"]
    for s in range(n_sub):
        g.live_step(delta_acc=dacc, r_crit=r_crit, rebuild=(s % 2 == 1))
    g.check()
    st = _state(g)
    # ---- the same in the oracle, rows in the order of its own builds ----
    t = oracle.build_tree(pos)
    orig = t.perm.copy()
    p, v = pos[orig].copy(), vel[orig].copy()
    boot, _ = oracle.walk_tree(t, eps=eps, mac_kind=1, mac_param=0.4)
    a = boot.astype(np.float32)
    amag = _amag32(a)
    lev, e_min, nlev = oracle.levels(a, eps, eta, max_levels)
    assert 2 ** (nlev - 1) == n_sub
    unit = 2.0 ** e_min
    tl = np.zeros(n, np.uint32)
    for s in range(n_sub):
        tn = s + 1
        pred = oracle.predict(p, v, a, tl, tn, unit)
        if s % 2 == 1:
            t = oracle.build_tree(pred)
            p, v, a, amag, tl, lev, orig, pred = p[t.perm], v[t.perm], a[t.perm], amag[t.perm], tl[t.perm], lev[t.perm], orig[t.perm], pred[t.perm]
            com, b = t.com, t.b
        else:
            com = oracle.moments(pred, t.head, t.num)[0]
            b = oracle.radius(pred, t.head, t.num, com)
        act = oracle.active_set(lev, tn)
        out, _ = oracle.walk(pred, t.head, t.num, t.child, t.nchild, com, b, eps=eps, mac_kind=0, mac_param=dacc, aold=amag, active=act, r_crit=r_crit)
        acc_new = out.astype(np.float32)
        p, v, a, tl, lev = p.copy(), v.copy(), a.copy(), tl.copy(), lev.copy()
        oracle.correct(act, pred, acc_new, tn, unit, p, v, a, tl, lev, eps=eps, eta=eta, e_min=e_min, max_levels=max_levels)
        amag[act] = _amag32(acc_new[act])
    # compare by original index
    gp, gv, gl = np.empty_like(st["pos_m"]), np.empty_like(st["vel"]), np.empty_like(st["level"])
    gp[st["orig"]], gv[st["orig"]] = st["pos_m"], st["vel"]
    op, ov = np.empty_like(p), np.empty_like(v)
    op[orig], ov[orig] = p, v
    assert np.abs(gp[:, :3] - op[:, :3]).max() < 1e-5 and np.abs(gv[:, :3] - ov[:, :3]).max() < 1e-4
    lev_new, _, _ = oracle.levels(a, eps, eta, max_levels)
    ol = np.empty_like(lev_new)
    ol[orig] = lev_new
    gl[st["orig"]] = st["level"]
    assert np.mean(gl != ol) < 2e-3
    g.close()
