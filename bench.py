#!/usr/bin/env python
"""bench.py -- whole-hot-path benchmark of the B200-native GOTHIC block-step cycle (driver contract).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME] [--n N]
    python bench.py --workload nfw_2p22_live | plummer_2p20_live | nfw_2p24_live | m31_2p24_live      (live block stepping only, see measure_live)

A "step" is one full block-step CYCLE of the workload (BASELINE.json configs[2], NFW sphere N = 2^24 by default):
    gothic_build_tree                                  (B1-B6: bbox, keys, sort, gather, nodes, moments)
    gothic_set_timesteps(acc)                          (T1: block levels from the current accelerations)
    for substep = 1 .. 2^(n_levels-1):
        gothic_set_timesteps(substep)                  (T2: ascending active list, count stays on the device)
        gothic_update_moments                          (B6 again: the paper recomputes pseudo-j every step)
        gothic_walk_tree(active, |a_old|, Delta_acc)   (W1-W6)
Positions are static (the configs carry no velocities), so the last substep (all particles active) refreshes every
acceleration and the next cycle starts from it.  `value` = interactions of the cycle / device time of the cycle,
inputs resident in HBM.  `e2e` = the same cycle through gothic_block_cycle_host with pinned HOST buffers (H2D of
positions + previous accelerations and D2H of the result inside the timed region).
Interactions are counted in a separate, identical, untimed replay ("in a separate run").

N > 1 (torchrun): the path is single-GPU by design (BASELINE.json north_star: "one GPU only"), so every rank runs an
independent replica (its own seed); no data-path collective; time = max over ranks; value = sum of interactions / time.

After the headline workload, rank 0 of an N = 1 run also times the other BASELINE.json configs (m31_2p24_block, hernquist_2p20,
plummer_2p13 and a reduced grid of the nfw_2p22_sweep: Delta_acc x active fraction) with a few steps each and reports them
under "other_configs" (walk ms, interactions, interactions/s, fraction of the FP32 peak at 24 flop, ms per block step);
--headline-only skips them.

--impl reference: times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample of the same
workload (the walks of every substep of one block cycle on a sample of i-groups; build, levels, moments untimed); rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "tree_walk_interactions_per_s_block_cycle"
UNIT = "interactions/s"
FLOP_PER_INTERACTION = 24          # 20 + rsqrt counted as 4 (the paper's GTX TITAN X convention); 20 and 28 also reported
THETA_BOOTSTRAP = 0.5              # DESIGN.md R7
# dram__bytes_read.sum + dram__bytes_write.sum per k_walk launch (mean over the substep launches of one cycle) is a profiler
# number: it is read from the tracked summary below (which names the commit and the command it was measured with), never
# measured here; null when the file has no entry for the workload
WALK_TRAFFIC_FILE = os.path.join(ROOT, "profiles", "walk_traffic.json")
OTHER_CONFIGS = ["m31_2p24_block", "hernquist_2p20", "plummer_2p13"]
SWEEP_LOG2_DELTA = [1, 5, 9, 13, 20]       # reduced grid of BASELINE.json configs[4]
SWEEP_ACTIVE = [0.01, 0.10, 1.00]
ETA, MAX_LEVELS = 0.5, 8           # BASELINE.json configs[2]


def _walk_traffic(workload: str):
    try:
        with open(WALK_TRAFFIC_FILE) as f:
            d = json.load(f)
        e = d["workloads"].get(workload)
        return (e["bytes_per_launch"], f"profiles/walk_traffic.json (ncu, commit {d['commit']})") if e else (None, None)
    except Exception:
        return None, None


def _peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0, "source": "fallback"}


class ClockSampler:
    """Samples SM clock / throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz, self.power = [], set(), None, []
        self._stop = threading.Event()
        self._t = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index or 0)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown, "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown, "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self._h) / 1000.0)
                r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.05)

    def __enter__(self):
        if self._nv is not None:
            self._t = threading.Thread(target=self._run, daemon=True)
            self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._t is not None:
            self._t.join()

    def summary(self) -> dict:
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "power_w_max": max(self.power) if self.power else None, "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------------------
REFERENCE_SCOPE = ("the walks (W1-W6) of every substep of one block cycle on a sample of i-groups, fp64 accumulation; the oracle's tree build, "
                   "levels, active lists and moments are not in the timed region (the GPU arm's cycle includes them); not like for like")


def _sample_ranges(n_groups: int, want: int, pieces: int):
    want = max(pieces, min(want, n_groups))
    per = max(1, want // pieces)
    out = []
    for k in range(pieces):
        lo = min(n_groups - per, (n_groups * k) // pieces)
        lo = max(lo, out[-1][1] if out else 0)
        hi = min(n_groups, lo + per)
        if hi > lo:
            out.append((lo, hi))
    return out


def oracle_bootstrap(oracle, tree, cfg):
    """|a_old| and the block levels of the FULL particle set from the oracle's own opening-angle bootstrap (R7, R6), so that a
    sample of i-groups sees the same cycle (finest level, number of substeps) as the whole system does.  Untimed set-up.
    Returns (aold, level or None, n_substeps)."""
    n, eps = cfg["n"], cfg["eps"]
    o, _ = oracle.walk_tree(tree, eps=eps, mac_kind=1, mac_param=THETA_BOOTSTRAP)
    aold = np.linalg.norm(o[:, :3], axis=1).astype(np.float32)
    if not cfg["block"]:
        return aold, None, 1
    lev, _, n_lev = oracle.levels(o.astype(np.float32), eps, ETA, MAX_LEVELS)
    return aold, lev, 1 << (n_lev - 1)


def oracle_cycle_sample(oracle, tree, cfg, r_crit: float, ranges, boot, G: int = 32):
    """The oracle's share of one step on the sampled i-groups: step() = the acceleration-MAC walk of every substep's active set among
    the sampled particles, levels and |a_old| taken from the full set's bootstrap (`boot` = oracle_bootstrap's result).
    Returns (step, n_substeps); step() returns the interactions it evaluated."""
    n, eps, dacc = cfg["n"], cfg["eps"], cfg["delta_acc"]
    aold, lev_all, n_sub = boot
    actives = [None]
    if cfg["block"]:
        sel = np.concatenate([np.arange(lo * G, min(n, hi * G), dtype=np.uint32) for lo, hi in ranges])
        lev = lev_all[sel]
        actives = []
        for s in range(1, n_sub + 1):
            ctz = (s & -s).bit_length() - 1
            actives.append(np.ascontiguousarray(sel[lev <= ctz]))

    def step():
        cnt = 0
        for act in actives:
            if act is not None and act.size == 0:
                continue
            for lo, hi in ranges:
                _, c = oracle.walk_tree(tree, eps=eps, mac_kind=0, mac_param=dacc, aold=aold, active=act, group_range=(lo, hi), r_crit=r_crit)
                cnt += c["interactions"]
        return cnt
    return step, len(actives)


def run_reference(args, rank: int, world: int):
    """The CPU oracle, as it stands, on the host cores: a bounded sample of the workload's block cycle."""
    if rank != 0:
        return
    import oracle
    from paper_1610_07279_b200 import workloads as W
    t0 = time.time()
    if args.workload.endswith("_live"):      # the live workloads' spheres at their initial positions: the oracle walks one block cycle's active sets
        pos, _, cfg = W.make_live_config(args.workload, seed=args.seed, n=args.n)
        cfg["block"] = True
    else:
        pos, cfg = W.make_config(args.workload, seed=args.seed, n=args.n)
    n, eps, dacc = cfg["n"], cfg["eps"], cfg["delta_acc"]
    r_crit = cfg["r_crit"] if args.r_crit is None else args.r_crit
    t_gen = time.time() - t0
    t0 = time.time()
    tree = oracle.build_tree(pos)
    t_build = time.time() - t0
    n_groups = (n + 31) // 32
    cores = oracle.num_threads()
    ranges = _sample_ranges(n_groups, args.ref_groups, 8)
    t0 = time.time()
    boot = oracle_bootstrap(oracle, tree, cfg)
    t_boot = time.time() - t0
    step, n_sub = oracle_cycle_sample(oracle, tree, cfg, r_crit, ranges, boot)
    for _ in range(args.warmup):
        step()
    t0 = time.time()
    inter = 0
    for _ in range(args.steps):
        inter += step()
    dt = time.time() - t0
    val = inter / dt
    sample = (f"{sum(hi - lo for lo, hi in ranges)} of {n_groups} i-groups (8 evenly spaced runs), all {n_sub} substeps of the block cycle, "
              f"levels and |a_old| from the oracle's bootstrap of all {n} particles, fp64 accumulation, {inter // max(args.steps, 1)} interactions per step; "
              f"oracle tree build {t_build:.1f} s and bootstrap {t_boot:.1f} s (untimed)")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": args.workload, "n": n, "eps": eps, "delta_acc": dacc, "r_crit": r_crit, "seed": args.seed},
            "reference_scope": REFERENCE_SCOPE,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "setup_s": {"generate": t_gen, "oracle_build": t_build, "oracle_bootstrap": t_boot}}
    print(json.dumps(line), flush=True)


def cpu_baseline(pos, cfg, r_crit: float, budget_s: float = 15.0) -> dict:
    """Oracle walks (fp64 sum, OpenMP over groups) of one block cycle on a sample of i-groups sized to ~budget_s."""
    import oracle
    n = cfg["n"]
    t0 = time.time()
    tree = oracle.build_tree(pos)
    t_build = time.time() - t0
    n_groups = (n + 31) // 32
    cores = oracle.num_threads()
    t0 = time.time()
    boot = oracle_bootstrap(oracle, tree, cfg)
    t_boot = time.time() - t0

    def run(ranges):
        step, n_sub = oracle_cycle_sample(oracle, tree, cfg, r_crit, ranges, boot)
        t0 = time.time()
        cnt = step()
        return cnt, time.time() - t0, n_sub

    probe = _sample_ranges(n_groups, 64 * cores, 8)
    t0 = time.time()
    cnt, dt, n_sub = run(probe)
    t_probe = time.time() - t0
    want = int(sum(hi - lo for lo, hi in probe) * budget_s / max(t_probe, 1e-3))
    ranges = _sample_ranges(n_groups, want, 8)
    cnt, dt, n_sub = run(ranges)
    ng = sum(hi - lo for lo, hi in ranges)
    return {"value": cnt / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{ng} of {n_groups} i-groups (8 evenly spaced runs), all {n_sub} substeps of the block cycle (levels and |a_old| from the oracle's bootstrap of "
                      f"all {n} particles), fp64 accumulation, {cnt} interactions in {dt:.2f} s; oracle tree build at full N took {t_build:.1f} s, the bootstrap "
                      f"{t_boot:.1f} s (not in the rate)",
            "scope": REFERENCE_SCOPE}


# ------------------------------------------------------------------------------------------------------------
def aggregate_over_ranks(dist, times_ms, counts, device):
    """Replicas only: no data-path collective.  The job's time is the MAX over ranks of each device time,
    its work the SUM over ranks of each count.  `dist` is torch.distributed (any backend) or None for one rank."""
    import torch
    t_all = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    i_all = torch.tensor(list(counts), dtype=torch.int64, device=device)
    if dist is not None:
        dist.all_reduce(t_all, op=dist.ReduceOp.MAX)
        dist.all_reduce(i_all, op=dist.ReduceOp.SUM)
    return [float(x) for x in t_all.tolist()], [int(x) for x in i_all.tolist()]


def measure_cycle(torch, W, B, workload: str, *, seed: int, n, r_crit, steps: int, warmup: int, dev, barrier, clock_index=None, with_e2e: bool = True):
    """Times `steps` block cycles of one workload on the current device (after `warmup` untimed ones) and replays them untimed with
    the interaction counter on.  Returns a dict of raw measurements of this rank."""
    pos_np, cfg = W.make_config(workload, seed=seed, n=n)
    n, eps, dacc = cfg["n"], cfg["eps"], cfg["delta_acc"]
    block, G = cfg["block"], cfg["group_size"]
    r_crit = cfg["r_crit"] if r_crit is None else r_crit

    g = B.Gothic(n, group_size=G)
    pos_host = torch.from_numpy(pos_np).pin_memory()
    pos = pos_host.to(dev, non_blocking=True)
    acc = torch.zeros(n, 4, dtype=torch.float32, device=dev)
    amag = torch.zeros(n, dtype=torch.float32, device=dev)
    level = torch.zeros(n, dtype=torch.uint8, device=dev)
    active = torch.zeros(n, dtype=torch.int32, device=dev)
    n_act = torch.zeros(1, dtype=torch.int32, device=dev)
    emin_nlev = torch.zeros(2, dtype=torch.int32, device=dev)

    # ---- untimed bootstrap (R7): opening-angle walk -> |a_old|, then one acceleration-MAC walk -------------
    g.build_tree(pos)
    g.walk_tree(acc, eps=eps, mac_kind=B.MAC_OPENING_ANGLE, mac_param=THETA_BOOTSTRAP, amag_out=amag, r_crit=r_crit)
    g.walk_tree(acc, eps=eps, mac_kind=B.MAC_ACCELERATION, mac_param=dacc, aold=amag, amag_out=amag, r_crit=r_crit)
    if block:
        g.set_timesteps(level, acc_pot=acc, eps=eps, eta=ETA, max_levels=MAX_LEVELS, emin_nlev_dev=emin_nlev)
        g.check()
        e_min, n_levels = (int(x) for x in emin_nlev.tolist())
    else:
        e_min, n_levels = 0, 1
    n_sub = 1 << (n_levels - 1)

    stage_names = ["build", "levels", "active", "moments", "walk"]

    def cycle(ev=None, counts=None):
        """One step.  ev: optional list collecting (stage, start_event, stop_event); counts: per-substep interaction tensor."""
        def timed(name, fn):
            if ev is None:
                fn()
                return
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            ev.append((name, a, b))
        timed("build", lambda: g.build_tree(pos))
        if block:
            timed("levels", lambda: g.set_timesteps(level, acc_pot=acc, eps=eps, eta=ETA, max_levels=MAX_LEVELS, emin_nlev_dev=emin_nlev))
        for s in range(1, n_sub + 1):
            if block:
                timed("active", lambda: g.set_timesteps(level, acc_pot=None, eps=eps, substep=s, active=active, n_active_dev=n_act))
                timed("moments", lambda: g.update_moments())
                timed("walk", lambda: g.walk_tree(acc, eps=eps, mac_kind=B.MAC_ACCELERATION, mac_param=dacc, aold=amag, active=active,
                                                   n_active_dev=n_act, amag_out=amag, r_crit=r_crit,
                                                   n_interactions=None if counts is None else counts[s - 1:s]))
            else:
                timed("walk", lambda: g.walk_tree(acc, eps=eps, mac_kind=B.MAC_ACCELERATION, mac_param=dacc, aold=amag, amag_out=amag, r_crit=r_crit,
                                                   n_interactions=None if counts is None else counts[s - 1:s]))

    for _ in range(warmup):
        cycle()
        g.check()       # the traversal-stack flag is sticky: one check validates every walk of the cycle
    snap = (acc.clone(), amag.clone(), level.clone())

    # ---- timed region: exactly K steps -------------------------------------------------------------------------------
    launches0 = g.launch_count()
    ev = []
    t_start, t_stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with ClockSampler(clock_index) as clk:
        t_start.record()
        for _ in range(steps):
            cycle(ev)
        t_stop.record()
        barrier()
    total_ms = t_start.elapsed_time(t_stop)
    launches = g.launch_count() - launches0
    g.check()
    if block:
        assert int(emin_nlev[1].item()) == n_levels, "the number of block levels changed between cycles"
    stage_ms = {k: 0.0 for k in stage_names}
    walk_ms_sub = np.zeros(n_sub)
    wi = 0
    for name, a, b in ev:
        ms = a.elapsed_time(b)
        stage_ms[name] += ms
        if name == "walk":
            walk_ms_sub[wi % n_sub] += ms
            wi += 1

    # ---- identical untimed replay with the interaction counter on ----------------------------------------------
    acc.copy_(snap[0]); amag.copy_(snap[1]); level.copy_(snap[2])
    counts = torch.zeros(n_sub, dtype=torch.int64, device=dev)
    act_counts = np.zeros(n_sub, np.int64)
    inter_sub = np.zeros(n_sub, np.int64)
    for _ in range(steps):
        counts.zero_()
        cycle(None, counts)
        g.check()
        inter_sub += counts.cpu().numpy()
    if block:   # active counts per substep (same every cycle: levels are recomputed from converged accelerations)
        for s in range(1, n_sub + 1):
            g.set_timesteps(level, acc_pot=None, eps=eps, substep=s, active=active, n_active_dev=n_act)
            act_counts[s - 1] = int(n_act.item())
    else:
        act_counts[:] = n

    # ---- e2e: same cycle through the host-buffer C-ABI call ---------------------------------------------------------------
    e2e = None
    if with_e2e and block:
        k_e2e = max(1, min(steps, 3))
        acc_prev_sorted = snap[0]
        perm = g.get_tree_view()["perm"].long()
        acc_prev_orig = torch.empty_like(acc_prev_sorted)
        acc_prev_orig[perm] = acc_prev_sorted
        h_prev = acc_prev_orig.cpu().pin_memory()
        h_prev0 = h_prev.clone().pin_memory()
        h_out = torch.empty(n, 4, dtype=torch.float32).pin_memory()
        h_lev = torch.empty(n, dtype=torch.uint8).pin_memory()
        del acc_prev_orig, perm
        kw = dict(eps=eps, delta_acc=dacc, eta=ETA, max_levels=MAX_LEVELS, level_host=h_lev, r_crit=r_crit)
        g.block_cycle_host(pos_host, h_prev, h_out, **kw)   # warm-up
        h_prev.copy_(h_prev0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        t0 = time.perf_counter()
        e0.record()
        a, b = h_prev, h_out
        for _ in range(k_e2e):
            g.block_cycle_host(pos_host, a, b, **kw)
            a, b = b, a
        e1.record()
        barrier()
        e2e_wall_ms = 1e3 * (time.perf_counter() - t0)
        e2e_ms = max(e0.elapsed_time(e1), e2e_wall_ms)     # host-synchronous call: wall clock covers the copies too
        # counted replay
        h_prev.copy_(h_prev0)
        a, b, e2e_inter = h_prev, h_out, 0
        for _ in range(k_e2e):
            info = g.block_cycle_host(pos_host, a, b, count=True, **kw)
            e2e_inter += info["interactions"]
            a, b = b, a
        e2e = {"ms": e2e_ms, "steps": k_e2e, "interactions": e2e_inter, "h2d": 2 * n * 16, "d2h": n * 16 + n}
    g.close()
    return {"cfg": cfg, "pos_np": pos_np, "n": n, "r_crit": r_crit, "n_levels": n_levels, "n_sub": n_sub, "steps": steps, "total_ms": total_ms,
            "stage_ms": stage_ms, "walk_ms_sub": walk_ms_sub, "walk_launches": wi, "inter_sub": inter_sub, "inter_total": int(inter_sub.sum()),
            "act_counts": act_counts, "launches": int(launches), "e2e": e2e, "clocks": clk.summary()}


def summarise(m: dict, alu_peak: float) -> dict:
    """The per-workload numbers north_star asks for: walk time, interactions/s, TFLOP/s, fraction of the FP32 peak, whole-step time."""
    K, n_sub = m["steps"], m["n_sub"]
    walk_rate = m["inter_total"] / (m["stage_ms"]["walk"] * 1e-3)
    return {"n": m["n"], "r_crit": m["r_crit"], "group_size": m["cfg"]["group_size"], "n_levels": m["n_levels"], "n_substeps": n_sub, "steps": K,
            "ms_per_cycle": m["total_ms"] / K, "ms_per_block_step": m["total_ms"] / K / n_sub,
            "interactions_per_cycle": m["inter_total"] // K, "interactions_per_s_cycle": m["inter_total"] / (m["total_ms"] * 1e-3),
            "walk_ms_per_cycle": m["stage_ms"]["walk"] / K, "walk_interactions_per_s": walk_rate,
            "walk_tflops_24": walk_rate * 24 / 1e12, "walk_frac_fp32_peak_24": walk_rate * FLOP_PER_INTERACTION / 1e12 / alu_peak,
            "all_active_walk_ms": m["walk_ms_sub"][-1] / K, "all_active_interactions": int(m["inter_sub"][-1] // K),
            "stage_ms_per_cycle": {k: v / K for k, v in m["stage_ms"].items()}, "gpu_launches": m["launches"],
            "e2e_ms_per_cycle": m["e2e"]["ms"] / m["e2e"]["steps"] if m["e2e"] else None, "clocks": m["clocks"]}


def measure_sweep(torch, W, B, dev, alu_peak: float, seed: int, reps: int = 3) -> dict:
    """Reduced grid of BASELINE.json configs[4] on the NFW 2^22 sphere: accuracy parameter x active fraction (random subsets, fixed
    seed): walk time (best of `reps`, CUDA events), interactions, interactions/s."""
    pos_np, cfg = W.make_config("nfw_2p22_sweep", seed=seed)
    n, eps, r_crit = cfg["n"], cfg["eps"], cfg["r_crit"]
    g = B.Gothic(n, group_size=cfg["group_size"])
    pos = torch.from_numpy(pos_np).to(dev)
    acc = torch.zeros(n, 4, dtype=torch.float32, device=dev)
    amag = torch.zeros(n, dtype=torch.float32, device=dev)
    cnt = torch.zeros(1, dtype=torch.int64, device=dev)
    g.build_tree(pos)
    g.walk_tree(acc, eps=eps, mac_kind=B.MAC_OPENING_ANGLE, mac_param=THETA_BOOTSTRAP, amag_out=amag, r_crit=r_crit)
    g.walk_tree(acc, eps=eps, mac_kind=B.MAC_ACCELERATION, mac_param=cfg["delta_acc"], aold=amag, amag_out=amag, r_crit=r_crit)
    points = []
    for frac in SWEEP_ACTIVE:
        act = None if frac >= 1.0 else torch.from_numpy(W.random_active_subset(n, frac).astype(np.int32)).to(dev)
        for ld in SWEEP_LOG2_DELTA:
            kw = dict(eps=eps, mac_kind=B.MAC_ACCELERATION, mac_param=2.0 ** -ld, aold=amag, active=act, r_crit=r_crit)
            cnt.zero_()
            g.walk_tree(acc, n_interactions=cnt, **kw)          # warm-up + count
            best = float("inf")
            for _ in range(reps):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                g.walk_tree(acc, **kw)
                b.record()
                torch.cuda.synchronize()
                best = min(best, a.elapsed_time(b))
            ni = int(cnt.item())
            points.append({"log2_delta_acc": -ld, "active_fraction": frac, "n_active": n if act is None else int(act.numel()), "walk_ms": best,
                           "interactions": ni, "interactions_per_s": ni / (best * 1e-3),
                           "frac_fp32_peak_24": ni / (best * 1e-3) * FLOP_PER_INTERACTION / 1e12 / alu_peak})
    g.check()
    g.close()
    return {"n": n, "eps": eps, "r_crit": r_crit, "reps": reps, "timing": "best of reps, CUDA events around gothic_walk_tree (group marking included)", "points": points}


def measure_live(torch, W, B, workload: str, *, seed: int, n, dev, alu_peak: float, intervals=(1, 2, 4, 12, "cycle", "auto"), cycles: int = 2) -> dict:
    """The paper's actual time-to-solution loop with MOVING particles through gothic_live_step: per block
    step predict all -> rebuild (every k-th step) or moments refresh -> active list -> walk -> correct with level migration, state on the
    device in tree order.  For each rebuild interval k: one warm-up cycle, then `cycles` block cycles timed with CUDA events
    (seconds per block step), then one more cycle replayed with the interaction counter read after every step (separate run).
    k = "auto": the rebuild decision of every step comes from paper_1610_07279_b200.tuner.RebuildTuner (eq. 8-12 in the
    form "rebuild when the walk time lost to the tree's age has reached t_make"), fed with the step's own CUDA-event times
    (gothic_live_timing: one event wait and a 4-byte read-back per step, inside the timed region); two warm-up cycles instead of one."""
    from paper_1610_07279_b200.tuner import RebuildTuner
    pos_np, vel_np, cfg = W.make_live_config(workload, seed=seed, n=n)
    n, eps, dacc, r_crit = cfg["n"], cfg["eps"], cfg["delta_acc"], cfg["r_crit"]
    pos, vel = torch.from_numpy(pos_np).to(dev), torch.from_numpy(vel_np).to(dev)
    out = {"workload": workload, "n": n, "eps": eps, "delta_acc": dacc, "r_crit": r_crit, "eta": ETA, "max_levels": MAX_LEVELS, "cycles_timed": cycles,
           "velocities": ("stand-in: Jeans dispersion of the spherically averaged total profile for halo and bulge, circular speed + 15 % dispersion for the disk "
                          "(workloads.m31_velocities)") if cfg["model"] == "m31_like" else "isotropic Gaussian, Jeans dispersion of the truncated profile (workloads.isotropic_velocities)", "rebuild_every": {}}
    for k in intervals:
        g = B.Gothic(n, group_size=cfg["group_size"])
        g.live_init(pos, vel, eps=eps, eta=ETA, max_levels=MAX_LEVELS, theta_boot=THETA_BOOTSTRAP)
        tuner = RebuildTuner() if k == "auto" else None

        def run_cycle(counter=None, log=None):
            st = g.live_get(arrays=False)
            for s in range(st["n_substeps"]):
                if tuner is not None:
                    rebuild = tuner.want_rebuild(s + 1)
                elif k == "cycle":
                    rebuild = s == 0
                else:
                    rebuild = (st["steps"] + s + 1) % k == 0      # the k-th step of every k: with k = 2, 4 the even (populous) substeps get the fresh tree
                g.live_step(delta_acc=dacc, r_crit=r_crit, rebuild=rebuild, n_interactions=counter)
                if tuner is not None:
                    tuner.observe(s + 1, rebuild, *g.live_timing())
                if log is not None:
                    now = g.live_get(arrays="n_active")
                    log.append((s + 1, int(now["steps_since_rebuild"]), int(now["n_active"].item()), int(counter.item())))
            return st["n_substeps"]

        run_cycle()                       # warm-up
        if tuner is not None:
            run_cycle()
        g.check()
        launches0 = g.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        steps = 0
        for _ in range(cycles):
            steps += run_cycle()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        launches = g.launch_count() - launches0
        g.check()
        counter = torch.zeros(1, dtype=torch.int64, device=dev)
        log = []
        n_sub = run_cycle(counter, log)
        g.check()
        inter = [b[3] - a for a, b in zip([0] + [x[3] for x in log[:-1]], log)]
        total = int(counter.item())
        out["rebuild_every"][str(k)] = {
            "sec_per_block_step": ms * 1e-3 / steps, "ms_per_cycle": ms / cycles, "block_steps_timed": steps, "n_substeps_last_cycle": n_sub,
            "interactions_per_cycle": total, "interactions_per_s": total * cycles / (ms * 1e-3) if steps == n_sub * cycles else None,
            "count_from": "replay cycle: the interactions of ONE later, untimed cycle (PAPER.md:331), scaled to the timed cycles; approximate, the particles have moved on",
            "gpu_launches_per_step": launches / steps,
            "steps": [{"substep": a, "steps_since_rebuild": b, "n_active": c, "interactions": i} for (a, b, c, _), i in zip(log, inter)]}
        if tuner is not None:
            out["rebuild_every"][str(k)]["tuner"] = {"rule": "rebuild when the walk time lost since the last rebuild >= t_make (eq. 8-12, PAPER.md:138-175)",
                                                     "t_make_ms": tuner.t_make, "intervals": tuner.intervals()[-32:]}
        g.close()
    return out


def run_ours(args, rank: int, world: int, local_rank: int):
    import torch
    from paper_1610_07279_b200 import workloads as W
    from paper_1610_07279_b200 import binding as B

    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    peaks = _peaks()
    props = torch.cuda.get_device_properties(dev)
    if args.workload.endswith("_live"):
        # live block stepping only: one line whose headline is the run with the tree rebuilt once per block cycle
        alu_peak = props.multi_processor_count * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
        with ClockSampler(local_rank) as clk:
            lv = measure_live(torch, W, B, args.workload, seed=args.seed + rank, n=args.n, dev=dev, alu_peak=alu_peak, cycles=max(1, args.steps))
        head = lv["rebuild_every"]["cycle"]
        (ms_max,), (inter_all,) = aggregate_over_ranks(dist, [head["ms_per_cycle"]], [head["interactions_per_cycle"]], dev)
        if rank == 0:
            print(json.dumps({"metric": METRIC, "value": inter_all / (ms_max * 1e-3), "unit": UNIT, "n_gpus": world, "steps": max(1, args.steps),
                              "warmup": 1, "ms_per_step": ms_max, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                              "data": "synthetic", "config": {"workload": args.workload, "n": lv["n"], "parallelism": "replicas" if world > 1 else "single_gpu"},
                              "sec_per_block_step": head["sec_per_block_step"], "live": lv, "clocks": clk.summary(),
                              "gpu_launches": int(head["gpu_launches_per_step"] * head["block_steps_timed"])}), flush=True)
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return
    m = measure_cycle(torch, W, B, args.workload, seed=args.seed + rank, n=args.n, r_crit=args.r_crit, steps=args.steps, warmup=args.warmup,
                      dev=dev, barrier=barrier, clock_index=local_rank)
    cfg, n, n_sub, n_levels, r_crit = m["cfg"], m["n"], m["n_sub"], m["n_levels"], m["r_crit"]
    eps, dacc = cfg["eps"], cfg["delta_acc"]
    total_ms, stage_ms, e2e, inter_total = m["total_ms"], m["stage_ms"], m["e2e"], m["inter_total"]

    # ---- max over ranks, aggregate ---------------------------------------------------------------------------------------
    (total_ms_max, walk_ms_max, e2e_ms_max), (inter_all, e2e_inter_all) = aggregate_over_ranks(
        dist, [total_ms, stage_ms["walk"], e2e["ms"] if e2e else 0.0], [inter_total, e2e["interactions"] if e2e else 0], dev)

    if rank == 0:
        K = args.steps
        value = inter_all / (total_ms_max * 1e-3)
        walk_rate = inter_total / (stage_ms["walk"] * 1e-3)            # this rank's walk stage
        alu_peak = props.multi_processor_count * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12      # TFLOP/s, DESIGN.md "Rooflines"
        achieved = walk_rate * FLOP_PER_INTERACTION / 1e12
        traffic, traffic_src = _walk_traffic(args.workload) if args.n is None else (None, None)
        # per particle: 309 B with the method's eight LSD passes (8 x 24 B); as run the sort is five passes + the fix-up scan (5 x 24 + 12 B): 249 B
        build_bytes_8pass = n * 309 + 0.24 * n * 150
        build_bytes = n * 249 + 0.24 * n * 150
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": total_ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": args.workload, "n": n, "eps": eps, "delta_acc": dacc, "r_crit": r_crit,
                       "r_crit_choice": "fixed per workload from a coarse sweep of the all-active walk time on a B200 (the paper auto-tunes it at run time, "
                                        "PAPER.md:122-126); see DESIGN.md section 7",
                       "eta": ETA, "max_levels": MAX_LEVELS, "seed": args.seed,
                       "group_size": cfg["group_size"], "n_leaf": 16, "key": "peano_hilbert", "n_levels": n_levels, "n_substeps": n_sub,
                       "parallelism": "replicas" if world > 1 else "single_gpu", "l2": "inputs_exceed_l2" if n * 16 > 126e6 else "inputs_fit_l2"},
            "sec_per_block_step": total_ms_max * 1e-3 / K / n_sub,
            # the same with the tree build amortised three ways: rebuilt every block step, every 12 (the paper's
            # measured mean interval), once per cycle (what the timed region did)
            "sec_per_block_step_rebuild_every": {
                "1": ((total_ms_max - stage_ms["build"]) / K / n_sub + stage_ms["build"] / K) * 1e-3,
                "12": ((total_ms_max - stage_ms["build"]) / K / n_sub + stage_ms["build"] / K / 12.0) * 1e-3,
                "cycle": total_ms_max * 1e-3 / K / n_sub},
            "interactions_per_cycle": inter_total // K,
            "stage_ms_per_cycle": {k: v / K for k, v in stage_ms.items()},
            "substeps": [{"substep": s + 1, "n_active": int(m["act_counts"][s]), "interactions": int(m["inter_sub"][s] // K),
                          "walk_ms": m["walk_ms_sub"][s] / K,
                          "interactions_per_s": float(m["inter_sub"][s] / max(m["walk_ms_sub"][s], 1e-9) * 1e3)} for s in range(n_sub)],
            "walk": {"interactions_per_s": walk_rate, "tflops_20": walk_rate * 20 / 1e12, "tflops_24": walk_rate * 24 / 1e12,
                     "tflops_28": walk_rate * 28 / 1e12, "frac_fp32_peak_24": achieved / alu_peak},
            "roofline": {"kernel": "k_walk", "bound": "alu", "achieved": achieved, "peak": alu_peak, "unit": "TFLOP/s", "frac": achieved / alu_peak,
                         "traffic": traffic, "traffic_unit": "bytes/launch", "traffic_source": traffic_src,
                         "flop_per_interaction": FLOP_PER_INTERACTION,
                         "avg_launch_ms": stage_ms["walk"] / max(m["walk_launches"], 1),
                         "peak_source": f"derived: {props.multi_processor_count} SM x 128 FP32 lanes x 2 flop x {peaks['sm_max_mhz']:.0f} MHz "
                                        f"(clock from MEASURED_PEAKS.json, {peaks['source']})"},
            # the HBM-bound part: algorithmic bytes of one build (bbox 16, keys 16 + 8, histogram 8, sort passes x 2 x 12,
            # gather 4 + 16 + 16, node events 2 x 8 B per particle; moments 16 + 16 + 4 + 1 B per particle and ~150 B per node); `frac` counts the
            # five sort passes + fix-up scan that run, `frac_8pass` what the same build would move with the plain eight-pass LSD sort
            "build_roofline": {"bound": "hbm", "achieved": build_bytes / (stage_ms["build"] / K * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
                               "unit": "GB/s", "frac": build_bytes / (stage_ms["build"] / K * 1e-3) / 1e9 / peaks["hbm_gbs"],
                               "bytes_per_particle": 249, "sort": "as run: 5 one-sweep passes + fix-up scan",
                               "frac_8pass": build_bytes_8pass / (stage_ms["build"] / K * 1e-3) / 1e9 / peaks["hbm_gbs"],
                               "ms": stage_ms["build"] / K, "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peaks['source']})"},
            "clocks": m["clocks"],
            "gpu_launches": m["launches"],
            "e2e": None,
        }
        if e2e:
            line["e2e"] = {"value": e2e_inter_all / (e2e_ms_max * 1e-3), "unit": UNIT, "h2d_bytes_per_step": e2e["h2d"],
                           "d2h_bytes_per_step": e2e["d2h"], "ms_per_step": e2e_ms_max / e2e["steps"], "steps": e2e["steps"]}
        if world == 1 and not args.headline_only:
            # the other BASELINE.json configs, a few steps each (north_star: "throughput on the synthetic models below")
            others = {}
            for name in OTHER_CONFIGS:
                if name == args.workload:
                    continue
                mo = measure_cycle(torch, W, B, name, seed=args.seed, n=None, r_crit=None, steps=args.other_steps, warmup=3, dev=dev,
                                   barrier=barrier, clock_index=local_rank, with_e2e=False)
                others[name] = summarise(mo, alu_peak)
                del mo
            others["nfw_2p22_sweep"] = measure_sweep(torch, W, B, dev, alu_peak, args.seed)
            line["other_configs"] = others
            # the same sphere with moving particles: predict -> rebuild / refresh -> walk -> correct (gothic_live_step), SURVEY.md 8f row 1
            line["live"] = measure_live(torch, W, B, "nfw_2p24_live", seed=args.seed, n=None, dev=dev, alu_peak=alu_peak, intervals=(1, 2, 4, "cycle", "auto"), cycles=2)
            # and the paper's headline model, 64 substeps per cycle: where the fixed per-step costs weigh most
            line["live_m31"] = measure_live(torch, W, B, "m31_2p24_live", seed=args.seed, n=None, dev=dev, alu_peak=alu_peak, intervals=(1, 2, 4, "auto"), cycles=1)
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(m["pos_np"], cfg, r_crit, args.cpu_budget)
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="nfw_2p24_block")
    ap.add_argument("--n", type=int, default=None, help="override N (debugging; the reported config then says so)")
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--r-crit", type=float, default=None, help="override the workload's critical separation (PAPER.md:122-126); inf = no group splitting")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--headline-only", action="store_true", help="skip the other BASELINE.json configs (other_configs)")
    ap.add_argument("--other-steps", type=int, default=2, help="timed cycles of each of the other configs")
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--ref-groups", type=int, default=65536, help="i-groups per step of the --impl reference sample")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
