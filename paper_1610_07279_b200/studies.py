"""Parameter studies of SURVEY.md section 8f row 4 on the CUDA path (one JSON line per measurement).

    python -m paper_1610_07279_b200.studies keys      Morton vs Peano-Hilbert ordering: ball radii of the
                                                      i-groups, interactions and walk time
    python -m paper_1610_07279_b200.studies refresh   moments-only refresh vs rebuilding the tree every step (PAPER.md:62,
                                                      :301, :331): interactions and walk time against steps since the build
    python -m paper_1610_07279_b200.studies balls     GEO vs EBS enclosing ball x the three MACs (App. B, Fig. 3-5):
                                                      interactions, walk time and median error at matched parameters

Everything runs through the C-ABI binding; torch is used for device memory and CUDA-event timing only."""
from __future__ import annotations

import argparse
import json

import numpy as np
import torch

from . import workloads as W
from .binding import BALL_CMP, BALL_COM, BALL_EBS, BALL_GEO, BALL_SEB, KEY_MORTON, KEY_PEANO_HILBERT, MAC_ACCELERATION, MAC_MULTIPOLE, MAC_OPENING_ANGLE, Gothic


def _timed(fn, reps=3):
    fn()
    torch.cuda.synchronize()
    best = float("inf")
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        torch.cuda.synchronize()
        best = min(best, a.elapsed_time(b))
    return best


def _walk(g, n, *, eps, mac_kind, mac_param, aold=None, r_crit=float("inf")):
    acc = torch.zeros(n, 4, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    g.walk_tree(acc, eps=eps, mac_kind=mac_kind, mac_param=mac_param, aold=aold, n_interactions=cnt, r_crit=r_crit)
    ms = _timed(lambda: g.walk_tree(acc, eps=eps, mac_kind=mac_kind, mac_param=mac_param, aold=aold, r_crit=r_crit))
    return acc, int(cnt.item()), ms


def _group_radii(pos_sorted: torch.Tensor, G: int = 32) -> np.ndarray:
    """GEO ball radius of every full i-group of the sorted order (host arithmetic on a copy: a diagnostic, not the path)."""
    n = (pos_sorted.shape[0] // G) * G
    p = pos_sorted[:n, :3].double().view(-1, G, 3)
    c = 0.5 * (p.min(1).values + p.max(1).values)
    return (p - c[:, None, :]).norm(dim=2).max(1).values.cpu().numpy()


def study_keys(n: int):
    pos_np, cfg = W.make_config("nfw_2p22_sweep", seed=1, n=n)
    eps, dacc = cfg["eps"], cfg["delta_acc"]
    pos = torch.from_numpy(pos_np).cuda()
    for name, kind in (("peano_hilbert", KEY_PEANO_HILBERT), ("morton", KEY_MORTON)):
        g = Gothic(n)
        build_ms = _timed(lambda: g.build_tree(pos, key_kind=kind))
        v = g.get_tree_view()
        amag = torch.zeros(n, device="cuda")
        acc = torch.zeros(n, 4, device="cuda")
        g.walk_tree(acc, eps=eps, mac_kind=MAC_OPENING_ANGLE, mac_param=0.5, amag_out=amag)
        _, cnt, ms = _walk(g, n, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=dacc, aold=amag, r_crit=cfg["r_crit"])
        _, cnt_u, ms_u = _walk(g, n, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=dacc, aold=amag)      # unsplit groups
        r = _group_radii(v["pos_m_sorted"])
        print(json.dumps({"study": "keys", "key": name, "n": n, "build_ms": build_ms, "n_nodes": v["n_nodes"], "walk_ms": ms, "interactions": cnt,
                          "interactions_per_particle": cnt / n, "r_crit": cfg["r_crit"], "walk_ms_unsplit": ms_u, "interactions_unsplit": cnt_u, "group_ball_radius_median": float(np.median(r)),
                          "group_ball_radius_p99": float(np.percentile(r, 99)), "group_ball_radius_mean": float(r.mean())}), flush=True)
        g.close()


def study_refresh(n: int, steps: int):
    """Plummer sphere with isotropic Gaussian velocities (sigma^2 = -Phi/6), shared step dt = 2^-7 (~1/200 of a crossing time)."""
    pos_np = W.plummer(n, seed=1)
    rng = np.random.default_rng(2)
    r = np.linalg.norm(pos_np[:, :3].astype(np.float64), axis=1)
    vel_np = np.zeros((n, 4), np.float32)
    vel_np[:, :3] = (rng.normal(size=(n, 3)) * np.sqrt(1.0 / (6.0 * np.sqrt(1.0 + r * r)))[:, None]).astype(np.float32)
    eps, dacc, dt, r_crit = 1.0 / 64, 2.0 ** -9, 2.0 ** -7, 0.5
    for mode in ("rebuild_every_step", "moments_only"):
        g = Gothic(n)
        g.build_tree(torch.from_numpy(pos_np).cuda())
        v = g.get_tree_view()
        perm = v["perm"].long()
        pos = v["pos_m_sorted"].clone()
        vel = torch.from_numpy(vel_np).cuda()[perm].contiguous()
        acc = torch.zeros(n, 4, device="cuda")
        amag = torch.zeros(n, device="cuda")
        g.walk_tree(acc, eps=eps, mac_kind=MAC_OPENING_ANGLE, mac_param=0.5, amag_out=amag)
        g.walk_tree(acc, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=dacc, aold=amag, amag_out=amag)
        t_last = torch.zeros(n, dtype=torch.int32, device="cuda")
        pred, acc_new = torch.zeros(n, 4, device="cuda"), torch.zeros(n, 4, device="cuda")
        for step in range(1, steps + 1):
            g.predict(pos, vel, acc, t_last, pred, t_now=step, dt_unit=dt)
            if mode == "rebuild_every_step":
                # re-sort the state into the new tree's order so that it stays aligned with the tree
                g.build_tree(pred)
                p2 = g.get_tree_view()["perm"].long()
                pos, vel, acc, t_last, pred, amag = (x[p2].contiguous() for x in (pos, vel, acc, t_last, pred, amag))
            else:
                g.update_moments(pred)                        # same topology, new positions
            cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
            ms = _timed(lambda: g.walk_tree(acc_new, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=dacc, aold=amag, r_crit=r_crit), reps=2)
            g.walk_tree(acc_new, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=dacc, aold=amag, n_interactions=cnt, r_crit=r_crit)
            g.correct(pred, acc_new, pos, vel, acc, t_last, t_now=step, dt_unit=dt)
            amag = torch.linalg.norm(acc[:, :3], dim=1).contiguous()
            g.check()
            if step in (1, 2, 4, 8, 12, 16, 24, 32, 48, 64) or step == steps:
                print(json.dumps({"study": "refresh", "mode": mode, "n": n, "steps_since_build": step if mode == "moments_only" else 0, "step": step,
                                  "walk_ms": ms, "interactions": int(cnt.item())}), flush=True)
        g.close()


def study_balls(n: int):
    pos_np, cfg = W.make_config("nfw_2p22_sweep", seed=1, n=n)
    eps = cfg["eps"]
    g = Gothic(n)
    g.build_tree(torch.from_numpy(pos_np).cuda())
    amag = torch.zeros(n, device="cuda")
    ref = torch.zeros(n, 4, device="cuda")
    g.walk_tree(ref, eps=eps, mac_kind=MAC_OPENING_ANGLE, mac_param=0.5, amag_out=amag)
    g.walk_tree(ref, eps=eps, mac_kind=MAC_ACCELERATION, mac_param=2.0 ** -22, aold=amag)        # tight walk as the yardstick
    for ball_name, ball in (("GEO", BALL_GEO), ("EBS", BALL_EBS), ("COM", BALL_COM), ("CMP", BALL_CMP), ("SEB", BALL_SEB)):
        g.set_ball(ball)
        for mac_name, mac, params in (("acceleration", MAC_ACCELERATION, [2.0 ** -e for e in (5, 7, 9, 11)]),
                                      ("multipole", MAC_MULTIPOLE, [2.0 ** -e for e in (0, 3, 6, 9)]),
                                      ("opening_angle", MAC_OPENING_ANGLE, [0.9, 0.7, 0.5, 0.3])):
            for prm in params:
                acc, cnt, ms = _walk(g, n, eps=eps, mac_kind=mac, mac_param=prm, aold=amag, r_crit=cfg["r_crit"])
                err = ((acc[:, :3] - ref[:, :3]).norm(dim=1) / ref[:, :3].norm(dim=1))
                print(json.dumps({"study": "balls", "ball": ball_name, "mac": mac_name, "param": prm, "n": n, "walk_ms": ms, "interactions": cnt,
                                  "err_median": float(err.median()), "err_p99": float(err.kthvalue(int(0.99 * n)).values)}), flush=True)
    g.close()


def study_sort(n: int):
    """The library comparison VERDICT r01 asked to state next to B3: torch.sort(stable=True) (CUB's radix sort of 64-bit keys, with 64-bit
    indices as payload) on the workload's own keys in their pre-sort order, against the whole gothic_build_tree (keys + sort + gather +
    nodes + moments) of the same particles.  Context only: nothing of the library links or calls it."""
    pos_np, cfg = W.make_config("nfw_2p24_block", seed=1, n=n)
    g = Gothic(n)
    pos = torch.from_numpy(pos_np).cuda()
    g.build_tree(pos)
    v = g.get_tree_view()
    inv = torch.empty(n, dtype=torch.int64, device="cuda")
    inv[v["perm"].long()] = torch.arange(n, device="cuda")
    keys_unsorted = v["key"][inv].contiguous()              # key of original particle i
    ms_torch = _timed(lambda: torch.sort(keys_unsorted, stable=True), reps=5)
    ms_build = _timed(lambda: g.build_tree(pos), reps=5)
    srt, idx = torch.sort(keys_unsorted, stable=True)
    same = bool(torch.equal(idx.int(), v["perm"])) and bool(torch.equal(srt, v["key"]))
    print(json.dumps({"study": "sort", "n": n, "torch_sort_stable_ms": ms_torch, "gothic_build_tree_ms": ms_build, "same_permutation": same}), flush=True)
    g.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("study", choices=["keys", "refresh", "balls", "sort"])
    ap.add_argument("--n", type=int, default=1 << 22)
    ap.add_argument("--steps", type=int, default=32)
    a = ap.parse_args()
    if a.study == "keys":
        study_keys(a.n)
    elif a.study == "refresh":
        study_refresh(min(a.n, 1 << 20), a.steps)
    elif a.study == "sort":
        study_sort(a.n)
    else:
        study_balls(a.n)


if __name__ == "__main__":
    main()
