"""Helpers for the -m gpu parity tests: run the CUDA path through the C-ABI binding and bring results to numpy."""
import numpy as np
import torch


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.view(dtype) if t.element_size() == torch.empty(0, dtype=dtype).element_size() else t.to(dtype)
    return t.cuda()


def view_to_numpy(v: dict) -> dict:
    out = dict(v)
    for k, t in v.items():
        if isinstance(t, torch.Tensor):
            a = t.cpu().numpy()
            if a.dtype == np.int32:
                a = a.view(np.uint32)
            elif a.dtype == np.int64:
                a = a.view(np.uint64)
            out[k] = a
    return out


def gpu_build(pos_m: np.ndarray, key_kind=0, n_leaf=16, group_size=32, node_max=0):
    from paper_1610_07279_b200.binding import Gothic
    g = Gothic(pos_m.shape[0], node_max=node_max, group_size=group_size)
    g.build_tree(dev(pos_m), key_kind=key_kind, n_leaf=n_leaf)
    return g, view_to_numpy(g.get_tree_view())


def gpu_walk(g, n, *, eps, mac_kind, mac_param, aold=None, active=None, count=True, amag=False, n_active_dev=None, r_crit=float("inf")):
    acc = torch.zeros(n, 4, dtype=torch.float32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda") if count else None
    am = torch.zeros(n, dtype=torch.float32, device="cuda") if amag else None
    act = None if active is None else dev(active.astype(np.uint32), torch.int32)
    g.walk_tree(acc, eps=eps, mac_kind=mac_kind, mac_param=mac_param, aold=None if aold is None else dev(aold.astype(np.float32)),
                active=act, n_active_dev=n_active_dev, amag_out=am, n_interactions=cnt, r_crit=r_crit)
    g.check()
    res = acc.cpu().numpy().astype(np.float64)
    return res, (int(cnt.item()) if count else None), (am.cpu().numpy() if amag else None)


def acc_rel_err(out, ref):
    return np.linalg.norm(out[:, :3] - ref[:, :3], axis=1) / np.linalg.norm(ref[:, :3], axis=1)
