"""CPU oracle for the GOTHIC hot path: TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
The arithmetic lives in gothic_oracle.cpp (plain C++, cited line by line against PAPER.md); this file is
ctypes/numpy marshalling only.  It imports nothing from paper_1610_07279_b200.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

_lib = None

_u32p = np.ctypeslib.ndpointer(np.uint32, flags="C_CONTIGUOUS")
_u64p = np.ctypeslib.ndpointer(np.uint64, flags="C_CONTIGUOUS")
_u8p = np.ctypeslib.ndpointer(np.uint8, flags="C_CONTIGUOUS")
_f32p = np.ctypeslib.ndpointer(np.float32, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")
_i32p = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.oracle_num_threads.restype = C.c_int
        L.oracle_encode_peano3d.restype = C.c_uint64
        L.oracle_encode_peano3d.argtypes = [C.c_int, C.c_uint64, C.c_uint64, C.c_uint64]
        L.oracle_decode_peano3d.restype = None
        L.oracle_decode_peano3d.argtypes = [C.c_int, C.c_uint64, _u64p]
        L.oracle_morton3d.restype = C.c_uint64
        L.oracle_morton3d.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64]
        L.oracle_root_box.restype = None
        L.oracle_root_box.argtypes = [_f32p, C.c_uint32, _f32p]
        L.oracle_keys.restype = None
        L.oracle_keys.argtypes = [_f32p, C.c_uint32, _f32p, C.c_int, _u64p]
        L.oracle_sort.restype = None
        L.oracle_sort.argtypes = [_u64p, C.c_uint32, _u64p, _u32p]
        L.oracle_build_tree.restype = C.c_int64
        L.oracle_build_tree.argtypes = [_u64p, C.c_uint32, C.c_int, C.c_uint32, _u32p, _u32p, _u32p, _u8p, _u8p, _u32p]
        L.oracle_moments.restype = None
        L.oracle_moments.argtypes = [_f32p, C.c_uint32, _u32p, _u32p, _f32p, _f32p]
        L.oracle_radius.restype = None
        L.oracle_radius.argtypes = [_f32p, C.c_uint32, _u32p, _u32p, _f32p, _f32p]
        L.oracle_levels.restype = None
        L.oracle_levels.argtypes = [_f32p, C.c_uint32, C.c_float, C.c_int, _u8p, _i32p]
        L.oracle_active.restype = C.c_uint32
        L.oracle_active.argtypes = [_u8p, C.c_uint32, C.c_uint32, _u32p]
        L.oracle_direct.restype = None
        L.oracle_direct.argtypes = [_f32p, C.c_uint32, C.c_void_p, C.c_uint32, C.c_double, _f64p]
        L.oracle_walk.restype = None
        L.oracle_b2.restype = None
        L.oracle_b2.argtypes = [_f32p, C.c_uint32, _u32p, _u32p, _f32p, _f32p]
        L.oracle_walk.argtypes = [_f32p, C.c_uint32, _u32p, _u32p, _u32p, _u8p, _f32p, _f32p, C.c_void_p,
                                  C.c_void_p, C.c_uint32, C.c_int, C.c_float, C.c_int, C.c_float, C.c_void_p,
                                  C.c_uint32, C.c_uint32, C.c_float, C.c_int, _f64p, _u64p]
        L.oracle_predict.restype = None
        L.oracle_predict.argtypes = [_f32p, _f32p, _f32p, _u32p, C.c_uint32, C.c_float, C.c_uint32, _f32p]
        L.oracle_correct.restype = None
        L.oracle_correct.argtypes = [_u32p, C.c_uint32, _f32p, _f32p, C.c_uint32, C.c_float, _f32p, _f32p, _f32p, _u32p,
                                     C.c_void_p, C.c_float, C.c_int, C.c_int]
        L.oracle_group_ball.restype = None
        L.oracle_group_ball.argtypes = [_f32p, _u32p, C.c_uint32, C.c_int, _f32p]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def encode_peano3d(nlev: int, x: int, y: int, z: int) -> int:
    return int(lib().oracle_encode_peano3d(nlev, x, y, z))


def decode_peano3d(nlev: int, key: int) -> tuple[int, int, int]:
    out = np.zeros(3, np.uint64)
    lib().oracle_decode_peano3d(nlev, key, out)
    return int(out[0]), int(out[1]), int(out[2])


def morton3d(x: int, y: int, z: int) -> int:
    return int(lib().oracle_morton3d(x, y, z))


def _pos(pos_m) -> np.ndarray:
    a = np.ascontiguousarray(pos_m, dtype=np.float32)
    assert a.ndim == 2 and a.shape[1] == 4
    return a


def root_box(pos_m) -> np.ndarray:
    pos_m = _pos(pos_m)
    box = np.zeros(4, np.float32)
    lib().oracle_root_box(pos_m, pos_m.shape[0], box)
    return box


def keys(pos_m, box, key_kind: int = 0) -> np.ndarray:
    pos_m = _pos(pos_m)
    out = np.zeros(pos_m.shape[0], np.uint64)
    lib().oracle_keys(pos_m, pos_m.shape[0], np.ascontiguousarray(box, np.float32), key_kind, out)
    return out


def sort(key) -> tuple[np.ndarray, np.ndarray]:
    key = np.ascontiguousarray(key, np.uint64)
    ks = np.zeros_like(key)
    perm = np.zeros(key.shape[0], np.uint32)
    lib().oracle_sort(key, key.shape[0], ks, perm)
    return ks, perm


class Tree:
    """Plain container of the canonical tree arrays (O4) and, once computed, the moments (O5)."""

    def __init__(self):
        self.n = 0
        self.n_nodes = 0
        self.box = None
        self.key = None
        self.perm = None
        self.pos_sorted = None
        self.head = self.num = self.child = self.level = self.nchild = self.level_ofs = None
        self.com = self.b = None

    @property
    def n_levels(self) -> int:
        return int(self.level.max()) + 1


def build_tree_from_keys(key_sorted, n_leaf: int = 16, node_cap: int | None = None) -> Tree:
    key_sorted = np.ascontiguousarray(key_sorted, np.uint64)
    n = key_sorted.shape[0]
    cap = int(node_cap) if node_cap is not None else max(2 * n, 64) * 4
    t = Tree()
    head = np.zeros(cap, np.uint32)
    num = np.zeros(cap, np.uint32)
    child = np.zeros(cap, np.uint32)
    level = np.zeros(cap, np.uint8)
    nchild = np.zeros(cap, np.uint8)
    level_ofs = np.zeros(23, np.uint32)
    m = lib().oracle_build_tree(key_sorted, n, n_leaf, cap, head, num, child, level, nchild, level_ofs)
    if m < 0:
        raise OverflowError("oracle_build_tree: node capacity exceeded")
    t.n, t.n_nodes, t.key = n, int(m), key_sorted
    t.head, t.num, t.child, t.level, t.nchild = head[:m].copy(), num[:m].copy(), child[:m].copy(), level[:m].copy(), nchild[:m].copy()
    t.level_ofs = level_ofs
    return t


def moments(pos_sorted, head, num) -> tuple[np.ndarray, np.ndarray]:
    pos_sorted = _pos(pos_sorted)
    m = head.shape[0]
    com = np.zeros((m, 4), np.float32)
    b = np.zeros(m, np.float32)
    lib().oracle_moments(pos_sorted, m, np.ascontiguousarray(head, np.uint32), np.ascontiguousarray(num, np.uint32), com, b)
    return com, b


def radius(pos_sorted, head, num, com) -> np.ndarray:
    """b_J about the given stored centres (second half of O5)."""
    m = head.shape[0]
    b = np.zeros(m, np.float32)
    lib().oracle_radius(_pos(pos_sorted), m, np.ascontiguousarray(head, np.uint32), np.ascontiguousarray(num, np.uint32),
                        np.ascontiguousarray(com, np.float32), b)
    return b


def build_tree(pos_m, key_kind: int = 0, n_leaf: int = 16, node_cap: int | None = None) -> Tree:
    """O1-O5 in order: root box, keys, stable sort, reorder, canonical tree, moments."""
    pos_m = _pos(pos_m)
    box = root_box(pos_m)
    k = keys(pos_m, box, key_kind)
    ks, perm = sort(k)
    t = build_tree_from_keys(ks, n_leaf, node_cap)
    t.box, t.perm = box, perm
    t.pos_sorted = np.ascontiguousarray(pos_m[perm])
    t.com, t.b = moments(t.pos_sorted, t.head, t.num)
    return t


def timestep_constant(eps: float, eta: float) -> np.float32:
    """c = (float)(eta^4 eps^2), formed in double then rounded once (SURVEY.md O7 note)."""
    return np.float32(float(eta) ** 4 * float(eps) ** 2)


def levels(acc_pot, eps: float, eta: float = 0.5, max_levels: int = 8) -> tuple[np.ndarray, int, int]:
    acc_pot = np.ascontiguousarray(acc_pot, np.float32)
    n = acc_pot.shape[0]
    lev = np.zeros(n, np.uint8)
    en = np.zeros(2, np.int32)
    lib().oracle_levels(acc_pot, n, float(timestep_constant(eps, eta)), max_levels, lev, en)
    return lev, int(en[0]), int(en[1])


def active_set(level, substep: int) -> np.ndarray:
    level = np.ascontiguousarray(level, np.uint8)
    out = np.zeros(level.shape[0], np.uint32)
    k = lib().oracle_active(level, level.shape[0], substep, out)
    return out[:k].copy()


def direct(pos_m, eps: float, targets=None) -> np.ndarray:
    """Brute-force eq. 1 in double.  Returns float64 [nt, 4] = (ax, ay, az, Phi)."""
    pos_m = _pos(pos_m)
    n = pos_m.shape[0]
    if targets is None:
        out = np.zeros((n, 4), np.float64)
        lib().oracle_direct(pos_m, n, None, 0, float(eps), out)
    else:
        targets = np.ascontiguousarray(targets, np.uint32)
        out = np.zeros((targets.shape[0], 4), np.float64)
        lib().oracle_direct(pos_m, n, targets.ctypes.data_as(C.c_void_p), targets.shape[0], float(eps), out)
    return out


def b2(pos_sorted, head, num, com) -> np.ndarray:
    """O5b, eq. 4: B_2 about the given stored centres."""
    m = head.shape[0]
    out = np.zeros(m, np.float32)
    lib().oracle_b2(_pos(pos_sorted), m, np.ascontiguousarray(head, np.uint32), np.ascontiguousarray(num, np.uint32),
                    np.ascontiguousarray(com, np.float32), out)
    return out


def walk(pos_sorted, head, num, child, nchild, com, b, *, eps: float, mac_kind: int, mac_param: float,
         aold=None, active=None, group_size: int = 32, group_range=None, r_crit: float = float("inf"), B2=None, ball_kind: int = 0):
    """O7.  Returns (out float64 [n,4] (only active rows written), counts dict).
    r_crit: critical separation of P:122-126 (reading R13); inf = no group splitting."""
    pos_sorted = _pos(pos_sorted)
    n = pos_sorted.shape[0]
    out = np.zeros((n, 4), np.float64)
    counts = np.zeros(4, np.uint64)
    if mac_kind == 0 and aold is None:
        raise ValueError("acceleration MAC needs aold")
    if mac_kind == 2 and B2 is None:
        raise ValueError("multipole MAC needs B2")
    b2_p = None
    if B2 is not None:
        B2 = np.ascontiguousarray(B2, np.float32)
        b2_p = B2.ctypes.data_as(C.c_void_p)
    aold_p = None
    if aold is not None:
        aold = np.ascontiguousarray(aold, np.float32)
        aold_p = aold.ctypes.data_as(C.c_void_p)
    act_p, n_act = None, n
    if active is not None:
        active = np.ascontiguousarray(active, np.uint32)
        act_p, n_act = active.ctypes.data_as(C.c_void_p), active.shape[0]
    n_groups = (n + group_size - 1) // group_size
    g_lo, g_hi = (0, n_groups) if group_range is None else group_range
    lib().oracle_walk(pos_sorted, n,
                      np.ascontiguousarray(head, np.uint32), np.ascontiguousarray(num, np.uint32),
                      np.ascontiguousarray(child, np.uint32), np.ascontiguousarray(nchild, np.uint8),
                      np.ascontiguousarray(com, np.float32), np.ascontiguousarray(b, np.float32), b2_p,
                      act_p, n_act, group_size, float(eps), mac_kind, float(mac_param), aold_p,
                      int(g_lo), int(g_hi), float(r_crit), int(ball_kind), out, counts)
    return out, dict(interactions=int(counts[0]), mac_tests=int(counts[1]), groups=int(counts[2]), list_entries=int(counts[3]))


def walk_tree(t: Tree, **kw):
    if kw.get("mac_kind") == 2 and "B2" not in kw:
        kw["B2"] = b2(t.pos_sorted, t.head, t.num, t.com)
    return walk(t.pos_sorted, t.head, t.num, t.child, t.nchild, t.com, t.b, **kw)


def group_ball(pos_sorted, members, ball_kind: int = 0) -> np.ndarray:
    """(r_I, b_I) as the walk forms it: ball_kind 0 = GEO, 1 = EBS (Ritter), 2 = COM, 3 = CMP, 4 = SEB (smallest enclosing ball), App. B P:568."""
    out = np.zeros(4, np.float32)
    members = np.ascontiguousarray(members, np.uint32)
    lib().oracle_group_ball(_pos(pos_sorted), members, members.shape[0], int(ball_kind), out)
    return out


def predict(pos_m, vel, acc_pot, t_last, t_now: int, dt_unit: float) -> np.ndarray:
    """O8, eq. 15-16: all j-particles to t_now.  Returns pos_pred float32 [n,4]."""
    pos_m = _pos(pos_m)
    n = pos_m.shape[0]
    out = np.zeros((n, 4), np.float32)
    lib().oracle_predict(pos_m, np.ascontiguousarray(vel, np.float32), np.ascontiguousarray(acc_pot, np.float32),
                         np.ascontiguousarray(t_last, np.uint32), int(t_now), float(dt_unit), n, out)
    return out


def correct(active, pos_pred, acc_new, t_now: int, dt_unit: float, pos_m, vel, acc_pot, t_last, level=None,
            eps: float = 0.0, eta: float = 0.5, e_min: int = 0, max_levels: int = 8):
    """O8, eq. 17 for the active i-particles, IN PLACE on pos_m, vel, acc_pot, t_last (and level: reading R15)."""
    for a, dt in ((pos_m, np.float32), (vel, np.float32), (acc_pot, np.float32), (t_last, np.uint32)):
        assert a.dtype == dt and a.flags.c_contiguous
    active = np.ascontiguousarray(active, np.uint32)
    lev_p = None
    if level is not None:
        assert level.dtype == np.uint8 and level.flags.c_contiguous
        lev_p = level.ctypes.data_as(C.c_void_p)
    lib().oracle_correct(active, active.shape[0], np.ascontiguousarray(pos_pred, np.float32), np.ascontiguousarray(acc_new, np.float32),
                         int(t_now), float(dt_unit), pos_m, vel, acc_pot, t_last, lev_p,
                         float(timestep_constant(eps, eta)) if level is not None else 0.0, int(e_min), int(max_levels))
