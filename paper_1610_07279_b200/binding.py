"""Thin ctypes binding over the C ABI in include/gothic.h: argument marshalling only.

Every function takes torch CUDA tensors (device memory + current stream are PyTorch's job, nothing else)
and passes raw pointers to libgothic_b200.so.  There is no CPU fallback: if the library is missing or a
call fails, a GothicError is raised."""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgothic_b200.so")

KEY_PEANO_HILBERT, KEY_MORTON = 0, 1
MAC_ACCELERATION, MAC_OPENING_ANGLE, MAC_MULTIPOLE = 0, 1, 2
BALL_GEO, BALL_EBS, BALL_COM, BALL_CMP, BALL_SEB = 0, 1, 2, 3, 4

EXPORTS = [
    "gothic_create", "gothic_destroy", "gothic_strerror", "gothic_last_cuda_error", "gothic_build_tree",
    "gothic_update_moments", "gothic_walk_tree", "gothic_set_timesteps", "gothic_get_tree_view", "gothic_check",
    "gothic_gravity_host", "gothic_block_cycle_host", "gothic_launch_count", "gothic_predict", "gothic_correct", "gothic_set_ball",
    "gothic_live_init", "gothic_live_step", "gothic_live_get", "gothic_live_timing", "gothic_active_list_static",
]
STATIC_ACTIVE_MAX_N = 1 << 26     # GOTHIC_STATIC_ACTIVE_MAX_N of include/gothic.h


class GothicError(RuntimeError):
    pass


class TreeViewStruct(C.Structure):
    _fields_ = [("n", C.c_uint32), ("n_nodes", C.c_uint32), ("n_levels_tree", C.c_uint32), ("group_size", C.c_uint32),
                ("box", C.c_float * 4),
                ("key", C.c_void_p), ("perm", C.c_void_p), ("pos_m_sorted", C.c_void_p),
                ("node_head", C.c_void_p), ("node_num", C.c_void_p), ("node_child", C.c_void_p),
                ("node_level", C.c_void_p), ("node_nchild", C.c_void_p), ("level_ofs", C.c_void_p),
                ("node_com", C.c_void_p), ("node_b", C.c_void_p), ("node_b2", C.c_void_p)]


class LiveStateStruct(C.Structure):
    _fields_ = [("n", C.c_uint32), ("t_now", C.c_uint32), ("n_substeps", C.c_uint32), ("e_min", C.c_int32), ("n_levels", C.c_int32),
                ("steps_since_rebuild", C.c_uint32), ("steps", C.c_ulonglong),
                ("pos_m", C.c_void_p), ("vel", C.c_void_p), ("acc_pot", C.c_void_p), ("amag", C.c_void_p), ("t_last", C.c_void_p),
                ("level", C.c_void_p), ("orig", C.c_void_p), ("active", C.c_void_p), ("n_active", C.c_void_p)]


_lib = None


def load_library():
    """Loads libgothic_b200.so (built in-tree by paper_1610_07279_b200.build).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise GothicError(f"{LIB_PATH} not found: run `python -m paper_1610_07279_b200.build` (no CPU fallback exists)")
    L = C.CDLL(LIB_PATH)
    vp, u32, i32, f32 = C.c_void_p, C.c_uint32, C.c_int, C.c_float
    L.gothic_create.restype = i32
    L.gothic_create.argtypes = [C.POINTER(vp), u32, u32, i32, C.c_size_t]
    L.gothic_destroy.restype = None
    L.gothic_destroy.argtypes = [vp]
    L.gothic_strerror.restype = C.c_char_p
    L.gothic_strerror.argtypes = [i32]
    L.gothic_last_cuda_error.restype = C.c_char_p
    L.gothic_last_cuda_error.argtypes = [vp]
    L.gothic_build_tree.restype = i32
    L.gothic_build_tree.argtypes = [vp, vp, u32, i32, i32, vp]
    L.gothic_update_moments.restype = i32
    L.gothic_update_moments.argtypes = [vp, vp, vp]
    L.gothic_walk_tree.restype = i32
    L.gothic_walk_tree.argtypes = [vp, vp, u32, vp, f32, i32, f32, f32, vp, vp, vp, vp, vp]
    L.gothic_set_timesteps.restype = i32
    L.gothic_set_timesteps.argtypes = [vp, vp, u32, f32, f32, i32, u32, vp, vp, vp, vp, vp]
    L.gothic_get_tree_view.restype = i32
    L.gothic_get_tree_view.argtypes = [vp, C.POINTER(TreeViewStruct), vp]
    L.gothic_check.restype = i32
    L.gothic_check.argtypes = [vp, vp]
    L.gothic_gravity_host.restype = i32
    L.gothic_gravity_host.argtypes = [vp, vp, u32, i32, i32, f32, i32, f32, f32, vp, vp, vp, vp]
    L.gothic_block_cycle_host.restype = i32
    L.gothic_block_cycle_host.argtypes = [vp, vp, vp, u32, i32, i32, f32, f32, i32, f32, f32, vp, vp, vp, vp, vp]
    L.gothic_set_ball.restype = i32
    L.gothic_set_ball.argtypes = [vp, i32]
    L.gothic_predict.restype = i32
    L.gothic_predict.argtypes = [vp, vp, vp, vp, vp, u32, f32, u32, vp, vp]
    L.gothic_correct.restype = i32
    L.gothic_correct.argtypes = [vp, vp, u32, vp, u32, vp, vp, u32, f32, vp, vp, vp, vp, vp, f32, f32, i32, i32, vp]
    L.gothic_live_init.restype = i32
    L.gothic_live_init.argtypes = [vp, vp, vp, u32, i32, i32, f32, f32, i32, f32, vp]
    L.gothic_live_step.restype = i32
    L.gothic_live_step.argtypes = [vp, f32, f32, i32, vp, vp]
    L.gothic_live_get.restype = i32
    L.gothic_live_get.argtypes = [vp, C.POINTER(LiveStateStruct)]
    L.gothic_live_timing.restype = i32
    L.gothic_live_timing.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_uint32)]
    L.gothic_active_list_static.restype = i32
    L.gothic_active_list_static.argtypes = [vp, u32, u32, vp, vp, vp]
    L.gothic_launch_count.restype = C.c_ulonglong
    L.gothic_launch_count.argtypes = [vp]
    _lib = L
    return L


def _ptr(t, dtype=None):
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise GothicError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise GothicError(f"expected dtype {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def active_list_static(level: torch.Tensor, substep: int, active: torch.Tensor, n_active_dev: torch.Tensor, n: int | None = None):
    """gothic_active_list_static: the ascending active list of `substep` from the block levels, with no context and no device
    allocation inside the library.  For hosts that cannot cudaMalloc while they run (device memory already committed to their own
    arrays or pool, or no room for cudaMalloc's device-wide synchronisation in the step loop): the scratch is a fixed 128 KiB array in
    the library image, so n <= STATIC_ACTIVE_MAX_N, and calls that may overlap on the GPU must be ordered by the caller.  The
    tensors are the caller's; `n` defaults to len(level) (pass it to exercise the size check without a 2^26 tensor)."""
    L = load_library()
    if not torch.cuda.is_available():
        raise GothicError("no CUDA device: the GOTHIC hot path has no CPU fallback")
    rc = L.gothic_active_list_static(_ptr(level, torch.uint8), int(level.shape[0] if n is None else n), int(substep),
                                     _ptr(active, torch.int32), _ptr(n_active_dev, torch.int32), _stream())
    if rc != 0:
        raise GothicError(f"gothic error {rc}: {L.gothic_strerror(rc).decode()}")


class _DevView:
    """Wraps a raw device pointer so that torch can alias it (__cuda_array_interface__)."""

    def __init__(self, ptr: int, count: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (count,), "typestr": typestr, "data": (int(ptr), False), "version": 2}


_TYPESTR = {torch.int64: "<i8", torch.int32: "<i4", torch.uint8: "|u1", torch.float32: "<f4"}


def _from_ptr(ptr: int, count: int, dtype: torch.dtype, device) -> torch.Tensor:
    """Copies `count` elements of device memory at `ptr` into a new tensor (parity tests only)."""
    if count == 0 or not ptr:
        return torch.empty(count, dtype=dtype, device=device)
    return torch.as_tensor(_DevView(ptr, count, _TYPESTR[dtype]), device=device).clone()


class Gothic:
    """One context = one tree + scratch on the current CUDA device.  Method names follow the C ABI."""

    def __init__(self, n_max: int, node_max: int = 0, group_size: int = 32, scratch_bytes: int = 0):
        self._L = load_library()
        if not torch.cuda.is_available():
            raise GothicError("no CUDA device: the GOTHIC hot path has no CPU fallback")
        self._ctx = C.c_void_p()
        self._chk(self._L.gothic_create(C.byref(self._ctx), n_max, node_max, group_size, scratch_bytes), create=True)
        self.n_max, self.group_size = n_max, group_size or 32
        self.device = torch.device("cuda", torch.cuda.current_device())

    def _chk(self, rc: int, create: bool = False):
        if rc != 0:
            msg = self._L.gothic_strerror(rc).decode()
            if rc == -4 and not create and self._ctx:
                msg += ": " + self._L.gothic_last_cuda_error(self._ctx).decode()
            raise GothicError(f"gothic error {rc}: {msg}")

    def close(self):
        if getattr(self, "_ctx", None):
            self._L.gothic_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the C-ABI calls -----------------------------------------------------------------------------------
    def build_tree(self, pos_m: torch.Tensor, key_kind: int = KEY_PEANO_HILBERT, n_leaf: int = 16):
        self._chk(self._L.gothic_build_tree(self._ctx, _ptr(pos_m, torch.float32), pos_m.shape[0], key_kind, n_leaf, _stream()))

    def update_moments(self, pos_m_sorted: torch.Tensor | None = None):
        self._chk(self._L.gothic_update_moments(self._ctx, _ptr(pos_m_sorted, torch.float32), _stream()))

    def walk_tree(self, acc_pot: torch.Tensor, *, eps: float, mac_kind: int, mac_param: float, aold: torch.Tensor | None = None,
                  active: torch.Tensor | None = None, n_active: int | None = None, n_active_dev: torch.Tensor | None = None,
                  amag_out: torch.Tensor | None = None, n_interactions: torch.Tensor | None = None, r_crit: float = float("inf")):
        na = 0
        if active is not None:
            na = int(active.shape[0] if n_active is None else n_active)
        self._chk(self._L.gothic_walk_tree(self._ctx, _ptr(active, torch.int32) if active is not None else None, na,
                                           _ptr(n_active_dev, torch.int32), float(eps), mac_kind, float(mac_param), float(r_crit),
                                           _ptr(aold, torch.float32), _ptr(acc_pot, torch.float32), _ptr(amag_out, torch.float32),
                                           _ptr(n_interactions, torch.int64), _stream()))

    def set_timesteps(self, level: torch.Tensor, *, acc_pot: torch.Tensor | None, eps: float, eta: float = 0.5, max_levels: int = 8,
                      substep: int = 1, active: torch.Tensor | None = None, n_active_dev: torch.Tensor | None = None,
                      emin_nlev_dev: torch.Tensor | None = None):
        self._chk(self._L.gothic_set_timesteps(self._ctx, _ptr(acc_pot, torch.float32), level.shape[0], float(eps), float(eta),
                                               max_levels, substep, _ptr(level, torch.uint8), _ptr(active, torch.int32),
                                               _ptr(n_active_dev, torch.int32), _ptr(emin_nlev_dev, torch.int32), _stream()))

    def predict(self, pos_m: torch.Tensor, vel: torch.Tensor, acc_pot: torch.Tensor, t_last: torch.Tensor, pos_pred: torch.Tensor, *,
                t_now: int, dt_unit: float):
        self._chk(self._L.gothic_predict(self._ctx, _ptr(pos_m, torch.float32), _ptr(vel, torch.float32), _ptr(acc_pot, torch.float32),
                                         _ptr(t_last, torch.int32), int(t_now), float(dt_unit), pos_m.shape[0], _ptr(pos_pred, torch.float32), _stream()))

    def correct(self, pos_pred: torch.Tensor, acc_new: torch.Tensor, pos_m: torch.Tensor, vel: torch.Tensor, acc_pot: torch.Tensor,
                t_last: torch.Tensor, *, t_now: int, dt_unit: float, active: torch.Tensor | None = None, n_active: int | None = None,
                n_active_dev: torch.Tensor | None = None, level: torch.Tensor | None = None, eps: float = 0.0, eta: float = 0.5,
                e_min: int = 0, max_levels: int = 8):
        na = 0
        if active is not None:
            na = int(active.shape[0] if n_active is None else n_active)
        self._chk(self._L.gothic_correct(self._ctx, _ptr(active, torch.int32) if active is not None else None, na, _ptr(n_active_dev, torch.int32),
                                         pos_m.shape[0], _ptr(pos_pred, torch.float32), _ptr(acc_new, torch.float32), int(t_now), float(dt_unit),
                                         _ptr(pos_m, torch.float32), _ptr(vel, torch.float32), _ptr(acc_pot, torch.float32), _ptr(t_last, torch.int32),
                                         _ptr(level, torch.uint8), float(eps), float(eta), int(e_min), int(max_levels), _stream()))

    def set_ball(self, ball_kind: int):
        self._chk(self._L.gothic_set_ball(self._ctx, int(ball_kind)))

    def check(self):
        self._chk(self._L.gothic_check(self._ctx, _stream()))

    def launch_count(self) -> int:
        return int(self._L.gothic_launch_count(self._ctx))

    def get_tree_view(self) -> dict:
        """Copies of the tree arrays as torch tensors (parity tests; synchronises)."""
        v = TreeViewStruct()
        self._chk(self._L.gothic_get_tree_view(self._ctx, C.byref(v), _stream()))
        torch.cuda.current_stream().synchronize()
        d, n, m = self.device, v.n, v.n_nodes
        return dict(
            n=n, n_nodes=m, n_levels_tree=v.n_levels_tree, group_size=v.group_size, box=[float(x) for x in v.box],
            key=_from_ptr(v.key, n, torch.int64, d), perm=_from_ptr(v.perm, n, torch.int32, d),
            pos_m_sorted=_from_ptr(v.pos_m_sorted, 4 * n, torch.float32, d).view(n, 4),
            node_head=_from_ptr(v.node_head, m, torch.int32, d), node_num=_from_ptr(v.node_num, m, torch.int32, d),
            node_child=_from_ptr(v.node_child, m, torch.int32, d), node_level=_from_ptr(v.node_level, m, torch.uint8, d),
            node_nchild=_from_ptr(v.node_nchild, m, torch.uint8, d), level_ofs=_from_ptr(v.level_ofs, 23, torch.int32, d),
            node_com=_from_ptr(v.node_com, 4 * m, torch.float32, d).view(m, 4), node_b=_from_ptr(v.node_b, m, torch.float32, d), node_b2=_from_ptr(v.node_b2, m, torch.float32, d),
        )

    def live_init(self, pos_m: torch.Tensor, vel: torch.Tensor, *, eps: float, eta: float = 0.5, max_levels: int = 8, theta_boot: float = 0.5,
                  key_kind: int = KEY_PEANO_HILBERT, n_leaf: int = 16):
        """Live block stepping (gothic_live_*): state kept on the device by the library, in tree order."""
        self._chk(self._L.gothic_live_init(self._ctx, _ptr(pos_m, torch.float32), _ptr(vel, torch.float32), pos_m.shape[0], key_kind, n_leaf,
                                           float(eps), float(eta), int(max_levels), float(theta_boot), _stream()))

    def live_step(self, *, delta_acc: float, r_crit: float = float("inf"), rebuild: bool = False, n_interactions: torch.Tensor | None = None):
        self._chk(self._L.gothic_live_step(self._ctx, float(delta_acc), float(r_crit), int(bool(rebuild)), _ptr(n_interactions, torch.int64), _stream()))

    def live_timing(self) -> tuple[float, float, int]:
        """(tree stage ms, active list + walk ms, n_active) of the last live_step, from the step's own CUDA events; waits for that step."""
        ms = (C.c_float * 2)()
        na = C.c_uint32(0)
        self._chk(self._L.gothic_live_timing(self._ctx, ms, C.byref(na)))
        return float(ms[0]), float(ms[1]), int(na.value)

    def live_get(self, arrays: bool | str = True) -> dict:
        """The clock of the live run and (arrays=True) copies of its state rows in tree order (tests, diagnostics); arrays="n_active": only the
        device count of the last step's active list."""
        v = LiveStateStruct()
        self._chk(self._L.gothic_live_get(self._ctx, C.byref(v)))
        d, n = self.device, v.n
        out = dict(n=n, t_now=v.t_now, n_substeps=v.n_substeps, e_min=v.e_min, n_levels=v.n_levels, steps_since_rebuild=v.steps_since_rebuild, steps=v.steps)
        if arrays == "n_active":
            out.update(n_active=_from_ptr(v.n_active, 1, torch.int32, d))
        elif arrays:
            torch.cuda.current_stream().synchronize()
            out.update(pos_m=_from_ptr(v.pos_m, 4 * n, torch.float32, d).view(n, 4), vel=_from_ptr(v.vel, 4 * n, torch.float32, d).view(n, 4),
                       acc_pot=_from_ptr(v.acc_pot, 4 * n, torch.float32, d).view(n, 4), amag=_from_ptr(v.amag, n, torch.float32, d),
                       t_last=_from_ptr(v.t_last, n, torch.int32, d), level=_from_ptr(v.level, n, torch.uint8, d), orig=_from_ptr(v.orig, n, torch.int32, d),
                       active=_from_ptr(v.active, n, torch.int32, d), n_active=_from_ptr(v.n_active, 1, torch.int32, d))
        return out

    def gravity_host(self, pos_m_host: torch.Tensor, acc_pot_host: torch.Tensor, *, eps: float, mac_kind: int, mac_param: float,
                     aold_host: torch.Tensor | None = None, perm_host: torch.Tensor | None = None,
                     key_kind: int = KEY_PEANO_HILBERT, n_leaf: int = 16, r_crit: float = float("inf")):
        """End to end with HOST (pinned) buffers: H2D, build, all-active walk, D2H."""
        for t in (pos_m_host, acc_pot_host, aold_host, perm_host):
            if t is not None and (t.is_cuda or not t.is_contiguous()):
                raise GothicError("gravity_host expects contiguous host tensors")
        hp = lambda t: None if t is None else C.c_void_p(t.data_ptr())
        self._chk(self._L.gothic_gravity_host(self._ctx, hp(pos_m_host), pos_m_host.shape[0], key_kind, n_leaf, float(eps), mac_kind,
                                              float(mac_param), float(r_crit), hp(aold_host), hp(acc_pot_host), hp(perm_host), _stream()))

    def block_cycle_host(self, pos_m_host: torch.Tensor, acc_prev_host: torch.Tensor, acc_pot_host: torch.Tensor, *, eps: float,
                         delta_acc: float, eta: float = 0.5, max_levels: int = 8, level_host: torch.Tensor | None = None,
                         count: bool = False, key_kind: int = KEY_PEANO_HILBERT, n_leaf: int = 16, r_crit: float = float("inf")) -> dict:
        """One full block-step cycle end to end with HOST (pinned) buffers: H2D, build, levels, all substeps, D2H."""
        for t in (pos_m_host, acc_prev_host, acc_pot_host, level_host):
            if t is not None and (t.is_cuda or not t.is_contiguous()):
                raise GothicError("block_cycle_host expects contiguous host tensors")
        hp = lambda t: None if t is None else C.c_void_p(t.data_ptr())
        info = (C.c_int32 * 4)()
        cnt = C.c_ulonglong(0)
        self._chk(self._L.gothic_block_cycle_host(self._ctx, hp(pos_m_host), hp(acc_prev_host), pos_m_host.shape[0], key_kind, n_leaf,
                                                  float(eps), float(eta), max_levels, float(delta_acc), float(r_crit), hp(acc_pot_host), hp(level_host),
                                                  C.cast(info, C.c_void_p), C.cast(C.pointer(cnt), C.c_void_p) if count else None, _stream()))
        return dict(e_min=info[0], n_levels=info[1], n_substeps=info[2], interactions=int(cnt.value) if count else None)
