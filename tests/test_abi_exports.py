"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol include/gothic.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "gothic.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gothic_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for must in ("gothic_build_tree", "gothic_walk_tree", "gothic_set_timesteps"):
        assert must in names


def test_library_exports_every_declared_symbol():
    from paper_1610_07279_b200 import build
    lib = ctypes.CDLL(build.build())
    for name in _declared():
        assert hasattr(lib, name), name


def test_binding_lists_same_names_and_fails_loudly_without_gpu():
    import torch
    from paper_1610_07279_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()
    assert binding.load_library().gothic_strerror(-3).decode().startswith("node pool")
    if not torch.cuda.is_available():
        with pytest.raises(binding.GothicError):
            binding.Gothic(128)
        # raw C call without a device must return an error code, not crash or fall back
        ctx = ctypes.c_void_p()
        assert binding.load_library().gothic_create(ctypes.byref(ctx), 128, 0, 32, 0) == -4


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1610_07279_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"import\s+oracle|from\s+oracle|oracle\.|oracle/|libgothic_oracle", text), f
