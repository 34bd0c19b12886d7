"""CPU-side check of the boundary: libqtt_b200.so builds, loads, and exports every function that
include/qtt.h and include/qtt_diag.h declare (no compute calls without a GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    names = set()
    for h in ("qtt.h", "qtt_diag.h"):
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        for m in re.finditer(r"\b(qtt_\w+)\s*\(", src):
            names.add(m.group(1))
    # typedef'd callback types are not functions
    return names - {"qtt_alloc_fn", "qtt_release_fn"}


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2406_17823_b200 import build, _lib
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    decl = declared_functions()
    assert len(decl) >= 30
    for name in sorted(decl):
        assert hasattr(lib, name), f"{name} declared in include/ but not exported"
    assert decl == set(_lib.PROTOTYPES), (decl ^ set(_lib.PROTOTYPES))


def test_context_creation_fails_loudly_without_gpu():
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2406_17823_b200 as q
    with pytest.raises(RuntimeError):
        q.Context()
