"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/demag.h declares (no compute calls without a GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "demag.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(demag_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for want in ("demag_plan_create", "demag_set_kernel", "demag_apply", "demag_energy",
                 "demag_apply_atomistic", "demag_plan_destroy"):
        assert want in names


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2308_08447_b200 import build, binding
    path = build.build()
    lib = ctypes.CDLL(path)
    for name in _declared():
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == _declared()


def test_binding_has_same_names():
    from paper_2308_08447_b200 import binding
    for name in _declared():
        if name != "demag_last_error":
            assert callable(getattr(binding, name)), name


def test_missing_library_fails_loudly(monkeypatch):
    from paper_2308_08447_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", "/nonexistent/libdemag_b200.so")
    monkeypatch.setenv("DEMAG_NO_AUTOBUILD", "1")
    with pytest.raises(ImportError):
        binding.lib()


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2308_08447_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "demag_oracle" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "oracle.py")).read()
    assert "import paper_2308_08447_b200" not in otxt and "from paper_2308_08447_b200" not in otxt


def test_launch_path_headers_do_not_read_the_environment():
    """demag_apply never touches the host environment: the tuning toggles are read in plan.cu at
    plan creation; the kernel and launcher headers hold no getenv."""
    csrc = os.path.join(ROOT, "paper_2308_08447_b200", "csrc")
    for f in os.listdir(csrc):
        if f.endswith(".cuh"):
            assert "getenv" not in open(os.path.join(csrc, f)).read(), f
