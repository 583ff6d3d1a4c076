"""CPU-side checks of the boundary: the C-ABI library builds with nvcc for sm_100a, loads, and exports every
symbol include/arc.h declares (no compute calls without a GPU)."""
import ctypes
import re
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def _declared():
    text = (ROOT / "include" / "arc.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(arc_[a-z_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for must in ("arc_create", "arc_step", "arc_stats", "arc_destroy"):
        assert must in names


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2606_21238_b200 import build

    lib = build.build()
    assert lib.exists()
    L = ctypes.CDLL(str(lib))
    for name in _declared():
        assert hasattr(L, name), f"{name} declared in arc.h but not exported"


def test_binding_lists_the_same_names_as_the_header():
    from paper_2606_21238_b200 import arc

    assert sorted(arc.EXPORTS) == _declared()


def test_library_is_sm100a_and_signatures_are_plain_c():
    from paper_2606_21238_b200 import build

    lib = build.build()
    out = subprocess.run(["cuobjdump", "-lelf", str(lib)], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    text = (ROOT / "include" / "arc.h").read_text()
    assert "torch" not in text and "std::" not in text


def test_oracle_and_cuda_path_share_no_code():
    """Neither side includes / imports the other (comments may mention the other side; code may not)."""
    pat_py = re.compile(r"^\s*(from|import)\s+oracle\b|^\s*from\s+\.+\s*oracle|liboracle", re.M)
    pat_c = re.compile(r"#include\s*[\"<][^\">]*oracle", re.M)
    for f in (ROOT / "paper_2606_21238_b200").rglob("*"):
        if f.suffix == ".py":
            assert not pat_py.search(f.read_text()), f
        elif f.suffix in (".cu", ".cuh", ".h"):
            assert not pat_c.search(f.read_text()), f
    assert not pat_c.search((ROOT / "include" / "arc.h").read_text())
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix == ".py":
            assert not re.search(r"^\s*(from|import)\s+paper_2606_21238_b200", f.read_text(), re.M), f
        elif f.suffix == ".cpp":
            assert not re.search(r"#include\s*\"[^\"]*(csrc|arc\.h|\.cuh)", f.read_text()), f
