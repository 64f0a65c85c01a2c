"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads, and exports every symbol
that include/aera_unfold.h declares. No compute calls (no GPU here)."""
import ctypes
import os
import re
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "aera_unfold.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(aera_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported():
    from paper_1507_07733_b200 import build
    lib = ctypes.CDLL(build.build())
    syms = _declared_symbols()
    assert {"aera_pattern_upload", "aera_unfold_batch", "aera_scan_directions"} <= set(syms)
    for s in syms:
        assert hasattr(lib, s), s


def test_binding_mirrors_header():
    import paper_1507_07733_b200.binding as b
    for s in _declared_symbols():
        assert s in b.EXPORTS
        assert hasattr(b, s) or s in ("aera_last_error",), s
    assert b.aera_version().startswith("aera_unfold")
    assert b.aera_launch_count() == 0 or b.aera_launch_count() > 0


def test_library_contains_sm100a_code_and_tma():
    from paper_1507_07733_b200 import build
    lib = build.build()
    out = subprocess.run(["cuobjdump", "-lelf", lib], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True).stdout
    assert "UBLKCP" in sass  # TMA bulk copy staging the pattern-table corner blocks


def test_oracle_and_product_share_no_code():
    """Neither side imports / includes / links the other."""
    imp = re.compile(r"^\s*(from|import)\s+(\S+)", re.M)
    inc = re.compile(r'^\s*#\s*include\s+[<"]([^>"]+)[>"]', re.M)
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1507_07733_b200")):
        if os.path.basename(dirpath) in ("build", "__pycache__"):
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                t = open(os.path.join(dirpath, f)).read()
                assert not any(m.group(2).split(".")[0] == "oracle" for m in imp.finditer(t)), f
                assert not any("oracle" in m.group(1) for m in inc.finditer(t)), f
                assert "liboracle" not in t, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            t = open(os.path.join(ROOT, "oracle", f)).read()
            mods = [m.group(2).split(".")[0] for m in imp.finditer(t)]
            assert "paper_1507_07733_b200" not in mods and "torch" not in mods and "aera_inputs" not in mods, f
            assert not any("aera_unfold" in m.group(1) or "cuda" in m.group(1) for m in inc.finditer(t)), f
            assert "libaera_unfold" not in t, f
