"""The C-ABI library builds, loads and exports every symbol include/submatrix.h declares
(no compute calls: this runs without a GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_header_symbols():
    from paper_2004_10811_b200 import build, binding
    path = build.build()
    L = ctypes.CDLL(path)
    hdr = open(os.path.join(ROOT, "include", "submatrix.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(sm_[a-z_]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    for name in sorted(declared):
        assert hasattr(L, name), f"{name} declared in submatrix.h but not exported"
    assert declared == set(binding.EXPORTS)


def test_struct_sizes_match_header():
    """ctypes mirrors must have the C layout (sizes checked against a tiny C program)."""
    import subprocess, tempfile
    from paper_2004_10811_b200 import binding as B
    src = '#include <stdio.h>\n#include "submatrix.h"\nint main(){printf("%zu %zu %zu\\n", sizeof(sm_options_t), sizeof(sm_plan_info_t), sizeof(sm_stats_t));return 0;}\n'
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "s.c")
        open(c, "w").write(src)
        exe = os.path.join(d, "s")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe], check=True)
        out = subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()
    assert [int(x) for x in out] == [ctypes.sizeof(B.sm_options_t), ctypes.sizeof(B.sm_plan_info_t),
                                     ctypes.sizeof(B.sm_stats_t)]


def test_strerror_and_missing_library_is_loud(monkeypatch):
    from paper_2004_10811_b200 import binding as B
    assert "structure" in B.sm_strerror(B.SM_ERR_STRUCTURE)
    assert "warning" in B.sm_strerror(B.SM_WARN_MU_NOT_CONVERGED)
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "LIB_PATH", "/nonexistent/libsubmatrix_b200.so")
    try:
        B.lib()
    except RuntimeError as e:
        assert "no CPU fallback" in str(e)
    else:
        raise AssertionError("missing library must raise")
