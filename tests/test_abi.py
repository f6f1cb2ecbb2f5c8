"""Host-side checks of the C-ABI boundary (no GPU): the library builds, loads, and exports every
symbol include/nh_b200.h declares; the ctypes structs mirror the C structs; the product package
does not import the oracle (and vice versa)."""
import ctypes as C
import os
import re
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HDR = os.path.join(ROOT, "include", "nh_b200.h")


def _declared_functions():
    src = open(HDR).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nh_[A-Za-z_0-9]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_1706_04551_b200 import build
    path = build.build()
    L = C.CDLL(path)
    names = _declared_functions()
    assert "nh_create" in names and "nh_step" in names and "nh_nonhydro_correct" in names
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/nh_b200.h but not exported"


def test_binding_lists_the_same_names():
    from paper_1706_04551_b200 import build
    build.build()
    from paper_1706_04551_b200 import nh
    assert sorted(nh.EXPORTS) == _declared_functions()
    nh.lib()  # argtypes set for all of them without a GPU


def test_struct_layouts_match_the_header():
    # compile a tiny C program against the header and compare sizeof/offsetof with ctypes
    from paper_1706_04551_b200 import build
    build.build()
    from paper_1706_04551_b200 import nh
    prog = r"""
#include <stdio.h>
#include <stddef.h>
#include "nh_b200.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu %zu\n", sizeof(nh_params), offsetof(nh_params, manning_n),
         offsetof(nh_params, breaking), offsetof(nh_params, solver_maxit), offsetof(nh_params, precision),
         sizeof(nh_info), offsetof(nh_info, iters_last));
  return 0;
}
"""
    import tempfile
    with tempfile.TemporaryDirectory() as d:
        src = os.path.join(d, "t.c")
        open(src, "w").write(prog)
        exe = os.path.join(d, "t")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), "-o", exe, src], check=True)
        out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout.split()
    got = [int(x) for x in out]
    P, I = nh.Params, nh.Info
    want = [C.sizeof(P), P.manning_n.offset, P.breaking.offset, P.solver_maxit.offset,
            P.precision.offset, C.sizeof(I), I.iters_last.offset]
    assert got == want


def test_default_params_without_gpu():
    from paper_1706_04551_b200 import build
    build.build()
    from paper_1706_04551_b200 import nh
    p = nh.default_params()
    assert p.g == 9.81 and p.cfl == 0.5 and p.delta == 1e-5 and p.solver_rtol == 1e-12
    assert p.time_order == 2 and p.nonhydro == 1 and p.precision == 64


def test_product_and_oracle_do_not_import_each_other():
    pkg = os.path.join(ROOT, "paper_1706_04551_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dirpath, f)).read()
                for bad in ("import oracle", "from oracle", "nh_oracle", "nho_"):
                    assert bad not in s, f"{f} reaches into the oracle ({bad})"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            s = open(os.path.join(ROOT, "oracle", f)).read()
            for bad in ("import paper_1706_04551_b200", "from paper_1706_04551_b200", "#include \"nh_b200.h\"",
                        "csrc/", "libnh_b200"):
                assert bad not in s.replace("(paper_1706_04551_b200/csrc,", ""), f"{f} reaches into the product ({bad})"


def test_missing_library_fails_loudly(tmp_path):
    # the binding must raise, not fall back, when libnh_b200.so is absent
    code = (
        "import sys; sys.path.insert(0, %r)\n"
        "from paper_1706_04551_b200 import nh\n"
        "nh.LIB_PATH = %r\n"
        "try:\n"
        "    nh.lib()\n"
        "except ImportError as e:\n"
        "    print('RAISED'); sys.exit(0)\n"
        "sys.exit(1)\n" % (ROOT, str(tmp_path / "nope.so")))
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True)
    assert r.returncode == 0 and "RAISED" in r.stdout
