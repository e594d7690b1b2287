"""CPU-side checks of the boundary: the C-ABI library builds, loads, and exports every symbol include/hough.h declares
(no compute calls: there is no GPU here).  Also: the product package never imports the oracle."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "hough.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hough_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2511_02742_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def test_header_declares_the_five_entry_points():
    names = declared_functions()
    for n in ("hough_plan_create", "hough_vote", "hough_find_clusters", "hough_assign_hits", "hough_plan_destroy"):
        assert n in names


def test_library_exports_every_declared_symbol(lib):
    for n in declared_functions():
        assert hasattr(lib, n), f"libhough.so does not export {n}"


def test_binding_lists_every_declared_symbol():
    from paper_2511_02742_b200 import hough
    assert sorted(hough.EXPORTS) == declared_functions()
    for n in hough.EXPORTS:
        assert hasattr(hough, n) or n in ("hough_strerror", "hough_last_cuda_error"), n


def test_header_compiles_as_plain_c(tmp_path):
    c = tmp_path / "t.c"
    c.write_text('#include "hough.h"\nint main(void){ hough_plan_desc_t d; hough_candidate_t c; (void)d; (void)c; '
                 'return sizeof(hough_candidate_t) == 32 ? 0 : 1; }\n')
    exe = tmp_path / "t"
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(c), "-o", str(exe)])
    assert subprocess.call([str(exe)]) == 0


def test_struct_layouts_match_the_binding(lib, tmp_path):
    from paper_2511_02742_b200 import hough
    fields = [n for n, _ in hough.hough_plan_desc_t._fields_]
    c = tmp_path / "s.c"
    c.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "hough.h"\nint main(void){ printf("%zu %zu", sizeof(hough_plan_desc_t), sizeof(hough_plan_info_t));\n'
                 + "".join(f'printf(" %zu", offsetof(hough_plan_desc_t, {f}));\n' for f in fields) + "return 0; }\n")
    exe = tmp_path / "s"
    subprocess.check_call(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), str(c), "-o", str(exe)])
    nums = [int(x) for x in subprocess.check_output([str(exe)]).split()]
    assert nums[0] == ctypes.sizeof(hough.hough_plan_desc_t) and nums[1] == ctypes.sizeof(hough.hough_plan_info_t)
    assert nums[2:] == [getattr(hough.hough_plan_desc_t, f).offset for f in fields]
    assert hough.CANDIDATE_DTYPE.itemsize == 32
    lib.hough_strerror.restype = ctypes.c_char_p
    assert lib.hough_strerror(0) == b"ok"
    assert lib.hough_version() >= 100


def test_argument_validation_needs_no_gpu(lib):
    from paper_2511_02742_b200 import hough
    hough.load_library()
    with pytest.raises(hough.HoughError) as ei:
        hough.hough_plan_create(0, 0, 0.0, 0.0, 0.0, 0, 0.0, 0, 0, 0, 0)
    assert ei.value.status == hough.HOUGH_EINVAL


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2511_02742_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f"{f} imports the oracle"
                assert not re.search(r"#include[^\n]*oracle", text), f"{f} includes an oracle header"
                assert "libhough_oracle" not in text and "hough_oracle.c" not in text, f"{f} links the oracle"
    code = "import sys; import paper_2511_02742_b200.hough, paper_2511_02742_b200.synth; " \
           "assert not any(m == 'oracle' or m.startswith('oracle.') for m in sys.modules)"
    subprocess.check_call([sys.executable, "-c", code], cwd=ROOT)


def test_the_build_step_depends_on_every_source_file():
    """A header missing from build.DEPENDS means an edit to it does not rebuild libhough.so (round 2: hough_track.cuh was missing)."""
    import os
    from paper_2511_02742_b200 import build as b
    csrc = os.path.join(os.path.dirname(b.__file__), "csrc")
    deps = {os.path.abspath(d) for d in b.DEPENDS}
    for f in os.listdir(csrc):
        assert os.path.abspath(os.path.join(csrc, f)) in deps, f
    assert any(d.endswith(os.path.join("include", "hough.h")) for d in deps)
    # and every #include "..." of the translation unit is one of them
    import re
    for src in b.SOURCES:
        for inc in re.findall(r'#include\s+"([^"]+)"', open(src).read()):
            assert os.path.abspath(os.path.join(os.path.dirname(src), inc)) in deps, inc


def test_enumerators_of_the_header_match_the_binding():
    """Every HOUGH_* enumerator with an explicit value in include/hough.h has the same value in the Python binding (and in the
    host-model driver of the tests)."""
    import os
    import re
    import sys
    from paper_2511_02742_b200 import hough as H
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    text = re.sub(r"/\*.*?\*/", " ", open(os.path.join(root, "include", "hough.h")).read(), flags=re.S)
    found = {name: int(val) for name, val in re.findall(r"\b(HOUGH_[A-Z0-9_]+)\s*=\s*(-?\d+)", text)}
    assert {"HOUGH_FLAG_THETA_WRAP", "HOUGH_STATUS_BAD_OFFSETS", "HOUGH_U16", "HOUGH_FIT_FOUND", "HOUGH_EINVAL"} <= set(found)
    checked = 0
    for name, val in found.items():
        if hasattr(H, name):
            assert getattr(H, name) == val, name
            checked += 1
    assert checked >= 10
    sys.path.insert(0, os.path.join(root, "tests", "emu"))
    import hough_emu as E
    assert (E.FLAG_GENERAL_ONLY, E.FLAG_SMALL_LISTS, E.FLAG_THETA_WRAP) == (found["HOUGH_FLAG_GENERAL_ONLY"], found["HOUGH_FLAG_SMALL_LISTS"], found["HOUGH_FLAG_THETA_WRAP"])
    assert (E.HOUGH_I32, E.HOUGH_U16) == (found["HOUGH_I32"], found["HOUGH_U16"])
