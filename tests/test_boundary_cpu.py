"""CPU-side checks of the C-ABI boundary: the library loads and exports exactly what
include/tcrnet.h declares; no compute call is made (there is no GPU here)."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2112_06613_b200 import build as b
    b.build()
    import paper_2112_06613_b200 as pkg
    return pkg.load_library()


def _declared():
    text = open(os.path.join(ROOT, "include", "tcrnet.h")).read()
    return sorted(set(re.findall(r"TCRNET_API\s+[\w\s\*]+?\b(tcrnet_\w+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    import paper_2112_06613_b200 as pkg
    declared = _declared()
    assert declared == sorted(pkg.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    # and nothing else leaks out of the library
    out = subprocess.run(["nm", "-D", "--defined-only", pkg.LIB_PATH], capture_output=True, text=True, check=True).stdout
    exported = sorted(l.split()[-1] for l in out.splitlines() if " T " in l)
    assert exported == declared


def test_version_and_strerror(lib):
    import paper_2112_06613_b200 as pkg
    assert pkg.version() == 100
    assert pkg.strerror(0) == "ok"
    for code in range(-9, 0):
        assert pkg.strerror(code) not in ("ok", "unknown status")
    assert pkg.strerror(-99) == "unknown status"


def test_argument_errors_without_a_device(lib):
    """Calls that must fail before touching CUDA."""
    import paper_2112_06613_b200 as pkg
    assert lib.tcrnet_create(None, 0, None, None) == pkg.ERR_ARG
    assert lib.tcrnet_build(None, 1, None) == pkg.ERR_ARG
    assert lib.tcrnet_get_stats(None, None) == pkg.ERR_ARG
    lib.tcrnet_destroy(None)  # NULL is allowed
    # the no-allocation call refuses what does not fit its static scratch before it looks at a pointer or at CUDA
    fake = ctypes.c_void_p(256)
    assert lib.tcrnet_row_ptr_noalloc(fake, pkg.NOALLOC_MAX_ROWS + 1, fake, None, None) == pkg.ERR_CAPACITY
    assert lib.tcrnet_row_ptr_noalloc(fake, -1, fake, None, None) == pkg.ERR_ARG
    assert lib.tcrnet_row_ptr_noalloc(fake, 10, None, None, None) == pkg.ERR_ARG


def test_product_fails_loudly_without_gpu():
    import torch
    import paper_2112_06613_b200 as pkg
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        pkg.TcrNet(0)


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "tcrnet.h"\nint main(void){ tcrnet_stats s; (void)s; return TCRNET_OK; }\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"),
                    "-c", str(src), "-o", str(tmp_path / "t.o")], check=True)


def test_stats_struct_layout_matches_header(tmp_path):
    """The ctypes mirror of tcrnet_stats has the C compiler's size and field offsets."""
    from paper_2112_06613_b200.binding import tcrnet_stats
    names = [n for n, _ in tcrnet_stats._fields_]
    body = "".join(f'printf("%zu\\n", offsetof(tcrnet_stats, {n}));' for n in names)
    src = tmp_path / "o.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "tcrnet.h"\n'
                   f'int main(void){{ printf("%zu\\n", sizeof(tcrnet_stats)); {body} return 0; }}\n')
    exe = tmp_path / "o"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    vals = [int(x) for x in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    assert vals[0] == ctypes.sizeof(tcrnet_stats)
    assert vals[1:] == [getattr(tcrnet_stats, n).offset for n in names]


def test_product_does_not_import_oracle():
    """The product path must not route through oracle/ (or any CPU fallback)."""
    pkg_dir = os.path.join(ROOT, "paper_2112_06613_b200")
    for dirpath, _, files in os.walk(pkg_dir):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), f
                assert "tcrnet_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            assert "paper_2112_06613_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "(paper_2112_06613_b200/)", ""), f
