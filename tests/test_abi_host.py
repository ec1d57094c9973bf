"""Host-side checks of the C-ABI library without a GPU: it loads, exports every symbol include/lgt.h
declares, the binding covers the same set, and the product path refuses to run without a device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "lgt.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lgt_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_2602_20516_b200 import build

    return ctypes.CDLL(build.build())


def test_header_symbols_exported(lib):
    names = declared_symbols()
    assert len(names) >= 30
    for n in names:
        assert hasattr(lib, n), n


def test_binding_covers_header():
    from paper_2602_20516_b200 import lgt

    assert sorted(lgt.SYMBOLS) == declared_symbols()
    for n in declared_symbols():
        assert callable(getattr(lgt, n, None)) or n in ("lgt_last_error", "lgt_stream"), n


def test_no_cpu_fallback():
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2602_20516_b200 import lgt

    with pytest.raises(lgt.LgtError) as e:
        lgt.lgt_create((4, 4, 4, 4), 5.5, 0.1, (1, 1, 1, -1))
    assert e.value.code == lgt.LGT_ECUDA
    with pytest.raises(RuntimeError):
        lgt.Lattice((4, 4, 4, 4), 5.5, 0.1, (1, 1, 1, -1))


def test_product_does_not_touch_oracle():
    """The package must not import, link or execute anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2602_20516_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle|liblgt_oracle|lgto_|#include.*oracle", src, re.M), \
                    os.path.join(dirpath, f)


def test_header_is_plain_c_and_links(tmp_path, lib):
    """include/lgt.h compiles as C99 with -Wall -Werror, and a C program links against liblgt.so and gets a clean status
    code (LGT_OK on a GPU box, LGT_ECUDA with a message here) instead of an abort."""
    import subprocess

    from paper_2602_20516_b200 import build

    src = tmp_path / "abi.c"
    src.write_text(r'''
#include <stdio.h>
#include <string.h>
#include "lgt.h"
int main(void) {
    const int dims[4] = {4, 4, 4, 4}, bc[4] = {1, 1, 1, -1}, ranks[2] = {0, 1};
    lgt_ctx* c = NULL;
    lgt_dd* d = NULL;
    int rc = lgt_create(&c, dims, 5.5, 0.1, bc, LGT_F64, 0, NULL);
    if (rc != LGT_OK && rc != LGT_ECUDA) return 1;
    if (rc == LGT_ECUDA && strlen(lgt_last_error(NULL)) == 0) return 2;
    if (rc == LGT_OK && lgt_destroy(c) != LGT_OK) return 3;
    if (lgt_create(&c, dims, 5.5, 0.1, bc, 7, 0, NULL) != LGT_EINVAL) return 4;   /* bad precision */
    if (lgt_dd_create(&d, dims, 3, 2, ranks, 5.5, 0.1, bc, LGT_F64, 0, NULL) != LGT_EINVAL) return 5;
    if (lgt_set_links(NULL, NULL) != LGT_EINVAL) return 6;
    printf("%s rc=%d\n", lgt_version(), rc);
    return 0;
}
''')
    exe = tmp_path / "abi"
    libdir = os.path.dirname(build.LIB)
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"), str(src),
                           "-o", str(exe), "-L", libdir, "-llgt", "-Wl,-rpath," + libdir])
    out = subprocess.run([str(exe)], capture_output=True, text=True)
    assert out.returncode == 0, (out.returncode, out.stdout, out.stderr)
    assert "lgt-b200" in out.stdout
