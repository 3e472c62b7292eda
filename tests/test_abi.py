"""No-GPU checks of the boundary: the C-ABI library builds, loads and exports every symbol include/lcs.h
declares; the product path fails loudly without a CUDA device (no CPU fallback); the binding's struct
matches the header."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_2209_13775_b200 import build
    return build.build()


def header_symbols():
    src = open(os.path.join(ROOT, "include", "lcs.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lcs_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(built_lib):
    lib = ctypes.CDLL(built_lib)
    syms = header_symbols()
    assert {"lcs_field_create", "lcs_locate", "lcs_advect", "lcs_cg_ftle"} <= set(syms)
    for s in syms:
        assert hasattr(lib, s), s
    from paper_2209_13775_b200 import lcs
    assert sorted(lcs.EXPORTS) == syms


def test_header_is_plain_c(tmp_path):
    """include/lcs.h compiles as C (no C++/torch types in the signatures)."""
    import subprocess
    src = tmp_path / "t.c"
    src.write_text('#include "lcs.h"\nint main(void){ lcs_field_desc d; (void)d; return (int)sizeof(lcs_field_desc); }\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(src), "-o", str(tmp_path / "t.o")])


def test_desc_struct_matches_header(tmp_path):
    import subprocess
    from paper_2209_13775_b200 import lcs
    src = tmp_path / "s.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "lcs.h"\nint main(void){printf("%zu %zu %zu %zu %zu %zu",'
                   'sizeof(lcs_field_desc), offsetof(lcs_field_desc, origin), offsetof(lcs_field_desc, n_vertices),'
                   'offsetof(lcs_field_desc, n_snapshots), offsetof(lcs_field_desc, times), offsetof(lcs_field_desc, compute_dtype));return 0;}\n')
    exe = tmp_path / "s"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    out = [int(x) for x in subprocess.check_output([str(exe)]).split()]
    D = lcs.lcs_field_desc
    assert out == [ctypes.sizeof(D), D.origin.offset, D.n_vertices.offset, D.n_snapshots.offset, D.times.offset, D.compute_dtype.offset]


def test_no_cpu_fallback(built_lib):
    """Without a CUDA device the product path must fail loudly (LCS_ERR_CUDA), never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2209_13775_b200 import lcs, inputs
    w = inputs.config1(ng=(4, 4), n_nodes=(5, 5))
    with pytest.raises(lcs.LcsError) as e:
        lcs.Field.from_workload(w)
    assert e.value.status == 5 and "no CPU fallback" in str(e.value)


def test_product_never_imports_oracle():
    """The product package must not import, include, link or load anything under oracle/ (comments may
    cite it), and the oracle must not import the CUDA binding."""
    pat = re.compile(r"(#\s*include[^\n]*oracle|^\s*(from|import)\s+[^\n]*oracle|CDLL\([^\n]*oracle|liblcs_oracle)", re.M)
    pkg = os.path.join(ROOT, "paper_2209_13775_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dirpath, fn)).read()), fn
    pat2 = re.compile(r"(#\s*include[^\n]*(csrc|lcs\.h)|^\s*(from|import)\s+[^\n]*paper_2209_13775_b200|liblcs\.so)", re.M)
    for fn in ("lcs_oracle.py", "lcs_oracle.c"):
        assert not pat2.search(open(os.path.join(ROOT, "oracle", fn)).read()), fn


def test_inputs_are_deterministic():
    from paper_2209_13775_b200 import inputs
    a, b = inputs.config2(ng=(8, 4), lattice=(9, 5)), inputs.config2(ng=(8, 4), lattice=(9, 5))
    assert np.array_equal(a.vertices, b.vertices) and np.array_equal(a.cells, b.cells) and np.array_equal(a.vel, b.vel)
    s = inputs.config1(ng=(4, 2)).seeds()
    assert np.allclose(s[0], [0.25, 0.25]) and np.allclose(s[1], [0.75, 0.25])        # cell-centred, axis 0 fastest
