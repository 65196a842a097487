"""CPU-side checks of the boundary: the CUDA library builds (nvcc cross-compiles sm_100a without a GPU), loads,
and exports every symbol include/refdef.h declares; without a CUDA device the entry points fail loudly
(RD_ECUDA) instead of falling back to anything.  No compute call is made here."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

import paper_2606_17971_b200 as pkg
from paper_2606_17971_b200 import binding, build as cuda_build


@pytest.fixture(scope="module")
def lib_path():
    return cuda_build.build()


def test_library_exports_every_declared_symbol(lib_path):
    declared = binding.declared_in_header()
    assert len(declared) >= 15
    assert sorted(declared) == sorted(binding.EXPORTS)
    assert sorted(pkg.exported_symbols(lib_path)) == sorted(binding.EXPORTS)


def test_struct_layouts_match_header(lib_path):
    # sizes the C compiler gives the report structs (gcc on the header) equal the ctypes mirrors
    src = r'''
    #include <stdio.h>
    #include "refdef.h"
    int main(void){ printf("%zu %zu %zu %zu\n", sizeof(rd_options), sizeof(rd_step_report), sizeof(rd_query_report), sizeof(rd_solve_report)); return 0; }
    '''
    import tempfile

    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "s.c")
        open(c, "w").write(src)
        exe = os.path.join(d, "s")
        subprocess.check_call(["gcc", "-I", os.path.join(os.path.dirname(binding.HERE), "include"), c, "-o", exe])
        sizes = [int(x) for x in subprocess.check_output([exe]).split()]
    assert sizes == [C.sizeof(binding._Options), C.sizeof(binding._StepReport), C.sizeof(binding._QueryReport),
                     C.sizeof(binding._SolveReport)]


def test_no_cpu_fallback(lib_path):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    rp = np.array([0, 1], dtype=np.int64)
    with pytest.raises(pkg.RefDefError, match="ecuda"):
        pkg.RefDef(rp, np.array([0], dtype=np.int32), np.array([1.0]), np.array([1.0]), 1e-4)


def test_default_options(lib_path):
    lib = pkg.load_library()
    o = binding._Options()
    lib.rd_default_options(C.byref(o))
    d = pkg.Options()
    assert (o.sigma_is_alpha, o.eps, o.eps_c, o.cg_cap, o.pdas_cap, o.replace_period, o.jacobi, o.c_is_diag, o.init,
            o.alg1_variant) == \
           (d.sigma_is_alpha, d.eps, d.eps_c, d.cg_cap, d.pdas_cap, d.replace_period, d.jacobi, d.c_is_diag, d.init,
            d.alg1_variant)


def test_product_never_imports_oracle():
    # the product package must not reference oracle/ (a product path through the oracle voids parity)
    for root, _, files in os.walk(binding.HERE):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(root, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "refdef_oracle" not in text, f
