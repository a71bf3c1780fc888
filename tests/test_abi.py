"""CPU-side checks of the C-ABI boundary (no compute): the library builds for sm_100a, loads, and
exports every symbol include/pbc_jk.h declares; the binding's struct layouts match the header;
without a CUDA device the library refuses loudly (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2410_22278_b200 import build, binding
    build.build()
    return binding.load()


def _header_symbols():
    txt = open(os.path.join(ROOT, "include", "pbc_jk.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(pbc_jk_[a-z0-9_]+)\s*\(", txt)))


def test_header_symbols_exported(lib):
    from paper_2410_22278_b200 import binding
    names = _header_symbols()
    assert len(names) >= 10
    for n in names:
        assert hasattr(lib, n), f"libpbc_jk.so does not export {n}"
    assert sorted(binding.SYMBOLS) == names


def test_struct_layout_matches_header():
    """sizeof of the binding's ctypes structs == sizeof computed by a C compiler from the header."""
    import subprocess
    import tempfile
    from paper_2410_22278_b200 import binding
    src = ('#include "pbc_jk.h"\n#include <stdio.h>\nint main(void){printf("%zu %zu %zu %zu %zu\\n",'
           "sizeof(pbc_cell),sizeof(pbc_atoms),sizeof(pbc_shells),sizeof(pbc_cutoffs),sizeof(pbc_jk_stats_t));return 0;}\n")
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "s.c")
        open(c, "w").write(src)
        exe = os.path.join(d, "s")
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe])
        sizes = [int(x) for x in subprocess.check_output([exe]).split()]
    mine = [C.sizeof(binding.pbc_cell), C.sizeof(binding.pbc_atoms), C.sizeof(binding.pbc_shells),
            C.sizeof(binding.pbc_cutoffs), C.sizeof(binding.pbc_jk_stats_t)]
    assert sizes == mine


def test_invalid_arguments_rejected(lib):
    out = C.c_void_p()
    assert lib.pbc_jk_create(None, None, None, 0.3, None, C.byref(out)) == -1
    assert not out.value
    assert b"null" in lib.pbc_jk_last_error(None)
    assert lib.pbc_jk_nbf(None) == -1
    assert lib.pbc_jk_destroy(None) == 0
    assert lib.pbc_jk_build(None, None, None, None, None) == -1


def test_no_cpu_fallback(lib):
    """On a box without a GPU pbc_jk_create must fail with PBC_JK_ERR_CUDA, not compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2410_22278_b200 import binding, workloads
    with pytest.raises(binding.PbcJKError) as ei:
        binding.PbcJK(workloads.tiny())
    assert ei.value.code == -3
    assert "no CPU fallback" in str(ei.value)


def test_product_does_not_import_oracle():
    """The product path never touches oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2410_22278_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) == "build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "pbc_jk_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2410_22278_b200 import" not in txt and "import paper_2410_22278_b200" not in txt, f
            assert "libpbc_jk.so" not in txt


def test_bench_peaks_helper_exports_and_refuses_without_gpu(lib):
    """bench.py's measurement helper (outside the product ABI) exports its five probes; without a device each fails."""
    from paper_2410_22278_b200 import binding
    hl = C.CDLL(binding.PEAKS_LIB_PATH)
    for name in ("fp64_fma", "fp32_fma", "fp64_dmma", "fp64_mixed_pipe", "fp64_dmma_loop"):
        f = getattr(hl, f"bench_{name}_peak")
        f.argtypes = [C.c_int32, C.POINTER(C.c_double)]
        f.restype = C.c_int
        import torch
        if not torch.cuda.is_available():
            v = C.c_double(-7.0)
            assert f(10, C.byref(v)) != 0 and v.value == -7.0
    # the product library holds none of them
    assert not hasattr(lib, "bench_fp64_dmma_peak")
