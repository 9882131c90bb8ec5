"""CPU-side checks of the boundary: libtdpd.so builds for sm_100a, loads, exports every symbol include/tdpd.h
declares, and the ctypes structs have the C layout.  No compute calls (there is no GPU here)."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def T():
    from paper_1611_06163_b200 import build
    build.build()
    import paper_1611_06163_b200 as T
    return T


def test_exports_every_declared_symbol(T):
    hdr = open(os.path.join(ROOT, "include", "tdpd.h")).read()
    declared = set(re.findall(r"\b(tdpd_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(T.SYMBOLS)
    L = T.load_library()
    for name in declared:
        assert hasattr(L, name), name
    nm = subprocess.run(["nm", "-D", "--defined-only", T.LIB_PATH], capture_output=True, text=True).stdout
    exported = set(re.findall(r" T (tdpd_[a-z_0-9]+)", nm))
    assert declared <= exported


def test_struct_layout_matches_header(T, tmp_path):
    src = tmp_path / "sz.c"
    src.write_text('#include "tdpd.h"\n#include <stdio.h>\n#include <stddef.h>\n'
                   'int main(void){printf("%zu %zu %zu %zu %zu\\n", sizeof(tdpd_params), sizeof(tdpd_rbc_params),'
                   'offsetof(tdpd_params, kappa), offsetof(tdpd_params, seed), offsetof(tdpd_params, body_mode));return 0;}\n')
    exe = tmp_path / "sz"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    a, b, c, d, e = map(int, subprocess.check_output([str(exe)]).split())
    assert a == ctypes.sizeof(T.Params) and b == ctypes.sizeof(T.RbcParams)
    assert c == T.Params.kappa.offset and d == T.Params.seed.offset and e == T.Params.body_mode.offset


def test_sass_is_sm100a_and_no_fallback(T):
    out = subprocess.run(["cuobjdump", "-lelf", T.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    import torch
    if not torch.cuda.is_available():
        import tdpd_workloads as W
        with pytest.raises(RuntimeError):
            T.Simulation(W.fluid_params((6, 6, 6), 1.0))   # fails loudly without a GPU: no CPU path


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1611_06163_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "tdpd_oracle" not in txt, f


def test_noalloc_sort_argument_checks_need_no_gpu(T):
    """tdpd_sort_cells_noalloc refuses bad sizes before it touches CUDA: checked here without a device; the binding's
    limit is the header's."""
    hdr = open(os.path.join(ROOT, "include", "tdpd.h")).read()
    assert int(re.search(r"#define TDPD_NOALLOC_MAX_N (\d+)", hdr).group(1)) == T.NOALLOC_MAX_N
    scratch = int(re.search(r"#define TDPD_NOALLOC_SCRATCH_BYTES (\d+)", hdr).group(1))
    assert scratch == 2 * 4 * T.NOALLOC_MAX_N + 128 * 1024
    with pytest.raises(T.TdpdError) as e:
        T.sort_cells_noalloc(256, 0, T.NOALLOC_MAX_N + 1, 16, 256, 256)
    assert e.value.code == -1 and "TDPD_NOALLOC_MAX_N" in str(e.value)
    for n, bits in ((-1, 16), (16, 0), (16, 33)):
        with pytest.raises(T.TdpdError) as e:
            T.sort_cells_noalloc(256, 0, n, bits, 256, 256)
        assert e.value.code == -1
    T.sort_cells_noalloc(0, 0, 0, 16, 0, 0)      # n = 0 is a no-op, also without a device
    with pytest.raises(T.TdpdError):
        T.sort_cells_noalloc(0, 0, 16, 16, 256, 256)   # NULL keys
