"""CPU-side checks of the CUDA path's boundary: the C-ABI library builds, loads and exports every symbol that
include/jump_b200.h declares; the ctypes structs have the C layout; no compute call is made (no GPU here)."""
import ctypes as C
import os
import re
import subprocess
import sys
import tempfile

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "jump_b200.h")


@pytest.fixture(scope="module")
def binding():
    from paper_2412_15073_b200 import build as b, binding
    b.build()
    return binding


def declared_symbols():
    txt = open(HEADER).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(jump_[a-z0-9_]+|baoab_step)\s*\(", txt)))


def test_library_exports_every_declared_symbol(binding):
    names = declared_symbols()
    assert {"jump_init", "jump_step", "baoab_step", "jump_respa_step", "jump_free"} <= set(names)
    lib = binding.lib()
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names


def test_ctypes_structs_match_the_c_layout(binding):
    src = r'''
#include <stdio.h>
#include <stddef.h>
#include "jump_b200.h"
int main(void) {
  printf("%zu %zu %zu\n", sizeof(jump_params), sizeof(jump_event), sizeof(jump_stats));
  printf("%zu %zu %zu %zu %zu\n", offsetof(jump_params, seed), offsetof(jump_params, box), offsetof(jump_params, r_mid),
         offsetof(jump_params, eps_jump), offsetof(jump_params, cell_edge));
  printf("%zu %zu %zu\n", offsetof(jump_stats, max_p), offsetof(jump_stats, max_row), offsetof(jump_stats, error));
  return 0; }
'''
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "t.c")
        open(c, "w").write(src)
        exe = os.path.join(d, "t")
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe])
        out = subprocess.check_output([exe]).decode().split()
    v = [int(x) for x in out]
    P, E, S = binding.jump_params, binding.jump_event, binding.jump_stats
    assert v[:3] == [C.sizeof(P), C.sizeof(E), C.sizeof(S)]
    assert v[3:8] == [P.seed.offset, P.box.offset, P.r_mid.offset, P.eps_jump.offset, P.cell_edge.offset]
    assert v[8:] == [S.max_p.offset, S.max_row.offset, S.error.offset]
    assert binding.EVENT_DTYPE.itemsize == C.sizeof(E)


def test_header_is_plain_c_and_has_no_torch_types():
    txt = open(HEADER).read()
    code = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    assert "torch" not in code.lower() and "at::" not in code and "std::" not in code and 'extern "C"' in code
    with tempfile.TemporaryDirectory() as d:     # compiles as C
        c = os.path.join(d, "t.c")
        open(c, "w").write('#include "jump_b200.h"\nint main(void) { return 0; }\n')
        subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", c, "-o", os.path.join(d, "t.o")])


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2412_15073_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "jump_oracle" not in txt and "from oracle" not in txt and "import oracle" not in txt, f


def test_no_gpu_means_a_loud_failure_not_a_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2412_15073_b200 import workloads as wl
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.JumpSim(wl.small_water(2), r_short=4.0, r_long=6.0)


def test_make_params_defaults(binding):
    p = binding.make_params(648, 18.64, 5.0, 9.0)
    assert p.r_mid == 7.0 and p.flags == 3 and p.n_inner == 4 and list(p.box) == [18.64] * 3
