"""CPU-only checks of the boundary: libfpcl.so builds, loads and exports every symbol include/fpcl.h declares, the
ctypes mirrors of the POD structs have the C sizes, and the flag constants agree with the header.  No compute call
is made (there is no GPU here)."""
import ctypes as C
import os
import re
import subprocess
import sys
import tempfile

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "fpcl.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2606_15622_b200 import build, fpcl
    build.build()
    return fpcl.load()


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fp_[a-z_]+)\s*\(", src)))


def test_exports_every_declared_symbol(lib):
    from paper_2606_15622_b200 import fpcl
    names = _declared()
    assert set(names) == set(fpcl.EXPORTS), (names, fpcl.EXPORTS)
    for n in names:
        assert hasattr(lib, n), n
    assert fpcl.fp_version().startswith("fpcl")


def test_struct_sizes_and_constants_match_header():
    from paper_2606_15622_b200 import fpcl
    prog = r'''
#include <stdio.h>
#include <stddef.h>
#include "fpcl.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu\n", sizeof(fp_wall), sizeof(fp_params), sizeof(fp_mlp),
         offsetof(fp_params, seed), offsetof(fp_params, wall), offsetof(fp_params, body_kind));
  printf("%u %u %u %u %u %u %u\n", FP_FLAG_EMPTY, FP_FLAG_LOWCOUNT, FP_FLAG_SINGULAR, FP_FLAG_ILLCOND, FP_FLAG_ALPHA,
         FP_FLAG_SKIPPED, FP_FLAG_NONFINITE);
  printf("%d %d %d %d\n", FP_ERR_ARG, FP_ERR_STATE, FP_ERR_CUDA, FP_ERR_UNSUPPORTED);
  return 0;
}'''
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "s.c")
        open(c, "w").write(prog)
        exe = os.path.join(d, "s")
        subprocess.check_call(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), c, "-o", exe])
        out = subprocess.check_output([exe]).decode().split("\n")
    sizes = [int(v) for v in out[0].split()]
    assert sizes[0] == C.sizeof(fpcl.FpWall)
    assert sizes[1] == C.sizeof(fpcl.FpParams)
    assert sizes[2] == C.sizeof(fpcl.FpMlp)
    assert sizes[3] == fpcl.FpParams.seed.offset
    assert sizes[4] == fpcl.FpParams.wall.offset
    assert sizes[5] == fpcl.FpParams.body_kind.offset
    flags = [int(v) for v in out[1].split()]
    assert flags == [fpcl.FLAG_EMPTY, fpcl.FLAG_LOWCOUNT, fpcl.FLAG_SINGULAR, fpcl.FLAG_ILLCOND, fpcl.FLAG_ALPHA,
                     fpcl.FLAG_SKIPPED, fpcl.FLAG_NONFINITE]
    errs = [int(v) for v in out[2].split()]
    assert errs == [fpcl.FP_ERR_ARG, fpcl.FP_ERR_STATE, fpcl.FP_ERR_CUDA, fpcl.FP_ERR_UNSUPPORTED]


def test_flag_constants_agree_with_oracle(orc):
    from paper_2606_15622_b200 import fpcl
    # the two sides define the interface constants independently; the tests are where they are compared
    for n in ("FLAG_EMPTY", "FLAG_LOWCOUNT", "FLAG_SINGULAR", "FLAG_ILLCOND", "FLAG_ALPHA", "FLAG_SKIPPED",
              "FLAG_NONFINITE"):
        assert getattr(fpcl, n) == getattr(orc, n)


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle: no file of the package mentions it as an import."""
    pkg = os.path.join(ROOT, "paper_2606_15622_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "fp_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "libfpcl" not in txt and "csrc/common" not in txt, f


def test_no_cpu_fallback_without_gpu():
    """Without a CUDA device the binding raises instead of computing anything on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2606_15622_b200 import fpcl, workloads
    cfg, _ = workloads.couette()
    with pytest.raises(fpcl.FpclError):
        fpcl.Context(cfg)
