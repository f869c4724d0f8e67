"""CPU-only checks of the product's host logic: the C-ABI library loads and exports every symbol
include/fts.h declares, argument validation works without a GPU, and the pencil-transform index
arithmetic of csrc/fts_pencil.h (run on the host as an emulated CTA) is correct and bank-conflict-free."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1204_5434_b200 import build
    return build.build()


def test_library_exports_every_declared_symbol(libpath):
    hdr = open(os.path.join(ROOT, "include", "fts.h")).read()
    declared = set(re.findall(r"\b(fts_[a-z_]+)\s*\(", hdr))
    assert {"fts_create", "fts_propagate", "fts_density_operators", "fts_scft_step", "fts_cl_step"} <= declared
    L = C.CDLL(libpath)
    for name in sorted(declared):
        assert hasattr(L, name), name
    from paper_1204_5434_b200 import binding
    assert set(binding.EXPORTS) == declared


def test_argument_validation_without_gpu(libpath):
    from paper_1204_5434_b200 import binding as B
    ok = B.make_params("diblock", fA=0.3, chiN=20.0)
    assert B.workspace_bytes((32, 32, 32), 100, ok) > 2 * 52 * 32 ** 3 * 16           # meet-in-the-middle: Ns/2 + 2 slices per propagator
    both = B.make_params("diblock", fA=0.3, chiN=20.0, store_both=1)
    assert B.workspace_bytes((32, 32, 32), 100, both) > 2 * 101 * 32 ** 3 * 16        # store_both: every slice of q and q+
    assert B.workspace_bytes((32, 32, 32), 100, ok, "f32") < B.workspace_bytes((32, 32, 32), 100, ok)
    # 1-D / 2-D grids are grids with dimensions of 1 (the ones do not change the memory layout)
    assert B.workspace_bytes((64, 1, 1), 100, ok) == B.workspace_bytes((1, 1, 64), 100, ok) == B.workspace_bytes((1, 64, 1), 100, ok)
    assert B.workspace_bytes((32, 16, 1), 100, ok) == B.workspace_bytes((1, 32, 16), 100, ok)
    for grid, Ns, p, status in [((32, 32, 12), 100, ok, 6),                           # not a power of two
                                ((1, 1, 1), 100, ok, 6),
                                ((4, 1, 1), 100, ok, 6),
                                ((512, 8, 8), 100, ok, 6),
                                ((32, 32, 32), 1, ok, 1),
                                ((32, 32, 32), 10, B.make_params("diblock", fA=0.33, chiN=20.0), 1),    # fA*Ns not integer
                                ((32, 32, 32), 10, B.make_params("diblock", fA=0.5, chiN=20.0), 1),     # odd Simpson block
                                ((32, 32, 32), 7, B.make_params("external"), 1)]:
        with pytest.raises(B.FtsError) as e:
            B.workspace_bytes(grid, Ns, p)
        assert e.value.status == status
    # config 5: two stores of 52 slices of 256^3 complex128 = 27.9 GB (BASELINE.json: "~27 GB"); 101 slices each with store_both = 54.2 GB
    n5 = B.workspace_bytes((256, 256, 256), 100, B.make_params("diblock", fA=0.5, chiN=15.0))
    assert 27.9e9 < n5 < 34e9
    n5b = B.workspace_bytes((256, 256, 256), 100, B.make_params("diblock", fA=0.5, chiN=15.0, store_both=1))
    assert 54e9 < n5b < 61e9


def test_pencil_transform_host_emulation(tmp_path):
    exe = str(tmp_path / "host_pencil_test")
    subprocess.run(["g++", "-std=c++17", "-O1", "-o", exe, os.path.join(ROOT, "tests", "host_pencil_test.cpp")], check=True)
    out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0 and "ALL OK" in out.stdout, out.stdout[-2000:]
    assert "FAIL" not in out.stdout.replace("FAILED", "")


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1204_5434_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"import\s+oracle|from\s+oracle|liboracle|oracle_[a-z]|oracle/", txt), f
