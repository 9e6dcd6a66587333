"""The C-ABI library loads and exports every symbol include/srpp.h declares; host-side validation
(no compute calls: this runs without a GPU)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from conftest import ROOT
from paper_1411_3396_b200 import binding, build as srpp_build


@pytest.fixture(scope="module")
def lib():
    srpp_build.build()
    return binding.load()


def test_header_symbols_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "srpp.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(srpp_[a-z_0-9]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None
    assert lib.srpp_version() == 1


def test_struct_layout_matches_header():
    assert C.sizeof(binding.SrppParams) == 3 * 4 + 3 * 4 + 4 + 4 + 6 * 4
    assert C.sizeof(binding.SrppStats) == 8 * 3 + 4 * 2 + 8 + 8 * 3
    assert C.sizeof(binding.SrppTimings) == 20
    assert C.sizeof(binding.SrppBlockInfo) == 48


def test_default_poly_bits():
    got = binding.default_poly().view(np.uint32)
    assert [int(v) for v in got] == [0x3EDEAD5D, 0xBE36288A, 0x3D2403BC, 0xBBB0860A, 0x39CFCFAA, 0xB74AC976]


def test_strerror_and_validation(lib):
    assert binding.strerror(0) == "ok"
    for code in range(-6, 0):
        assert binding.strerror(code) not in ("ok", "unknown status")
    good = binding.make_params((32.0,) * 3, (10,) * 3, 3.0, 0.1)
    assert binding.workspace_bytes(good, 32768) > 32768 * (16 + 24 + 4)     # sorted float4 + fp64 accumulators + perm at least
    # geometry: fewer than 3 cells, cell smaller than rc, too many cells
    for box, nc in (((32.0,) * 3, (2, 10, 10)), ((32.0,) * 3, (11, 10, 10)), ((4096.0,) * 3, (300, 300, 300))):
        with pytest.raises(binding.SrppError) as e:
            binding.workspace_bytes(binding.make_params(box, nc, 3.0, 0.1), 10)
        assert e.value.status == -2
    # invalid arguments
    for kw in (dict(eps=0.0), dict(eps=-1.0), dict(rcut=0.0), dict(eps=float("nan")), dict(rcut=float("inf"))):
        args = dict(rcut=3.0, eps=0.1)
        args.update(kw)
        with pytest.raises(binding.SrppError) as e:
            binding.workspace_bytes(binding.make_params((32.0,) * 3, (10,) * 3, **args), 10)
        assert e.value.status == -1
    bad_poly = binding.default_poly()
    bad_poly[3] = np.inf
    with pytest.raises(binding.SrppError):
        binding.workspace_bytes(binding.make_params((32.0,) * 3, (10,) * 3, 3.0, 0.1, bad_poly), 10)
    with pytest.raises(binding.SrppError) as e:
        binding.workspace_bytes(good, -1)
    assert e.value.status == -1
    with pytest.raises(binding.SrppError) as e:
        binding.workspace_bytes(good, 2 ** 31)
    assert e.value.status == -1


def test_create_argument_errors(lib):
    good = binding.make_params((32.0,) * 3, (10,) * 3, 3.0, 0.1)
    ctx = C.c_void_p()
    assert lib.srpp_create(C.byref(ctx), C.byref(good), None, 1 << 20, None) == -1        # null workspace
    assert lib.srpp_create(C.byref(ctx), C.byref(good), 0x1010, 1 << 30, None) == -4      # misaligned
    assert lib.srpp_create(C.byref(ctx), C.byref(good), 0x1000, 16, None) == -4           # too small
    assert lib.srpp_create(None, C.byref(good), 0x1000, 1 << 30, None) == -1
    # calls on a null context fail cleanly
    assert lib.srpp_build_mesh(None, None, 0) == -1
    assert lib.srpp_accel(None, None) == -1
    assert lib.srpp_accel_kick(None, None, None, C.c_float(0.1)) == -1
    assert lib.srpp_get_mesh(None, None, None, None) == -1
    lib.srpp_destroy(None)


def test_no_cpu_fallback_without_gpu(lib):
    """Without a CUDA device srpp_create reports SRPP_ERR_CUDA: the product path has no CPU route."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    good = binding.make_params((32.0,) * 3, (10,) * 3, 3.0, 0.1)
    ctx = C.c_void_p()
    assert lib.srpp_create(C.byref(ctx), C.byref(good), 0x1000, 1 << 30, None) == -6
    with pytest.raises(RuntimeError):
        binding.Solver((32.0,) * 3, (10,) * 3, n_max=10)


def test_product_does_not_import_oracle():
    """The package and bench's product arm never reference oracle/ (it is test infrastructure)."""
    pkg = os.path.join(ROOT, "paper_1411_3396_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "srpp_oracle" not in txt, f
    src = open(os.path.join(ROOT, "oracle", "srpp_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "srpp.h" not in src and "import paper_1411_3396_b200" not in src and "binding" not in src
