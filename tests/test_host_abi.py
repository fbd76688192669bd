"""CPU-side checks of the boundary: the library builds/loads, exports every symbol include/gx.h
declares, fails loudly without a GPU, and the host-side helper logic is right.  No compute calls."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2209_06731_b200 import binding, build
    build.build()
    return binding.load()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "gx.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gx_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    from paper_2209_06731_b200 import binding
    names = _declared_symbols()
    assert "gx_grid_create" in names and "gx_geometry_set" in names
    assert "gx_nonlinear_rhs" in names and "gx_rhs" in names
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTED) == names


def test_no_torch_types_in_the_c_abi():
    src = open(os.path.join(ROOT, "include", "gx.h")).read()
    assert "torch" not in src.lower() and "at::" not in src and "Tensor" not in src
    assert 'extern "C"' in src


def test_fails_loudly_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2209_06731_b200 import binding as B
    with pytest.raises(B.GxError) as e:
        B.gx_grid_create(16, 16, 4, 2, 2, 1)
    assert e.value.code == B.GX_ERR_CUDA
    h = ctypes.c_void_p()
    assert lib.gx_grid_create(15, 16, 4, 2, 2, 1, ctypes.byref(h)) == B.GX_ERR_ARG
    assert lib.gx_grid_create(16, 16, 4, 2, 2, 1, None) == B.GX_ERR_ARG
    assert lib.gx_query(None, 0, None) == B.GX_ERR_ARG
    assert lib.gx_last_error(None) == b"null handle"


def test_product_path_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2209_06731_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "gx_oracle" not in txt and "libgxconv" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2209_06731_b200 import" not in txt and "libgx.so" not in txt, f


def test_config_shapes_match_survey_table():
    from paper_2209_06731_b200 import inputs as I
    expect = {"tiny": (11, 6, 2, 4224), "cyclone": (127, 22, 5, 2145792), "kinetic": (85, 22, 5, 3829760),
              "hires": (171, 32, 11, 22413312), "stellarator": (127, 64, 8, 74907648)}
    for name, (nakx, naky, J, gel) in expect.items():
        c = I.named_config(name)
        assert (c.nakx, c.naky, c.nj, int(np.prod(c.g_shape))) == (nakx, naky, J, gel)
    assert I.named_config("cyclone").grid_point_moments == 9437184
