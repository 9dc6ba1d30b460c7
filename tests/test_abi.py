"""CPU checks of the boundary: libmgrhd.so builds for sm_100a, loads, exports every symbol that
include/mgrhd.h declares, validates arguments on the host, and fails loudly (no CPU fallback)
when no CUDA device can be used.  No compute calls here.
"""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "mgrhd.h")


@pytest.fixture(scope="module")
def binding():
    from paper_2407_18304_b200 import binding, build

    build.build()
    binding.load_library()
    return binding


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mgrhd_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(binding):
    names = declared_functions()
    assert len(names) >= 10
    lib = ctypes.CDLL(binding.LIB_PATH)
    for name in names:
        assert hasattr(lib, name), f"{name} declared in include/mgrhd.h but not exported"
    assert sorted(binding.EXPORTS) == names


def test_struct_layouts_match_header(binding):
    """ctypes mirrors: field counts/sizes implied by the header."""
    assert ctypes.sizeof(binding.Units) == 5 * 8
    assert ctypes.sizeof(binding.State) == 11 * 8            # ... + Srad
    assert ctypes.sizeof(binding.OpacityModel) == 128        # 2 pointers, controls, kind / T_ref / p_T / NT / lnT0 / dlnT / table, outer_mode
    assert ctypes.sizeof(binding.Stats) == (9 + 2 * 64) * 8
    src = open(HEADER).read()
    assert "#define MGRHD_MAX_GROUPS 64" in src and "#define MGRHD_HIST 64" in src
    assert binding.MAX_GROUPS == 64 and binding.HIST == 64


def _init(binding, edges, kappa, alpha, **kw):
    return binding.Context(edges, kappa, alpha, **kw)


def test_init_argument_errors(binding):
    e = np.array([1.0, 2.0, 4.0])
    k = np.ones(2)
    a = np.zeros(2)
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_EDGES"):
        _init(binding, np.array([1.0, 4.0, 2.0]), k, a)
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_EDGES"):
        _init(binding, np.array([-1.0, 2.0, 4.0]), k, a)
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_ALPHA"):
        _init(binding, np.array([0.0, 2.0, 4.0]), k, np.array([-1.0, 0.0]))
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_ALPHA"):
        _init(binding, np.array([1.0, 2.0, np.inf]), k, np.array([0.0, -2.0]))
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_RANGE"):
        _init(binding, e, k, a, gamma=1.0)
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_RANGE"):
        _init(binding, e, k, a, a_rad=0.0)
    for bad_k in (0.0, -1.0, np.inf, np.nan):           # kappa = 0 makes Eq. 42 singular (1/chi_E)
        with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_RANGE"):
            _init(binding, e, np.array([1.0, bad_k]), a)
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_ARG"):
        _init(binding, e, k, a, closure=2)
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_ARG"):
        _init(binding, e, k, a, spectrum=2)
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_ARG"):
        _init(binding, e, k, a, opacity_kind=3)
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_ARG"):
        _init(binding, e, k, a, outer_mode=2)
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_RANGE"):
        _init(binding, e, k, a, opacity_kind=1, T_ref=0.0, p_T=1.5)
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_ARG"):
        _init(binding, e, None, None, opacity_kind=2)                                   # no table
    tab = np.zeros((3, 4))
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_ALPHA"):
        _init(binding, np.array([0.0, 2.0, 4.0]), None, None, opacity_kind=2, lnk_edge=tab)   # Eq. 20 needs finite edges > 0
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_RANGE"):
        _init(binding, e, None, None, opacity_kind=2, lnk_edge=tab, dlnT=0.0)
    bad = tab.copy()
    bad[1, 2] = np.nan
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_RANGE"):
        _init(binding, e, None, None, opacity_kind=2, lnk_edge=bad)
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_ARG"):
        _init(binding, np.arange(67.0) + 1, np.ones(66), np.zeros(66))   # Nq > MGRHD_MAX_GROUPS


def test_no_cpu_fallback(binding):
    """Without a CUDA device a valid mgrhd_init must fail with MGRHD_ERR_CUDA, never compute."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present; the loud-failure path is exercised on the CPU box")
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_CUDA"):
        _init(binding, np.array([1.0, 2.0, 4.0]), np.ones(2), np.zeros(2))
    with pytest.raises(binding.MgrhdError, match="MGRHD_ERR_CUDA"):
        binding.measure_dfma_peak()


def test_product_does_not_import_oracle():
    """The product package must not reference oracle/ (and the oracle must not reference the product's csrc)."""
    pkg = os.path.join(ROOT, "paper_2407_18304_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "mgrhd_oracle" not in txt and "liboracle" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "mgrhd_oracle.cpp")).read()
    assert "#include \"" not in otxt          # system headers only
    opy = open(os.path.join(ROOT, "oracle", "oracle.py")).read()
    assert "paper_2407_18304_b200" not in opy
