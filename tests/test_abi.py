"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol include/ctqmc.h declares;
the Python binding mirrors the C names; the product path fails loudly (no CPU fallback) when there is no device."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    with open(os.path.join(ROOT, "include", "ctqmc.h")) as fh:
        text = fh.read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ctqmc_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_2010_08482_b200 import build
    build.build()          # nvcc cross-compiles for sm_100a without a GPU
    import paper_2010_08482_b200 as L
    return L


def test_header_symbols_are_exported(lib):
    names = _declared_symbols()
    assert {"ctqmc_load_impurity", "ctqmc_trace_batch", "ctqmc_bound_batch", "ctqmc_free_impurity",
            "ctqmc_last_error"} <= set(names)
    dll = ctypes.CDLL(lib.LIB_PATH)
    for n in names:
        assert hasattr(dll, n), f"{n} is declared in include/ctqmc.h but not exported by {lib.LIB_PATH}"


def test_binding_lists_every_header_symbol(lib):
    assert sorted(lib.EXPORTS) == _declared_symbols()
    for n in lib.EXPORTS:
        assert hasattr(lib, n), f"binding has no function {n}"


def test_header_constants_match_binding(lib):
    with open(os.path.join(ROOT, "include", "ctqmc.h")) as fh:
        text = fh.read()
    for name, val in re.findall(r"#define\s+(CTQMC_[A-Z0-9_]+)\s+(-?\d+)", text):
        if hasattr(lib.binding, name):
            assert getattr(lib.binding, name) == int(val), name


def test_sass_is_sm100a_with_fp64_tensor_ops(lib):
    """The shipped library holds sm_100a code and FP64 tensor-core instructions (DMMA) -- not a stub."""
    import subprocess
    cuobjdump = "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-lelf", lib.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run([cuobjdump, "-sass", lib.LIB_PATH], capture_output=True, text=True).stdout
    assert "DMMA" in sass


def test_argument_errors_without_device(lib):
    """Argument validation happens before any CUDA call, so it is observable on a CPU-only box; a well-formed load
    must FAIL (no device, no CPU fallback) rather than silently succeed."""
    import torch
    with pytest.raises(lib.CtqmcError) as ei:
        class Bad:
            dims = np.array([0], np.int32); energy = np.zeros(0); n_symbols = 1; is_complex = False
            blk_symbol = np.zeros(0, np.int32); blk_src = np.zeros(0, np.int32); blk_dst = np.zeros(0, np.int32)
            blk_offset = np.zeros(0, np.int64); blk_data = np.zeros(0)
        lib.ctqmc_load_impurity(Bad(), 0)
    assert ei.value.code == lib.binding.CTQMC_ERR_ARG
    assert "dim" in lib.ctqmc_last_error()
    if not torch.cuda.is_available():
        class Good:
            dims = np.array([1], np.int32); energy = np.zeros(1); n_symbols = 1; is_complex = False
            blk_symbol = np.zeros(0, np.int32); blk_src = np.zeros(0, np.int32); blk_dst = np.zeros(0, np.int32)
            blk_offset = np.zeros(0, np.int64); blk_data = np.zeros(0)
        with pytest.raises(lib.CtqmcError) as ei:
            lib.ctqmc_load_impurity(Good(), 0)
        assert ei.value.code in (lib.binding.CTQMC_ERR_CUDA, lib.binding.CTQMC_ERR_OOM, lib.binding.CTQMC_ERR_UNSUPPORTED)


def test_product_path_does_not_import_oracle():
    """The oracle is test infrastructure: nothing under the package (or workloads/) may import it."""
    for base in ("paper_2010_08482_b200", "workloads"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, base)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".h")):
                    with open(os.path.join(dirpath, f)) as fh:
                        src = fh.read()
                    assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), os.path.join(dirpath, f)
    for dirpath, _, files in os.walk(os.path.join(ROOT, "oracle")):
        for f in files:
            if f.endswith(".py"):
                with open(os.path.join(dirpath, f)) as fh:
                    assert "paper_2010_08482_b200" not in re.sub(r'""".*?"""', "", fh.read(), flags=re.S)
