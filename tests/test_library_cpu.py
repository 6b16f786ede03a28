"""CPU-side checks of the C-ABI library: it loads, exports every symbol declared in
include/phoebe_elph.h, and its host logic (argument validation, workspace sizing)
behaves as the header says.  No compute call is made (there is no GPU here)."""
import ctypes
import os
import re

import pytest

from paper_2111_14999_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def test_every_declared_symbol_is_exported(lib):
    header = open(os.path.join(ROOT, "include", "phoebe_elph.h")).read()
    declared = set(re.findall(r"\b(phoebe_elph_[a-z0-9_]+)\s*\(", header))
    declared -= {"phoebe_elph_ctx", "phoebe_elph_dims"}
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None
    # ... and nothing else: the product ABI is the hot path's calls, measurement aids live in their own library
    import subprocess
    syms = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True).stdout
    exported = set(re.findall(r" T (phoebe_elph_[a-z0-9_]+)", syms))
    assert exported == declared, exported ^ declared
    probes = binding.load_probes()
    pheader = open(os.path.join(ROOT, "include", "phoebe_elph_probes.h")).read()
    pdecl = set(re.findall(r"\b(phoebe_elph_[a-z0-9_]+)\s*\(", pheader))
    assert pdecl == set(binding.PROBE_EXPORTS)
    for name in pdecl:
        assert getattr(probes, name) is not None


def test_version(lib):
    assert "sm_100a" in binding.version()


def test_workspace_bytes_monotone_and_budget(lib):
    d = binding.Dims(343, 343, 8, 6, 8, 8, 4096)
    nbytes, nq = binding.workspace_bytes(d, 10 << 30)
    assert nq == 4096 and 0 < nbytes < (1 << 30)
    # a budget just below what 4096 q need gives a smaller batch that fits
    nbytes2, nq2 = binding.workspace_bytes(d, nbytes - 1)
    assert nq2 < 4096 and nbytes2 <= nbytes - 1
    # nq_max = 0 means "as many as fit"
    d0 = binding.Dims(343, 343, 8, 6, 8, 8, 0)
    nbytes3, nq3 = binding.workspace_bytes(d0, 1 << 30)
    assert nq3 > 4096 and nbytes3 <= (1 << 30)
    # too small for anything
    with pytest.raises(binding.PhoebeElphError) as e:
        binding.workspace_bytes(d, 1 << 10)
    assert e.value.code == -5


def test_large_config_fits_180GB(lib):
    d = binding.Dims(343, 343, 32, 30, 32, 32, 16384)
    gW = 16 * 343 * 343 * 32 * 32 * 30
    nbytes, nq = binding.workspace_bytes(d, 170 * 10**9 - gW)
    assert nq == 16384 and gW + nbytes < 170 * 10**9


@pytest.mark.parametrize("bad", [
    (0, 343, 8, 6, 8, 8, 16), (343, 0, 8, 6, 8, 8, 16), (343, 343, 8, 6, 9, 8, 16),
    (343, 343, 8, 6, 8, 0, 16), (343, 343, 8, 0, 8, 8, 16), (343, 343, 8, 6, 8, 8, -1),
    (343, 343, 8, 6, 8, 8, 16, 33), (343, 343, 8, 6, 8, 8, 16, -1),
])
def test_bad_dims_rejected(lib, bad):
    with pytest.raises(binding.PhoebeElphError) as e:
        binding.workspace_bytes(binding.Dims(*bad), 1 << 30)
    assert e.value.code == -2


def test_null_and_error_codes_without_gpu(lib):
    d = binding.Dims(27, 27, 2, 3, 2, 2, 64)
    ctx = ctypes.c_void_p(0)
    # null pointers
    assert lib.phoebe_elph_setup(ctypes.byref(ctx), None, None, None, None, None, ctypes.byref(d), None, 0, None) == -1
    assert lib.phoebe_elph_set_k(None, None, None, 1) == -1
    assert lib.phoebe_elph_q_batch(None, 1, 1, None, None, None, None, None) == -1
    assert lib.phoebe_elph_destroy(None) == -1
    assert lib.phoebe_elph_last_error(None) == b""
    # misaligned g_W pointer
    Re = (ctypes.c_double * 81)()
    assert lib.phoebe_elph_setup(ctypes.byref(ctx), 0x1008, Re, Re, None, None, ctypes.byref(d), 0x10000, 1 << 30,
                                 None) == -3
    # workspace too small
    assert lib.phoebe_elph_setup(ctypes.byref(ctx), 0x1000, Re, Re, None, None, ctypes.byref(d), 0x10000, 16, None) == -5
    # non-positive degeneracy
    assert lib.phoebe_elph_setup(ctypes.byref(ctx), 0x1000, Re, Re, Re, None, ctypes.byref(d), 0x10000, 1 << 30,
                                 None) == -2


def test_no_cpu_fallback(lib):
    """Without a CUDA device the product path must fail loudly, not fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    d = binding.Dims(27, 27, 2, 3, 2, 2, 64)
    ctx = ctypes.c_void_p(0)
    Re = (ctypes.c_double * 81)()
    rc = lib.phoebe_elph_setup(ctypes.byref(ctx), 0x1000, Re, Re, None, None, ctypes.byref(d), 0x10000, 1 << 30, None)
    assert rc == -6 and not ctx.value
    t = ctypes.c_double(0)
    assert binding.load_probes().phoebe_elph_probe_fp64(1, 10, None, ctypes.byref(t)) == -6
    import numpy as np
    with pytest.raises(binding.PhoebeElphError) as e:
        binding.ElphContext(torch.zeros((1, 1, 1, 1, 1), dtype=torch.complex128), np.zeros((1, 3)), np.zeros((1, 3)),
                            nq_max=1)
    assert e.value.code == -6


def test_product_path_does_not_import_oracle():
    for fn in ("binding.py", "harness.py", "workloads.py", "build.py", "__init__.py"):
        src = open(os.path.join(ROOT, "paper_2111_14999_b200", fn)).read()
        assert not re.search(r"^\s*(import|from)\s+oracle", src, re.M), fn
    for fn in os.listdir(os.path.join(ROOT, "paper_2111_14999_b200", "csrc")):
        assert "oracle" not in open(os.path.join(ROOT, "paper_2111_14999_b200", "csrc", fn)).read(), fn
