"""CPU-side checks of the C-ABI boundary: the library builds, loads, exports every symbol that
include/dgpe.h declares, validates its arguments, and fails loudly (no CPU fallback) without a GPU.
No compute call is made here."""
import ctypes as C
import os
import re

import pytest
import torch

from paper_1610_05329_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "dgpe.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dgpe_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported():
    L = binding.lib()
    names = declared_symbols()
    assert len(names) >= 18
    for n in names:
        assert hasattr(L, n), n
    assert set(binding.EXPORTS) == set(names)


def test_header_cites_the_paper_for_each_stage():
    text = open(os.path.join(ROOT, "include", "dgpe.h")).read()
    for cite in ("P:L31", "P:L33", "P:L39", "P:L45", "P:L130", "P:L132", "BJ:north_star", "BJ:configs[0]"):
        assert cite in text, cite


@pytest.mark.parametrize("args,frag", [
    ((64, 64, 34, .1, .1, .1, .01, 1, 1, 1, 1, 1, 0), "2^a 3^b 5^c 7^d 11^e 13^f"),       # 34 = 2*17
    ((64, 64, 54, .1, .1, .1, .01, 1, 1, 1, 1, 1, 3), "mode"),
    ((2, 64, 64, .1, .1, .1, .01, 1, 1, 1, 1, 1, 0), "< 4"),
    ((64, 64, 27, .1, .1, .1, .01, 1, 1, 1, 1, 1, 0), "even"),
    ((64, 76, 64, .1, .1, .1, .01, 1, 1, 1, 1, 1, 0), "2^a 3^b 5^c 7^d 11^e 13^f"),       # 76 = 4*19
    ((64, 64, 64, .1, -.1, .1, .01, 1, 1, 1, 1, 1, 0), "positive"),
    ((64, 64, 64, .1, .1, .1, 0.0, 1, 1, 1, 1, 1, 0), "positive"),
    ((2048, 64, 64, .1, .1, .1, .01, 1, 1, 1, 1, 1, 0), "> 1024"),
])
def test_create_rejects_bad_arguments(args, frag):
    L = binding.lib()
    h = L.dgpe_create(*args)
    assert not h
    assert frag in binding.last_error()


def test_null_arguments_are_errors_not_crashes():
    L = binding.lib()
    out = (C.c_double * 4)()
    assert L.dgpe_step(None, None, 1) == binding.ERR_ARG
    assert L.dgpe_step_host(None, None, 1) == binding.ERR_ARG
    assert L.dgpe_norm(None, None, out) == binding.ERR_ARG
    assert L.dgpe_sweep(None, None, 0) == binding.ERR_ARG
    assert L.dgpe_set_stream(None, None) == binding.ERR_ARG
    L.dgpe_destroy(None)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_gpu_means_failure_not_fallback():
    L = binding.lib()
    h = L.dgpe_create(64, 64, 64, .25, .25, .25, .005, 1, 1, 1, 20., 5., 0)
    assert not h
    assert "CUDA" in binding.last_error() or "cuda" in binding.last_error()
    with pytest.raises(RuntimeError):
        binding.Dgpe(64, 64, 64, .25, .25, .25, .005, 1, 1, 1, 20., 5., 0)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1610_05329_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "dgpe_oracle" not in src, f


def test_header_is_plain_c():
    """The boundary is a C ABI: include/dgpe.h must compile as C99 (no C++-only constructs, no torch or CUDA types)."""
    import shutil
    import subprocess
    if not shutil.which("gcc"):
        pytest.skip("gcc not found")
    hdr = os.path.join(ROOT, "include", "dgpe.h")
    res = subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-fsyntax-only", "-x", "c", hdr], capture_output=True, text=True)
    assert res.returncode == 0, res.stderr
    code = re.sub(r"/\*.*?\*/", "", open(hdr).read(), flags=re.S)        # the declarations, comments stripped
    assert "torch" not in code and "cudaStream_t" not in code and "#include" not in code
