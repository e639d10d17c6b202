"""CPU-only checks of the boundary: librbq_b200.so builds for sm_100a without a GPU, loads, and exports
every function include/rbq.h declares (and nothing in the binding is missing); the binding refuses to
compute without a CUDA device (no CPU fallback); the product package does not import the oracle.
No compute call is made here.
"""
import ctypes as C
import re
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def lib_path():
    from paper_2606_31519_b200 import build
    return build.build()


def declared_functions():
    text = (ROOT / "include" / "rbq.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rbq_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for need in ["rbq_encode_keys", "rbq_append_tokens", "rbq_estimate_scores", "rbq_topp_select",
                 "rbq_sparse_attention", "rbq_decode_step"]:
        assert need in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = C.CDLL(str(lib_path))
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} declared in include/rbq.h but not exported"
    out = subprocess.run(["nm", "-D", "--defined-only", str(lib_path)], capture_output=True, text=True).stdout
    exported = set(re.findall(r" T (rbq_[a-z0-9_]+)$", out, flags=re.M))
    assert set(declared_functions()) <= exported


def test_binding_covers_the_header(lib_path):
    from paper_2606_31519_b200 import binding
    assert sorted(binding.EXPORTS) == declared_functions()
    lib = binding.load()
    for name in binding.EXPORTS:
        assert getattr(lib, name).argtypes is not None
        assert hasattr(binding, name) or name in ("rbq_last_error",)


def test_library_is_sm100a_only(lib_path):
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-lelf", str(lib_path)], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_no_cpu_fallback_without_gpu(lib_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2606_31519_b200 import binding
    cfg = binding.rbq_config(1, 1, 1, 128, 64, 0, 0, 0, 0, 0.0, 0, 1, 0)
    with pytest.raises(binding.RbqError):
        binding.rbq_create(cfg)
    h = C.c_void_p()
    assert binding.load().rbq_create(C.byref(cfg), C.byref(h)) == -4         # RBQ_ERR_CUDA from the C ABI itself


def test_product_does_not_touch_the_oracle():
    pkg = ROOT / "paper_2606_31519_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")) + [ROOT / "include" / "rbq.h"]:
        src = f.read_text()
        assert "rbq_ref" not in src and "rbq_oracle" not in src and "import oracle" not in src, f
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".c"):
            src = f.read_text()
            assert "paper_2606_31519_b200" not in src.replace("paper_2606_31519_b200/csrc (the CUDA path)", "").replace(
                "(paper_2606_31519_b200/csrc, binding.py)", ""), f
