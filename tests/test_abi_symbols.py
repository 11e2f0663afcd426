"""The C-ABI library loads and exports every symbol include/rfim_pt.h declares (no GPU, no compute)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_1508_06268_b200 import build
    return build.build()


def _declared():
    txt = open(os.path.join(ROOT, "include", "rfim_pt.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(rfim_pt_[a-z0-9_]+)\s*\(", txt)))


def test_every_declared_symbol_is_exported_and_bound(built_lib):
    from paper_1508_06268_b200 import binding
    lib = binding.load()
    declared = _declared()
    assert len(declared) >= 30
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in rfim_pt.h but not exported"
    assert sorted(binding.SIGNATURES) == declared, "binding.SIGNATURES and rfim_pt.h disagree"


def test_library_is_built_for_sm_100a(built_lib):
    import subprocess
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-lelf", built_lib], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_product_does_not_reach_the_oracle():
    # the product path must never import, link or read anything under oracle/
    pkg = os.path.join(ROOT, "paper_1508_06268_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f), errors="ignore").read()
                assert "import oracle" not in txt and "from oracle" not in txt and "rfim_oracle" not in txt, f
                for line in txt.splitlines():
                    if line.lstrip().startswith("#include"):
                        assert "oracle" not in line, (f, line)


def test_create_without_gpu_fails_loudly(built_lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1508_06268_b200 import binding
    with pytest.raises(RuntimeError):
        binding.RfimPT(8, 2, 1.0, 1.0, 0, seed=1)
    # and the raw C entry point refuses too (no CPU fallback inside the library)
    import ctypes
    h = ctypes.c_void_p()
    rc = binding.load().rfim_pt_create(ctypes.byref(h), 8, 2, 1.0, 1.0, 0, 1)
    assert rc == binding.ECUDA and not h.value
