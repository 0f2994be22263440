"""The C-ABI library loads and exports every symbol include/gf.h declares (no GPU needed, no compute calls);
without a CUDA device the product path fails loudly instead of falling back to anything."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "gf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gf_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_1209_4008_b200 import build

    build.build()  # nvcc cross-compiles sm_100a without a GPU
    import paper_1209_4008_b200 as m

    return m


def test_header_and_binding_agree(lib):
    declared = _declared_symbols()
    assert len(declared) >= 15
    assert declared == sorted(lib.SIGNATURES)


def test_library_exports_every_declared_symbol(lib):
    cdll = lib.load_library()
    for name in _declared_symbols():
        assert getattr(cdll, name) is not None, name


def test_sm100a_code_is_embedded(lib):
    import subprocess

    out = subprocess.run(["cuobjdump", "-lelf", lib.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_no_cpu_fallback(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(lib.GFError) as err:
        lib.gf_create(4, 4, 4, 4, lib.GF_FP64, lib.GF_LANDAU)
    assert err.value.code == lib.GF_ECUDA
    with pytest.raises(RuntimeError):
        lib.GaugeFixer((4, 4, 4, 4))


def test_create_rejects_bad_extents_before_touching_the_device(lib):
    for dims in [(3, 4, 4, 4), (4, 4, 4, 0), (4, 5, 4, 4), (-2, 4, 4, 4)]:
        with pytest.raises(lib.GFError) as err:
            lib.gf_create(*dims, lib.GF_FP64, lib.GF_LANDAU)
        assert err.value.code == lib.GF_EINVAL


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1209_4008_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "gf_oracle" not in src and "liborc" not in src, f
