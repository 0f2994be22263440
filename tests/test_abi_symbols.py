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


def test_kp_tables_are_what_their_generator_writes():
    """csrc/gf_kp_tables.inc (constants of the fp64 annealing draw's -ln u / sin / cos) is the output of the committed
    generator, and its table obeys what the kernel relies on: r_j has at most 10 significant bits (m r_j - 1 exact),
    |m r_j - 1| < 0.006 over the bin, T_j = -ln r_j (minus ln 2 in the upper half), last bin exactly (1/2, 0)."""
    import math
    import re
    import subprocess
    import sys

    here = os.path.join(ROOT, "paper_1209_4008_b200", "csrc")
    out = subprocess.run([sys.executable, os.path.join(here, "gen_kp_tables.py")], capture_output=True, text=True, check=True).stdout
    with open(os.path.join(here, "gf_kp_tables.inc")) as fh:
        assert fh.read() == out
    rows = re.findall(r"\{(0x[0-9a-fp.+-]+), (-?0x[0-9a-fp.+-]+)\}", out)
    assert len(rows) == 128
    for j, (r, t) in enumerate(rows):
        r, t = float.fromhex(r), float.fromhex(t)
        assert (r * 1024).is_integer() and 0.5 <= r <= 1.0
        lo, hi = 1 + j / 128, 1 + (j + 1) / 128
        assert max(abs(lo * r - 1), abs(hi * r - 1)) < 0.006
        want = -math.log(r) - (math.log(2) if j >= 64 else 0.0)
        assert abs(t - want) <= 2e-16
    assert rows[127] == ("0x1.0000000000000p-1", "0x0.0p+0")


def test_theta_static_refuses_oversized_lattices_before_touching_the_device(lib):
    """gf_theta_static (no allocation, fixed 1 MiB scratch inside the library): the size check is host arithmetic and
    comes before any CUDA call, so it can be checked without a GPU."""
    assert lib.gf_theta_static_max_partials() == 131072
    with pytest.raises(lib.GFError) as err:
        lib.gf_theta_static((64, 64, 64, 130), lib.GF_FP32, lib.GF_LANDAU, 12, 256, 256, stream=0)
    assert err.value.code == lib.GF_EINVAL
    assert "133120" in str(err.value) and "131072" in str(err.value)
    for dims in [(3, 4, 4, 4), (4, 4, 4, 0)]:
        with pytest.raises(lib.GFError) as err:
            lib.gf_theta_static(dims, lib.GF_FP64, lib.GF_LANDAU, 18, 256, 256, stream=0)
        assert err.value.code == lib.GF_EINVAL
