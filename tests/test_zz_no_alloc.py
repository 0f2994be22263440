"""gf_theta_static: theta for host programs that cannot allocate GPU memory (collected last on purpose).

Some users of this library run it inside a program that took the whole GPU into its own memory pool when it
started, or that shares the GPU under a fixed memory budget; a cudaMalloc made behind their back fails or takes
memory they have promised elsewhere, and each cudaMalloc / cudaFree stalls the device in the middle of their loop.
Every other reduction goes through a gf_ctx, whose creation allocates.  gf_theta_static (include/gf.h) takes only the
caller's field and the caller's output buffer; its block partials go to a fixed 1 MiB array inside libgf.so that all
calls on a GPU share and that keeps the previous call's contents.

What is checked: the new entry point gives the numbers of the existing path (gf_theta / gf_theta_slices on a context:
same kernels, same summation order) on two calls in a row -- the second on a smaller lattice, so that it runs over
whatever the first left in the shared array -- and then on the first field again; and a lattice beyond the array's
size is refused with a message, not truncated.  The tolerance is the one tests/test_gpu_parity.py uses for the
reductions (relative 1e-10).

The file sorts after every other test file: `pytest -x` stops at the first failure, so a failure here cannot hide
another test.  It needs nothing from the tests before it and passes alone in a fresh process as well.
"""
import numpy as np
import pytest

import gf_inputs

pytestmark = pytest.mark.gpu

RTOL = 1e-10  # tests/test_gpu_parity.py::test_functional_and_theta


@pytest.fixture(scope="module")
def gfm():
    import torch

    assert torch.cuda.is_available()
    import paper_1209_4008_b200 as m

    m.load_library()  # fails loudly if the CUDA library is missing
    return m


def _existing_path(fx):
    """theta through the context: (whole lattice or max over slices as the gauge says, per-timeslice values)"""
    return fx.theta(), np.array(fx.theta_slices())


def _static_path(gfm, fx, out):
    """theta through gf_theta_static into the caller's buffer `out` (Nt + 2 doubles on the device)"""
    import torch

    out.fill_(float("nan"))  # every entry must be written by the call
    gfm.gf_theta_static(fx.dims, fx.precision, fx.gauge, fx.R, fx.U, out)
    torch.cuda.current_stream().synchronize()
    return out.cpu().numpy()


def _check(gfm, fx, out):
    theta, slices = _existing_path(fx)
    got = _static_path(gfm, fx, out)
    Nt = fx.dims[3]
    assert np.all(np.isfinite(got[: Nt + 2]))
    np.testing.assert_allclose(got[2 : 2 + Nt], slices, rtol=RTOL, atol=0)
    assert got[1] == pytest.approx(slices.max(), rel=RTOL)
    assert got[0] == pytest.approx(slices.mean(), rel=1e-9)  # equal slice volumes: the lattice value is their mean
    assert (got[1] if fx.gauge == gfm.GF_COULOMB else got[0]) == pytest.approx(theta, rel=RTOL)


@pytest.mark.parametrize("precision,R,gauge", [("fp64", 18, "landau"), ("fp32", 12, "coulomb"), ("fp32", 18, "landau"),
                                               ("fp64", 12, "coulomb")])
def test_two_calls_in_a_row_match_the_context_path(gfm, precision, R, gauge):
    import torch

    big, small = (16, 12, 10, 8), (6, 4, 4, 4)  # several blocks per timeslice with a ragged last one; one block
    fx_big = gfm.GaugeFixer(big, precision=precision, gauge=gauge, reals_per_link=R)
    fx_small = gfm.GaugeFixer(small, precision=precision, gauge=gauge, reals_per_link=R)
    fx_big.load(gf_inputs.smooth_random(big, 0.4, 31))
    fx_small.load(gf_inputs.smooth_random(small, 0.4, 32))
    fx_big.overrelax(1.7, 2)  # partly fixed: theta no longer O(1), slices differ
    fx_small.overrelax(1.7, 2)
    torch.cuda.synchronize()
    out_big = torch.empty(big[3] + 2, dtype=torch.float64, device="cuda")
    out_small = torch.empty(small[3] + 2, dtype=torch.float64, device="cuda")
    _check(gfm, fx_big, out_big)      # first call: leaves its partials in the shared array
    _check(gfm, fx_small, out_small)  # second call, straight after: must not see them
    _check(gfm, fx_big, out_big)      # and the first field again gives the first answer
    fx_big.close()
    fx_small.close()


def test_same_call_twice_is_bit_identical(gfm):
    import torch

    dims = (8, 8, 8, 8)
    fx = gfm.GaugeFixer(dims, precision="fp64")
    fx.load(gf_inputs.smooth_random(dims, 0.4, 33))
    out = torch.empty(dims[3] + 2, dtype=torch.float64, device="cuda")
    first = _static_path(gfm, fx, out).copy()
    second = _static_path(gfm, fx, out)
    assert np.array_equal(first, second)
    fx.close()


def test_lattice_beyond_the_builtin_scratch_is_refused(gfm):
    import torch

    limit = gfm.gf_theta_static_max_partials()
    assert limit == 131072
    # 2 * Nt * ceil(Nx/2 * Ny * Nz / 256): 64^3 x 128 uses the array exactly, 64^3 x 130 is one step too far
    dummy = torch.zeros(64, dtype=torch.float64, device="cuda")  # never read: the call must stop before any launch
    with pytest.raises(gfm.GFError) as err:
        gfm.gf_theta_static((64, 64, 64, 130), gfm.GF_FP32, gfm.GF_LANDAU, 12, dummy, dummy)
    assert err.value.code == gfm.GF_EINVAL
    assert "133120" in str(err.value) and "131072" in str(err.value)
    with pytest.raises(gfm.GFError) as err:
        gfm.gf_theta_static((8, 8, 8, 7), gfm.GF_FP32, gfm.GF_LANDAU, 12, dummy, dummy)
    assert err.value.code == gfm.GF_EINVAL
    with pytest.raises(gfm.GFError) as err:
        gfm.gf_theta_static((8, 8, 8, 8), gfm.GF_FP32, gfm.GF_LANDAU, 15, dummy, dummy)
    assert err.value.code == gfm.GF_EINVAL
    torch.cuda.synchronize()
