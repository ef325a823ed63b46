"""mg_residual_norm_static: the residual norm for callers that cannot allocate.

Some users of libmg have no way to call cudaMalloc at the moment they want ||rhs - A p||: a
flow solver that gave all device memory to its own pool at start-up (the paper does this,
PAPER.md section 4.2), or a convergence monitor inside a running time loop, where the
device-wide synchronisation of cudaMalloc / cudaFree would stall the host application.  Every
other entry point needs a handle, and making a handle allocates.  This entry point takes only
the caller's inputs and output and keeps its per-block partial sums in a fixed array inside the
library (128 KB, at most 2^27 cells).

The test compares it with the existing path (`Multigrid.residual`, i.e. mg_set_density +
mg_residual on a handle) on two calls in a row with different grids, densities and boundary
types, within the norm tolerance of tests/test_gpu_parity.py (relative 1e-10).  The second
grid is smaller than the first, so a call that read slots left over from the one before
would fail.  The file sorts last on purpose: `pytest -x` stops at the first failure and a
failure here must not hide the parity tests.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

NORM_RTOL = 1e-10          # the bar of tests/test_gpu_parity.py for residual norms


@pytest.fixture(scope="module")
def mgmod():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2605_30082_b200 as m
    return m


def fields(uniform, seed, n):
    shape = (n[2], n[1], n[0])
    rho = np.exp(uniform(seed, shape, np.log(1.2), np.log(998.0)))
    rhs = uniform(seed + 1, shape)
    p = uniform(seed + 2, shape)
    return [torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0") for a in (rho, rhs, p)]


def existing_path(mgmod, n, h, bc, rho, rhs, p):
    g = mgmod.Multigrid(n, h, bc)
    g.set_density(rho)
    ref = g.residual(rhs, p)
    g.close()
    return ref


def test_two_calls_in_a_row_match_the_handle_path(mgmod, uniform):
    # ragged against the 8192-cell chunks; walls on different axes; the second grid is smaller
    cases = [((72, 40, 36), 1.0 / 72, (0, 1, 1), 11), ((24, 48, 20), 1.0 / 48, (1, 0, 0), 23)]
    inputs = [fields(uniform, seed, n) for n, _, _, seed in cases]
    outs = [torch.full((1,), -1.0, dtype=torch.float64, device="cuda:0") for _ in cases]
    # both calls back to back on one stream, nothing in between
    for (n, h, bc, _), (rho, rhs, p), out in zip(cases, inputs, outs):
        mgmod.residual_norm_static(n, h, bc, rho, rhs, p, out)
    got = [float(o.item()) for o in outs]
    for (n, h, bc, _), (rho, rhs, p), val in zip(cases, inputs, got):
        ref = existing_path(mgmod, n, h, bc, rho, rhs, p)
        assert ref > 0.0
        assert abs(val - ref) <= NORM_RTOL * ref, (n, bc, val, ref)
    # the same inputs once more: the array now holds the second call's sums
    (n, h, bc, _), (rho, rhs, p) = cases[0], inputs[0]
    again = torch.zeros(1, dtype=torch.float64, device="cuda:0")
    mgmod.residual_norm_static(n, h, bc, rho, rhs, p, again)
    assert float(again.item()) == got[0]          # fixed summation tree: same bits


def test_sizes_beyond_the_static_array_are_refused(mgmod):
    from paper_2605_30082_b200 import binding as B

    L = B.lib()
    import ctypes as C

    bc = (C.c_int * 3)(0, 0, 0)
    one = torch.zeros(8, dtype=torch.float64, device="cuda:0")
    ptr = one.data_ptr()
    # 1024 x 512 x 512 = 2^28 cells > MG_STATIC_MAX_CELLS; rejected before any pointer is used
    assert L.mg_residual_norm_static(1024, 512, 512, 1.0, bc, ptr, ptr, ptr, ptr, None) == B.MG_EINVAL
    msg = L.mg_last_cuda_error().decode()
    assert "MG_STATIC_MAX_CELLS" in msg and str(B.MG_STATIC_MAX_CELLS) in msg
    assert 512 ** 3 == B.MG_STATIC_MAX_CELLS       # the largest grid it takes is the paper's per-device load
    bad = (C.c_int * 3)(0, 2, 0)                    # Dirichlet sides are mg_create6's
    assert L.mg_residual_norm_static(8, 8, 8, 1.0, bad, ptr, ptr, ptr, ptr, None) == B.MG_EINVAL
    assert L.mg_residual_norm_static(8, 8, 8, 1.0, bc, None, ptr, ptr, ptr, None) == B.MG_EINVAL


def test_largest_admitted_grid(mgmod):
    """512^3 = MG_STATIC_MAX_CELLS exactly: every slot of the static array is in use."""
    n, h, bc = (512, 512, 512), 1.0 / 512, (0, 0, 1)
    gen = torch.Generator(device="cuda:0").manual_seed(5)
    shape = (n[2], n[1], n[0])
    rho = torch.exp(torch.rand(shape, dtype=torch.float64, device="cuda:0", generator=gen) * 6.7 + 0.18)
    rhs = torch.rand(shape, dtype=torch.float64, device="cuda:0", generator=gen) - 0.5
    p = torch.rand(shape, dtype=torch.float64, device="cuda:0", generator=gen) - 0.5
    out = torch.zeros(1, dtype=torch.float64, device="cuda:0")
    mgmod.residual_norm_static(n, h, bc, rho, rhs, p, out)
    val = float(out.item())
    ref = existing_path(mgmod, n, h, bc, rho, rhs, p)
    assert abs(val - ref) <= NORM_RTOL * ref, (val, ref)
