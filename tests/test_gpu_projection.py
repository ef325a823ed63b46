"""GPU parity of the projection steps (mg_project_rhs, mg_project_correct, mg_project) against
the CPU oracle: bit-exact fields (both sides implement C10 / C11 with IEEE fp64 sub, add, mul,
fma), the solve inside mg_project to the tolerances of the pressure solve."""
import itertools
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle.mgo import Oracle  # noqa: E402
from workloads import make_workload  # noqa: E402

P, N = 0, 1


@pytest.fixture(scope="module")
def mgmod():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2605_30082_b200 as m
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def host(t):
    return t.detach().cpu().numpy()


def staggered(uniform, seed, shape, bc):
    u, v, w = (uniform(seed + q, shape) for q in range(3))
    if bc[0] == N:
        u[:, :, 0] = 0.0
    if bc[1] == N:
        v[:, 0, :] = 0.0
    if bc[2] == N:
        w[0, :, :] = 0.0
    return u, v, w


SHAPES = [((32, 32, 32), (P, P, P)), ((48, 32, 24), (N, P, N)), ((40, 24, 56), (P, N, P)),
          ((64, 16, 8), (N, N, N)), ((8, 8, 8), (P, P, N)), ((72, 40, 36), (P, N, N)),
          ((130, 34, 18), (N, P, P))]       # 130: ragged against the 64-cell strips, two strips + 2


@pytest.mark.parametrize("n,bc", SHAPES)
def test_rhs_and_correct_bit_exact(mgmod, uniform, n, bc):
    h, dt = 1.0 / n[0], 3.0e-3
    shp = (n[2], n[1], n[0])
    rho = np.exp(uniform(5, shp, math.log(1.2), math.log(998.0)))
    o = Oracle(n, h, bc)
    o.set_density(rho)
    g = mgmod.Multigrid(n, h, bc)
    g.set_density(dev(rho))
    u, v, w = staggered(uniform, 50, shp, bc)
    p = uniform(60, shp)
    # rhs
    fo = o.project_rhs(u, v, w, dt)
    fg = torch.empty(shp, dtype=torch.float64, device="cuda:0")
    g.project_rhs(dev(u), dev(v), dev(w), dt, fg)
    assert np.array_equal(fo, host(fg))
    # correction
    uo, vo, wo = u.copy(), v.copy(), w.copy()
    o.project_correct(p, dt, uo, vo, wo)
    ug, vg, wg = dev(u), dev(v), dev(w)
    g.project_correct(dev(p), dt, ug, vg, wg)
    assert np.array_equal(uo, host(ug)) and np.array_equal(vo, host(vg)) and np.array_equal(wo, host(wg))


def test_whole_projection_step_config3_twin(mgmod, uniform):
    """rhs -> solve -> correct on the 64^3 drop-film twin: same cycle count as the oracle, p to
    1e-9, corrected velocity to 1e-9 of its scale, and the projected field is divergence-free
    to the residual of the solve."""
    w_ = make_workload(3, 64)
    dt = 1.0e-2
    o = Oracle(w_.n, w_.h, w_.bc, w_.nu1, w_.nu2)
    o.set_density(w_.rho)
    g = mgmod.Multigrid(w_.n, w_.h, w_.bc, w_.nu1, w_.nu2)
    g.set_density(dev(w_.rho))
    u, v, w = staggered(uniform, 70, o.shape, w_.bc)
    # oracle
    fo = o.project_rhs(u, v, w, dt)
    po = np.zeros(o.shape)
    so, co, ro, ho = o.solve(fo, po, w_.rtol, 60)
    uo, vo, wo = u.copy(), v.copy(), w.copy()
    o.project_correct(po, dt, uo, vo, wo)
    # CUDA path
    ug, vg, wg = dev(u), dev(v), dev(w)
    pg = torch.zeros(o.shape, dtype=torch.float64, device="cuda:0")
    rhs = torch.empty_like(pg)
    sg, cg, rg = g.project(ug, vg, wg, dt, pg, rhs, w_.rtol, 60)
    assert (sg, cg) == (so, co)
    assert np.array_equal(fo, host(rhs))
    assert rg == pytest.approx(ro, rel=1e-10)
    assert np.abs(host(pg) - po).max() <= 1e-9 * np.abs(po).max()
    scale = max(np.abs(uo).max(), np.abs(vo).max(), np.abs(wo).max())
    for a, b in ((uo, ug), (vo, vg), (wo, wg)):
        assert np.abs(a - host(b)).max() <= 1e-9 * scale
    d = torch.empty_like(pg)
    g.project_rhs(ug, vg, wg, dt, d)
    assert float(torch.linalg.vector_norm(d)) <= 2 * w_.rtol * float(np.sqrt((fo ** 2).sum()))


def test_projection_error_codes(mgmod):
    from paper_2605_30082_b200 import binding as B
    g = mgmod.Multigrid(8, 0.125, (P, P, P))
    z = torch.zeros(g.shape, dtype=torch.float64, device="cuda:0")
    for bad in (0.0, -1.0, float("nan"), float("inf")):
        with pytest.raises(B.MgError) as e:
            g.project_rhs(z, z, z, bad, z.clone())
        assert e.value.code == B.MG_EINVAL
        with pytest.raises(B.MgError):
            g.project_correct(z, bad, z.clone(), z.clone(), z.clone())
