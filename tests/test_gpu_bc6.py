"""GPU parity of per-side boundary conditions with Dirichlet walls (mg_create6; SURVEY 8(f) rank 3,
DESIGN.md R24): the CUDA path (level-generic kernels with wall logic) against the CPU
oracle (mgo_create6), element by element on identical seeded inputs.  Bars as in
test_gpu_parity.py: single steps and cycles bit-exact, norms 1e-10, p after the solve 1e-9.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle.mgo import Oracle  # noqa: E402

P, N, D = 0, 1, 2
NORM_RTOL = 1e-10
P_RTOL = 1e-9

PAPER_BOX = (N, D, N, D, N, D)      # symmetry planes x-, y-; no-slip base z-; outflow x+, y+, z+

CASES = [
    ((32, 32, 32), PAPER_BOX),
    ((96, 64, 48), PAPER_BOX),               # several tiles and z-chunks of the TMA kernel
    ((64, 72, 32), (D, N, D, D, D, N)),
    ((48, 32, 24), (D, D, P, P, N, D)),
    ((40, 24, 56), (P, P, D, N, D, D)),
    ((64, 64, 64), (N, N, N, N, N, D)),
    ((72, 40, 36), (D, N, N, N, P, P)),
]


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


def random_rho(uniform, seed, shape):
    return np.exp(uniform(seed, shape, np.log(1.2), np.log(998.0)))


def pair(mgmod, n, bc, nu=(2, 2), rho=None, coarse_sweeps=32, cycle_type=0, kernels=1):
    from paper_2605_30082_b200 import binding as B

    o = Oracle(n, 1.0 / n[0], bc, nu[0], nu[1], coarse_sweeps)
    g = mgmod.Multigrid(n, 1.0 / n[0], bc, nu[0], nu[1], coarse_sweeps)
    g.set_option(B.MG_OPT_KERNELS, kernels)      # 1 (default): TMA sweeps on level 0; 0: level-generic kernels only
    o.set_cycle_type(cycle_type)
    g.set_cycle_type(cycle_type)
    if rho is not None:
        o.set_density(rho)
        g.set_density(dev(rho))
    return o, g


@pytest.mark.parametrize("n,bc", CASES)
def test_steps_bit_exact_with_dirichlet_walls(mgmod, uniform, n, bc):
    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, bc, rho=random_rho(uniform, 121, shp))
    assert o.num_levels == g.num_levels
    for lvl in range(o.num_levels):
        lshp = o.level_shape(lvl)
        for bo, bg in zip(o.faces(lvl), g.level_faces(lvl)):        # minus faces incl. the minus walls
            assert np.array_equal(bo, host(bg)), f"faces level {lvl}"
        f, p0 = uniform(130 + lvl, lshp), uniform(140 + lvl, lshp)
        po, pg, fd = p0.copy(), dev(p0), dev(f)
        for colour in (0, 1, 0):
            o.smooth_half(colour, f, po, lvl)
            g.level_smooth_half(lvl, colour, fd, pg)
            assert np.array_equal(po, host(pg)), f"half sweep colour {colour} level {lvl}"
        # the residual sees every wall coefficient (plus walls included)
        assert np.array_equal(o.residual_level(f, po, lvl), host(g.level_residual(lvl, fd, pg))), f"residual level {lvl}"
        if lvl < o.num_levels - 1:
            fc_o = o.restrict(o.residual_level(f, po, lvl), lvl)
            assert np.array_equal(fc_o, host(g.level_residual_restrict(lvl, fd, pg)))
            e = uniform(150 + lvl, o.level_shape(lvl + 1))
            o.prolong_add(e, po, lvl)
            g.level_prolong_add(lvl, dev(e), pg)
            assert np.array_equal(po, host(pg)), f"prolong level {lvl}"


@pytest.mark.parametrize("n,bc", CASES)
@pytest.mark.parametrize("sweeps", [1, 2, 3])
def test_level0_sweeps_and_tails_with_dirichlet_walls(mgmod, uniform, n, bc, sweeps):
    """The TMA kernel on level 0 (k_rbt WALLS): sweeps, fused pairs, restriction and norm tails."""
    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, bc, rho=random_rho(uniform, 126, shp))
    f, p0 = uniform(127, shp), uniform(128, shp)
    po = p0.copy()
    for _ in range(sweeps):
        o.sweep(f, po, 0)
    pg = dev(p0)
    g.level_smooth(0, sweeps, dev(f), pg)
    assert np.array_equal(po, host(pg))
    pg = dev(p0)
    fc_g = g.level_smooth_restrict(0, sweeps, dev(f), pg)
    assert np.array_equal(po, host(pg))
    assert np.array_equal(o.restrict(o.residual_level(f, po, 0), 0), host(fc_g))
    pg = dev(p0)
    nrm = g.level_smooth_norm(sweeps, dev(f), pg)
    assert np.array_equal(po, host(pg))
    assert nrm == pytest.approx(o.residual(f, po), rel=NORM_RTOL)


@pytest.mark.parametrize("n,bc", CASES)
@pytest.mark.parametrize("cycle_type", [0, 1], ids=["V", "F"])
@pytest.mark.parametrize("kernels,cta", [(0, 0), (1, 1), (1, 0)])
def test_cycles_bit_exact_with_dirichlet_walls(mgmod, uniform, n, bc, cycle_type, kernels, cta):
    from paper_2605_30082_b200 import binding as B

    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, bc, nu=(3, 3), rho=random_rho(uniform, 122, shp), coarse_sweeps=8, cycle_type=cycle_type,
                kernels=kernels)
    g.set_option(B.MG_OPT_COARSE_CTA, cta)      # levels <= 16^3 in the persistent CTA (wall logic included) or launch by launch
    f = uniform(123, shp) + 0.25          # non-singular: the rhs need not be mean-free
    po, pg, fd = np.zeros(shp), dev(np.zeros(shp)), dev(f)
    for cyc in range(3):
        o.vcycle(f, po)
        g.vcycle(fd, pg)
        assert np.array_equal(po, host(pg)), f"cycle {cyc}"
    assert g.residual(fd, pg) == pytest.approx(o.residual(f, po), rel=NORM_RTOL)


# stored-face levels of a solver with Dirichlet sides in the TMA kernel (k_rbt<.., CELL = false, WALLS>):
# the plus-wall faces wx, wy are patched into the bx / by tiles, wz replaces the zero-filled bz plane
FACE_CASES = [
    ((96, 64, 48), PAPER_BOX),                      # level 1 = 48 x 32 x 24: one tile, all three plus walls Dirichlet
    ((64, 72, 32), (D, N, D, D, D, N)),
    ((64, 64, 64), (N, N, N, N, N, D)),
    ((160, 144, 64), PAPER_BOX),                    # level 1 = 80 x 72 x 32: several tiles in x and y
    ((144, 160, 96), (P, P, D, D, N, D)),           # periodic images in x along the Dirichlet y walls; level 2 streams too
    ((128, 136, 64), (D, D, P, P, D, N)),           # periodic images in y along the Dirichlet x walls
    ((136, 128, 80), (N, D, N, D, P, P)),           # periodic z
]


@pytest.mark.parametrize("n,bc", FACE_CASES)
@pytest.mark.parametrize("fuse", [1, 3])
def test_face_levels_streamed_with_dirichlet_walls(mgmod, uniform, n, bc, fuse):
    from paper_2605_30082_b200 import binding as B

    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, bc, rho=random_rho(uniform, 161, shp))
    g.set_option(B.MG_OPT_FACE_STREAM_LOG2, 0)
    g.set_option(B.MG_OPT_SWEEP_FUSE, fuse)
    g.set_option(B.MG_OPT_TAIL_FUSION, 2)
    tested = 0
    for lvl in range(1, o.num_levels - 1):
        lshp = o.level_shape(lvl)
        if min(lshp[1], lshp[2]) < 32 or lshp[0] < 16:
            break
        tested += 1
        f, p0 = uniform(162 + lvl, lshp), uniform(166 + lvl, lshp)
        fd = dev(f)
        for sweeps in (1, 2, 3, 4):
            po = p0.copy()
            for _ in range(sweeps):
                o.sweep(f, po, lvl)
            pg = dev(p0)
            g.level_smooth(lvl, sweeps, fd, pg)
            assert np.array_equal(po, host(pg)), f"level {lvl}, {sweeps} sweeps"
            fc_o = o.restrict(o.residual_level(f, po, lvl), lvl)
            pg = dev(p0)
            fc_g = g.level_smooth_restrict(lvl, sweeps, fd, pg)
            assert np.array_equal(po, host(pg)), f"level {lvl}, {sweeps} sweeps + tail: p"
            assert np.array_equal(fc_o, host(fc_g)), f"level {lvl}, {sweeps} sweeps + tail: coarse rhs"
    assert tested >= 1


@pytest.mark.parametrize("n,bc", FACE_CASES)
@pytest.mark.parametrize("cycle_type", [0, 1], ids=["V", "F"])
@pytest.mark.parametrize("tails", [1, 2])
def test_cycles_face_levels_streamed_with_dirichlet_walls(mgmod, uniform, n, bc, cycle_type, tails):
    from paper_2605_30082_b200 import binding as B

    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, bc, nu=(3, 3), rho=random_rho(uniform, 171, shp), coarse_sweeps=8, cycle_type=cycle_type)
    g.set_option(B.MG_OPT_FACE_STREAM_LOG2, 0)
    g.set_option(B.MG_OPT_TAIL_FUSION, tails)
    f = uniform(172, shp) + 0.25
    po, pg, fd = np.zeros(shp), dev(np.zeros(shp)), dev(f)
    for cyc in range(2):
        o.vcycle(f, po)
        g.vcycle(fd, pg)
        assert np.array_equal(po, host(pg)), f"cycle {cyc}"
    assert g.residual(fd, pg) == pytest.approx(o.residual(f, po), rel=NORM_RTOL)


@pytest.mark.parametrize("size", [64, 256])
def test_solve_on_the_papers_box(mgmod, uniform, size):
    """Drop-film densities in the paper's box: no-slip base, symmetry planes, outflow planes;
    at 64^3 and at config 3's full 256^3 (level 0 runs the TMA kernel with walls, two sweeps per
    pass from 2^26 cells only, so 256^3 takes the one-sweep passes)."""
    from workloads import make_workload

    w = make_workload(3, size)
    o, g = pair(mgmod, w.n, PAPER_BOX, nu=(w.nu1, w.nu2), rho=w.rho)
    f = w.rhs + 0.1                        # no compatibility condition with a Dirichlet wall
    po = np.zeros(o.shape)
    so, co, ro, ho = o.solve(f, po, w.rtol, 60)
    pg = dev(np.zeros(o.shape))
    sg, cg, rg, hg = g.solve(dev(f), pg, w.rtol, 60)
    assert so == 0 and (sg, cg) == (so, co)
    hg = np.array(hg)
    assert np.all(np.abs(hg / ho - 1) <= NORM_RTOL), (hg, ho)
    pgh = host(pg)
    assert np.abs(pgh - po).max() <= P_RTOL * np.abs(po).max()
    assert abs(po.mean()) > 1e-6 * np.abs(po).max()          # no mean was removed on either side


def test_dirichlet_solver_refuses_what_it_does_not_define(mgmod):
    from paper_2605_30082_b200 import binding as B

    g = mgmod.Multigrid((16, 16, 16), 1.0 / 16, PAPER_BOX)
    z = torch.zeros(g.shape, dtype=torch.float64, device="cuda:0")
    with pytest.raises(B.MgError):
        g.project_rhs(z, z, z, 1.0, z.clone())
    for bad in [(P, N, P, P, P, P), (3, 3, N, N, N, N)]:
        with pytest.raises(B.MgError):
            mgmod.Multigrid((16, 16, 16), 1.0 / 16, bad)


def test_six_entry_form_without_dirichlet_is_the_streaming_path(mgmod, uniform):
    """(P,P,P,P,N,N) through mg_create6 = (P,P,N) through mg_create: same kernels, same bits."""
    n = (64, 64, 64)
    shp = (64, 64, 64)
    rho = random_rho(uniform, 124, shp)
    f = uniform(125, shp)
    f -= f.mean()
    outs = []
    for bc in ((P, P, N), (P, P, P, P, N, N)):
        g = mgmod.Multigrid(n, 1.0 / 64, bc, 3, 3)
        g.set_density(dev(rho))
        p = dev(np.zeros(shp))
        g.vcycle(dev(f), p)
        outs.append(host(p))
    assert np.array_equal(outs[0], outs[1])
