"""GPU parity: the CUDA path (through the C ABI of include/mg.h) against the CPU oracle,
element by element on identical seeded inputs.

Bars (BASELINE.json north_star): fields of single steps and of V-cycles are
compared BIT-EXACTLY (both sides implement the expression trees C1-C9 with IEEE fp64
add/mul/fma/div); per-cycle residual norms within relative 1e-10 (the two sides only
differ in the summation order of the norm); p after the solve within 1e-9 max-abs
relative (the mean that is subtracted comes from differently ordered sums).
"""
import itertools

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle.mgo import Oracle  # noqa: E402
from workloads import make_workload  # noqa: E402

P, N = 0, 1
NORM_RTOL = 1e-10
P_RTOL = 1e-9


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


def pair(mgmod, n, h, bc, nu=(2, 2), rho=None, coarse_sweeps=32, **opts):
    o = Oracle(n, h, bc, nu[0], nu[1], coarse_sweeps)
    g = mgmod.Multigrid(n, h, bc, nu[0], nu[1], coarse_sweeps)
    from paper_2605_30082_b200 import binding as B
    for key, name in ((B.MG_OPT_KERNELS, "kernels"), (B.MG_OPT_GRAPH, "graph"), (B.MG_OPT_COARSE_CTA, "coarse_cta"),
                      (B.MG_OPT_TAIL_FUSION, "tails"), (B.MG_OPT_SWEEP_FUSE, "fuse"),
                      (B.MG_OPT_FACE_STREAM_LOG2, "face_log2"), (B.MG_OPT_PROLONG_FUSE, "head")):
        if name in opts:
            g.set_option(key, opts[name])
    if "cycle_type" in opts:
        o.set_cycle_type(opts["cycle_type"])
        g.set_cycle_type(opts["cycle_type"])
    if rho is not None:
        o.set_density(rho)
        g.set_density(dev(rho))
    return o, g


def random_rho(uniform, seed, shape):
    return np.exp(uniform(seed, shape, np.log(1.2), np.log(998.0)))


SHAPES = [
    ((32, 32, 32), (P, P, P)),
    ((32, 32, 32), (P, P, N)),
    ((48, 32, 24), (N, P, N)),     # non-cubic, coarsest 12x8x6
    ((40, 24, 56), (P, N, P)),     # ragged against every tile size, single coarsening
    ((64, 16, 8), (N, N, N)),
    ((8, 8, 8), (P, P, N)),
    ((4, 4, 4), (P, P, P)),        # single level
    ((72, 40, 36), (P, N, N)),     # streaming kernels: ragged tiles in x and y, walls in y and z
    ((64, 64, 64), (N, P, N)),     # streaming kernels on two levels, wall in x
    ((128, 32, 64), (P, P, P)),    # several x tiles, periodic wrap everywhere
]


# --------------------------------------------------------------------------- #
# single steps, every level, bit exact
# --------------------------------------------------------------------------- #
@pytest.mark.parametrize("n,bc", SHAPES)
def test_steps_bit_exact(mgmod, uniform, n, bc):
    h = 1.0 / n[0]
    rho = random_rho(uniform, 5, (n[2], n[1], n[0]))
    o, g = pair(mgmod, n, h, bc, rho=rho)
    assert o.num_levels == g.num_levels
    for lvl in range(o.num_levels):
        assert o.level_dims(lvl) == g.level_dims(lvl)
        shp = o.level_shape(lvl)
        # coefficients (A0)
        for bo, bg in zip(o.faces(lvl), g.level_faces(lvl)):
            assert np.array_equal(bo, host(bg)), f"faces level {lvl}"
        f, p0 = uniform(10 + lvl, shp), uniform(20 + lvl, shp)
        # half sweeps (A1/A6), both colours in order
        po, pg = p0.copy(), dev(p0)
        fd = dev(f)
        for colour in (0, 1, 0):
            o.smooth_half(colour, f, po, lvl)
            g.level_smooth_half(lvl, colour, fd, pg)
            assert np.array_equal(po, host(pg)), f"half sweep colour {colour} level {lvl}"
        # full sweeps through whichever kernels the cycle uses
        po2, pg2 = p0.copy(), dev(p0)
        for _ in range(3):
            o.sweep(f, po2, lvl)
        g.level_smooth(lvl, 3, fd, pg2)
        assert np.array_equal(po2, host(pg2)), f"3 sweeps level {lvl}"
        # residual (A2)
        assert np.array_equal(o.residual_level(f, po, lvl), host(g.level_residual(lvl, fd, pg)))
        if lvl < o.num_levels - 1:
            # residual + restriction (A2+A3)
            fc_o = o.restrict(o.residual_level(f, po, lvl), lvl)
            assert np.array_equal(fc_o, host(g.level_residual_restrict(lvl, fd, pg)))
            # prolongation + correction (A5)
            e = uniform(30 + lvl, o.level_shape(lvl + 1))
            o.prolong_add(e, po, lvl)
            g.level_prolong_add(lvl, dev(e), pg)
            assert np.array_equal(po, host(pg)), f"prolong level {lvl}"


# --------------------------------------------------------------------------- #
# fused tails of the TMA sweep kernel (SURVEY §8(a) A2+A3 behind the last pre-sweep, A7 behind
# the last post-sweep): p and the coarse right-hand side bit-exact, norm 1e-10
# --------------------------------------------------------------------------- #
TAIL_SHAPES = [
    ((64, 64, 64), (P, P, P)),
    ((64, 64, 64), (N, N, N)),
    ((72, 40, 36), (P, N, N)),      # ragged tiles, x periodic through a shifted last tile
    ((136, 72, 96), (N, P, P)),     # several tiles per axis and several z-chunks
    ((32, 32, 32), (P, P, N)),
]


@pytest.mark.parametrize("n,bc", TAIL_SHAPES)
@pytest.mark.parametrize("sweeps", [1, 2, 3])
def test_fused_restrict_tail_bit_exact(mgmod, uniform, n, bc, sweeps):
    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, 1.0 / n[0], bc, rho=random_rho(uniform, 51, shp))
    f, p0 = uniform(52, shp), uniform(53, shp)
    po = p0.copy()
    for _ in range(sweeps):
        o.sweep(f, po, 0)
    fc_o = o.restrict(o.residual_level(f, po, 0), 0)
    pg = dev(p0)
    fc_g = g.level_smooth_restrict(0, sweeps, dev(f), pg)
    assert np.array_equal(po, host(pg))
    assert np.array_equal(fc_o, host(fc_g))


@pytest.mark.parametrize("n,bc", TAIL_SHAPES)
@pytest.mark.parametrize("sweeps", [1, 2])
def test_fused_norm_tail(mgmod, uniform, n, bc, sweeps):
    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, 1.0 / n[0], bc, rho=random_rho(uniform, 54, shp))
    f, p0 = uniform(55, shp), uniform(56, shp)
    po = p0.copy()
    for _ in range(sweeps):
        o.sweep(f, po, 0)
    pg = dev(p0)
    nrm = g.level_smooth_norm(sweeps, dev(f), pg)
    assert np.array_equal(po, host(pg))
    assert nrm == pytest.approx(o.residual(f, po), rel=NORM_RTOL)


def _seeded_shapes(count, seed):
    """Extents 4k in [32, 108] (x, y) and [16, 68] (z), so that there are at least two levels, with a
    random boundary set: tile edges, shifted last tiles, patched images and z-chunk seams fall at
    many different offsets."""
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(count):
        n = (int(rng.integers(8, 28)) * 4, int(rng.integers(8, 28)) * 4, int(rng.integers(4, 18)) * 4)
        out.append((n, tuple(int(b) for b in rng.integers(0, 2, size=3))))
    return out


@pytest.mark.parametrize("n,bc", _seeded_shapes(12, 20262))
def test_tma_kernel_on_seeded_ragged_shapes(mgmod, uniform, n, bc):
    """Every instance of the level-0 TMA kernel (one sweep, two sweeps per pass, restriction tail,
    norm tail, prolongation head) on shapes drawn at random: p and the coarse rhs bit-exact."""
    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, 1.0 / n[0], bc, rho=random_rho(uniform, 301, shp), fuse=3, head=1)
    f, p0 = uniform(302, shp), uniform(303, shp)
    po = p0.copy()
    for _ in range(3):
        o.sweep(f, po, 0)
    pg = dev(p0)
    g.level_smooth(0, 3, dev(f), pg)                       # in-place sweep + one two-sweep pass
    assert np.array_equal(po, host(pg))
    pg = dev(p0)
    fc_g = g.level_smooth_restrict(0, 3, dev(f), pg)       # two-sweep pass + one sweep with the tail
    assert np.array_equal(po, host(pg))
    assert np.array_equal(o.restrict(o.residual_level(f, po, 0), 0), host(fc_g))
    pg = dev(p0)
    nrm = g.level_smooth_norm(3, dev(f), pg)
    assert np.array_equal(po, host(pg))
    assert nrm == pytest.approx(o.residual(f, po), rel=NORM_RTOL)
    e = uniform(304, o.level_shape(1))
    po2 = p0.copy()
    o.prolong_add(e, po2, 0)
    for _ in range(2):
        o.sweep(f, po2, 0)
    pg = dev(p0)
    g.level_prolong_smooth(0, 2, dev(e), dev(f), pg)
    assert np.array_equal(po2, host(pg))


@pytest.mark.parametrize("n,bc", TAIL_SHAPES + [((128, 64, 48), (P, N, P))])
@pytest.mark.parametrize("sweeps", [1, 2, 3])
def test_fused_prolongation_head_bit_exact(mgmod, uniform, n, bc, sweeps):
    """SURVEY 8(a) A5 + A6: prolongation, correction and the first post-sweep in one pass of the TMA
    kernel (the p plane is staged as p_old + P e), then the remaining sweeps; p bit-exact.
    (MG_OPT_PROLONG_FUSE = 1; off by default because the separate prolongation pass is faster.)"""
    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, 1.0 / n[0], bc, rho=random_rho(uniform, 54, shp), head=1)
    f, p0 = uniform(55, shp), uniform(56, shp)
    e = uniform(57, o.level_shape(1))
    po = p0.copy()
    o.prolong_add(e, po, 0)
    for _ in range(sweeps):
        o.sweep(f, po, 0)
    pg = dev(p0)
    g.level_prolong_smooth(0, sweeps, dev(e), dev(f), pg)
    assert np.array_equal(po, host(pg))


@pytest.mark.parametrize("fuse", [1, 2, 3])
@pytest.mark.parametrize("sweeps", [2, 4, 5])
def test_two_sweeps_fused_per_pass_bit_exact(mgmod, uniform, sweeps, fuse):
    """MG_OPT_SWEEP_FUSE = 3: temporal blocking, two red-black sweeps per pass of k_rbt<2> at every
    size; = 2 (default): where it pays (not at this size); = 1: one sweep per pass."""
    from paper_2605_30082_b200 import binding as B
    n, bc = (136, 72, 96), (P, N, P)
    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, 1.0 / n[0], bc, rho=random_rho(uniform, 57, shp))
    g.set_option(B.MG_OPT_SWEEP_FUSE, fuse)
    f, p0 = uniform(58, shp), uniform(59, shp)
    po = p0.copy()
    for _ in range(sweeps):
        o.sweep(f, po, 0)
    pg = dev(p0)
    g.level_smooth(0, sweeps, dev(f), pg)
    assert np.array_equal(po, host(pg))


# --------------------------------------------------------------------------- #
# the TMA sweep kernel on the stored-face levels (>= 1): forced onto small levels with
# MG_OPT_FACE_STREAM_LOG2 = 0 (by default only levels of 2^20 cells and more take it).
# Sweeps, fused pairs of sweeps and the restriction tail bit-exact on level 1 and 2;
# periodic wrap (patched images), walls (zero fill, masked updates) and ragged tiles.
# --------------------------------------------------------------------------- #
FACE_SHAPES = [
    ((64, 64, 64), (P, P, P)),
    ((64, 64, 64), (N, N, N)),
    ((136, 72, 96), (N, P, P)),
    ((80, 144, 64), (P, N, N)),
    ((128, 128, 128), (P, P, N)),     # level 1 = 64^3 and level 2 = 32^3 both stream
]


@pytest.mark.parametrize("n,bc", FACE_SHAPES)
@pytest.mark.parametrize("fuse", [1, 3])
def test_face_levels_streamed_bit_exact(mgmod, uniform, n, bc, fuse):
    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, 1.0 / n[0], bc, rho=random_rho(uniform, 61, shp), fuse=fuse, face_log2=0, tails=2)
    for lvl in range(1, o.num_levels - 1):
        lshp = o.level_shape(lvl)                      # (nz, ny, nx)
        if min(lshp[1], lshp[2]) < 32 or lshp[0] < 16:
            break
        f, p0 = uniform(62 + lvl, lshp), uniform(66 + lvl, lshp)
        fd = dev(f)
        for sweeps in (1, 2, 3, 4):
            po = p0.copy()
            for _ in range(sweeps):
                o.sweep(f, po, lvl)
            pg = dev(p0)
            g.level_smooth(lvl, sweeps, fd, pg)
            assert np.array_equal(po, host(pg)), f"level {lvl}, {sweeps} sweeps"
            # the same sweeps with residual + restriction fused behind the last one
            fc_o = o.restrict(o.residual_level(f, po, lvl), lvl)
            pg = dev(p0)
            fc_g = g.level_smooth_restrict(lvl, sweeps, fd, pg)
            assert np.array_equal(po, host(pg)), f"level {lvl}, {sweeps} sweeps + tail: p"
            assert np.array_equal(fc_o, host(fc_g)), f"level {lvl}, {sweeps} sweeps + tail: coarse rhs"


@pytest.mark.parametrize("n,bc", FACE_SHAPES)
@pytest.mark.parametrize("nu", [(2, 2), (3, 3)])
@pytest.mark.parametrize("tails", [1, 2])
def test_vcycle_face_levels_streamed_bit_exact(mgmod, uniform, n, bc, nu, tails):
    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, 1.0 / n[0], bc, nu=nu, rho=random_rho(uniform, 71, shp), coarse_sweeps=8, face_log2=0,
                tails=tails)
    f = uniform(72, shp)
    f -= f.mean()
    po, pg, fd = np.zeros(shp), dev(np.zeros(shp)), dev(f)
    for cyc in range(2):
        o.vcycle(f, po)
        g.vcycle(fd, pg)
        assert np.array_equal(po, host(pg)), f"cycle {cyc}"


# --------------------------------------------------------------------------- #
# V-cycles: every kernel-selection combination gives the oracle's iterate bit for bit
# --------------------------------------------------------------------------- #
OPTS = [dict(kernels=k, graph=gr, coarse_cta=c) for k, gr, c in itertools.product((0, 1), (0, 1), (0, 1))]
OPTS += [dict(kernels=1, graph=1, coarse_cta=1, tails=0), dict(kernels=1, graph=1, coarse_cta=1, head=1),
         dict(kernels=1, graph=0, coarse_cta=1, fuse=1), dict(kernels=1, graph=1, coarse_cta=1, fuse=3)]


@pytest.mark.parametrize("n,bc", SHAPES[:5] + SHAPES[7:])
@pytest.mark.parametrize("opts", OPTS, ids=lambda d: "k%d-g%d-c%d-t%d-f%d-h%d" % (d["kernels"], d["graph"], d["coarse_cta"], d.get("tails", 1), d.get("fuse", 2), d.get("head", 0)))
@pytest.mark.parametrize("nu", [(2, 2), (3, 3), (1, 0)])
def test_vcycle_bit_exact(mgmod, uniform, n, bc, opts, nu):
    h = 1.0 / n[0]
    shp = (n[2], n[1], n[0])
    rho = random_rho(uniform, 7, shp)
    o, g = pair(mgmod, n, h, bc, nu=nu, rho=rho, coarse_sweeps=8, **opts)
    f = uniform(8, shp)
    f -= f.mean()
    po, pg, fd = np.zeros(shp), dev(np.zeros(shp)), dev(f)
    for cyc in range(3):
        o.vcycle(f, po)
        g.vcycle(fd, pg)
        assert np.array_equal(po, host(pg)), f"cycle {cyc}"
    assert g.residual(fd, pg) == pytest.approx(o.residual(f, po), rel=NORM_RTOL)


# --------------------------------------------------------------------------- #
# F- and W-cycles (mg_set_cycle_type, DESIGN R23): the iterate of every
# cycle bit for bit, with the levels <= 16^3 inside the coarse CTA (its own recursion) and
# launch by launch, graph and no graph; then whole solves
# --------------------------------------------------------------------------- #
CYCLE_SHAPES = [((32, 32, 32), (P, P, N)), ((64, 64, 64), (N, P, N)), ((72, 40, 36), (P, N, N)),
                ((128, 128, 128), (P, P, P))]


@pytest.mark.parametrize("n,bc", CYCLE_SHAPES)
@pytest.mark.parametrize("cycle_type", [1, 2], ids=["F", "W"])
@pytest.mark.parametrize("opts", [dict(), dict(coarse_cta=0, graph=0), dict(kernels=0), dict(face_log2=0)],
                         ids=["default", "no-cta-no-graph", "reference-kernels", "faces-streamed"])
def test_f_and_w_cycles_bit_exact(mgmod, uniform, n, bc, cycle_type, opts):
    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, 1.0 / n[0], bc, nu=(2, 1), rho=random_rho(uniform, 91, shp), coarse_sweeps=6,
                cycle_type=cycle_type, **opts)
    f = uniform(92, shp)
    f -= f.mean()
    po, pg, fd = np.zeros(shp), dev(np.zeros(shp)), dev(f)
    for cyc in range(3):
        o.vcycle(f, po)
        g.vcycle(fd, pg)
        assert np.array_equal(po, host(pg)), f"cycle {cyc}"


@pytest.mark.parametrize("cycle_type", [1, 2], ids=["F", "W"])
@pytest.mark.parametrize("cfg,n", [(3, 64), (3, 128), (2, 64)])
def test_solve_with_f_and_w_cycles(mgmod, cfg, n, cycle_type):
    check_solve(mgmod, make_workload(cfg, n), cycle_type=cycle_type)


# --------------------------------------------------------------------------- #
# solves on the BASELINE configs (and scaled twins): norms 1e-10, p 1e-9
# --------------------------------------------------------------------------- #
def check_solve(mgmod, w, max_cycles=40, **opts):
    o, g = pair(mgmod, w.n, w.h, w.bc, nu=(w.nu1, w.nu2), rho=w.rho, **opts)
    po = np.zeros(o.shape)
    so, co, ro, ho = o.solve(w.rhs, po, w.rtol, max_cycles)
    pg = dev(np.zeros(o.shape))
    sg, cg, rg, hg = g.solve(dev(w.rhs), pg, w.rtol, max_cycles)
    assert (sg, cg) == (so, co)
    hg = np.array(hg)
    assert np.abs(hg - ho).max() <= NORM_RTOL * ho[0] and np.all(np.abs(hg / ho - 1) <= NORM_RTOL), (hg, ho)
    assert rg == pytest.approx(ro, rel=NORM_RTOL)
    pgh = host(pg)
    assert np.abs(pgh - po).max() <= P_RTOL * np.abs(po).max()
    assert abs(pgh.mean()) <= 1e-12 * np.abs(pgh).max()
    return o, g, po, pgh, ho


def test_solve_config1(mgmod):
    w = make_workload(1)
    o, g, po, pg, hist = check_solve(mgmod, w)
    assert len(hist) - 1 <= 12 and np.abs(pg - w.p_exact).max() <= 1e-10


@pytest.mark.parametrize("cfg,n", [(2, 64), (2, 128), (3, 64), (3, 128), (5, 128)])
def test_solve_config_twins(mgmod, cfg, n):
    check_solve(mgmod, make_workload(cfg, n))


@pytest.mark.parametrize("opts", [dict(kernels=0, graph=0, coarse_cta=0), dict(kernels=1, graph=1, coarse_cta=0)],
                         ids=["reference-kernels", "fused-no-cta"])
def test_solve_kernel_variants_agree(mgmod, opts):
    check_solve(mgmod, make_workload(3, 64), **opts)


def test_solve_host_buffers(mgmod):
    w = make_workload(3, 64)
    o, g = pair(mgmod, w.n, w.h, w.bc, nu=(w.nu1, w.nu2))
    o.set_density(w.rho)
    po = np.zeros(o.shape)
    so, co, ro, ho = o.solve(w.rhs, po, w.rtol, 40)
    rho_h = torch.from_numpy(w.rho).pin_memory()
    rhs_h = torch.from_numpy(w.rhs).pin_memory()
    p_h = torch.empty(o.shape, dtype=torch.float64).pin_memory()
    sg, cg, rg, hg = g.solve_host(rho_h, rhs_h, p_h, w.rtol, 40)
    assert (sg, cg) == (so, co)
    assert np.all(np.abs(np.array(hg) / ho - 1) <= NORM_RTOL)
    assert np.abs(p_h.numpy() - po).max() <= P_RTOL * np.abs(po).max()


# --------------------------------------------------------------------------- #
# paths of the boundary that the tests above do not reach
# --------------------------------------------------------------------------- #
@pytest.mark.parametrize("n,bc", [((72, 40, 36), (P, N, N)), ((64, 64, 64), (P, P, N))])
def test_residual_field_and_norm(mgmod, uniform, n, bc):
    """mg_residual with r_dev: the field alone (norm2_host NULL) and field + norm in one call
    (DESIGN §3 C6, R15): r bit-exact, the norm within 1e-10."""
    shp = (n[2], n[1], n[0])
    o, g = pair(mgmod, n, 1.0 / n[0], bc, rho=random_rho(uniform, 41, shp))
    f, p = uniform(42, shp), uniform(43, shp)
    nrm_o, r_o = o.residual(f, p, want_field=True)
    fd, pd = dev(f), dev(p)
    r1 = torch.full(shp, np.nan, dtype=torch.float64, device="cuda:0")
    g.residual_field(fd, pd, r1)
    assert np.array_equal(r_o, host(r1))
    r2 = torch.full(shp, np.nan, dtype=torch.float64, device="cuda:0")
    nrm_g = g.residual(fd, pd, r2)
    assert np.array_equal(r_o, host(r2))
    assert nrm_g == pytest.approx(nrm_o, rel=NORM_RTOL)
    assert g.residual(fd, pd) == pytest.approx(nrm_o, rel=NORM_RTOL)


def test_warm_started_solve_after_density_replacement(mgmod):
    """The time-sequence path (bench.py --sequence): solve, replace the
    density, solve again from the previous solution.
    (a) Identical inputs: each GPU solve starts from the ORACLE's previous solution, so both
        sides see the same bits: cycle counts equal, norms 1e-10 relative, p 1e-9.
    (b) The GPU's own chain: its starting iterate differs from the oracle's by the rounding of
        the subtracted mean (C9 leaves the summation order free, ~1e-18 relative).  That
        perturbation is amplified relative to the shrinking residual (SURVEY §8(c) "parity
        hazard"), so the chain is held to SURVEY's stated fallback reading
        |d||r_k||| <= 1e-10 ||r_0||, plus equal cycle counts and p within 1e-9."""
    from workloads import sequence_density
    w = make_workload(3, 64)
    o, g = pair(mgmod, w.n, w.h, w.bc, nu=(w.nu1, w.nu2))
    po, pg, fd = np.zeros(o.shape), dev(np.zeros(o.shape)), dev(w.rhs)
    for step in range(3):
        rho = sequence_density(3, 64, step, 3)
        o.set_density(rho)
        g.set_density(dev(rho))
        pg_same = dev(po)                                     # (a): the oracle's starting iterate
        so, co, ro, ho = o.solve(w.rhs, po, w.rtol, 40)       # po, pg: previous step's solution
        sa, ca, ra, ha = g.solve(fd, pg_same, w.rtol, 40)
        assert (sa, ca) == (so, co), f"step {step}"
        assert np.all(np.abs(np.array(ha) / ho - 1) <= NORM_RTOL), f"step {step}"
        assert np.abs(host(pg_same) - po).max() <= P_RTOL * np.abs(po).max(), f"step {step}"
        sg, cg, rg, hg = g.solve(fd, pg, w.rtol, 40)          # (b): the GPU's own chain
        assert (sg, cg) == (so, co), f"step {step}"
        assert np.abs(np.array(hg) - ho).max() <= NORM_RTOL * ho[0], f"step {step}"
        assert np.abs(host(pg) - po).max() <= P_RTOL * np.abs(po).max(), f"step {step}"
        if step:
            assert co < 10                                     # the warm start pays


def test_library_owned_workspace(mgmod, uniform):
    """mg_create (cudaMalloc workspace owned by the handle) instead of mg_create_in."""
    n, bc = (64, 32, 48), (P, N, P)
    shp = (n[2], n[1], n[0])
    rho = random_rho(uniform, 44, shp)
    o = Oracle(n, 1.0 / 64, bc, 2, 2)
    g = mgmod.Multigrid(n, 1.0 / 64, bc, 2, 2, own_workspace=True)
    o.set_density(rho)
    g.set_density(dev(rho))
    f = uniform(45, shp)
    f -= f.mean()
    po, pg, fd = np.zeros(shp), dev(np.zeros(shp)), dev(f)
    for cyc in range(2):
        o.vcycle(f, po)
        g.vcycle(fd, pg)
        assert np.array_equal(po, host(pg))
    g.close()


def test_full_solve_config3_256(mgmod):
    """BASELINE configs[2] at its full size (256^3 drop-film, V(3,3), 1e-8): the whole solve,
    every norm of the history and the solution, in the launch configuration bench.py times."""
    check_solve(mgmod, make_workload(3))


def test_misaligned_device_pointer_is_rejected(mgmod):
    from paper_2605_30082_b200 import binding as B
    g = mgmod.Multigrid((8, 8, 8), 0.125, (P, P, P))
    buf = torch.zeros(8 * 8 * 8 + 1, dtype=torch.float64, device="cuda:0")
    ok = buf[:512]
    st = B.lib().mg_vcycle(g._h, ok.data_ptr() + 8, ok.data_ptr())
    assert st == B.MG_EINVAL


# --------------------------------------------------------------------------- #
# edge cases and error behaviour of the boundary
# --------------------------------------------------------------------------- #
def test_error_codes_and_degenerate_inputs(mgmod, uniform):
    from paper_2605_30082_b200 import binding as B
    for bad in [((7, 8, 8), 0.1, (P, P, P)), ((8, 8, 2), 0.1, (P, P, P)), ((8, 8, 8), -1.0, (P, P, P)),
                ((8, 8, 8), 0.1, (P, 3, P))]:
        with pytest.raises(B.MgError) as ei:
            mgmod.Multigrid(*bad)
        assert ei.value.code == B.MG_EINVAL
    g = mgmod.Multigrid((8, 8, 8), 0.125, (P, P, P))
    rho = np.ones((8, 8, 8))
    rho[1, 2, 3] = 0.0
    with pytest.raises(B.MgError) as ei:
        g.set_density(dev(rho))
    assert ei.value.code == B.MG_EINVAL
    rho[1, 2, 3] = np.nan
    with pytest.raises(B.MgError):
        g.set_density(dev(rho))
    g.set_density(dev(np.ones((8, 8, 8))))
    f = uniform(3, (8, 8, 8))
    p = dev(np.full((8, 8, 8), 0.25))
    with pytest.raises(B.MgError) as ei:
        g.solve(dev(f + 1.0), p, 1e-8, 5)
    assert ei.value.code == B.MG_EINCOMPATIBLE
    assert np.all(host(p) == 0.25)                       # p untouched
    f -= f.mean()
    st, cyc, rel, hist = g.solve(dev(f), p, 1e-14, 2)
    assert st == B.MG_NOT_CONVERGED and cyc == 2 and len(hist) == 3
    # max_cycles = 0: only the initial residual and the mean removal
    p = dev(uniform(4, (8, 8, 8)))
    st, cyc, rel, hist = g.solve(dev(f), p, 1e-8, 0)
    assert st == B.MG_NOT_CONVERGED and cyc == 0 and len(hist) == 1 and abs(host(p).mean()) < 1e-16
    # zero right-hand side, zero guess: converged immediately with p = 0
    z = dev(np.zeros((8, 8, 8)))
    st, cyc, rel, hist = g.solve(z, dev(np.zeros((8, 8, 8))), 1e-8, 5)
    assert st == B.MG_OK and cyc == 0 and hist == [0.0]
    assert g.stat(B.MG_STAT_KERNEL_LAUNCHES) > 0 and g.stat(B.MG_STAT_WORKSPACE_BYTES) > 0


def test_default_density_is_one(mgmod, uniform):
    n = (16, 16, 16)
    o, g = pair(mgmod, n, 1 / 16, (P, P, N))           # no set_density on either side
    f = uniform(2, (16, 16, 16))
    f -= f.mean()
    po, pg = np.zeros((16, 16, 16)), dev(np.zeros((16, 16, 16)))
    o.vcycle(f, po)
    g.vcycle(dev(f), pg)
    assert np.array_equal(po, host(pg))


def test_density_can_be_replaced(mgmod, uniform):
    w = make_workload(3, 32)
    o, g = pair(mgmod, w.n, w.h, w.bc, nu=(3, 3), rho=random_rho(uniform, 1, (32, 32, 32)))
    pg, po = dev(np.zeros(o.shape)), np.zeros(o.shape)
    g.vcycle(dev(w.rhs), pg)                              # graph captured with the first density
    o.vcycle(w.rhs, po)
    o.set_density(w.rho)
    g.set_density(dev(w.rho))
    g.vcycle(dev(w.rhs), pg)
    o.vcycle(w.rhs, po)
    assert np.array_equal(po, host(pg))


# --------------------------------------------------------------------------- #
# full sizes, in the launch configuration bench.py times (graph replay, streaming kernels)
# --------------------------------------------------------------------------- #
def _full_size_cycles(mgmod, cfg, cycles):
    w = make_workload(cfg)
    o, g = pair(mgmod, w.n, w.h, w.bc, nu=(w.nu1, w.nu2), rho=w.rho)
    shp = o.shape
    po = np.zeros(shp)
    pg, fd = dev(po), dev(w.rhs)
    for cyc in range(cycles):
        o.vcycle(w.rhs, po)
        g.vcycle(fd, pg)
        assert np.array_equal(po, host(pg)), f"config {cfg} cycle {cyc}"
    assert g.residual(fd, pg) == pytest.approx(o.residual(w.rhs, po), rel=NORM_RTOL)
    o.close()
    g.close()


def test_full_size_config4_bit_exact(mgmod):
    """512^3 drop-film (BASELINE configs[3], the bench workload): every cell of two V(3,3)
    cycles equals the oracle's, and the residual norm agrees to 1e-10."""
    _full_size_cycles(mgmod, 4, 2)


@pytest.mark.parametrize("cycle_type", [0, 1], ids=["V", "F"])
def test_full_size_config4_whole_solve(mgmod, cycle_type):
    """The timed workload itself (512^3 drop-film, V(3,3), rtol 1e-8), solved to the end with V-cycles
    (17) and with F-cycles (11) in bench.py's launch configuration (default options: graph replay,
    two-sweep passes, fused tails): cycle count, every norm of the history to 1e-10, p to 1e-9."""
    w = make_workload(4)
    o, g, po, pg, hist = check_solve(mgmod, w, max_cycles=40, cycle_type=cycle_type)
    assert len(hist) - 1 == (17 if cycle_type == 0 else 11)
    o.close()
    g.close()


def test_full_size_config5_bit_exact(mgmod):
    """1024^3 (BASELINE configs[4], the largest size): one V(3,3) cycle, every cell.  Needs
    ~60 GB of host memory for the oracle and ~52 GB on the device; skipped on smaller boxes."""
    import os
    host_gb = os.sysconf("SC_PAGE_SIZE") * os.sysconf("SC_PHYS_PAGES") / 2**30
    dev_gb = torch.cuda.get_device_properties(0).total_memory / 2**30
    if host_gb < 100 or dev_gb < 100:
        pytest.skip(f"needs >= 100 GB host and device memory (have {host_gb:.0f} / {dev_gb:.0f})")
    _full_size_cycles(mgmod, 5, 1)


def test_streaming_sweep_is_reproducible_under_repetition(mgmod, uniform):
    """The streaming sweep synchronises its rows with one barrier every second step and reuses
    its exchange and staging slots cyclically; a missing ordering would show up as run-to-run
    differences.  40 repetitions of two sweeps on the same input (several x / y tiles and
    z-chunks, a Neumann wall) must all give the oracle's bits."""
    n, bc = (136, 72, 96), (P, N, P)
    h = 1.0 / n[0]
    shp = (n[2], n[1], n[0])
    rho = random_rho(uniform, 9, shp)
    o, g = pair(mgmod, n, h, bc, rho=rho)
    f, p0 = uniform(10, shp), uniform(11, shp)
    po = p0.copy()
    o.sweep(f, po, 0); o.sweep(f, po, 0)
    fd = dev(f)
    for rep in range(40):
        pg = dev(p0)
        g.level_smooth(0, 2, fd, pg)
        assert np.array_equal(po, host(pg)), f"repetition {rep}"
