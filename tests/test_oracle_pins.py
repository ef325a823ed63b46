"""Pins of the CPU oracle against what the mathematics fixes (no GPU, no self-reference).

Each test names the oracle function it pins and the plausible mistake it catches.
Sources: BASELINE.json north_star ("discrete sine eigenmodes ... closed-form lambda;
operator symmetry; zero-mean compatibility; second-order convergence on a manufactured
solution; dense direct solve on an 8^3 grid") and SURVEY.md §4.
"""
import itertools
import math

import numpy as np
import pytest

from oracle import mgo
from oracle.mgo import Oracle
from workloads import make_workload

P, N = 0, 1
ALL_BC = list(itertools.product((P, N), repeat=3))


def centres(n, h):
    return (np.arange(n) + 0.5) * h


def mode_1d(kind, k, n, h):
    """Eigenvector of the 1-D constant-coefficient operator and its eigenvalue."""
    x = centres(n, h)
    L = n * h
    if kind == "psin":
        return np.sin(2 * math.pi * k * x / L), -(4.0 / h ** 2) * math.sin(math.pi * k / n) ** 2
    if kind == "pcos":
        return np.cos(2 * math.pi * k * x / L), -(4.0 / h ** 2) * math.sin(math.pi * k / n) ** 2
    if kind == "ncos":
        return np.cos(math.pi * k * x / L), -(4.0 / h ** 2) * math.sin(math.pi * k / (2 * n)) ** 2
    raise KeyError(kind)


# --------------------------------------------------------------------------- #
# 1. eigenmodes: pins apply / residual_level (stencil weights, 1/h^2, sign, 1/rho,
#    periodic wrap vs Neumann wall, axis order nx != ny != nz)
# --------------------------------------------------------------------------- #
@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("rho0", [1.0, 935.0])
def test_constant_density_eigenmodes(bc, rho0):
    n = (16, 12, 8)            # nx, ny, nz all different: catches transposed axes
    h = 1.0 / 16
    o = Oracle(n, h, bc)
    o.set_density(np.full(o.shape, rho0))
    ks = (3, 2, 1)
    vecs, lam = [], 0.0
    for ax in range(3):
        kind = "ncos" if bc[ax] == N else ("psin" if ax != 1 else "pcos")
        v, l1 = mode_1d(kind, ks[ax], n[ax], h)
        vecs.append(v)
        lam += l1
    lam /= rho0
    v = vecs[2][:, None, None] * vecs[1][None, :, None] * vecs[0][None, None, :]
    Av = o.apply(v)
    scale = abs(lam) * np.abs(v).max()
    assert np.abs(Av - lam * v).max() <= 1e-12 * scale
    # r = f - A p vanishes for f = lambda v  (pins residual_level's sign convention)
    r = o.residual_level(lam * v, v)
    assert np.abs(r).max() <= 1e-12 * scale
    # and does not vanish for the wrong sign
    assert np.abs(o.residual_level(-lam * v, v)).max() > 0.5 * scale


def test_config1_eigenvalue_value():
    w = make_workload(1)
    o = Oracle(w.n, w.h, w.bc)
    Ap = o.apply(w.p_exact)
    assert w.eigenvalue == pytest.approx(-(12 / w.h ** 2) * math.sin(math.pi / 32) ** 2, rel=1e-15)
    assert np.abs(Ap - w.eigenvalue * w.p_exact).max() < 1e-11


# --------------------------------------------------------------------------- #
# 2. algebraic structure with random positive density: pins set_density's faces
#    (shared by both cells, wall faces zero) and apply
# --------------------------------------------------------------------------- #
@pytest.mark.parametrize("bc", ALL_BC)
def test_symmetry_rowsums_colsums_definiteness(bc, uniform):
    n = (8, 12, 16)
    o = Oracle(n, 0.125, bc)
    rho = np.exp(uniform(11, o.shape, math.log(1.2), math.log(998.0)))
    o.set_density(rho)
    x, y = uniform(12, o.shape), uniform(13, o.shape)
    Ax, Ay = o.apply(x), o.apply(y)
    big = np.abs(Ax).max() * x.size
    assert abs(np.vdot(x, Ay) - np.vdot(y, Ax)) <= 1e-13 * big          # symmetry
    assert np.abs(o.apply(np.ones(o.shape))).max() == 0.0               # A 1 = 0
    assert abs(float(np.sum(Ax, dtype=np.longdouble))) <= 1e-12 * big   # 1^T A = 0
    assert np.vdot(x, Ax) < 0.0                                         # negative semi-definite
    # every level's operator has the same structure (coarse faces shared, walls zero)
    for lvl in range(1, o.num_levels):
        shp = o.level_shape(lvl)
        xl, yl = uniform(20 + lvl, shp), uniform(30 + lvl, shp)
        Axl, Ayl = o.apply(xl, lvl), o.apply(yl, lvl)
        bigl = np.abs(Axl).max() * xl.size
        assert abs(np.vdot(xl, Ayl) - np.vdot(yl, Axl)) <= 1e-13 * bigl
        assert np.abs(o.apply(np.ones(shp), lvl)).max() <= 1e-12 * np.abs(Axl).max()
        assert np.vdot(xl, Axl) < 0.0


def test_faces_are_harmonic_mean_reciprocals_and_walls_zero():
    # two-cell check of R4 independent of the oracle's own expression:
    # beta = 1 / (2 ra rb / (ra + rb))
    o = Oracle((4, 4, 4), 0.25, (P, P, N))
    rho = np.ones(o.shape)
    rho[:, :, 0], rho[:, :, 1], rho[:, :, 2], rho[:, :, 3] = 2.0, 8.0, 1.0, 4.0
    o.set_density(rho)
    bx, by, bz = o.faces(0)
    harm = lambda a, b: 1.0 / (2 * a * b / (a + b))
    assert np.allclose(bx[:, :, 1], harm(2.0, 8.0), rtol=1e-15)
    assert np.allclose(bx[:, :, 0], harm(4.0, 2.0), rtol=1e-15)      # periodic wrap face
    assert np.allclose(by[:, :, 1], 1.0 / 8.0, rtol=1e-15)
    assert np.all(bz[0] == 0.0) and np.all(bz[1:] > 0.0)             # Neumann wall
    # the other reading, 2/(ra+rb), differs: make sure we are not computing it
    assert not np.allclose(bx[:, :, 1], 2.0 / (2.0 + 8.0))


# --------------------------------------------------------------------------- #
# 3. layered medium: exact discrete solution by prefix sums.  Pins the face rule at a
#    density jump (R4 vs the 2/(ra+rb) reading) and the whole solve.
# --------------------------------------------------------------------------- #
def test_layered_medium_prefix_sum_solution(uniform):
    n, h = 16, 1.0 / 16
    o = Oracle((n, n, n), h, (P, P, N), 2, 2)
    rho_z = np.where(np.arange(n) < 5, 935.0, 1.2)
    rho_z[5] = 0.3 * 935.0 + 0.7 * 1.2
    fz = uniform(5, (n,))
    fz -= fz.mean()
    rho = np.broadcast_to(rho_z[:, None, None], o.shape).copy()
    f = np.broadcast_to(fz[:, None, None], o.shape).copy()
    o.set_density(rho)
    p = np.zeros(o.shape)
    st, cyc, rel, hist = o.solve(f, p, 1e-13, 60)
    assert st == mgo.OK
    # closed form: flux through face k+1/2 is h * sum_{m<=k} f_m
    beta = 0.5 * (1.0 / rho_z[:-1] + 1.0 / rho_z[1:])
    pz = np.zeros(n)
    pz[1:] = np.cumsum(h * h * np.cumsum(fz)[:-1] / beta)
    pz -= pz.mean()
    assert np.abs(p - pz[:, None, None]).max() <= 1e-9 * np.abs(pz).max()
    # the rejected reading beta = 2/(ra+rb) gives a measurably different answer
    beta2 = 2.0 / (rho_z[:-1] + rho_z[1:])
    pz2 = np.zeros(n)
    pz2[1:] = np.cumsum(h * h * np.cumsum(fz)[:-1] / beta2)
    pz2 -= pz2.mean()
    assert np.abs(pz2 - pz).max() > 1e-3 * np.abs(pz).max()


# --------------------------------------------------------------------------- #
# 4. manufactured smooth solution with smooth variable density: second order.
#    Pins operator + solve as a discretisation of div((1/rho) grad p).
# --------------------------------------------------------------------------- #
def _manufactured(n, bc_z):
    h = 1.0 / n
    x = centres(n, h)
    X, Y, Z = x[None, None, :], x[None, :, None], x[:, None, None]
    tp = 2 * math.pi
    # c = 1/rho smooth, periodic in x,y; z-dependence compatible with both bcs
    c = 1.0 + 0.5 * np.sin(tp * X) * np.cos(tp * Y) + 0.25 * np.cos(tp * Z)
    cx = 0.5 * tp * np.cos(tp * X) * np.cos(tp * Y) + 0 * Z
    cy = -0.5 * tp * np.sin(tp * X) * np.sin(tp * Y) + 0 * Z
    cz = -0.25 * tp * np.sin(tp * Z) + 0 * X + 0 * Y
    if bc_z == N:   # dp/dz = 0 at z = 0, 1
        g, gz, gzz = np.cos(math.pi * Z), -math.pi * np.sin(math.pi * Z), -math.pi ** 2 * np.cos(math.pi * Z)
    else:
        g, gz, gzz = np.sin(tp * Z), tp * np.cos(tp * Z), -tp ** 2 * np.sin(tp * Z)
    a, ax_, axx = np.sin(tp * X), tp * np.cos(tp * X), -tp ** 2 * np.sin(tp * X)
    b, by_, byy = np.cos(2 * tp * Y), -2 * tp * np.sin(2 * tp * Y), -(2 * tp) ** 2 * np.cos(2 * tp * Y)
    p = a * b * g
    f = c * (axx * b * g + a * byy * g + a * b * gzz) + cx * ax_ * b * g + cy * a * by_ * g + cz * a * b * gz
    return h, 1.0 / c, p - p.mean(), f - f.mean()


@pytest.mark.parametrize("bc_z", [P, N])
def test_manufactured_solution_second_order(bc_z):
    errs = []
    for n in (16, 32, 64):
        h, rho, p_true, f = _manufactured(n, bc_z)
        o = Oracle((n, n, n), h, (P, P, bc_z), 2, 2)
        o.set_density(rho)
        p = np.zeros(o.shape)
        st, *_ = o.solve(f, p, 1e-11, 60)
        assert st == mgo.OK
        errs.append(np.abs(p - p_true).max())
    r1, r2 = errs[0] / errs[1], errs[1] / errs[2]
    assert 3.3 < r1 < 4.8 and 3.6 < r2 < 4.4, (errs, r1, r2)


# --------------------------------------------------------------------------- #
# 5. dense direct solve at 8^3: pins solve incl. null-space handling, all bcs
# --------------------------------------------------------------------------- #
@pytest.mark.parametrize("bc", [(P, P, P), (P, P, N), (N, N, N)])
def test_dense_direct_solve_8cubed(bc, uniform):
    n = 8
    o = Oracle((n, n, n), 1.0 / n, bc, 2, 2)
    rho = np.exp(uniform(41, o.shape, math.log(1.2), math.log(998.0)))
    o.set_density(rho)
    N3 = n ** 3
    A = np.empty((N3, N3))
    e = np.zeros(N3)
    for c in range(N3):
        e[c] = 1.0
        A[:, c] = o.apply(e.reshape(o.shape)).reshape(-1)
        e[c] = 0.0
    assert np.abs(A - A.T).max() <= 1e-12 * np.abs(A).max()
    ev = np.linalg.eigvalsh(0.5 * (A + A.T))
    assert ev[-1] == pytest.approx(0.0, abs=1e-9 * abs(ev[0]))     # exactly one zero eigenvalue
    assert ev[-2] < -1e-6 * abs(ev[0])
    f = uniform(42, o.shape)
    f -= f.mean()
    # mean-constrained dense solve: [A 1; 1^T 0][p; mu] = [f; 0]
    K = np.zeros((N3 + 1, N3 + 1))
    K[:N3, :N3] = A
    K[:N3, N3] = 1.0
    K[N3, :N3] = 1.0
    sol = np.linalg.solve(K, np.concatenate([f.reshape(-1), [0.0]]))
    p_dense = sol[:N3].reshape(o.shape)
    p = np.zeros(o.shape)
    st, cyc, rel, hist = o.solve(f, p, 1e-13, 200)
    assert st == mgo.OK
    assert abs(p.mean()) <= 1e-15 * np.abs(p).max() * N3
    assert np.abs(p - p_dense).max() <= 1e-9 * np.abs(p_dense).max()


# --------------------------------------------------------------------------- #
# 6. smoother invariants: pins smooth_half (update formula, colouring, order)
# --------------------------------------------------------------------------- #
@pytest.mark.parametrize("bc", [(P, P, P), (P, N, N)])
def test_half_sweep_zeroes_residual_on_its_colour(bc, uniform):
    n = (8, 8, 12)
    o = Oracle(n, 0.125, bc)
    o.set_density(np.exp(uniform(51, o.shape, 0.0, 6.0)))
    f, p = uniform(52, o.shape), uniform(53, o.shape)
    k, j, i = np.indices(o.shape)
    red = ((i + j + k) & 1) == 0
    p_before = p.copy()
    o.smooth_half(0, f, p)
    assert np.array_equal(p[~red], p_before[~red])           # black untouched
    assert not np.array_equal(p[red], p_before[red])
    r = o.residual_level(f, p)
    scale = np.abs(f).max() + np.abs(o.apply(p)).max()
    assert np.abs(r[red]).max() <= 1e-13 * scale
    assert np.abs(r[~red]).max() > 1e-3 * scale
    o.smooth_half(1, f, p)
    r = o.residual_level(f, p)
    assert np.abs(r[~red]).max() <= 1e-13 * scale            # black now exact ...
    assert np.abs(r[red]).max() > 1e-3 * scale               # ... red no longer: order is red, black


def test_exact_solution_is_fixed_point_of_sweep_and_vcycle(uniform):
    n = 16
    o = Oracle((n, n, n), 1.0 / n, (P, P, N), 2, 2)
    o.set_density(np.exp(uniform(61, o.shape, 0.0, 5.0)))
    p_true = uniform(62, o.shape)
    f = o.apply(p_true)
    p = p_true.copy()
    o.sweep(f, p)
    assert np.abs(p - p_true).max() <= 1e-12 * np.abs(p_true).max()
    o.vcycle(f, p)
    assert np.abs(p - p_true).max() <= 1e-11 * np.abs(p_true).max()


# --------------------------------------------------------------------------- #
# 7. transfer invariants: pins restrict (weights 1/8) and prolong_add (3/4, 1/4, ghosts)
# --------------------------------------------------------------------------- #
def test_restriction_invariants(uniform):
    o = Oracle((8, 12, 16), 0.125, (P, P, N))
    r = uniform(71, o.shape)
    fc = o.restrict(r)
    assert fc.shape == (8, 6, 4)
    assert np.allclose(o.restrict(np.full(o.shape, 3.25)), 3.25, rtol=0, atol=0)
    assert 8 * fc.sum() == pytest.approx(r.sum(), abs=1e-12 * np.abs(r).sum())
    # brute force on the definition: mean over the 2x2x2 block
    want = r.reshape(8, 2, 6, 2, 4, 2).mean(axis=(1, 3, 5))
    assert np.abs(fc - want).max() <= 1e-15
    # a single non-zero child lands in exactly one parent with weight 1/8
    d = np.zeros(o.shape)
    d[5, 6, 3] = 8.0                      # (k,j,i) -> parent (2,3,1)
    fd = o.restrict(d)
    assert fd[2, 3, 1] == 1.0 and np.count_nonzero(fd) == 1


@pytest.mark.parametrize("bc", [(P, P, P), (N, N, N), (P, N, P)])
def test_prolongation_invariants(bc, uniform):
    n = (8, 12, 16)
    o = Oracle(n, 0.125, bc)
    cshape = o.level_shape(1)
    # constants are reproduced
    p = np.zeros(o.shape)
    o.prolong_add(np.full(cshape, 2.5), p)
    assert np.all(p == 2.5)
    # adds to p rather than overwriting
    p = np.full(o.shape, 1.0)
    o.prolong_add(np.full(cshape, 2.0), p)
    assert np.all(p == 3.0)
    # mass: sum(P e) = 8 sum(e) for periodic and for clamped (Neumann) ghosts alike
    e = uniform(72, cshape)
    p = np.zeros(o.shape)
    o.prolong_add(e, p)
    assert p.sum() == pytest.approx(8 * e.sum(), abs=1e-12 * np.abs(e).sum())
    # linear functions are reproduced exactly at fine cells whose 2x2x2 coarse
    # neighbourhood does not touch a boundary
    (cx, cy, cz), hc = o.level_dims(1)
    K, J, I = np.indices(cshape)
    lin = 0.3 * (I + 0.5) * hc - 0.7 * (J + 0.5) * hc + 1.1 * (K + 0.5) * hc
    p = np.zeros(o.shape)
    o.prolong_add(lin, p)
    k, j, i = np.indices(o.shape)
    hf = 0.125
    want = 0.3 * (i + 0.5) * hf - 0.7 * (j + 0.5) * hf + 1.1 * (k + 0.5) * hf
    inner = (slice(1, -1),) * 3
    assert np.abs(p[inner] - want[inner]).max() <= 1e-14


def test_prolongation_weights_of_a_delta():
    o = Oracle((8, 8, 8), 0.125, (P, P, P))
    e = np.zeros((4, 4, 4))
    e[2, 1, 1] = 64.0                     # coarse (K,J,I) = (2,1,1)
    p = np.zeros(o.shape)
    o.prolong_add(e, p)
    # per axis a coarse cell I contributes 1/4,3/4,3/4,1/4 to fine cells 2I-1..2I+2
    w = np.array([0.25, 0.75, 0.75, 0.25])
    want = np.zeros(o.shape)
    want[3:7, 1:5, 1:5] = 64.0 * w[:, None, None] * w[None, :, None] * w[None, None, :]
    assert np.array_equal(p, want)
    assert sorted(set(np.unique(p))) == [0.0, 1.0, 3.0, 9.0, 27.0]


def test_prolongation_neumann_wall_clamps():
    o = Oracle((8, 8, 8), 0.125, (P, P, N))
    e = np.zeros((4, 4, 4))
    e[0] = 1.0                            # bottom coarse layer
    p = np.zeros(o.shape)
    o.prolong_add(e, p)
    assert np.all(p[0] == 1.0)            # 3/4 e0 + 1/4 e0 (clamped ghost), not wrapped
    assert np.all(p[1] == 0.75) and np.all(p[2] == 0.25) and np.all(p[3:] == 0.0)
    op = Oracle((8, 8, 8), 0.125, (P, P, P))
    q = np.zeros(op.shape)
    op.prolong_add(e, q)
    assert np.all(q[0] == 0.75) and np.all(q[7] == 0.25)     # periodic: wraps instead


# --------------------------------------------------------------------------- #
# 8. coefficient hierarchy (R8 is a convention: only its invariants can be pinned)
# --------------------------------------------------------------------------- #
def test_coarse_faces_invariants(uniform):
    o = Oracle((16, 16, 16), 1.0 / 16, (P, N, N))
    o.set_density(np.full(o.shape, 4.0))
    for lvl in range(o.num_levels):
        bx, by, bz = o.faces(lvl)
        assert np.all(bx == 0.25)
        assert np.all(by[:, 0, :] == 0.0) and np.all(by[:, 1:, :] == 0.25)
        assert np.all(bz[0] == 0.0) and np.all(bz[1:] == 0.25)
    # layered in z: a coarse x-face is the mean over its two z-layers
    rho_z = np.exp(uniform(81, (16,), 0.0, 5.0))
    o.set_density(np.broadcast_to(rho_z[:, None, None], o.shape).copy())
    bx0, _, bz0 = o.faces(0)
    bx1, _, bz1 = o.faces(1)
    assert np.allclose(bx1[:, 0, 0], 0.5 * (bx0[0::2, 0, 0] + bx0[1::2, 0, 0]), rtol=1e-15)
    assert np.allclose(bz1[:, 3, 3], bz0[0::2, 3, 3], rtol=1e-15)   # even child's minus face


@pytest.mark.parametrize("bc", [(P, P, P), (P, N, N), (N, N, N)])
def test_coarse_faces_brute_force_3d(bc, uniform):
    """Pins mgo_set_density's coarse levels: with a fully 3-D
    random density every face of level l >= 1 must be the mean of the FOUR level l-1 faces of the
    same direction that lie on it, i.e. the minus faces of the even child across the face and
    of its three neighbours in the two tangential directions, written out as numpy slices of
    faces(l-1) in (k, j, i) order.  Catches: taking the odd child's face, averaging over the
    wrong pair of directions, dropping one of the four faces (each changes the value when
    the density varies in all three directions)."""
    n = (32, 16, 16)                      # nx != ny: catches a swapped axis as well
    o = Oracle(n, 1.0 / 16, bc)
    o.set_density(np.exp(uniform(83, o.shape, 0.0, 6.0)))
    assert o.num_levels >= 3
    for lvl in range(1, o.num_levels):
        fx, fy, fz = o.faces(lvl - 1)
        bx, by, bz = o.faces(lvl)
        # x-face of coarse cell (I,J,K): fine x-minus faces at i = 2I, j in {2J,2J+1}, k in {2K,2K+1}
        ex = 0.25 * ((fx[0::2, 0::2, 0::2] + fx[0::2, 1::2, 0::2]) + (fx[1::2, 0::2, 0::2] + fx[1::2, 1::2, 0::2]))
        # y-face: fine y-minus faces at j = 2J, i in {2I,2I+1}, k in {2K,2K+1}
        ey = 0.25 * ((fy[0::2, 0::2, 0::2] + fy[0::2, 0::2, 1::2]) + (fy[1::2, 0::2, 0::2] + fy[1::2, 0::2, 1::2]))
        # z-face: fine z-minus faces at k = 2K, i in {2I,2I+1}, j in {2J,2J+1}
        ez = 0.25 * ((fz[0::2, 0::2, 0::2] + fz[0::2, 0::2, 1::2]) + (fz[0::2, 1::2, 0::2] + fz[0::2, 1::2, 1::2]))
        for got, exp in ((bx, ex), (by, ey), (bz, ez)):
            assert got.shape == exp.shape
            assert np.all(np.abs(got - exp) <= np.spacing(np.abs(exp)))     # 1 ulp
        # the random field really separates the candidates (odd child / wrong pair / 3 of 4)
        odd = 0.25 * ((fx[0::2, 0::2, 1::2] + fx[0::2, 1::2, 1::2]) + (fx[1::2, 0::2, 1::2] + fx[1::2, 1::2, 1::2]))
        assert np.abs(odd - ex).max() > 1e-3 * np.abs(ex).max()
        # Neumann axes keep their wall face exactly zero on every level
        if bc[0] == N: assert np.all(bx[:, :, 0] == 0.0)
        if bc[1] == N: assert np.all(by[:, 0, :] == 0.0)
        if bc[2] == N: assert np.all(bz[0] == 0.0)


def test_coarsest_level_runs_exactly_coarse_sweeps_sweeps(uniform):
    """Pins R13's count in vcycle(): on a one-level hierarchy (6^3 cannot be halved, R7) a cycle
    is nothing but `coarse_sweeps` red-black sweeps from the incoming p, each of which is the
    pinned smooth_half(0) then smooth_half(1).  Catches a wrong count (e.g. coarse_sweeps/8) and
    a coarsest solve that restarts from zero."""
    o = Oracle((6, 6, 6), 1.0 / 6, (P, N, P), 2, 2, 5)
    assert o.num_levels == 1
    o.set_density(np.exp(uniform(85, o.shape, 0.0, 3.0)))
    f = uniform(86, o.shape)
    f -= f.mean()
    p0 = uniform(87, o.shape)
    p = p0.copy()
    o.vcycle(f, p)
    q = p0.copy()
    for it in range(5):
        o.smooth_half(0, f, q)
        o.smooth_half(1, f, q)
        if it == 3:
            assert not np.array_equal(p, q)          # four sweeps are not enough
    assert np.array_equal(p, q)


# --------------------------------------------------------------------------- #
# 9. end to end on config 1 (known solution), API behaviour, thread independence
# --------------------------------------------------------------------------- #
def test_config1_converges_to_known_solution():
    w = make_workload(1)
    o = Oracle(w.n, w.h, w.bc, w.nu1, w.nu2)
    assert o.num_levels == 4 and o.level_dims(3)[0] == (4, 4, 4)      # "down to 4^3"
    o.set_density(w.rho)
    p = np.zeros(o.shape)
    st, cyc, rel, hist = o.solve(w.rhs, p, w.rtol, 30)
    assert st == mgo.OK and cyc <= 12 and rel <= 1e-10
    assert np.all(np.diff(hist) < 0)
    assert np.abs(p - w.p_exact).max() <= 1e-10
    # hist[k] really is ||f - A p_k||: recompute the last one independently via apply
    assert hist[-1] == pytest.approx(np.linalg.norm((w.rhs - o.apply(p)).ravel()), rel=1e-12)


def test_solve_measures_r0_from_the_incoming_p(uniform):
    """Pins R15 in mgo_solve: r_0 = ||f - A p_0|| of the INCOMING p (not ||f||), hist[0] is that
    number, the stop is the first k with hist[k] <= rtol * hist[0], and the statuses of the two
    degenerate calls.  Built from the pinned apply() and numpy's norm only.  p_0 is chosen so that
    ||f - A p_0|| is about 1000 ||f||: with r_0 read as ||f|| the same rtol would need several
    more cycles, with hist[0] = 2 r_0 one fewer could pass, so each misreading moves `cyc`."""
    o = Oracle((16, 16, 16), 1.0 / 16, (P, N, P), 2, 2)
    o.set_density(np.exp(uniform(301, o.shape, np.log(1.2), np.log(998.0))))
    f = uniform(302, o.shape)
    f -= f.mean()
    p0 = 1000.0 * uniform(303, o.shape) * np.linalg.norm(f.ravel()) / np.linalg.norm(o.apply(uniform(303, o.shape)).ravel())
    r0 = np.linalg.norm((f - o.apply(p0)).ravel())
    assert r0 > 500.0 * np.linalg.norm(f.ravel())
    rtol = 1e-4
    p = p0.copy()
    st, cyc, rel, hist = o.solve(f, p, rtol, 40)
    assert st == mgo.OK and len(hist) == cyc + 1
    assert hist[0] == pytest.approx(r0, rel=1e-13)
    # every entry is the residual of the iterate it belongs to: replay the cycles by hand
    q = p0.copy()
    for k in range(1, cyc + 1):
        o.vcycle(f, q)
        assert hist[k] == pytest.approx(np.linalg.norm((f - o.apply(q)).ravel()), rel=1e-12)
    # stop at the FIRST k below rtol * r0, measured against r0 of the incoming p
    below = [k for k in range(cyc + 1) if hist[k] <= rtol * r0]
    assert below == [cyc]
    assert hist[cyc] > rtol * np.linalg.norm(f.ravel())          # ||f|| as r_0 would have gone on
    assert hist[cyc - 1] > rtol * 2.0 * r0                        # 2 r_0 would still stop here or earlier ...
    assert rel == pytest.approx(hist[cyc] / r0, rel=1e-13)        # ... but relres pins the denominator
    assert np.array_equal(p, q - q.mean()) or np.abs(p - (q - q.mean())).max() <= 1e-13 * np.abs(q).max()
    # max_cycles = 0: not converged, no cycle run, only the mean removed
    p = p0.copy()
    st, cyc0, rel0, hist0 = o.solve(f, p, rtol, 0)
    assert st == mgo.NOT_CONVERGED and cyc0 == 0 and len(hist0) == 1
    assert hist0[0] == pytest.approx(r0, rel=1e-13) and rel0 == 1.0
    assert np.abs(p - (p0 - p0.mean())).max() <= 1e-13 * np.abs(p0).max()
    # rhs = 0 from p = 0: r_0 = 0 counts as converged at once
    z = np.zeros(o.shape)
    st, cycz, relz, histz = o.solve(z, z.copy(), rtol, 5)
    assert st == mgo.OK and cycz == 0 and list(histz) == [0.0] and relz == 0.0


def test_level_counts_of_the_configs():
    for n, levels in [(32, 4), (128, 6), (256, 7)]:
        o = Oracle((n, n, n), 1.0 / n, (P, P, N))
        assert o.num_levels == levels
    assert Oracle((48, 48, 48), 1 / 48, (P, P, P)).level_dims(3)[0] == (6, 6, 6)


def test_error_codes(uniform):
    with pytest.raises(mgo.OracleError):
        Oracle((7, 8, 8), 0.1, (P, P, P))
    with pytest.raises(mgo.OracleError):
        Oracle((8, 8, 8), -1.0, (P, P, P))
    with pytest.raises(mgo.OracleError):
        Oracle((8, 8, 8), 0.1, (P, 2, P))
    o = Oracle((8, 8, 8), 0.125, (P, P, P))
    bad = np.ones(o.shape)
    bad[1, 2, 3] = -1.0
    with pytest.raises(mgo.OracleError):
        o.set_density(bad)
    f = uniform(91, o.shape)
    with pytest.raises(mgo.OracleError) as ei:
        o.solve(f + 1.0, np.zeros(o.shape), 1e-8, 5)
    assert ei.value.code == mgo.EINCOMPATIBLE
    f -= f.mean()
    st, cyc, rel, hist = o.solve(f, np.zeros(o.shape), 1e-14, 2)
    assert st == mgo.NOT_CONVERGED and cyc == 2 and len(hist) == 3


def test_fields_do_not_depend_on_thread_count():
    w = make_workload(3, 32)
    out = []
    for t in (1, 4):
        mgo.set_threads(t)
        o = Oracle(w.n, w.h, w.bc, w.nu1, w.nu2)
        o.set_density(w.rho)
        p = np.zeros(o.shape)
        st, cyc, rel, hist = o.solve(w.rhs, p, w.rtol, 30)
        out.append((p.copy(), hist))
    mgo.set_threads(0)
    assert np.array_equal(out[0][0], out[1][0])
    assert np.array_equal(out[0][1], out[1][1])


def test_drop_film_twin_converges_like_the_probe():
    # SURVEY 8(c) probe (ballpark, not golden): drop-film 64^3 V(3,3): ~10 cycles to 1e-8,
    # first-cycle residual may rise.  Guards against silent changes of R4/R8.
    w = make_workload(3, 64)
    o = Oracle(w.n, w.h, w.bc, w.nu1, w.nu2)
    o.set_density(w.rho)
    p = np.zeros(o.shape)
    st, cyc, rel, hist = o.solve(w.rhs, p, w.rtol, 30)
    assert st == mgo.OK and 8 <= cyc <= 14
    r = o.residual(w.rhs, p)
    assert r == pytest.approx(hist[-1], rel=1e-9)       # mean removal leaves the residual alone
    assert abs(p.mean()) < 1e-12 * np.abs(p).max()
