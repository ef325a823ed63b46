"""Pins of the oracle's per-side boundary conditions with Dirichlet walls (mgo_create6; SURVEY 8(f)
rank 3, R24; the paper's box has a no-slip base, symmetry planes and "continuous" outflow
planes).  No GPU.

What they catch: a wall coefficient that is not 2 (a_c + a_c) (a_c + a_c alone, or the Neumann 0),
a wall neighbour value that is not 0, the minus and the plus wall of an axis mixed up, a wall that
leaks onto a periodic axis, a coarse wall that is not the mean of its four finer wall faces, a
prolongation ghost that is not -e_boundary, a mean removed from (or a compatibility check applied
to) a non-singular system.
"""
import itertools
import math

import numpy as np
import pytest

from oracle import mgo
from oracle.mgo import Oracle

P, N, D = 0, 1, 2


def centres(n, h):
    return (np.arange(n) + 0.5) * h


def axis_mode(bm, bp, k, n, h):
    """Eigenvector and eigenvalue of the 1-D second difference (1/h^2)(v[i-1] - 2 v[i] + v[i+1]) with
    ghost rules v[-1] = v[n-1] (P), v[0] (N), -v[0] (D) and alike on the plus side; x_i = (i+1/2)h."""
    i = np.arange(n) + 0.5
    if (bm, bp) == (P, P):
        th = 2.0 * math.pi * k / n
        v = np.cos(th * i) + np.sin(th * i)
    elif (bm, bp) == (N, N):
        th = math.pi * k / n
        v = np.cos(th * i)
    elif (bm, bp) == (D, D):
        th = math.pi * (k + 1) / n
        v = np.sin(th * i)
    elif (bm, bp) == (N, D):
        th = math.pi * (k + 0.5) / n
        v = np.cos(th * i)
    elif (bm, bp) == (D, N):
        th = math.pi * (k + 0.5) / n
        v = np.sin(th * i)
    else:
        raise ValueError
    return v, -(4.0 / h ** 2) * math.sin(th / 2.0) ** 2


SIDES = [(P, P), (N, N), (D, D), (N, D), (D, N)]


@pytest.mark.parametrize("sx,sy,sz", [c for c in itertools.product(SIDES, repeat=3) if D in c[0] + c[1] + c[2]][::3])
def test_constant_density_eigenmodes_with_dirichlet_walls(sx, sy, sz):
    n, h, rho0 = (12, 8, 16), 1.0 / 16, 3.0
    o = Oracle(n, h, sx + sy + sz)
    o.set_density(np.full(o.shape, rho0))
    vx, lx = axis_mode(*sx, 2, n[0], h)
    vy, ly = axis_mode(*sy, 1, n[1], h)
    vz, lz = axis_mode(*sz, 3, n[2], h)
    v = vz[:, None, None] * vy[None, :, None] * vx[None, None, :]
    lam = (lx + ly + lz) / rho0
    assert np.abs(o.apply(v) - lam * v).max() <= 1e-11 * abs(lam) * np.abs(v).max()


def test_wall_faces_values_and_sides(uniform):
    """Level 0: minus wall in entry 0 of the minus-face array, plus wall in wx / wy / wz; Dirichlet
    2 (a + a) = 2/rho of the wall cell, Neumann 0; a periodic axis has no wall."""
    n = (8, 12, 16)
    o = Oracle(n, 1.0 / 8, (D, N, P, P, N, D))
    rho = np.exp(uniform(101, o.shape, 0.0, 5.0))
    o.set_density(rho)
    bx, by, bz = o.faces(0)
    wx, wy, wz = o.walls(0)
    a = 0.5 / rho
    assert np.array_equal(bx[:, :, 0], 2.0 * (a[:, :, 0] + a[:, :, 0]))        # x-: Dirichlet
    assert np.array_equal(wx, np.zeros_like(wx))                               # x+: Neumann
    assert np.array_equal(by[:, 0, :], a[:, 0, :] + a[:, -1, :])               # y periodic: wrap face
    assert np.array_equal(wy, np.zeros_like(wy))
    assert np.array_equal(bz[0], np.zeros_like(bz[0]))                         # z-: Neumann
    assert np.array_equal(wz, 2.0 * (a[-1] + a[-1]))                           # z+: Dirichlet


@pytest.mark.parametrize("bc", [(D, D, D, D, D, D), (N, D, P, P, D, N)])
def test_coarse_walls_are_means_of_the_four_finer_wall_faces(uniform, bc):
    n = (16, 16, 32)
    o = Oracle(n, 1.0 / 16, bc)
    o.set_density(np.exp(uniform(102, o.shape, math.log(1.2), math.log(998.0))))
    for lvl in range(1, o.num_levels):
        fx, fy, fz = o.walls(lvl - 1)
        cx, cy, cz = o.walls(lvl)
        for f, c in ((fx, cx), (fy, cy), (fz, cz)):
            # C3 order: pairs over the faster in-plane axis first, then over the slower one
            want = 0.25 * ((f[0::2, 0::2] + f[0::2, 1::2]) + (f[1::2, 0::2] + f[1::2, 1::2]))
            assert np.array_equal(c, want), f"level {lvl}"
        # and the minus walls through the ordinary C3 rule
        fbx, fby, fbz = o.faces(lvl - 1)
        cbx, cby, cbz = o.faces(lvl)
        want = 0.25 * ((fbx[0::2, 0::2, 0] + fbx[0::2, 1::2, 0]) + (fbx[1::2, 0::2, 0] + fbx[1::2, 1::2, 0]))
        assert np.array_equal(cbx[:, :, 0], want)
    # constant density: every Dirichlet wall on every level is 2 / rho
    o.set_density(np.full(o.shape, 4.0))
    for lvl in range(o.num_levels):
        for w, side in zip(o.walls(lvl), (bc[1], bc[3], bc[5])):
            assert np.all(w == (0.5 if side == D else 0.0))


@pytest.mark.parametrize("bc", [(N, D, P, P, N, D), (D, D, N, N, P, P), (N, N, N, N, N, D)])
def test_symmetry_and_strict_definiteness(uniform, bc):
    n = (8, 12, 8)
    o = Oracle(n, 1.0 / 8, bc)
    o.set_density(np.exp(uniform(103, o.shape, math.log(1.2), math.log(998.0))))
    x, y = uniform(104, o.shape), uniform(105, o.shape)
    Ax, Ay = o.apply(x), o.apply(y)
    assert abs(float((x * Ay).sum()) - float((y * Ax).sum())) <= 1e-12 * np.abs(x).sum() * np.abs(Ay).max()
    assert float((x * Ax).sum()) < 0.0
    one = np.ones(o.shape)
    assert float((one * o.apply(one)).sum()) < 0.0          # constants are no longer in the null space


def test_layered_medium_with_dirichlet_top(uniform):
    """rho = rho(z), f = f(z), Neumann bottom, Dirichlet top, periodic x / y: the discrete solution
    follows from flux continuity, bottom up: beta_{k+1/2} (p_{k+1} - p_k) = h^2 sum_{m<=k} f_m, and
    at the top wall beta_w (0 - p_{n-1}) = h^2 sum_m f_m with beta_w = 2 (a + a) = 2 / rho_{n-1}."""
    n, h = 32, 1.0 / 32
    o = Oracle((8, 8, n), h, (P, P, P, P, N, D))
    rho_z = np.where(np.arange(n) < 10, 935.0, 1.2) * (1.0 + 0.1 * np.cos(np.arange(n)))
    fz = uniform(106, (n,))
    o.set_density(np.broadcast_to(rho_z[:, None, None], o.shape).copy())
    f = np.broadcast_to(fz[:, None, None], o.shape).copy()
    a = 0.5 / rho_z
    p = np.zeros(n)
    F = np.cumsum(fz) * h * h
    p[n - 1] = -F[n - 1] / (2.0 * (a[n - 1] + a[n - 1]))
    for k in range(n - 2, -1, -1):
        p[k] = p[k + 1] - F[k] / (a[k] + a[k + 1])
    q = np.zeros(o.shape)
    st, cyc, rel, hist = o.solve(f, q, 1e-13, 200)
    assert st == mgo.OK
    assert np.abs(q - p[:, None, None]).max() <= 1e-9 * np.abs(p).max()


@pytest.mark.parametrize("bc", [(N, D, N, D, N, D), (D, D, P, P, N, N)])
def test_dense_direct_solve_8cubed_nonsingular(uniform, bc):
    n = 8
    o = Oracle((n, n, n), 1.0 / n, bc, 2, 2)
    o.set_density(np.exp(uniform(107, o.shape, math.log(1.2), math.log(998.0))))
    N3 = n ** 3
    A = np.empty((N3, N3))
    e = np.zeros(N3)
    for c in range(N3):
        e[c] = 1.0
        A[:, c] = o.apply(e.reshape(o.shape)).reshape(-1)
        e[c] = 0.0
    assert np.abs(A - A.T).max() <= 1e-12 * np.abs(A).max()
    assert np.linalg.eigvalsh(0.5 * (A + A.T))[-1] < 0.0                 # no zero eigenvalue
    f = uniform(108, o.shape) + 0.3                                      # NOT mean-free: must be accepted
    p_dense = np.linalg.solve(A, f.reshape(-1)).reshape(o.shape)
    p = np.zeros(o.shape)
    st, cyc, rel, hist = o.solve(f, p, 1e-13, 300)
    assert st == mgo.OK
    assert np.abs(p - p_dense).max() <= 1e-9 * np.abs(p_dense).max()     # and no mean was removed
    assert abs(p_dense.mean()) > 1e-6 * np.abs(p_dense).max()


def test_prolongation_ghost_beyond_a_dirichlet_wall():
    """A coarse delta in the wall cell: the fine cell next to the wall gets 3/4 e - 1/4 e = e/2 per
    Dirichlet axis (Neumann: 3/4 + 1/4 = e).  A function linear in the distance to the wall is
    reproduced exactly up to the wall."""
    o = Oracle((16, 16, 16), 1.0 / 16, (D, N, N, N, N, D))
    e = np.zeros(o.level_shape(1))
    e[0, 0, 0] = 1.0                     # coarse cell at x-: Dirichlet, y-: Neumann, z-: Neumann
    out = o.prolong_add(e, np.zeros(o.shape), 0)
    assert out[0, 0, 0] == 0.5 * 1.0 * 1.0
    assert out[0, 0, 1] == 0.75
    e[:] = 0.0
    e[-1, 0, 0] = 1.0                    # z+ is Dirichlet, x- too
    out = o.prolong_add(e, np.zeros(o.shape), 0)
    assert out[-1, 0, 0] == 0.25 and out[-2, 0, 0] == 0.5 * 0.75
    # linear in the distance to the x- wall: coarse centres at (I + 1/2) H, fine at (i + 1/2) h, H = 2h
    H, h = 2.0 / 16, 1.0 / 16
    lin = np.broadcast_to(((np.arange(8) + 0.5) * H)[None, None, :], o.level_shape(1)).copy()
    out = o.prolong_add(lin, np.zeros(o.shape), 0)
    want = (np.arange(16) + 0.5) * h
    assert np.abs(out[4, 4, :15] - want[:15]).max() <= 1e-15       # the last cell sees the Neumann clamp


@pytest.mark.parametrize("n", [32, 64])
def test_manufactured_solution_second_order_with_outflow_walls(n):
    """Smooth p* vanishing on the Dirichlet walls (x+, z+), even across the Neumann walls (x-, z-),
    periodic in y, smooth variable density: the error of the discrete solution drops 4x per refinement."""
    errs = []
    for m in (n, 2 * n):
        h = 1.0 / m
        o = Oracle((m, m, m), h, (N, D, P, P, N, D), 2, 2)
        x = centres(m, h)
        Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
        ps = np.cos(0.5 * math.pi * X) * np.cos(2 * math.pi * Y) * np.cos(1.5 * math.pi * Z)
        rho = 1.0 + 0.5 * np.sin(2 * math.pi * Y) * np.cos(math.pi * X)
        o.set_density(rho)
        # rhs from the continuous operator div((1/rho) grad p*), evaluated at cell centres
        b = 1.0 / rho
        bx_ = -b * b * (-0.5 * math.pi * np.sin(2 * math.pi * Y) * np.sin(math.pi * X))
        by_ = -b * b * (math.pi * np.cos(2 * math.pi * Y) * np.cos(math.pi * X))
        px = -0.5 * math.pi * np.sin(0.5 * math.pi * X) * np.cos(2 * math.pi * Y) * np.cos(1.5 * math.pi * Z)
        py = -2 * math.pi * np.cos(0.5 * math.pi * X) * np.sin(2 * math.pi * Y) * np.cos(1.5 * math.pi * Z)
        lap = -((0.5 * math.pi) ** 2 + (2 * math.pi) ** 2 + (1.5 * math.pi) ** 2) * ps
        f = b * lap + bx_ * px + by_ * py
        p = np.zeros(o.shape)
        st, cyc, rel, _ = o.solve(f, p, 1e-12, 100)
        assert st == mgo.OK
        errs.append(np.abs(p - ps).max())
    assert 3.3 <= errs[0] / errs[1] <= 4.7, errs


def test_paper_box_converges_and_exact_solution_is_fixed_point(uniform):
    """No-slip base (Neumann for p), symmetry planes x-, y- (Neumann), outflow x+, y+, z+ (Dirichlet)."""
    bc = (N, D, N, D, N, D)
    o = Oracle((32, 32, 32), 1.0 / 32, bc, 3, 3)
    o.set_density(np.exp(uniform(109, o.shape, math.log(1.2), math.log(998.0))))
    p_true = uniform(110, o.shape)
    f = o.apply(p_true)
    p = p_true.copy()
    o.vcycle(f, p)
    assert np.abs(p - p_true).max() <= 1e-11 * np.abs(p_true).max()
    q = np.zeros(o.shape)
    st, cyc, rel, hist = o.solve(f, q, 1e-10, 60)
    assert st == mgo.OK and cyc <= 25
    assert np.abs(q - p_true).max() <= 1e-7 * np.abs(p_true).max()


def test_create6_argument_checks():
    for bad in [(P, N, P, P, P, P), (N, P, N, N, N, N), (3, 3, N, N, N, N), (N, N, N, N, -1, N)]:
        with pytest.raises(mgo.OracleError):
            Oracle((8, 8, 8), 1.0 / 8, bad)
    o = Oracle((8, 8, 8), 1.0 / 8, (N, D, N, N, N, N))
    z = np.zeros(o.shape)
    with pytest.raises(mgo.OracleError):           # PCG / projection: periodic and Neumann sides only
        o.precondition(z)


def test_three_entry_form_equals_six_entry_form(uniform):
    """mgo_create(bc[3]) is mgo_create6 with both sides alike."""
    n = (16, 8, 8)
    rho = np.exp(uniform(111, (8, 8, 16), 0.0, 5.0))
    f = uniform(112, (8, 8, 16))
    f -= f.mean()
    outs = []
    for bc in ((P, N, N), (P, P, N, N, N, N)):
        o = Oracle(n, 1.0 / 16, bc)
        o.set_density(rho)
        outs.append(o.vcycle(f, np.zeros(o.shape)))
    assert np.array_equal(outs[0], outs[1])
