"""Pins of the oracle's projection steps (mgo_project_rhs, mgo_project_correct; SURVEY 8(f)
rank 2, R21/C10/C11) against what the mathematics fixes.  No GPU.

Mistakes they are chosen to catch: a wrong staggering (plus instead of minus face), a wrong
sign or a missing 1/h or 1/dt, a transposed axis, the cell density instead of the face
coefficient, a wall face that moves, a wrap that is off by one.
"""
import itertools
import math

import numpy as np
import pytest

from oracle.mgo import Oracle

P, N = 0, 1
ALL_BC = list(itertools.product((P, N), repeat=3))


def staggered_fields(uniform, seed, shape, bc):
    u, v, w = (uniform(seed + q, shape) for q in range(3))
    # no-penetration walls: the wrap face of a Neumann axis is the wall
    if bc[0] == N:
        u[:, :, 0] = 0.0
    if bc[1] == N:
        v[:, 0, :] = 0.0
    if bc[2] == N:
        w[0, :, :] = 0.0
    return u, v, w


def test_rhs_of_linear_and_constant_fields():
    """u = x on the faces (x_face = i*h), v = w = const: div = 1 in the interior, so f = 1/dt
    there; catches a missing 1/h or 1/dt and a plus/minus-face mix-up (which would shift the
    jump cell of the periodic wrap to the other end)."""
    n, h, dt = (16, 12, 8), 0.125, 0.25
    o = Oracle(n, h, (P, P, P))
    x = np.arange(n[0]) * h
    u = np.broadcast_to(x, (n[2], n[1], n[0])).copy()
    v = np.full_like(u, 3.0)
    w = np.full_like(u, -2.0)
    f = o.project_rhs(u, v, w, dt)
    assert np.allclose(f[:, :, :-1], 1.0 / dt, rtol=1e-14, atol=0)
    # the wrap face closes the loop: last cell sees u[0] - u[nx-1] = -(nx-1)h
    assert np.allclose(f[:, :, -1], -(n[0] - 1) / dt, rtol=1e-14, atol=0)
    # each axis separately: a transposed axis would put the jump in the wrong direction
    y = np.arange(n[1]) * h
    v2 = np.broadcast_to(y[None, :, None], u.shape).copy()
    f2 = o.project_rhs(np.zeros_like(u), v2, np.zeros_like(u), dt)
    assert np.allclose(f2[:, :-1, :], 1.0 / dt, rtol=1e-14, atol=0) and np.allclose(f2[:, -1, :], -(n[1] - 1) / dt)
    z = np.arange(n[2]) * h
    w2 = np.broadcast_to(z[:, None, None], u.shape).copy()
    f3 = o.project_rhs(np.zeros_like(u), np.zeros_like(u), w2, dt)
    assert np.allclose(f3[:-1, :, :], 1.0 / dt, rtol=1e-14, atol=0) and np.allclose(f3[-1, :, :], -(n[2] - 1) / dt)


@pytest.mark.parametrize("bc", ALL_BC)
def test_rhs_is_compatible(bc, uniform):
    """Discrete Gauss theorem: with periodic axes and closed walls the divergence sums to zero
    (telescoping), so the assembled rhs passes the solver's compatibility test."""
    n, h, dt = (12, 16, 8), 1.0 / 16, 1e-3
    o = Oracle(n, h, bc)
    u, v, w = staggered_fields(uniform, 11, o.shape, bc)
    f = o.project_rhs(u, v, w, dt)
    assert abs(f.sum()) <= 1e-11 * np.abs(f).sum()


@pytest.mark.parametrize("bc", [(P, P, P), (P, P, N), (N, P, N), (N, N, N)])
def test_divergence_after_correction_is_dt_times_residual(bc, uniform):
    """For ANY p: div(u - dt beta grad p)/dt = f - A p cell by cell.  Ties project_rhs and
    project_correct to the operator pinned in test_oracle_pins.py: a wrong sign, a cell-centred
    instead of a face coefficient, or a minus/plus-face slip in either function breaks it."""
    n, h, dt = (12, 8, 16), 1.0 / 16, 0.02
    o = Oracle(n, h, bc)
    rho = np.exp(uniform(5, o.shape, math.log(1.2), math.log(998.0)))
    o.set_density(rho)
    u, v, w = staggered_fields(uniform, 21, o.shape, bc)
    p = uniform(31, o.shape)
    f = o.project_rhs(u, v, w, dt)
    r = f - o.apply(p)
    u2, v2, w2 = u.copy(), v.copy(), w.copy()
    o.project_correct(p, dt, u2, v2, w2)
    d = o.project_rhs(u2, v2, w2, dt)
    scale = np.abs(f).max() + np.abs(o.apply(p)).max()
    assert np.abs(d - r).max() <= 1e-12 * scale
    # walls do not move
    if bc[0] == N:
        assert np.all(u2[:, :, 0] == 0.0)
    if bc[1] == N:
        assert np.all(v2[:, 0, :] == 0.0)
    if bc[2] == N:
        assert np.all(w2[0, :, :] == 0.0)


def test_correction_closed_form_constant_density():
    """rho = 2 => beta = 1/2 on every face; p = sin mode in x only: u changes by
    -dt/(2h) (p_i - p_{i-1}), v and w do not change."""
    n, h, dt = 16, 1.0 / 16, 0.1
    o = Oracle(n, h, (P, P, P))
    o.set_density(np.full(o.shape, 2.0))
    x = (np.arange(n) + 0.5) * h
    p1 = np.sin(2 * math.pi * x)
    p = np.broadcast_to(p1, o.shape).copy()
    u = np.zeros(o.shape); v = np.ones(o.shape); w = np.ones(o.shape)
    o.project_correct(p, dt, u, v, w)
    expect = -dt / (2.0 * h) * (p1 - np.roll(p1, 1))
    assert np.allclose(u, np.broadcast_to(expect, o.shape), rtol=1e-13, atol=1e-15)
    assert np.all(v == 1.0) and np.all(w == 1.0)


def test_projection_makes_the_field_divergence_free(uniform):
    """The whole step on a small drop-like density: rhs -> solve -> correct leaves a
    divergence of dt * (final residual), i.e. 1e-10 of the initial one."""
    n, h, dt = 32, 1.0 / 32, 1e-2
    bc = (P, P, N)
    o = Oracle(n, h, bc, 2, 2)
    zc, yc, xc = np.meshgrid(*(3 * [(np.arange(n) + 0.5) * h]), indexing="ij")
    rho = np.where((xc - 0.5) ** 2 + (yc - 0.5) ** 2 + (zc - 0.4) ** 2 < 0.2 ** 2, 998.0, 1.2)
    o.set_density(rho)
    u, v, w = staggered_fields(uniform, 41, o.shape, bc)
    f = o.project_rhs(u, v, w, dt)
    p = np.zeros(o.shape)
    st, cyc, rel, hist = o.solve(f, p, 1e-10, 60)
    assert st == 0
    o.project_correct(p, dt, u, v, w)
    d = o.project_rhs(u, v, w, dt)
    assert np.sqrt((d ** 2).sum()) <= 2e-10 * np.sqrt((f ** 2).sum())


def test_projection_error_codes(uniform):
    o = Oracle(8, 0.125, (P, P, P))
    z = np.zeros(o.shape)
    from oracle.mgo import OracleError
    for bad_dt in (0.0, -1.0, float("nan"), float("inf")):
        with pytest.raises(OracleError):
            o.project_rhs(z, z, z, bad_dt)
        with pytest.raises(OracleError):
            o.project_correct(z, bad_dt, z.copy(), z.copy(), z.copy())
