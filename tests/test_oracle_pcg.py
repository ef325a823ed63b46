"""Pins of the oracle's MG-preconditioned CG (mgo_restrict_adj, mgo_precondition, mgo_solve_pcg;
SURVEY 8(f) rank 1, R22 / C12-C14).  No GPU.

What they catch: a restriction that is not the transpose of the prolongation (weights, wall
clamp, wrap), a preconditioner that is not symmetric (post-smoothing in the wrong order, the
8-child mean left in), a sign slip in alpha / beta, a search direction built from the wrong
vectors.
"""
import itertools
import math

import numpy as np
import pytest

from oracle.mgo import Oracle

P, N = 0, 1
ALL_BC = list(itertools.product((P, N), repeat=3))


def zero_mean(a):
    return a - a.mean()


@pytest.mark.parametrize("bc", ALL_BC)
def test_restrict_adj_is_the_scaled_transpose_of_prolongation(bc, uniform):
    """8 (R' r).e = r.(P e) for random r, e: pins every weight of R', the Neumann clamp and the
    periodic wrap against the prolongation that test_oracle_pins.py pins on its own."""
    n = (16, 12, 8)
    o = Oracle(n, 1.0 / 16, bc)
    r = uniform(3, o.level_shape(0))
    e = uniform(4, o.level_shape(1))
    Pe = o.prolong_add(e, np.zeros(o.level_shape(0)), 0)
    lhs = 8.0 * float((o.restrict_adj(r, 0) * e).sum())
    rhs = float((r * Pe).sum())
    assert abs(lhs - rhs) <= 1e-12 * (np.abs(r).sum() * np.abs(e).max())


def test_restrict_adj_preserves_constants_and_mass():
    o = Oracle((16, 16, 16), 1.0 / 16, (P, N, N))
    one = np.ones(o.level_shape(0))
    assert np.allclose(o.restrict_adj(one, 0), 1.0, rtol=0, atol=1e-15)
    r = np.zeros(o.level_shape(0)); r[5, 6, 7] = 1.0
    assert abs(o.restrict_adj(r, 0).sum() * 8.0 - 1.0) <= 1e-15


@pytest.mark.parametrize("bc", [(P, P, P), (P, P, N), (N, N, N)])
def test_preconditioner_is_symmetric_and_definite(bc, uniform):
    """x.M y = y.M x and x.M x < 0 on zero-mean fields (M approximates the inverse of the
    negative semi-definite A).  The plain V-cycle fails the first by ~1e-2 (checked below)."""
    n = (16, 16, 16)
    o = Oracle(n, 1.0 / 16, bc, 2, 2, 8)
    o.set_density(np.exp(uniform(5, o.shape, math.log(1.2), math.log(998.0))))
    x = zero_mean(uniform(6, o.shape))
    y = zero_mean(uniform(7, o.shape))
    Mx, My = o.precondition(x), o.precondition(y)
    a, b = float((x * My).sum()), float((y * Mx).sum())
    assert abs(a - b) <= 1e-10 * (np.abs(x).sum() * np.abs(My).max())
    assert float((x * Mx).sum()) < 0.0 and float((y * My).sum()) < 0.0
    # the unsymmetric cycle of mgo_vcycle is measurably not symmetric
    Vx = o.vcycle(x, np.zeros(o.shape)); Vy = o.vcycle(y, np.zeros(o.shape))
    assert abs(float((x * Vy).sum()) - float((y * Vx).sum())) > 1e-6 * abs(a)


@pytest.mark.parametrize("bc", [(P, P, P), (N, P, N)])
def test_pcg_matches_dense_solve_8cubed(bc, uniform):
    """PCG reaches the minimum-norm solution of the dense 8^3 system."""
    n = 8
    o = Oracle(n, 1.0 / n, bc, 2, 2, 8)
    o.set_density(np.exp(uniform(8, o.shape, math.log(1.2), math.log(998.0))))
    N3 = n ** 3
    A = np.empty((N3, N3))
    for c in range(N3):
        ec = np.zeros(N3); ec[c] = 1.0
        A[:, c] = o.apply(ec.reshape(o.shape)).reshape(-1)
    f = zero_mean(uniform(9, o.shape))
    x = np.linalg.lstsq(A, f.reshape(-1), rcond=None)[0]
    x -= x.mean()
    p = np.zeros(o.shape)
    st, it, rel, hist = o.solve_pcg(f, p, 1e-12, 50)
    assert st == 0 and it <= 20
    assert np.abs(p.reshape(-1) - x).max() <= 1e-9 * np.abs(x).max()
    # the recurrence residual is the true residual
    assert o.residual(f, p) <= 2e-12 * hist[0] + 1e-13 * hist[0]


def test_pcg_needs_fewer_iterations_than_v_cycles_on_the_drop_film_twin():
    from workloads import make_workload
    w = make_workload(3, 32)
    o = Oracle(w.n, w.h, w.bc, w.nu1, w.nu2)
    o.set_density(w.rho)
    pv = np.zeros(o.shape)
    _, cyc, _, _ = o.solve(w.rhs, pv, w.rtol, 60)
    pc = np.zeros(o.shape)
    st, it, rel, hist = o.solve_pcg(w.rhs, pc, w.rtol, 60)
    assert st == 0 and it < cyc
    assert o.residual(w.rhs, pc) <= 1.01 * w.rtol * hist[0]
    assert np.abs(pc - pv).max() <= 1e-5 * np.abs(pv).max()      # both solve the same system to 1e-8
    assert all(b < a for a, b in zip(hist[2:], hist[3:]))        # monotone once started


def test_pcg_error_codes(uniform):
    from oracle.mgo import OracleError, EINVAL, EINCOMPATIBLE
    o = Oracle(8, 0.125, (P, P, P), 2, 3)
    f = zero_mean(uniform(1, o.shape))
    with pytest.raises(OracleError) as e:
        o.solve_pcg(f, np.zeros(o.shape), 1e-8, 10)          # nu1 != nu2: not symmetric
    assert e.value.code == EINVAL
    o.set_cycle(2, 2)
    with pytest.raises(OracleError) as e:
        o.solve_pcg(f + 1.0, np.zeros(o.shape), 1e-8, 10)
    assert e.value.code == EINCOMPATIBLE
