"""Pins of the oracle's F- and W-cycles (mgo_set_cycle_type, R23).
No GPU.

The cycle index is a schedule over steps that tests/test_oracle_pins.py pins one by one (sweep,
residual, restriction, prolongation).  What these tests fix about the schedule itself:

* the visit sequence: the event trace of an independent recursion written from the textbook
  definition (V: one visit of the coarse problem, W: two, F: an F visit then a V visit), replayed
  through the single-step calls, gives the same field bit for bit; a cycle that visits a level
  once too often or too seldom, zeroes the correction before the second visit, or recurses with
  the wrong index fails;
* closed forms of the visit counts per level (V: 1; W: 2^l; F: l + 1);
* the exact solution is a fixed point, and the iteration converges to the dense direct solution
  of a 16^3 problem (three levels, so V, F and W differ);
* on a two-level hierarchy the three cycles coincide.
"""
import math

import numpy as np
import pytest

from oracle import mgo
from oracle.mgo import Oracle

P, N = 0, 1
V, F, W = 0, 1, 2


def reference_cycle(o, lvl, p, f, typ, nu1, nu2, coarse_sweeps, trace):
    """The cycle written out from its definition on top of the oracle's single steps."""
    trace.append(lvl)
    last = o.num_levels - 1
    if lvl == last:
        for _ in range(coarse_sweeps):
            o.sweep(f, p, lvl)
        return
    for _ in range(nu1):
        o.sweep(f, p, lvl)
    fc = o.restrict(o.residual_level(f, p, lvl), lvl)
    e = np.zeros(o.level_shape(lvl + 1))
    reference_cycle(o, lvl + 1, e, fc, typ, nu1, nu2, coarse_sweeps, trace)
    if lvl + 1 < last:
        if typ == W:
            reference_cycle(o, lvl + 1, e, fc, W, nu1, nu2, coarse_sweeps, trace)
        elif typ == F:
            reference_cycle(o, lvl + 1, e, fc, V, nu1, nu2, coarse_sweeps, trace)
    o.prolong_add(e, p, lvl)
    for _ in range(nu2):
        o.sweep(f, p, lvl)


@pytest.mark.parametrize("typ", [V, F, W])
@pytest.mark.parametrize("n,bc", [((32, 32, 32), (P, P, N)), ((48, 32, 16), (N, P, P))])
def test_cycle_equals_the_recursion_over_single_steps(uniform, typ, n, bc):
    o = Oracle(n, 1.0 / n[0], bc, 2, 1, 5)
    o.set_density(np.exp(uniform(81, o.shape, math.log(1.2), math.log(998.0))))
    o.set_cycle_type(typ)
    f = uniform(82, o.shape)
    f -= f.mean()
    p = uniform(83, o.shape)
    q = p.copy()
    trace = []
    reference_cycle(o, 0, q, f, typ, 2, 1, 5, trace)
    o.vcycle(f, p)
    assert np.array_equal(p, q)
    # visits per level: V 1, W 2^l (the coarsest level is visited once per visit of its parent),
    # F l + 1 (same exception)
    L = o.num_levels
    visits = [trace.count(l) for l in range(L)]
    if typ == V:
        want = [1] * L
    elif typ == W:
        want = [2 ** l for l in range(L - 1)] + [2 ** (L - 2)]
    else:
        want = [l + 1 for l in range(L - 1)] + [L - 1]
    assert visits == want


def test_cycle_types_coincide_on_two_levels(uniform):
    outs = []
    for typ in (V, F, W):
        o = Oracle((8, 8, 8), 1.0 / 8, (P, N, P), 2, 2)
        assert o.num_levels == 2
        o.set_density(np.exp(uniform(84, o.shape, 0.0, 5.0)))
        o.set_cycle_type(typ)
        f = uniform(85, o.shape)
        f -= f.mean()
        outs.append(o.vcycle(f, np.zeros(o.shape)))
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


@pytest.mark.parametrize("typ", [F, W])
def test_exact_solution_is_a_fixed_point(uniform, typ):
    n = 32
    o = Oracle((n, n, n), 1.0 / n, (P, P, N), 3, 3)
    o.set_density(np.exp(uniform(86, o.shape, 0.0, 5.0)))
    o.set_cycle_type(typ)
    p_true = uniform(87, o.shape)
    f = o.apply(p_true)
    p = p_true.copy()
    o.vcycle(f, p)
    assert np.abs(p - p_true).max() <= 1e-11 * np.abs(p_true).max()


@pytest.mark.parametrize("typ", [F, W])
def test_dense_direct_solve_16cubed(uniform, typ):
    """Three levels (16, 8, 4): the F- and W-cycle differ from the V-cycle and must still converge
    to the solution of the mean-constrained dense system built from the oracle's operator."""
    n = 16
    o = Oracle((n, n, n), 1.0 / n, (P, P, N), 2, 2)
    assert o.num_levels == 3
    o.set_density(np.exp(uniform(88, o.shape, math.log(1.2), math.log(998.0))))
    N3 = n ** 3
    K = np.zeros((N3 + 1, N3 + 1))
    e = np.zeros(N3)
    for c in range(N3):
        e[c] = 1.0
        K[:N3, c] = o.apply(e.reshape(o.shape)).reshape(-1)
        e[c] = 0.0
    K[:N3, N3] = 1.0
    K[N3, :N3] = 1.0
    f = uniform(89, o.shape)
    f -= f.mean()
    p_dense = np.linalg.solve(K, np.concatenate([f.reshape(-1), [0.0]]))[:N3].reshape(o.shape)
    o.set_cycle_type(typ)
    p = np.zeros(o.shape)
    st, cyc, rel, hist = o.solve(f, p, 1e-13, 200)
    assert st == mgo.OK
    assert np.abs(p - p_dense).max() <= 1e-9 * np.abs(p_dense).max()
    # and it is a different iteration from the V-cycle's
    o.set_cycle_type(V)
    pv = np.zeros(o.shape)
    o.vcycle(f, pv)
    o.set_cycle_type(typ)
    pt = np.zeros(o.shape)
    o.vcycle(f, pt)
    assert not np.array_equal(pv, pt)


def test_f_and_w_cycles_need_no_more_cycles_than_v_on_the_drop_film_twin():
    """64^3 twin of config 3/4 (measured: V 10, F 9, W 9 cycles to 1e-8)."""
    from workloads import make_workload

    w = make_workload(3, 64)
    counts = {}
    for typ in (V, F, W):
        o = Oracle(w.n, w.h, w.bc, w.nu1, w.nu2)
        o.set_cycle_type(typ)
        o.set_density(w.rho)
        st, cyc, rel, _ = o.solve(w.rhs, np.zeros(o.shape), w.rtol, 40)
        assert st == mgo.OK
        counts[typ] = cyc
    assert counts[F] <= counts[V] and counts[W] <= counts[F]


def test_cycle_type_argument_is_checked():
    o = Oracle((8, 8, 8), 1.0 / 8, (P, P, P))
    for bad in (-1, 3):
        with pytest.raises(mgo.OracleError):
            o.set_cycle_type(bad)
