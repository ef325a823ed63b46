"""Pins for the seeded input generators (workloads/): PRNG known answers and the
structure the recipes of SURVEY.md 8(d) promise.  No solver arithmetic involved."""
from pathlib import Path

import numpy as np
import pytest

from workloads import CONFIGS, make_workload, splitmix64_uniform

GOLDEN = Path(__file__).parent / "golden"


def test_splitmix64_known_answers():
    for line in (GOLDEN / "splitmix64_kat.txt").read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        seed, *outs = (int(t) for t in line.split())
        u = splitmix64_uniform(seed, len(outs))
        want = np.array([(z >> 11) * 2.0 ** -53 for z in outs])
        assert np.array_equal(u, want)
        # offset draws continue the same stream
        assert np.array_equal(splitmix64_uniform(seed, 2, offset=len(outs) - 2), want[-2:])
    assert 0.0 <= splitmix64_uniform(7, 1000).min() and splitmix64_uniform(7, 1000).max() < 1.0


def test_config1_is_an_eigenmode_recipe():
    w = make_workload(1)
    assert w.n == (32, 32, 32) and w.bc == (0, 0, 0) and (w.nu1, w.nu2) == (2, 2) and w.rtol == 1e-10
    assert w.eigenvalue == pytest.approx(-118.05523720255212, rel=1e-14)
    assert np.all(w.rho == 1.0)
    assert np.array_equal(w.rhs, w.eigenvalue * w.p_exact)
    assert abs(w.rhs.sum()) < 1e-9


@pytest.mark.parametrize("cfg,n", [(2, 32), (3, 32), (3, 64), (5, 64)])
def test_density_phases_and_mean_free_rhs(cfg, n):
    w = make_workload(cfg, n)
    assert w.rho.shape == (n, n, n) and w.rhs.shape == (n, n, n)
    assert w.rho.min() >= 1.2 and w.rho.max() <= 998.0
    assert (w.rho == 1.2).any() and (w.rho == 998.0).any()      # pure-phase cells are exact
    mean = float(np.sum(w.rhs, dtype=np.longdouble)) / w.rhs.size
    assert abs(mean) <= 1e-13 * np.sqrt(np.mean(w.rhs ** 2))
    if cfg in (3, 5):
        assert w.bc == (0, 0, 1)
        assert (w.rho == 935.0).any()
        # air far above the film and the drop
        assert np.all(w.rho[-n // 4:] == 1.2)
    # mixed cells exist and are 1/64-quantised combinations
    mixed = w.rho[(w.rho != 1.2) & (w.rho != 998.0) & (w.rho != 935.0)]
    assert mixed.size > 0


def test_film_fraction_layer():
    # n = 64: film_top = 0.10 = 6.4 h -> layer k = 6 has 2 of 4 z-samples below 6.4 (6.125, 6.375)
    w = make_workload(3, 64)
    far = w.rho[:, 2, 2]           # a column far from the drop
    assert np.all(far[:6] == 935.0)
    assert far[6] == pytest.approx(935.0 * 0.5 + 1.2 * 0.5, rel=1e-15)
    assert np.all(far[7:] == 1.2)


def test_sphere_volume():
    w = make_workload(2, 64)
    frac = (w.rho - 1.2) / (998.0 - 1.2)
    vol = frac.sum() / 64 ** 3
    assert vol == pytest.approx(4.0 / 3.0 * np.pi * 0.25 ** 3, rel=2e-3)
    # symmetric under reflection of each axis (centred sphere, symmetric sub-samples)
    assert np.allclose(w.rho, w.rho[::-1], rtol=0, atol=1e-12)
    assert np.allclose(w.rho, w.rho[:, ::-1], rtol=0, atol=1e-12)
    assert np.allclose(w.rho, w.rho[:, :, ::-1], rtol=0, atol=1e-12)


def test_generation_is_reproducible():
    a, b = make_workload(3, 32), make_workload(3, 32)
    assert np.array_equal(a.rho, b.rho) and np.array_equal(a.rhs, b.rhs)
    assert not np.array_equal(make_workload(2, 32).rhs, make_workload(3, 32).rhs)
    assert set(CONFIGS) == {1, 2, 3, 4, 5}


def test_velocity_field_reproduces_the_rhs_of_config3():
    """The materialised 16-mode staggered velocity is the field behind the workload's rhs:
    its divergence (oracle C10, dt = 1) equals rhs up to rounding and the removed mean, and it
    has closed walls in z."""
    import numpy as np
    from oracle.mgo import Oracle
    from workloads import make_workload, velocity_field

    w = make_workload(3, 32)
    u, v, ww = velocity_field(w.n, w.h, w.seed)
    assert np.all(ww[0] == 0.0)
    o = Oracle(w.n, w.h, w.bc)
    f = o.project_rhs(u, v, ww, 1.0)
    f -= f.mean()
    assert np.abs(f - w.rhs).max() <= 1e-10 * np.abs(w.rhs).max()
