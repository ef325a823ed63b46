"""The branch-free reciprocal of the TMA sweep kernels (rt_rcp_fast, csrc/mg_rbt_kernels.cuh) against
the definition C5 uses: the correctly rounded 1.0 / D, taken from the HOST's IEEE division (numpy),
bit for bit -- not from the values the parity tests happen to visit.

mg_set_density admits the sequence while every a = 0.5/rho lies in [2^-900, 2^900]; a diagonal D is
a sum of at most six faces a_c + a_nb (or 4 a_c at a Dirichlet wall), so D ranges over
[2^-900, 2^905).  Covered: 1.3e8 seeded values with uniform exponent over that range and random
mantissas, every exponent of the range with the extreme mantissas (0, 1 ulp, all ones, all ones - 1 ulp),
both signs.  Then a parity case whose density leaves the admitted range mid-life, so that the handle
drops its graph and runs the kernels built on the library reciprocal (FR = false) against the oracle
(that the switch happened is checked through the kernel names ncu lists, profiles/r3_cycle.md; here the
fields must simply stay bit-exact across it).
"""
import ctypes as C

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

E_LO, E_HI = -900, 904


@pytest.fixture(scope="module")
def mgmod():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2605_30082_b200 as m
    return m


def both_reciprocals(mgmod, d):
    from paper_2605_30082_b200 import binding as B

    dd = torch.from_numpy(d).to("cuda:0")
    fast, libv = torch.empty_like(dd), torch.empty_like(dd)
    st = B.lib().mg_test_rcp(dd.data_ptr(), dd.numel(), fast.data_ptr(), libv.data_ptr(),
                             torch.cuda.current_stream().cuda_stream)
    assert st == 0
    return fast.cpu().numpy(), libv.cpu().numpy()


def from_bits(sign, expo, mant):
    bits = (sign.astype(np.uint64) << np.uint64(63)) | ((expo + 1023).astype(np.uint64) << np.uint64(52)) | mant.astype(np.uint64)
    return bits.view(np.float64)


def test_extreme_mantissas_at_every_exponent(mgmod):
    expo = np.arange(E_LO, E_HI + 1, dtype=np.int64)
    top = (1 << 52) - 1
    mants = np.array([0, 1, 2, 3, top, top - 1, 1 << 51, (1 << 51) - 1, (1 << 51) + 1, 0x5555555555555, 0xAAAAAAAAAAAAA], dtype=np.uint64)
    e, m = np.meshgrid(expo, mants, indexing="ij")
    for sign in (0, 1):
        d = from_bits(np.full(e.size, sign), e.ravel(), m.ravel())
        want = 1.0 / d
        fast, libv = both_reciprocals(mgmod, d)
        assert np.array_equal(libv.view(np.uint64), want.view(np.uint64))
        assert np.array_equal(fast.view(np.uint64), want.view(np.uint64))


@pytest.mark.parametrize("chunk", range(8))
def test_seeded_values_over_the_admitted_range(mgmod, chunk):
    n = 1 << 24                                     # 8 chunks: 1.34e8 values
    rng = np.random.Generator(np.random.Philox(key=20260530 + chunk))
    expo = rng.integers(E_LO, E_HI + 1, n, dtype=np.int64)
    mant = rng.integers(0, 1 << 52, n, dtype=np.uint64)
    sign = (rng.integers(0, 4, n, dtype=np.int64) == 0)           # a quarter negative
    d = from_bits(sign, expo, mant)
    want = 1.0 / d
    fast, libv = both_reciprocals(mgmod, d)
    assert np.array_equal(libv.view(np.uint64), want.view(np.uint64))
    bad = np.nonzero(fast.view(np.uint64) != want.view(np.uint64))[0]
    assert bad.size == 0, (bad.size, d[bad[:4]], fast[bad[:4]], want[bad[:4]])


@pytest.mark.parametrize("n,bc,opts", [((72, 40, 36), (0, 1, 1), {}),
                                       ((128, 64, 64), (1, 0, 1), {"face_log2": 0, "fuse": 3}),
                                       ((64, 64, 64), (0, 0, 1), {"head": 1, "fuse": 3})],
                         ids=["default", "faces-streamed-two-sweeps", "head"])
def test_density_outside_the_range_switches_to_the_library_reciprocal(mgmod, uniform, n, bc, opts):
    """rho so large that a = 0.5/rho < 2^-900 in some cells: mg_set_density must notice, drop the
    captured graph and run the FR = false kernels; the cycle stays the oracle's bit for bit.  Then
    back to an ordinary density (fast path again) on the same handle."""
    from oracle.mgo import Oracle

    from paper_2605_30082_b200 import binding as B

    shp = (n[2], n[1], n[0])
    h = 1.0 / n[0]
    rho_ok = np.exp(uniform(41, shp, np.log(1.2), np.log(998.0)))
    rho_wide = rho_ok.copy()
    # isolated cells (no two adjacent) with a = 0.5/rho = 2^-906, below the admitted 2^-900: every face and
    # diagonal stays an ordinary number (the neighbours' a dominates), so nothing overflows, but
    # mg_set_density must still leave the branch-free reciprocal
    rho_wide[3::7, 3::5, 3::9] = 2.0 ** 905
    f = uniform(42, shp)
    f -= f.mean()
    o = Oracle(n, h, bc, 3, 3, 8)
    g = mgmod.Multigrid(n, h, bc, 3, 3, 8)
    for key, name in ((B.MG_OPT_FACE_STREAM_LOG2, "face_log2"), (B.MG_OPT_SWEEP_FUSE, "fuse"), (B.MG_OPT_PROLONG_FUSE, "head")):
        if name in opts:
            g.set_option(key, opts[name])
    fd = torch.from_numpy(f).to("cuda:0")
    po, pg = np.zeros(shp), torch.zeros(shp, dtype=torch.float64, device="cuda:0")
    for rho in (rho_ok, rho_wide, rho_wide, rho_ok):
        o.set_density(rho)
        g.set_density(torch.from_numpy(rho).to("cuda:0"))
        for _ in range(2):
            o.vcycle(f, po)
            g.vcycle(fd, pg)
            assert np.array_equal(po, pg.cpu().numpy())
        # the sweeps, the fused tails and the two-sweep pass one by one on level 0
        q_o, q_g = po.copy(), pg.clone()
        o.sweep(f, q_o)
        o.sweep(f, q_o)
        g.level_smooth(0, 2, fd, q_g)
        assert np.array_equal(q_o, q_g.cpu().numpy())
        fc = g.level_smooth_restrict(0, 1, fd, q_g)
        o.sweep(f, q_o)
        assert np.array_equal(q_o, q_g.cpu().numpy())
        assert np.array_equal(o.restrict(o.residual_level(f, q_o)), fc.cpu().numpy())
