"""The five BASELINE.json configs as seeded synthetic inputs.

Array convention everywhere in this repo: dense fp64, x fastest,
``idx = i + nx*(j + ny*k)``; as numpy that is a C-contiguous array of shape
``(nz, ny, nx)``.  Unit cube, ``h = 1/nx``, cell centre ``x_i = (i + 1/2) h``.

Nothing here is solver arithmetic: densities follow the volume-fraction mixing of
PAPER.md:47-52 (eq. 5) with fractions from 4^3 sub-sampling, the
right-hand sides are closed-form / seeded fields.  The generator's own rounding
never enters a parity comparison because the very same buffers go to both sides.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional, Tuple

import numpy as np

PERIODIC = 0
NEUMANN = 1

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64_uniform(seed: int, count: int, offset: int = 0) -> np.ndarray:
    """`count` uniform doubles in [0,1) from splitmix64 seeded with `seed`.

    Draw number ``q`` (0-based, ``q = offset + t``) is the q-th output of the
    sequential generator ``s += GOLDEN; z = mix(s)``; since the state is a pure
    counter this vectorises.  ``u = (z >> 11) * 2^-53``.
    """
    with np.errstate(over="ignore"):
        q = np.arange(offset + 1, offset + count + 1, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + q * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


class _Stream:
    """Sequential reader over the splitmix64 stream of one seed."""

    def __init__(self, seed: int):
        self.seed = seed
        self.pos = 0

    def uniform(self, count: int = 1) -> np.ndarray:
        u = splitmix64_uniform(self.seed, count, self.pos)
        self.pos += count
        return u

    def real(self, lo: float, hi: float) -> float:
        return lo + (hi - lo) * float(self.uniform()[0])

    def integer(self, lo: int, hi: int) -> int:
        return lo + int(math.floor(float(self.uniform()[0]) * (hi - lo + 1)))


@dataclass
class Workload:
    name: str
    n: Tuple[int, int, int]            # (nx, ny, nz)
    h: float
    bc: Tuple[int, int, int]           # per axis: 0 periodic, 1 homogeneous Neumann
    rho: np.ndarray                    # (nz, ny, nx) fp64
    rhs: np.ndarray                    # (nz, ny, nx) fp64, mean-free
    nu1: int
    nu2: int
    rtol: float
    coarse_sweeps: int = 32
    seed: Optional[int] = None
    p_exact: Optional[np.ndarray] = None
    eigenvalue: Optional[float] = None
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def ncells(self) -> int:
        return self.n[0] * self.n[1] * self.n[2]


# --------------------------------------------------------------------------- #
# density: phases by 4^3 sub-sampling, arithmetic (volume-weighted) mixing
# --------------------------------------------------------------------------- #
def _mixed_density(n, h, rho_air, film_top, rho_film, sphere_c, sphere_r, rho_drop):
    """rho = sum_phase rho_phase * f_phase, f_phase = (#sample points in phase)/64.

    Sample points of cell (i,j,k): ((i + (s+1/2)/4) h, ...), s = 0..3 per axis
    (SURVEY R19).  A point inside the sphere is drop (drop wins over film, R18);
    else below ``film_top`` it is film; else air.  ``film_top = None`` = no film.
    """
    nx, ny, nz = n
    sub = (np.arange(4) + 0.5) / 4.0
    zs = (np.arange(nz)[:, None] + sub[None, :]) * h              # (nz, 4)
    filmz = (zs < film_top) if film_top is not None else np.zeros_like(zs, bool)

    n_film = 16 * filmz.sum(axis=1)                                # (nz,)
    f_film = (n_film / 64.0)[:, None, None]
    f_air = ((64 - n_film) / 64.0)[:, None, None]
    rho = np.empty((nz, ny, nx), dtype=np.float64)
    rho[...] = rho_film * f_film + rho_air * f_air if film_top is not None else rho_air

    if sphere_r is None:
        return rho
    cx, cy, cz = sphere_c
    lo = [max(0, int(math.floor((c - sphere_r) / h)) - 1) for c in (cx, cy, cz)]
    hi = [min(m, int(math.ceil((c + sphere_r) / h)) + 1) for c, m in zip((cx, cy, cz), (nx, ny, nz))]
    for c, m in zip((cx, cy, cz), (nx, ny, nz)):
        assert c - sphere_r > 0.0 and c + sphere_r < m * h, "sphere must not cross the box boundary"
    xs = ((np.arange(lo[0], hi[0])[:, None] + sub[None, :]) * h).reshape(-1)
    ys = ((np.arange(lo[1], hi[1])[:, None] + sub[None, :]) * h).reshape(-1)
    dx2 = (xs - cx) ** 2
    dy2 = (ys - cy) ** 2
    bx, by = hi[0] - lo[0], hi[1] - lo[1]
    r2 = sphere_r * sphere_r
    chunk = 8
    for k0 in range(lo[2], hi[2], chunk):
        k1 = min(hi[2], k0 + chunk)
        ck = k1 - k0
        zz = zs[k0:k1].reshape(-1)                                  # (ck*4,)
        inside = ((zz - cz) ** 2)[:, None, None] + dy2[None, :, None] + dx2[None, None, :] < r2
        # per z-sub-layer count of the 16 (y,x) sub-samples inside the sphere
        layer = inside.reshape(ck, 4, by, 4, bx, 4).sum(axis=(3, 5))      # (ck,4,by,bx)
        n_drop = layer.sum(axis=1)
        n_filmc = (filmz[k0:k1][:, :, None, None] * (16 - layer)).sum(axis=1)
        n_airc = 64 - n_drop - n_filmc
        rho[k0:k1, lo[1]:hi[1], lo[0]:hi[0]] = (
            rho_drop * (n_drop / 64.0) + rho_film * (n_filmc / 64.0) + rho_air * (n_airc / 64.0)
        )
    return rho


def _remove_mean(f: np.ndarray) -> np.ndarray:
    mean = float(np.sum(f, dtype=np.longdouble) / np.longdouble(f.size))
    f -= mean
    return f


# --------------------------------------------------------------------------- #
# right-hand sides
# --------------------------------------------------------------------------- #
def _rhs_noise(n, seed):
    nx, ny, nz = n
    u = splitmix64_uniform(seed, nx * ny * nz)
    f = (-1.0 + 2.0 * u).reshape(nz, ny, nx)
    return _remove_mean(f)


def _rhs_velocity_divergence(n, h, seed, nmodes=16):
    """f = (Dx u + Dy v + Dz w)/h of a 16-mode staggered velocity field, dt = 1.

    u on x-faces, v on y-faces, w on z-faces (w = 0 on both z walls), so the
    discrete compatibility sum(f) = 0 holds by telescoping.
    Terms are accumulated in a fixed order with elementwise numpy ops only
    (no BLAS), so the field is reproducible.
    """
    nx, ny, nz = n
    st = _Stream(seed)
    xi_f = np.arange(nx) * h
    xi_c = (np.arange(nx) + 0.5) * h
    yj_f = np.arange(ny) * h
    yj_c = (np.arange(ny) + 0.5) * h
    zk_c = (np.arange(nz) + 0.5) * h
    planes, zvecs = [], []
    two_pi = 2.0 * math.pi
    for _ in range(nmodes):
        kx = st.integer(-4, 4)
        ky = st.integer(-4, 4)
        kz = st.integer(1, 4)
        phi = two_pi * float(st.uniform()[0])
        ax = st.real(-1.0, 1.0)
        ay = st.real(-1.0, 1.0)
        az = st.real(-1.0, 1.0)
        ux = np.cos(two_pi * (kx * xi_f[None, :] + ky * yj_c[:, None]) + phi)   # x-faces
        vy = np.cos(two_pi * (kx * xi_c[None, :] + ky * yj_f[:, None]) + phi)   # y-faces
        wc = np.cos(two_pi * (kx * xi_c[None, :] + ky * yj_c[:, None]) + phi)   # centres
        dxy = ax * (np.roll(ux, -1, axis=1) - ux) + ay * (np.roll(vy, -1, axis=0) - vy)
        cz = np.cos(math.pi * kz * zk_c)
        sz = np.sin(math.pi * kz * np.arange(nz + 1) * h)
        sz[0] = 0.0
        sz[nz] = 0.0
        planes.append((dxy, az * wc))
        zvecs.append((cz, sz[1:] - sz[:-1]))
    f = np.zeros((nz, ny, nx), dtype=np.float64)
    chunk = 8
    for k0 in range(0, nz, chunk):
        k1 = min(nz, k0 + chunk)
        blk = f[k0:k1]
        for (dxy, wz), (cz, dsz) in zip(planes, zvecs):
            blk += dxy[None, :, :] * cz[k0:k1, None, None]
            blk += wz[None, :, :] * dsz[k0:k1, None, None]
    f *= 1.0 / h
    return _remove_mean(f)


def velocity_field(n, h, seed, nmodes=16):
    """The staggered velocity behind _rhs_velocity_divergence, materialised: u on the minus
    x-faces, v on the minus y-faces, w on the minus z-faces of every cell (w = 0 on the bottom
    wall k = 0, which is also the top wall of the wrapped array).  Same seed stream, same modes;
    input for the projection steps (mg_project_rhs with dt = 1 reproduces the workload's rhs up
    to rounding and the removed mean).  Returns (u, v, w), each (nz, ny, nx) fp64."""
    nx, ny, nz = n
    st = _Stream(seed)
    xi_f = np.arange(nx) * h
    xi_c = (np.arange(nx) + 0.5) * h
    yj_f = np.arange(ny) * h
    yj_c = (np.arange(ny) + 0.5) * h
    zk_c = (np.arange(nz) + 0.5) * h
    two_pi = 2.0 * math.pi
    u = np.zeros((nz, ny, nx), dtype=np.float64)
    v = np.zeros_like(u)
    w = np.zeros_like(u)
    chunk = 8
    for _ in range(nmodes):
        kx = st.integer(-4, 4)
        ky = st.integer(-4, 4)
        kz = st.integer(1, 4)
        phi = two_pi * float(st.uniform()[0])
        ax = st.real(-1.0, 1.0)
        ay = st.real(-1.0, 1.0)
        az = st.real(-1.0, 1.0)
        ux = ax * np.cos(two_pi * (kx * xi_f[None, :] + ky * yj_c[:, None]) + phi)
        vy = ay * np.cos(two_pi * (kx * xi_c[None, :] + ky * yj_f[:, None]) + phi)
        wc = az * np.cos(two_pi * (kx * xi_c[None, :] + ky * yj_c[:, None]) + phi)
        cz = np.cos(math.pi * kz * zk_c)
        sz = np.sin(math.pi * kz * np.arange(nz) * h)      # minus z-face of plane k is at z = k h
        sz[0] = 0.0
        for k0 in range(0, nz, chunk):
            k1 = min(nz, k0 + chunk)
            u[k0:k1] += ux[None, :, :] * cz[k0:k1, None, None]
            v[k0:k1] += vy[None, :, :] * cz[k0:k1, None, None]
            w[k0:k1] += wc[None, :, :] * sz[k0:k1, None, None]
    return u, v, w


# --------------------------------------------------------------------------- #
# the five configs
# --------------------------------------------------------------------------- #
CONFIGS = {
    1: dict(n=32, bc=(0, 0, 0), nu=(2, 2), rtol=1e-10, seed=None,
            what="periodic cube, rho=1, rhs = lambda * sin(2pi x)sin(2pi y)sin(2pi z)"),
    2: dict(n=128, bc=(0, 0, 0), nu=(2, 2), rtol=1e-8, seed=1002,
            what="periodic cube, centred sphere r=0.25 rho 998 in / 1.2 out, noise rhs"),
    3: dict(n=256, bc=(0, 0, 1), nu=(3, 3), rtol=1e-8, seed=1003,
            what="drop-film box: film z<0.10 rho 935, drop r=0.1 at z=0.15 rho 998, air 1.2"),
    4: dict(n=512, bc=(0, 0, 1), nu=(3, 3), rtol=1e-8, seed=1004,
            what="as config 3 at 512^3 (the paper's per-device load, PAPER.md:196,218)"),
    5: dict(n=1024, bc=(0, 0, 1), nu=(3, 3), rtol=1e-8, seed=1005,
            what="drop-film box: film z<0.05, drop r=0.05 at z=0.10, 998/935/1.2"),
}


def make_workload(config: int, n: Optional[int] = None) -> Workload:
    """Build config `config` (1..5).  `n` overrides the cells per axis (scaled twin
    of the same recipe, used by the parity tests at sizes the oracle finishes fast)."""
    c = CONFIGS[config]
    nn = int(n if n is not None else c["n"])
    shape = (nn, nn, nn)
    h = 1.0 / nn
    nu1, nu2 = c["nu"]
    name = f"config{config}_{nn}"
    if config == 1:
        xc = (np.arange(nn) + 0.5) * h
        s = np.sin(2.0 * math.pi * xc)
        p_exact = s[:, None, None] * s[None, :, None] * s[None, None, :]
        lam = -(12.0 / (h * h)) * math.sin(math.pi / nn) ** 2
        rho = np.ones((nn, nn, nn), dtype=np.float64)
        rhs = lam * p_exact
        return Workload(name, shape, h, c["bc"], rho, rhs, nu1, nu2, c["rtol"],
                        p_exact=p_exact, eigenvalue=lam, note=c["what"])
    if config == 2:
        rho = _mixed_density(shape, h, 1.2, None, 0.0, (0.5, 0.5, 0.5), 0.25, 998.0)
        rhs = _rhs_noise(shape, c["seed"])
    elif config in (3, 4):
        rho = _mixed_density(shape, h, 1.2, 0.10, 935.0, (0.5, 0.5, 0.15), 0.10, 998.0)
        rhs = _rhs_velocity_divergence(shape, h, c["seed"])
    elif config == 5:
        rho = _mixed_density(shape, h, 1.2, 0.05, 935.0, (0.5, 0.5, 0.10), 0.05, 998.0)
        rhs = _rhs_velocity_divergence(shape, h, c["seed"])
    else:
        raise KeyError(config)
    return Workload(name, shape, h, c["bc"], rho, rhs, nu1, nu2, c["rtol"],
                    seed=c["seed"], note=c["what"])


def sequence_density(config: int, n: Optional[int], step: int, nsteps: int) -> np.ndarray:
    """Density of time step `step` (0 .. nsteps-1) of a drop falling onto the film (the paper's
    subject): the geometry of configs 3-5 with the drop
    centre starting 0.8 radii above its config position and ending exactly there, in equal
    steps.  Same sub-sampling and mixing as the configs (R19); seeded by nothing (closed form)."""
    assert config in (3, 4, 5) and 0 <= step < nsteps
    c = CONFIGS[config]
    nn = int(n if n is not None else c["n"])
    film, r, cz = (0.10, 0.10, 0.15) if config in (3, 4) else (0.05, 0.05, 0.10)
    lift = 0.8 * r * (1.0 - step / max(1, nsteps - 1))
    return _mixed_density((nn, nn, nn), 1.0 / nn, 1.2, film, 935.0, (0.5, 0.5, cz + lift), r, 998.0)
