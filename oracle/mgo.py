"""ctypes front end of the CPU oracle (libmgo.so).  TEST INFRASTRUCTURE ONLY.

May be imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` legs, never by the product package.  It imports nothing from
``paper_2605_30082_b200``.  See oracle/mgo.h for what is computed and the citations.
"""
from __future__ import annotations

import ctypes as C
import hashlib
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = [_HERE / "mgo.c", _HERE / "mgo.h"]

OK, NOT_CONVERGED, EINVAL, ENOMEM, EINCOMPATIBLE, EDIVERGED = 0, 1, -1, -2, -4, -5


def _cpu_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("flags"):
                    return " fma" in line
    except OSError:
        pass
    return False


def build(force: bool = False) -> Path:
    """Compile mgo.c -> oracle/_build/libmgo-<tag>.so (tag = source + flag hash)."""
    flags = ["-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-fopenmp"]
    if _cpu_has_fma():
        flags.append("-mfma")   # fma() -> one hardware instruction; same rounding as libm's
    hsh = hashlib.sha1()
    for p in _SRC:
        hsh.update(p.read_bytes())
    hsh.update(" ".join(flags).encode())
    out = _HERE / "_build" / f"libmgo-{hsh.hexdigest()[:12]}.so"
    if out.exists() and not force:
        return out
    out.parent.mkdir(exist_ok=True)
    tmp = out.with_suffix(f".tmp{os.getpid()}")
    cmd = ["gcc", *flags, "-o", str(tmp), str(_SRC[0]), "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    os.replace(tmp, out)
    return out


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        vp = C.c_void_p
        L.mgo_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, ip, C.POINTER(vp)]
        L.mgo_create6.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, ip, C.POINTER(vp)]
        L.mgo_destroy.argtypes = [vp]
        L.mgo_get_walls.argtypes = [vp, C.c_int, dp, dp, dp]
        L.mgo_destroy.restype = None
        L.mgo_set_cycle.argtypes = [vp, C.c_int, C.c_int, C.c_int]
        L.mgo_set_cycle_type.argtypes = [vp, C.c_int]
        L.mgo_set_density.argtypes = [vp, dp]
        L.mgo_vcycle.argtypes = [vp, dp, dp]
        L.mgo_residual.argtypes = [vp, dp, dp, dp, dp]
        L.mgo_solve.argtypes = [vp, dp, dp, C.c_double, C.c_int, ip, dp, dp]
        L.mgo_num_levels.argtypes = [vp]
        L.mgo_level_dims.argtypes = [vp, C.c_int, ip, dp]
        L.mgo_get_faces.argtypes = [vp, C.c_int, dp, dp, dp]
        L.mgo_apply.argtypes = [vp, C.c_int, dp, dp]
        L.mgo_smooth_half.argtypes = [vp, C.c_int, C.c_int, dp, dp]
        L.mgo_residual_level.argtypes = [vp, C.c_int, dp, dp, dp]
        L.mgo_restrict.argtypes = [vp, C.c_int, dp, dp]
        L.mgo_prolong_add.argtypes = [vp, C.c_int, dp, dp]
        L.mgo_solve_pcg.argtypes = [vp, dp, dp, C.c_double, C.c_int, ip, dp, dp]
        L.mgo_precondition.argtypes = [vp, dp, dp]
        L.mgo_restrict_adj.argtypes = [vp, C.c_int, dp, dp]
        L.mgo_project_rhs.argtypes = [vp, dp, dp, dp, C.c_double, dp]
        L.mgo_project_correct.argtypes = [vp, dp, C.c_double, dp, dp, dp]
        L.mgo_threads.restype = C.c_int
        L.mgo_set_threads.argtypes = [C.c_int]
        L.mgo_set_threads.restype = None
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__(f"mgo error {code}")
        self.code = code


def _chk(code, allowed=(OK,)):
    if code not in allowed:
        raise OracleError(code)
    return code


class Oracle:
    """Host-array multigrid oracle.  Arrays are numpy fp64 of shape (nz, ny, nx)."""

    def __init__(self, n, h, bc, nu1=2, nu2=2, coarse_sweeps=32):
        nx, ny, nz = (n, n, n) if np.isscalar(n) else n
        self.n = (int(nx), int(ny), int(nz))
        self.h = float(h)
        self.bc = tuple(int(b) for b in bc)
        self._h = C.c_void_p()
        if len(self.bc) == 6:           # R24: one type per side (x-, x+, y-, y+, z-, z+); 2 = Dirichlet
            bca = (C.c_int * 6)(*self.bc)
            _chk(lib().mgo_create6(self.n[0], self.n[1], self.n[2], self.h, bca, C.byref(self._h)))
        else:
            bca = (C.c_int * 3)(*self.bc)
            _chk(lib().mgo_create(self.n[0], self.n[1], self.n[2], self.h, bca, C.byref(self._h)))
        _chk(lib().mgo_set_cycle(self._h, nu1, nu2, coarse_sweeps))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().mgo_destroy(self._h)
            self._h = None

    __del__ = close

    # ---- geometry
    @property
    def shape(self):
        return (self.n[2], self.n[1], self.n[0])

    @property
    def num_levels(self):
        return lib().mgo_num_levels(self._h)

    def level_dims(self, level):
        d = (C.c_int * 3)()
        hl = C.c_double()
        _chk(lib().mgo_level_dims(self._h, level, d, C.byref(hl)))
        return (d[0], d[1], d[2]), hl.value

    def level_shape(self, level):
        (nx, ny, nz), _ = self.level_dims(level)
        return (nz, ny, nx)

    def _arr(self, a, level=0):
        a = np.ascontiguousarray(a, dtype=np.float64)
        assert a.shape == self.level_shape(level), (a.shape, self.level_shape(level))
        return a

    # ---- the calls of the boundary
    def set_cycle(self, nu1, nu2, coarse_sweeps=32):
        _chk(lib().mgo_set_cycle(self._h, nu1, nu2, coarse_sweeps))

    def set_cycle_type(self, type):
        """0 = V (default), 1 = F, 2 = W (R23)."""
        _chk(lib().mgo_set_cycle_type(self._h, int(type)))

    def set_density(self, rho):
        _chk(lib().mgo_set_density(self._h, _dp(self._arr(rho))))

    def vcycle(self, rhs, p):
        """One V-cycle in place on p (p must be a C-contiguous fp64 array)."""
        assert p.flags["C_CONTIGUOUS"] and p.dtype == np.float64 and p.shape == self.shape
        _chk(lib().mgo_vcycle(self._h, _dp(self._arr(rhs)), _dp(p)))
        return p

    def residual(self, rhs, p, want_field=False):
        nrm = C.c_double()
        r = np.empty(self.shape) if want_field else None
        _chk(lib().mgo_residual(self._h, _dp(self._arr(rhs)), _dp(self._arr(p)),
                                _dp(r) if want_field else None, C.byref(nrm)))
        return (nrm.value, r) if want_field else nrm.value

    def solve(self, rhs, p, rtol, max_cycles):
        """Returns (status, cycles, relres, hist[0..cycles]); p updated in place."""
        assert p.flags["C_CONTIGUOUS"] and p.dtype == np.float64 and p.shape == self.shape
        cyc = C.c_int()
        rel = C.c_double()
        hist = np.zeros(max_cycles + 1)
        st = lib().mgo_solve(self._h, _dp(self._arr(rhs)), _dp(p), rtol, max_cycles,
                             C.byref(cyc), C.byref(rel), _dp(hist))
        if st < 0:
            raise OracleError(st)
        return st, cyc.value, rel.value, hist[: cyc.value + 1].copy()

    # ---- MG-preconditioned CG
    def solve_pcg(self, rhs, p, rtol, max_iter):
        """Returns (status, iterations, relres, hist[0..iterations]); p updated in place."""
        assert p.flags["C_CONTIGUOUS"] and p.dtype == np.float64 and p.shape == self.shape
        it = C.c_int()
        rel = C.c_double()
        hist = np.zeros(max_iter + 1)
        st = lib().mgo_solve_pcg(self._h, _dp(self._arr(rhs)), _dp(p), rtol, max_iter,
                                 C.byref(it), C.byref(rel), _dp(hist))
        if st < 0:
            raise OracleError(st)
        return st, it.value, rel.value, hist[: it.value + 1].copy()

    def precondition(self, r):
        z = np.empty(self.shape)
        _chk(lib().mgo_precondition(self._h, _dp(self._arr(r)), _dp(z)))
        return z

    def walls(self, level=0):
        """Plus-wall face coefficients (wx[nz, ny], wy[nz, nx], wz[ny, nx]) of a level."""
        nz, ny, nx = self.level_shape(level)
        wx, wy, wz = np.empty((nz, ny)), np.empty((nz, nx)), np.empty((ny, nx))
        _chk(lib().mgo_get_walls(self._h, level, _dp(wx), _dp(wy), _dp(wz)))
        return wx, wy, wz

    def restrict_adj(self, r, level=0):
        fc = np.empty(self.level_shape(level + 1))
        _chk(lib().mgo_restrict_adj(self._h, level, _dp(self._arr(r, level)), _dp(fc)))
        return fc

    # ---- projection steps
    def project_rhs(self, u, v, w, dt):
        f = np.empty(self.shape)
        _chk(lib().mgo_project_rhs(self._h, _dp(self._arr(u)), _dp(self._arr(v)), _dp(self._arr(w)),
                                   float(dt), _dp(f)))
        return f

    def project_correct(self, p, dt, u, v, w):
        for a in (u, v, w):
            assert a.flags["C_CONTIGUOUS"] and a.dtype == np.float64 and a.shape == self.shape
        _chk(lib().mgo_project_correct(self._h, _dp(self._arr(p)), float(dt), _dp(u), _dp(v), _dp(w)))
        return u, v, w

    # ---- step level
    def faces(self, level):
        shp = self.level_shape(level)
        bx, by, bz = np.empty(shp), np.empty(shp), np.empty(shp)
        _chk(lib().mgo_get_faces(self._h, level, _dp(bx), _dp(by), _dp(bz)))
        return bx, by, bz

    def apply(self, p, level=0):
        out = np.empty(self.level_shape(level))
        _chk(lib().mgo_apply(self._h, level, _dp(self._arr(p, level)), _dp(out)))
        return out

    def smooth_half(self, colour, f, p, level=0):
        assert p.flags["C_CONTIGUOUS"] and p.dtype == np.float64
        _chk(lib().mgo_smooth_half(self._h, level, colour, _dp(self._arr(f, level)), _dp(p)))
        return p

    def sweep(self, f, p, level=0):
        self.smooth_half(0, f, p, level)
        self.smooth_half(1, f, p, level)
        return p

    def residual_level(self, f, p, level=0):
        r = np.empty(self.level_shape(level))
        _chk(lib().mgo_residual_level(self._h, level, _dp(self._arr(f, level)),
                                      _dp(self._arr(p, level)), _dp(r)))
        return r

    def restrict(self, r, level=0):
        fc = np.empty(self.level_shape(level + 1))
        _chk(lib().mgo_restrict(self._h, level, _dp(self._arr(r, level)), _dp(fc)))
        return fc

    def prolong_add(self, e, p, level=0):
        assert p.flags["C_CONTIGUOUS"] and p.dtype == np.float64
        _chk(lib().mgo_prolong_add(self._h, level, _dp(self._arr(e, level + 1)), _dp(p)))
        return p


def threads() -> int:
    return lib().mgo_threads()


def set_threads(n: int) -> None:
    lib().mgo_set_threads(n)
