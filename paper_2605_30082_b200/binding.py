"""ctypes binding of libmg: argument marshalling only (include/mg.h has the semantics).

Tensors are torch CUDA fp64 tensors of shape (nz, ny, nx) (x fastest); torch supplies
device memory and the stream, nothing else.  Every ``mg_*`` entry point of the header
is reachable as ``lib().mg_*``; :class:`Multigrid` wraps a handle.
"""
from __future__ import annotations

import ctypes as C

from . import _build

MG_OK, MG_NOT_CONVERGED = 0, 1
MG_EINVAL, MG_ENOMEM, MG_ECUDA, MG_EINCOMPATIBLE, MG_EDIVERGED = -1, -2, -3, -4, -5
MG_BC_PERIODIC, MG_BC_NEUMANN = 0, 1
MG_OPT_KERNELS, MG_OPT_GRAPH, MG_OPT_COARSE_CTA, MG_OPT_SWEEP_FUSE, MG_OPT_TAIL_FUSION = 1, 2, 3, 4, 5
MG_OPT_FACE_STREAM_LOG2 = 6
MG_OPT_PROLONG_FUSE = 7
MG_CYCLE_V, MG_CYCLE_F, MG_CYCLE_W = 0, 1, 2
MG_STAT_KERNEL_LAUNCHES, MG_STAT_WORKSPACE_BYTES, MG_STAT_LAUNCHES_PER_VCYCLE = 1, 2, 3
MG_STAT_EXTRA_DEVICE_BYTES = 4

_vp, _dp, _ip = C.c_void_p, C.c_void_p, C.POINTER(C.c_int)   # device pointers travel as integers
_hp = C.POINTER(C.c_double)

SIGNATURES = {
    "mg_workspace_bytes": (C.c_size_t, [C.c_int, C.c_int, C.c_int]),
    "mg_create": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_double, _ip, C.POINTER(_vp)]),
    "mg_create_in": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_double, _ip, _vp, C.c_size_t, C.POINTER(_vp)]),
    "mg_create6": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_double, _ip, C.POINTER(_vp)]),
    "mg_create6_in": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_double, _ip, _vp, C.c_size_t, C.POINTER(_vp)]),
    "mg_destroy": (None, [_vp]),
    "mg_set_stream": (C.c_int, [_vp, _vp]),
    "mg_set_cycle_type": (C.c_int, [_vp, C.c_int]),
    "mg_set_cycle": (C.c_int, [_vp, C.c_int, C.c_int, C.c_int]),
    "mg_set_option": (C.c_int, [_vp, C.c_int, C.c_int]),
    "mg_get_stat": (C.c_int, [_vp, C.c_int, C.POINTER(C.c_longlong)]),
    "mg_set_density": (C.c_int, [_vp, _dp]),
    "mg_vcycle": (C.c_int, [_vp, _dp, _dp]),
    "mg_residual": (C.c_int, [_vp, _dp, _dp, _dp, _hp]),
    "mg_solve": (C.c_int, [_vp, _dp, _dp, C.c_double, C.c_int, _ip, _hp, _hp]),
    "mg_solve_pcg": (C.c_int, [_vp, _dp, _dp, C.c_double, C.c_int, _ip, _hp, _hp]),
    "mg_precondition": (C.c_int, [_vp, _dp, _dp]),
    "mg_level_prolong_smooth": (C.c_int, [_vp, C.c_int, C.c_int, _dp, _dp, _dp]),
    "mg_level_restrict_adj": (C.c_int, [_vp, C.c_int, _dp, _dp]),
    "mg_solve_host": (C.c_int, [_vp, _vp, _vp, _vp, C.c_double, C.c_int, _ip, _hp, _hp]),
    "mg_project_rhs": (C.c_int, [_vp, _dp, _dp, _dp, C.c_double, _dp]),
    "mg_project_correct": (C.c_int, [_vp, _dp, C.c_double, _dp, _dp, _dp]),
    "mg_project": (C.c_int, [_vp, _dp, _dp, _dp, C.c_double, _dp, _dp, C.c_double, C.c_int, _ip, _hp]),
    "mg_residual_norm_static": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_double, _ip, _dp, _dp, _dp, _dp, _vp]),
    "mg_test_rcp": (C.c_int, [_dp, C.c_size_t, _dp, _dp, _vp]),
    "mg_strerror": (C.c_char_p, [C.c_int]),
    "mg_last_cuda_error": (C.c_char_p, []),
    "mg_num_levels": (C.c_int, [_vp]),
    "mg_level_dims": (C.c_int, [_vp, C.c_int, _ip, _hp]),
    "mg_level_faces": (C.c_int, [_vp, C.c_int, _dp, _dp, _dp]),
    "mg_level_smooth_half": (C.c_int, [_vp, C.c_int, C.c_int, _dp, _dp]),
    "mg_level_smooth": (C.c_int, [_vp, C.c_int, C.c_int, _dp, _dp]),
    "mg_level_residual": (C.c_int, [_vp, C.c_int, _dp, _dp, _dp]),
    "mg_level_residual_restrict": (C.c_int, [_vp, C.c_int, _dp, _dp, _dp]),
    "mg_level_prolong_add": (C.c_int, [_vp, C.c_int, _dp, _dp]),
    "mg_level_smooth_restrict": (C.c_int, [_vp, C.c_int, C.c_int, _dp, _dp, _dp]),
    "mg_level_smooth_norm": (C.c_int, [_vp, C.c_int, _dp, _dp, _hp]),
}

_lib = None


def lib():
    """The loaded libmg (built on demand).  Raises if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(str(path))
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)          # AttributeError = header/library mismatch
            fn.restype, fn.argtypes = res, args
        L._path = str(path)
        _lib = L
    return _lib


class MgError(RuntimeError):
    def __init__(self, code, detail=None):
        msg = lib().mg_strerror(code).decode()
        if code == MG_ECUDA:
            msg += ": " + lib().mg_last_cuda_error().decode()
        elif detail:
            msg += ": " + detail
        super().__init__(f"libmg error {code}: {msg}")
        self.code = code


def _chk(code, ok=(MG_OK,)):
    if code not in ok:
        raise MgError(code)
    return code


def workspace_bytes(nx, ny, nz):
    return lib().mg_workspace_bytes(nx, ny, nz)


def _ptr(t, shape=None):
    import torch

    if t is None:
        return None
    assert isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous(), \
        "expected a contiguous CUDA float64 tensor"
    if shape is not None:
        assert tuple(t.shape) == tuple(shape), (tuple(t.shape), tuple(shape))
    assert t.data_ptr() % 16 == 0, "device arrays must be 16-byte aligned (include/mg.h)"
    return t.data_ptr()


MG_STATIC_MAX_CELLS = 1 << 27


def residual_norm_static(n, h, bc, rho, rhs, p, out, stream=None):
    """``out[0] = ||rhs - A p||_2`` through mg_residual_norm_static: no handle, and the library
    allocates nothing (its scratch is a fixed array inside libmg, good for up to
    MG_STATIC_MAX_CELLS cells; larger grids raise MgError(MG_EINVAL)).  Meant for callers that
    cannot allocate device memory where they need the norm: a solver whose memory all sits in
    its own pool, or a monitor inside a running time loop that must not trigger cudaMalloc's
    device-wide synchronisation.  ``out`` is the caller's own 1-element CUDA float64 tensor;
    the call is asynchronous on ``stream`` (default: torch's current stream).  Calls share the
    scratch array, so do not let two of them overlap on one GPU."""
    import torch

    nx, ny, nz = (n, n, n) if isinstance(n, int) else n
    shape = (int(nz), int(ny), int(nx))
    assert isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64 and out.numel() == 1
    bca = (C.c_int * 3)(*[int(b) for b in bc])
    with torch.cuda.device(out.device):
        st = stream if stream is not None else torch.cuda.current_stream(out.device)
        code = lib().mg_residual_norm_static(int(nx), int(ny), int(nz), float(h), bca, _ptr(rho, shape),
                                             _ptr(rhs, shape), _ptr(p, shape), out.data_ptr(), st.cuda_stream)
    if code == MG_EINVAL and lib().mg_last_cuda_error():
        raise MgError(code, lib().mg_last_cuda_error().decode())
    _chk(code)
    return out


class Multigrid:
    """Handle to one solver.  n = (nx, ny, nz) or a single int; bc per axis (0 periodic,
    1 Neumann), or six entries, one per side x-, x+, y-, y+, z-, z+ (2 = Dirichlet: mg_create6).
    Device storage comes from a torch tensor (mg_create_in); the stream is
    torch's current stream at construction unless ``stream`` is given."""

    def __init__(self, n, h, bc, nu1=2, nu2=2, coarse_sweeps=32, stream=None, device="cuda:0",
                 own_workspace=False):
        import torch

        nx, ny, nz = (n, n, n) if isinstance(n, int) else n
        self.n = (int(nx), int(ny), int(nz))
        self.shape = (self.n[2], self.n[1], self.n[0])
        self.device = torch.device(device)
        L = lib()
        self._h = _vp()
        need = L.mg_workspace_bytes(*self.n)
        if need == 0:
            raise MgError(MG_EINVAL)
        with torch.cuda.device(self.device):
            bc = [int(b) for b in bc]
            bca = (C.c_int * len(bc))(*bc)
            create, create_in = (L.mg_create6, L.mg_create6_in) if len(bc) == 6 else (L.mg_create, L.mg_create_in)
            if own_workspace:           # mg_create: the library allocates with cudaMalloc
                self._ws = None
                _chk(create(*self.n, float(h), bca, C.byref(self._h)))
            else:
                self._ws = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
                base = (self._ws.data_ptr() + 255) // 256 * 256
                _chk(create_in(*self.n, float(h), bca, base, need, C.byref(self._h)))
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            _chk(L.mg_set_stream(self._h, self.stream.cuda_stream))
        _chk(L.mg_set_cycle(self._h, nu1, nu2, coarse_sweeps))

    def close(self):
        if getattr(self, "_h", None):
            lib().mg_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- configuration
    def set_cycle(self, nu1, nu2, coarse_sweeps=32):
        _chk(lib().mg_set_cycle(self._h, nu1, nu2, coarse_sweeps))

    def set_cycle_type(self, type):
        """0 = V (default), 1 = F, 2 = W."""
        _chk(lib().mg_set_cycle_type(self._h, int(type)))

    def set_option(self, key, value):
        _chk(lib().mg_set_option(self._h, key, value))

    def stat(self, key):
        v = C.c_longlong()
        _chk(lib().mg_get_stat(self._h, key, C.byref(v)))
        return v.value

    @property
    def num_levels(self):
        return lib().mg_num_levels(self._h)

    def level_dims(self, level):
        d = (C.c_int * 3)()
        h = C.c_double()
        _chk(lib().mg_level_dims(self._h, level, d, C.byref(h)))
        return (d[0], d[1], d[2]), h.value

    def level_shape(self, level):
        (nx, ny, nz), _ = self.level_dims(level)
        return (nz, ny, nx)

    # ---- the calls of the boundary
    def set_density(self, rho):
        _chk(lib().mg_set_density(self._h, _ptr(rho, self.shape)))

    def vcycle(self, rhs, p):
        _chk(lib().mg_vcycle(self._h, _ptr(rhs, self.shape), _ptr(p, self.shape)))
        return p

    def residual(self, rhs, p, r=None):
        nrm = C.c_double()
        _chk(lib().mg_residual(self._h, _ptr(rhs, self.shape), _ptr(p, self.shape),
                               _ptr(r, self.shape), C.byref(nrm)))
        return nrm.value

    def residual_field(self, rhs, p, r):
        """r = rhs - A p only (no norm, asynchronous)."""
        _chk(lib().mg_residual(self._h, _ptr(rhs, self.shape), _ptr(p, self.shape), _ptr(r, self.shape), None))
        return r

    def solve(self, rhs, p, rtol, max_cycles):
        """Returns (status, cycles, relres, hist[0..cycles]); p updated in place."""
        cyc, rel = C.c_int(), C.c_double()
        hist = (C.c_double * (max_cycles + 1))()
        st = lib().mg_solve(self._h, _ptr(rhs, self.shape), _ptr(p, self.shape), float(rtol),
                            int(max_cycles), C.byref(cyc), C.byref(rel), hist)
        if st < 0:
            raise MgError(st)
        return st, cyc.value, rel.value, list(hist[: cyc.value + 1])

    def solve_pcg(self, rhs, p, rtol, max_iter):
        """MG-preconditioned CG: returns (status, iterations, relres, hist[0..iterations])."""
        it, rel = C.c_int(), C.c_double()
        hist = (C.c_double * (max_iter + 1))()
        st = lib().mg_solve_pcg(self._h, _ptr(rhs, self.shape), _ptr(p, self.shape), float(rtol),
                                int(max_iter), C.byref(it), C.byref(rel), hist)
        if st < 0:
            raise MgError(st)
        return st, it.value, rel.value, list(hist[: it.value + 1])

    def precondition(self, r, z):
        _chk(lib().mg_precondition(self._h, _ptr(r, self.shape), _ptr(z, self.shape)))
        return z

    def level_restrict_adj(self, level, r):
        import torch

        fc = torch.empty(self.level_shape(level + 1), dtype=torch.float64, device=self.device)
        _chk(lib().mg_level_restrict_adj(self._h, level, _ptr(r, self.level_shape(level)), _ptr(fc)))
        return fc

    def solve_host(self, rho_host, rhs_host, p_host, rtol, max_cycles):
        """Host-buffer variant: CPU torch tensors (ideally pinned) of shape (nz,ny,nx)."""
        cyc, rel = C.c_int(), C.c_double()
        hist = (C.c_double * (max_cycles + 1))()
        for t in (rho_host, rhs_host, p_host):
            assert t is None or (not t.is_cuda and t.is_contiguous() and tuple(t.shape) == self.shape)
        st = lib().mg_solve_host(self._h, rho_host.data_ptr() if rho_host is not None else None,
                                 rhs_host.data_ptr(), p_host.data_ptr(), float(rtol), int(max_cycles),
                                 C.byref(cyc), C.byref(rel), hist)
        if st < 0:
            raise MgError(st)
        return st, cyc.value, rel.value, list(hist[: cyc.value + 1])

    # ---- projection steps either side of the solve
    def project_rhs(self, u, v, w, dt, f):
        _chk(lib().mg_project_rhs(self._h, _ptr(u, self.shape), _ptr(v, self.shape), _ptr(w, self.shape),
                                  float(dt), _ptr(f, self.shape)))
        return f

    def project_correct(self, p, dt, u, v, w):
        _chk(lib().mg_project_correct(self._h, _ptr(p, self.shape), float(dt), _ptr(u, self.shape),
                                      _ptr(v, self.shape), _ptr(w, self.shape)))

    def project(self, u, v, w, dt, p, rhs, rtol, max_cycles):
        """rhs -> solve -> correct; returns (status, cycles, relres)."""
        cyc, rel = C.c_int(), C.c_double()
        st = lib().mg_project(self._h, _ptr(u, self.shape), _ptr(v, self.shape), _ptr(w, self.shape), float(dt),
                              _ptr(p, self.shape), _ptr(rhs, self.shape), float(rtol), int(max_cycles),
                              C.byref(cyc), C.byref(rel))
        if st < 0:
            raise MgError(st)
        return st, cyc.value, rel.value

    # ---- single steps
    def level_faces(self, level):
        import torch

        shp = self.level_shape(level)
        out = [torch.empty(shp, dtype=torch.float64, device=self.device) for _ in range(3)]
        _chk(lib().mg_level_faces(self._h, level, *[_ptr(t) for t in out]))
        return out

    def level_smooth_half(self, level, colour, f, p):
        _chk(lib().mg_level_smooth_half(self._h, level, colour, _ptr(f, self.level_shape(level)),
                                        _ptr(p, self.level_shape(level))))
        return p

    def level_smooth(self, level, sweeps, f, p):
        _chk(lib().mg_level_smooth(self._h, level, sweeps, _ptr(f, self.level_shape(level)),
                                   _ptr(p, self.level_shape(level))))
        return p

    def level_residual(self, level, f, p):
        import torch

        r = torch.empty(self.level_shape(level), dtype=torch.float64, device=self.device)
        _chk(lib().mg_level_residual(self._h, level, _ptr(f, r.shape), _ptr(p, r.shape), _ptr(r)))
        return r

    def level_residual_restrict(self, level, f, p):
        import torch

        fc = torch.empty(self.level_shape(level + 1), dtype=torch.float64, device=self.device)
        shp = self.level_shape(level)
        _chk(lib().mg_level_residual_restrict(self._h, level, _ptr(f, shp), _ptr(p, shp), _ptr(fc)))
        return fc

    def level_smooth_restrict(self, level, sweeps, f, p):
        import torch

        fc = torch.empty(self.level_shape(level + 1), dtype=torch.float64, device=self.device)
        shp = self.level_shape(level)
        _chk(lib().mg_level_smooth_restrict(self._h, level, sweeps, _ptr(f, shp), _ptr(p, shp), _ptr(fc)))
        return fc

    def level_smooth_norm(self, sweeps, f, p):
        nrm = C.c_double()
        _chk(lib().mg_level_smooth_norm(self._h, sweeps, _ptr(f, self.shape), _ptr(p, self.shape), C.byref(nrm)))
        return nrm.value

    def level_prolong_smooth(self, level, sweeps, e, f, p):
        _chk(lib().mg_level_prolong_smooth(self._h, level, int(sweeps), _ptr(e, self.level_shape(level + 1)),
                                           _ptr(f, self.level_shape(level)), _ptr(p, self.level_shape(level))))
        return p

    def level_prolong_add(self, level, e, p):
        _chk(lib().mg_level_prolong_add(self._h, level, _ptr(e, self.level_shape(level + 1)),
                                        _ptr(p, self.level_shape(level))))
        return p
