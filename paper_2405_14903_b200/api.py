"""Thin ctypes binding of the C-ABI library (include/nf.h).  Argument marshalling only: every step of the hot
path runs in the CUDA kernels of csrc/.  torch is used for device memory and streams (PAPER.md:L145 exposes the
simulator to PyTorch the same way).  There is no CPU fallback: if libnf_b200.so is missing this module raises.

Function names follow include/nf.h one to one (`Grid.project` -> nf_project, ...)."""
import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnf_b200.so")

NF_OK, NF_NOT_CONVERGED = 0, 1
NF_ERR_INVALID, NF_ERR_ALLOC, NF_ERR_CUDA, NF_ERR_STATE = -1, -2, -3, -4
BC_CLOSED, BC_DIRICHLET = 0, 1

_c_float_p = ctypes.c_void_p  # raw device (or host) addresses
_c_host_float_p = ctypes.POINTER(ctypes.c_float)
_c_host_double_p = ctypes.POINTER(ctypes.c_double)
_SIGNATURES = {
    "nf_version": (ctypes.c_char_p, []),
    "nf_grid_create": (ctypes.c_int, [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_float,
                                      ctypes.POINTER(ctypes.c_void_p)]),
    "nf_grid_destroy": (None, [ctypes.c_void_p]),
    "nf_set_stream": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "nf_set_dt_rho": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_float]),
    "nf_set_domain_bc": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_float]),
    "nf_set_solver_options": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int]),
    "nf_set_coarse_sweeps": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_int]),
    "nf_get_sweeps": (ctypes.c_int, [ctypes.c_void_p] + [ctypes.POINTER(ctypes.c_int)] * 4),
    "nf_set_coarse_relaxation": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_float]),
    "nf_get_coarse_relaxation": (ctypes.c_float, [ctypes.c_void_p]),
    "nf_set_pressure_lo": (ctypes.c_int, [ctypes.c_void_p, _c_float_p]),
    "nf_set_solid": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 4),
    "nf_set_weights": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 3),
    "nf_get_weights": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 3),
    "nf_set_solid_velocity": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 3),
    "nf_solve": (ctypes.c_int, [ctypes.c_void_p, _c_float_p, _c_float_p, ctypes.c_float, ctypes.c_int]),
    "nf_project": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 4 + [ctypes.c_float, ctypes.c_int]),
    "nf_project_adjoint": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 14 + [ctypes.c_float, ctypes.c_int]),
    "nf_solve_batch": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_float,
                                      ctypes.c_int, ctypes.POINTER(ctypes.c_int)]),
    "nf_project_batch": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int] + [ctypes.c_void_p] * 4 +
                         [ctypes.c_float, ctypes.c_int, ctypes.POINTER(ctypes.c_int)]),
    "nf_project_adjoint_batch": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int] + [ctypes.c_void_p] * 14 +
                                 [ctypes.c_float, ctypes.c_int, ctypes.POINTER(ctypes.c_int)]),
    "nf_advect": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 3 + [ctypes.c_float]),
    "nf_max_speed": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 3 + [ctypes.POINTER(ctypes.c_float)]),
    "nf_viscosity": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 3 + [ctypes.c_float, ctypes.c_float]),
    "nf_advect_adjoint": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 6 + [ctypes.c_float]),
    "nf_weights_adjoint": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 4),
    "nf_geom_sdf": (ctypes.c_int, [ctypes.c_void_p, _c_host_float_p] + [ctypes.c_int] * 4 + [_c_float_p]),
    "nf_geom_sdf_adjoint": (ctypes.c_int, [ctypes.c_void_p, _c_host_float_p] + [ctypes.c_int] * 4 +
                            [_c_float_p, _c_host_double_p]),
    "nf_geom_csg": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int] + [_c_float_p] * 3),
    "nf_geom_csg_adjoint": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int] + [_c_float_p] * 5),
    "nf_geom_velocity": (ctypes.c_int, [ctypes.c_void_p, _c_host_float_p, _c_host_float_p] + [ctypes.c_int] * 3 +
                         [ctypes.c_float] + [_c_float_p] * 3),
    "nf_geom_velocity_adjoint": (ctypes.c_int, [ctypes.c_void_p, _c_host_float_p] + [ctypes.c_int] * 3 +
                                 [ctypes.c_float] + [_c_float_p] * 3 + [_c_host_double_p]),
    "nf_apply_A": (ctypes.c_int, [ctypes.c_void_p, _c_float_p, _c_float_p]),
    "nf_vcycle": (ctypes.c_int, [ctypes.c_void_p, _c_float_p, _c_float_p]),
    "nf_set_host_async": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int]),
    "nf_host_sync": (ctypes.c_int, [ctypes.c_void_p]),
    "nf_project_host": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 4 + [ctypes.c_float, ctypes.c_int]),
    "nf_project_adjoint_host": (ctypes.c_int, [ctypes.c_void_p] + [_c_float_p] * 7 + [ctypes.c_float, ctypes.c_int]),
    "nf_last_solve_info": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_int),
                                          ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_float)]),
    "nf_grid_info": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_int),
                                    ctypes.POINTER(ctypes.c_longlong), ctypes.POINTER(ctypes.c_int)]),
    "nf_grid_components": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int)]),
    "nf_profile_enable": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int]),
    "nf_profile_get": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_char_p),
                                      ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_longlong)]),
    "nf_launch_count": (ctypes.c_longlong, [ctypes.c_void_p]),
    "nf_last_error": (ctypes.c_char_p, [ctypes.c_void_p]),
    "nf_max_speed_static": (ctypes.c_int, [_c_float_p] * 3 + [ctypes.c_int] * 3 + [ctypes.c_void_p, _c_float_p]),
    "nf_static_last_error": (ctypes.c_char_p, []),
}
EXPORTED_SYMBOLS = tuple(_SIGNATURES)

_lib = None


def load_library(path=None):
    """dlopen libnf_b200.so and declare every signature of include/nf.h.  Raises if the library is missing."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise RuntimeError("%s not found: build it with `python -m paper_2405_14903_b200.build` "
                           "(there is no CPU fallback)" % path)
    lib = ctypes.CDLL(path)
    for name, (res, args) in _SIGNATURES.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


class NfError(RuntimeError):
    pass


class NfNotConvergedWarning(RuntimeWarning):
    """A solve hit maxit: the best iterate was written (NF_NOT_CONVERGED), the caller's tolerance was not met."""


def _bound(fn):
    """Hot-path methods run on the torch stream that is current when they are called (the handle is re-bound if it
    changed since the last call) and with the handle's device current, so that the library's kernels are ordered with
    the caller's torch ops on the same stream."""
    import functools

    @functools.wraps(fn)
    def wrapper(self, *a, **k):
        import torch
        if torch.cuda.current_device() != self.device.index:
            with torch.cuda.device(self.device):
                self._bind_stream()
                return fn(self, *a, **k)
        self._bind_stream()
        return fn(self, *a, **k)
    return wrapper


def _ptr(t):
    """Device (or host) address of a contiguous float32 torch tensor; None -> NULL."""
    if t is None:
        return None
    import torch
    if not isinstance(t, torch.Tensor):
        raise TypeError("expected a torch.Tensor or None")
    if t.dtype != torch.float32 or not t.is_contiguous():
        raise ValueError("arrays must be contiguous float32 tensors")
    return ctypes.c_void_p(t.data_ptr())


class Grid:
    """Owner of one nf_grid handle.  Tensors are passed by address; shapes follow include/nf.h:
    p (nz,ny,nx), u (nz,ny,nx+1), v (nz,ny+1,nx), w (nz+1,ny,nx), sdf (nz+1,ny+1,nx+1)."""

    def __init__(self, nx, ny, nz, dx, device=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2405_14903_b200 needs a CUDA device (there is no CPU fallback)")
        self.lib = load_library()
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self.nx, self.ny, self.nz, self.dx = int(nx), int(ny), int(nz), float(dx)
        h = ctypes.c_void_p()
        with torch.cuda.device(self.device):
            rc = self.lib.nf_grid_create(self.nx, self.ny, self.nz, self.dx, ctypes.byref(h))
        if rc != NF_OK:
            raise NfError("nf_grid_create failed with %d" % rc)
        self.h = h
        self._stream = None
        self.warn_not_converged = True
        self._bind_stream()

    # -- shapes -------------------------------------------------------------------------------------------
    @property
    def shape_p(self):
        return (self.nz, self.ny, self.nx)

    @property
    def shape_u(self):
        return (self.nz, self.ny, self.nx + 1)

    @property
    def shape_v(self):
        return (self.nz, self.ny + 1, self.nx)

    @property
    def shape_w(self):
        return (self.nz + 1, self.ny, self.nx)

    @property
    def shape_sdf(self):
        return (self.nz + 1, self.ny + 1, self.nx + 1)

    def _bind_stream(self):
        import torch
        s = torch.cuda.current_stream(self.device).cuda_stream
        if s != self._stream:
            self._check(self.lib.nf_set_stream(self.h, ctypes.c_void_p(s)), "nf_set_stream")
            self._stream = s

    def _check(self, rc, name, allow_not_converged=True):
        if rc == NF_NOT_CONVERGED and allow_not_converged and self.warn_not_converged:
            import warnings
            warnings.warn("%s: the solve stopped at maxit without reaching the tolerance (NF_NOT_CONVERGED); the "
                          "result is the best iterate" % name, NfNotConvergedWarning, stacklevel=3)
        if rc == NF_OK or (allow_not_converged and rc == NF_NOT_CONVERGED):
            return rc
        msg = self.lib.nf_last_error(self.h)
        raise NfError("%s failed with %d: %s" % (name, rc, msg.decode() if msg else ""))

    def _expect(self, t, shape, name, host=False):
        if t is None:
            return
        if tuple(t.shape) != tuple(shape):
            raise ValueError("%s has shape %s, expected %s" % (name, tuple(t.shape), tuple(shape)))
        if host and t.is_cuda:
            raise ValueError("%s must be a host tensor" % name)
        if not host and not t.is_cuda:
            raise ValueError("%s must be a CUDA tensor" % name)

    def close(self):
        if getattr(self, "h", None):
            self.lib.nf_grid_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- configuration ------------------------------------------------------------------------------------
    def set_stream(self, stream):
        """Bind the handle to `stream` now (every hot-path call re-binds to the torch stream current at that call)."""
        self._check(self.lib.nf_set_stream(self.h, ctypes.c_void_p(stream.cuda_stream)), "nf_set_stream")
        self._stream = stream.cuda_stream

    @_bound
    def set_dt_rho(self, dt_over_rho):
        self._check(self.lib.nf_set_dt_rho(self.h, float(dt_over_rho)), "nf_set_dt_rho")

    def set_domain_bc(self, face, bc_type, p_value=0.0):
        self._check(self.lib.nf_set_domain_bc(self.h, int(face), int(bc_type), float(p_value)), "nf_set_domain_bc")

    def set_solver_options(self, nu_pre=1, nu_post=1, flags=0):
        self._check(self.lib.nf_set_solver_options(self.h, nu_pre, nu_post, flags), "nf_set_solver_options")

    @_bound
    def set_coarse_sweeps(self, nu_level1=2, nu_deeper=None):
        nd = nu_level1 if nu_deeper is None else nu_deeper
        self._check(self.lib.nf_set_coarse_sweeps(self.h, int(nu_level1), int(nd)), "nf_set_coarse_sweeps")

    @_bound
    def set_coarse_relaxation(self, omega=1.0):
        self._check(self.lib.nf_set_coarse_relaxation(self.h, float(omega)), "nf_set_coarse_relaxation")

    def coarse_relaxation(self):
        return float(self.lib.nf_get_coarse_relaxation(self.h))

    def sweeps(self):
        """(nu_fine_pre, nu_fine_post, nu_level1, nu_deeper) in force."""
        v = [ctypes.c_int() for _ in range(4)]
        self._check(self.lib.nf_get_sweeps(self.h, *[ctypes.byref(x) for x in v]), "nf_get_sweeps")
        return tuple(x.value for x in v)

    def set_pressure_lo(self, lo):
        """Install (or remove with None) the cell array that receives the low-order part of the next pressures."""
        self._expect(lo, self.shape_p, "lo")
        self._lo_keepalive = lo
        self._check(self.lib.nf_set_pressure_lo(self.h, _ptr(lo)), "nf_set_pressure_lo")

    @_bound
    def set_solid(self, sdf, us=None, vs=None, ws=None):
        self._expect(sdf, self.shape_sdf, "sdf")
        self._expect(us, self.shape_u, "us"); self._expect(vs, self.shape_v, "vs"); self._expect(ws, self.shape_w, "ws")
        self._check(self.lib.nf_set_solid(self.h, _ptr(sdf), _ptr(us), _ptr(vs), _ptr(ws)), "nf_set_solid")

    @_bound
    def set_weights(self, au, av, aw):
        self._expect(au, self.shape_u, "au"); self._expect(av, self.shape_v, "av"); self._expect(aw, self.shape_w, "aw")
        self._check(self.lib.nf_set_weights(self.h, _ptr(au), _ptr(av), _ptr(aw)), "nf_set_weights")

    @_bound
    def get_weights(self):
        import torch
        au = torch.empty(self.shape_u, dtype=torch.float32, device=self.device)
        av = torch.empty(self.shape_v, dtype=torch.float32, device=self.device)
        aw = torch.empty(self.shape_w, dtype=torch.float32, device=self.device)
        self._check(self.lib.nf_get_weights(self.h, _ptr(au), _ptr(av), _ptr(aw)), "nf_get_weights")
        return au, av, aw

    @_bound
    def set_solid_velocity(self, us=None, vs=None, ws=None):
        self._expect(us, self.shape_u, "us"); self._expect(vs, self.shape_v, "vs"); self._expect(ws, self.shape_w, "ws")
        self._check(self.lib.nf_set_solid_velocity(self.h, _ptr(us), _ptr(vs), _ptr(ws)), "nf_set_solid_velocity")

    # -- hot path -----------------------------------------------------------------------------------------
    @_bound
    def solve(self, rhs, p, tol=1e-6, maxit=200):
        self._expect(rhs, self.shape_p, "rhs"); self._expect(p, self.shape_p, "p")
        return self._check(self.lib.nf_solve(self.h, _ptr(rhs), _ptr(p), float(tol), int(maxit)), "nf_solve")

    @_bound
    def project(self, u, v, w, p, tol=1e-6, maxit=200):
        self._expect(u, self.shape_u, "u"); self._expect(v, self.shape_v, "v"); self._expect(w, self.shape_w, "w")
        self._expect(p, self.shape_p, "p")
        return self._check(self.lib.nf_project(self.h, _ptr(u), _ptr(v), _ptr(w), _ptr(p), float(tol), int(maxit)),
                           "nf_project")

    @_bound
    def project_adjoint(self, gu, gv, gw, p_saved=None, uhat=None, galpha=None, gus=None, y_out=None, tol=1e-6,
                        maxit=200):
        self._expect(gu, self.shape_u, "gu"); self._expect(gv, self.shape_v, "gv"); self._expect(gw, self.shape_w, "gw")
        self._expect(p_saved, self.shape_p, "p_saved"); self._expect(y_out, self.shape_p, "y_out")
        uh = uhat if uhat is not None else (None, None, None)
        ga = galpha if galpha is not None else (None, None, None)
        gs = gus if gus is not None else (None, None, None)
        for trip, nm in ((uh, "uhat"), (ga, "galpha"), (gs, "gus")):
            self._expect(trip[0], self.shape_u, nm + "_u"); self._expect(trip[1], self.shape_v, nm + "_v")
            self._expect(trip[2], self.shape_w, nm + "_w")
        rc = self.lib.nf_project_adjoint(self.h, _ptr(gu), _ptr(gv), _ptr(gw), _ptr(p_saved), _ptr(uh[0]), _ptr(uh[1]),
                                         _ptr(uh[2]), _ptr(ga[0]), _ptr(ga[1]), _ptr(ga[2]), _ptr(gs[0]), _ptr(gs[1]),
                                         _ptr(gs[2]), _ptr(y_out), float(tol), int(maxit))
        return self._check(rc, "nf_project_adjoint")

    @_bound
    def advect(self, u, v, w, dt):
        self._expect(u, self.shape_u, "u"); self._expect(v, self.shape_v, "v"); self._expect(w, self.shape_w, "w")
        self._check(self.lib.nf_advect(self.h, _ptr(u), _ptr(v), _ptr(w), float(dt)), "nf_advect")

    @_bound
    def max_speed(self, u, v, w):
        """max over all faces of |u|, |v|, |w| (synchronises)."""
        self._expect(u, self.shape_u, "u"); self._expect(v, self.shape_v, "v"); self._expect(w, self.shape_w, "w")
        out = ctypes.c_float()
        self._check(self.lib.nf_max_speed(self.h, _ptr(u), _ptr(v), _ptr(w), ctypes.byref(out)), "nf_max_speed")
        return out.value

    @_bound
    def viscosity(self, u, v, w, nu, dt):
        """Explicit viscosity step, in place; symmetric, so the backward pass calls it on the gradient (Eq. 8)."""
        self._expect(u, self.shape_u, "u"); self._expect(v, self.shape_v, "v"); self._expect(w, self.shape_w, "w")
        self._check(self.lib.nf_viscosity(self.h, _ptr(u), _ptr(v), _ptr(w), float(nu), float(dt)), "nf_viscosity")

    # ---- NEXT-2: parametric geometry (host parameter vectors: any float sequence / NumPy array) ----
    @staticmethod
    def geom_n_params(K, N):
        return 2 + K * (2 + 2 * N)

    def _geom_vec(self, v, K, N, name):
        import numpy as np
        a = np.ascontiguousarray(np.asarray(v, dtype=np.float32))
        if a.shape != (self.geom_n_params(K, N),):
            raise ValueError("%s: expected %d values" % (name, self.geom_n_params(K, N)))
        return a, a.ctypes.data_as(_c_host_float_p)

    @_bound
    def geom_sdf(self, params, K, N, M, sdf, complement=False):
        self._expect(sdf, self.shape_sdf, "sdf")
        _keep, pp = self._geom_vec(params, K, N, "params")
        self._check(self.lib.nf_geom_sdf(self.h, pp, int(K), int(N), int(M), 1 if complement else 0, _ptr(sdf)),
                    "nf_geom_sdf")

    @_bound
    def geom_sdf_adjoint(self, params, K, N, M, gsdf, complement=False):
        """-> NumPy float64 vector dJ/dparams (synchronises)."""
        import numpy as np
        self._expect(gsdf, self.shape_sdf, "gsdf")
        _keep, pp = self._geom_vec(params, K, N, "params")
        out = np.zeros(self.geom_n_params(K, N), dtype=np.float64)
        self._check(self.lib.nf_geom_sdf_adjoint(self.h, pp, int(K), int(N), int(M), 1 if complement else 0, _ptr(gsdf),
                                                 out.ctypes.data_as(_c_host_double_p)), "nf_geom_sdf_adjoint")
        return out

    @_bound
    def geom_csg(self, op, a, b, out):
        for t, n in ((a, "a"), (b, "b"), (out, "out")):
            self._expect(t, self.shape_sdf, n)
        self._check(self.lib.nf_geom_csg(self.h, {"union": 0, "intersection": 1}[op], _ptr(a), _ptr(b), _ptr(out)),
                    "nf_geom_csg")

    @_bound
    def geom_csg_adjoint(self, op, a, b, gout, ga, gb):
        for t, n in ((a, "a"), (b, "b"), (gout, "gout"), (ga, "ga"), (gb, "gb")):
            self._expect(t, self.shape_sdf, n)
        self._check(self.lib.nf_geom_csg_adjoint(self.h, {"union": 0, "intersection": 1}[op], _ptr(a), _ptr(b),
                                                 _ptr(gout), _ptr(ga), _ptr(gb)), "nf_geom_csg_adjoint")

    @_bound
    def geom_velocity(self, params, pdot, K, N, M, us, vs, ws, band=float("inf")):
        for t, s, n in ((us, self.shape_u, "us"), (vs, self.shape_v, "vs"), (ws, self.shape_w, "ws")):
            if t is not None:
                self._expect(t, s, n)
        _k1, pp = self._geom_vec(params, K, N, "params")
        _k2, pd = self._geom_vec(pdot, K, N, "pdot")
        self._check(self.lib.nf_geom_velocity(self.h, pp, pd, int(K), int(N), int(M), float(band), _ptr(us), _ptr(vs),
                                              _ptr(ws)), "nf_geom_velocity")

    @_bound
    def geom_velocity_adjoint(self, params, K, N, M, gus, gvs, gws, band=float("inf")):
        """-> NumPy float64 vector dJ/dpdot (synchronises)."""
        import numpy as np
        for t, s, n in ((gus, self.shape_u, "gus"), (gvs, self.shape_v, "gvs"), (gws, self.shape_w, "gws")):
            if t is not None:
                self._expect(t, s, n)
        _keep, pp = self._geom_vec(params, K, N, "params")
        out = np.zeros(self.geom_n_params(K, N), dtype=np.float64)
        self._check(self.lib.nf_geom_velocity_adjoint(self.h, pp, int(K), int(N), int(M), float(band), _ptr(gus),
                                                      _ptr(gvs), _ptr(gws), out.ctypes.data_as(_c_host_double_p)),
                    "nf_geom_velocity_adjoint")
        return out

    @_bound
    def advect_adjoint(self, u0, v0, w0, gu, gv, gw, dt):
        for t, s, n in ((u0, self.shape_u, "u0"), (v0, self.shape_v, "v0"), (w0, self.shape_w, "w0"),
                        (gu, self.shape_u, "gu"), (gv, self.shape_v, "gv"), (gw, self.shape_w, "gw")):
            self._expect(t, s, n)
        self._check(self.lib.nf_advect_adjoint(self.h, _ptr(u0), _ptr(v0), _ptr(w0), _ptr(gu), _ptr(gv), _ptr(gw),
                                               float(dt)), "nf_advect_adjoint")

    @_bound
    def weights_adjoint(self, gau, gav, gaw, gsdf):
        self._expect(gau, self.shape_u, "gau"); self._expect(gav, self.shape_v, "gav")
        self._expect(gaw, self.shape_w, "gaw"); self._expect(gsdf, self.shape_sdf, "gsdf")
        self._check(self.lib.nf_weights_adjoint(self.h, _ptr(gau), _ptr(gav), _ptr(gaw), _ptr(gsdf)),
                    "nf_weights_adjoint")

    @_bound
    def apply_A(self, p, q):
        self._expect(p, self.shape_p, "p"); self._expect(q, self.shape_p, "q")
        self._check(self.lib.nf_apply_A(self.h, _ptr(p), _ptr(q)), "nf_apply_A")

    @_bound
    def vcycle(self, r, z):
        self._expect(r, self.shape_p, "r"); self._expect(z, self.shape_p, "z")
        self._check(self.lib.nf_vcycle(self.h, _ptr(r), _ptr(z)), "nf_vcycle")

    # -- host-buffer variants (e2e timing) ------------------------------------------------------------------
    @_bound
    def project_host(self, u, v, w, p, tol=1e-6, maxit=200):
        self._expect(u, self.shape_u, "u", host=True); self._expect(v, self.shape_v, "v", host=True)
        self._expect(w, self.shape_w, "w", host=True); self._expect(p, self.shape_p, "p", host=True)
        return self._check(self.lib.nf_project_host(self.h, _ptr(u), _ptr(v), _ptr(w), _ptr(p), float(tol),
                                                    int(maxit)), "nf_project_host")

    @_bound
    def project_adjoint_host(self, gu, gv, gw, tol=1e-6, maxit=200):
        self._expect(gu, self.shape_u, "gu", host=True); self._expect(gv, self.shape_v, "gv", host=True)
        self._expect(gw, self.shape_w, "gw", host=True)
        return self._check(self.lib.nf_project_adjoint_host(self.h, _ptr(gu), _ptr(gv), _ptr(gw), None, None, None,
                                                            None, float(tol), int(maxit)), "nf_project_adjoint_host")

    def set_host_async(self, on=True):
        self._check(self.lib.nf_set_host_async(self.h, 1 if on else 0), "nf_set_host_async")

    def host_sync(self):
        self._check(self.lib.nf_host_sync(self.h), "nf_host_sync")

    # -- info -------------------------------------------------------------------------------------------------
    def last_solve_info(self):
        it, rr, ms = ctypes.c_int(), ctypes.c_float(), ctypes.c_float()
        self._check(self.lib.nf_last_solve_info(self.h, ctypes.byref(it), ctypes.byref(rr), ctypes.byref(ms)),
                    "nf_last_solve_info")
        return dict(iters=it.value, relres=rr.value, ms=ms.value)

    def info(self):
        lv, na, sg = ctypes.c_int(), ctypes.c_longlong(), ctypes.c_int()
        self._check(self.lib.nf_grid_info(self.h, ctypes.byref(lv), ctypes.byref(na), ctypes.byref(sg)), "nf_grid_info")
        return dict(levels=lv.value, active_cells=na.value, singular=sg.value)

    def components(self):
        """(number of fluid components, number of singular ones) of the current weights (R12)."""
        nc, ns = ctypes.c_int(), ctypes.c_int()
        self._check(self.lib.nf_grid_components(self.h, ctypes.byref(nc), ctypes.byref(ns)), "nf_grid_components")
        return nc.value, ns.value

    def profile_enable(self, on=True):
        self._check(self.lib.nf_profile_enable(self.h, 1 if on else 0), "nf_profile_enable")

    def profile(self):
        """{class name: (ms, launches)} accumulated since profile_enable(True)."""
        out, idx = {}, 0
        while True:
            nm, ms, n = ctypes.c_char_p(), ctypes.c_double(), ctypes.c_longlong()
            rc = self.lib.nf_profile_get(self.h, idx, ctypes.byref(nm), ctypes.byref(ms), ctypes.byref(n))
            if rc != NF_OK:
                break
            out[nm.value.decode()] = (ms.value, n.value)
            idx += 1
        return out

    def launch_count(self):
        return int(self.lib.nf_launch_count(self.h))


# ---- batched entry points (include/nf.h "NEXT-4"): n grids of equal extents on one stream ---------------------------------
def _ptr_array(tensors):
    """HOST array of device addresses (None -> NULL array)."""
    if tensors is None:
        return None
    arr = (ctypes.c_void_p * len(tensors))()
    for i, t in enumerate(tensors):
        arr[i] = _ptr(t).value if t is not None else None
    return arr


def _batch_prologue(grids):
    import torch
    g0 = grids[0]
    if any(g.device != g0.device for g in grids):
        raise ValueError("a batch lives on one device")
    for g in grids:
        g._bind_stream()  # every handle of the batch on the current torch stream
    h = (ctypes.c_void_p * len(grids))(*[g.h for g in grids])
    return g0, h, (ctypes.c_int * len(grids))()


def solve_batch(grids, rhs, p, tol=1e-6, maxit=200):
    """nf_solve_batch: rhs, p = lists of n cell tensors.  Returns the list of per-grid status codes."""
    g0, h, st = _batch_prologue(grids)
    rc = g0.lib.nf_solve_batch(h, len(grids), _ptr_array(rhs), _ptr_array(p), float(tol), int(maxit), st)
    g0._check(rc, "nf_solve_batch")
    return list(st)


def project_batch(grids, U, p, tol=1e-6, maxit=200):
    """nf_project_batch: U = list of n (u, v, w) triples (in place), p = list of n cell tensors."""
    g0, h, st = _batch_prologue(grids)
    rc = g0.lib.nf_project_batch(h, len(grids), _ptr_array([a[0] for a in U]), _ptr_array([a[1] for a in U]),
                                 _ptr_array([a[2] for a in U]), _ptr_array(p), float(tol), int(maxit), st)
    g0._check(rc, "nf_project_batch")
    return list(st)


def project_adjoint_batch(grids, G, y, p_saved=None, uhat=None, galpha=None, gus=None, tol=1e-6, maxit=200):
    """nf_project_adjoint_batch: G = list of n (gu, gv, gw) triples (in place: dJ/dU -> dJ/dUhat), y = list of n cell
    tensors (the adjoint variable, required); p_saved / uhat / galpha / gus: lists as in Grid.project_adjoint or None."""
    g0, h, st = _batch_prologue(grids)
    col = lambda L, c: None if L is None else _ptr_array([a[c] for a in L])
    rc = g0.lib.nf_project_adjoint_batch(h, len(grids), col(G, 0), col(G, 1), col(G, 2), _ptr_array(p_saved),
                                         col(uhat, 0), col(uhat, 1), col(uhat, 2), col(galpha, 0), col(galpha, 1),
                                         col(galpha, 2), col(gus, 0), col(gus, 1), col(gus, 2), _ptr_array(y),
                                         float(tol), int(maxit), st)
    g0._check(rc, "nf_project_adjoint_batch")
    return list(st)


def max_speed_static(u, v, w, out, stream=None):
    """nf_max_speed_static: max over all faces of |u|, |v|, |w| into the one-element DEVICE tensor `out`, without a
    handle and without any allocation (fixed scratch inside the library, include/nf.h).  Enqueued on `stream`
    (default: torch's current stream of the tensors' device); no synchronisation.  Calls that overlap on the GPU race
    on the shared scratch.  Raises NfError for sizes beyond the scratch (u + v + w faces > 268 435 456)."""
    import torch
    lib = load_library()
    nz, ny, nx = u.shape[0], u.shape[1], u.shape[2] - 1
    if tuple(v.shape) != (nz, ny + 1, nx) or tuple(w.shape) != (nz + 1, ny, nx):
        raise ValueError("u, v, w must be (nz, ny, nx+1), (nz, ny+1, nx), (nz+1, ny, nx)")
    for t in (u, v, w, out):
        if not t.is_cuda or t.device != u.device:
            raise ValueError("nf_max_speed_static takes device tensors on one device")
    if out.numel() != 1:
        raise ValueError("out must hold one float32")
    with torch.cuda.device(u.device):
        s = stream if stream is not None else torch.cuda.current_stream()
        rc = lib.nf_max_speed_static(_ptr(u), _ptr(v), _ptr(w), int(nx), int(ny), int(nz),
                                     ctypes.c_void_p(s.cuda_stream), _ptr(out))
    if rc != 0:
        raise NfError("nf_max_speed_static failed (%d): %s" % (rc, lib.nf_static_last_error().decode()))
    return out
