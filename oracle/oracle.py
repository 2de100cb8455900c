"""ctypes face of the CPU oracle (oracle/sldg_oracle.c) -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It never imports the CUDA package and shares no code with it.
All arrays are numpy float64, C-contiguous, flat layout as in sldg_oracle.c's header
(x_1 fastest; as a numpy array the shape is (D_last, ..., D_1, D_0)).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        dp, ip, vp, lg = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p, C.c_long
        fp = C.POINTER(C.c_float)
        sig = {
            "orc_gauss_legendre": (None, [C.c_int, dp, dp]),
            "orc_lagrange": (C.c_double, [C.c_int, dp, C.c_int, C.c_double]),
            "orc_AB": (None, [C.c_int, C.c_double, dp, dp]),
            "orc_sweep_line": (None, [C.c_int, C.c_int, C.c_double, dp, dp, lg]),
            "orc_create": (vp, [C.c_int, C.c_int, ip, C.c_int, dp]),
            "orc_destroy": (None, [vp]),
            "orc_set_threads": (None, [vp, C.c_int]),
            "orc_max_threads": (C.c_int, []),
            "orc_field_elems": (lg, [vp]),
            "orc_rho_elems": (lg, [vp]),
            "orc_node_coords": (None, [vp, C.c_int, dp]),
            "orc_sweep_axis": (None, [vp, dp, dp, C.c_int, dp, C.c_int, C.c_int]),
            "orc_advect_x": (None, [vp, dp, dp, C.c_double]),
            "orc_advect_v": (None, [vp, dp, dp, dp, C.c_double]),
            "orc_density": (None, [vp, dp, dp]),
            "orc_poisson": (None, [vp, dp, dp]),
            "orc_step": (None, [vp, dp, dp, dp, dp, C.c_double]),
            "orc_mass": (C.c_double, [vp, dp]),
            "orc_electric_energy": (C.c_double, [vp, dp]),
            "orc_sweep_axis_f32": (None, [vp, fp, fp, C.c_int, dp, C.c_int, C.c_int]),
            "orc_advect_x_f32": (None, [vp, fp, fp, C.c_double]),
            "orc_advect_v_f32": (None, [vp, fp, fp, dp, C.c_double]),
            "orc_density_f32": (None, [vp, fp, dp]),
            "orc_step_f32": (None, [vp, fp, fp, dp, dp, C.c_double]),
            "orc_mass_f32": (C.c_double, [vp, fp]),
            "orc_lagrange_deriv": (C.c_double, [C.c_int, dp, C.c_int, C.c_double]),
            "orc_sipg_sigma_default": (C.c_double, [C.c_int]),
            "orc_sipg_MB": (None, [C.c_int, C.c_double, dp, dp]),
            "orc_sipg_apply": (None, [vp, C.c_double, dp, dp]),
            "orc_sipg_rhs": (None, [vp, dp, dp]),
            "orc_grad_phi": (None, [vp, dp, dp]),
            "orc_poisson_cg": (C.c_int, [vp, C.c_double, dp, dp, dp, C.c_double, C.c_int, dp]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(_lib, name)
            fn.restype, fn.argtypes = res, args
    return _lib


def _p(a):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _pf(a):
    assert a.dtype == np.float32 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_float))


def gauss_legendre(n):
    xi, w = np.empty(n), np.empty(n)
    lib().orc_gauss_legendre(n, _p(xi), _p(w))
    return xi, w


def lagrange(xi, l, z):
    xi = np.ascontiguousarray(xi, dtype=np.float64)
    return lib().orc_lagrange(len(xi), _p(xi), l, float(z))


def AB(k, alpha):
    A, B = np.empty((k + 1, k + 1)), np.empty((k + 1, k + 1))
    lib().orc_AB(k, float(alpha), _p(A), _p(B))
    return A, B


def sweep_line(k, u, delta):
    """u: 1-D array of N*(k+1) nodal values of one line; returns the line shifted by delta cells."""
    u = np.ascontiguousarray(u, dtype=np.float64)
    n = u.size // (k + 1)
    assert n * (k + 1) == u.size
    out = np.empty_like(u)
    lib().orc_sweep_line(k, n, float(delta), _p(u), _p(out), 1)
    return out


def lagrange_deriv(xi, l, z):
    xi = np.ascontiguousarray(xi, dtype=np.float64)
    return lib().orc_lagrange_deriv(len(xi), _p(xi), l, float(z))


def sipg_sigma_default(k):
    return lib().orc_sipg_sigma_default(k)


def sipg_MB(k, sigma):
    """M, B of the SIPG block-tridiagonal matrix (reading I)."""
    M, B = np.empty((k + 1, k + 1)), np.empty((k + 1, k + 1))
    lib().orc_sipg_MB(k, float(sigma), _p(M), _p(B))
    return M, B


class Oracle:
    """Mirror of the solver's problem statement: create(dim_x, dim_v, cells, degree, domain)."""

    def __init__(self, dim_x, dim_v, cells, degree, domain, threads=1):
        self.dx, self.dv, self.d, self.k = dim_x, dim_v, dim_x + dim_v, degree
        self.cells = [int(c) for c in cells]
        self.domain = [float(v) for v in np.asarray(domain, dtype=np.float64).ravel()]
        assert len(self.cells) == self.d and len(self.domain) == 2 * self.d
        ca = (C.c_int * self.d)(*self.cells)
        da = (C.c_double * (2 * self.d))(*self.domain)
        self._h = lib().orc_create(dim_x, dim_v, ca, degree, da)
        if not self._h:
            raise ValueError("orc_create rejected the arguments")
        self.D = [c * (degree + 1) for c in self.cells]
        self.nf = lib().orc_field_elems(self._h)
        self.X = lib().orc_rho_elems(self._h)
        self.shape = tuple(reversed(self.D))            # numpy shape, x_1 last (fastest)
        self.xshape = tuple(reversed(self.D[:dim_x]))
        self.set_threads(threads)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    def set_threads(self, t):
        self.threads = max(1, int(t))
        lib().orc_set_threads(self._h, self.threads)

    def node_coords(self, axis):
        out = np.empty(self.D[axis])
        lib().orc_node_coords(self._h, axis, _p(out))
        return out

    def sweep_axis(self, f, axis, delta, mode=None, saxis=None):
        """One sweep along `axis` with a caller-given delta table (cells).
        x axis (axis < dx): delta indexed by the node of v-axis dx+axis; v axis: by flat x-node."""
        if mode is None:
            mode = 0 if axis < self.dx else 1
        if saxis is None:
            saxis = self.dx + axis if mode == 0 else -1
        delta = np.ascontiguousarray(delta, dtype=np.float64)
        assert delta.size == (self.D[saxis] if mode == 0 else self.X)
        fin = np.ascontiguousarray(f, dtype=np.float64).reshape(-1)
        out = np.empty_like(fin)
        lib().orc_sweep_axis(self._h, _p(fin), _p(out), axis, _p(delta), mode, saxis)
        return out.reshape(self.shape)

    def advect_x(self, f, tau):
        g = np.array(f, dtype=np.float64, order="C").reshape(-1)
        tmp = np.empty_like(g)
        lib().orc_advect_x(self._h, _p(g), _p(tmp), float(tau))
        return g.reshape(self.shape)

    def advect_v(self, f, E, tau):
        g = np.array(f, dtype=np.float64, order="C").reshape(-1)
        tmp = np.empty_like(g)
        E = np.ascontiguousarray(E, dtype=np.float64).reshape(-1)
        assert E.size == self.dx * self.X
        lib().orc_advect_v(self._h, _p(g), _p(tmp), _p(E), float(tau))
        return g.reshape(self.shape)

    def density(self, f):
        fin = np.ascontiguousarray(f, dtype=np.float64).reshape(-1)
        rho = np.empty(self.X)
        lib().orc_density(self._h, _p(fin), _p(rho))
        return rho.reshape(self.xshape)

    def poisson(self, rho):
        r = np.ascontiguousarray(rho, dtype=np.float64).reshape(-1)
        E = np.empty(self.dx * self.X)
        lib().orc_poisson(self._h, _p(r), _p(E))
        return E.reshape((self.dx,) + self.xshape)

    def step(self, f, dt):
        """One Strang step; returns (f_new, rho, E) with rho, E from the middle of the step."""
        g = np.array(f, dtype=np.float64, order="C").reshape(-1)
        tmp = np.empty_like(g)
        rho, E = np.empty(self.X), np.empty(self.dx * self.X)
        lib().orc_step(self._h, _p(g), _p(tmp), _p(rho), _p(E), float(dt))
        return g.reshape(self.shape), rho.reshape(self.xshape), E.reshape((self.dx,) + self.xshape)

    def mass(self, f):
        return lib().orc_mass(self._h, _p(np.ascontiguousarray(f, dtype=np.float64).reshape(-1)))

    def electric_energy(self, E):
        return lib().orc_electric_energy(self._h, _p(np.ascontiguousarray(E, dtype=np.float64).reshape(-1)))

    # ---- CGdG Poisson solver
    def sipg_apply(self, u, sigma=None):
        sigma = sipg_sigma_default(self.k) if sigma is None else sigma
        u = np.ascontiguousarray(u, dtype=np.float64).reshape(-1)
        out = np.empty(self.X)
        lib().orc_sipg_apply(self._h, float(sigma), _p(u), _p(out))
        return out.reshape(self.xshape)

    def sipg_rhs(self, rho):
        r = np.ascontiguousarray(rho, dtype=np.float64).reshape(-1)
        b = np.empty(self.X)
        lib().orc_sipg_rhs(self._h, _p(r), _p(b))
        return b.reshape(self.xshape)

    def grad_phi(self, phi):
        u = np.ascontiguousarray(phi, dtype=np.float64).reshape(-1)
        E = np.empty(self.dx * self.X)
        lib().orc_grad_phi(self._h, _p(u), _p(E))
        return E.reshape((self.dx,) + self.xshape)

    def poisson_cg(self, rho, phi0=None, tol=1e-3, maxiter=None, sigma=None):
        """Algorithm 1 from the starting vector phi0 (zeros if None).  Returns (E, phi, iterations, relres)."""
        sigma = sipg_sigma_default(self.k) if sigma is None else sigma
        if maxiter is None:
            maxiter = 4 * int(round(self.X ** (1.0 / self.dx))) + 20         # PAPER.md:567, safety factor 4
        r = np.ascontiguousarray(rho, dtype=np.float64).reshape(-1)
        phi = np.zeros(self.X) if phi0 is None else np.array(phi0, dtype=np.float64, order="C").reshape(-1)
        E, info = np.empty(self.dx * self.X), np.empty(2)
        it = lib().orc_poisson_cg(self._h, float(sigma), _p(r), _p(phi), _p(E), float(tol), int(maxiter), _p(info))
        return E.reshape((self.dx,) + self.xshape), phi.reshape(self.xshape), it, float(info[0])

    # ---- single precision mode (reading W): float32 storage and sweep arithmetic, fp64 field solve
    def sweep_axis_f32(self, f, axis, delta, mode=None, saxis=None):
        if mode is None:
            mode = 0 if axis < self.dx else 1
        if saxis is None:
            saxis = self.dx + axis if mode == 0 else -1
        delta = np.ascontiguousarray(delta, dtype=np.float64)
        assert delta.size == (self.D[saxis] if mode == 0 else self.X)
        fin = np.ascontiguousarray(f, dtype=np.float32).reshape(-1)
        out = np.empty_like(fin)
        lib().orc_sweep_axis_f32(self._h, _pf(fin), _pf(out), axis, _p(delta), mode, saxis)
        return out.reshape(self.shape)

    def advect_x_f32(self, f, tau):
        g = np.array(f, dtype=np.float32, order="C").reshape(-1)
        tmp = np.empty_like(g)
        lib().orc_advect_x_f32(self._h, _pf(g), _pf(tmp), float(tau))
        return g.reshape(self.shape)

    def advect_v_f32(self, f, E, tau):
        g = np.array(f, dtype=np.float32, order="C").reshape(-1)
        tmp = np.empty_like(g)
        E = np.ascontiguousarray(E, dtype=np.float64).reshape(-1)
        assert E.size == self.dx * self.X
        lib().orc_advect_v_f32(self._h, _pf(g), _pf(tmp), _p(E), float(tau))
        return g.reshape(self.shape)

    def density_f32(self, f):
        fin = np.ascontiguousarray(f, dtype=np.float32).reshape(-1)
        rho = np.empty(self.X)
        lib().orc_density_f32(self._h, _pf(fin), _p(rho))
        return rho.reshape(self.xshape)

    def step_f32(self, f, dt):
        g = np.array(f, dtype=np.float32, order="C").reshape(-1)
        tmp = np.empty_like(g)
        rho, E = np.empty(self.X), np.empty(self.dx * self.X)
        lib().orc_step_f32(self._h, _pf(g), _pf(tmp), _p(rho), _p(E), float(dt))
        return g.reshape(self.shape), rho.reshape(self.xshape), E.reshape((self.dx,) + self.xshape)

    def mass_f32(self, f):
        return lib().orc_mass_f32(self._h, _pf(np.ascontiguousarray(f, dtype=np.float32).reshape(-1)))
