"""ctypes binding with the same names as include/sldg.h (argument marshalling only).

PyTorch supplies device memory and the stream; nothing here computes.  This module never
imports anything under oracle/.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBNAME = "libsldg_b200.so"

NKINDS = 12
ABI_VERSION = 3          # SLDG_ABI_VERSION of the include/sldg.h these argument lists were written against
MAX_DIM = 6
KIND_NAMES = ["sweep_axis0_tma", "sweep_slow_axis", "rho", "poisson", "shift_tables", "copies", "sweep_fused_x", "sweep_fused_v", "sweep_fused_x_double", "sweep_fused_v3", "sweep_fused_x3_double", "table_uploads"]

_vp, _dp, _ip, _ll = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_longlong
_llp = C.POINTER(C.c_longlong)

# name -> (restype, argtypes); every symbol include/sldg.h declares
EXPORTS = {
    "sldg_abi_version": (C.c_int, []),
    "sldg_create": (C.c_int, [C.POINTER(_vp), C.c_int, C.c_int, _ip, C.c_int, _dp]),
    "sldg_create_prec": (C.c_int, [C.POINTER(_vp), C.c_int, C.c_int, _ip, C.c_int, _dp, C.c_int]),
    "sldg_precision": (C.c_int, [_vp]),
    "sldg_destroy": (C.c_int, [_vp]),
    "sldg_set_stream": (C.c_int, [_vp, _vp]),
    "sldg_workspace_bytes": (C.c_size_t, [_vp]),
    "sldg_set_workspace": (C.c_int, [_vp, _vp, C.c_size_t]),
    "sldg_advect_x": (C.c_int, [_vp, _vp, C.c_double]),
    "sldg_advect_v": (C.c_int, [_vp, _vp, _vp, C.c_double]),
    "sldg_density": (C.c_int, [_vp, _vp, _vp]),
    "sldg_poisson": (C.c_int, [_vp, _vp, _vp]),
    "sldg_step": (C.c_int, [_vp, _vp, C.c_double]),
    "sldg_graph_active": (C.c_int, [_vp]),
    "sldg_step_to": (C.c_int, [_vp, _vp, _vp, C.c_double, C.c_int]),
    "sldg_workspace_field": (_vp, [_vp]),
    "sldg_plan_query_step_to": (C.c_int, [C.c_int, C.c_int, _ip, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                          C.POINTER(C.c_longlong)]),
    "sldg_steps": (C.c_int, [_vp, _vp, C.c_double, C.c_int]),
    "sldg_step_host": (C.c_int, [_vp, _vp, _vp, _vp, C.c_double, C.c_int]),
    "sldg_field_elems": (_ll, [_vp]),
    "sldg_rho_elems": (_ll, [_vp]),
    "sldg_nodes": (C.c_int, [_vp, C.c_int]),
    "sldg_node_coords": (C.c_int, [_vp, C.c_int, _dp]),
    "sldg_last_rho": (_vp, [_vp]),
    "sldg_last_E": (_vp, [_vp]),
    "sldg_electric_energy": (C.c_int, [_vp, _vp, _dp]),
    "sldg_mass": (C.c_int, [_vp, _vp, _dp]),
    "sldg_strerror": (C.c_char_p, [C.c_int]),
    "sldg_last_cuda_error": (C.c_int, [_vp]),
    "sldg_AB": (C.c_int, [C.c_int, C.c_double, C.c_int, _dp, _dp]),
    "sldg_gauss_legendre": (C.c_int, [C.c_int, _dp, _dp]),
    "sldg_advect_axis": (C.c_int, [_vp, _vp, C.c_int, _dp]),
    "sldg_timing_enable": (C.c_int, [_vp, C.c_int]),
    "sldg_timing_read": (C.c_int, [_vp, _llp, _dp]),
    "sldg_launch_count": (_ll, [_vp]),
    "sldg_timing_axis": (C.c_int, [_vp, _llp, _dp]),
    "sldg_set_option": (C.c_int, [_vp, C.c_char_p, _ll]),
    "sldg_poisson_cg": (C.c_int, [_vp, _vp, _vp, C.c_double, C.c_int]),
    "sldg_set_poisson_solver": (C.c_int, [_vp, C.c_int, C.c_double, C.c_int, C.c_double]),
    "sldg_cg_reset": (C.c_int, [_vp]),
    "sldg_cg_info": (C.c_int, [_vp, _ip, _dp]),
    "sldg_last_phi": (_vp, [_vp]),
    "sldg_sipg_matrices": (C.c_int, [C.c_int, C.c_double, _dp, _dp]),
    "sldg_density_static": (C.c_int, [_vp, _vp, _ll, _ll, C.c_int, _vp, _vp, _ip]),
    "sldg_density_static_max_x": (_ll, []),
    "sldg_plan_query": (C.c_int, [C.c_int, C.c_int, _ip, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                  C.POINTER(C.c_longlong)]),
}

_lib = None


class SldgError(RuntimeError):
    pass


def library_path():
    return os.path.join(_HERE, _LIBNAME)


def lib():
    """Load the in-tree CUDA library.  Fails loudly if it was not built (no fallback)."""
    global _lib
    if _lib is None:
        path = library_path()
        if not os.path.exists(path):
            raise SldgError(f"{path} is missing: run `python -m paper_2110_14557_b200.build` "
                            "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(path)
        for name, (res, args) in EXPORTS.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        if L.sldg_abi_version() != ABI_VERSION:
            raise SldgError(f"{path} has ABI version {L.sldg_abi_version()}, this binding was written for {ABI_VERSION}: rebuild")
        _lib = L
    return _lib


def _check(code, ctx=None):
    if code != 0:
        msg = lib().sldg_strerror(code).decode()
        if ctx is not None and code == -3:
            msg += f" [cudaError {lib().sldg_last_cuda_error(ctx)}]"
        raise SldgError(f"sldg error {code}: {msg}")


def _ptr(t):
    """Device (or pinned host) pointer of a contiguous float64 torch tensor."""
    import torch
    assert isinstance(t, torch.Tensor) and t.dtype == torch.float64 and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def AB(degree, alpha, device_arith=False):
    """sldg_AB: the library's A(alpha), B(alpha) (host-only call; no device needed)."""
    import numpy as np
    n = degree + 1
    A, B = np.empty((n, n)), np.empty((n, n))
    _check(lib().sldg_AB(int(degree), float(alpha), 1 if device_arith else 0,
                         A.ctypes.data_as(_dp), B.ctypes.data_as(_dp)))
    return A, B


def sipg_matrices(degree, sigma=0.0):
    import numpy as np
    M, B = np.empty((degree + 1, degree + 1)), np.empty((degree + 1, degree + 1))
    _check(lib().sldg_sipg_matrices(int(degree), float(sigma), M.ctypes.data_as(_dp), B.ctypes.data_as(_dp)))
    return M, B


def plan_query(dim_x, dim_v, cells, degree, nsteps, precision="f64", shifts_below_one=True, fuse_v=1, x_double=1, fuse_v3=1):
    """sldg_plan_query (host-only call): passes over f that sldg_step (nsteps == 0) / sldg_steps(nsteps) would launch.
    -> dict(x_passes, v_passes, rho_passes, field_solves, copies, launches)"""
    cells_c = (C.c_int * len(cells))(*[int(c) for c in cells])
    out = (C.c_longlong * 6)()
    _check(lib().sldg_plan_query(int(dim_x), int(dim_v), cells_c, int(degree), 1 if precision == "f32" else 0, int(nsteps),
                                 1 if shifts_below_one else 0, int(fuse_v), int(fuse_v3), int(x_double), out))
    return dict(zip(("x_passes", "v_passes", "rho_passes", "field_solves", "copies", "launches"), [int(v) for v in out]))


def plan_query_step_to(dim_x, dim_v, cells, degree, precision="f64", end_of_step_field=False, shifts_below_one=True, fuse_v=1,
                       x_double=1, fuse_v3=1):
    """sldg_plan_query_step_to (host-only call): passes over f of one sldg_step_to call; same dict as plan_query."""
    cells_c = (C.c_int * len(cells))(*[int(c) for c in cells])
    out = (C.c_longlong * 6)()
    _check(lib().sldg_plan_query_step_to(int(dim_x), int(dim_v), cells_c, int(degree), 1 if precision == "f32" else 0,
                                         1 if end_of_step_field else 0, 1 if shifts_below_one else 0, int(fuse_v), int(fuse_v3),
                                         int(x_double), out))
    return dict(zip(("x_passes", "v_passes", "rho_passes", "field_solves", "copies", "launches"), [int(v) for v in out]))


def gauss_legendre(degree):
    """sldg_gauss_legendre: the library's nodes and weights on [0,1] (host-only call)."""
    import numpy as np
    xi, w = np.empty(degree + 1), np.empty(degree + 1)
    _check(lib().sldg_gauss_legendre(int(degree), xi.ctypes.data_as(_dp), w.ctypes.data_as(_dp)))
    return xi, w


def density_static_max_x():
    return int(lib().sldg_density_static_max_x())


def density_static(f, Wv, rho=None, stream=None):
    """sldg_density_static: rho[x] = sum_v Wv[v] f[v, x] without a context, a workspace or any device allocation inside the
    library (for callers that cannot allocate; the partial sums use a fixed 8 MiB array inside the library, so X is limited to
    density_static_max_x() and calls that overlap on the GPU must be ordered by the caller).  f: contiguous CUDA tensor, float64
    or float32, whose leading dimensions are the v axes and whose trailing dimensions are the x axes; Wv: float64 CUDA tensor
    with one weight per v row (its size fixes V, X = f.numel() / V).  Passing rho avoids the one torch allocation made here."""
    import torch
    assert f.is_cuda and f.is_contiguous() and f.dtype in (torch.float64, torch.float32)
    assert Wv.is_cuda and Wv.is_contiguous() and Wv.dtype == torch.float64
    V = Wv.numel()
    assert V > 0 and f.numel() % V == 0
    X = f.numel() // V
    if rho is None:
        rho = torch.empty(X, dtype=torch.float64, device=f.device)
    assert rho.is_cuda and rho.is_contiguous() and rho.dtype == torch.float64 and rho.numel() == X
    st = stream if stream is not None else torch.cuda.current_stream(f.device)
    err = C.c_int(0)
    with torch.cuda.device(f.device):
        code = lib().sldg_density_static(C.c_void_p(f.data_ptr()), C.c_void_p(Wv.data_ptr()), X, V,
                                         1 if f.dtype == torch.float32 else 0, C.c_void_p(rho.data_ptr()),
                                         C.c_void_p(st.cuda_stream), C.byref(err))
    if code != 0:
        raise SldgError(f"sldg error {code}: {lib().sldg_strerror(code).decode()}" + (f" [cudaError {err.value}]" if code == -3 else ""))
    return rho


class Sldg:
    """One solver context: sldg_create(dim_x, dim_v, cells, degree, domain) plus a torch-owned workspace."""

    def __init__(self, dim_x, dim_v, cells, degree, domain, device="cuda:0", stream=None, precision="f64"):
        """precision "f32": single precision mode (sldg_create_prec, SLDG_F32): f tensors are float32."""
        import torch
        self.precision = precision
        self.dtype = {"f64": torch.float64, "f32": torch.float32}[precision]
        self._h = None
        L = lib()
        if not torch.cuda.is_available():
            raise SldgError("no CUDA device: the SLDG path has no CPU fallback")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.dx, self.dv, self.d, self.k = dim_x, dim_v, dim_x + dim_v, degree
        self.cells = [int(c) for c in cells]
        dom = [float(v) for v in domain]
        assert len(self.cells) == self.d and len(dom) == 2 * self.d
        h = _vp()
        _check(L.sldg_create_prec(C.byref(h), dim_x, dim_v, (C.c_int * self.d)(*self.cells), degree,
                                  (C.c_double * (2 * self.d))(*dom), 1 if precision == "f32" else 0))
        self._h = h
        self.D = [L.sldg_nodes(h, a) for a in range(self.d)]
        self.nf = L.sldg_field_elems(h)
        self.X = L.sldg_rho_elems(h)
        self.shape = tuple(reversed(self.D))
        self.xshape = tuple(reversed(self.D[:dim_x]))
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.stream = st
        _check(L.sldg_set_stream(h, C.c_void_p(st.cuda_stream)))
        nbytes = L.sldg_workspace_bytes(h)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        off = (-self.workspace.data_ptr()) % 256
        _check(L.sldg_set_workspace(h, C.c_void_p(self.workspace.data_ptr() + off), nbytes), h)

    def close(self):
        if self._h is not None:
            lib().sldg_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- helpers
    def _fp(self, t):
        """pointer of a contiguous f tensor of the context's precision"""
        import torch
        assert isinstance(t, torch.Tensor) and t.dtype == self.dtype and t.is_contiguous(), (t.dtype, self.dtype)
        return C.c_void_p(t.data_ptr())

    def node_coords(self, axis):
        import numpy as np
        out = np.empty(self.D[axis])
        _check(lib().sldg_node_coords(self._h, axis, out.ctypes.data_as(_dp)))
        return out

    def empty_field(self):
        import torch
        return torch.empty(self.shape, dtype=self.dtype, device=self.device)

    def AB(self, alpha, device_arith=False):
        return AB(self.k, alpha, device_arith)

    # ---- hot path (names as in include/sldg.h)
    def advect_x(self, f, dt):
        _check(lib().sldg_advect_x(self._h, self._fp(f), float(dt)), self._h)

    def advect_v(self, f, E, dt):
        _check(lib().sldg_advect_v(self._h, self._fp(f), _ptr(E), float(dt)), self._h)

    def density(self, f, rho=None):
        import torch
        if rho is None:
            rho = torch.empty(self.xshape, dtype=torch.float64, device=self.device)
        _check(lib().sldg_density(self._h, self._fp(f), _ptr(rho)), self._h)
        return rho

    def poisson(self, rho, E=None):
        import torch
        if E is None:
            E = torch.empty((self.dx,) + self.xshape, dtype=torch.float64, device=self.device)
        _check(lib().sldg_poisson(self._h, _ptr(rho), _ptr(E)), self._h)
        return E

    def poisson_cg(self, rho, E=None, tol=1e-3, maxiter=0):
        import torch
        if E is None:
            E = torch.empty((self.dx,) + self.xshape, dtype=torch.float64, device=self.device)
        _check(lib().sldg_poisson_cg(self._h, _ptr(rho), _ptr(E), float(tol), int(maxiter)), self._h)
        return E

    def set_poisson_solver(self, solver, tol=1e-3, maxiter=0, sigma=0.0):
        _check(lib().sldg_set_poisson_solver(self._h, int(solver), float(tol), int(maxiter), float(sigma)), self._h)

    def cg_reset(self):
        _check(lib().sldg_cg_reset(self._h), self._h)

    def cg_info(self):
        it, rel = C.c_int(), C.c_double()
        _check(lib().sldg_cg_info(self._h, C.byref(it), C.byref(rel)), self._h)
        return it.value, rel.value

    def last_phi(self):
        return self._view(lib().sldg_last_phi(self._h), self.xshape)

    def step(self, f, dt):
        _check(lib().sldg_step(self._h, self._fp(f), float(dt)), self._h)

    def step_to(self, f_in, f_out, dt, end_of_step_field=False):
        _check(lib().sldg_step_to(self._h, self._fp(f_in), self._fp(f_out), float(dt), 1 if end_of_step_field else 0), self._h)

    def workspace_field(self):
        """The |f|-value buffer inside the workspace as a tensor VIEW (no copy): a valid f_out / f_in of step_to."""
        ptr = lib().sldg_workspace_field(self._h)
        off = ptr - self.workspace.data_ptr()
        nbytes = self.nf * (4 if self.precision == "f32" else 8)
        return self.workspace[off:off + nbytes].view(self.dtype).reshape(self.shape)

    def graph_active(self):
        return bool(lib().sldg_graph_active(self._h))

    def steps(self, f, dt, nsteps):
        _check(lib().sldg_steps(self._h, self._fp(f), float(dt), int(nsteps)), self._h)

    def step_host(self, f_host, f_dev, dt, nsteps=1, E_host=None):
        _check(lib().sldg_step_host(self._h, self._fp(f_host), self._fp(f_dev),
                                    _ptr(E_host) if E_host is not None else None, float(dt), int(nsteps)), self._h)

    def advect_axis(self, f, axis, delta):
        import numpy as np
        d = np.ascontiguousarray(np.asarray(delta, dtype=np.float64))
        want = self.D[self.dx + axis] if axis < self.dx else self.X
        assert d.size == want, (d.size, want)
        _check(lib().sldg_advect_axis(self._h, self._fp(f), int(axis), d.ctypes.data_as(_dp)), self._h)

    def last_rho(self):
        return self._view(lib().sldg_last_rho(self._h), self.xshape)

    def last_E(self):
        return self._view(lib().sldg_last_E(self._h), (self.dx,) + self.xshape)

    def _view(self, ptr, shape):
        """Copy of a workspace region as a torch tensor (device)."""
        import torch
        base = self.workspace.data_ptr()
        off = ptr - base
        n = 1
        for s in shape:
            n *= s
        return self.workspace[off:off + 8 * n].view(torch.float64).reshape(shape).clone()

    def electric_energy(self, E):
        out = C.c_double()
        _check(lib().sldg_electric_energy(self._h, _ptr(E), C.byref(out)), self._h)
        return out.value

    def mass(self, f):
        out = C.c_double()
        _check(lib().sldg_mass(self._h, self._fp(f), C.byref(out)), self._h)
        return out.value

    # ---- instrumentation
    def timing_enable(self, on=True):
        _check(lib().sldg_timing_enable(self._h, 1 if on else 0))

    def timing_read(self):
        """-> (per kind {name: (launches, ms)}, per axis [(launches, ms)])  since the last read; synchronises."""
        n = (C.c_longlong * NKINDS)()
        ms = (C.c_double * NKINDS)()
        _check(lib().sldg_timing_read(self._h, n, ms), self._h)
        an = (C.c_longlong * MAX_DIM)()
        ams = (C.c_double * MAX_DIM)()
        _check(lib().sldg_timing_axis(self._h, an, ams))
        kinds = {KIND_NAMES[i]: (int(n[i]), float(ms[i])) for i in range(NKINDS)}
        axes = [(int(an[i]), float(ams[i])) for i in range(self.d)]
        return kinds, axes

    def launch_count(self):
        return int(lib().sldg_launch_count(self._h))

    def set_option(self, name, value):
        _check(lib().sldg_set_option(self._h, name.encode(), int(value)))
