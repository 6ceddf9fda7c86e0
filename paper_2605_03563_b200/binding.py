"""Thin Python binding over the C ABI of include/poisson.h — argument marshalling only.

Every step of the path runs in the CUDA kernels of libpoisson_b200.so; there is no CPU fallback and a missing
library is a hard error.  PyTorch is used by callers for device memory and streams; tensors are passed as raw
device pointers (`tensor.data_ptr()`).  Function names mirror the C entry points.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpoisson_b200.so")

CARTESIAN, SPHERICAL = 0, 1
BC_DIRICHLET_GHOST, BC_PERIODIC, BC_NEUMANN0, BC_AXIS = 0, 1, 2, 3
F64, MIXED = 0, 1
OK, NOT_CONVERGED, BREAKDOWN = 0, 1, 2
INVALID_ARG, UNSUPPORTED, CUDA_ERROR, OUT_OF_MEMORY = -1, -2, -3, -4
OPT_KERNEL_PATH, OPT_RESTRICTION, OPT_POLL_INTERVAL, OPT_JACOBI, OPT_RECORD_HISTORY, OPT_TIME_KERNELS = 0, 1, 2, 3, 4, 5
OPT_SOR_HALFSTEPS, OPT_FUSED_RESTRICT, OPT_BICG_RESTART_EPS = 6, 7, 8
OPT_TILE_CFG, OPT_PLANE_SPLIT, OPT_APPLY_BULK, OPT_COMPACT_ORDER = 9, 10, 11, 12
PATH_AUTO, PATH_GENERIC, PATH_PLANE = 0, 1, 2

SYMBOLS = [
    "poisson_create", "poisson_destroy", "poisson_last_error", "poisson_set_option", "poisson_set_option_f64",
    "poisson_bicgstab_stats", "poisson_apply_laplacian",
    "poisson_rbsor_sweep", "poisson_cg_solve", "poisson_bicgstab_solve", "poisson_mg_vcycle", "poisson_multipole_bc",
    "poisson_set_ghost_faces", "poisson_get_ghost_face", "poisson_face_len", "poisson_residual_norm",
    "poisson_get_history", "poisson_kernel_launches", "poisson_kernel_classes", "poisson_kernel_name",
    "poisson_kernel_class_launches", "poisson_kernel_time", "poisson_reset_kernel_times",
    "poisson_apply_laplacian_host", "poisson_rbsor_sweep_host", "poisson_cg_solve_host",
    "poisson_bicgstab_solve_host", "poisson_mg_vcycle_host", "poisson_multipole_bc_host",
    "poisson_spai_smooth", "poisson_mgv_vcycle", "poisson_mgv_vcycle_host",
    "poisson_rbsor_cheby", "poisson_rbsor_local", "poisson_pcg_solve", "poisson_multipole_inner_moments",
    "poisson_residual_norm_static", "poisson_residual_norm_static_error", "poisson_compact_rhs",
]

_lib = None


class PoissonError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("poisson error %d: %s" % (code, msg))
        self.code = code


def lib():
    """Load the CUDA library; fails loudly if it has not been built (python -m paper_2605_03563_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("CUDA extension %s is missing: run `python -m paper_2605_03563_b200.build` "
                              "(there is no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        L.poisson_last_error.restype = C.c_char_p
        L.poisson_last_error.argtypes = [C.c_void_p]
        L.poisson_residual_norm_static_error.restype = C.c_char_p
        L.poisson_residual_norm_static_error.argtypes = []
        L.poisson_face_len.restype = C.c_long
        L.poisson_face_len.argtypes = [C.c_void_p, C.c_int]
        L.poisson_kernel_launches.restype = C.c_long
        L.poisson_kernel_launches.argtypes = [C.c_void_p]
        L.poisson_kernel_name.restype = C.c_char_p
        L.poisson_kernel_name.argtypes = [C.c_int]
        L.poisson_kernel_class_launches.restype = C.c_long
        L.poisson_kernel_class_launches.argtypes = [C.c_void_p, C.c_int]
        _lib = L
    return _lib


def kernel_classes():
    """Names of the kernel classes (rows of the hot path), indexed by class id."""
    L = lib()
    return [L.poisson_kernel_name(i).decode() for i in range(L.poisson_kernel_classes())]


def _ptr(t):
    """Device (or pinned host) pointer of a torch tensor / numpy array / raw integer address."""
    if t is None:
        return C.c_void_p(0)
    if isinstance(t, int):
        return C.c_void_p(t)
    if hasattr(t, "ctypes"):  # numpy array (host entry points only)
        assert t.flags.c_contiguous, "arrays must be contiguous"
        return C.c_void_p(t.ctypes.data)
    assert t.is_contiguous(), "arrays must be contiguous"
    return C.c_void_p(t.data_ptr())


def residual_norm_static(shape, spacing, d_phi, d_rhs, d_norm, stream=0):
    """||rhs - L phi||_2 into the device double d_norm, through the entry point that allocates nothing (static
    scratch; include/poisson.h).  Queued on `stream` (a raw cudaStream_t, 0 = default stream); does not synchronise."""
    rc = lib().poisson_residual_norm_static((C.c_int * 3)(*[int(s) for s in shape]),
                                            (C.c_double * 3)(*[float(h) for h in spacing]), _ptr(d_phi), _ptr(d_rhs),
                                            _ptr(d_norm), C.c_void_p(int(stream)))
    if rc != OK:
        raise PoissonError(rc, lib().poisson_residual_norm_static_error().decode())
    return rc


class Poisson:
    """Owner of one poisson_t handle."""

    def __init__(self, shape, spacing=None, origin=None, edges=None, coord=CARTESIAN, order=2, bc=(0,) * 6,
                 stream=None):
        L = lib()
        self.shape = tuple(int(s) for s in shape)
        sh = (C.c_int * 3)(*self.shape)
        sp = (C.c_double * 3)(*(spacing if spacing is not None else (1.0, 1.0, 1.0)))
        og = (C.c_double * 3)(*(origin if origin is not None else (0.0, 0.0, 0.0)))
        bcs = (C.c_int * 6)(*[int(b) for b in bc])
        ed = None
        if edges is not None:
            self._edges = [(C.c_double * len(e))(*[float(x) for x in e]) for e in edges]
            ed = (C.POINTER(C.c_double) * 3)(*[C.cast(e, C.POINTER(C.c_double)) for e in self._edges])
        h = C.c_void_p(0)
        st = C.c_void_p(int(stream) if stream is not None else 0)
        rc = L.poisson_create(C.byref(h), sh, sp, og, ed, int(coord), int(order), bcs, st)
        if rc != OK:
            raise PoissonError(rc, L.poisson_last_error(None).decode())
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            lib().poisson_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc < 0:
            raise PoissonError(rc, lib().poisson_last_error(self.h).decode())
        return rc

    @property
    def size(self):
        return self.shape[0] * self.shape[1] * self.shape[2]

    def last_error(self):
        return lib().poisson_last_error(self.h).decode()

    def set_option(self, option, value):
        self._check(lib().poisson_set_option(self.h, int(option), int(value)))

    def set_option_f64(self, option, value):
        self._check(lib().poisson_set_option_f64(self.h, int(option), C.c_double(value)))

    def bicgstab_stats(self):
        """(near-breakdown restarts, failed true-residual confirmations) of the last BiCGSTAB solve."""
        a, b = C.c_int(0), C.c_int(0)
        self._check(lib().poisson_bicgstab_stats(self.h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def kernel_launches(self):
        return int(lib().poisson_kernel_launches(self.h))

    def kernel_class_launches(self):
        L = lib()
        return {n: int(L.poisson_kernel_class_launches(self.h, i)) for i, n in enumerate(kernel_classes())}

    def kernel_time(self, kernel_class):
        """(total ms, launches) of the event-timed launches of one class (set OPT_TIME_KERNELS first)."""
        ms, cnt = C.c_double(0.0), C.c_long(0)
        self._check(lib().poisson_kernel_time(self.h, int(kernel_class), C.byref(ms), C.byref(cnt)))
        return ms.value, cnt.value

    def reset_kernel_times(self):
        self._check(lib().poisson_reset_kernel_times(self.h))

    def face_len(self, f):
        return int(lib().poisson_face_len(self.h, int(f)))

    def apply_laplacian(self, d_phi, d_out):
        self._check(lib().poisson_apply_laplacian(self.h, _ptr(d_phi), _ptr(d_out)))

    def apply_laplacian_host(self, h_phi, h_out):
        self._check(lib().poisson_apply_laplacian_host(self.h, _ptr(h_phi), _ptr(h_out)))

    def residual_norm(self, d_phi, d_rhs):
        out = C.c_double(0.0)
        self._check(lib().poisson_residual_norm(self.h, _ptr(d_phi), _ptr(d_rhs), C.byref(out)))
        return out.value

    def rbsor_sweep(self, d_phi, d_rhs, omega, nsweeps, want_resnorm=False):
        out = C.c_double(0.0)
        self._check(lib().poisson_rbsor_sweep(self.h, _ptr(d_phi), _ptr(d_rhs), C.c_double(omega), int(nsweeps),
                                              C.byref(out) if want_resnorm else None))
        return out.value if want_resnorm else None

    def rbsor_sweep_host(self, h_phi, h_rhs, omega, nsweeps, want_resnorm=False):
        out = C.c_double(0.0)
        self._check(lib().poisson_rbsor_sweep_host(self.h, _ptr(h_phi), _ptr(h_rhs), C.c_double(omega), int(nsweeps),
                                                   C.byref(out) if want_resnorm else None))
        return out.value if want_resnorm else None

    def rbsor_cheby(self, d_phi, d_rhs, nsweeps, r_jacobi=0.0, start_n=1, want_resnorm=False):
        out = C.c_double(0.0)
        self._check(lib().poisson_rbsor_cheby(self.h, _ptr(d_phi), _ptr(d_rhs), C.c_double(r_jacobi), int(nsweeps),
                                              int(start_n), C.byref(out) if want_resnorm else None))
        return out.value if want_resnorm else None

    def rbsor_local(self, d_phi, d_rhs, nsweeps, start_n=1, want_resnorm=False):
        out = C.c_double(0.0)
        self._check(lib().poisson_rbsor_local(self.h, _ptr(d_phi), _ptr(d_rhs), int(nsweeps), int(start_n),
                                              C.byref(out) if want_resnorm else None))
        return out.value if want_resnorm else None

    def pcg_solve(self, d_phi, d_rhs, rtol=1e-8, max_iter=10000, fixed_iters=0):
        return self._krylov(lib().poisson_pcg_solve, d_phi, d_rhs, rtol, max_iter, fixed_iters)

    def multipole_inner_moments(self, lmax):
        buf = (C.c_double * ((lmax + 1) ** 2))()
        self._check(lib().poisson_multipole_inner_moments(self.h, buf, int(lmax)))
        return list(buf)

    def _krylov(self, fn, d_phi, d_rhs, rtol, max_iter, fixed_iters):
        it, rr = C.c_int(0), C.c_double(0.0)
        rc = self._check(fn(self.h, _ptr(d_phi), _ptr(d_rhs), C.c_double(rtol), int(max_iter), int(fixed_iters),
                            C.byref(it), C.byref(rr)))
        return dict(status=rc, iters=it.value, relres=rr.value)

    def cg_solve(self, d_phi, d_rhs, rtol=1e-8, max_iter=10000, fixed_iters=0):
        return self._krylov(lib().poisson_cg_solve, d_phi, d_rhs, rtol, max_iter, fixed_iters)

    def cg_solve_host(self, h_phi, h_rhs, rtol=1e-8, max_iter=10000, fixed_iters=0):
        return self._krylov(lib().poisson_cg_solve_host, h_phi, h_rhs, rtol, max_iter, fixed_iters)

    def bicgstab_solve(self, d_phi, d_rhs, rtol=1e-8, max_iter=10000, fixed_iters=0):
        return self._krylov(lib().poisson_bicgstab_solve, d_phi, d_rhs, rtol, max_iter, fixed_iters)

    def bicgstab_solve_host(self, h_phi, h_rhs, rtol=1e-8, max_iter=10000, fixed_iters=0):
        return self._krylov(lib().poisson_bicgstab_solve_host, h_phi, h_rhs, rtol, max_iter, fixed_iters)

    def get_history(self, n):
        buf = (C.c_double * n)()
        self._check(lib().poisson_get_history(self.h, buf, int(n)))
        return list(buf)

    def mg_vcycle(self, d_phi, d_rhs, nu1=2, nu2=2, coarsest_n=8, coarsest_sweeps=50, precision=F64, ncycles=1,
                  want_resnorms=True):
        buf = (C.c_double * (ncycles + 1))()
        rc = self._check(lib().poisson_mg_vcycle(self.h, _ptr(d_phi), _ptr(d_rhs), int(nu1), int(nu2),
                                                 int(coarsest_n), int(coarsest_sweeps), int(precision), int(ncycles),
                                                 buf if want_resnorms else None))
        return dict(status=rc, resnorms=list(buf) if want_resnorms else None)

    def mg_vcycle_host(self, h_phi, h_rhs, nu1=2, nu2=2, coarsest_n=8, coarsest_sweeps=50, precision=F64, ncycles=1,
                       want_resnorms=True):
        buf = (C.c_double * (ncycles + 1))()
        rc = self._check(lib().poisson_mg_vcycle_host(self.h, _ptr(h_phi), _ptr(h_rhs), int(nu1), int(nu2),
                                                      int(coarsest_n), int(coarsest_sweeps), int(precision),
                                                      int(ncycles), buf if want_resnorms else None))
        return dict(status=rc, resnorms=list(buf) if want_resnorms else None)

    def spai_smooth(self, d_phi, d_rhs, spai=None, nsteps=1):
        sp = (C.c_double * 5)(*spai) if spai is not None else None
        self._check(lib().poisson_spai_smooth(self.h, _ptr(d_phi), _ptr(d_rhs), sp, int(nsteps)))

    def compact_rhs(self, d_f_ext, d_out):
        self._check(lib().poisson_compact_rhs(self.h, _ptr(d_f_ext), _ptr(d_out)))

    def mgv_vcycle(self, d_phi, d_rhs, nu1=1, nu2=1, coarsest_n=3, spai=None, cg_rtol=1e-3, precision=F64, ncycles=1,
                   want_resnorms=True, _fn=None):
        sp = (C.c_double * 5)(*spai) if spai is not None else None
        buf = (C.c_double * (ncycles + 1))()
        fn = _fn or lib().poisson_mgv_vcycle
        rc = self._check(fn(self.h, _ptr(d_phi), _ptr(d_rhs), int(nu1), int(nu2), int(coarsest_n), sp,
                            C.c_double(cg_rtol), int(precision), int(ncycles), buf if want_resnorms else None))
        return dict(status=rc, resnorms=list(buf) if want_resnorms else None)

    def mgv_vcycle_host(self, h_phi, h_rhs, **kw):
        return self.mgv_vcycle(h_phi, h_rhs, _fn=lib().poisson_mgv_vcycle_host, **kw)

    def multipole_bc(self, d_rho, G, lmax, want_moments=True, _fn=None):
        nq = (lmax + 1) ** 2
        buf = (C.c_double * nq)()
        fn = _fn or lib().poisson_multipole_bc
        self._check(fn(self.h, _ptr(d_rho), C.c_double(G), int(lmax), buf if want_moments else None))
        return list(buf) if want_moments else None

    def multipole_bc_host(self, h_rho, G, lmax, want_moments=True):
        return self.multipole_bc(h_rho, G, lmax, want_moments, _fn=lib().poisson_multipole_bc_host)

    def set_ghost_faces(self, d_faces):
        arr = (C.c_void_p * 6)(*[_ptr(f) for f in d_faces])
        self._check(lib().poisson_set_ghost_faces(self.h, arr))

    def get_ghost_face(self, f, d_out):
        self._check(lib().poisson_get_ghost_face(self.h, int(f), _ptr(d_out)))
