"""ORACLE — TEST INFRASTRUCTURE ONLY.  ctypes wrapper around oracle/liboracle.so (plain C++ CPU oracle).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from the CUDA package.
"""
import ctypes as C
import importlib.util
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))

CARTESIAN, SPHERICAL = 0, 1
BC_DIRICHLET_GHOST, BC_PERIODIC, BC_NEUMANN0, BC_AXIS = 0, 1, 2, 3

# PAPER.md:176-182 Table 1, row "Order 2": omega, alpha, beta, gamma, delta of the SPAI smoother (Eq. 15-16)
SPAI_ORDER2 = (1.3699, 0.1432, 0.0284, 0.0081, 0.0025)
# rows "Order 4" and "Order 6" (for the compact radius-1 discretisations of PAPER.md:172).  The delta of order 6 is
# printed as 0.0909, a copy of the mu column (reading C20): taken as 0.0150, the middle of the interval
# [0.0140, 0.0160] on which the local-Fourier smoothing factor of Eq. 17 is smallest with the other printed values.
SPAI_ORDER4 = (0.9363, 0.2807, 0.0329, 0.0166, 0.0044)
SPAI_ORDER6 = (0.3543, 0.7064, 0.1005, 0.0363, 0.0150)
SPAI = {2: SPAI_ORDER2, 4: SPAI_ORDER4, 6: SPAI_ORDER6}

_lib = None


def lib():
    global _lib
    if _lib is None:
        spec = importlib.util.spec_from_file_location("_oracle_build", os.path.join(_HERE, "build.py"))
        mod = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mod)
        _lib = C.CDLL(mod.build())
        _lib.orc_create.restype = C.c_void_p
        _lib.orc_residual_norm.restype = C.c_double
        _lib.orc_multipole_potential.restype = C.c_double
        _lib.orc_r_ghost_out.restype = C.c_double
        _lib.orc_face_len.restype = C.c_long
        _lib.orc_jacobi_radius.restype = C.c_double
        _lib.orc_local_jacobi_radius.restype = C.c_double
        _lib.orc_multipole_inner_potential.restype = C.c_double
    return _lib


def _p(a, ct=C.c_double):
    return a.ctypes.data_as(C.POINTER(ct)) if a is not None else None


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def set_threads(n):
    lib().orc_set_threads(int(n))


def get_threads():
    return int(lib().orc_get_threads())


class Oracle:
    """One grid + operator.  Arrays are numpy, shape (nz, ny, nx) i.e. axis 0 of the method is the last numpy axis."""

    def __init__(self, shape, spacing=None, origin=None, edges=None, coord=CARTESIAN, order=2, bc=(0,) * 6):
        L = lib()
        self.shape = tuple(int(s) for s in shape)  # (n0, n1, n2), n0 fastest
        self.npshape = self.shape[::-1]
        self.coord, self.order = coord, order
        self.bc = tuple(int(b) for b in bc)
        sh = (C.c_int * 3)(*self.shape)
        sp = (C.c_double * 3)(*(spacing if spacing is not None else (1.0, 1.0, 1.0)))
        og = (C.c_double * 3)(*(origin if origin is not None else (0.0, 0.0, 0.0)))
        self.spacing = tuple(sp)
        self.origin = tuple(og)
        bcs = (C.c_int * 6)(*self.bc)
        if edges is not None:
            self._edges = [_f64(e) for e in edges]
            ed = (C.POINTER(C.c_double) * 3)(*[_p(e) for e in self._edges])
        else:
            ed = None
        self.h = C.c_void_p(L.orc_create(sh, sp, og, ed, coord, order, bcs))

    def __del__(self):
        try:
            if self.h:
                lib().orc_destroy(self.h)
                self.h = None
        except Exception:
            pass

    @property
    def size(self):
        return self.shape[0] * self.shape[1] * self.shape[2]

    def set_gamma(self, gamma):
        lib().orc_set_gamma(self.h, C.c_double(gamma))

    def face_len(self, f):
        return int(lib().orc_face_len(self.h, f))

    def set_ghost_face(self, f, v):
        v = _f64(v).ravel()
        assert v.size == self.face_len(f)
        lib().orc_set_ghost_face(self.h, f, _p(v))

    def get_ghost_face(self, f):
        v = np.zeros(self.face_len(f))
        lib().orc_get_ghost_face(self.h, f, _p(v))
        return v

    def apply(self, phi, use_ghost=True):
        phi = _f64(phi)
        out = np.empty_like(phi)
        lib().orc_apply(self.h, _p(phi), _p(out), int(use_ghost))
        return out

    def apply_f32(self, phi, use_ghost=True):
        phi = np.ascontiguousarray(phi, dtype=np.float32)
        out = np.empty_like(phi)
        lib().orc_apply_f32(self.h, _p(phi, C.c_float), _p(out, C.c_float), int(use_ghost))
        return out

    def diag(self):
        out = np.empty(self.npshape)
        lib().orc_diag(self.h, _p(out))
        return out

    def residual_norm(self, phi, rhs):
        phi, rhs = _f64(phi), _f64(rhs)
        return float(lib().orc_residual_norm(self.h, _p(phi), _p(rhs)))

    def rbsor_half(self, phi, rhs, omega, colour):
        """In place on phi (must be a contiguous float64 array)."""
        assert phi.dtype == np.float64 and phi.flags.c_contiguous
        rhs = _f64(rhs)
        lib().orc_rbsor_half(self.h, _p(phi), _p(rhs), C.c_double(omega), int(colour))

    def rbsor(self, phi, rhs, omega, nsweeps, want_resnorm=False):
        assert phi.dtype == np.float64 and phi.flags.c_contiguous
        rhs = _f64(rhs)
        rn = C.c_double(0.0)
        lib().orc_rbsor(self.h, _p(phi), _p(rhs), C.c_double(omega), int(nsweeps),
                        C.byref(rn) if want_resnorm else None)
        return rn.value if want_resnorm else None

    def rbsor_f32(self, phi, rhs, omega, nsweeps):
        assert phi.dtype == np.float32 and phi.flags.c_contiguous
        rhs = np.ascontiguousarray(rhs, dtype=np.float32)
        lib().orc_rbsor_f32(self.h, _p(phi, C.c_float), _p(rhs, C.c_float), C.c_float(omega), int(nsweeps))

    def _krylov(self, fn, phi, rhs, rtol, max_iter, fixed_iters, want_history, extra=()):
        assert phi.dtype == np.float64 and phi.flags.c_contiguous
        rhs = _f64(rhs)
        iters, relres = C.c_int(0), C.c_double(0.0)
        nh = (fixed_iters if fixed_iters > 0 else max_iter) + 1
        hist = np.zeros(nh) if want_history else None
        st = fn(self.h, _p(phi), _p(rhs), C.c_double(rtol), int(max_iter), int(fixed_iters), *extra,
                C.byref(iters), C.byref(relres), _p(hist))
        out = dict(status=int(st), iters=iters.value, relres=relres.value)
        if want_history:
            out["history"] = hist[: iters.value + 1]
        return out

    def cg(self, phi, rhs, rtol=1e-8, max_iter=10000, fixed_iters=0, want_history=False):
        return self._krylov(lib().orc_cg, phi, rhs, rtol, max_iter, fixed_iters, want_history)

    def bicgstab(self, phi, rhs, rtol=1e-8, max_iter=10000, fixed_iters=0, jacobi=1, want_history=False):
        return self._krylov(lib().orc_bicgstab, phi, rhs, rtol, max_iter, fixed_iters, want_history,
                            extra=(int(jacobi),))

    def pcg(self, phi, rhs, rtol=1e-8, max_iter=10000, fixed_iters=0, want_history=False):
        """CG preconditioned by the symmetrised red-black Gauss-Seidel sweep (row f3)."""
        return self._krylov(lib().orc_pcg, phi, rhs, rtol, max_iter, fixed_iters, want_history)

    def gs_precond(self, v, sign=-1, symmetric=True):
        v = _f64(v)
        z = np.zeros_like(v)
        lib().orc_gs_precond(self.h, _p(v), _p(z), int(sign), int(bool(symmetric)))
        return z

    def jacobi_radius(self):
        return float(lib().orc_jacobi_radius(self.h))

    def local_jacobi_radius(self, i, j):
        return float(lib().orc_local_jacobi_radius(self.h, int(i), int(j)))

    def rbsor_cheby(self, phi, rhs, nsweeps, rJ=None, start_n=1):
        """Chebyshev-accelerated omega sequence (Eq. 6), one omega per colour half-sweep; returns the omegas used."""
        assert phi.dtype == np.float64 and phi.flags.c_contiguous
        rhs = _f64(rhs)
        om = np.zeros(2 * nsweeps)
        rJ = self.jacobi_radius() if rJ is None else rJ
        lib().orc_rbsor_cheby(self.h, _p(phi), _p(rhs), C.c_double(rJ), int(nsweeps), int(start_n), _p(om))
        return om

    def rbsor_local(self, phi, rhs, nsweeps, start_n=1):
        assert phi.dtype == np.float64 and phi.flags.c_contiguous
        rhs = _f64(rhs)
        lib().orc_rbsor_local(self.h, _p(phi), _p(rhs), int(nsweeps), int(start_n))

    def multipole_bc2(self, rho, G, lmax):
        """(outer moments, inner moments): fills the outer and — on a spherical grid with a Dirichlet inner face — the
        inner ghost shell (Eq. 19-22)."""
        rho = _f64(rho)
        q, qb = np.zeros((lmax + 1) ** 2), np.zeros((lmax + 1) ** 2)
        lib().orc_multipole_bc2(self.h, _p(rho), C.c_double(G), int(lmax), _p(q), _p(qb))
        return q, qb

    def multipole_inner_moments(self, rho, lmax):
        rho = _f64(rho)
        q = np.zeros((lmax + 1) ** 2)
        lib().orc_multipole_inner_moments(self.h, _p(rho), int(lmax), _p(q))
        return q

    @staticmethod
    def set_bicgstab_restart_eps(eps):
        """Near-breakdown threshold of BiCGSTAB (default 1e-12); tests raise it to force the restart branch."""
        fn = lib().orc_set_bicgstab_restart_eps
        fn.argtypes = [C.c_double]
        fn.restype = None
        fn(float(eps))

    @staticmethod
    def bicgstab_stats():
        """(restarts, failed true-residual confirmations) of the last bicgstab call."""
        a, b = C.c_int(0), C.c_int(0)
        lib().orc_bicgstab_stats(C.byref(a), C.byref(b))
        return a.value, b.value

    def vcycle(self, phi, rhs, nu1=2, nu2=2, coarsest_n=8, coarsest_sweeps=50, precision=0, restriction=0,
               ncycles=1):
        assert phi.dtype == np.float64 and phi.flags.c_contiguous
        rhs = _f64(rhs)
        rn = np.zeros(ncycles + 1)
        st = lib().orc_vcycle(self.h, _p(phi), _p(rhs), int(nu1), int(nu2), int(coarsest_n), int(coarsest_sweeps),
                              int(precision), int(restriction), int(ncycles), _p(rn))
        return dict(status=int(st), resnorms=rn)

    def restrict(self, r, restriction=0):
        r = _f64(r)
        fc = np.zeros(tuple(s // 2 for s in self.npshape))
        lib().orc_restrict(self.h, _p(r), _p(fc), int(restriction))
        return fc

    def prolong_add(self, ec, phi, coarse_gamma):
        assert phi.dtype == np.float64 and phi.flags.c_contiguous
        ec = _f64(ec)
        lib().orc_prolong_add(self.h, _p(ec), _p(phi), C.c_double(coarse_gamma))

    # ---- the paper's own multigrid (oracle/mgv.cpp) ----
    def spai_smooth(self, phi, rhs, spai=None, nsteps=1, order=2):
        """order 4 / 6: the compact operator, zero boundary values, rhs = compact_rhs(...) (oracle/mgv.cpp)."""
        assert phi.dtype == np.float64 and phi.flags.c_contiguous
        rhs, sp = _f64(rhs), _f64(np.array(SPAI[order] if spai is None else spai))
        lib().orc_spai_smooth(self.h, _p(phi), _p(rhs), _p(sp), int(nsteps), int(order))

    def mgv_vcycle(self, phi, rhs, nu1=1, nu2=1, coarsest_n=3, spai=None, cg_rtol=1e-3, storage_f32=False,
                   ncycles=1, order=2):
        assert phi.dtype == np.float64 and phi.flags.c_contiguous
        rhs, sp = _f64(rhs), _f64(np.array(SPAI[order] if spai is None else spai))
        rn = np.zeros(ncycles + 1)
        fn = lib().orc_mgv_vcycle
        fn.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_double, C.c_int,
                       C.c_int, C.c_void_p, C.c_int]
        st = fn(self.h, phi.ctypes.data, rhs.ctypes.data, int(nu1), int(nu2), int(coarsest_n), sp.ctypes.data,
                float(cg_rtol), int(bool(storage_f32)), int(ncycles), rn.ctypes.data, int(order))
        return dict(status=int(st), resnorms=rn)

    def compact_apply(self, v, order):
        """L_h v with the compact radius-1 Laplacian of the given order, zero values outside the grid."""
        v = _f64(v)
        out = np.zeros_like(v)
        rc = lib().orc_compact_apply(self.h, int(order), _p(v), _p(out))
        assert rc == 0
        return out

    def mgv_galerkin_stencil(self, level, I, J, K, order=2):
        out = np.zeros(27)
        rc = lib().orc_mgv_galerkin_stencil(self.h, int(level), int(I), int(J), int(K), _p(out), int(order))
        assert rc == 0
        return out.reshape(3, 3, 3)

    def mgv_restrict(self, r):
        r = _f64(r)
        bc = np.zeros(tuple((s - 1) // 2 for s in self.npshape))
        lib().orc_mgv_restrict(self.h, _p(r), _p(bc))
        return bc

    def mgv_prolong_add(self, ec, x):
        assert x.dtype == np.float64 and x.flags.c_contiguous
        ec = _f64(ec)
        lib().orc_mgv_prolong_add(self.h, _p(ec), _p(x))

    def multipole_moments(self, rho, lmax):
        rho = _f64(rho)
        q = np.zeros((lmax + 1) ** 2)
        lib().orc_multipole_moments(self.h, _p(rho), int(lmax), _p(q))
        return q

    def multipole_bc(self, rho, G, lmax):
        rho = _f64(rho)
        q = np.zeros((lmax + 1) ** 2)
        lib().orc_multipole_bc(self.h, _p(rho), C.c_double(G), int(lmax), _p(q))
        return q

    def centres(self, axis):
        out = np.zeros(self.shape[axis])
        lib().orc_centres(self.h, int(axis), _p(out))
        return out

    def r_ghost_out(self):
        return float(lib().orc_r_ghost_out(self.h))


def compact_rhs(f_ext, order):
    """B f of the compact scheme of the given order (oracle/mgv.cpp compact_rhs): f_ext carries two extra layers per side
    (numpy shape (n2+4, n1+4, n0+4)); returns shape (n2, n1, n0)."""
    f_ext = _f64(f_ext)
    n = (C.c_int * 3)(f_ext.shape[2] - 4, f_ext.shape[1] - 4, f_ext.shape[0] - 4)
    out = np.zeros((f_ext.shape[0] - 4, f_ext.shape[1] - 4, f_ext.shape[2] - 4))
    fn = lib().orc_compact_rhs
    fn.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
    rc = fn(n, int(order), f_ext.ctypes.data, out.ctypes.data)
    assert rc == 0
    return out


def multipole_inner_potential(qbar, lmax, G, x, y, z):
    qbar = _f64(qbar)
    return float(lib().orc_multipole_inner_potential(_p(qbar), int(lmax), C.c_double(G), C.c_double(x), C.c_double(y),
                                                     C.c_double(z)))


def multipole_potential(q, lmax, G, x, y, z):
    q = _f64(q)
    return float(lib().orc_multipole_potential(_p(q), int(lmax), C.c_double(G), C.c_double(x), C.c_double(y),
                                               C.c_double(z)))
