"""Pins for the oracle's stencil apply (oracle/grid.hpp, oracle/apply.cpp) — SURVEY.md §8(c) C1, C5."""
import math

import numpy as np
import pytest

import pyoracle as po
from helpers import dense_matrix, make_oracle
from paper_2605_03563_b200 import workloads as wl

D6 = (po.BC_DIRICHLET_GHOST,) * 6
P6 = (po.BC_PERIODIC,) * 6


def test_7pt_sine_is_eigenvector():
    # PAPER.md:43-45 Eq. 1 discretised with second differences: sin(pi x)sin(pi y)sin(pi z) on the vertex grid is an
    # exact eigenvector with eigenvalue -(12/h^2) sin^2(pi h/2).
    w = wl.config1(16)
    o = make_oracle(w)
    h = w["spacing"][0]
    lam = -(12.0 / h ** 2) * math.sin(math.pi * h / 2) ** 2
    out = o.apply(w["exact"])
    assert np.abs(out - lam * w["exact"]).max() <= 1e-12 * abs(lam)


def test_7pt_quadratic_exact_with_anisotropic_spacing_and_ghosts():
    # a transposed spacing or a mis-placed ghost face fails this: L(a x^2 + b y^2 + c z^2 + xy + z) = 2(a+b+c)
    shape, h, org = (7, 5, 6), (0.1, 0.25, 0.4), (0.3, -0.2, 1.0)
    w = dict(shape=shape, spacing=h, origin=org, bc=D6)
    o = make_oracle(w)
    f = lambda x, y, z: 1.5 * x * x - 2.0 * y * y + 0.7 * z * z + x * y + z
    X, Y, Z = wl._mesh(shape, org, h)
    faces = wl.analytic_ghost_faces(w, f)
    for k in range(6):
        o.set_ghost_face(k, faces[k])
    out = o.apply(np.ascontiguousarray(f(X, Y, Z) + 0 * (X + Y + Z)))
    assert np.abs(out - 2 * (1.5 - 2.0 + 0.7)).max() < 1e-10


def test_7pt_symmetric_negative_definite_dense_8cubed():
    o = po.Oracle((8, 8, 8), (0.1, 0.1, 0.1), bc=D6)
    A = dense_matrix(o)
    assert np.abs(A - A.T).max() == 0.0
    ev = np.linalg.eigvalsh(A)
    assert ev.max() < 0
    # closed-form spectrum of the Dirichlet second-difference operator
    lam1 = -(4 / 0.01) * math.sin(math.pi / 18) ** 2
    assert abs(ev.max() - 3 * lam1) < 1e-9 * abs(lam1)


def test_7pt_inner_product_symmetry_random():
    shape = (12, 9, 10)
    o = po.Oracle(shape, (0.2, 0.3, 0.5), bc=D6)
    u, v = wl.random_field(shape, 1), wl.random_field(shape, 2)
    a, b = np.vdot(u, o.apply(v, use_ghost=False)), np.vdot(o.apply(u, use_ghost=False), v)
    assert abs(a - b) <= 1e-13 * abs(a)


@pytest.mark.parametrize("n", [16, 32, 64])
def test_19pt_periodic_fourier_symbol(n):
    # textbook 6th-order central second difference (PAPER.md:172 names only the radius): symbol
    # (-49/18 + 3 cos t - (3/10) cos 2t + (1/45) cos 3t)/h^2, t = 2 pi k/n
    h = 1.0 / n
    o = po.Oracle((n, n, n), (h, h, h), order=6, bc=P6)
    x = h * np.arange(n)
    for (kx, ky, kz) in ((1, 0, 0), (0, 2, 0), (1, 2, 3)):
        u = np.cos(2 * math.pi * (kx * x[None, None, :] + ky * x[None, :, None] + kz * x[:, None, None]))
        sym = sum((-49 / 18 + 3 * math.cos(t) - 0.3 * math.cos(2 * t) + math.cos(3 * t) / 45) / h ** 2
                  for t in (2 * math.pi * kx / n, 2 * math.pi * ky / n, 2 * math.pi * kz / n))
        out = o.apply(np.ascontiguousarray(u))
        assert np.abs(out - sym * u).max() <= 1e-11 * abs(sym)


def test_19pt_sixth_order_convergence():
    errs = []
    for n in (32, 64, 128):
        h = 1.0 / n
        t = 2 * math.pi / n
        sym = (-49 / 18 + 3 * math.cos(t) - 0.3 * math.cos(2 * t) + math.cos(3 * t) / 45) / h ** 2
        errs.append(abs(sym / (-(2 * math.pi) ** 2) - 1))
    # SURVEY.md C1 probe values 1.02e-7, 1.60e-9, 2.49e-11 (64x per doubling)
    assert errs[0] == pytest.approx(1.02e-7, rel=0.02)
    assert errs[0] / errs[1] == pytest.approx(64, rel=0.03)
    assert errs[1] / errs[2] == pytest.approx(64, rel=0.05)


def test_19pt_dirichlet_three_ghost_layers_polynomial_exact():
    # degree <= 7 polynomials are differentiated exactly by the radius-3 stencil; needs all three ghost layers
    shape, h, org = (6, 7, 5), (0.1, 0.2, 0.15), (0.05, -0.3, 0.2)
    w = dict(shape=shape, spacing=h, origin=org, bc=D6, order=6)
    o = make_oracle(w)
    f = lambda x, y, z: x ** 6 - 2 * y ** 5 + 0.5 * z ** 4 + x * y * z
    lap = lambda x, y, z: 30 * x ** 4 - 40 * y ** 3 + 6 * z ** 2
    faces = wl.analytic_ghost_faces(w, f, R=3)
    for k in range(6):
        o.set_ghost_face(k, faces[k])
    X, Y, Z = wl._mesh(shape, org, h)
    out = o.apply(np.ascontiguousarray(f(X, Y, Z)))
    assert np.abs(out - lap(X, Y, Z)).max() < 1e-9


def test_19pt_symmetric_dense():
    o = po.Oracle((8, 8, 8), (0.1, 0.1, 0.1), order=6, bc=P6)
    A = dense_matrix(o)
    assert np.abs(A - A.T).max() < 1e-12
    assert np.abs(A.sum(axis=1)).max() < 1e-10  # constants are the null space


# ---- spherical operator (SURVEY.md C5 pins) -------------------------------------------------------------------------
def _sph(nr=32, nt=16, nph=32):
    re, te, pe = wl.spherical_edges(nr, nt, nph)
    bc = (po.BC_NEUMANN0, po.BC_DIRICHLET_GHOST, po.BC_AXIS, po.BC_AXIS, po.BC_PERIODIC, po.BC_PERIODIC)
    return po.Oracle((nr, nt, nph), edges=(re, te, pe), coord=po.SPHERICAL, bc=bc), (re, te, pe)


def test_spherical_volume_scaled_operator_is_symmetric():
    o, (re, te, pe) = _sph(8, 4, 8)
    A = dense_matrix(o)
    rc = np.sqrt(re[:-1] * re[1:])
    V = (rc ** 2 * np.diff(re))[None, None, :] * np.sin(0.5 * (te[:-1] + te[1:]))[None, :, None] * np.ones((8, 1, 1))
    VA = V.reshape(-1)[:, None] * A
    assert np.abs(VA - VA.T).max() <= 1e-13 * np.abs(VA).max()
    assert np.abs(A - A.T).max() > 1e-3 * np.abs(A).max()  # and L itself is not symmetric


def test_spherical_constants_and_one_over_r():
    o, (re, te, pe) = _sph()
    nr = 32
    one = np.ones(o.npshape)
    out = o.apply(one, use_ghost=False)
    scale = np.abs(o.diag())
    assert np.abs(out[:, :, : nr - 1] / scale[:, :, : nr - 1]).max() < 1e-14  # rows not touching the outer ghost
    # 1/r is discretely harmonic on rows i >= 1: face radius = geometric mean of neighbouring centres
    rc = o.centres(0)
    u = np.ascontiguousarray(np.broadcast_to(1.0 / rc[None, None, :], o.npshape))
    o.set_ghost_face(1, np.full(o.face_len(1), 1.0 / o.r_ghost_out()))
    out = o.apply(u)
    assert np.abs(out[:, :, 1:] / (scale[:, :, 1:] * u[:, :, 1:])).max() < 5e-14


def test_spherical_second_order_on_r_cos_theta():
    errs = []
    for (nr, nt, nph) in ((32, 16, 32), (64, 32, 64)):
        o, _ = _sph(nr, nt, nph)
        rc, tc = o.centres(0), o.centres(1)
        u = np.ascontiguousarray(np.broadcast_to(rc[None, None, :] * np.cos(tc)[None, :, None], o.npshape))
        o.set_ghost_face(1, np.ascontiguousarray(
            np.broadcast_to(o.r_ghost_out() * np.cos(tc)[None, :], (nph, nt))).ravel())
        out = o.apply(u)  # z is harmonic: L z = 0 up to truncation
        rel = np.abs(out[:, :, 1:]) * rc[None, None, 1:]  # the terms of L(r cos th) are of size 2 cos(th)/r
        errs.append(rel.max())
    assert errs[0] < 3e-2
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.1)


# ---- Cartesian zero-flux (Neumann) faces: the diagonal modification of oracle/grid.hpp diag() -------------------------
N6 = (po.BC_NEUMANN0,) * 6


def test_7pt_all_neumann_box_annihilates_constants_and_has_cosine_eigenvectors():
    # PAPER.md:43-45 Eq. 1 with zero normal flux through every face (cell-centred: the mirror ghost equals the adjacent
    # interior value, which removes one off-diagonal coefficient and lowers the diagonal by the same amount).  Then
    # every row sums to zero (L 1 = 0 on ALL rows, faces/edges/corners included) and cos(m pi (i+1/2)/n) per axis is an
    # exact eigenvector with eigenvalue -(4/h^2) sin^2(m pi/(2n)) (textbook DCT-II spectrum).  Dropping the `d -= c`
    # on a face breaks both on that face's rows.
    shape, h = (9, 6, 7), (0.2, 0.35, 0.15)
    o = po.Oracle(shape, h, bc=N6)
    out = o.apply(np.ones(o.npshape), use_ghost=False)
    assert np.abs(out).max() <= 1e-12 * 2 * sum(1 / s ** 2 for s in h)
    for m in ((1, 0, 0), (0, 2, 0), (0, 0, 3), (2, 1, 4), (8, 5, 6)):
        cx = np.cos(m[0] * math.pi * (np.arange(shape[0]) + 0.5) / shape[0])
        cy = np.cos(m[1] * math.pi * (np.arange(shape[1]) + 0.5) / shape[1])
        cz = np.cos(m[2] * math.pi * (np.arange(shape[2]) + 0.5) / shape[2])
        u = np.ascontiguousarray(cz[:, None, None] * cy[None, :, None] * cx[None, None, :])
        lam = -sum((4 / h[a] ** 2) * math.sin(m[a] * math.pi / (2 * shape[a])) ** 2 for a in range(3))
        assert np.abs(o.apply(u, use_ghost=False) - lam * u).max() <= 1e-12 * 2 * sum(1 / s ** 2 for s in h)


def test_7pt_mixed_neumann_dirichlet_faces_dense_matrix():
    # one Neumann face per axis (low x, high y, low z), ghost-Dirichlet on the others: still symmetric, and per axis the
    # matrix is tridiag(1,-2,1)/h^2 with one -1 corner (mirror ghost on one side, ghost value at distance h on the
    # other), whose eigenvalues are -(4/h^2) sin^2((2m+1) pi / (2(2n+1))), m = 0..n-1 (textbook Neumann-Dirichlet second
    # difference).  The 3-D spectrum is the sum over the axes.
    shape, h = (5, 4, 6), (0.3, 0.2, 0.25)
    bc = (po.BC_NEUMANN0, po.BC_DIRICHLET_GHOST, po.BC_DIRICHLET_GHOST, po.BC_NEUMANN0, po.BC_NEUMANN0,
          po.BC_DIRICHLET_GHOST)
    o = po.Oracle(shape, h, bc=bc)
    A = dense_matrix(o)
    assert np.abs(A - A.T).max() == 0.0
    ev = np.sort(np.linalg.eigvalsh(A))
    ax = [np.array([-(4 / h[a] ** 2) * math.sin((2 * m + 1) * math.pi / (2 * (2 * shape[a] + 1))) ** 2
                    for m in range(shape[a])]) for a in range(3)]
    want = np.sort((ax[2][:, None, None] + ax[1][None, :, None] + ax[0][None, None, :]).ravel())
    assert np.abs(ev - want).max() <= 1e-11 * np.abs(want).max()
