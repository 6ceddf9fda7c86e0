"""Pins for the oracle's multipole boundary (oracle/multipole.cpp) — SURVEY.md §8(c) C6; Eq. 19-20."""
import math

import numpy as np
import pytest
from scipy.special import eval_legendre

import pyoracle as po
from helpers import make_oracle
from paper_2605_03563_b200 import workloads as wl

D6 = (po.BC_DIRICHLET_GHOST,) * 6


def _grid(n=9, h=0.25):
    # odd n: the centre cell sits at the origin
    o = -(n // 2) * h
    return po.Oracle((n, n, n), (h, h, h), origin=(o, o, o), bc=D6), n, h, o


def _point_mass(n, h, o, pos, M):
    rho = np.zeros((n, n, n))
    i, j, k = (int(round((p - o) / h)) for p in pos)
    rho[k, j, i] = M / h ** 3
    return rho


def test_point_mass_at_origin_has_only_monopole():
    g, n, h, o = _grid()
    q = g.multipole_moments(_point_mass(n, h, o, (0, 0, 0), 2.5), 6)
    assert q[0] == pytest.approx(2.5, rel=1e-14)
    assert np.abs(q[1:]).max() < 1e-15


def test_point_mass_on_z_axis():
    g, n, h, o = _grid()
    a, M, L = 0.75, 1.7, 8
    q = g.multipole_moments(_point_mass(n, h, o, (0, 0, a), M), L)
    for l in range(L + 1):
        for m in range(-l, l + 1):
            want = M * a ** l if m == 0 else 0.0
            assert q[l * l + l + m] == pytest.approx(want, rel=1e-13, abs=1e-15)


def test_sign_and_index_convention_cos_for_m_positive():
    # sine harmonics take m < 0, cosine harmonics m >= 0
    g, n, h, o = _grid()
    qx = g.multipole_moments(_point_mass(n, h, o, (0.5, 0, 0), 1.0), 2)
    qy = g.multipole_moments(_point_mass(n, h, o, (0, 0.5, 0), 1.0), 2)
    l1 = lambda m: 1 + 1 + m
    assert qx[l1(1)] == pytest.approx(0.5) and abs(qx[l1(-1)]) < 1e-16 and abs(qx[l1(0)]) < 1e-16
    assert qy[l1(-1)] == pytest.approx(0.5) and abs(qy[l1(1)]) < 1e-16
    # l = 2, on the x axis: r^2 S_22 = (sqrt(3)/2)(x^2 - y^2), r^2 S_20 = (2z^2-x^2-y^2)/2
    assert qx[4 + 2 + 2] == pytest.approx(math.sqrt(3) / 2 * 0.25)
    assert qx[4 + 2 + 0] == pytest.approx(-0.125)


def test_ghost_values_equal_truncated_legendre_sum_bruteforce():
    # addition theorem: sum_m S_lm(x) S_lm(x') = P_l(cos gamma), so Eq. 19-20 give
    #   Phi(x) = -G sum_cells rho dV sum_{l<=lmax} r'^l / r^{l+1} P_l(cos gamma), whatever the harmonic convention
    n, h = 8, 0.125
    org = -0.5 + h / 2
    w = dict(shape=(n, n, n), spacing=(h,) * 3, origin=(org,) * 3, bc=D6)
    o = make_oracle(w)
    rho = wl.random_field((n, n, n), 51, 0.0, 1.0)
    # keep the mass away from the boundary as the paper recommends
    rho[:2] = rho[-2:] = 0
    rho[:, :2] = rho[:, -2:] = 0
    rho[:, :, :2] = rho[:, :, -2:] = 0
    G, L = 1.3, 5
    o.multipole_bc(rho, G, L)
    x = org + h * np.arange(n)
    Xc, Yc, Zc = np.meshgrid(x, x, x, indexing="ij")  # any order: summed over all cells
    src = np.stack([Xc.ravel(), Yc.ravel(), Zc.ravel()], 1)
    m = (rho.transpose(2, 1, 0)).ravel() * h ** 3       # rho[k,j,i] -> [i,j,k] to match src
    rs = np.linalg.norm(src, axis=1)
    for f in range(6):
        got = o.get_ghost_face(f).reshape(n, n)
        a = f // 2
        a1, a2 = (1, 2) if a == 0 else ((0, 2) if a == 1 else (0, 1))
        for (q2, q1) in ((0, 0), (3, 5), (7, 2)):
            p = np.zeros(3)
            p[a] = org + h * (n if f & 1 else -1)
            p[a1], p[a2] = x[q1], x[q2]
            r = np.linalg.norm(p)
            cg = (src @ p) / (rs * r)
            want = -G * sum(np.sum(m * rs ** l * eval_legendre(l, cg)) / r ** (l + 1) for l in range(L + 1))
            assert got[q2, q1] == pytest.approx(want, rel=1e-12)


def test_large_lmax_tends_to_newton_sum():
    # the ideal boundary condition is the direct Newton sum; the expansion converges to it
    n, h = 8, 0.125
    org = -0.5 + h / 2
    o = po.Oracle((n, n, n), (h,) * 3, origin=(org,) * 3, bc=D6)
    rho = np.zeros((n, n, n))
    rho[3:5, 3:5, 2:5] = wl.random_field((3, 2, 2), 52, 0.5, 1.5)
    x = org + h * np.arange(n)
    p = np.array([org - h, x[2], x[5]])
    kk, jj, ii = np.nonzero(rho)
    newton = -sum(rho[k, j, i] * h ** 3 / np.linalg.norm(p - np.array([x[i], x[j], x[k]])) for k, j, i in zip(kk, jj, ii))
    errs = []
    for L in (2, 6, 12):
        q = o.multipole_moments(rho, L)
        errs.append(abs(po.multipole_potential(q, L, 1.0, *p) - newton) / abs(newton))
    assert errs[0] > errs[1] > errs[2] and errs[2] < 1e-6


def test_two_sphere_moments():
    # exterior multipoles of the paper's two-sphere set-up are those of two point masses,
    # q_l0 = 0.4^l + 2 (-0.2)^l, q_lm = 0 (m != 0), up to sampling error
    w = wl.two_spheres(64)
    o = make_oracle(w)
    q = o.multipole_moments(w["rho"], 4)
    for l in range(5):
        assert q[l * l + l] == pytest.approx(0.4 ** l + 2 * (-0.2) ** l, abs=2e-2)  # point sampling of a 2.5-cell-radius sphere
        for m in range(1, l + 1):
            assert abs(q[l * l + l + m]) < 2e-3 and abs(q[l * l + l - m]) < 2e-3


def test_spherical_grid_moments_of_uniform_shell():
    # exact cell volumes: a uniform-density spherical grid has q_00 = mass of the shell, everything else 0
    re, te, pe = wl.spherical_edges(16, 8, 16, 0.1, 1.0)
    bc = (po.BC_NEUMANN0, po.BC_DIRICHLET_GHOST, po.BC_AXIS, po.BC_AXIS, po.BC_PERIODIC, po.BC_PERIODIC)
    o = po.Oracle((16, 8, 16), edges=(re, te, pe), coord=po.SPHERICAL, bc=bc)
    q = o.multipole_bc(np.ones(o.npshape), 1.0, 4)
    M = 4 / 3 * math.pi * (1 - 0.1 ** 3)
    assert q[0] == pytest.approx(M, rel=1e-13)
    # odd-l moments vanish by the grid's mirror symmetry; even l > 0 only up to the midpoint rule in theta
    assert abs(q[2]) < 1e-13 * M and abs(q[1 + 1 + 1]) < 1e-13 * M
    ghost = o.get_ghost_face(1)
    assert np.allclose(ghost, -M / o.r_ghost_out(), rtol=2e-2)


def test_config2_ghosts_close_to_point_mass_potential():
    # SURVEY.md C6 probe: 1.2e-5 relative at 128^3 with lmax = 4; at 32^3 the sampled sphere is coarser
    w = wl.config2(32)
    o = make_oracle(w)
    o.multipole_bc(w["rho"], 1.0, 4)
    faces = wl.analytic_ghost_faces(w, lambda x, y, z: wl.uniform_sphere_potential(x, y, z, w["centre"], 0.25, 1.0))
    for f in range(6):
        assert np.abs(o.get_ghost_face(f) / faces[f] - 1).max() < 2e-3
