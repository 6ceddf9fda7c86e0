"""Pins for the oracle's multigrid V-cycle (oracle/vcycle.cpp) — SURVEY.md §8(c) C7."""
import math

import numpy as np
import pytest

import pyoracle as po
from helpers import dense_matrix, make_oracle, rel_l2
from paper_2605_03563_b200 import workloads as wl

D6 = (po.BC_DIRICHLET_GHOST,) * 6


def test_restriction_and_prolongation_preserve_constants():
    o = po.Oracle((16, 16, 16), (0.1,) * 3, bc=D6)
    one_f = np.ones(o.npshape)
    fc = o.restrict(one_f)
    assert np.abs(fc[1:-1, 1:-1, 1:-1] - 1).max() < 1e-15     # R 1 = 1 away from the boundary (Eq. 13 normalisation)
    assert fc[0, 0, 0] == pytest.approx((7 / 8) ** 3)          # one out-of-range residual per axis at a corner
    mean = o.restrict(one_f, restriction=1)
    assert np.abs(mean - 1).max() < 1e-15
    phi = np.zeros(o.npshape)
    o.prolong_add(np.ones((8, 8, 8)), phi, coarse_gamma=0.0)
    assert np.abs(phi[2:-2, 2:-2, 2:-2] - 1).max() < 1e-15    # P 1 = 1 ("P preserves constant functions")
    phi = np.zeros(o.npshape)
    o.prolong_add(np.ones((8, 8, 8)), phi, coarse_gamma=1 / 3)
    # level-1 closure: the interpolant vanishes at the finest ghost centre; first fine cell = 3/4 + 1/4 (-1/3)
    assert phi[5, 5, 0] == pytest.approx(0.75 - 0.25 / 3)


def test_prolongation_is_eight_times_restriction_transpose():
    o = po.Oracle((12, 8, 10), (0.1,) * 3, bc=D6)
    u = wl.random_field((6, 4, 5), 21)
    v = wl.random_field((12, 8, 10), 22)
    Pu = np.zeros(o.npshape)
    o.prolong_add(u, Pu, coarse_gamma=0.0)
    lhs, rhs = np.vdot(Pu, v), 8 * np.vdot(u, o.restrict(v))
    assert abs(lhs - rhs) <= 1e-13 * abs(lhs)


def test_prolongation_is_trilinear():
    # a linear function sampled at coarse cell centres is reproduced at fine cell centres (interior)
    o = po.Oracle((16, 16, 16), (0.1,) * 3, origin=(0.05,) * 3, bc=D6)
    xc = 0.1 + 0.2 * np.arange(8)
    xf = 0.05 + 0.1 * np.arange(16)
    lin = lambda x, y, z: 1 + 2 * x - 3 * y + 0.5 * z
    ec = lin(xc[None, None, :], xc[None, :, None], xc[:, None, None])
    phi = np.zeros(o.npshape)
    o.prolong_add(ec, phi, coarse_gamma=0.0)
    ex = lin(xf[None, None, :], xf[None, :, None], xf[:, None, None])
    assert np.abs(phi - ex)[1:-1, 1:-1, 1:-1].max() < 1e-14


def test_two_level_cycle_equals_dense_two_grid_operator():
    # error propagation of one V(1,1) cycle 8^3 -> 4^3 with an exact coarse solve:
    #   E = S (I - P A_c^-1 R A_f) S   (Eq. 11 with E_{N} = A_N^-1, Eq. 12)
    nf = 8
    h = 2.0 / nf
    of = po.Oracle((nf,) * 3, (h,) * 3, origin=(-1 + h / 2,) * 3, bc=D6)
    oc = po.Oracle((nf // 2,) * 3, (2 * h,) * 3, origin=(-1 + h,) * 3, bc=D6)
    oc.set_gamma(1 / 3)
    Af, Ac = dense_matrix(of), dense_matrix(oc)
    N, Nc = nf ** 3, (nf // 2) ** 3
    R = np.zeros((Nc, N))
    P = np.zeros((N, Nc))
    S = np.zeros((N, N))
    e = np.zeros(of.npshape)
    for c in range(N):
        e.reshape(-1)[c] = 1
        R[:, c] = of.restrict(e).reshape(-1)
        s = e.copy()
        of.rbsor(s, np.zeros_like(s), 1.0, 1)   # homogeneous GS sweep = error propagation of the smoother
        S[:, c] = s.reshape(-1)
        e.reshape(-1)[c] = 0
    ec = np.zeros(oc.npshape)
    for c in range(Nc):
        ec.reshape(-1)[c] = 1
        p = np.zeros(of.npshape)
        of.prolong_add(ec, p, coarse_gamma=1 / 3)
        P[:, c] = p.reshape(-1)
        ec.reshape(-1)[c] = 0
    E = S @ (np.eye(N) - P @ np.linalg.solve(Ac, R @ Af)) @ S
    rhs = wl.random_field((nf,) * 3, 31)
    exact = np.linalg.solve(Af, rhs.reshape(-1))
    phi0 = wl.random_field((nf,) * 3, 32)
    phi = phi0.copy()
    of.vcycle(phi, rhs, nu1=1, nu2=1, coarsest_n=4, coarsest_sweeps=400, ncycles=1)
    err_expected = E @ (phi0.reshape(-1) - exact)
    assert np.abs((phi.reshape(-1) - exact) - err_expected).max() <= 1e-12 * np.abs(exact).max()
    assert max(abs(np.linalg.eigvals(E))) < 0.25


def _blob_problem(n):
    w = wl.config3(n)
    o = make_oracle(w)
    X, Y, Z = wl._mesh(w["shape"], w["origin"], w["spacing"])

    def pot(x, y, z):
        from scipy.special import erf
        out = 0.0
        for (c, sg, amp) in w["blobs"]:
            d = np.sqrt((x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2)
            out = out - amp * (2 * math.pi) ** 1.5 * sg ** 3 * erf(d / (math.sqrt(2) * sg)) / d
        return out

    for k, fa in enumerate(wl.analytic_ghost_faces(w, pot)):
        o.set_ghost_face(k, fa)
    return w, o


def test_vcycle_factors_grid_independent_and_second_order():
    factors, errs = {}, {}
    for n in (32, 64):
        w, o = _blob_problem(n)
        phi = np.zeros_like(w["rhs"])
        res = o.vcycle(phi, w["rhs"], ncycles=8)["resnorms"]
        ratios = res[1:] / res[:-1]
        assert np.all(ratios < 0.2)          # SURVEY.md C7 probe: 0.058 -> 0.149 with the gamma closure
        factors[n] = (res[-1] / res[0]) ** (1 / 8)   # mean convergence rate, Eq. 18
        errs[n] = rel_l2(phi, w["exact"])
    assert factors[64] == pytest.approx(factors[32], rel=0.25)
    assert errs[32] / errs[64] == pytest.approx(4.0, rel=0.15)   # O(h^2) against the erf potential
    assert errs[32] == pytest.approx(1.5e-3, rel=0.5)            # SURVEY.md §8(d) probe (different RNG)


def test_mixed_precision_tracks_fp64():
    w, o = _blob_problem(32)
    a, b = np.zeros_like(w["rhs"]), np.zeros_like(w["rhs"])
    ra = o.vcycle(a, w["rhs"], ncycles=8)["resnorms"]
    rb = o.vcycle(b, w["rhs"], ncycles=8, precision=1)["resnorms"]
    assert np.allclose(rb[1:6] / rb[0], ra[1:6] / ra[0], rtol=0.05)
    assert rel_l2(b, a) < 1e-6


def test_vcycle_fixed_point_is_discrete_solution():
    n = 8
    h = 2.0 / n
    o = po.Oracle((n,) * 3, (h,) * 3, origin=(-1 + h / 2,) * 3, bc=D6)
    rhs = wl.random_field((n,) * 3, 41)
    exact = np.linalg.solve(dense_matrix(o), rhs.reshape(-1)).reshape(rhs.shape)
    for restriction in (0, 1):
        phi = np.zeros_like(rhs)
        o.vcycle(phi, rhs, coarsest_n=4, coarsest_sweeps=50, restriction=restriction, ncycles=25)
        assert rel_l2(phi, exact) < 1e-12


def test_coarsest_level_sor_uses_omega_opt_of_the_8cubed_operator():
    # DESIGN.md reading C7 / PAPER.md:65-76 Eq. 3-4: the coarsest level is solved by SOR sweeps at omega_opt =
    # 2/(1+sin(pi/(n+1))) of an n-unknowns-per-axis Dirichlet operator (r_J = cos(pi/(n+1))).  At omega_opt every
    # eigenvalue of the SOR iteration matrix has modulus omega_opt - 1 (Young's theory; the red-black ordering is
    # consistently ordered), so the residual contracts asymptotically like k (omega_opt-1)^k: between 30 and 50 sweeps
    # the mean factor per sweep is (50/30)^(1/20) (omega_opt - 1) = 1.026 * 0.4903 = 0.503.  With pi/n instead of
    # pi/(n+1) (omega = 1.4465 < omega_opt) the spectral radius is ((omega r_J + sqrt(omega^2 r_J^2 - 4(omega-1)))/2)^2
    # = 0.646, far outside the band.  On a single-level hierarchy (grid == coarsest grid) a "V-cycle" is exactly that solve.
    n = 8
    h = 2.0 / n
    o = po.Oracle((n,) * 3, (h,) * 3, origin=(-1 + h / 2,) * 3, bc=D6)
    rhs = wl.random_field((n,) * 3, 43)
    res = {}
    for sweeps in (30, 50):
        phi = np.zeros_like(rhs)
        res[sweeps] = o.vcycle(phi, rhs, coarsest_n=n, coarsest_sweeps=sweeps, ncycles=1)["resnorms"][1]
    factor = (res[50] / res[30]) ** (1 / 20)
    w_opt = 2 / (1 + math.sin(math.pi / (n + 1)))
    assert factor == pytest.approx((50 / 30) ** (1 / 20) * (w_opt - 1), rel=0.03)
    assert factor < 0.53
