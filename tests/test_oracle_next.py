"""Pins for the oracle's SURVEY.md §8 "next" rows f3 and f4: multi-colour Gauss-Seidel preconditioning (PAPER.md:107-123
Eq. 9-10), the Chebyshev / position-dependent omega sequences (Eq. 6-7), the inner multipole expansion
(Eq. 21-22)."""
import math
import os

import numpy as np
import pytest

import pyoracle as po
from helpers import dense_matrix, rel_l2
from paper_2605_03563_b200 import workloads as wl

D6 = (po.BC_DIRICHLET_GHOST,) * 6
GOLD = os.path.join(os.path.dirname(__file__), "golden")
COUNTS = {(r[0], int(r[1])): (int(r[2]), int(r[3]))
          for r in (l.split() for l in open(os.path.join(GOLD, "paper_table3_counts.txt")) if l[0] != "#")}


def _two_sphere(n=64):
    w = wl.two_spheres(n)
    o = po.Oracle(w["shape"], w["spacing"], w["origin"], bc=w["bc"])
    for f, a in enumerate(wl.analytic_ghost_faces(w, w["potential"])):
        o.set_ghost_face(f, a)
    return w, o


def _sph(nr=8, nt=4, nph=8, inner=po.BC_NEUMANN0):
    re, te, pe = wl.spherical_edges(nr, nt, nph)
    bc = (inner, po.BC_DIRICHLET_GHOST, po.BC_AXIS, po.BC_AXIS, po.BC_PERIODIC, po.BC_PERIODIC)
    return po.Oracle((nr, nt, nph), edges=(re, te, pe), coord=po.SPHERICAL, bc=bc), (re, te, pe)


# ---- f4: Chebyshev acceleration, Eq. 6 -------------------------------------------------------------------------------
def test_chebyshev_sequence_decreases_to_omega_opt_of_eq3():
    o = po.Oracle((32,) * 3, (1 / 33,) * 3, origin=(1 / 33,) * 3, bc=D6)
    rJ = o.jacobi_radius()
    assert rJ == pytest.approx(math.cos(math.pi / 33), rel=1e-15)            # Eq. 4, N = n + 1 (C0)
    phi = np.zeros(o.npshape)
    om = o.rbsor_cheby(phi, np.zeros(o.npshape), 300, start_n=0)
    assert om[0] == 1.0 and om[1] == pytest.approx(1 / (1 - rJ ** 2 / 2), rel=1e-15)   # omega_0, omega_1
    assert np.all(np.diff(om[1:]) <= 0) and np.all(np.diff(om[1:60]) < 0)     # monotone from omega_1 on (then converged)
    w_opt = 2 / (1 + math.sqrt(1 - rJ ** 2))                                  # Eq. 3, the fixed point of the recurrence
    assert om[-1] == pytest.approx(w_opt, rel=1e-12) and om[-1] >= w_opt
    assert np.array_equal(o.rbsor_cheby(phi, np.zeros(o.npshape), 5, start_n=1), om[1:11])   # "starting from n = 1"


def test_chebyshev_half_sweeps_use_one_omega_each_and_converge_to_the_discrete_solution():
    shape, h = (8, 8, 8), (0.1, 0.1, 0.1)
    o = po.Oracle(shape, h, bc=D6)
    o.set_ghost_face(0, wl.hash_uniform(5, np.arange(o.face_len(0))))
    rhs = wl.random_field(shape, 3)
    # composition pin: the same iterate as explicit half-sweeps driven by the returned sequence
    a = wl.random_field(shape, 4)
    b = a.copy()
    om = o.rbsor_cheby(a, rhs, 3, start_n=1)
    for m in range(6):
        o.rbsor_half(b, rhs, om[m], m & 1)
    assert np.array_equal(a, b)
    exact = np.linalg.solve(dense_matrix(o), (rhs - o.apply(np.zeros(o.npshape))).reshape(-1)).reshape(rhs.shape)
    phi = np.zeros_like(rhs)
    o.rbsor_cheby(phi, rhs, 120)
    assert rel_l2(phi, exact) < 1e-12


def test_chebyshev_needs_fewer_sweeps_than_table3_fixed_omega():
    # "the first steps of the SOR iteration may be more accurate"; Table 3 prints 130 / 187 sweeps at 64^3 for
    # the fixed omega_opt,a of Eq. 5.  With the sequence of Eq. 6 (from n = 1) the same reductions take fewer sweeps.
    w, o = _two_sphere(64)
    r0 = o.residual_norm(np.zeros_like(w["rhs"]), w["rhs"])
    want4, want6 = COUNTS[("SOR", 64)]
    got = {}
    for nsw in (100, 113, 150, 162):
        phi = np.zeros_like(w["rhs"])
        o.rbsor_cheby(phi, w["rhs"], nsw, start_n=1)
        got[nsw] = o.residual_norm(phi, w["rhs"]) / r0
    assert got[113] < 1e-4 < got[100] and 113 < want4
    assert got[162] < 1e-6 < got[150] and 162 < want6


# ---- f4: position-dependent omega, Eq. 7 -----------------------------------------------------------------------------
def test_local_jacobi_radius_is_eq7():
    o, (re, te, pe) = _sph(8, 4, 8)
    for i, j in ((0, 0), (3, 1), (7, 3)):
        r, th = math.sqrt(re[i] * re[i + 1]), 0.5 * (te[j] + te[j + 1])
        a, b, c = (re[i + 1] - re[i]) ** -2, (r * (te[1] - te[0])) ** -2, (r * math.sin(th) * (pe[1] - pe[0])) ** -2
        want = (math.cos(math.pi / 8) * a + math.cos(math.pi / 4) * b + math.cos(math.pi / 8) * c) / (a + b + c)
        assert o.local_jacobi_radius(i, j) == pytest.approx(want, rel=1e-14)
    # "Equation (7) can also be adapted to a ... Cartesian grid by omitting the metric factors" -> Eq. 4 on a uniform one
    oc = po.Oracle((8, 6, 4), (0.1, 0.2, 0.3), bc=D6)
    assert oc.local_jacobi_radius(2, 3) == oc.jacobi_radius()


def test_local_omega_sor_converges_to_the_gauss_seidel_fixed_point_and_faster():
    # "This approach also converges to the same value as Gauss-Seidel, and it is experimentally observed to
    # improve speed of convergence for nonuniform and curvilinear grids."
    o, _ = _sph(8, 4, 8)
    ghost = wl.hash_uniform(4, np.arange(o.face_len(1)))
    o.set_ghost_face(1, ghost)
    rhs = wl.random_field(o.shape, 6)
    exact = np.linalg.solve(dense_matrix(o), (rhs - o.apply(np.zeros(o.npshape))).reshape(-1)).reshape(rhs.shape)
    phi = np.zeros_like(rhs)
    o.rbsor_local(phi, rhs, 400)
    assert rel_l2(phi, exact) < 1e-10
    w = wl.config5(32, 16, 32)
    o = po.Oracle(w["shape"], edges=w["edges"], coord=po.SPHERICAL, bc=w["bc"])
    o.multipole_bc(w["rho"], 1.0, 8)
    a, b = np.zeros_like(w["rhs"]), np.zeros_like(w["rhs"])
    o.rbsor_local(a, w["rhs"], 400)
    o.rbsor(b, w["rhs"], 1.0, 400)
    assert o.residual_norm(a, w["rhs"]) < 0.02 * o.residual_norm(b, w["rhs"])


# ---- f4: inner multipole expansion, Eq. 21-22 ------------------------------------------------------------------------
def test_inner_moments_of_a_point_mass_and_the_inner_potential():
    # a single cell of mass M at radius a on the z axis-ish direction: qbar_l0-like closed forms hold through the addition
    # theorem: Phi_inner(x) = -G M sum_l r^l / a^(l+1) P_l(cos gamma) -> -G M / |x - x'| for r < a as lmax grows
    o, (re, te, pe) = _sph(16, 8, 16, inner=po.BC_DIRICHLET_GHOST)
    rho = np.zeros(o.npshape)
    i, j, k = 11, 2, 5
    rho[k, j, i] = 3.0
    rc, tc, pc = o.centres(0), o.centres(1), o.centres(2)
    dV = (re[i + 1] ** 3 - re[i] ** 3) / 3 * (math.cos(te[j]) - math.cos(te[j + 1])) * (pe[k + 1] - pe[k])
    M = 3.0 * dV
    src = rc[i] * np.array([math.sin(tc[j]) * math.cos(pc[k]), math.sin(tc[j]) * math.sin(pc[k]), math.cos(tc[j])])
    qb = o.multipole_inner_moments(rho, 16)
    assert qb[0] == pytest.approx(M / rc[i], rel=1e-13)                       # l = 0: M / a
    x = 0.2 * rc[i] * np.array([0.3, -0.5, 0.81])
    direct = -2.0 * M / np.linalg.norm(x - src)
    errs = [abs(po.multipole_inner_potential(qb, L, 2.0, *x) - direct) / abs(direct) for L in (2, 8, 16)]
    assert errs[0] > errs[1] > errs[2] and errs[2] < 1e-9                     # geometric in (r/a)^(lmax+1)
    # brute force: the truncated Legendre sum, convention-independent (addition theorem)
    cg = float(x @ src / (np.linalg.norm(x) * rc[i]))
    P = [1.0, cg]
    for l in range(2, 9):
        P.append(((2 * l - 1) * cg * P[l - 1] - (l - 1) * P[l - 2]) / l)
    want = -2.0 * M * sum(np.linalg.norm(x) ** l / rc[i] ** (l + 1) * P[l] for l in range(9))
    assert po.multipole_inner_potential(qb, 8, 2.0, *x) == pytest.approx(want, rel=1e-12)


def test_multipole_bc_fills_the_inner_ghost_shell_with_eq21_and_the_outer_with_eq19():
    o, (re, te, pe) = _sph(16, 8, 16, inner=po.BC_DIRICHLET_GHOST)
    rho = np.zeros(o.npshape)
    rho[:, :, 6:10] = wl.random_field((4, 8, 16), 8, 0.1, 1.0)                # a shell well inside (r_in, r_out)
    q, qb = o.multipole_bc2(rho, 1.5, 6)
    assert np.array_equal(q, o.multipole_moments(rho, 6)) and np.array_equal(qb, o.multipole_inner_moments(rho, 6))
    tc, pc = o.centres(1), o.centres(2)
    r_in = re[0] * math.sqrt(re[0] / re[1])
    inner, outer = o.get_ghost_face(0).reshape(16, 8), o.get_ghost_face(1).reshape(16, 8)
    for (jj, kk) in ((0, 0), (3, 7), (7, 15)):
        d = np.array([math.sin(tc[jj]) * math.cos(pc[kk]), math.sin(tc[jj]) * math.sin(pc[kk]), math.cos(tc[jj])])
        assert inner[kk, jj] == po.multipole_inner_potential(qb, 6, 1.5, *(r_in * d))
        assert outer[kk, jj] == po.multipole_potential(q, 6, 1.5, *(o.r_ghost_out() * d))
    # with Neumann at r_in (BASELINE config 5) the inner shell does not exist
    on, _ = _sph(16, 8, 16)
    on.multipole_bc(rho, 1.5, 6)
    assert np.array_equal(on.get_ghost_face(1), o.get_ghost_face(1))


# ---- f3: multi-colour Gauss-Seidel preconditioner, Eq. 9-10 ----------------------------------------------------------
def _colour_perm(o):
    n0, n1, n2 = o.shape
    idx = np.arange(n0 * n1 * n2)
    i, j, k = idx % n0, (idx // n0) % n1, idx // (n0 * n1)
    red = ((i + j + k) & 1) == 0
    return np.concatenate([idx[red], idx[~red]]), int(red.sum())


def test_gs_preconditioner_is_the_block_lower_triangular_solve_of_eq10():
    # order the unknowns red then black: A = [[D_R, N_RB], [N_BR, D_B]] (Eq. 9), B = [[D_R, 0], [N_BR, D_B]] (Eq. 10)
    for o in (po.Oracle((6, 5, 4), (0.1, 0.15, 0.2), bc=D6), _sph(8, 4, 8)[0]):
        L = dense_matrix(o)
        perm, nr = _colour_perm(o)
        for sign in (+1, -1):
            A = sign * L[np.ix_(perm, perm)]
            assert np.count_nonzero(A[:nr, :nr] - np.diag(np.diag(A[:nr, :nr]))) == 0      # D_R, D_B are diagonal:
            assert np.count_nonzero(A[nr:, nr:] - np.diag(np.diag(A[nr:, nr:]))) == 0      # two colours suffice
            B = A.copy()
            B[:nr, nr:] = 0.0
            v = wl.random_field(o.shape, 31)
            z = o.gs_precond(v, sign=sign, symmetric=False)
            want = np.linalg.solve(B, v.reshape(-1)[perm])
            assert np.abs(z.reshape(-1)[perm] - want).max() <= 1e-12 * np.abs(want).max()


def test_symmetrised_gs_preconditioner_is_symmetric_positive_definite():
    o = po.Oracle((6, 5, 4), (0.1, 0.15, 0.2), bc=D6)
    n = o.size
    Minv = np.zeros((n, n))
    e = np.zeros(o.npshape)
    for c in range(n):
        e.reshape(-1)[c] = 1.0
        Minv[:, c] = o.gs_precond(e, sign=-1, symmetric=True).reshape(-1)
        e.reshape(-1)[c] = 0.0
    assert np.abs(Minv - Minv.T).max() <= 1e-14 * np.abs(Minv).max()
    assert np.linalg.eigvalsh(0.5 * (Minv + Minv.T)).min() > 0
    # it is the symmetric Gauss-Seidel splitting: M = (D + Lo) D^-1 (D + Lo^T) in the red-black ordering
    A = -dense_matrix(o)
    perm, nr = _colour_perm(o)
    Ap = A[np.ix_(perm, perm)]
    D, Lo = np.diag(np.diag(Ap)), np.tril(Ap, -1)
    M = (D + Lo) @ np.linalg.inv(D) @ (D + Lo.T)
    assert np.abs(np.linalg.inv(M) - Minv[np.ix_(perm, perm)]).max() <= 1e-12 * np.abs(Minv).max()
    # the forward-only B^-1 of Eq. 10 is NOT symmetric — which is why CG takes the symmetrised sweep (C15)
    u, v = wl.random_field(o.shape, 1), wl.random_field(o.shape, 2)
    a, b = np.vdot(u, o.gs_precond(v, symmetric=False)), np.vdot(o.gs_precond(u, symmetric=False), v)
    assert abs(a - b) > 1e-3 * abs(a)


def test_pcg_matches_dense_solve_and_halves_table3_counts():
    shape, h = (8, 8, 8), (0.1, 0.12, 0.09)
    o = po.Oracle(shape, h, bc=D6)
    o.set_ghost_face(3, wl.hash_uniform(9, np.arange(o.face_len(3))))
    rhs = wl.random_field(shape, 3)
    exact = np.linalg.solve(dense_matrix(o), (rhs - o.apply(np.zeros(o.npshape))).reshape(-1)).reshape(rhs.shape)
    phi = np.zeros_like(rhs)
    res = o.pcg(phi, rhs, rtol=1e-13, max_iter=300)
    assert res["status"] == 0 and rel_l2(phi, exact) < 1e-11
    # "Applying an iterative method directly to A rarely gives sufficiently good convergence"; Table 3's
    # CG2 counts at 64^3 (125 / 171, unpreconditioned) drop to about half with the Gauss-Seidel preconditioner
    w, o = _two_sphere(64)
    want4, want6 = COUNTS[("CG2", 64)]
    for tol, want in ((1e-4, want4), (1e-6, want6)):
        phi = np.zeros_like(w["rhs"])
        res = o.pcg(phi, w["rhs"], rtol=tol, max_iter=1000)
        assert res["status"] == 0 and 0.4 * want <= res["iters"] <= 0.6 * want
        assert o.residual_norm(phi, w["rhs"]) <= tol * o.residual_norm(np.zeros_like(phi), w["rhs"]) * (1 + 1e-9)


def test_bicgstab_with_eq10_preconditioner_matches_dense_lu_and_beats_jacobi_scaling():
    o, _ = _sph(8, 4, 8)
    o.set_ghost_face(1, wl.hash_uniform(4, np.arange(o.face_len(1))))
    rhs = wl.random_field(o.shape, 6)
    exact = np.linalg.solve(dense_matrix(o), (rhs - o.apply(np.zeros(o.npshape))).reshape(-1)).reshape(rhs.shape)
    phi = np.zeros_like(rhs)
    res = o.bicgstab(phi, rhs, rtol=1e-11, max_iter=2000, jacobi=2)
    assert res["status"] == 0 and rel_l2(phi, exact) < 1e-9
    w = wl.config5(32, 16, 32)
    o = po.Oracle(w["shape"], edges=w["edges"], coord=po.SPHERICAL, bc=w["bc"])
    o.multipole_bc(w["rho"], 1.0, 8)
    its = {}
    for pre in (1, 2):
        phi = np.zeros_like(w["rhs"])
        res = o.bicgstab(phi, w["rhs"], rtol=1e-8, max_iter=5000, jacobi=pre)
        assert res["status"] == 0
        assert o.residual_norm(phi, w["rhs"]) <= 1e-8 * o.residual_norm(np.zeros_like(phi), w["rhs"]) * 1.001
        its[pre] = res["iters"]
    assert its[2] < 0.7 * its[1]
