"""Pins for the compact radius-1 discretisations of order 4 and 6 ("Spotz & Carey 1996"; the paper
prints no coefficients — DESIGN.md reading C19 derives them) and their SPAI smoothers (Table 1 rows 4 and 6) in the
oracle (oracle/mgv.cpp).  What fixes them independently of the oracle: the order at which the discretisation error of
a manufactured solution falls under refinement, the exact eigenvalues on sine modes, symmetry, a dense solve, the
smoothing factors of Table 1 and the convergence factors of Table 2."""
import itertools
import math

import numpy as np
import pytest

import pyoracle as po
from helpers import rel_l2

D6 = (po.BC_DIRICHLET_GHOST,) * 6
PI = math.pi


def _vertex_grid(n):
    h = 1.0 / (n + 1)
    return po.Oracle((n,) * 3, (h,) * 3, origin=(h,) * 3, bc=D6), h


def _sine(n, a, b, c, ext=0):
    """sin(a pi x) sin(b pi y) sin(c pi z) on the interior vertices of the unit cube (+ ext layers per side)."""
    h = 1.0 / (n + 1)
    x = h * (np.arange(-ext, n + ext) + 1)
    return np.ascontiguousarray(np.sin(c * PI * x)[:, None, None] * np.sin(b * PI * x)[None, :, None]
                                * np.sin(a * PI * x)[None, None, :])


def _lam(order, t1, t2, t3):
    """h^2 times the eigenvalue of the compact Laplacian on a Fourier mode, from the definition in second differences
    d_a^2 -> 2 cos(theta_a) - 2 (not from the stencil weights the oracle tabulates)."""
    d = [2 * math.cos(t) - 2 for t in (t1, t2, t3)]
    s1 = d[0] + d[1] + d[2]
    s2 = d[0] * d[1] + d[1] * d[2] + d[2] * d[0]
    s3 = d[0] * d[1] * d[2]
    return s1 + (s2 / 6 if order >= 4 else 0.0) + (s3 / 30 if order == 6 else 0.0)


@pytest.mark.parametrize("order", [2, 4, 6])
def test_compact_operator_has_the_closed_form_eigenvalues_on_sine_modes(order):
    n = 7
    o, h = _vertex_grid(n)
    for a, b, c in itertools.product((1, 2, 5, 7), repeat=3):
        u = _sine(n, a, b, c)
        lam = _lam(order, a * PI * h, b * PI * h, c * PI * h) / h ** 2
        assert np.abs(o.compact_apply(u, order) - lam * u).max() <= 1e-11 * abs(lam)


@pytest.mark.parametrize("order,rate", [(4, 4), (6, 6)])
def test_truncation_error_of_operator_and_right_hand_side_falls_at_the_formal_order(order, rate):
    # L_h u - B f for lap u = f, u = sin(pi x) sin(2 pi y) sin(pi z) (f = -6 pi^2 u, zero on the boundary): O(h^order).
    # A wrong edge / corner weight or a wrong 1/12, 1/240, 1/90 leaves an O(h^2) or O(h^4) term and fails the rate.
    errs = []
    for n in (7, 15, 31):
        o, h = _vertex_grid(n)
        u = _sine(n, 1, 2, 1)
        f_ext = -6 * PI ** 2 * _sine(n, 1, 2, 1, ext=2)
        errs.append(np.abs(o.compact_apply(u, order) - po.compact_rhs(f_ext, order)).max())
    r1, r2 = math.log2(errs[0] / errs[1]), math.log2(errs[1] / errs[2])
    assert rate - 0.35 < r2 < rate + 0.35 and r1 > rate - 0.8, (errs, r1, r2)


@pytest.mark.parametrize("order,rate", [(4, 4), (6, 6)])
def test_solution_error_falls_at_the_formal_order(order, rate):
    # the whole chain: transformed right-hand side, V-cycles of the paper's multigrid to a residual of 1e-11, error
    # against the exact solution under refinement 7^3 -> 15^3 -> 31^3
    errs = []
    for n in (7, 15, 31):
        o, h = _vertex_grid(n)
        u = _sine(n, 1, 1, 2)
        b = po.compact_rhs(-6 * PI ** 2 * _sine(n, 1, 1, 2, ext=2), order)
        phi = np.zeros_like(u)
        res = o.mgv_vcycle(phi, b, nu1=2, nu2=2, ncycles=14, order=order, cg_rtol=1e-6)["resnorms"]
        assert res[-1] <= 1e-10 * res[0]
        errs.append(np.abs(phi - u).max())
    r2 = math.log2(errs[1] / errs[2])
    assert rate - 0.4 < r2 < rate + 0.4, errs
    assert errs[2] < {4: 2e-6, 6: 5e-8}[order]


@pytest.mark.parametrize("order", [4, 6])
def test_compact_operator_is_symmetric_negative_definite_and_the_vcycle_solves_the_dense_system(order):
    n = 5
    o, h = _vertex_grid(n)
    N = n ** 3
    A = np.zeros((N, N))
    for c in range(N):
        e = np.zeros(N)
        e[c] = 1.0
        A[:, c] = o.compact_apply(e.reshape(n, n, n), order).reshape(-1)
    assert np.abs(A - A.T).max() <= 1e-12 * np.abs(A).max()
    assert np.linalg.eigvalsh(A).max() < 0
    rng = np.random.default_rng(5)
    b = rng.standard_normal((n, n, n))
    phi = np.zeros_like(b)
    o.mgv_vcycle(phi, b, nu1=2, nu2=2, coarsest_n=2, ncycles=30, order=order, cg_rtol=1e-10)
    assert rel_l2(phi, np.linalg.solve(A, b.reshape(-1)).reshape(n, n, n)) <= 1e-10


def _mu(order, sp, m=49):
    """Eq. 17 on a sample of T = [-pi,pi]^3 without [-pi/2,pi/2]^3 (symmetric in the signs: [0,pi]^3 suffices)."""
    om, al, be, ga, de = sp
    t = np.linspace(0.0, PI, m)
    T1, T2, T3 = np.meshgrid(t, t, t, indexing="ij")
    c1, c2, c3 = np.cos(T1), np.cos(T2), np.cos(T3)
    d1, d2, d3 = 2 * c1 - 2, 2 * c2 - 2, 2 * c3 - 2
    lam = d1 + d2 + d3
    if order >= 4:
        lam = lam + (d1 * d2 + d2 * d3 + d3 * d1) / 6
    if order == 6:
        lam = lam + d1 * d2 * d3 / 30
    M = al + 2 * be * (c1 + c2 + c3) + 4 * ga * (c1 * c2 + c2 * c3 + c3 * c1) + 8 * de * c1 * c2 * c3
    S = 1 + om * M * lam                         # A = -L_h
    hi = (T1 >= PI / 2 - 1e-12) | (T2 >= PI / 2 - 1e-12) | (T3 >= PI / 2 - 1e-12)
    return np.abs(S[hi]).max()


def test_table1_rows_4_and_6_belong_to_the_compact_operators():
    # With the 4-digit coefficients the paper prints, Eq. 17 gives 0.104 (order 4; the paper quotes an "approximate"
    # 0.0828) and 0.112 (order 6, delta by reading C20; quoted 0.0909) — the same 10-25 % above the quoted value as row 2
    # (0.2076 against 0.1888).  Rows and operators that do not belong together are far off: row 4 on the 7-point operator
    # or row 2 on the 19-point one give > 0.3.
    mu4, mu6 = _mu(4, po.SPAI_ORDER4), _mu(6, po.SPAI_ORDER6)
    assert 0.0828 <= mu4 <= 0.105 and 0.0909 <= mu6 <= 0.113
    assert _mu(2, po.SPAI_ORDER4) > 0.3 and _mu(4, po.SPAI_ORDER2) > 0.3 and _mu(6, po.SPAI_ORDER4) > 0.3
    # reading C20: the printed delta of row 6 (0.0909, a copy of the mu column) makes the iteration diverge
    assert _mu(6, po.SPAI_ORDER6[:4] + (0.0909,)) > 1.0
    # and 0.0150 sits on the flat minimum of mu over delta
    assert all(_mu(6, po.SPAI_ORDER6[:4] + (d,)) >= mu6 - 1e-9 for d in (0.012, 0.013, 0.017, 0.018))


@pytest.mark.parametrize("order", [4, 6])
def test_spai_step_multiplies_sine_modes_by_the_symbol(order):
    n = 7
    o, h = _vertex_grid(n)
    om, al, be, ga, de = po.SPAI[order]
    for a, b, c in itertools.product((1, 3, 4, 7), repeat=3):
        u = _sine(n, a, b, c)
        v = u.copy()
        o.spai_smooth(v, np.zeros_like(u), nsteps=1, order=order)
        c1, c2, c3 = (math.cos(q * PI * h) for q in (a, b, c))
        M = al + 2 * be * (c1 + c2 + c3) + 4 * ga * (c1 * c2 + c2 * c3 + c3 * c1) + 8 * de * c1 * c2 * c3
        s = 1 + om * M * _lam(order, a * PI * h, b * PI * h, c * PI * h)
        assert np.abs(v - s * u).max() <= 1e-13


def test_vcycle_convergence_factors_of_table2():
    # PAPER.md Table 2 (511^3, seven coarse levels): residual factors per V(1,1) cycle 0.102 / 0.065 / 0.068 for orders
    # 2 / 4 / 6.  The factor a cycle settles to is grid-independent: on the two-sphere problem at 31^3 (three coarse
    # levels) the eighth cycle gives 0.091 / 0.067 / 0.068.  The V(2,2) means of eight cycles (paper: 0.028 / 0.017 /
    # 0.018) depend on the size and on the number of cycles averaged and only have to come out in the same order.
    from paper_2605_03563_b200 import workloads as wl
    n = 31
    o, h = _vertex_grid(n)
    b = wl.two_spheres(n, cell_centred=False)["rhs"]
    last, mean2 = {}, {}
    for order in (2, 4, 6):
        phi = np.zeros_like(b)
        r = o.mgv_vcycle(phi, b, nu1=1, nu2=1, ncycles=8, order=order)["resnorms"]
        last[order] = r[8] / r[7]
        phi = np.zeros_like(b)
        r = o.mgv_vcycle(phi, b, nu1=2, nu2=2, ncycles=8, order=order)["resnorms"]
        mean2[order] = (r[8] / r[0]) ** 0.125
    assert last[4] == pytest.approx(0.065, rel=0.08) and last[6] == pytest.approx(0.068, rel=0.08)
    assert last[2] == pytest.approx(0.102, rel=0.15)
    assert last[4] < last[6] < last[2]
    assert mean2[2] == pytest.approx(0.028, rel=0.1)
    assert mean2[4] < mean2[6] < mean2[2] and mean2[4] == pytest.approx(0.017, rel=0.45)
