"""Pins for the oracle's red-black SOR (oracle/rbsor.cpp) — SURVEY.md §8(c) C2; Table 3."""
import math
import os

import numpy as np
import pytest

import pyoracle as po
from helpers import dense_matrix, make_oracle
from paper_2605_03563_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
D6 = (po.BC_DIRICHLET_GHOST,) * 6


def test_fixed_point_is_dense_solve_8cubed():
    shape, h = (8, 8, 8), (0.11, 0.13, 0.17)
    o = po.Oracle(shape, h, bc=D6)
    A = dense_matrix(o)
    rhs = wl.random_field(shape, 7)
    exact = np.linalg.solve(A, rhs.reshape(-1)).reshape(rhs.shape)
    phi = np.zeros_like(rhs)
    o.rbsor(phi, rhs, 1.5, 400)
    assert np.abs(phi - exact).max() <= 1e-12 * np.abs(exact).max()


def test_fixed_point_with_inhomogeneous_ghosts():
    # harmonic quadratic: the discrete solution with analytic ghosts and rhs = L f is f itself
    shape, h, org = (6, 7, 8), (0.2, 0.2, 0.2), (0.1, 0.2, 0.3)
    w = dict(shape=shape, spacing=h, origin=org, bc=D6)
    o = make_oracle(w)
    f = lambda x, y, z: x * x - 2 * y * y + z * z + 3 * x * z + 1.0
    for k, fa in enumerate(wl.analytic_ghost_faces(w, f)):
        o.set_ghost_face(k, fa)
    X, Y, Z = wl._mesh(shape, org, h)
    phi = np.zeros(o.npshape)
    o.rbsor(phi, np.zeros(o.npshape), 1.4, 300)
    assert np.abs(phi - f(X, Y, Z)).max() < 1e-11


def test_config1_closed_form_plateau_and_golden_trajectory():
    w = wl.config1()
    o = make_oracle(w)
    h = w["spacing"][0]
    assert w["omega"] == pytest.approx(1.8263905415884214, abs=1e-15)
    phi = np.zeros_like(w["rhs"])
    r0 = o.residual_norm(phi, w["rhs"])
    gold = np.loadtxt(os.path.join(GOLD, "config1_sor_trajectory.txt"))
    for row in gold:
        rn = o.rbsor(phi, w["rhs"], w["omega"], 10, want_resnorm=True)
        assert rn / r0 == pytest.approx(row[1], rel=0.02)
        assert np.abs(phi - w["exact"]).max() == pytest.approx(row[2], rel=0.02)
    # converged discrete solution = c_h sin sin sin, c_h = pi^2 h^2/(4 sin^2(pi h/2))
    ch = math.pi ** 2 * h ** 2 / (4 * math.sin(math.pi * h / 2) ** 2)
    assert ch - 1 == pytest.approx(7.5559e-4, rel=1e-4)
    o.rbsor(phi, w["rhs"], w["omega"], 20)
    assert np.abs(phi - ch * w["exact"]).max() < 1e-13
    assert np.abs(phi - w["exact"]).max() == pytest.approx((ch - 1) * math.sin(16 * math.pi / 33) ** 3, rel=1e-9)


def test_asymptotic_factor_is_omega_opt_minus_one():
    # Young's theory for consistently ordered matrices: rho(SOR at omega_opt) = omega_opt - 1 (Eq. 3)
    w = wl.config1()
    o = make_oracle(w)
    phi = np.zeros_like(w["rhs"])
    o.rbsor(phi, w["rhs"], w["omega"], 60)
    r60 = o.residual_norm(phi, w["rhs"])
    o.rbsor(phi, w["rhs"], w["omega"], 60)
    r120 = o.residual_norm(phi, w["rhs"])
    factor = (r120 / r60) ** (1 / 60)
    # at omega_opt the iteration matrix has a Jordan block: the observed factor approaches omega-1 from above
    assert factor == pytest.approx(w["omega"] - 1, rel=0.04)
    assert w["omega"] - 1 == pytest.approx(0.82639, abs=1e-5)


def test_second_order_under_refinement():
    errs = []
    for n in (32, 65):
        w = wl.config1(n)
        o = make_oracle(w)
        phi = np.zeros_like(w["rhs"])
        o.rbsor(phi, w["rhs"], w["omega"], 160 if n == 32 else 330)
        errs.append(np.abs(phi - w["exact"]).max())
    assert errs[1] == pytest.approx(1.888e-4, rel=2e-3)
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.01)


@pytest.mark.parametrize("omega", [1.0, 1.5, 1.8263905415884214, 1.95])
def test_energy_never_increases(omega):
    # Ostrowski-Reich: for SPD A = -L and 0 < omega < 2 every relaxation step lowers E = 1/2 phi'A phi - b'phi
    shape = (16, 16, 16)
    o = po.Oracle(shape, (1 / 17,) * 3, bc=D6)
    rhs = wl.random_field(shape, 11)
    phi = np.zeros_like(rhs)

    def energy(p):
        Ap = -o.apply(p, use_ghost=False)
        return 0.5 * np.vdot(p, Ap) + np.vdot(rhs, p)  # b = -rhs

    e_prev = energy(phi)
    for half in range(60):
        o.rbsor_half(phi, rhs, omega, half & 1)
        e = energy(phi)
        assert e <= e_prev + 1e-12 * abs(e_prev)
        e_prev = e


def test_paper_table3_sor_counts_64():
    # SOR with omega_opt,a = 2/(1+pi/N) needs 130 / 187 sweeps at 64^3
    counts = {(r[0], int(r[1])): (int(r[2]), int(r[3]))
              for r in (l.split() for l in open(os.path.join(GOLD, "paper_table3_counts.txt")) if l[0] != "#")}
    n = 64
    w = wl.two_spheres(n)
    o = make_oracle(w)
    for k, fa in enumerate(wl.analytic_ghost_faces(w, w["potential"])):
        o.set_ghost_face(k, fa)
    phi = np.zeros_like(w["rhs"])
    om = 2 / (1 + math.pi / n)
    r0 = o.residual_norm(phi, w["rhs"])
    c4 = c6 = None
    for s in range(1, 260):
        rn = o.rbsor(phi, w["rhs"], om, 1, want_resnorm=True)
        if c4 is None and rn / r0 < 1e-4:
            c4 = s
        if rn / r0 < 1e-6:
            c6 = s
            break
    assert (c4, c6) == counts[("SOR", 64)]


def test_f32_sweep_tracks_f64():
    w = wl.config1(16)
    o = make_oracle(w)
    p64 = np.zeros_like(w["rhs"])
    p32 = np.zeros(w["rhs"].shape, dtype=np.float32)
    o.rbsor(p64, w["rhs"], 1.0, 5)
    o.rbsor_f32(p32, w["rhs"].astype(np.float32), 1.0, 5)
    assert np.abs(p32 - p64).max() < 2e-6 * np.abs(p64).max()
