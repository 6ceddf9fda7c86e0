"""The five BASELINE.json configs at FULL size, run to convergence on the GPU (-m gpu).

north_star: "converged solutions within 10x the residual tolerance" — read (C8) as: the TRUE residual of the
GPU solution, evaluated with the ORACLE's operator, is within 10 x rtol x ||r0||.  Where a closed form exists the
discretisation error is checked against the figure the oracle pins predict.  The oracle does not have to run the
solvers here (its one residual evaluation per config takes seconds); step-by-step solver parity is in
test_gpu_parity.py (reduced sizes) and test_gpu_fullsize.py (full sizes, short fixed counts).
"""
import math

import numpy as np
import pytest
import torch

import pyoracle as po
from gpu_helpers import dev, host, make_pair, rel_l2
from paper_2605_03563_b200 import binding as pb
from paper_2605_03563_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def test_config1_sor_200_sweeps_plateau():
    w = wl.config1()
    o, g = make_pair(w)
    d_phi, d_rhs = dev(np.zeros_like(w["rhs"])), dev(w["rhs"])
    r0 = o.residual_norm(np.zeros_like(w["rhs"]), w["rhs"])
    rn = g.rbsor_sweep(d_phi, d_rhs, w["omega"], 200, want_resnorm=True)
    phi = host(d_phi)
    assert rn / r0 < 1e-12
    assert o.residual_norm(phi, w["rhs"]) / r0 < 1e-12                       # the oracle's operator agrees
    assert np.abs(phi - w["exact"]).max() == pytest.approx(7.5303e-4, rel=1e-4)  # (c_h - 1) sin^3(16 pi / 33)


def test_config2_cg_uniform_sphere_128():
    w = wl.config2(128)
    o, g = make_pair(w)
    o.multipole_bc(w["rho"], w["G"], w["lmax"])
    g.multipole_bc(dev(w["rho"]), w["G"], w["lmax"], want_moments=False)
    d_phi = dev(np.zeros_like(w["rhs"]))
    res = g.cg_solve(d_phi, dev(w["rhs"]), rtol=w["rtol"], max_iter=5000)
    assert res["status"] == pb.OK and res["relres"] <= w["rtol"]
    assert 380 <= res["iters"] <= 500                                         # probe: 435 iterations at 128^3
    phi = host(d_phi)
    r0 = o.residual_norm(np.zeros_like(phi), w["rhs"])
    assert o.residual_norm(phi, w["rhs"]) / r0 <= 10 * w["rtol"]
    assert rel_l2(phi, w["exact"]) < 1e-4                                     # second order: 5.5e-5 at 128^3


@pytest.mark.parametrize("precision", [pb.F64, pb.MIXED])
def test_config3_ten_vcycles_256(precision):
    w = wl.config3(256)
    o, g = make_pair(w)
    o.multipole_bc(w["rho"], w["G"], w["lmax"])
    g.multipole_bc(dev(w["rho"]), w["G"], w["lmax"], want_moments=False)
    d_phi = dev(np.zeros_like(w["rhs"]))
    rn = np.array(g.mg_vcycle(d_phi, dev(w["rhs"]), precision=precision, ncycles=10)["resnorms"])
    assert np.all(rn[1:] / rn[:-1] < 0.2) and rn[-1] / rn[0] < 1e-8          # probe: 0.06 -> 0.15 per cycle, 2-4e-10 total
    phi = host(d_phi)
    assert o.residual_norm(phi, w["rhs"]) == pytest.approx(rn[-1], rel=1e-3 if precision == pb.F64 else 5e-2)
    assert rel_l2(phi, w["exact"]) < 1e-4                                     # O(h^2) + lmax = 8 truncation floor


def test_config4_cg6_periodic_512_converged():
    w = wl.config4(512)
    o, g = make_pair(w)
    rhs = w["rhs"]
    d_x = dev(np.zeros_like(rhs))
    res = g.cg_solve(d_x, dev(rhs), rtol=w["rtol"], max_iter=6000)
    assert res["status"] == pb.OK and res["relres"] <= w["rtol"]
    x = host(d_x)
    assert abs(x.mean()) <= 1e-12 * np.abs(x).max()                          # null space removed
    true = np.linalg.norm((rhs - o.apply(x)).ravel()) / np.linalg.norm(rhs.ravel())
    assert true <= 10 * w["rtol"]


def test_config5_bicgstab_spherical_converged():
    w = wl.config5()
    o, g = make_pair(w)
    o.multipole_bc(w["rho"], w["G"], w["lmax"])
    g.multipole_bc(dev(w["rho"]), w["G"], w["lmax"], want_moments=False)
    d_x = dev(np.zeros_like(w["rhs"]))
    res = g.bicgstab_solve(d_x, dev(w["rhs"]), rtol=w["rtol"], max_iter=40000)
    # rtol = 1e-8 is the accuracy fp64 can attain on this grid (r in [0.01, 1] log-spaced: eps |L| |x| / |rhs| ~ 1e-8;
    # DESIGN.md reading C4): the recurrence passes the threshold again and again while the TRUE residual, which is what
    # the solver reports, hovers at 0.99-1.07e-8.  Whether one of its confirmations lands below 1e-8 (OK) or the budget
    # of 30 runs out first (NOT_CONVERGED, honestly reported) changes with one ulp in the ghost values.  Either way the
    # solution meets north_star's bar: true residual within 10 x the tolerance, evaluated by the oracle's operator.
    confirm_failed = g.bicgstab_stats()[1]
    if res["status"] == pb.OK:
        assert res["relres"] <= w["rtol"]
    else:
        assert res["status"] == pb.NOT_CONVERGED and confirm_failed >= 30 and res["relres"] <= 1.2 * w["rtol"]
    assert res["iters"] < 20000
    x = host(d_x)
    r0 = o.residual_norm(np.zeros_like(x), w["rhs"])
    true = o.residual_norm(x, w["rhs"]) / r0
    assert true <= 10 * w["rtol"] and true == pytest.approx(res["relres"], rel=1e-3)
