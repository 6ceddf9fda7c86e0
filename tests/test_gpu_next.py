"""GPU parity of rows f3 and f4 (-m gpu): Chebyshev / position-dependent omega sequences (Eq. 6-7), the
inner multipole expansion (Eq. 21-22), CG preconditioned by the multi-colour Gauss-Seidel sweep (Eq. 9-10)."""
import numpy as np
import pytest
import torch

import pyoracle as po
from gpu_helpers import dev, host, make_pair, pointwise_scaled, rel_l2, set_faces, stencil_scale
from paper_2605_03563_b200 import binding as pb
from paper_2605_03563_b200 import workloads as wl

pytestmark = pytest.mark.gpu
D6 = (po.BC_DIRICHLET_GHOST,) * 6
PATHS = [pb.PATH_GENERIC, pb.PATH_PLANE]


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("shape", [(32, 32, 32), (33, 18, 7), (64, 48, 40)])
def test_rbsor_chebyshev_sequence_matches_oracle(path, shape):
    w = dict(shape=shape, spacing=(0.1, 0.12, 0.09), origin=(0, 0, 0), bc=D6)
    o, g = make_pair(w, path)
    set_faces(o, g, [wl.hash_uniform(7 + f, np.arange(o.face_len(f))) - 0.5 for f in range(6)])
    rhs = wl.random_field(shape, 8)
    for start in (0, 1):
        phi_c = wl.random_field(shape, 9)
        d_phi = dev(phi_c)
        for nsw in (1, 2, 5):     # odd and even sweep counts: one- and two-sweep fused passes
            o.rbsor_cheby(phi_c, rhs, nsw, start_n=start)
            rn = g.rbsor_cheby(d_phi, dev(rhs), nsw, start_n=start, want_resnorm=True)
            assert pointwise_scaled(host(d_phi), phi_c, stencil_scale(phi_c, rhs * 0.003)) <= 1e-13
            assert rn == pytest.approx(o.residual_norm(phi_c, rhs), rel=1e-10)
    # an explicit Jacobi radius travels through the ABI
    phi_c = np.zeros(o.npshape)
    d_phi = dev(phi_c)
    o.rbsor_cheby(phi_c, rhs, 3, rJ=0.9)
    g.rbsor_cheby(d_phi, dev(rhs), 3, r_jacobi=0.9)
    assert pointwise_scaled(host(d_phi), phi_c, stencil_scale(phi_c, rhs * 0.003)) <= 1e-13


def test_config1_chebyshev_converges_in_fewer_sweeps_than_fixed_omega():
    w = wl.config1()
    o, g = make_pair(w)
    r0 = o.residual_norm(np.zeros_like(w["rhs"]), w["rhs"])
    a, b = dev(np.zeros_like(w["rhs"])), dev(np.zeros_like(w["rhs"]))
    ra = g.rbsor_cheby(a, dev(w["rhs"]), 60, want_resnorm=True)
    rb = g.rbsor_sweep(b, dev(w["rhs"]), w["omega"], 60, want_resnorm=True)
    assert ra < 0.5 * rb and ra / r0 < 1e-3
    phi_c = np.zeros_like(w["rhs"])
    o.rbsor_cheby(phi_c, w["rhs"], 60)
    assert pointwise_scaled(host(a), phi_c, stencil_scale(phi_c, w["rhs"] / (6 / w["spacing"][0] ** 2))) <= 1e-13


def test_rbsor_local_omega_spherical_matches_oracle():
    w = wl.config5(32, 16, 32)
    o, g = make_pair(w)
    o.multipole_bc(w["rho"], w["G"], w["lmax"])
    g.multipole_bc(dev(w["rho"]), w["G"], w["lmax"], want_moments=False)
    phi_c = np.zeros_like(w["rhs"])
    d_phi = dev(phi_c)
    for nsw, start in ((1, 1), (4, 1), (3, 0)):
        o.rbsor_local(phi_c, w["rhs"], nsw, start_n=start)
        rn = g.rbsor_local(d_phi, dev(w["rhs"]), nsw, start_n=start, want_resnorm=True)
        assert rel_l2(host(d_phi), phi_c) <= 1e-12
        assert rn == pytest.approx(o.residual_norm(phi_c, w["rhs"]), rel=1e-9)
    # Cartesian: Eq. 7 without metric factors is Eq. 4 -> the uniform Chebyshev sequence
    wc = dict(shape=(24, 20, 16), spacing=(0.1, 0.12, 0.09), origin=(0, 0, 0), bc=D6)
    oc, gc = make_pair(wc)
    rhs = wl.random_field(wc["shape"], 3)
    a, b = dev(np.zeros(oc.npshape)), dev(np.zeros(oc.npshape))
    gc.rbsor_local(a, dev(rhs), 4)
    gc.rbsor_cheby(b, dev(rhs), 4)
    assert rel_l2(host(a), host(b)) <= 1e-14


def test_inner_multipole_expansion_matches_oracle():
    re, te, pe = wl.spherical_edges(32, 16, 32)
    bc = (po.BC_DIRICHLET_GHOST, po.BC_DIRICHLET_GHOST, po.BC_AXIS, po.BC_AXIS, po.BC_PERIODIC, po.BC_PERIODIC)
    w = dict(shape=(32, 16, 32), edges=(re, te, pe), coord=po.SPHERICAL, bc=bc)
    o, g = make_pair(w)
    rho = np.zeros(o.npshape)
    rho[:, :, 10:22] = wl.random_field((12, 16, 32), 8, 0.1, 1.0)
    for lmax in (0, 3, 8):
        q_c, qb_c = o.multipole_bc2(rho, 1.5, lmax)
        q_g = np.array(g.multipole_bc(dev(rho), 1.5, lmax))
        qb_g = np.array(g.multipole_inner_moments(lmax))
        for l in range(lmax + 1):
            sl = slice(l * l, (l + 1) * (l + 1))
            assert np.abs(q_g[sl] - q_c[sl]).max() <= 1e-12 * np.abs(q_c[sl]).max() + 1e-16 * abs(q_c[0])
            assert np.abs(qb_g[sl] - qb_c[sl]).max() <= 1e-12 * np.abs(qb_c[sl]).max() + 1e-16 * abs(qb_c[0])
        for f in (0, 1):
            buf = torch.empty(g.face_len(f), device="cuda", dtype=torch.float64)
            g.get_ghost_face(f, buf)
            want = o.get_ghost_face(f)
            assert np.abs(host(buf) - want).max() <= 1e-12 * np.abs(want).max()
    # the operator then uses the inner shell: same apply on both sides
    phi = wl.random_field(w["shape"], 6)
    d_out = torch.empty(phi.shape, device="cuda", dtype=torch.float64)
    g.apply_laplacian(dev(phi), d_out)
    assert pointwise_scaled(host(d_out), o.apply(phi), o.diag() * stencil_scale(phi) + 1.0) <= 1e-12
    with pytest.raises(pb.PoissonError):
        make_pair(wl.config5(16, 8, 16))[1].multipole_inner_moments(4)     # Neumann inner face: no inner expansion


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("n", [32, 64])
def test_pcg_gauss_seidel_preconditioned_matches_oracle(path, n):
    w = wl.config2(n)
    o, g = make_pair(w, path)
    o.multipole_bc(w["rho"], w["G"], w["lmax"])
    g.multipole_bc(dev(w["rho"]), w["G"], w["lmax"], want_moments=False)
    g.set_option(pb.OPT_RECORD_HISTORY, 1)
    for fixed in (10, 40):
        phi_c = np.zeros_like(w["rhs"])
        d_phi = dev(phi_c)
        res_c = o.pcg(phi_c, w["rhs"], fixed_iters=fixed, want_history=True)
        res_g = g.pcg_solve(d_phi, dev(w["rhs"]), fixed_iters=fixed)
        assert res_g["iters"] == fixed and res_g["status"] == pb.OK
        assert rel_l2(host(d_phi), phi_c) <= 1e-10
        assert np.allclose(g.get_history(fixed + 1), res_c["history"], rtol=1e-8)
    phi_c = np.zeros_like(w["rhs"])
    d_phi = dev(phi_c)
    res_c = o.pcg(phi_c, w["rhs"], rtol=1e-8, max_iter=2000)
    res_g = g.pcg_solve(d_phi, dev(w["rhs"]), rtol=1e-8, max_iter=2000)
    assert res_g["status"] == pb.OK and abs(res_g["iters"] - res_c["iters"]) <= 1
    b_norm = o.residual_norm(np.zeros_like(phi_c), w["rhs"])
    assert o.residual_norm(host(d_phi), w["rhs"]) <= 10 * 1e-8 * b_norm
    # about half the iterations of unpreconditioned CG on the same problem
    res_u = g.cg_solve(dev(np.zeros_like(w["rhs"])), dev(w["rhs"]), rtol=1e-8, max_iter=2000)
    assert res_g["iters"] < 0.65 * res_u["iters"]
    assert rel_l2(host(d_phi), w["exact"]) < {32: 2e-3, 64: 5e-4}[n]


def test_pcg_statuses_and_unsupported_grids():
    w = wl.config2(32)
    o, g = make_pair(w)
    d_phi, d_rhs = dev(np.zeros_like(w["rhs"])), dev(w["rhs"])
    res = g.pcg_solve(d_phi, d_rhs, rtol=1e-12, max_iter=3)
    assert res["status"] == pb.NOT_CONVERGED and res["iters"] == 3
    res = g.pcg_solve(d_phi, d_rhs, rtol=1e-9, max_iter=300)          # warm start
    assert res["status"] == pb.OK
    res = g.pcg_solve(dev(np.zeros_like(w["rhs"])), dev(np.zeros_like(w["rhs"])), rtol=1e-8, max_iter=10)
    assert res["status"] == pb.OK and res["iters"] == 0
    x = torch.zeros(512, device="cuda", dtype=torch.float64)
    with pytest.raises(pb.PoissonError) as e:
        pb.Poisson((8, 8, 8), (0.1,) * 3, order=6, bc=(po.BC_PERIODIC,) * 6).pcg_solve(x, x.clone())
    assert e.value.code == pb.UNSUPPORTED


@pytest.mark.parametrize("which", ["spherical", "cartesian"])
def test_bicgstab_gauss_seidel_preconditioned_matches_oracle(which):
    # BiCGSTAB right-preconditioned by the block lower-triangular B of Eq. 10 (POISSON_OPT_JACOBI = 2)
    w = wl.config5(32, 16, 32) if which == "spherical" else wl.config2(32)
    o, g = make_pair(w)
    o.multipole_bc(w["rho"], w["G"], w["lmax"])
    g.multipole_bc(dev(w["rho"]), w["G"], w["lmax"], want_moments=False)
    g.set_option(pb.OPT_JACOBI, 2)
    g.set_option(pb.OPT_RECORD_HISTORY, 1)
    for fixed in (3, 10):
        phi_c = np.zeros_like(w["rhs"])
        d_phi = dev(phi_c)
        res_c = o.bicgstab(phi_c, w["rhs"], fixed_iters=fixed, jacobi=2, want_history=True)
        res_g = g.bicgstab_solve(d_phi, dev(w["rhs"]), fixed_iters=fixed)
        assert res_g["iters"] == fixed and res_g["status"] == pb.OK
        # north_star's 1e-10 while rounding differences are not amplified (3 iterations); at 10 the erratic BiCGSTAB
        # recurrence on the spherical operator amplifies a 1-ulp input perturbation of the ORACLE itself beyond that
        # (C8): then 10 x that sensitivity, capped at 1e-6, is the bound
        tol_x, tol_h = 1e-10, 1e-7
        if fixed > 3:
            x2 = np.zeros_like(w["rhs"])
            eps = np.finfo(np.float64).eps * np.abs(w["rhs"]).max()
            h2 = o.bicgstab(x2, w["rhs"] + eps * wl.random_field(w["shape"], 77), fixed_iters=fixed, jacobi=2,
                            want_history=True)["history"]
            sens_x = rel_l2(x2, phi_c)
            sens_h = float(np.max(np.abs(np.array(h2) - res_c["history"]) / res_c["history"]))
            tol_x, tol_h = min(max(1e-10, 10 * sens_x), 1e-6), min(max(1e-7, 10 * sens_h), 1e-6)
            print("GS-BiCGSTAB %s %d its: oracle 1-ulp sensitivity %.2e / %.2e -> tolerances %.2e / %.2e"
                  % (which, fixed, sens_x, sens_h, tol_x, tol_h))
        assert rel_l2(host(d_phi), phi_c) <= tol_x
        assert np.allclose(g.get_history(fixed + 1), res_c["history"], rtol=tol_h)
    phi_c = np.zeros_like(w["rhs"])
    d_phi = dev(phi_c)
    res_c = o.bicgstab(phi_c, w["rhs"], rtol=1e-8, max_iter=3000, jacobi=2)
    res_g = g.bicgstab_solve(d_phi, dev(w["rhs"]), rtol=1e-8, max_iter=3000)
    assert res_g["status"] == pb.OK and res_c["status"] == 0
    b_norm = o.residual_norm(np.zeros_like(phi_c), w["rhs"])
    assert o.residual_norm(host(d_phi), w["rhs"]) <= 10 * 1e-8 * b_norm
    # fewer iterations than with Jacobi scaling (the default) on the same problem
    g.set_option(pb.OPT_JACOBI, 1)
    res_j = g.bicgstab_solve(dev(np.zeros_like(w["rhs"])), dev(w["rhs"]), rtol=1e-8, max_iter=3000)
    assert res_g["iters"] < 0.8 * res_j["iters"]
