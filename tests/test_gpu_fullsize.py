"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (-m gpu).

The oracle is slow but finishes one operator application / sweep / V-cycle / Krylov iteration on these grids in
seconds with its OpenMP pointwise loops, so the comparison is still element by element over the WHOLE grid for the
pointwise rows and relative L2 for short fixed-count solver runs (C8).  Also: the different kernel paths
(generic direct-load kernels vs the fused / staged ones) must agree bit for bit on pointwise work.
"""
import math

import numpy as np
import pytest
import torch

import pyoracle as po
from gpu_helpers import dev, host, make_pair, pointwise_scaled, rel_l2, stencil_scale
from paper_2605_03563_b200 import binding as pb
from paper_2605_03563_b200 import workloads as wl

pytestmark = pytest.mark.gpu
D6 = (po.BC_DIRICHLET_GHOST,) * 6
P6 = (po.BC_PERIODIC,) * 6


def gface(g, f):
    out = torch.empty(g.face_len(f), device="cuda", dtype=torch.float64)
    g.get_ghost_face(f, out)
    return host(out)


@pytest.fixture(scope="module")
def c3():
    """Config 3 grid (256^3, Dirichlet ghosts from the multipole expansion, lmax = 8) on both sides."""
    w = wl.config3(256)
    o, g = make_pair(w)
    o.multipole_bc(w["rho"], w["G"], w["lmax"])
    g.multipole_bc(dev(w["rho"]), w["G"], w["lmax"], want_moments=False)
    return w, o, g


def test_config3_ghost_faces_256(c3):
    w, o, g = c3
    for f in range(6):
        got = gface(g, f)
        want = o.get_ghost_face(f)
        assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max()


def test_apply_and_residual_256(c3):
    w, o, g = c3
    phi = wl.random_field(w["shape"], 31)
    want = o.apply(phi)
    d_phi, d_out = dev(phi), torch.empty(phi.shape, device="cuda", dtype=torch.float64)
    g.apply_laplacian(d_phi, d_out)
    d = 2 * 3 / w["spacing"][0] ** 2
    assert pointwise_scaled(host(d_out), want, d * stencil_scale(phi) + 1.0) <= 1e-13
    rn = g.residual_norm(d_phi, dev(w["rhs"]))
    assert rn == pytest.approx(o.residual_norm(phi, w["rhs"]), rel=1e-12)


def test_rbsor_two_sweeps_256(c3):
    w, o, g = c3
    phi_c = wl.random_field(w["shape"], 32)
    d_phi, d_rhs = dev(phi_c), dev(w["rhs"])
    omega = 2.0 / (1.0 + math.sin(math.pi / 257))
    d = 2 * 3 / w["spacing"][0] ** 2
    for nsw in (2, 1):   # an even count (pure ping-pong) and an odd one (final copy back)
        o.rbsor(phi_c, w["rhs"], omega, nsw)
        g.rbsor_sweep(d_phi, d_rhs, omega, nsw)
        assert pointwise_scaled(host(d_phi), phi_c, stencil_scale(phi_c, w["rhs"] / d)) <= 1e-13


@pytest.mark.parametrize("precision,tol", [(pb.F64, 1e-10), (pb.MIXED, 1e-5)])
def test_vcycle_256(c3, precision, tol):
    w, o, g = c3
    phi_c = np.zeros_like(w["rhs"])
    d_phi = dev(phi_c)
    rc = o.vcycle(phi_c, w["rhs"], precision=precision, ncycles=2)["resnorms"]
    rg = np.array(g.mg_vcycle(d_phi, dev(w["rhs"]), precision=precision, ncycles=2)["resnorms"])
    assert rel_l2(host(d_phi), phi_c) <= tol
    assert np.allclose(rg, rc, rtol=1e-6 if precision == pb.F64 else 2e-2)
    assert np.all(rg[1:] / rg[:-1] < 0.2)


def test_cg_19pt_periodic_512_three_iterations():
    """Config 4 grid (512^3 periodic, 19-point): white-noise right-hand side (the filtered field of config 4 needs a
    134 M-point host FFT; the kernels do not care), three CG iterations, and one operator application."""
    n = 512
    w = dict(shape=(n, n, n), spacing=(1.0 / n,) * 3, origin=(0.0,) * 3, order=6, bc=P6)
    o, g = make_pair(w)
    rhs = wl.random_field(w["shape"], 41)
    rhs -= rhs.mean()
    want = o.apply(rhs)
    d_rhs, d_out = dev(rhs), torch.empty(rhs.shape, device="cuda", dtype=torch.float64)
    g.apply_laplacian(d_rhs, d_out)
    c = n * n
    assert pointwise_scaled(host(d_out), want, (49 / 18) * 3 * c * stencil_scale(rhs)) <= 1e-13
    del want, d_out
    x_c = np.zeros_like(rhs)
    d_x = dev(x_c)
    o.cg(x_c, rhs, fixed_iters=3)
    res = g.cg_solve(d_x, d_rhs, fixed_iters=3)
    assert res["iters"] == 3
    assert rel_l2(host(d_x), x_c) <= 1e-10


def test_bicgstab_config5_full_size_five_iterations():
    w = wl.config5()
    o, g = make_pair(w)
    o.multipole_bc(w["rho"], w["G"], w["lmax"])
    g.multipole_bc(dev(w["rho"]), w["G"], w["lmax"], want_moments=False)
    got, want = gface(g, 1), o.get_ghost_face(1)
    assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max()
    x_c = np.zeros_like(w["rhs"])
    d_x = dev(x_c)
    o.bicgstab(x_c, w["rhs"], fixed_iters=5)
    res = g.bicgstab_solve(d_x, dev(w["rhs"]), fixed_iters=5)
    assert res["iters"] == 5
    assert rel_l2(host(d_x), x_c) <= 1e-10


# ---- the kernel paths agree bit for bit on pointwise work -------------------------------------------------------------
@pytest.mark.parametrize("shape", [(64, 64, 64), (96, 40, 34), (128, 128, 40)])
def test_paths_bit_identical(shape):
    w = dict(shape=shape, spacing=(0.1, 0.12, 0.09), origin=(0, 0, 0), bc=D6)
    outs = []
    for path in (pb.PATH_GENERIC, pb.PATH_PLANE):
        g = pb.Poisson(shape, w["spacing"], w["origin"], bc=D6)
        g.set_option(pb.OPT_KERNEL_PATH, path)
        faces = [dev(wl.hash_uniform(300 + f, np.arange(g.face_len(f))) - 0.5) for f in range(6)]
        g.set_ghost_faces(faces)
        phi, rhs = dev(wl.random_field(shape, 51)), dev(wl.random_field(shape, 52))
        out = torch.empty_like(phi)
        g.apply_laplacian(phi, out)
        g.rbsor_sweep(phi, rhs, 1.4, 3)
        g.mg_vcycle(phi, rhs, ncycles=1) if all(s % 8 == 0 for s in shape) else None
        outs.append((host(out), host(phi)))
    assert np.array_equal(outs[0][0], outs[1][0]), "apply: generic vs staged kernels"
    assert np.array_equal(outs[0][1], outs[1][1]), "SOR / V-cycle: generic vs fused kernels"


def test_sor_two_sweeps_per_pass_option():
    """POISSON_OPT_SOR_HALFSTEPS = 4 (two sweeps per HBM pass) gives the same bits as one sweep per pass."""
    shape = (128, 64, 48)
    outs = []
    for nhs in (2, 4):
        g = pb.Poisson(shape, (0.1, 0.1, 0.1), (0, 0, 0), bc=D6)
        g.set_option(pb.OPT_KERNEL_PATH, pb.PATH_PLANE)
        g.set_option(pb.OPT_SOR_HALFSTEPS, nhs)
        phi, rhs = dev(wl.random_field(shape, 61)), dev(wl.random_field(shape, 62))
        g.rbsor_sweep(phi, rhs, 1.7, 5)
        outs.append(host(phi))
    assert np.array_equal(outs[0], outs[1])


def test_fused_residual_restriction_option():
    """POISSON_OPT_FUSED_RESTRICT: the one-pass residual + restriction kernel gives the same bits as the two kernels."""
    shape = (128, 64, 64)
    outs = []
    for mode in (1, 2):
        g = pb.Poisson(shape, (0.1, 0.1, 0.1), (0, 0, 0), bc=D6)
        g.set_option(pb.OPT_FUSED_RESTRICT, mode)
        faces = [dev(wl.hash_uniform(400 + f, np.arange(g.face_len(f))) - 0.5) for f in range(6)]
        g.set_ghost_faces(faces)
        for precision in (pb.F64, pb.MIXED):
            for restriction in (0, 1):
                g.set_option(pb.OPT_RESTRICTION, restriction)
                phi, rhs = dev(wl.random_field(shape, 71)), dev(wl.random_field(shape, 72))
                g.mg_vcycle(phi, rhs, precision=precision, ncycles=2)
                outs.append(host(phi))
    n = len(outs) // 2
    for a, b in zip(outs[:n], outs[n:]):
        assert np.array_equal(a, b)


# ---- edge cases of the fused / staged kernels ---------------------------------------------------------------------------
N6 = (po.BC_NEUMANN0, po.BC_DIRICHLET_GHOST, po.BC_DIRICHLET_GHOST, po.BC_NEUMANN0, po.BC_NEUMANN0, po.BC_DIRICHLET_GHOST)


@pytest.mark.parametrize("shape", [(2, 2, 2), (4, 6, 2), (2, 40, 3), (66, 14, 5), (130, 30, 9), (64, 2, 70)])
@pytest.mark.parametrize("bc", [D6, N6])
def test_small_and_ragged_grids_through_the_fused_kernels(shape, bc):
    """Tiny, thin and ragged grids (tiles mostly outside the domain, runs shorter than the wavefront, one plane) with
    Dirichlet ghosts and with Neumann faces, forced through k_apply7 / k_sor_fused (kernel path 2)."""
    w = dict(shape=shape, spacing=(0.1, 0.07, 0.13), origin=(0.0, 0.1, 0.2), bc=bc)
    o, g = make_pair(w, pb.PATH_PLANE)
    faces = [wl.hash_uniform(500 + f, np.arange(o.face_len(f))) - 0.5 if bc[f] == po.BC_DIRICHLET_GHOST else None
             for f in range(6)]
    from gpu_helpers import set_faces
    set_faces(o, g, faces)
    phi_c, rhs = wl.random_field(shape, 81), wl.random_field(shape, 82)
    d_phi, d_rhs = dev(phi_c), dev(rhs)
    d_out = torch.empty_like(d_phi)
    g.apply_laplacian(d_phi, d_out)
    c = [1 / 0.1 ** 2, 1 / 0.07 ** 2, 1 / 0.13 ** 2]
    assert pointwise_scaled(host(d_out), o.apply(phi_c), 2 * sum(c) * stencil_scale(phi_c) + 1.0) <= 1e-13
    assert g.residual_norm(d_phi, d_rhs) == pytest.approx(o.residual_norm(phi_c, rhs), rel=1e-12)
    for nhs in (2, 4):
        g.set_option(pb.OPT_SOR_HALFSTEPS, nhs)
        for nsw in (1, 2, 5):
            o.rbsor(phi_c, rhs, 1.2, nsw)
            g.rbsor_sweep(d_phi, d_rhs, 1.2, nsw)
            assert pointwise_scaled(host(d_phi), phi_c, stencil_scale(phi_c, rhs * 0.002)) <= 1e-13


def test_vcycle_anisotropic_spacing_and_non_cubic_grid():
    """V-cycles on a 128 x 64 x 32 grid with three different spacings (every level has its own tile geometry)."""
    w = dict(shape=(128, 64, 32), spacing=(0.01, 0.013, 0.017), origin=(0.0, 0.0, 0.0), bc=D6)
    o, g = make_pair(w)
    from gpu_helpers import set_faces
    set_faces(o, g, [wl.hash_uniform(600 + f, np.arange(o.face_len(f))) - 0.5 for f in range(6)])
    rhs = wl.random_field(w["shape"], 91)
    for precision, tol in ((pb.F64, 1e-10), (pb.MIXED, 1e-5)):
        phi_c = np.zeros_like(rhs)
        d_phi = dev(phi_c)
        o.vcycle(phi_c, rhs, precision=precision, ncycles=3)
        g.mg_vcycle(d_phi, dev(rhs), precision=precision, ncycles=3)
        assert rel_l2(host(d_phi), phi_c) <= tol
