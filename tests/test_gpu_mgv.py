"""GPU parity of the paper's own multigrid (rows f1, f2): SPAI smoother, vertex-centred Galerkin V-cycle, fp32 coarse
storage — the CUDA path through the C ABI against oracle/mgv.cpp on the same inputs (-m gpu)."""
import numpy as np
import pytest
import torch

import pyoracle as po
from gpu_helpers import dev, host, make_pair, rel_l2, set_faces
from paper_2605_03563_b200 import binding as pb
from paper_2605_03563_b200 import workloads as wl

pytestmark = pytest.mark.gpu
D6 = (po.BC_DIRICHLET_GHOST,) * 6


def _pair(shape, h, seed=None):
    w = dict(shape=shape, spacing=(h,) * 3, origin=(h,) * 3, bc=D6)
    o, g = make_pair(w)
    if seed is not None:
        set_faces(o, g, [wl.hash_uniform(seed + f, np.arange(o.face_len(f))) - 0.5 for f in range(6)])
    return o, g


@pytest.mark.parametrize("shape", [(31, 31, 31), (63, 31, 15), (37, 20, 9), (64, 48, 40), (127, 63, 31)])
def test_spai_smoother_matches_oracle(shape):
    o, g = _pair(shape, 1.0 / 64, seed=11)
    rhs = wl.random_field(shape, 8) * 100
    phi_c = wl.random_field(shape, 9)
    d_phi, d_rhs = dev(phi_c), dev(rhs)
    for nsteps in (1, 2, 3):
        o.spai_smooth(phi_c, rhs, nsteps=nsteps)
        g.spai_smooth(d_phi, d_rhs, nsteps=nsteps)
        # pointwise: per-step differences are rounding-order only (a 27-term sum against partial sums)
        assert np.abs(host(d_phi) - phi_c).max() <= 1e-13 * np.abs(phi_c).max()
    # custom coefficients travel through the ABI
    sp = (1.1, 0.15, 0.03, 0.01, 0.002)
    o.spai_smooth(phi_c, rhs, spai=sp, nsteps=2)
    g.spai_smooth(d_phi, d_rhs, spai=sp, nsteps=2)
    assert np.abs(host(d_phi) - phi_c).max() <= 1e-13 * np.abs(phi_c).max()


@pytest.mark.parametrize("n,nu", [(31, 1), (63, 1), (63, 2), (63, 3)])
def test_mgv_vcycle_two_spheres_matches_oracle_and_table2(n, nu):
    w = wl.two_spheres(n, cell_centred=False)
    o, g = make_pair(w)
    set_faces(o, g, wl.analytic_ghost_faces(w, w["potential"]))
    for precision, tol in ((pb.F64, 1e-10), (pb.MIXED, 1e-5)):
        phi_c = np.zeros_like(w["rhs"])
        d_phi = dev(phi_c)
        rc = o.mgv_vcycle(phi_c, w["rhs"], nu1=nu, nu2=nu, storage_f32=precision == pb.MIXED, ncycles=4)["resnorms"]
        rg = np.array(g.mgv_vcycle(d_phi, dev(w["rhs"]), nu1=nu, nu2=nu, precision=precision, ncycles=4)["resnorms"])
        assert rel_l2(host(d_phi), phi_c) <= tol
        assert np.allclose(rg, rc, rtol=1e-6 if precision == pb.F64 else 2e-2)
    if n == 63:   # the CUDA path reproduces the paper's convergence factors too (tests/golden/paper_table2_rho.txt)
        want, m = {1: (0.102, 4), 2: (0.028, 3), 3: (0.013, 2)}[nu]
        assert (rg[m] / rg[0]) ** (1.0 / m) == pytest.approx(want, rel=0.2)


def test_mgv_vcycle_anisotropic_shape_and_early_coarsest_level():
    shape = (63, 31, 47)     # 47 -> 23 -> 11 -> 5; 31 -> 15 -> 7 -> 3: three coarse levels
    o, g = _pair(shape, 1.0 / 64, seed=21)
    rhs = wl.random_field(shape, 5) * 50
    for cn in (3, 7):
        phi_c = np.zeros_like(rhs)
        d_phi = dev(phi_c)
        rc = o.mgv_vcycle(phi_c, rhs, nu1=2, nu2=1, coarsest_n=cn, cg_rtol=1e-6, ncycles=3)["resnorms"]
        rg = np.array(g.mgv_vcycle(d_phi, dev(rhs), nu1=2, nu2=1, coarsest_n=cn, cg_rtol=1e-6, ncycles=3)["resnorms"])
        assert rel_l2(host(d_phi), phi_c) <= 1e-10
        assert np.allclose(rg, rc, rtol=1e-6)
        assert rg[3] / rg[0] < 1e-3


def test_mgv_host_entry_and_errors():
    w = wl.two_spheres(31, cell_centred=False)
    o, g = make_pair(w)
    set_faces(o, g, wl.analytic_ghost_faces(w, w["potential"]))
    h_phi, h_rhs = np.zeros_like(w["rhs"]), np.ascontiguousarray(w["rhs"])
    g.mgv_vcycle_host(h_phi, h_rhs, ncycles=2)
    d_phi = dev(np.zeros_like(w["rhs"]))
    g.mgv_vcycle(d_phi, dev(w["rhs"]), ncycles=2)
    assert np.array_equal(h_phi, host(d_phi))
    phi_c = np.zeros_like(w["rhs"])
    o.mgv_vcycle(phi_c, w["rhs"], ncycles=2)
    assert rel_l2(h_phi, phi_c) <= 1e-10
    x = torch.zeros(32 ** 3, device="cuda", dtype=torch.float64)
    with pytest.raises(pb.PoissonError) as e:      # even sizes admit no vertex-centred coarse level
        pb.Poisson((32, 32, 32), (0.1,) * 3, bc=D6).mgv_vcycle(x, x.clone())
    assert e.value.code == pb.UNSUPPORTED
    with pytest.raises(pb.PoissonError) as e:      # isotropic spacing only
        pb.Poisson((31, 31, 31), (0.1, 0.1, 0.2), bc=D6).spai_smooth(x, x.clone())
    assert e.value.code == pb.UNSUPPORTED
