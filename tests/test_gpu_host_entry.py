"""The six *_host entry points (include/poisson.h "End-to-end variants with HOST buffers") against the oracle and
against their device twins (-m gpu).  bench.py's `e2e` leg runs through exactly these calls."""
import numpy as np
import pytest
import torch

import pyoracle as po
from gpu_helpers import dev, host, make_pair, pointwise_scaled, rel_l2, stencil_scale
from paper_2605_03563_b200 import binding as pb
from paper_2605_03563_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _buf(a, pinned):
    """Host buffer for the C ABI: pageable numpy array, or a numpy view of pinned torch memory."""
    if not pinned:
        return np.ascontiguousarray(a).copy(), None
    t = torch.from_numpy(np.ascontiguousarray(a)).clone().pin_memory()
    return t.numpy(), t   # keep t alive


@pytest.mark.parametrize("pinned", [False, True])
def test_apply_rbsor_vcycle_host_match_oracle_and_device_twins(pinned):
    w = wl.config3(32)
    o, g = make_pair(w)
    # multipole_bc_host: moments and ghost faces
    h_rho, keep0 = _buf(w["rho"], pinned)
    q_c = o.multipole_bc(w["rho"], w["G"], w["lmax"])
    q_g = np.array(g.multipole_bc_host(h_rho, w["G"], w["lmax"]))
    for l in range(w["lmax"] + 1):
        sl = slice(l * l, (l + 1) * (l + 1))
        assert np.abs(q_g[sl] - q_c[sl]).max() <= 1e-12 * np.abs(q_c[sl]).max() + 1e-16 * abs(q_c[0])
    for f in range(6):
        buf = torch.empty(g.face_len(f), device="cuda", dtype=torch.float64)
        g.get_ghost_face(f, buf)
        want = o.get_ghost_face(f)
        assert np.abs(host(buf) - want).max() <= 1e-12 * np.abs(want).max()
    # apply_laplacian_host
    phi = wl.random_field(w["shape"], 5)
    h_phi, keep1 = _buf(phi, pinned)
    h_out, keep2 = _buf(np.zeros_like(phi), pinned)
    g.apply_laplacian_host(h_phi, h_out)
    want = o.apply(phi)
    scale = 2 * 3 / w["spacing"][0] ** 2 * stencil_scale(phi) + 1.0
    assert pointwise_scaled(h_out, want, scale) <= 1e-13
    d_out = torch.empty(phi.shape, device="cuda", dtype=torch.float64)
    g.apply_laplacian(dev(phi), d_out)
    assert np.array_equal(h_out, host(d_out))          # bit-identical to the device twin
    assert np.array_equal(h_phi, phi)                  # the input buffer is untouched
    # rbsor_sweep_host with the residual norm
    phi_c = phi.copy()
    rn_c = o.rbsor(phi_c, w["rhs"], 1.4, 3, want_resnorm=True)
    h_rhs, keep3 = _buf(w["rhs"], pinned)
    rn_g = g.rbsor_sweep_host(h_phi, h_rhs, 1.4, 3, want_resnorm=True)
    d = 2 * 3 / w["spacing"][0] ** 2
    assert pointwise_scaled(h_phi, phi_c, stencil_scale(phi_c, w["rhs"] / d)) <= 1e-13
    assert rn_g == pytest.approx(rn_c, rel=1e-10)
    d_phi = dev(phi)
    g.rbsor_sweep(d_phi, dev(w["rhs"]), 1.4, 3)
    assert np.array_equal(h_phi, host(d_phi))
    # mg_vcycle_host, fp64 and mixed
    for precision, tol in ((pb.F64, 1e-10), (pb.MIXED, 1e-5)):
        x_c = np.zeros_like(phi)
        rc = o.vcycle(x_c, w["rhs"], precision=precision, ncycles=3)["resnorms"]
        h_x, keep4 = _buf(np.zeros_like(phi), pinned)
        rg = np.array(g.mg_vcycle_host(h_x, h_rhs, precision=precision, ncycles=3)["resnorms"])
        assert rel_l2(h_x, x_c) <= tol
        assert np.allclose(rg, rc, rtol=1e-6 if precision == pb.F64 else 2e-2)
        d_x = dev(np.zeros_like(phi))
        g.mg_vcycle(d_x, dev(w["rhs"]), precision=precision, ncycles=3)
        assert np.array_equal(h_x, host(d_x))


@pytest.mark.parametrize("pinned", [False, True])
def test_cg_and_bicgstab_host_match_oracle_and_device_twins(pinned):
    w = wl.config2(32)
    o, g = make_pair(w)
    o.multipole_bc(w["rho"], w["G"], w["lmax"])
    g.multipole_bc_host(np.ascontiguousarray(w["rho"]), w["G"], w["lmax"], want_moments=False)
    h_rhs, keep0 = _buf(w["rhs"], pinned)
    x_c = np.zeros_like(w["rhs"])
    o.cg(x_c, w["rhs"], fixed_iters=25)
    h_x, keep1 = _buf(np.zeros_like(x_c), pinned)
    res = g.cg_solve_host(h_x, h_rhs, fixed_iters=25)
    assert res["status"] == pb.OK and res["iters"] == 25
    assert rel_l2(h_x, x_c) <= 1e-10
    d_x = dev(np.zeros_like(x_c))
    g.cg_solve(d_x, dev(w["rhs"]), fixed_iters=25)
    assert np.array_equal(h_x, host(d_x))
    # soft status travels through the host variant, and the iterate still comes back (warm start)
    h_x[...] = 0.0
    res = g.cg_solve_host(h_x, h_rhs, rtol=1e-12, max_iter=5)
    assert res["status"] == pb.NOT_CONVERGED and res["iters"] == 5 and np.abs(h_x).max() > 0
    res = g.cg_solve_host(h_x, h_rhs, rtol=1e-8, max_iter=500)
    assert res["status"] == pb.OK
    assert o.residual_norm(h_x, w["rhs"]) <= 10 * 1e-8 * o.residual_norm(np.zeros_like(h_x), w["rhs"])

    w = wl.config5(32, 16, 32)
    o, g = make_pair(w)
    o.multipole_bc(w["rho"], w["G"], w["lmax"])
    g.multipole_bc_host(np.ascontiguousarray(w["rho"]), w["G"], w["lmax"], want_moments=False)
    h_rhs, keep2 = _buf(w["rhs"], pinned)
    x_c = np.zeros_like(w["rhs"])
    o.bicgstab(x_c, w["rhs"], fixed_iters=5)
    h_x, keep3 = _buf(np.zeros_like(x_c), pinned)
    res = g.bicgstab_solve_host(h_x, h_rhs, fixed_iters=5)
    assert res["status"] == pb.OK and res["iters"] == 5
    assert rel_l2(h_x, x_c) <= 1e-10
    d_x = dev(np.zeros_like(x_c))
    g.bicgstab_solve(d_x, dev(w["rhs"]), fixed_iters=5)
    assert np.array_equal(h_x, host(d_x))


def test_host_entry_points_reject_null_pointers():
    g = pb.Poisson((8, 8, 8), (0.1,) * 3, bc=(po.BC_DIRICHLET_GHOST,) * 6)
    a = np.zeros((8, 8, 8))
    for call in (lambda: g.apply_laplacian_host(None, a), lambda: g.rbsor_sweep_host(a, None, 1.0, 1),
                 lambda: g.cg_solve_host(None, a), lambda: g.bicgstab_solve_host(a, None),
                 lambda: g.mg_vcycle_host(None, a), lambda: g.multipole_bc_host(None, 1.0, 2)):
        with pytest.raises(pb.PoissonError) as e:
            call()
        assert e.value.code == pb.INVALID_ARG
