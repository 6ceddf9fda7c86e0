"""GPU parity of the compact radius-1 discretisations of order 4 and 6 in the
paper's multigrid: right-hand-side transform, SPAI steps with rows 4 / 6 of Table 1, Galerkin V-cycles and their residual
norms — the CUDA path through the C ABI against oracle/mgv.cpp on the same inputs (-m gpu)."""
import math

import numpy as np
import pytest
import torch

import pyoracle as po
from gpu_helpers import dev, host, make_pair, rel_l2
from paper_2605_03563_b200 import binding as pb
from paper_2605_03563_b200 import workloads as wl

pytestmark = pytest.mark.gpu
D6 = (po.BC_DIRICHLET_GHOST,) * 6


def _pair(shape, h, order):
    o, g = make_pair(dict(shape=shape, spacing=(h,) * 3, origin=(h,) * 3, bc=D6))
    g.set_option(pb.OPT_COMPACT_ORDER, order)
    return o, g


@pytest.mark.parametrize("order", [2, 4, 6])
@pytest.mark.parametrize("shape", [(31, 31, 31), (37, 20, 9), (64, 48, 40)])
def test_compact_rhs_matches_oracle(shape, order):
    o, g = _pair(shape, 1.0 / 64, order)
    ext = (shape[0] + 4, shape[1] + 4, shape[2] + 4)
    f_ext = wl.random_field(ext, 31)
    want = po.compact_rhs(f_ext, order)
    d_out = torch.empty(shape[::-1], dtype=torch.float64, device="cuda")
    g.compact_rhs(dev(f_ext), d_out)
    assert np.abs(host(d_out) - want).max() <= 1e-13 * np.abs(f_ext).max()


@pytest.mark.parametrize("order", [4, 6])
@pytest.mark.parametrize("shape", [(31, 31, 31), (63, 31, 15), (37, 20, 9), (64, 48, 40), (127, 63, 31)])
def test_compact_spai_smoother_matches_oracle(shape, order):
    o, g = _pair(shape, 1.0 / 64, order)
    rhs = wl.random_field(shape, 8) * 100
    phi_c = wl.random_field(shape, 9)
    d_phi, d_rhs = dev(phi_c), dev(rhs)
    for nsteps in (1, 2, 3):
        o.spai_smooth(phi_c, rhs, nsteps=nsteps, order=order)      # Table 1 row of the order on both sides
        g.spai_smooth(d_phi, d_rhs, nsteps=nsteps)
        assert np.abs(host(d_phi) - phi_c).max() <= 1e-13 * np.abs(phi_c).max()


@pytest.mark.parametrize("order", [4, 6])
@pytest.mark.parametrize("n,nu", [(31, 1), (63, 1), (63, 2)])
def test_compact_vcycle_matches_oracle(n, nu, order):
    h = 1.0 / (n + 1)
    o, g = _pair((n,) * 3, h, order)
    rhs = wl.two_spheres(n, cell_centred=False)["rhs"]
    for precision, tol in ((pb.F64, 1e-10), (pb.MIXED, 1e-5)):
        phi_c = np.zeros_like(rhs)
        d_phi = dev(phi_c)
        rc = o.mgv_vcycle(phi_c, rhs, nu1=nu, nu2=nu, storage_f32=precision == pb.MIXED, ncycles=4,
                          order=order)["resnorms"]
        rg = np.array(g.mgv_vcycle(d_phi, dev(rhs), nu1=nu, nu2=nu, precision=precision, ncycles=4)["resnorms"])
        assert rel_l2(host(d_phi), phi_c) <= tol
        assert np.allclose(rg, rc, rtol=1e-6 if precision == pb.F64 else 2e-2)
        assert np.all(rg[1:] < 0.1 * rg[:-1])


@pytest.mark.parametrize("order,rate", [(4, 4), (6, 6)])
def test_compact_solution_error_falls_at_the_formal_order_on_the_gpu(order, rate):
    # the whole CUDA chain on a manufactured solution (u = sin(pi x) sin(pi y) sin(2 pi z), zero on the boundary):
    # poisson_compact_rhs, then V-cycles to a residual of 1e-10; the error against u falls by 2^order per refinement
    errs = []
    for n in (15, 31, 63):
        hh = 1.0 / (n + 1)
        o, g = _pair((n,) * 3, hh, order)
        x = hh * (np.arange(-2, n + 2) + 1)
        ue = np.sin(2 * math.pi * x)[:, None, None] * np.sin(math.pi * x)[None, :, None] * np.sin(math.pi * x)[None, None, :]
        d_b = torch.empty((n,) * 3, dtype=torch.float64, device="cuda")
        g.compact_rhs(dev(-6 * math.pi ** 2 * ue), d_b)
        d_phi = torch.zeros((n,) * 3, dtype=torch.float64, device="cuda")
        res = g.mgv_vcycle(d_phi, d_b, nu1=2, nu2=2, ncycles=12, cg_rtol=1e-6)["resnorms"]
        assert res[-1] <= 1e-9 * res[0]
        errs.append(np.abs(host(d_phi) - ue[2:-2, 2:-2, 2:-2]).max())
    r = math.log2(errs[1] / errs[2])
    assert rate - 0.4 < r < rate + 0.4, errs


def test_compact_order_errors():
    o, g = make_pair(dict(shape=(15, 15, 15), spacing=(0.1,) * 3, origin=(0.1,) * 3, bc=D6))
    with pytest.raises(pb.PoissonError) as e:
        g.set_option(pb.OPT_COMPACT_ORDER, 3)
    assert e.value.code == pb.INVALID_ARG
    g.set_option(pb.OPT_COMPACT_ORDER, 4)
    g.set_ghost_faces([dev(np.ones(g.face_len(f))) for f in range(6)])
    x = torch.zeros(15 ** 3, dtype=torch.float64, device="cuda")
    with pytest.raises(pb.PoissonError) as e:     # ghost values cannot feed a 19- / 27-point stencil
        g.spai_smooth(x, x.clone())
    assert e.value.code == pb.UNSUPPORTED and "right-hand side" in str(e.value)
    g2 = pb.Poisson((15, 15, 15), (0.1, 0.1, 0.2), (0.1,) * 3, bc=D6)
    with pytest.raises(pb.PoissonError) as e:     # sixth order assumes isotropic spacing
        g2.set_option(pb.OPT_COMPACT_ORDER, 6)
    assert e.value.code == pb.UNSUPPORTED
