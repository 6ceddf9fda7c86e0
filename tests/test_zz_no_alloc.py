"""poisson_residual_norm_static (include/poisson.h): the residual norm through the entry point that allocates nothing —
its block partials live in a static device array of the library — against the handle-based poisson_residual_norm on
the same inputs, twice in a row (the second call on a smaller grid with other data, so stale scratch contents beyond
its own partials and from the first call must not leak into it).  Collected last (file name) on purpose."""
import numpy as np
import pytest
import torch

from paper_2605_03563_b200 import binding as pb
from paper_2605_03563_b200 import workloads as wl

pytestmark = pytest.mark.gpu

D6 = (pb.BC_DIRICHLET_GHOST,) * 6
RTOL = 1e-12   # the tolerance of the other norm / reduction comparisons (different summation order, fp64)


def _case(shape, spacing, seed):
    g = pb.Poisson(shape, spacing, (0.0, 0.0, 0.0), bc=D6)   # fresh handle: ghost values zero
    phi = torch.from_numpy(wl.random_field(shape, seed)).to("cuda").contiguous()
    rhs = torch.from_numpy(wl.random_field(shape, seed + 1)).to("cuda").contiguous()
    return g, phi, rhs


def test_static_scratch_residual_norm_matches_the_handle_path_twice_in_a_row():
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    cases = [((160, 72, 50), (0.1, 0.12, 0.09), 901), ((33, 9, 17), (0.2, 0.1, 0.3), 903)]
    prepared = [(shape, spacing) + _case(shape, spacing, seed) for shape, spacing, seed in cases]
    wants = [g.residual_norm(phi, rhs) for _, _, g, phi, rhs in prepared]
    torch.cuda.synchronize()
    for n, ((shape, spacing, g, phi, rhs), want) in enumerate(zip(prepared, wants)):
        free_before = torch.cuda.mem_get_info()[0]
        pb.residual_norm_static(shape, spacing, phi, rhs, out, stream)
        torch.cuda.synchronize()
        got = float(out.item())
        assert want > 0 and abs(got - want) <= RTOL * want, (shape, got, want)
        if n > 0:   # (the first call may load the module) no device memory was taken by the call
            assert torch.cuda.mem_get_info()[0] >= free_before
    # and again on the first inputs: same bits as the first time (fixed summation order, shared scratch overwritten)
    shape, spacing, g, phi, rhs = prepared[0]
    pb.residual_norm_static(shape, spacing, phi, rhs, out, stream)
    torch.cuda.synchronize()
    first = float(out.item())
    pb.residual_norm_static(shape, spacing, phi, rhs, out, stream)
    torch.cuda.synchronize()
    assert float(out.item()) == first and abs(first - wants[0]) <= RTOL * wants[0]


def test_static_scratch_rejects_grids_beyond_its_size_and_host_pointers():
    x = torch.zeros(8, dtype=torch.float64, device="cuda")
    with pytest.raises(pb.PoissonError) as e:
        pb.residual_norm_static((1024, 1024, 600), (0.1,) * 3, x, x, x)    # 32 * 128 * 38 blocks > 32768
    assert e.value.code == pb.UNSUPPORTED and "static scratch" in str(e.value)
    h = np.zeros(8)
    with pytest.raises(pb.PoissonError) as e:
        pb.residual_norm_static((2, 2, 2), (0.1,) * 3, h, x, x)
    assert e.value.code == pb.INVALID_ARG
    with pytest.raises(pb.PoissonError) as e:
        pb.residual_norm_static((2, 0, 2), (0.1,) * 3, x, x, x)
    assert e.value.code == pb.INVALID_ARG
