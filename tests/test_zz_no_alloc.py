"""The entry point that allocates nothing (tdx_helmholtz_thomas_lines_static: scratch in a static device array of the
library, include/tdx.h) against the existing path (tdx_helmholtz_wavenumber_solve, mode THOMAS, per-line shifts: scratch
in a workspace the grid cudaMallocs) -- same kernel, so the results must agree to the tests' 1e-12 (they are bit-equal) --
on two calls in a row with different right-hand sides (the array keeps the first call's contents), against the oracle,
and the refusal of sizes beyond the static array.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

import oracle as orc
from paper_1812_01178_b200 import binding as tdx
from paper_1812_01178_b200 import inputs

pytestmark = pytest.mark.gpu
BCS = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
TOL = 1e-12


def relerr(x, ref):
    return float(np.max(np.abs(x - ref)) / np.max(np.abs(ref)))


def test_static_scratch_solve_matches_the_allocating_path_twice_in_a_row():
    nx, ny, nz = 96, 72, 40                                      # ragged: nx not a multiple of the 128-thread block
    nm = nz // 2 + 1
    assert nx * ny * nm <= tdx.STATIC_SCRATCH_DOUBLES
    yf = inputs.faces_tanh_one_sided(ny, 3.0)
    grid = tdx.Grid(nx, ny, nz, inputs.faces_uniform(nx, 2.0), yf, inputs.faces_uniform(nz, 1.0), bcs=BCS)
    kx2 = inputs.modified_wavenumbers_x(nx, 2.0)
    kz2 = inputs.modified_wavenumbers_z(nz, 1.0)
    dkx, dkz = torch.from_numpy(kx2).cuda(), torch.from_numpy(kz2).cuda()
    tdx.static_scratch_setup(0)
    for call, seed in enumerate((41, 42)):                       # two calls in a row, different data
        rhs = inputs.rhs_complex_uniform((nm, ny, nx), seed) * (1.0 + 9.0 * call)
        a = torch.from_numpy(rhs).cuda()
        b = torch.from_numpy(rhs).cuda()
        grid.helmholtz_wavenumber_solve(tdx.MODE_THOMAS, 1, kx2, kz2, a)          # existing path: grid-owned workspace
        n0 = tdx.kernel_launch_count()
        grid.helmholtz_thomas_lines_static(nm, dkx, dkz, b)                      # static scratch, device wavenumbers
        assert tdx.kernel_launch_count() == n0 + 1
        torch.cuda.synchronize()
        got, want = b.cpu().numpy(), a.cpu().numpy()
        assert relerr(got, want) < TOL, (call, relerr(got, want))
        ref = orc.helmholtz_solve(rhs.copy(), yf, kx2, kz2, orc.MODE_THOMAS, 1)
        assert relerr(got, ref) < TOL, (call, relerr(got, ref))
        assert got[0, 0, 0] == 0.0                               # the pinned point of mode (0, 0)
    grid.close()


def test_static_scratch_limit_is_enforced_before_any_launch():
    nx, ny, nz = 256, 128, 256                                   # 256 * 128 * 129 doubles > the static array
    nm = nz // 2 + 1
    assert nx * ny * nm > tdx.STATIC_SCRATCH_DOUBLES
    grid = tdx.Grid(nx, ny, nz, inputs.faces_uniform(nx, 1.0), inputs.faces_uniform(ny, 1.0), inputs.faces_uniform(nz, 1.0), bcs=BCS)
    dkx = torch.zeros(nx, dtype=torch.float64, device="cuda")
    dkz = torch.ones(nm, dtype=torch.float64, device="cuda")
    t = torch.ones(16, dtype=torch.complex128, device="cuda")    # never touched: the size check comes first
    n0 = tdx.kernel_launch_count()
    with pytest.raises(tdx.TdxError) as e:
        grid.helmholtz_thomas_lines_static(nm, dkx, dkz, t)
    assert e.value.status == tdx.ERR_UNSUPPORTED and "TDX_STATIC_SCRATCH_DOUBLES" in str(e.value)
    assert tdx.kernel_launch_count() == n0
    with pytest.raises(tdx.TdxError) as e:
        grid.helmholtz_thomas_lines_static(0, dkx, dkz, t)
    assert e.value.status == tdx.ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert bool((t == 1).all())
    grid.close()
