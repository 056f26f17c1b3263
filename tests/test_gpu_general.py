"""GPU parity of tdx_general_solve (per-line coefficients, diagonal pivoting) against the
dense LAPACK oracle.  Tolerance: the systems are random and NOT dominant, so the forward error of any backward-stable
solver is kappa(A) * eps per line; each line is gated at 50 * kappa(A_line) * eps (kappa from the oracle's dense
matrices), and the whole field at a relative residual of 1e-13."""
import numpy as np
import pytest
import torch

import general as ogen
import oracle as orc
from paper_1812_01178_b200 import binding as tdx
from paper_1812_01178_b200 import inputs

pytestmark = pytest.mark.gpu
BCS = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_DIRICHLET)
EPS = 2.220446049250313e-16


def _setup(nx, ny, nz, seed, diag_scale):
    faces = (inputs.faces_uniform(nx, 1.0), inputs.faces_uniform(ny, 1.0), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    n = nx * ny * nz
    a = inputs.uniform_pm1(seed, n, stream=1).reshape(nz, ny, nx)
    b = diag_scale * inputs.uniform_pm1(seed, n, stream=2).reshape(nz, ny, nx)
    c = inputs.uniform_pm1(seed, n, stream=3).reshape(nz, ny, nx)
    d = inputs.uniform_pm1(seed, n, stream=4).reshape(nz, ny, nx)
    return grid, a, b, c, d


def _solve(grid, direction, pivoting, a, b, c, d):
    ta, tb, tc = (torch.from_numpy(v).cuda() for v in (a, b, c))
    td = torch.from_numpy(d).cuda()
    work = torch.empty(9 * d.size + 64, dtype=torch.uint8, device="cuda")
    grid.general_solve(direction, pivoting, ta, tb, tc, td, work)
    torch.cuda.synchronize()
    assert torch.equal(ta.cpu(), torch.from_numpy(a)) and torch.equal(tb.cpu(), torch.from_numpy(b))   # coefficients untouched
    return td.cpu().numpy()


@pytest.mark.parametrize("direction,shape", [(1, (150, 48, 6)), (2, (34, 5, 40)), (1, (4, 2, 3)), (1, (5, 3, 2)), (2, (130, 1 + 1, 1 + 2))])
def test_non_dominant_random_systems_with_pivoting(direction, shape):
    nx, ny, nz = shape
    grid, a, b, c, d = _setup(nx, ny, nz, 700 + nx, 0.3)
    axis = 1 if direction == 1 else 0
    got = _solve(grid, direction, True, a, b, c, d)
    ref, A = ogen.general_solve(a, b, c, d, axis)
    cond = np.linalg.cond(A)
    n = d.shape[axis]
    err = np.max(np.abs(np.moveaxis(got - ref, axis, -1).reshape(-1, n)), axis=1)
    scale = np.max(np.abs(np.moveaxis(ref, axis, -1).reshape(-1, n)), axis=1)
    assert np.all(err <= 50 * cond * EPS * scale), float(np.max(err / (cond * EPS * scale)))
    # residual of the equations themselves
    r = b * got
    gm = np.moveaxis(got, axis, 0); rm = np.moveaxis(r, axis, 0); am = np.moveaxis(a, axis, 0); cm = np.moveaxis(c, axis, 0)
    rm[1:] += am[1:] * gm[:-1]
    rm[:-1] += cm[:-1] * gm[1:]
    assert np.max(np.abs(r - d)) <= 1e-13 * (np.max(np.abs(got)) * 3.0 + 1.0)
    grid.close()


def test_zero_diagonals_need_the_2x2_pivots():
    """Every second diagonal entry is exactly zero: plain Thomas (pivoting = 0) breaks down, the pivoting solve is exact."""
    nx, ny, nz = 64, 40, 3
    grid, a, b, c, d = _setup(nx, ny, nz, 800, 1.0)
    b[:, ::2, :] = 0.0
    a = np.sign(a) * (0.5 + np.abs(a)); c = np.sign(c) * (0.5 + np.abs(c))      # couplings bounded away from zero
    got = _solve(grid, 1, True, a, b, c, d)
    ref, A = ogen.general_solve(a, b, c, d, 1)
    cond = np.linalg.cond(A)
    err = np.max(np.abs(np.moveaxis(got - ref, 1, -1).reshape(-1, ny)), axis=1)
    scale = np.max(np.abs(np.moveaxis(ref, 1, -1).reshape(-1, ny)), axis=1)
    assert np.all(err <= 50 * cond * EPS * scale)
    bad = _solve(grid, 1, False, a, b, c, d)
    assert not np.all(np.isfinite(bad))                          # b_0 = 0: the first division of plain Thomas
    grid.close()


def test_dominant_systems_equal_thomas_with_and_without_pivoting():
    nx, ny, nz = 32, 30, 4
    grid, a, b, c, d = _setup(nx, ny, nz, 810, 1.0)
    b = 2.5 + np.abs(b)
    x1 = _solve(grid, 1, True, a, b, c, d)
    x0 = _solve(grid, 1, False, a, b, c, d)
    assert np.array_equal(x0, x1)                                # dominant rows always take the 1x1 pivot
    for k, i in ((0, 0), (3, 31), (2, 7)):
        ref = orc.thomas(np.ascontiguousarray(a[k, :, i]), np.ascontiguousarray(b[k, :, i]), np.ascontiguousarray(c[k, :, i]),
                         np.ascontiguousarray(d[k, :, i]))
        assert np.max(np.abs(x1[k, :, i] - ref)) <= 1e-12 * np.max(np.abs(ref))
    with pytest.raises(tdx.TdxError) as e:
        _solve(grid, 0, True, a, b, c, d)
    assert e.value.status == tdx.ERR_UNSUPPORTED
    grid.close()
