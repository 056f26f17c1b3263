"""GPU parity of tdx_general_solve / tdx_general_cyclic_solve (per-line coefficients, diagonal pivoting; SURVEY 8(f) N4,
PAPER.md:L174) against the dense LAPACK oracle, along x, y and z.  Tolerance: the random systems are NOT dominant, so the
forward error of any backward-stable solver is kappa(A) * eps per line; each line is gated at 50 * kappa(A_line) * eps
(kappa from the oracle's dense matrices), and the whole field at a relative residual of 1e-13.  The partition kernel
hands lines with a numerically singular partition block to the per-line path: both paths are exercised (the count of
such lines is asserted: none on weakly dominant systems, some on the random ones)."""
import numpy as np
import pytest
import torch

import general as ogen
import oracle as orc
from paper_1812_01178_b200 import binding as tdx
from paper_1812_01178_b200 import inputs

pytestmark = pytest.mark.gpu
BCS = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_DIRICHLET)
AXIS = {0: 2, 1: 1, 2: 0}                                       # array axis of a sweep direction
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


def _solve(grid, direction, pivoting, a, b, c, d, cyclic=False, method=tdx.GENERAL_FORCE_PARTITION, pivot_partitions=False):
    """method: the partition kernel is forced wherever it applies (it is the default only for x lines), so that it is the
    path under test; periodic lines and very short lines take the per-line kernel whatever is asked."""
    n = d.shape[AXIS[direction]]
    P = max(2, -(-n // 8))
    pivoting = int(pivoting) | (method if (not cyclic and n // P >= 2 and P <= 512) else 0) | (tdx.GENERAL_PIVOT_PARTITIONS if pivot_partitions else 0)
    ta, tb, tc = (torch.from_numpy(v).cuda() for v in (a, b, c))
    td = torch.from_numpy(d).cuda()
    work = torch.empty(25 * d.size + 64, dtype=torch.uint8, device="cuda")
    (grid.general_cyclic_solve if cyclic else grid.general_solve)(direction, pivoting, ta, tb, tc, td, work)
    torch.cuda.synchronize()
    assert torch.equal(ta.cpu(), torch.from_numpy(a)) and torch.equal(tb.cpu(), torch.from_numpy(b))   # coefficients untouched
    return td.cpu().numpy()


@pytest.mark.parametrize("pivot_partitions", [False, True])       # optimistic plain elimination first / pivots inside the partitions
@pytest.mark.parametrize("cyclic", [False, True])
@pytest.mark.parametrize("direction,shape", [(1, (150, 48, 6)), (2, (34, 5, 40)), (1, (4, 2, 3)), (1, (5, 3, 2)), (2, (130, 1 + 1, 1 + 2)),
                                             (0, (64, 9, 7)), (0, (203, 5, 3)), (0, (9, 4, 4)), (1, (32, 288, 2)), (1, (17, 101, 3))])
def test_non_dominant_random_systems_with_pivoting(direction, shape, cyclic, pivot_partitions):
    nx, ny, nz = shape
    grid, a, b, c, d = _setup(nx, ny, nz, 700 + nx, 0.3)
    axis = AXIS[direction]
    if cyclic and d.shape[axis] < 3:
        pytest.skip("periodic lines need n >= 3")
    if cyclic and pivot_partitions:
        pytest.skip("periodic lines take the per-line kernel either way")
    got = _solve(grid, direction, True, a, b, c, d, cyclic, pivot_partitions=pivot_partitions)
    ref, A = ogen.general_solve(a, b, c, d, axis, cyclic)
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
    if cyclic:
        rm[0] += am[0] * gm[-1]
        rm[-1] += cm[-1] * gm[0]
    assert np.max(np.abs(r - d)) <= 1e-13 * (np.max(np.abs(got)) * 3.0 + 1.0)
    nfb = grid.general_fallback_count()
    nlines = d.size // n
    assert 0 <= nfb <= nlines
    if not cyclic and n >= 64:
        assert nfb > 0                                           # random non-dominant blocks: some line always has a bad 8-row block
    grid.close()


@pytest.mark.parametrize("direction", [0, 1, 2])
def test_weakly_dominant_per_line_systems_take_the_partition_path_only(direction):
    """The paper's case (L172-174): Poisson-like rows |b| = |a| + |c| + eps with a different eps on every line, given as
    explicit per-line coefficients.  No partition block is singular: no line may fall back, and the result is within
    the kappa * eps gate of the dense oracle."""
    nx, ny, nz = 40, 36, 34
    grid, a, b, c, d = _setup(nx, ny, nz, 900 + direction, 1.0)
    a = -(0.2 + np.abs(a)); c = -(0.2 + np.abs(c))
    eps = 10.0 ** (-6.0 * np.abs(b))                                               # 1e-6 ... 1 per entry
    axis = AXIS[direction]
    eps = np.broadcast_to(np.take(eps, [0], axis=axis), eps.shape).copy()          # one shift per line
    am = np.moveaxis(a, axis, 0); cm = np.moveaxis(c, axis, 0)
    am[0] = 0.0; cm[-1] = 0.0                                                      # the cut ends, so that every row is dominant
    b = -(a + c) + eps
    got = _solve(grid, direction, True, a, b, c, d)
    assert grid.general_fallback_count() == 0
    ref, A = ogen.general_solve(a, b, c, d, axis)
    cond = np.linalg.cond(A)
    n = d.shape[axis]
    err = np.max(np.abs(np.moveaxis(got - ref, axis, -1).reshape(-1, n)), axis=1)
    scale = np.max(np.abs(np.moveaxis(ref, axis, -1).reshape(-1, n)), axis=1)
    assert np.all(err <= 50 * cond * EPS * scale), float(np.max(err / (cond * EPS * scale)))
    assert np.array_equal(got, _solve(grid, direction, False, a, b, c, d))         # dominant rows always take the 1x1 pivot
    lines = _solve(grid, direction, True, a, b, c, d, method=tdx.GENERAL_FORCE_LINES)   # the other method: same answer to the gate
    errl = np.max(np.abs(np.moveaxis(lines - ref, axis, -1).reshape(-1, n)), axis=1)
    assert np.all(errl <= 50 * cond * EPS * scale)
    dflt = _solve(grid, direction, True, a, b, c, d, method=0)                     # default: the partition method in every direction
    assert np.array_equal(dflt, got)
    grid.close()


@pytest.mark.parametrize("direction", [0, 1, 2])
def test_default_method_is_chosen_on_the_device_from_a_sample_of_the_rows(direction):
    """method = 0 with pivoting: a sample of the rows decides on the device (no host synchronisation) -- mostly non-dominant
    rows: the per-line kernel solves every line at once (bit-equal to TDX_GENERAL_FORCE_LINES, the count of lines that left
    the partition method = all); dominant rows, also with a few wild lines in between: the optimistic partition pass
    (bit-equal to TDX_GENERAL_FORCE_PARTITION)."""
    nx, ny, nz = 72, 64, 40
    grid, a, b, c, d = _setup(nx, ny, nz, 1300 + direction, 0.3)
    nlines = d.size // d.shape[AXIS[direction]]
    dflt = _solve(grid, direction, True, a, b, c, d, method=0)
    n_dflt = grid.general_fallback_count()
    forced_l = _solve(grid, direction, True, a, b, c, d, method=tdx.GENERAL_FORCE_LINES)
    forced_p = _solve(grid, direction, True, a, b, c, d, method=tdx.GENERAL_FORCE_PARTITION)
    n_part = grid.general_fallback_count()
    assert np.array_equal(dflt, forced_l) and n_dflt == nlines and 0 < n_part < nlines
    # dominant rows with 5 % wild lines: the partition pass, whatever the direction
    axis = AXIS[direction]
    n = d.shape[axis]
    pick = inputs.uniform_pm1(78, nlines, stream=5)
    shape = list(d.shape); shape[axis] = 1
    wild = np.broadcast_to((0.5 * (pick + 1.0) < 0.05).reshape(shape), d.shape)
    b2 = np.where(wild, b, np.abs(a) + np.abs(c) + 0.5 + np.abs(b))
    dflt = _solve(grid, direction, True, a, b2, c, d, method=0)
    n_dflt = grid.general_fallback_count()
    forced_p = _solve(grid, direction, True, a, b2, c, d, method=tdx.GENERAL_FORCE_PARTITION)
    assert np.array_equal(dflt, forced_p) and n_dflt == grid.general_fallback_count() <= int(wild.sum()) // n
    grid.close()


@pytest.mark.parametrize("nx", [256, 512, 768, 1024, 2048])
@pytest.mark.parametrize("kind", ["weak", "strong", "random"])
def test_x_lines_of_many_partitions(nx, kind):
    """Long x lines: 32 to 256 partitions per line (1 to 8 warps of one CTA work on a line; 5 to 8 reduction steps), several
    lines per CTA with a partly filled last CTA.  'weak': |b| = |a| + |c| + eps, eps down to 1e-6 (couplings that do not
    decay: every reduction step runs; lines of tame blocks are accepted WITHOUT a residual check, so only the oracle sees a
    wrong reduced solve); 'strong': decayed spikes (the early exit); 'random': non-dominant lines, re-solved ones included.
    Gate: kappa * eps per line against the dense LAPACK oracle."""
    ny, nz = 3, 2
    grid, a, b, c, d = _setup(nx, ny, nz, 1200 + nx, 0.3 if kind == "random" else 1.0)
    if kind != "random":
        a = -(0.2 + np.abs(a)); c = -(0.2 + np.abs(c))
        eps = 10.0 ** (-6.0 * np.abs(b)) if kind == "weak" else 2.0 + np.abs(b)
        eps = np.broadcast_to(eps[:, :, :1], eps.shape).copy()                      # one shift per line
        a[:, :, 0] = 0.0; c[:, :, -1] = 0.0
        b = -(a + c) + eps
    got = _solve(grid, 0, True, a, b, c, d)
    assert tdx.last_launch().startswith("k_general_part<8,0,1,1>") and "block=(%d," % (nx // 8) in tdx.last_launch().replace(" ", "")
    nfb = grid.general_fallback_count()
    if kind != "random":
        assert nfb == 0
    ref, A = ogen.general_solve(a, b, c, d, 2)
    cond = np.linalg.cond(A)
    err = np.max(np.abs(got - ref).reshape(-1, nx), axis=1)
    scale = np.max(np.abs(ref).reshape(-1, nx), axis=1)
    assert np.all(err <= 50 * cond * EPS * scale), float(np.max(err / (cond * EPS * scale)))
    grid.close()


@pytest.mark.parametrize("direction", [0, 1, 2])
@pytest.mark.parametrize("share", [0.06, 0.6])
def test_mixed_lines_only_the_lines_that_need_pivots_are_re_solved(direction, share):
    """Dominant lines with a share of lines in between whose every second diagonal entry is exactly zero (plain elimination
    divides by zero there; the 2x2 pivots solve them).  The re-solve of the lines the partition kernel does not vouch for has
    two forms (k_general_lines: from the list when they are few, every line in memory order with the accepted ones skipped
    when they are more than a third): both must leave the accepted lines alone and solve the others to the gate, and the
    count of re-solved lines is exactly the number of zero-diagonal lines."""
    nx, ny, nz = {0: (64, 24, 20), 1: (40, 64, 12), 2: (24, 20, 64)}[direction]
    grid, a, b, c, d = _setup(nx, ny, nz, 950 + direction, 1.0)
    axis = AXIS[direction]
    n = d.shape[axis]
    a = np.sign(a) * (0.5 + np.abs(a)); c = np.sign(c) * (0.5 + np.abs(c))          # couplings bounded away from zero
    pick = inputs.uniform_pm1(77, d.size // n, stream=5)                            # one draw per line
    shape = list(d.shape); shape[axis] = 1
    wild = np.broadcast_to((0.5 * (pick + 1.0) < share).reshape(shape), d.shape)
    nwild = int(wild.sum()) // n
    assert 0 < nwild < d.size // n
    odd = np.zeros(n, dtype=bool); odd[::2] = True
    shp = [1, 1, 1]; shp[axis] = n
    bz = np.where(odd.reshape(shp), 0.0, b)                                          # zero on every second row
    b = np.where(wild, bz, np.abs(a) + np.abs(c) + 0.5 + np.abs(b))
    got = _solve(grid, direction, True, a, b, c, d)
    nfb = grid.general_fallback_count()
    assert nfb == nwild, (nfb, nwild)
    assert (nfb * 3 > d.size // n) == (share > 0.5), (nfb, d.size // n)              # the branch this case is meant to take
    ref, A = ogen.general_solve(a, b, c, d, axis)
    cond = np.linalg.cond(A)
    err = np.max(np.abs(np.moveaxis(got - ref, axis, -1).reshape(-1, n)), axis=1)
    scale = np.max(np.abs(np.moveaxis(ref, axis, -1).reshape(-1, n)), axis=1)
    assert np.all(err <= 50 * cond * EPS * scale), float(np.max(err / (cond * EPS * scale)))
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
    got_pp = _solve(grid, 1, True, a, b, c, d, pivot_partitions=True)
    assert np.all(np.max(np.abs(np.moveaxis(got_pp - ref, 1, -1).reshape(-1, ny)), axis=1) <= 50 * cond * EPS * np.max(np.abs(np.moveaxis(ref, 1, -1).reshape(-1, ny)), axis=1))
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
    xx = _solve(grid, 0, True, a, b, c, d)                       # x lines as well (round 1: TDX_ERR_UNSUPPORTED)
    refx, _ = ogen.general_solve(a, b, c, d, 2)
    assert np.max(np.abs(xx - refx)) <= 1e-12 * np.max(np.abs(refx))
    grid.close()
