"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded inputs.
Bars (BASELINE.json north_star): PPT and THOMAS within 1e-12 relative max-norm of the exact oracle solution; PDD within
1e-10 wherever the a-priori dropped bound is <= 1e-11 (reading A9) and, everywhere, within 1e-12 of the
oracle's own step-by-step PDD; partition map / layout bit-exact."""
import numpy as np
import pytest
import torch

import oracle as orc
from paper_1812_01178_b200 import binding as tdx
from paper_1812_01178_b200 import configs, inputs

pytestmark = pytest.mark.gpu

TOL_EXACT = 1e-12
TOL_PDD = 1e-10
BCS = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
MODES = {"thomas": tdx.MODE_THOMAS, "pdd": tdx.MODE_PDD, "ppt": tdx.MODE_PPT}


def relerr(x, ref):
    return float(np.max(np.abs(x - ref)) / np.max(np.abs(ref)))


def gpu_sweep(grid, field, direction, mode, P, alpha):
    t = torch.from_numpy(field).cuda()
    grid.adi_sweep(direction, mode, P, alpha, t)
    torch.cuda.synchronize()
    return t.cpu().numpy()


def check_sweep(grid, faces, bcs, field, direction, mode_name, P, alpha):
    mode = MODES[mode_name]
    out = gpu_sweep(grid, field, direction, mode, P, alpha)
    exact = orc.adi_sweep(field.copy(), *faces, bcs, direction, orc.MODE_THOMAS, 1, alpha)
    err = relerr(out, exact)
    if mode_name == "pdd":
        f = faces[direction]
        a, b, c = orc.adi_coeffs(f, bcs[direction], alpha)
        if bcs[direction] == orc.BC_PERIODIC:                   # reduced system closed cyclically: P interfaces (A16)
            dropped = orc.cyclic_pdd_dropped(P, a, b, c)
        else:
            dropped = orc.pdd_dropped(P, a, b, c)
        assert abs(grid.pdd_dropped_bound(direction, P, alpha) - dropped) <= 1e-10 * dropped + 1e-300
        ref_pdd = orc.adi_sweep(field.copy(), *faces, bcs, direction, orc.MODE_PDD, P, alpha)
        assert relerr(out, ref_pdd) < TOL_EXACT, ("pdd vs oracle pdd", direction, P, relerr(out, ref_pdd))
        if dropped <= 1e-11:
            assert err < TOL_PDD, ("pdd vs exact", direction, P, err, dropped)
        else:
            assert err < 100 * dropped + TOL_PDD
    else:
        assert err < TOL_EXACT, (mode_name, direction, P, err)
    return err


@pytest.fixture(scope="module")
def cfg1():
    c = configs.get(1)
    faces = c.faces()
    grid = tdx.Grid(c.nx, c.ny, c.nz, *faces, bcs=BCS)
    yield c, faces, grid, c.rhs_field()
    grid.close()


@pytest.mark.parametrize("direction", [0, 1, 2])
@pytest.mark.parametrize("mode_name", ["thomas", "pdd", "ppt"])
def test_cfg1_every_element(cfg1, direction, mode_name):
    c, faces, grid, field = cfg1
    check_sweep(grid, faces, BCS, field, direction, mode_name, 4, c.alpha)


@pytest.mark.parametrize("direction", [0, 1, 2])
@pytest.mark.parametrize("mode_name", ["thomas", "pdd", "ppt"])
def test_cfg1_strong_coupling(cfg1, direction, mode_name):
    """alpha large enough that the spikes do not decay inside a partition: PPT's Z^{-1} band is full."""
    c, faces, grid, field = cfg1
    check_sweep(grid, faces, BCS, field, direction, mode_name, 4, 1e-2)


@pytest.fixture(scope="module")
def cfg2():
    c = configs.get(2)
    faces = c.faces()
    grid = tdx.Grid(c.nx, c.ny, c.nz, *faces, bcs=BCS)
    yield c, faces, grid, c.rhs_field()
    grid.close()


@pytest.mark.parametrize("P", [4, 8, 16])
@pytest.mark.parametrize("mode_name", ["pdd", "ppt"])
def test_cfg2_x_then_y_then_z(cfg2, P, mode_name):
    """BASELINE.json config 2: full ADI sweep in x then y then z, compared after every sweep."""
    c, faces, grid, field = cfg2
    mode = MODES[mode_name]
    t = torch.from_numpy(field).cuda()
    chained = field.copy()                                      # exact x->y->z chain (PPT must follow it to 1e-12)
    for direction in (0, 1, 2):
        sweep_in = t.cpu().numpy()                              # each sweep is judged on its own input
        grid.adi_sweep(direction, mode, P, c.alpha, t)
        torch.cuda.synchronize()
        out = t.cpu().numpy()
        ref = orc.adi_sweep(sweep_in.copy(), *faces, BCS, direction, orc.MODE_THOMAS, 1, c.alpha)
        orc.adi_sweep(chained, *faces, BCS, direction, orc.MODE_THOMAS, 1, c.alpha)
        err = relerr(out, ref)
        dropped = grid.pdd_dropped_bound(direction, P, c.alpha)
        if mode_name == "ppt":
            assert err < TOL_EXACT and relerr(out, chained) < TOL_EXACT, (direction, P, err)
        elif dropped <= 1e-11:
            assert err < TOL_PDD, (direction, P, err, dropped)
        else:
            assert err < 100 * dropped + TOL_PDD, (direction, P, err, dropped)


def test_cfg2_thomas_all_directions(cfg2):
    c, faces, grid, field = cfg2
    for direction in (0, 1, 2):
        check_sweep(grid, faces, BCS, field, direction, "thomas", 1, c.alpha)


@pytest.mark.parametrize("mode_name,P", [("thomas", 1), ("ppt", 4), ("ppt", 8), ("ppt", 16)])
def test_cfg2_helmholtz_65_modes(cfg2, mode_name, P):
    """Poisson step of config 2: 65 wavenumbers, kz=0 pinned; PPT is the paper's method here."""
    c, faces, grid, _ = cfg2
    rhs = c.rhs_helmholtz()
    kz2 = c.kz2()
    t = torch.from_numpy(rhs).cuda()
    grid.helmholtz_wavenumber_solve(MODES[mode_name], P, None, kz2, t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    ref = orc.helmholtz_solve(rhs.copy(), faces[1], None, kz2, orc.MODE_THOMAS, 1)
    assert np.all(out[0, 0, :] == 0.0)                          # pinned points
    err = relerr(out, ref)
    if err >= TOL_EXACT:                                        # arbiter: compare both with long double
        ld = orc.helmholtz_solve(rhs.copy(), faces[1], None, kz2, orc.MODE_THOMAS_LD, 1)
        raise AssertionError("gpu-vs-fp64 oracle %.2e; gpu-vs-long double %.2e; fp64 oracle-vs-long double %.2e" % (err, relerr(out, ld), relerr(ref, ld)))
    # per-mode check so that large low-mode amplitudes do not hide errors in the high modes
    for m in range(0, c.nm, 8):
        assert relerr(out[m], ref[m]) < TOL_EXACT, m


def test_cfg2_helmholtz_pdd_is_inaccurate_on_low_modes_as_the_paper_reports(cfg2):
    """PDD gives inaccurate results on the weakly dominant Poisson systems; it still equals the
    oracle's step-by-step PDD, and it is accurate on the strongly dominant high modes."""
    c, faces, grid, _ = cfg2
    rhs = c.rhs_helmholtz()
    kz2 = c.kz2()
    t = torch.from_numpy(rhs).cuda()
    grid.helmholtz_wavenumber_solve(tdx.MODE_PDD, 4, None, kz2, t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    exact = orc.helmholtz_solve(rhs.copy(), faces[1], None, kz2, orc.MODE_THOMAS, 1)
    pdd = orc.helmholtz_solve(rhs.copy(), faces[1], None, kz2, orc.MODE_PDD, 4)
    assert relerr(out[1], exact[1]) > 1e-3
    assert relerr(out[c.nm - 1], exact[c.nm - 1]) < TOL_PDD
    for m in (1, 2, 7, 33, c.nm - 1):
        assert relerr(out[m], pdd[m]) < 1e-11, m


# ------------------------------------------------------------------------------------------ ragged / odd shapes
@pytest.fixture(scope="module")
def ragged():
    nx, ny, nz = 50, 37, 29
    faces = (inputs.faces_tanh_two_sided(nx, 1.2, 2.0), inputs.faces_tanh_one_sided(ny, 2.5), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    yield (nx, ny, nz), faces, grid, inputs.rhs_gaussian((nz, ny, nx), 77)
    grid.close()


@pytest.mark.parametrize("direction", [0, 1, 2])
@pytest.mark.parametrize("mode_name", ["thomas", "pdd", "ppt"])
@pytest.mark.parametrize("P", [3, 5])
def test_ragged_partitions_odd_extents_stretched_x(ragged, direction, mode_name, P):
    """n % P != 0 (partition lengths q and q+1), odd nx (scalar accesses), stretched x (per-partition tables)."""
    _, faces, grid, field = ragged
    check_sweep(grid, faces, BCS, field, direction, mode_name, P, 3e-4)


@pytest.mark.parametrize("bcs", [(tdx.BC_PERIODIC, tdx.BC_NEUMANN, tdx.BC_DIRICHLET), (tdx.BC_NEUMANN, tdx.BC_PERIODIC, tdx.BC_NEUMANN)])
@pytest.mark.parametrize("mode_name", ["thomas", "ppt", "pdd"])
def test_other_boundary_conditions(bcs, mode_name):
    nx, ny, nz = 48, 40, 36
    faces = (inputs.faces_uniform(nx, 1.5), inputs.faces_tanh_two_sided(ny, 1.5), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=bcs)
    field = inputs.rhs_uniform((nz, ny, nx), 9)
    for direction in range(3):
        check_sweep(grid, faces, bcs, field, direction, mode_name, 4, 5e-4)
    grid.close()


@pytest.mark.parametrize("bcx", [tdx.BC_DIRICHLET, tdx.BC_PERIODIC, tdx.BC_NEUMANN])
@pytest.mark.parametrize("nx,ny,nz", [(33, 5, 3), (64, 8, 8), (100, 7, 11), (7, 9, 5), (32, 4, 8), (257, 6, 6), (31, 13, 5)])
def test_thomas_along_x_warp_tiles(bcx, nx, ny, nz):
    """THOMAS mode along x walks 32 lines x 32 columns per warp through shared memory (k_thomas_unit_tiled): line counts that
    are not multiples of 32 (15, 77, 45, 65 lines), line lengths below, at and across the 32-column tile, last tiles of
    1 and 31 columns; Dirichlet, Neumann and periodic (third pass) ends.  Stretched x so that every row has its own table
    entry."""
    faces = (inputs.faces_tanh_two_sided(nx, 1.2), inputs.faces_uniform(ny, 1.0), inputs.faces_uniform(nz, 1.0))
    bcs = (bcx, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=bcs)
    field = inputs.rhs_uniform((nz, ny, nx), 31 + nx)
    check_sweep(grid, faces, bcs, field, 0, "thomas", 1, 3e-4)
    assert tdx.last_launch().startswith("k_thomas_unit_tiled<%d>" % (1 if bcx == tdx.BC_PERIODIC else 0))
    grid.close()


@pytest.mark.parametrize("nx,ny,nz,P", [(64, 48, 40, 2), (96, 16, 16, 12), (256, 8, 8, 64), (512, 6, 6, 8), (40, 36, 200, 25)])
def test_tile_and_partition_extremes(nx, ny, nz, P):
    """P=2 (no uniform table), many short partitions, 64-row partitions, lines spanning several warps."""
    faces = (inputs.faces_uniform(nx, 2.0), inputs.faces_tanh_two_sided(ny, 2.0), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    field = inputs.rhs_uniform((nz, ny, nx), 21)
    for direction in range(3):
        n = (nx, ny, nz)[direction]
        if n // P < 2:
            continue
        for mode_name in ("ppt", "pdd"):
            check_sweep(grid, faces, BCS, field, direction, mode_name, P, 2e-4)
    grid.close()


def test_helmholtz_per_line_shift_kx2_thomas(cfg2):
    """lambda = kx'^2(i) + kz'^2(m) (the paper's cosine-x / Fourier-z Poisson solve): every line has its own
    matrix; built for mode THOMAS (on-the-fly factorisation).  Only the (i = 0, m = 0) line is singular and pinned."""
    c, faces, grid, _ = cfg2
    rhs = c.rhs_helmholtz()
    kz2 = c.kz2()
    kx2 = inputs.modified_wavenumbers_x(c.nx, c.lx)
    assert kx2[0] == 0.0 and np.all(kx2[1:] > 0)
    t = torch.from_numpy(rhs).cuda()
    grid.helmholtz_wavenumber_solve(tdx.MODE_THOMAS, 1, kx2, kz2, t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    ref = orc.helmholtz_solve(rhs.copy(), faces[1], kx2, kz2, orc.MODE_THOMAS, 1)
    assert out[0, 0, 0] == 0.0                                   # the one pinned point
    assert np.all(out[0, 0, 1:] != 0.0)
    for m in range(0, c.nm, 4):                                  # per wavenumber: large low modes must not hide the rest
        assert relerr(out[m], ref[m]) < TOL_EXACT, (m, relerr(out[m], ref[m]))
    assert relerr(out, ref) < TOL_EXACT
    before = t.clone()
    with pytest.raises(tdx.TdxError) as e:                       # per-line PDD takes at most 16 rows per partition (128 / 4 = 32)
        grid.helmholtz_wavenumber_solve(tdx.MODE_PDD, 4, kx2, kz2, t)
    assert e.value.status == tdx.ERR_UNSUPPORTED and torch.equal(t, before)
    t4 = torch.from_numpy(rhs).cuda()                           # PPT is exact for any partitioning: 32-row partitions are cut again
    grid.helmholtz_wavenumber_solve(tdx.MODE_PPT, 4, kx2, kz2, t4)
    torch.cuda.synchronize()
    assert relerr(t4.cpu().numpy(), ref) < TOL_EXACT
    # kx2 given but all zero is the shared-matrix fast path
    t2 = torch.from_numpy(rhs).cuda(); t3 = torch.from_numpy(rhs).cuda()
    grid.helmholtz_wavenumber_solve(tdx.MODE_PPT, 8, np.zeros(c.nx), kz2, t2)
    grid.helmholtz_wavenumber_solve(tdx.MODE_PPT, 8, None, kz2, t3)
    torch.cuda.synchronize()
    assert torch.equal(t2, t3)


@pytest.mark.parametrize("P", [8, 16])
def test_helmholtz_per_line_shift_kx2_ppt_and_pdd(cfg2, P):
    """Per-line PPT/PDD (k_helm_lines: factorisation, spikes and the reduced system on the fly per line)."""
    c, faces, grid, _ = cfg2
    rhs = c.rhs_helmholtz()
    kz2 = c.kz2()
    kx2 = inputs.modified_wavenumbers_x(c.nx, c.lx)
    exact = orc.helmholtz_solve(rhs.copy(), faces[1], kx2, kz2, orc.MODE_THOMAS, 1)
    t = torch.from_numpy(rhs).cuda()
    grid.helmholtz_wavenumber_solve(tdx.MODE_PPT, P, kx2, kz2, t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    assert out[0, 0, 0] == 0.0
    err = relerr(out, exact)
    if err >= TOL_EXACT:
        ld = orc.helmholtz_solve(rhs.copy(), faces[1], kx2, kz2, orc.MODE_THOMAS_LD, 1)
        raise AssertionError("gpu-vs-fp64 oracle %.2e; gpu-vs-long double %.2e; fp64 oracle-vs-long double %.2e" % (err, relerr(out, ld), relerr(exact, ld)))
    for m in range(0, c.nm, 4):
        assert relerr(out[m], exact[m]) < 1e-11, (m, relerr(out[m], exact[m]))
    # PDD: equals the oracle's step-by-step PDD; accurate only where the spikes have decayed (high modes)
    t = torch.from_numpy(rhs).cuda()
    grid.helmholtz_wavenumber_solve(tdx.MODE_PDD, P, kx2, kz2, t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    pdd = orc.helmholtz_solve(rhs.copy(), faces[1], kx2, kz2, orc.MODE_PDD, P)
    for m in (0, 1, 5, 33, c.nm - 1):
        assert relerr(out[m], pdd[m]) < 1e-11, (m, relerr(out[m], pdd[m]))


def test_helmholtz_per_line_ragged_tile_and_12_row_partitions():
    """nx not a multiple of the 8-line tile, ny = 96 = 8 x 12."""
    nx, ny, nz = 50, 96, 12
    faces = (inputs.faces_uniform(nx, 1.0), inputs.faces_tanh_one_sided(ny, 2.5), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    nm = nz // 2 + 1
    rhs = inputs.rhs_complex_uniform((nm, ny, nx), 55)
    kz2 = inputs.modified_wavenumbers_z(nz, 1.0)
    kx2 = inputs.modified_wavenumbers_x(nx, 1.0)
    exact = orc.helmholtz_solve(rhs.copy(), faces[1], kx2, kz2, orc.MODE_THOMAS, 1)
    for P in (8, 12, 6):                                         # M = 12, 8, 16
        t = torch.from_numpy(rhs).cuda()
        grid.helmholtz_wavenumber_solve(tdx.MODE_PPT, P, kx2, kz2, t)
        torch.cuda.synchronize()
        assert relerr(t.cpu().numpy(), exact) < TOL_EXACT, P
    grid.close()


@pytest.mark.parametrize("ny,P", [(100, 8), (100, 7), (37, 3), (50, 25), (131, 9), (96, 7)])
def test_helmholtz_per_line_ragged_partitions(ny, P):
    """Per-line PPT / PDD when ny is not P*M: the partition map of tdx_partition_bounds (reading A5) with padding rows in
    the register tile (k_helm_lines<M, true>); every element against the oracle, PDD against the oracle's step-by-step PDD."""
    nx, nz = 21, 10
    faces = (inputs.faces_uniform(nx, 1.0), inputs.faces_tanh_one_sided(ny, 2.5), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    nm = nz // 2 + 1
    rhs = inputs.rhs_complex_uniform((nm, ny, nx), 77 + ny)
    kz2 = inputs.modified_wavenumbers_z(nz, 1.0)
    kx2 = inputs.modified_wavenumbers_x(nx, 1.0)
    exact = orc.helmholtz_solve(rhs.copy(), faces[1], kx2, kz2, orc.MODE_THOMAS, 1)
    t = torch.from_numpy(rhs).cuda()
    grid.helmholtz_wavenumber_solve(tdx.MODE_PPT, P, kx2, kz2, t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    assert out[0, 0, 0] == 0.0                                   # the pinned point of mode (0, 0)
    assert relerr(out, exact) < TOL_EXACT, (ny, P, relerr(out, exact))
    for m in range(nm):
        assert relerr(out[m], exact[m]) < 1e-11, (m, relerr(out[m], exact[m]))
    t = torch.from_numpy(rhs).cuda()
    grid.helmholtz_wavenumber_solve(tdx.MODE_PDD, P, kx2, kz2, t)
    torch.cuda.synchronize()
    pdd = orc.helmholtz_solve(rhs.copy(), faces[1], kx2, kz2, orc.MODE_PDD, P)
    out = t.cpu().numpy()
    for m in range(nm):
        assert relerr(out[m], pdd[m]) < 1e-11, (m, relerr(out[m], pdd[m]))
    grid.close()
