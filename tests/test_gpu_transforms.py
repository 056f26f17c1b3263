"""GPU parity (through the C ABI) of the transforms around the Poisson y-solves and of the whole direct Poisson solve
 against oracle/transforms.py (dense-sum definitions) on the same seeded inputs.
Tolerances: transforms 1e-12 relative max-norm (an N-point FFT in fp64 is good to ~log2(N) eps, the dense-sum oracle to
~N eps); Poisson: see test_poisson_solve_cfg2."""
import numpy as np
import pytest
import torch

import oracle as orc
import transforms as otr
from paper_1812_01178_b200 import binding as tdx
from paper_1812_01178_b200 import configs, inputs

pytestmark = pytest.mark.gpu
BCS = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
TOL = 1e-12


def relerr(x, ref):
    return float(np.max(np.abs(x - ref)) / np.max(np.abs(ref)))


def make_grid(nx, ny, nz, lx=2.0):
    faces = (inputs.faces_uniform(nx, lx), inputs.faces_tanh_one_sided(ny, 2.5), inputs.faces_uniform(nz, 1.0))
    return faces, tdx.Grid(nx, ny, nz, *faces, bcs=BCS)


# every kernel instantiation: nx = 16 .. 4096; line counts that leave a partial last CTA (ny*nz not a multiple of 2*LP)
@pytest.mark.parametrize("nx,ny,nz", [(16, 5, 16), (32, 3, 16), (64, 5, 16), (128, 7, 16), (256, 9, 16), (512, 3, 16),
                                      (1024, 3, 16), (2048, 3, 16), (4096, 3, 16),
                                      (48, 5, 16), (96, 3, 16), (192, 5, 16), (384, 3, 16), (768, 3, 16), (1536, 3, 16), (3072, 3, 16)])
def test_dct_x_forward_and_inverse(nx, ny, nz):
    faces, grid = make_grid(nx, ny, nz)
    x = inputs.rhs_uniform((nz, ny, nx), 100 + nx)
    t = torch.from_numpy(x).cuda()
    grid.dct_x(False, t)
    torch.cuda.synchronize()
    X = t.cpu().numpy()
    ref = otr.dct_x(x)
    assert relerr(X, ref) < TOL, relerr(X, ref)
    # per line too: a line with a small spectrum must not hide behind a large one
    worst = np.max(np.abs(X - ref), axis=-1) / np.max(np.abs(ref), axis=-1)
    assert np.max(worst) < 1e-11
    t2 = torch.from_numpy(ref).cuda()                      # inverse, fed with the oracle's spectrum
    grid.dct_x(True, t2)
    torch.cuda.synchronize()
    assert relerr(t2.cpu().numpy(), otr.idct_x(ref)) < TOL
    grid.dct_x(True, t)                                    # round trip on the device
    torch.cuda.synchronize()
    assert relerr(t.cpu().numpy(), x) < TOL
    grid.close()


def test_dct_x_one_hot_touches_only_its_line_and_is_the_cosine_row():
    nx, ny, nz = 64, 6, 16
    faces, grid = make_grid(nx, ny, nz)
    x = np.zeros((nz, ny, nx)); x[5, 3, 9] = 1.0
    t = torch.from_numpy(x).cuda()
    grid.dct_x(False, t)
    torch.cuda.synchronize()
    X = t.cpu().numpy()
    row = np.cos(np.pi * np.arange(nx) * 9.5 / nx)
    assert np.max(np.abs(X[5, 3] - row)) < 1e-14
    X[5, 3] = 0.0
    # lines (5,2) and (5,3) are the re/im parts of one complex transform: the partner sees rounding residue only
    assert np.max(np.abs(X[5, 2])) < 4e-16
    X[5, 2] = 0.0
    assert not X.any()                                      # every other line is exactly zero
    grid.close()


@pytest.mark.parametrize("nx,ny,nz", [(16, 3, 16), (50, 4, 32), (64, 3, 64), (34, 2, 128), (32, 3, 256), (36, 2, 512), (18, 2, 1024),
                                      (34, 3, 48), (16, 2, 96), (50, 2, 192), (18, 3, 384), (36, 2, 768), (20, 2, 1536)])
def test_rfft_z_forward_and_inverse(nx, ny, nz):
    """nx even but not a multiple of the 32-wide column tile: ragged last tile."""
    faces = (inputs.faces_uniform(nx, 1.0), inputs.faces_tanh_one_sided(ny, 2.5), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    nm = nz // 2 + 1
    f = inputs.rhs_uniform((nz, ny, nx), 200 + nz)
    tin = torch.from_numpy(f).cuda()
    spec = torch.full((nm, ny, nx), float("nan"), dtype=torch.complex128, device="cuda")
    grid.rfft_z(tin, spec)
    torch.cuda.synchronize()
    assert torch.equal(tin.cpu(), torch.from_numpy(f))       # input untouched
    F = spec.cpu().numpy()
    ref = otr.rfft_z(f)
    assert relerr(F, ref) < TOL, relerr(F, ref)
    assert np.all(F[0].imag == 0.0) and np.all(F[-1].imag == 0.0)
    col = np.max(np.abs(F - ref), axis=0) / np.max(np.abs(ref), axis=0)     # per column
    assert np.max(col) < 1e-11
    G = inputs.rhs_complex_uniform((nm, ny, nx), 300 + nz)   # arbitrary spectrum, imaginary DC / Nyquist parts included
    tg = torch.from_numpy(G).cuda()
    back = torch.full((nz, ny, nx), float("nan"), dtype=torch.float64, device="cuda")
    grid.irfft_z(tg, back)
    torch.cuda.synchronize()
    assert relerr(back.cpu().numpy(), otr.irfft_z(G, nz)) < TOL
    grid.irfft_z(spec, back)                                 # round trip
    torch.cuda.synchronize()
    assert relerr(back.cpu().numpy(), f) < TOL
    grid.close()


def test_transform_error_paths_leave_data_untouched():
    nx, ny, nz = 40, 4, 24                                   # neither 2^k nor 3 * 2^k (k >= 4)
    faces = (inputs.faces_uniform(nx, 1.0), inputs.faces_tanh_one_sided(ny, 2.5), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    x = inputs.rhs_uniform((nz, ny, nx), 7)
    t = torch.from_numpy(x).cuda()
    spec = torch.zeros((nz // 2 + 1, ny, nx), dtype=torch.complex128, device="cuda")
    for call in (lambda: grid.dct_x(False, t), lambda: grid.rfft_z(t, spec), lambda: grid.irfft_z(spec, t),
                 lambda: grid.poisson_solve(tdx.MODE_THOMAS, 1, None, None, t, spec)):
        with pytest.raises(tdx.TdxError) as e:
            call()
        assert e.value.status == tdx.ERR_UNSUPPORTED
    torch.cuda.synchronize()
    assert np.array_equal(t.cpu().numpy(), x) and not spec.cpu().numpy().any()
    grid.close()
    faces, grid = make_grid(32, 16, 16)
    t = torch.zeros((16, 16, 32), dtype=torch.float64, device="cuda")
    spec = torch.zeros((9, 16, 32), dtype=torch.complex128, device="cuda")
    with pytest.raises(tdx.TdxError) as e:
        grid.rfft_z(t, t)                                    # in place is not defined
    assert e.value.status == tdx.ERR_INVALID_ARG
    with pytest.raises(tdx.TdxError) as e:
        grid.poisson_solve(tdx.MODE_PPT, 9, None, None, t, spec)   # 16 rows / 9 partitions: fewer than 2 rows each
    assert e.value.status == tdx.ERR_BAD_PARTITION
    t.fill_(1.5)
    bad = np.full(32, 1.0); bad[7] = float("nan")
    with pytest.raises(tdx.TdxError) as e:                       # a bad wavenumber is caught before the first transform runs
        grid.poisson_solve(tdx.MODE_THOMAS, 1, bad, None, t, spec)
    assert e.value.status == tdx.ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert bool((t == 1.5).all())
    grid.close()


@pytest.fixture(scope="module")
def cfg2():
    c = configs.get(2)
    faces = c.faces()
    grid = tdx.Grid(c.nx, c.ny, c.nz, *faces, bcs=BCS)
    yield c, faces, grid
    grid.close()


@pytest.mark.parametrize("mode,P", [(tdx.MODE_THOMAS, 1), (tdx.MODE_PPT, 8), (tdx.MODE_PPT, 16)])
def test_poisson_solve_cfg2(cfg2, mode, P):
    """Whole direct solve on config 2 (256x128x128) against the oracle's composition, same wavenumber arrays on both sides.
    Tolerance: the y-systems of the lowest modes are nearly singular (|b| = |a| + |c| + lambda with lambda down to
    kx'^2(1) ~ (pi/Lx)^2 against off-diagonals ~ 1/dy_min^2), so rounding differences between two
    correct fp64 solvers are amplified there.  Measured on B200: 3e-14 (THOMAS) to 1e-13 (PPT) on phi, 6e-13 on the
    residual (the oracle's own residual: 3e-12); gates: 2e-12 on phi (north_star's 1e-12 for one solve, doubled for the
    four transforms around it), 1e-11 on the residual."""
    c, faces, grid = cfg2
    f = c.rhs_field()
    kx2, kz2 = otr.modified_wavenumbers(c.nx, c.nz, c.lx, 1.0)
    ref = otr.poisson_solve(f, faces[1], c.lx, 1.0)
    t = torch.from_numpy(f).cuda()
    work = torch.empty((c.nz // 2 + 1, c.ny, c.nx), dtype=torch.complex128, device="cuda")
    grid.poisson_solve(mode, P, kx2, kz2, t, work)
    torch.cuda.synchronize()
    phi = t.cpu().numpy()
    err = relerr(phi, ref)
    assert err < 2e-12, err
    r = otr.laplacian(phi, faces[1], c.lx, 1.0) - f
    r[:, 0, :] -= np.mean(r[:, 0, :])                        # the pinned row of the mean mode carries the compatibility defect
    assert np.max(np.abs(r)) < 1e-11 * np.max(np.abs(f)), np.max(np.abs(r)) / np.max(np.abs(f))
    # wavenumbers computed by the library (NULL): same answer to rounding of lambda
    t2 = torch.from_numpy(f).cuda()
    grid.poisson_solve(mode, P, None, None, t2, work)
    torch.cuda.synchronize()
    assert relerr(t2.cpu().numpy(), ref) < 2e-12


def test_poisson_solve_factor_three_sizes():
    """nx = 96 = 3 * 32, nz = 48 = 3 * 16 (the paper's own grid, 3072 x 256 x 768, has a factor 3 in x and z: L182, L314)."""
    nx, ny, nz = 96, 32, 48
    faces, grid = make_grid(nx, ny, nz, lx=2.0)
    phi = inputs.rhs_uniform((nz, ny, nx), 33)
    f = otr.laplacian(phi, faces[1], 2.0, 1.0)
    work = torch.empty((nz // 2 + 1, ny, nx), dtype=torch.complex128, device="cuda")
    ref = otr.poisson_solve(f, faces[1], 2.0, 1.0)
    for mode, P in ((tdx.MODE_THOMAS, 1), (tdx.MODE_PPT, 4)):
        t = torch.from_numpy(f).cuda()
        grid.poisson_solve(mode, P, None, None, t, work)
        torch.cuda.synchronize()
        got = t.cpu().numpy()
        assert relerr(got, ref) < 2e-12, (mode, P, relerr(got, ref))
        assert relerr(got, phi - np.mean(phi[:, 0, :])) < 1e-9
    grid.close()


def test_poisson_solve_manufactured_small_every_element():
    """32x32x16 with phi manufactured through the physical-space Laplacian of the oracle: the GPU solve returns phi up to
    the constant the pin fixes."""
    nx, ny, nz = 32, 32, 16
    faces, grid = make_grid(nx, ny, nz, lx=2.0)
    phi = inputs.rhs_uniform((nz, ny, nx), 31)
    f = otr.laplacian(phi, faces[1], 2.0, 1.0)
    work = torch.empty((nz // 2 + 1, ny, nx), dtype=torch.complex128, device="cuda")
    for mode, P in ((tdx.MODE_THOMAS, 1), (tdx.MODE_PPT, 4), (tdx.MODE_PPT, 2), (tdx.MODE_PPT, 3), (tdx.MODE_PPT, 5)):   # 3, 5: ragged partitions
        t = torch.from_numpy(f).cuda()
        grid.poisson_solve(mode, P, None, None, t, work)
        torch.cuda.synchronize()
        got = t.cpu().numpy()
        assert relerr(got, phi - np.mean(phi[:, 0, :])) < 1e-9, (mode, P)
        assert relerr(got, otr.poisson_solve(f, faces[1], 2.0, 1.0)) < 2e-12, (mode, P)
    grid.close()
