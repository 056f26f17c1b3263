"""Pins for oracle/transforms.py: the cosine / Fourier transforms written out as
dense sums and the direct Poisson solve built from them, checked against things that are not themselves: independent
library FFTs (numpy.fft, scipy.fft), closed forms, the eigen-relations with the second differences (which tie the
transforms to the modified wavenumbers the y-solves are shifted by), and the residual of the discrete Poisson equation
applied in physical space."""
import numpy as np
import pytest
import scipy.fft

import oracle as orc
import transforms as otr
from paper_1812_01178_b200 import inputs


def rel(x, ref):
    return float(np.max(np.abs(x - ref)) / np.max(np.abs(ref)))


@pytest.mark.parametrize("N", [4, 16, 30, 64])
def test_dct_matches_scipy_type2_and_inverse_round_trips(N):
    x = inputs.uniform_pm1(11, 3 * 5 * N).reshape(3, 5, N)
    X = otr.dct_x(x)
    assert rel(X, 0.5 * scipy.fft.dct(x, type=2, axis=-1)) < 1e-13          # scipy's type 2 carries a factor 2
    assert rel(otr.idct_x(X), x) < 1e-13
    assert rel(otr.idct_x(X), scipy.fft.idct(2.0 * X, type=2, axis=-1)) < 1e-13


def test_dct_closed_forms():
    N = 32
    n = np.arange(N)
    c = np.full((1, 1, N), 2.5)
    X = otr.dct_x(c)
    assert abs(X[0, 0, 0] - 2.5 * N) < 1e-12 and np.max(np.abs(X[0, 0, 1:])) < 1e-12      # constant -> k = 0 only
    for q in (1, 5, 31):
        x = np.cos(np.pi * q * (n + 0.5) / N).reshape(1, 1, N)
        X = otr.dct_x(x)[0, 0]
        e = np.zeros(N); e[q] = N / 2.0                                                   # orthogonality of the cosines
        assert np.max(np.abs(X - e)) < 1e-12
    d = np.zeros((1, 1, N)); d[0, 0, 7] = 1.0
    assert np.max(np.abs(otr.dct_x(d)[0, 0] - np.cos(np.pi * np.arange(N) * 7.5 / N))) < 1e-13   # a row of the definition


def test_dct_diagonalises_the_neumann_second_difference_with_kx2():
    """DCT(delta2_x u)_k = -kx'^2(k) DCT(u)_k: the reading T3 and inputs.modified_wavenumbers_x are the same thing."""
    N, lx = 48, 3.0
    u = inputs.uniform_pm1(5, N)
    dx = lx / N
    up = np.concatenate([u[:1], u, u[-1:]])
    d2 = (up[2:] - 2 * u + up[:-2]) / dx ** 2
    kx2, _ = otr.modified_wavenumbers(N, 8, lx, 1.0)
    lhs = otr.dct_x(d2.reshape(1, 1, N))[0, 0]
    rhs = -kx2 * otr.dct_x(u.reshape(1, 1, N))[0, 0]
    assert np.max(np.abs(lhs - rhs)) < 1e-10 * np.max(np.abs(rhs))
    assert np.allclose(kx2, inputs.modified_wavenumbers_x(N, lx), rtol=1e-12, atol=0.0)     # the input generator's 2(1-cos) form


@pytest.mark.parametrize("nz", [4, 16, 30, 64])
def test_rfft_matches_numpy_and_inverse_round_trips(nz):
    f = inputs.uniform_pm1(12, nz * 3 * 6).reshape(nz, 3, 6)
    F = otr.rfft_z(f)
    assert F.shape == (nz // 2 + 1, 3, 6)
    assert rel(F, np.fft.rfft(f, axis=0)) < 1e-13
    assert rel(otr.irfft_z(F, nz), f) < 1e-13
    G = F + 0.0
    G[0] += 0.37j; G[-1] -= 1.1j                       # imaginary parts of the DC and Nyquist terms do not enter
    assert rel(otr.irfft_z(G, nz), np.fft.irfft(G, n=nz, axis=0)) < 1e-13
    assert rel(otr.irfft_z(G, nz), f) < 1e-13


def test_rfft_closed_forms_and_parseval():
    nz = 32
    k = np.arange(nz)
    d = np.zeros((nz, 1, 1)); d[3, 0, 0] = 1.0
    F = otr.rfft_z(d)[:, 0, 0]
    assert np.max(np.abs(F - np.exp(-2j * np.pi * np.arange(nz // 2 + 1) * 3 / nz))) < 1e-13
    f = (np.cos(2 * np.pi * 5 * k / nz) + 0.5 * np.sin(2 * np.pi * 2 * k / nz)).reshape(nz, 1, 1)
    F = otr.rfft_z(f)[:, 0, 0]
    e = np.zeros(nz // 2 + 1, dtype=complex); e[5] = nz / 2; e[2] = -0.25j * nz
    assert np.max(np.abs(F - e)) < 1e-12
    g = inputs.uniform_pm1(3, nz).reshape(nz, 1, 1)
    G = otr.rfft_z(g)[:, 0, 0]
    w = np.full(nz // 2 + 1, 2.0); w[0] = w[-1] = 1.0
    assert abs(np.sum(w * np.abs(G) ** 2) / nz - np.sum(g ** 2)) < 1e-12 * np.sum(g ** 2)


def test_rfft_diagonalises_the_periodic_second_difference_with_kz2():
    nz, lz = 40, 1.0
    u = inputs.uniform_pm1(6, nz)
    dz = lz / nz
    d2 = (np.roll(u, -1) - 2 * u + np.roll(u, 1)) / dz ** 2
    _, kz2 = otr.modified_wavenumbers(8, nz, 1.0, lz)
    lhs = otr.rfft_z(d2.reshape(nz, 1, 1))[:, 0, 0]
    rhs = -kz2 * otr.rfft_z(u.reshape(nz, 1, 1))[:, 0, 0]
    assert np.max(np.abs(lhs - rhs)) < 1e-10 * np.max(np.abs(rhs))
    assert np.allclose(kz2, inputs.modified_wavenumbers_z(nz, lz), rtol=1e-12, atol=0.0)


def test_laplacian_y_part_is_the_helmholtz_matrix_of_the_oracle():
    """The physical-space operator used to pin the Poisson solve agrees with the tridiagonal coefficients the y-solves use."""
    ny = 20
    yf = inputs.faces_tanh_one_sided(ny, 2.0)
    a, b, c, pinned = orc.helmholtz_coeffs(yf, 0.0)
    assert pinned
    # un-pin row 0 (lambda = 0 lines are pinned in the solve; the operator itself has b0 = -(c0))
    A = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    phi = inputs.uniform_pm1(9, ny)
    full = otr.laplacian(phi.reshape(1, ny, 1), yf, 1.0, 1.0)[0, :, 0]      # nx = nz = 1: x and z parts vanish
    assert np.max(np.abs((A @ phi)[1:] - full[1:])) < 1e-9 * np.max(np.abs(full))


@pytest.mark.parametrize("shape", [(8, 12, 16), (16, 10, 6)])
def test_poisson_solve_inverts_the_discrete_laplacian(shape):
    """Manufactured: f = L phi for a random phi; the solve returns phi up to the additive constant the pin fixes
    (mode (0,0) is pinned to 0 at j = 0, i.e. the x-z mean of row j = 0 vanishes)."""
    nz, ny, nx = shape
    lx, lz = 2.0, 1.0
    yf = inputs.faces_tanh_one_sided(ny, 2.0)
    phi = inputs.uniform_pm1(21, nz * ny * nx).reshape(nz, ny, nx)
    f = otr.laplacian(phi, yf, lx, lz)
    got = otr.poisson_solve(f, yf, lx, lz)
    shift = np.mean(phi[:, 0, :])
    assert abs(np.mean(got[:, 0, :])) < 1e-12
    assert rel(got, phi - shift) < 1e-10
    # and the residual of the equation itself, everywhere except the pinned row of the mean mode
    r = otr.laplacian(got, yf, lx, lz) - f
    assert np.max(np.abs(r)) < 1e-9 * np.max(np.abs(f))


def test_poisson_solve_of_a_single_separable_mode_is_the_closed_form():
    """f = cos(pi p (i+1/2)/nx) cos(2 pi r k/nz) g(j): phi is the same x-z mode times the solution of one y-system."""
    nz, ny, nx, p, r = 16, 14, 12, 3, 2
    lx, lz = 1.5, 1.0
    yf = inputs.faces_tanh_two_sided(ny, 2.0)
    g = inputs.uniform_pm1(4, ny)
    cx = np.cos(np.pi * p * (np.arange(nx) + 0.5) / nx)
    cz = np.cos(2 * np.pi * r * np.arange(nz) / nz)
    f = cz[:, None, None] * g[None, :, None] * cx[None, None, :]
    kx2, kz2 = otr.modified_wavenumbers(nx, nz, lx, lz)
    a, b, c, _ = orc.helmholtz_coeffs(yf, kx2[p] + kz2[r])
    A = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    y = np.linalg.solve(A, g)
    want = cz[:, None, None] * y[None, :, None] * cx[None, None, :]
    assert rel(otr.poisson_solve(f, yf, lx, lz), want) < 1e-11
