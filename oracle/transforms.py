"""Transforms around the Poisson y-solves and the whole direct Poisson solve -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

PAPER.md:L45 (section 2.2): "The Poisson equation is solved directly using half-range cosine transform in the
streamwise x-direction and Fourier transform in the spanwise z-direction.  Complex-numbered tridiagonal matrices in the
wall-normal y-direction are inverted, after which the pseudo-pressure phi is obtained via inverse transforms."
PAPER.md:L172: the main diagonal of those matrices is a + c plus "the modified wavenumbers coming from the half-cosine
transform in the x-direction followed by the Fourier transform in the z-direction".

Every transform here is its plain definition written out as a dense sum (a matrix of cosines / complex exponentials
applied with a library matmul, fp64; arguments reduced exactly in integer arithmetic before cos/sin); nothing is blocked,
factored or reordered.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It imports nothing from paper_1812_01178_b200 and shares no code or table with csrc/.
Every function is pinned by tests/test_oracle_transform_pins.py (independent library FFTs, closed forms, eigen-relations
with the second differences, manufactured Poisson solutions); nothing here is "parity unpinned".

Readings (T1-T3):
  T1  half-range cosine transform of cell-centred values (pressure sits at cell centres, L41; Neumann walls):
      X_k = sum_n x_n cos(pi k (n + 1/2) / N), k = 0..N-1 (unnormalised);
      inverse x_n = (1/N) [ X_0 + 2 sum_{k>=1} X_k cos(pi k (n + 1/2) / N) ].
  T2  Fourier transform in z of real data, non-redundant half: F_m = sum_k f_k exp(-2 pi i m k / N), m = 0..N/2;
      inverse f_k = (1/N) [ Re F_0 + (-1)^k Re F_{N/2} + 2 Re sum_{0<m<N/2} F_m exp(+2 pi i m k / N) ].
  T3  the transformed equation for mode (i, m) is (delta2_y - kx'^2(i) - kz'^2(m)) phi^ = f^ with
      kx'^2(i) = 2(1 - cos(pi i / Nx)) / dx^2 and kz'^2(m) = 2(1 - cos(2 pi m / Nz)) / dz^2 (the eigenvalues of the
      Neumann / periodic second differences on the uniform x and z grids); mode (0, 0) is singular and pinned at j = 0.
"""
import numpy as np

import oracle as _orc  # oracle/oracle.py (the Thomas y-solves)


def _cos_table(N):
    """C[k][n] = cos(pi k (2n+1) / (2N)); the integer k(2n+1) is reduced modulo 4N before the division."""
    k = np.arange(N, dtype=np.int64)[:, None]
    n = np.arange(N, dtype=np.int64)[None, :]
    q = (k * (2 * n + 1)) % (4 * N)
    return np.cos(np.pi * q.astype(np.float64) / (2.0 * N))


def dct_x(field_zyx):
    """T1 forward along the last (x) axis; returns a new array."""
    N = field_zyx.shape[-1]
    return field_zyx @ _cos_table(N).T


def idct_x(spec_zyx):
    """T1 inverse along the last (x) axis; returns a new array."""
    N = spec_zyx.shape[-1]
    Cm = _cos_table(N).copy()          # [k][n]
    Cm[1:, :] *= 2.0
    return (spec_zyx @ Cm) / N


def _exp_table(N, rows, sign):
    """E[m][k] = exp(sign * 2 pi i m k / N) for m < rows; m k reduced modulo N exactly."""
    m = np.arange(rows, dtype=np.int64)[:, None]
    k = np.arange(N, dtype=np.int64)[None, :]
    q = (m * k) % N
    ang = 2.0 * np.pi * q.astype(np.float64) / N
    return np.cos(ang) + sign * 1j * np.sin(ang)


def rfft_z(field_zyx):
    """T2 forward along the first (z) axis: real [nz][ny][nx] -> complex128 [nz/2+1][ny][nx]."""
    nz, ny, nx = field_zyx.shape
    assert nz % 2 == 0
    E = _exp_table(nz, nz // 2 + 1, -1.0)
    out = E @ field_zyx.reshape(nz, ny * nx).astype(np.complex128)
    return np.ascontiguousarray(out.reshape(nz // 2 + 1, ny, nx))


def irfft_z(spec_myx, nz):
    """T2 inverse: complex [nz/2+1][ny][nx] -> real [nz][ny][nx].  The imaginary parts of F_0 and F_{nz/2} do not enter."""
    nm, ny, nx = spec_myx.shape
    assert nm == nz // 2 + 1
    F = spec_myx.reshape(nm, ny * nx)
    E = _exp_table(nz, nm, +1.0).T                           # [k][m] = exp(+2 pi i m k / N)
    w = np.full(nm, 2.0); w[0] = 1.0; w[-1] = 1.0
    G = F.copy()
    G[0] = G[0].real; G[-1] = G[-1].real
    out = ((E * w[None, :]) @ G).real / nz
    return np.ascontiguousarray(out.reshape(nz, ny, nx))


def modified_wavenumbers(nx, nz, lx, lz):
    """T3: (kx'^2[nx], kz'^2[nz/2+1]); entry 0 of each is exactly 0."""
    i = np.arange(nx, dtype=np.float64)
    m = np.arange(nz // 2 + 1, dtype=np.float64)
    dx, dz = lx / nx, lz / nz
    # 2(1 - cos t) written as 4 sin^2(t/2): the same number without the cancellation at small t (relative error ~1e-16
    # instead of ~1e-16/t^2 -- the lowest modes are the nearly singular ones, L172)
    kx2 = 4.0 * np.sin(0.5 * np.pi * i / nx) ** 2 / (dx * dx)
    kz2 = 4.0 * np.sin(np.pi * m / nz) ** 2 / (dz * dz)
    kx2[0] = 0.0; kz2[0] = 0.0
    return kx2, kz2


def poisson_solve(f_zyx, yf, lx, lz):
    """Direct Poisson solve of L45 in the paper's order: cosine transform in x, Fourier transform in z, y-solves
    (Thomas, the oracle's own), inverse Fourier transform, inverse cosine transform.  Returns phi [nz][ny][nx].
    Neumann in x and y, periodic in z; mode (0,0) pinned at j = 0 (T3)."""
    nz, ny, nx = f_zyx.shape
    kx2, kz2 = modified_wavenumbers(nx, nz, lx, lz)
    spec = rfft_z(dct_x(f_zyx))
    _orc.helmholtz_solve(spec, np.asarray(yf, dtype=np.float64), kx2, kz2, _orc.MODE_THOMAS, 1)
    return idct_x(irfft_z(spec, nz))


def laplacian(phi_zyx, yf, lx, lz):
    """The discrete operator the solve inverts, applied directly in physical space (used by the pins only):
    second differences, Neumann (mirror) ends in x and y, periodic in z, cell-centred stretched y."""
    nz, ny, nx = phi_zyx.shape
    dx, dz = lx / nx, lz / nz
    out = np.zeros_like(phi_zyx)
    px = np.concatenate([phi_zyx[:, :, :1], phi_zyx, phi_zyx[:, :, -1:]], axis=2)
    out += (px[:, :, 2:] - 2.0 * phi_zyx + px[:, :, :-2]) / (dx * dx)
    out += (np.roll(phi_zyx, -1, axis=0) - 2.0 * phi_zyx + np.roll(phi_zyx, 1, axis=0)) / (dz * dz)
    yf = np.asarray(yf, dtype=np.float64)
    d = np.diff(yf)                                     # cell widths
    yc = 0.5 * (yf[1:] + yf[:-1])
    h = np.diff(yc)                                     # centre-to-centre
    flux = np.zeros((nz, ny + 1, nx))
    flux[:, 1:ny, :] = (phi_zyx[:, 1:, :] - phi_zyx[:, :-1, :]) / h[None, :, None]   # zero flux through the walls
    out += (flux[:, 1:, :] - flux[:, :-1, :]) / d[None, :, None]
    return out
