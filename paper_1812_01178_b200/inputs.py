"""Seeded synthetic inputs shared by the tests, the oracle callers and bench.py.

This module holds NONE of the method's arithmetic (no metrics, coefficients, eliminations): only the
grid-face generators, the wavenumber shifts handed to the Helmholtz entry point, and counter-based random
right-hand sides, i.e. the *inputs* of the hot path (recipe: DESIGN.md "Input recipe").
numpy only; imports neither the CUDA binding nor the oracle.
"""
import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix64(x):
    """splitmix64 finaliser on a uint64 array (counter-based: value depends on (seed, index) only)."""
    x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
    x ^= x >> np.uint64(30)
    x = (x * np.uint64(0xBF58476D1CE4E5B9)) & _M64
    x ^= x >> np.uint64(27)
    x = (x * np.uint64(0x94D049BB133111EB)) & _M64
    x ^= x >> np.uint64(31)
    return x


def _u01(seed, stream, start, count):
    """53-bit uniforms in [0,1) for linear indices start..start+count-1 of (seed, stream)."""
    with np.errstate(over="ignore"):
        idx = np.arange(start, start + count, dtype=np.uint64)
        key = _mix64(np.uint64(seed) * np.uint64(0xD1342543DE82EF95) + np.uint64(stream))
        h = _mix64(idx ^ key)
    return (h >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def uniform_pm1(seed, count, start=0, stream=0, chunk=1 << 24):
    """uniform[-1,1) doubles, value = f(seed, stream, linear index)."""
    out = np.empty(count, dtype=np.float64)
    for s in range(0, count, chunk):
        n = min(chunk, count - s)
        out[s:s + n] = 2.0 * _u01(seed, stream, start + s, n) - 1.0
    return out


def gaussian(seed, count, start=0, chunk=1 << 24):
    """N(0,1) doubles by Box-Muller on two counter-based uniforms per value."""
    out = np.empty(count, dtype=np.float64)
    for s in range(0, count, chunk):
        n = min(chunk, count - s)
        u1 = _u01(seed, 1, start + s, n)
        u2 = _u01(seed, 2, start + s, n)
        out[s:s + n] = np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)
    return out


# ---- grid faces (N+1 strictly increasing coordinates per direction) -------------------------------------
def faces_uniform(n, length):
    return length * np.arange(n + 1, dtype=np.float64) / n


def faces_tanh_two_sided(n, gamma, length=1.0):
    """clustered at both walls: f_j = L/2 [1 + tanh(g(2j/N-1))/tanh g] (configs 1-3)."""
    j = np.arange(n + 1, dtype=np.float64)
    f = 0.5 * length * (1.0 + np.tanh(gamma * (2.0 * j / n - 1.0)) / np.tanh(gamma))
    f[0], f[-1] = 0.0, length
    return f


def faces_tanh_one_sided(n, gamma, length=1.0):
    """clustered at y=0 only: f_j = L [1 - tanh(g(1-j/N))/tanh g] (configs 4-5, boundary-layer like)."""
    j = np.arange(n + 1, dtype=np.float64)
    f = length * (1.0 - np.tanh(gamma * (1.0 - j / n)) / np.tanh(gamma))
    f[0], f[-1] = 0.0, length
    return f


def modified_wavenumbers_z(nz, lz=1.0):
    """kz'^2(m) = 2(1-cos(2 pi m/Nz))/dz^2, m = 0..Nz/2: the shifts passed to the Helmholtz entry point."""
    m = np.arange(nz // 2 + 1, dtype=np.float64)
    dz = lz / nz
    k = 2.0 * (1.0 - np.cos(2.0 * np.pi * m / nz)) / (dz * dz)
    k[0] = 0.0
    return k


def modified_wavenumbers_x(nx, lx):
    """kx'^2(i) = 2(1-cos(pi i/Nx))/dx^2 (half-range cosine, cell centred)."""
    i = np.arange(nx, dtype=np.float64)
    dx = lx / nx
    k = 2.0 * (1.0 - np.cos(np.pi * i / nx)) / (dx * dx)
    k[0] = 0.0
    return k


# ---- right-hand sides -------------------------------------------------------------------------------------
def rhs_uniform(shape_zyx, seed):
    nz, ny, nx = shape_zyx
    return uniform_pm1(seed, nz * ny * nx).reshape(nz, ny, nx)


def rhs_gaussian(shape_zyx, seed):
    nz, ny, nx = shape_zyx
    return gaussian(seed, nz * ny * nx).reshape(nz, ny, nx)


def rhs_smooth_modes(shape_zyx, seed, lx, ly=1.0, lz=1.0, noise=1e-3):
    """sum of 4 smooth modes sin(2 pi p x/Lx) cos(pi q y/Ly) cos(2 pi r z/Lz) at cell centres of a
    uniform reference lattice + noise*uniform[-1,1] (configs 4-5)."""
    nz, ny, nx = shape_zyx
    x = (np.arange(nx) + 0.5) / nx
    y = (np.arange(ny) + 0.5) / ny
    z = (np.arange(nz) + 0.5) / nz
    out = np.empty((nz, ny, nx), dtype=np.float64)
    modes = ((1, 1, 1), (2, 3, 1), (3, 2, 4), (5, 7, 3))
    sx = [np.sin(2 * np.pi * p * x) for p, _, _ in modes]
    cy = [np.cos(np.pi * q * y) for _, q, _ in modes]
    cz = [np.cos(2 * np.pi * r * z) for _, _, r in modes]
    for k in range(nz):
        plane = np.zeros((ny, nx))
        for t in range(4):
            plane += cz[t][k] * np.outer(cy[t], sx[t])
        plane += noise * uniform_pm1(seed, ny * nx, start=k * ny * nx).reshape(ny, nx)
        out[k] = plane
    return out


def rhs_complex_uniform(shape_myx, seed):
    """complex128 [nm][ny][nx], re and im uniform[-1,1) from two streams."""
    nm, ny, nx = shape_myx
    n = nm * ny * nx
    out = np.empty(n, dtype=np.complex128)
    out.real = uniform_pm1(seed, n, stream=3)
    out.imag = uniform_pm1(seed, n, stream=4)
    return out.reshape(nm, ny, nx)
