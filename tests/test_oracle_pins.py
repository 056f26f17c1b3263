"""Pins for the CPU oracle (oracle/oracle.c): every function is checked against something OTHER than itself --
dense Gaussian elimination / LAPACK on tiny systems, exact rational arithmetic, manufactured solutions through a
dense matvec, eigen closed forms, the structure the paper prints (tests/golden/Z_n12_p4.txt), the dominance
invariants PAPER.md:L162 / L172, and the paper's qualitative claims about PDD (L152, L164, L172).  CPU only."""
import os
import re
from fractions import Fraction

import numpy as np
import pytest
import scipy.linalg

import oracle as orc
from paper_1812_01178_b200 import configs, inputs

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
rng = np.random.default_rng(1234)


def random_dominant(n, margin=0.5, cyclic=False):
    a = rng.uniform(-1, 1, n); c = rng.uniform(-1, 1, n)
    b = (np.abs(a) + np.abs(c) + margin) * rng.choice([-1.0, 1.0], n)
    if not cyclic:
        a[0] = 0.0; c[-1] = 0.0
    return a, b, c


def banded_solve(a, b, c, d):
    """LAPACK gbsv (partial pivoting) through scipy: an independent library routine."""
    n = b.size
    ab = np.zeros((3, n)); ab[0, 1:] = c[:-1]; ab[1] = b; ab[2, :-1] = a[1:]
    return scipy.linalg.solve_banded((1, 1), ab, d)


def relerr(x, ref):
    return np.max(np.abs(x - ref)) / np.max(np.abs(ref))


# ---------------------------------------------------------------- partition map
@pytest.mark.parametrize("n,P", [(12, 4), (32, 4), (288, 16), (288, 32), (100, 7), (4096, 128), (17, 8), (9, 4)])
def test_partition_bounds_matches_array_split(n, P):
    st = orc.partition_bounds(n, P)
    sizes = [len(s) for s in np.array_split(np.arange(n), P)]       # numpy: first n%P parts get one more
    assert list(np.diff(st)) == sizes and st[0] == 0 and st[-1] == n


def test_partition_bounds_rejects_short_partitions():
    with pytest.raises(RuntimeError):
        orc.partition_bounds(7, 4)


# ---------------------------------------------------------------- Thomas / cyclic / dense GE
@pytest.mark.parametrize("n", [2, 3, 5, 8, 16])
def test_thomas_vs_dense_ge_and_lapack(n):
    a, b, c = random_dominant(n)
    d = rng.uniform(-1, 1, n)
    A = orc.dense_from_tridiag(a, b, c)
    x = orc.thomas(a, b, c, d)
    assert relerr(x, orc.dense_solve(A, d)) < 1e-14
    assert relerr(x, np.linalg.solve(A, d)) < 1e-14               # LAPACK, independent of oracle_dense_solve
    assert relerr(x, banded_solve(a, b, c, d)) < 1e-14
    assert relerr(orc.thomas(a, b, c, d, long_double=True), x) < 1e-14


def test_dense_from_tridiag_layout():
    a = np.array([9., 1., 2., 3.]); b = np.array([10., 20., 30., 40.]); c = np.array([5., 6., 7., 8.])
    A = orc.dense_from_tridiag(a, b, c)
    assert np.array_equal(A, np.array([[10, 5, 0, 0], [1, 20, 6, 0], [0, 2, 30, 7], [0, 0, 3, 40.]]))
    Ac = orc.dense_from_tridiag(a, b, c, cyclic=True)
    assert Ac[0, 3] == 9.0 and Ac[3, 0] == 8.0


def test_dense_solve_needs_pivoting_case():
    A = np.array([[0.0, 2.0, 1.0], [1.0, 1.0, 0.0], [3.0, 0.0, 1.0]]); d = np.array([1.0, 2.0, 3.0])
    assert relerr(orc.dense_solve(A, d), np.linalg.solve(A, d)) < 1e-15


def exact_rational_solve(a, b, c, d, cyclic=False):
    n = len(b)
    M = [[Fraction(0)] * (n + 1) for _ in range(n)]
    for j in range(n):
        M[j][j] = Fraction(b[j]); M[j][n] = Fraction(d[j])
        if j > 0: M[j][j - 1] = Fraction(a[j])
        if j < n - 1: M[j][j + 1] = Fraction(c[j])
    if cyclic:
        M[0][n - 1] += Fraction(a[0]); M[n - 1][0] += Fraction(c[n - 1])
    for k in range(n):
        piv = next(i for i in range(k, n) if M[i][k] != 0)
        M[k], M[piv] = M[piv], M[k]
        for i in range(k + 1, n):
            f = M[i][k] / M[k][k]
            if f: M[i] = [mi - f * mk for mi, mk in zip(M[i], M[k])]
    x = [Fraction(0)] * n
    for i in range(n - 1, -1, -1):
        x[i] = (M[i][n] - sum(M[i][j] * x[j] for j in range(i + 1, n))) / M[i][i]
    return np.array([float(v) for v in x])


def test_thomas_and_cyclic_vs_exact_rational_arithmetic():
    n = 9
    a, b, c = random_dominant(n, cyclic=True)
    d = rng.uniform(-1, 1, n)
    a0, c0 = a.copy(), c.copy(); a0[0] = 0; c0[-1] = 0
    assert relerr(orc.thomas(a0, b, c0, d), exact_rational_solve(a0, b, c0, d)) < 5e-16 * 20
    assert relerr(orc.thomas(a0, b, c0, d, long_double=True), exact_rational_solve(a0, b, c0, d)) < 3e-16
    assert relerr(orc.cyclic_thomas(a, b, c, d), exact_rational_solve(a, b, c, d, cyclic=True)) < 1e-14


@pytest.mark.parametrize("n", [16, 64, 257])
def test_manufactured_solution_dense_matvec(n):
    a, b, c = random_dominant(n)
    x = rng.normal(size=n)
    d = orc.dense_from_tridiag(a, b, c) @ x
    assert relerr(orc.thomas(a, b, c, d), x) < 1e-13
    ac, bc_, cc = random_dominant(n, cyclic=True)
    dc = orc.dense_from_tridiag(ac, bc_, cc, cyclic=True) @ x
    assert relerr(orc.cyclic_thomas(ac, bc_, cc, dc), x) < 1e-13


@pytest.mark.parametrize("n,k", [(16, 1), (16, 7), (512, 3), (512, 200)])
def test_dirichlet_eigen_closed_form(n, k):
    """constant rows (a,b,a): eigenvectors sin(jk pi/(n+1)), eigenvalues b + 2a cos(k pi/(n+1))."""
    av, bv = -0.3, 1.6
    a = np.full(n, av); b = np.full(n, bv); c = np.full(n, av)
    j = np.arange(1, n + 1)
    d = np.sin(j * k * np.pi / (n + 1))
    lam = bv + 2 * av * np.cos(k * np.pi / (n + 1))
    assert relerr(orc.thomas(a, b, c, d), d / lam) < 1e-13     # sin(j k pi/(n+1)) itself carries ~j*k*eps


@pytest.mark.parametrize("n,k", [(16, 0), (16, 5), (512, 17)])
def test_cyclic_eigen_closed_form(n, k):
    """circulant (a,b,a): eigenvectors cos(2 pi k j/n), eigenvalues b + 2a cos(2 pi k/n)."""
    av, bv = -0.4, 1.9
    a = np.full(n, av); b = np.full(n, bv); c = np.full(n, av)
    d = np.cos(2 * np.pi * k * np.arange(n) / n)
    lam = bv + 2 * av * np.cos(2 * np.pi * k / n)
    assert relerr(orc.cyclic_thomas(a, b, c, d), d / lam) < 1e-14


@pytest.mark.parametrize("n", [5, 12, 16])
def test_cyclic_vs_dense(n):
    a, b, c = random_dominant(n, cyclic=True)
    d = rng.uniform(-1, 1, n)
    A = orc.dense_from_tridiag(a, b, c, cyclic=True)
    assert relerr(orc.cyclic_thomas(a, b, c, d), np.linalg.solve(A, d)) < 1e-14
    assert relerr(orc.cyclic_thomas(a, b, c, d), orc.dense_solve(A, d)) < 1e-14


# ---------------------------------------------------------------- metrics and coefficients
def test_metrics_uniform_and_linear_exactness():
    n, L = 16, 2.0
    lo, up = orc.metrics(inputs.faces_uniform(n, L), orc.BC_DIRICHLET)
    h = L / n
    assert np.allclose(lo, 1 / h**2, rtol=1e-14) and np.allclose(up, 1 / h**2, rtol=1e-14)
    f = inputs.faces_tanh_one_sided(40, 3.0)
    lo, up = orc.metrics(f, orc.BC_DIRICHLET)
    cen = 0.5 * (f[1:] + f[:-1])
    u = 3.0 * cen - 1.0                                  # linear: delta2 u = 0 on interior rows of any grid
    d2 = up[1:-1] * (u[2:] - u[1:-1]) - lo[1:-1] * (u[1:-1] - u[:-2])
    assert np.max(np.abs(d2)) < 1e-9 * np.max(up)
    # independent restatement of hm/hp at one interior cell and at both ends (mirrored ghost)
    j = 7
    assert np.isclose(lo[j], 1 / ((cen[j] - cen[j - 1]) * (f[j + 1] - f[j])), rtol=1e-14)
    assert np.isclose(up[j], 1 / ((cen[j + 1] - cen[j]) * (f[j + 1] - f[j])), rtol=1e-14)
    assert np.isclose(lo[0], 1 / (f[1] - f[0])**2, rtol=1e-14) and np.isclose(up[-1], 1 / (f[-1] - f[-2])**2, rtol=1e-14)
    lop, upp = orc.metrics(f, orc.BC_PERIODIC)
    hper = 0.5 * ((f[1] - f[0]) + (f[-1] - f[-2]))
    assert np.isclose(lop[0], 1 / (hper * (f[1] - f[0])), rtol=1e-14) and np.isclose(upp[-1], 1 / (hper * (f[-1] - f[-2])), rtol=1e-14)


def test_delta2_quadratic_exact_on_uniform_grid():
    n, L, alpha = 32, 1.0, 1e-2
    f = inputs.faces_uniform(n, L)
    a, b, c = orc.adi_coeffs(f, orc.BC_DIRICHLET, alpha)
    cen = 0.5 * (f[1:] + f[:-1]); u = cen**2
    Au = orc.dense_from_tridiag(a, b, c) @ u
    assert np.allclose(Au[1:-1], u[1:-1] - alpha * 2.0, rtol=0, atol=1e-12)     # (I - alpha d2) x^2 = x^2 - 2 alpha


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_adi_dominance_invariant(cfg):
    """PAPER.md:L162 |b_j| = |a_j| + |c_j| + 1 (interior rows equality, boundary rows >=)."""
    c_ = configs.get(cfg)
    for f, bc in zip(c_.faces(), (orc.BC_DIRICHLET, orc.BC_DIRICHLET, orc.BC_PERIODIC)):
        a, b, c = orc.adi_coeffs(f, bc, c_.alpha)
        margin = np.abs(b) - np.abs(a) - np.abs(c)
        assert np.all(a <= 0) and np.all(c <= 0) and np.all(b > 0)
        inner = slice(1, -1) if bc != orc.BC_PERIODIC else slice(None)
        tol = 4 * np.finfo(float).eps * np.max(np.abs(b))          # b = 1 - a - c is rounded once per operation
        assert np.allclose(margin[inner], 1.0, rtol=0, atol=tol)
        assert np.all(margin >= 1.0 - tol)
        if bc == orc.BC_DIRICHLET:
            assert a[0] == 0.0 and c[-1] == 0.0
        else:
            assert a[0] != 0.0 and c[-1] != 0.0
    # alpha per BASELINE.json: dt/(2 Re)
    assert c_.alpha == {1: 5e-7, 2: 5e-7, 3: 5e-8, 4: 5e-8, 5: 5e-9}[cfg]


def test_adi_alpha_zero_is_identity_bit_exact():
    f = inputs.faces_tanh_two_sided(32, 2.0)
    a, b, c = orc.adi_coeffs(f, orc.BC_DIRICHLET, 0.0)
    d = rng.uniform(-1, 1, 32)
    assert np.array_equal(orc.thomas(a, b, c, d), d)
    assert np.array_equal(orc.partitioned_line(4, orc.MODE_PPT, a, b, c, d), d)
    assert np.array_equal(orc.partitioned_line(4, orc.MODE_PDD, a, b, c, d), d)


def test_adi_neumann_rows():
    f = inputs.faces_tanh_two_sided(16, 2.0)
    a, b, c = orc.adi_coeffs(f, orc.BC_NEUMANN, 1e-3)
    assert a[0] == 0 and c[-1] == 0 and np.isclose(b[0] + c[0], 1.0) and np.isclose(b[-1] + a[-1], 1.0)
    # constants are preserved by (I - alpha d2) with Neumann ends
    assert np.allclose(orc.dense_from_tridiag(a, b, c) @ np.ones(16), 1.0, atol=1e-14)


@pytest.mark.parametrize("lam", [0.0, 39.47, 1e4])
def test_helmholtz_invariant_and_pin(lam):
    """PAPER.md:L172 |b_j| = |a_j| + |c_j| + eps, eps = lambda (modified wavenumber)."""
    f = inputs.faces_tanh_one_sided(48, 3.0)
    a, b, c, pinned = orc.helmholtz_coeffs(f, lam)
    margin = np.abs(b) - np.abs(a) - np.abs(c)
    rows = slice(1, None) if lam == 0.0 else slice(None)
    assert np.allclose(margin[rows], lam, rtol=1e-9, atol=1e-6 * np.max(np.abs(b)) * 1e-9)
    assert pinned == (lam == 0.0)
    if pinned:
        assert b[0] == 1.0 and c[0] == 0.0
    assert a[0] == 0.0 and c[-1] == 0.0 and np.all(a[1:] > 0) and np.all(c[:-1] > 0 if not pinned else c[1:-1] > 0)


@pytest.mark.parametrize("k", [0, 1, 5])
def test_helmholtz_neumann_eigen_closed_form(k):
    """uniform grid, Neumann: eigenvectors cos(pi k (j+1/2)/n), eigenvalues -(2-2cos(pi k/n))/h^2 - lambda."""
    n, lam = 32, 7.5
    h = 1.0 / n
    a, b, c, _ = orc.helmholtz_coeffs(inputs.faces_uniform(n, 1.0), lam)
    d = np.cos(np.pi * k * (np.arange(n) + 0.5) / n)
    ev = -(2 - 2 * np.cos(np.pi * k / n)) / h**2 - lam
    assert relerr(orc.thomas(a, b, c, d), d / ev) < 1e-12


def test_modified_wavenumber_is_eigenvalue_of_periodic_delta2():
    """inputs.modified_wavenumbers_z is the symbol of the periodic second difference the ADI z-operator uses."""
    nz = 16
    f = inputs.faces_uniform(nz, 1.0)
    a, b, c = orc.adi_coeffs(f, orc.BC_PERIODIC, 1.0)            # I - delta2
    A = orc.dense_from_tridiag(a, b, c, cyclic=True)
    kz2 = inputs.modified_wavenumbers_z(nz)
    for m in (0, 1, 5, 8):
        e = np.cos(2 * np.pi * m * np.arange(nz) / nz)
        assert np.allclose(A @ e, (1.0 + kz2[m]) * e, atol=1e-9)
