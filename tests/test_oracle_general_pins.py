"""Pins for oracle/general.py: the dense LAPACK solve of per-line tridiagonal systems against things
that are not itself -- manufactured solutions through an independent mat-vec, the oracle's own Thomas on dominant
systems (plain C, different code), exact rational arithmetic on a tiny system with a zero pivot."""
from fractions import Fraction

import numpy as np

import general as ogen
import oracle as orc
from paper_1812_01178_b200 import inputs


def _fields(shape, seed, diag_scale):
    n = int(np.prod(shape))
    a = inputs.uniform_pm1(seed, n, stream=1).reshape(shape)
    b = diag_scale * inputs.uniform_pm1(seed, n, stream=2).reshape(shape)
    c = inputs.uniform_pm1(seed, n, stream=3).reshape(shape)
    return a, b, c


def _matvec(a, b, c, x, axis, cyclic=False):
    y = b * x
    xm = np.moveaxis(x, axis, 0); am = np.moveaxis(a, axis, 0); cm = np.moveaxis(c, axis, 0); ym = np.moveaxis(y, axis, 0)
    ym[1:] += am[1:] * xm[:-1]
    ym[:-1] += cm[:-1] * xm[1:]
    if cyclic:
        ym[0] += am[0] * xm[-1]
        ym[-1] += cm[-1] * xm[0]
    return y


def test_manufactured_solutions_along_x_and_periodic_lines():
    shape = (5, 7, 18)
    for axis, cyclic in ((2, False), (2, True), (1, True), (0, True)):
        a, b, c = _fields(shape, 61 + axis, 0.3)
        x = inputs.uniform_pm1(63, int(np.prod(shape))).reshape(shape)
        d = _matvec(a, b, c, x, axis, cyclic)
        got, A = ogen.general_solve(a, b, c, d, axis, cyclic)
        cond = np.linalg.cond(A)
        err = np.max(np.abs(np.moveaxis(got - x, axis, -1).reshape(len(cond), -1)), axis=1)
        assert np.all(err <= 1e-14 * cond * 10), float(np.max(err / cond))
        if cyclic:                                               # the corners really are part of the system
            plain, _ = ogen.general_solve(a, b, c, d, axis, False)
            assert np.max(np.abs(plain - x)) > 1e-3


def test_periodic_dominant_systems_agree_with_the_c_cyclic_thomas():
    shape = (2, 21, 3)
    a, b, c = _fields(shape, 71, 1.0)
    b = 3.0 + np.abs(b)
    d = inputs.uniform_pm1(72, int(np.prod(shape))).reshape(shape)
    got, _ = ogen.general_solve(a, b, c, d, 1, cyclic=True)
    for k in range(shape[0]):
        for i in range(shape[2]):
            ref = orc.cyclic_thomas(np.ascontiguousarray(a[k, :, i]), np.ascontiguousarray(b[k, :, i]), np.ascontiguousarray(c[k, :, i]),
                                    np.ascontiguousarray(d[k, :, i]))
            assert np.max(np.abs(got[k, :, i] - ref)) < 1e-14


def test_manufactured_solutions_non_dominant_both_axes():
    shape = (6, 20, 8)
    for axis in (1, 0):
        a, b, c = _fields(shape, 41 + axis, 0.3)                  # small diagonals: far from dominant
        x = inputs.uniform_pm1(43, int(np.prod(shape))).reshape(shape)
        d = _matvec(a, b, c, x, axis)
        got, A = ogen.general_solve(a, b, c, d, axis)
        cond = np.linalg.cond(A)
        err = np.max(np.abs(np.moveaxis(got - x, axis, -1).reshape(len(cond), -1)), axis=1)
        assert np.all(err <= 1e-14 * cond * 10), float(np.max(err / cond))


def test_dominant_systems_agree_with_the_c_thomas():
    shape = (2, 24, 3)
    a, b, c = _fields(shape, 51, 1.0)
    b = 3.0 + np.abs(b)                                          # strictly dominant
    d = inputs.uniform_pm1(52, int(np.prod(shape))).reshape(shape)
    got, _ = ogen.general_solve(a, b, c, d, 1)
    for k in range(shape[0]):
        for i in range(shape[2]):
            ref = orc.thomas(np.ascontiguousarray(a[k, :, i]), np.ascontiguousarray(b[k, :, i]), np.ascontiguousarray(c[k, :, i]),
                             np.ascontiguousarray(d[k, :, i]))
            assert np.max(np.abs(got[k, :, i] - ref)) < 1e-14


def test_zero_pivot_system_exact_rational():
    """b_0 = 0: Thomas without pivoting divides by zero; the system itself is regular.  Exact solution by Cramer's rule
    in rational arithmetic."""
    a = np.array([0.0, 2.0, 1.0]); b = np.array([0.0, 1.0, 3.0]); c = np.array([1.0, -1.0, 0.0]); d = np.array([1.0, 2.0, 5.0])
    A = [[Fraction(0), Fraction(1), Fraction(0)], [Fraction(2), Fraction(1), Fraction(-1)], [Fraction(0), Fraction(1), Fraction(3)]]
    rhs = [Fraction(1), Fraction(2), Fraction(5)]
    def det(M):
        return (M[0][0] * (M[1][1] * M[2][2] - M[1][2] * M[2][1]) - M[0][1] * (M[1][0] * M[2][2] - M[1][2] * M[2][0])
                + M[0][2] * (M[1][0] * M[2][1] - M[1][1] * M[2][0]))
    D = det(A)
    want = []
    for col in range(3):
        M = [row[:] for row in A]
        for r in range(3):
            M[r][col] = rhs[r]
        want.append(float(det(M) / D))
    got, _ = ogen.general_solve(a.reshape(1, 3, 1), b.reshape(1, 3, 1), c.reshape(1, 3, 1), d.reshape(1, 3, 1), 1)
    assert np.max(np.abs(got[0, :, 0] - np.array(want))) < 1e-15
