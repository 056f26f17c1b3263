"""Pins for the face-located ADI operator of the oracle (the wall-normal velocity component lives on
the y-faces of the staggered grid): closed forms, invariants, dense elimination, reduction to the
cell-centred operator on a uniform grid."""
import numpy as np
import pytest

import oracle as orc
from paper_1812_01178_b200 import inputs


def _dense(a, b, c, cyclic=False):
    n = len(b)
    A = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    if cyclic:
        A[0, n - 1] += a[0]; A[n - 1, 0] += c[n - 1]
    return A


def test_face_second_difference_is_exact_on_quadratics_on_a_stretched_grid():
    n = 24
    f = inputs.faces_tanh_one_sided(n, 2.5)
    alpha = -1.0                                                # (I - alpha d2) with alpha = -1: rows of I + d2
    a, b, c = orc.adi_coeffs_face(f, orc.BC_DIRICHLET, alpha)
    # interior faces i = 1..n-3 (rows that kept both couplings): d2 applied to v = 3 y^2 - 2 y + 1 must give 6 exactly
    y = f[1:]                                                   # row i sits at face f_{i+1}
    v = 3 * y ** 2 - 2 * y + 1
    for i in range(1, n - 2):
        d2 = a[i] * v[i - 1] + (b[i] - 1.0) * v[i] + c[i] * v[i + 1]
        assert abs(d2 - 6.0) < 1e-6 * max(1.0, abs(b[i])), (i, d2)


def test_face_operator_invariants_and_wall_rows():
    n = 32
    f = inputs.faces_tanh_two_sided(n, 2.0)
    alpha = 5e-4
    a, b, c = orc.adi_coeffs_face(f, orc.BC_DIRICHLET, alpha)
    assert a[0] == 0.0 and c[n - 2] == 0.0
    assert (a[n - 1], b[n - 1], c[n - 1]) == (0.0, 1.0, 0.0)    # wall face: identity row
    i = np.arange(1, n - 2)
    assert np.allclose(b[i] - np.abs(a[i]) - np.abs(c[i]), 1.0, rtol=0, atol=1e-12)
    assert np.all(b[[0, n - 2]] - np.abs(a[[0, n - 2]]) - np.abs(c[[0, n - 2]]) > 1.0)   # wall-adjacent rows: more dominant
    assert np.all(a[1:n - 1] < 0) and np.all(c[:n - 2] < 0)


def test_face_equals_centre_coefficients_on_a_uniform_grid():
    n, L, alpha = 20, 2.0, 3e-3
    f = inputs.faces_uniform(n, L)
    h = L / n
    a, b, c = orc.adi_coeffs_face(f, orc.BC_DIRICHLET, alpha)
    ac, bc_, cc = orc.adi_coeffs(f, orc.BC_DIRICHLET, alpha)
    assert np.allclose(a[1:n - 1], -alpha / h ** 2) and np.allclose(c[:n - 2], -alpha / h ** 2)
    assert np.allclose(a[1:n - 1], ac[1:n - 1]) and np.allclose(b[1:n - 2], bc_[1:n - 2])
    ap, bp, cp = orc.adi_coeffs_face(f, orc.BC_PERIODIC, alpha)                       # periodic uniform: identical operators
    aq, bq, cq = orc.adi_coeffs(f, orc.BC_PERIODIC, alpha)
    assert np.allclose(ap, aq) and np.allclose(bp, bq) and np.allclose(cp, cq)


def test_face_dirichlet_sine_eigenvector_closed_form():
    """Uniform grid, faces f_1..f_{n-1} with v = 0 at f_0 and f_n: sin(k pi y / L) is an eigenvector of the n-1 interior
    rows with eigenvalue 1 + alpha (2 - 2 cos(k pi / n)) / h^2; the wall row passes its right-hand side through."""
    n, L, alpha, k = 16, 1.0, 2e-3, 3
    f = inputs.faces_uniform(n, L)
    h = L / n
    a, b, c = orc.adi_coeffs_face(f, orc.BC_DIRICHLET, alpha)
    y = f[1:]
    d = np.sin(k * np.pi * y / L); d[n - 1] = 0.7
    x = orc.thomas(a, b, c, d)
    lam = 1.0 + alpha * (2.0 - 2.0 * np.cos(k * np.pi / n)) / h ** 2
    assert np.allclose(x[:n - 1], d[:n - 1] / lam, rtol=0, atol=1e-14)
    assert x[n - 1] == 0.7


@pytest.mark.parametrize("bc", [orc.BC_DIRICHLET, orc.BC_PERIODIC])
def test_face_sweep_vs_dense_solve(bc):
    nx, ny, nz = 5, 12, 4
    faces = (inputs.faces_uniform(nx, 1.0), inputs.faces_tanh_one_sided(ny, 2.0), inputs.faces_uniform(nz, 1.0))
    bcs = (orc.BC_DIRICHLET, bc, orc.BC_PERIODIC)
    field = inputs.rhs_uniform((nz, ny, nx), 5)
    alpha = 1e-2
    out = orc.adi_sweep_at(field.copy(), *faces, bcs, 1, 1, orc.MODE_THOMAS, 1, alpha)
    a, b, c = orc.adi_coeffs_face(faces[1], bc, alpha)
    A = _dense(a, b, c, cyclic=(bc == orc.BC_PERIODIC))
    for k in range(nz):
        for i in range(nx):
            ref = np.linalg.solve(A, field[k, :, i])
            assert np.allclose(out[k, :, i], ref, rtol=0, atol=1e-13)
    # loc = 0 is the cell-centred sweep
    assert np.array_equal(orc.adi_sweep_at(field.copy(), *faces, bcs, 1, 0, orc.MODE_THOMAS, 1, alpha),
                          orc.adi_sweep(field.copy(), *faces, bcs, 1, orc.MODE_THOMAS, 1, alpha))


def test_face_neumann_is_rejected():
    with pytest.raises(Exception):
        orc.adi_coeffs_face(inputs.faces_uniform(8, 1.0), orc.BC_NEUMANN, 1e-3)
