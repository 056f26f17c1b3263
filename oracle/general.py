"""Batched tridiagonal systems with per-line coefficients -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

PAPER.md:L174: the Poisson y-systems are solved with "a parallel tridiagonal solver with diagonal pivoting [3]" because
they are not safely dominant (L172).  What such a solver must return has a plain definition -- the solution of A x = d --
so the oracle is that definition: every line's matrix is assembled densely and handed to LAPACK's general solver
(numpy.linalg.solve: LU with partial pivoting, fp64).  Nothing of the GPU's pivoting strategy is restated here.
Only tests/ may import this.  It imports nothing from paper_1812_01178_b200.
Pinned by tests/test_oracle_general_pins.py (manufactured solutions through an independent mat-vec along x, y and z, also
periodic; the C Thomas / cyclic Thomas on dominant systems; an exact rational zero-pivot system); nothing here is
"parity unpinned".
"""
import numpy as np


def dense_lines(a, b, c, axis, cyclic=False):
    """a, b, c: [nz][ny][nx] coefficient fields; returns [lines][n][n] dense matrices of the lines along `axis` (2 = x, 1 = y,
    0 = z in array terms) in the order of np.moveaxis(field, axis, -1).reshape(-1, n).  cyclic: a of a line's first row
    couples it to the last row and c of the last row to the first (the periodic direction; "spanwisely
    periodic"), entries (0, n-1) and (n-1, 0) of the dense matrix."""
    am = np.moveaxis(a, axis, -1).reshape(-1, a.shape[axis])
    bm = np.moveaxis(b, axis, -1).reshape(-1, a.shape[axis])
    cm = np.moveaxis(c, axis, -1).reshape(-1, a.shape[axis])
    L, n = bm.shape
    A = np.zeros((L, n, n))
    idx = np.arange(n)
    A[:, idx, idx] = bm
    A[:, idx[1:], idx[:-1]] = am[:, 1:]          # a_j couples row j to row j-1 (a of the first row is not part of the system)
    A[:, idx[:-1], idx[1:]] = cm[:, :-1]         # c_j couples row j to row j+1 (c of the last row is not part of the system)
    if cyclic:
        A[:, 0, n - 1] += am[:, 0]
        A[:, n - 1, 0] += cm[:, n - 1]
    return A


def general_solve(a, b, c, d, axis, cyclic=False):
    """Solution field of the per-line systems along `axis`; also returns the dense matrices (for condition numbers)."""
    A = dense_lines(a, b, c, axis, cyclic)
    n = d.shape[axis]
    dm = np.moveaxis(d, axis, -1).reshape(-1, n)
    x = np.linalg.solve(A, dm[:, :, None])[:, :, 0]
    shp = np.moveaxis(d, axis, -1).shape
    return np.ascontiguousarray(np.moveaxis(x.reshape(shp), -1, axis)), A
