"""ctypes wrapper over oracle/liboracle.so -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
All arithmetic lives in oracle.c (plain C, fp64, cited to PAPER.md); this file only marshals numpy arrays.
It imports nothing from paper_1812_01178_b200.
"""
import ctypes as C
import os
import sys
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, _HERE)
import build as _build  # noqa: E402  (oracle/build.py)
sys.path.pop(0)

_lib = C.CDLL(_build.build())

BC_DIRICHLET, BC_PERIODIC, BC_NEUMANN = 0, 1, 2
MODE_THOMAS, MODE_PDD, MODE_PPT, MODE_THOMAS_LD = 0, 1, 2, 3

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def _p(arr):
    return arr.ctypes.data_as(_dp) if arr is not None else None


def _c(x):
    return np.ascontiguousarray(x, dtype=np.float64)


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError("oracle: %s failed (rc=%d)" % (what, rc))


_lib.oracle_pdd_dropped.restype = C.c_double
_lib.oracle_cyclic_pdd_dropped.restype = C.c_double
_lib.oracle_cyclic_pdd_outer_dropped.restype = C.c_double
_lib.oracle_pdd_dropped.argtypes = [C.c_int, C.c_int, _dp, _dp, _dp]


def num_threads():
    return int(_lib.oracle_num_threads())


def set_num_threads(n):
    """OpenMP threads of the loops over lines (timing only: no result depends on it).  Returns the count now in force."""
    return int(_lib.oracle_set_num_threads(C.c_int(int(n))))


def partition_bounds(n, P):
    st = np.zeros(P + 1, dtype=np.int32)
    _chk(_lib.oracle_partition_bounds(C.c_int(n), C.c_int(P), st.ctypes.data_as(_ip)), "partition_bounds")
    return st


def metrics(faces, bc):
    f = _c(faces); n = f.size - 1
    lo = np.empty(n); up = np.empty(n)
    _chk(_lib.oracle_metrics(C.c_int(n), _p(f), C.c_int(bc), _p(lo), _p(up)), "metrics")
    return lo, up


def adi_coeffs(faces, bc, alpha):
    f = _c(faces); n = f.size - 1
    a = np.empty(n); b = np.empty(n); c = np.empty(n)
    _chk(_lib.oracle_adi_coeffs(C.c_int(n), _p(f), C.c_int(bc), C.c_double(alpha), _p(a), _p(b), _p(c)), "adi_coeffs")
    return a, b, c


def adi_coeffs_face(faces, bc, alpha):
    f = _c(faces); n = f.size - 1
    a = np.empty(n); b = np.empty(n); c = np.empty(n)
    _chk(_lib.oracle_adi_coeffs_face(C.c_int(n), _p(f), C.c_int(bc), C.c_double(alpha), _p(a), _p(b), _p(c)), "adi_coeffs_face")
    return a, b, c


def helmholtz_coeffs(faces, lam):
    f = _c(faces); n = f.size - 1
    a = np.empty(n); b = np.empty(n); c = np.empty(n); pinned = C.c_int(0)
    _chk(_lib.oracle_helmholtz_coeffs(C.c_int(n), _p(f), C.c_double(lam), _p(a), _p(b), _p(c), C.byref(pinned)), "helmholtz_coeffs")
    return a, b, c, bool(pinned.value)


def thomas(a, b, c, d, long_double=False):
    a, b, c, d = _c(a), _c(b), _c(c), _c(d)
    x = np.empty_like(d)
    fn = _lib.oracle_thomas_ld if long_double else _lib.oracle_thomas
    _chk(fn(C.c_int(d.size), _p(a), _p(b), _p(c), _p(d), _p(x)), "thomas")
    return x


def cyclic_thomas(a, b, c, d):
    a, b, c, d = _c(a), _c(b), _c(c), _c(d)
    x = np.empty_like(d)
    _chk(_lib.oracle_cyclic_thomas(C.c_int(d.size), _p(a), _p(b), _p(c), _p(d), _p(x)), "cyclic_thomas")
    return x


def dense_solve(A, d):
    A, d = _c(A), _c(d)
    x = np.empty_like(d)
    _chk(_lib.oracle_dense_solve(C.c_int(d.size), _p(A), _p(d), _p(x)), "dense_solve")
    return x


def dense_from_tridiag(a, b, c, cyclic=False):
    a, b, c = _c(a), _c(b), _c(c)
    n = b.size
    A = np.empty((n, n))
    _chk(_lib.oracle_dense_from_tridiag(C.c_int(n), _p(a), _p(b), _p(c), C.c_int(int(cyclic)), _p(A)), "dense_from_tridiag")
    return A


def local_solves(P, a, b, c, d):
    a, b, c, d = _c(a), _c(b), _c(c), _c(d)
    n = b.size
    xt = np.empty(n); v = np.empty(n); w = np.empty(n)
    _chk(_lib.oracle_local_solves(C.c_int(n), C.c_int(P), _p(a), _p(b), _p(c), _p(d), _p(xt), _p(v), _p(w)), "local_solves")
    return xt, v, w


def build_Z(n, P, v, w, pdd=False):
    v, w = _c(v), _c(w)
    K = 2 * (P - 1)
    Z = np.empty((K, K))
    _chk(_lib.oracle_build_Z(C.c_int(n), C.c_int(P), _p(v), _p(w), C.c_int(int(pdd)), _p(Z)), "build_Z")
    return Z


def build_Zbar(Z):
    Z = _c(Z)
    Zb = np.empty_like(Z)
    _chk(_lib.oracle_build_Zbar(C.c_int(Z.shape[0]), _p(Z), _p(Zb)), "build_Zbar")
    return Zb


def pdd_dropped(P, a, b, c):
    a, b, c = _c(a), _c(b), _c(c)
    return float(_lib.oracle_pdd_dropped(C.c_int(b.size), C.c_int(P), _p(a), _p(b), _p(c)))


def cyclic_pdd_dropped(P, a, b, c):
    """a-priori bound of PDD on a periodic line (reduced system closed cyclically): every partition's far spike ends."""
    a, b, c = _c(a), _c(b), _c(c)
    return float(_lib.oracle_cyclic_pdd_dropped(C.c_int(b.size), C.c_int(P), _p(a), _p(b), _p(c)))


def cyclic_pdd_line(P, a, b, c, d, return_spikes=False):
    """PDD on one periodic line, P interfaces (oracle_cyclic_pdd_line); optionally the spikes v, w (each length n)."""
    a, b, c, d = _c(a), _c(b), _c(c), _c(d)
    x = np.empty_like(d)
    sp = np.zeros(2 * d.size)
    _chk(_lib.oracle_cyclic_pdd_line(C.c_int(d.size), C.c_int(P), _p(a), _p(b), _p(c), _p(d), _p(x), _p(sp)), "cyclic_pdd_line")
    return (x, sp[:d.size].copy(), sp[d.size:].copy()) if return_spikes else x


def cyclic_pdd_outer_line(P, a, b, c, d):
    """PDD on one periodic line by the OUTER rank-1 split (SURVEY 8(c) C2's oracle definition; oracle_cyclic_pdd_outer_line)."""
    a, b, c, d = _c(a), _c(b), _c(c), _c(d)
    x = np.empty_like(d)
    _chk(_lib.oracle_cyclic_pdd_outer_line(C.c_int(d.size), C.c_int(P), _p(a), _p(b), _p(c), _p(d), _p(x)), "cyclic_pdd_outer_line")
    return x


def cyclic_pdd_outer_dropped(P, a, b, c):
    """a-priori bound of the outer-split PDD: the far spike ends of the split matrix A'."""
    a, b, c = _c(a), _c(b), _c(c)
    return float(_lib.oracle_cyclic_pdd_outer_dropped(C.c_int(b.size), C.c_int(P), _p(a), _p(b), _p(c)))


def partitioned_line(P, mode, a, b, c, d, return_y=False):
    a, b, c, d = _c(a), _c(b), _c(c), _c(d)
    x = np.empty_like(d)
    y = np.zeros(max(2 * (P - 1), 1))
    _chk(_lib.oracle_partitioned_line(C.c_int(d.size), C.c_int(P), C.c_int(mode), _p(a), _p(b), _p(c), _p(d), _p(x), _p(y)), "partitioned_line")
    return (x, y[:2 * (P - 1)]) if return_y else x


def cyclic_line(P, mode, a, b, c, d):
    a, b, c, d = _c(a), _c(b), _c(c), _c(d)
    x = np.empty_like(d)
    _chk(_lib.oracle_cyclic_line(C.c_int(d.size), C.c_int(P), C.c_int(mode), _p(a), _p(b), _p(c), _p(d), _p(x)), "cyclic_line")
    return x


def _field(field, shape):
    assert field.dtype == np.float64 and field.flags.c_contiguous and field.shape == shape, "field must be C-contiguous float64 %r" % (shape,)


def adi_sweep(field_zyx, xf, yf, zf, bcs, direction, mode, P, alpha):
    """In place on field_zyx (numpy [nz][ny][nx] float64). bcs = (bcx, bcy, bcz)."""
    nz, ny, nx = field_zyx.shape
    _field(field_zyx, (nz, ny, nx))
    xf, yf, zf = _c(xf), _c(yf), _c(zf)
    _chk(_lib.oracle_adi_sweep(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(xf), _p(yf), _p(zf),
                               C.c_int(bcs[0]), C.c_int(bcs[1]), C.c_int(bcs[2]), C.c_int(direction), C.c_int(mode),
                               C.c_int(P), C.c_double(alpha), _p(field_zyx)), "adi_sweep")
    return field_zyx


def adi_sweep_at(field_zyx, xf, yf, zf, bcs, direction, loc, mode, P, alpha):
    """As adi_sweep with the unknowns of `direction` at cell centres (loc 0) or faces (loc 1)."""
    nz, ny, nx = field_zyx.shape
    _field(field_zyx, (nz, ny, nx))
    xf, yf, zf = _c(xf), _c(yf), _c(zf)
    _chk(_lib.oracle_adi_sweep_at(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(xf), _p(yf), _p(zf),
                                  C.c_int(bcs[0]), C.c_int(bcs[1]), C.c_int(bcs[2]), C.c_int(direction), C.c_int(loc),
                                  C.c_int(mode), C.c_int(P), C.c_double(alpha), _p(field_zyx)), "adi_sweep_at")
    return field_zyx


def sweep_coeffs(field_zyx, direction, mode, P, periodic, a, b, c):
    nz, ny, nx = field_zyx.shape
    _field(field_zyx, (nz, ny, nx))
    a, b, c = _c(a), _c(b), _c(c)
    _chk(_lib.oracle_sweep_coeffs(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_int(direction), C.c_int(mode), C.c_int(P),
                                  C.c_int(int(periodic)), _p(a), _p(b), _p(c), _p(field_zyx)), "sweep_coeffs")
    return field_zyx


def cyclic_solve(field_zyx, direction, mode, P, a, b, c):
    return sweep_coeffs(field_zyx, direction, mode, P, True, a, b, c)


def helmholtz_solve(field_myx, yf, kx2, kz2, mode, P):
    """In place on complex128 [nm][ny][nx]."""
    nm, ny, nx = field_myx.shape
    assert field_myx.dtype == np.complex128 and field_myx.flags.c_contiguous
    yf, kz2 = _c(yf), _c(kz2)
    kx2 = _c(kx2) if kx2 is not None else None
    view = field_myx.view(np.float64)
    _chk(_lib.oracle_helmholtz_solve(C.c_int(nx), C.c_int(ny), C.c_int(nm), _p(yf), _p(kx2), _p(kz2), C.c_int(mode),
                                     C.c_int(P), _p(view)), "helmholtz_solve")
    return field_myx
