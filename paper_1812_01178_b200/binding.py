"""Thin ctypes binding over csrc/libtdx.so (C ABI in include/tdx.h): argument marshalling ONLY.
Every step of the path runs in the CUDA kernels behind the C ABI.  PyTorch is used by callers for device memory
and streams; this module accepts raw device pointers (int) or anything with .data_ptr() (torch tensors).
Fails loudly (ImportError/RuntimeError) when the library is missing: there is no CPU fallback and this module
never imports oracle/."""
import ctypes as C
import os

import numpy as np

from . import build as _build

DIR_X, DIR_Y, DIR_Z = 0, 1, 2
MODE_THOMAS, MODE_PDD, MODE_PPT = 0, 1, 2
BC_DIRICHLET, BC_PERIODIC, BC_NEUMANN = 0, 1, 2
LOC_CENTER, LOC_FACE = 0, 1
GENERAL_PIVOT, GENERAL_FORCE_PARTITION, GENERAL_FORCE_LINES, GENERAL_PIVOT_PARTITIONS = 1, 16, 32, 64
OK, ERR_INVALID_ARG, ERR_BAD_PARTITION, ERR_ALLOC, ERR_CUDA, ERR_UNSUPPORTED, ERR_PDD_BOUND = 0, -1, -2, -3, -4, -5, -6

EXPORTS = ("tdx_grid_create", "tdx_grid_destroy", "tdx_grid_set_pdd_strict", "tdx_partition_bounds", "tdx_adi_sweep", "tdx_adi_sweep_at", "tdx_adi_step",
           "tdx_helmholtz_wavenumber_solve", "tdx_dct_x", "tdx_rfft_z", "tdx_irfft_z", "tdx_poisson_solve", "tdx_static_scratch_setup", "tdx_helmholtz_thomas_lines_static", "tdx_general_solve", "tdx_general_cyclic_solve", "tdx_general_fallback_count", "tdx_slab_create", "tdx_slab_destroy", "tdx_slab_eliminate", "tdx_slab_correct", "tdx_slab_dropped_bound", "tdx_cyclic_solve", "tdx_adi_sweep_host", "tdx_adi_step_host",
           "tdx_helmholtz_wavenumber_solve_host", "tdx_step_host", "tdx_step_host_async", "tdx_step_host_wait", "tdx_pdd_dropped_bound", "tdx_kernel_launch_count",
           "tdx_status_string", "tdx_last_error", "tdx_last_launch", "tdx_version")

_dp = C.POINTER(C.c_double)
_lib = None


class TdxError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("%s: %s" % (status_string(status), msg))
        self.status = status


def lib():
    """Load (building if the sources are newer) csrc/libtdx.so.  Raises if it cannot be had."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if _build.stale():
            path = _build.build()
        if not os.path.exists(path):
            raise ImportError("libtdx.so missing at %s: the CUDA extension is the only implementation" % path)
        L = C.CDLL(path)
        L.tdx_status_string.restype = C.c_char_p
        L.tdx_last_error.restype = C.c_char_p
        L.tdx_version.restype = C.c_char_p
        L.tdx_last_launch.restype = C.c_char_p
        L.tdx_kernel_launch_count.restype = C.c_longlong
        L.tdx_grid_create.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_void_p)]
        L.tdx_grid_destroy.argtypes = [C.c_void_p]
        L.tdx_grid_set_pdd_strict.argtypes = [C.c_void_p, C.c_double]
        L.tdx_partition_bounds.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_int)]
        L.tdx_adi_sweep.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_void_p, C.c_void_p]
        L.tdx_adi_sweep_at.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_void_p, C.c_void_p]
        L.tdx_adi_step.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, C.POINTER(C.c_int), C.c_void_p, C.c_void_p]
        L.tdx_helmholtz_wavenumber_solve.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, _dp, _dp, C.c_void_p, C.c_void_p]
        L.tdx_cyclic_solve.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, C.c_void_p, C.c_void_p]
        L.tdx_adi_sweep_host.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_void_p]
        L.tdx_adi_step_host.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_void_p]
        L.tdx_helmholtz_wavenumber_solve_host.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, _dp, _dp, C.c_void_p]
        L.tdx_step_host.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_void_p, C.c_int, C.c_int, _dp, C.c_void_p]
        L.tdx_step_host_async.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_void_p, C.c_int, C.c_int, _dp, C.c_void_p]
        L.tdx_step_host_wait.argtypes = [C.c_void_p, C.c_int]
        L.tdx_dct_x.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.tdx_rfft_z.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.tdx_irfft_z.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.tdx_poisson_solve.argtypes = [C.c_void_p, C.c_int, C.c_int, _dp, _dp, C.c_void_p, C.c_void_p, C.c_void_p]
        L.tdx_general_solve.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.tdx_general_cyclic_solve.argtypes = L.tdx_general_solve.argtypes
        L.tdx_general_fallback_count.argtypes = [C.c_void_p, C.POINTER(C.c_longlong)]
        L.tdx_static_scratch_setup.argtypes = [C.c_int]
        L.tdx_helmholtz_thomas_lines_static.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.tdx_slab_create.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, _dp, C.c_int, C.c_double, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_void_p)]
        L.tdx_slab_destroy.argtypes = [C.c_void_p]
        L.tdx_slab_eliminate.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.tdx_slab_correct.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.tdx_slab_dropped_bound.argtypes = [C.c_void_p, _dp]
        L.tdx_pdd_dropped_bound.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, _dp]
        _lib = L
    return _lib


def status_string(status):
    return lib().tdx_status_string(C.c_int(status)).decode()


def last_error():
    return lib().tdx_last_error().decode()


def last_launch():
    """Kernel name (with template arguments) and launch shape of this thread's last PDD / PPT sweep launch."""
    return lib().tdx_last_launch().decode()


def version():
    return lib().tdx_version().decode()


def kernel_launch_count():
    return int(lib().tdx_kernel_launch_count())


def _chk(rc):
    if rc != OK:
        raise TdxError(rc, last_error())


def _host(arr):
    if arr is None:
        return None, None
    a = np.ascontiguousarray(arr, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def _devptr(x):
    return C.c_void_p(int(x.data_ptr()) if hasattr(x, "data_ptr") else int(x))


def _hostptr(arr, nbytes):
    assert isinstance(arr, np.ndarray) and arr.flags.c_contiguous and arr.nbytes == nbytes, "host buffer: C-contiguous, %d bytes" % nbytes
    return C.c_void_p(arr.ctypes.data)


STATIC_SCRATCH_DOUBLES = 2359296


def static_scratch_setup(device=0):
    _chk(lib().tdx_static_scratch_setup(int(device)))


def partition_bounds(n, P):
    st = (C.c_int * (P + 1))()
    _chk(lib().tdx_partition_bounds(n, P, st))
    return np.array(st[:], dtype=np.int32)


class Grid:
    """tdx_grid_create / tdx_grid_destroy.  faces: host arrays of n+1 face coordinates."""

    def __init__(self, nx, ny, nz, xf, yf, zf, bcs=(BC_DIRICHLET, BC_DIRICHLET, BC_PERIODIC), device=0):
        self.nx, self.ny, self.nz = nx, ny, nz
        self._h = C.c_void_p()
        (_, px), (_, py), (_, pz) = _host(xf), _host(yf), _host(zf)
        assert len(xf) == nx + 1 and len(yf) == ny + 1 and len(zf) == nz + 1
        _chk(lib().tdx_grid_create(nx, ny, nz, px, py, pz, bcs[0], bcs[1], bcs[2], device, C.byref(self._h)))

    def close(self):
        if self._h:
            lib().tdx_grid_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_pdd_strict(self, max_dropped):
        _chk(lib().tdx_grid_set_pdd_strict(self._h, float(max_dropped)))

    def adi_sweep(self, direction, mode, P, alpha, rhs, stream=0):
        _chk(lib().tdx_adi_sweep(self._h, direction, mode, P, alpha, _devptr(rhs), C.c_void_p(stream)))

    def adi_sweep_at(self, direction, loc, mode, P, alpha, rhs, stream=0):
        _chk(lib().tdx_adi_sweep_at(self._h, direction, loc, mode, P, alpha, _devptr(rhs), C.c_void_p(stream)))

    def adi_step(self, mode, Px, Py, Pz, alpha, ncomp, loc, rhs, stream=0):
        """loc: None or ncomp*3 ints (loc[c*3+dir]); rhs: device buffer of ncomp fields stored back to back."""
        arr = None
        if loc is not None:
            flat = [int(v) for v in np.asarray(loc).reshape(-1)]
            assert len(flat) == ncomp * 3
            arr = (C.c_int * len(flat))(*flat)
        _chk(lib().tdx_adi_step(self._h, mode, Px, Py, Pz, alpha, ncomp, arr, _devptr(rhs), C.c_void_p(stream)))

    def helmholtz_wavenumber_solve(self, mode, P, kx2, kz2, rhs, stream=0):
        kz, pkz = _host(kz2)
        _, pkx = _host(kx2)
        _chk(lib().tdx_helmholtz_wavenumber_solve(self._h, mode, P, kz.size, pkx, pkz, _devptr(rhs), C.c_void_p(stream)))

    def helmholtz_thomas_lines_static(self, nm, kx2_dev, kz2_dev, rhs, stream=0):
        """The entry point that allocates nothing: kx2_dev / kz2_dev are DEVICE arrays; scratch is the library's static array."""
        _chk(lib().tdx_helmholtz_thomas_lines_static(self._h, int(nm), _devptr(kx2_dev), _devptr(kz2_dev), _devptr(rhs), C.c_void_p(stream)))

    def dct_x(self, inverse, field, stream=0):
        _chk(lib().tdx_dct_x(self._h, int(inverse), _devptr(field), C.c_void_p(stream)))

    def rfft_z(self, field_in, spec_out, stream=0):
        _chk(lib().tdx_rfft_z(self._h, _devptr(field_in), _devptr(spec_out), C.c_void_p(stream)))

    def irfft_z(self, spec_in, field_out, stream=0):
        _chk(lib().tdx_irfft_z(self._h, _devptr(spec_in), _devptr(field_out), C.c_void_p(stream)))

    def poisson_solve(self, mode, P, kx2, kz2, field, spec_work, stream=0):
        _, pkx = _host(kx2)
        _, pkz = _host(kz2)
        _chk(lib().tdx_poisson_solve(self._h, mode, P, pkx, pkz, _devptr(field), _devptr(spec_work), C.c_void_p(stream)))

    def general_solve(self, direction, pivoting, a, b, c, rhs, work, stream=0):
        _chk(lib().tdx_general_solve(self._h, direction, int(pivoting), _devptr(a), _devptr(b), _devptr(c), _devptr(rhs), _devptr(work), C.c_void_p(stream)))

    def general_cyclic_solve(self, direction, pivoting, a, b, c, rhs, work, stream=0):
        _chk(lib().tdx_general_cyclic_solve(self._h, direction, int(pivoting), _devptr(a), _devptr(b), _devptr(c), _devptr(rhs), _devptr(work), C.c_void_p(stream)))

    def general_fallback_count(self):
        out = C.c_longlong(0)
        _chk(lib().tdx_general_fallback_count(self._h, C.byref(out)))
        return int(out.value)

    def cyclic_solve(self, direction, mode, P, a, b, c, rhs, stream=0):
        (_, pa), (_, pb), (_, pc) = _host(a), _host(b), _host(c)
        _chk(lib().tdx_cyclic_solve(self._h, direction, mode, P, pa, pb, pc, _devptr(rhs), C.c_void_p(stream)))

    def adi_sweep_host(self, direction, mode, P, alpha, host_rhs):
        _chk(lib().tdx_adi_sweep_host(self._h, direction, mode, P, alpha, _hostptr(host_rhs, self.nx * self.ny * self.nz * 8)))

    def adi_step_host(self, mode, Px, Py, Pz, alpha, host_rhs):
        _chk(lib().tdx_adi_step_host(self._h, mode, Px, Py, Pz, alpha, _hostptr(host_rhs, self.nx * self.ny * self.nz * 8)))

    def helmholtz_wavenumber_solve_host(self, mode, P, kx2, kz2, host_rhs):
        kz, pkz = _host(kz2)
        _, pkx = _host(kx2)
        _chk(lib().tdx_helmholtz_wavenumber_solve_host(self._h, mode, P, kz.size, pkx, pkz,
                                                       _hostptr(host_rhs, self.nx * self.ny * kz.size * 16)))

    def step_host(self, mode, Px, Py, Pz, alpha, host_field, Ph, kz2, host_helm):
        """Pipelined whole step on host buffers (either may be None)."""
        kz, pkz = _host(kz2) if host_helm is not None else (None, None)
        pf = _hostptr(host_field, self.nx * self.ny * self.nz * 8) if host_field is not None else None
        ph = _hostptr(host_helm, self.nx * self.ny * kz.size * 16) if host_helm is not None else None
        _chk(lib().tdx_step_host(self._h, mode, Px, Py, Pz, alpha, pf, Ph, kz.size if kz is not None else 0, pkz, ph))

    def step_host_async(self, slot, mode, Px, Py, Pz, alpha, host_field, Ph, kz2, host_helm):
        """The pipelined step enqueued only (slot 0 or 1); the host buffers are valid after step_host_wait(slot)."""
        kz, pkz = _host(kz2) if host_helm is not None else (None, None)
        pf = _hostptr(host_field, self.nx * self.ny * self.nz * 8) if host_field is not None else None
        ph = _hostptr(host_helm, self.nx * self.ny * kz.size * 16) if host_helm is not None else None
        _chk(lib().tdx_step_host_async(self._h, slot, mode, Px, Py, Pz, alpha, pf, Ph, kz.size if kz is not None else 0, pkz, ph))

    def step_host_wait(self, slot):
        _chk(lib().tdx_step_host_wait(self._h, slot))

    def pdd_dropped_bound(self, direction, P, alpha):
        out = C.c_double(0.0)
        _chk(lib().tdx_pdd_dropped_bound(self._h, direction, P, alpha, C.byref(out)))
        return out.value


class Slab:
    """tdx_slab_t: one rank's share of a slab-decomposed sweep (include/tdx.h).  Holds a reference to its grid."""

    def __init__(self, slab_grid, direction, rank, nranks, faces_global, bc_global, alpha, across, local_mode, P_local):
        f, pf = _host(faces_global)
        self._grid = slab_grid
        self._h = C.c_void_p()
        self.rank, self.nranks, self.direction = rank, nranks, direction
        _chk(lib().tdx_slab_create(slab_grid._h, direction, rank, nranks, f.size - 1, pf, bc_global, float(alpha), across,
                                   local_mode, P_local, C.byref(self._h)))

    def close(self):
        if self._h:
            lib().tdx_slab_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def eliminate(self, field, iface_out, stream=0):
        _chk(lib().tdx_slab_eliminate(self._h, _devptr(field), _devptr(iface_out), C.c_void_p(stream)))

    def correct(self, field, iface_own, iface_nbr, stream=0):
        _chk(lib().tdx_slab_correct(self._h, _devptr(field), _devptr(iface_own), _devptr(iface_nbr) if iface_nbr is not None else None, C.c_void_p(stream)))

    def dropped_bound(self):
        out = C.c_double(0.0)
        _chk(lib().tdx_slab_dropped_bound(self._h, C.byref(out)))
        return out.value
