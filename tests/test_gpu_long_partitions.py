"""GPU parity for partitions longer than one thread keeps in registers (1 <= P <= 128, floor(n/P) >= 2 --
any partition length; PAPER.md:L112 m = n/p for any p).  The library cuts such partitions again inside the thread block
(two-level plans) and must return the result of the CALLER's P: PPT exact (1e-12 of the oracle's
Thomas), PDD = the oracle's step-by-step PDD with the caller's P (1e-12), also where the couplings PDD deletes are
visible (alpha = 1e-3: the spikes decay to 1e-2 ... 1e-7 over such a partition), so a composite that approximated anything
else would fail.  Gates: 1e-12 at the configs' weak coupling; 1e-11 at alpha = 1e-3, where cond(A) reaches 1e3-1e4 and two
backward-stable algorithms may differ by that much.
Also here: the strict PDD switch (TDX_ERR_PDD_BOUND) and the per-line Helmholtz solve with long partitions."""
import numpy as np
import pytest
import torch

import oracle as orc
from paper_1812_01178_b200 import binding as tdx
from paper_1812_01178_b200 import configs, inputs

pytestmark = pytest.mark.gpu

BCS = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
MODES = {"pdd": tdx.MODE_PDD, "ppt": tdx.MODE_PPT}


def relerr(x, ref):
    return float(np.max(np.abs(x - ref)) / np.max(np.abs(ref)))


def grid_for(direction, n, other=(12, 10)):
    """n points along `direction`, a few along the others (even x extent); stretched along y, uniform else."""
    dims = [other[0], other[1], other[1]]
    dims[direction] = n
    if direction != 0 and dims[0] % 2:
        dims[0] += 1
    nx, ny, nz = dims
    faces = (inputs.faces_uniform(nx, 1.0), inputs.faces_tanh_two_sided(ny, 2.0), inputs.faces_uniform(nz, 1.0))
    return (nx, ny, nz), faces


def dropped_of(faces, direction, P, alpha):
    a, b, c = orc.adi_coeffs(faces[direction], BCS[direction], alpha)
    return orc.cyclic_pdd_dropped(P, a, b, c) if BCS[direction] == orc.BC_PERIODIC else orc.pdd_dropped(P, a, b, c)


# (direction, n, P): 128-row and 100-row partitions, ragged ones (n % P != 0 and rows % sub-partitions != 0), 2 partitions
CASES = [(0, 512, 4), (0, 400, 4), (0, 203, 2), (0, 1024, 8), (0, 330, 3), (0, 192, 2), (0, 96, 2),
         (1, 256, 2), (1, 400, 4), (1, 205, 2), (1, 130, 2), (1, 66, 1 + 1),
         (2, 256, 2), (2, 300, 3), (2, 205, 2), (2, 512, 4)]


@pytest.mark.parametrize("direction,n,P", CASES)
@pytest.mark.parametrize("mode_name", ["ppt", "pdd"])
@pytest.mark.parametrize("alpha", [1e-6, 1e-3])
def test_long_partitions_every_element(direction, n, P, mode_name, alpha):
    (nx, ny, nz), faces = grid_for(direction, n)
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    field = inputs.rhs_uniform((nz, ny, nx), 17 + n + P)
    t = torch.from_numpy(field).cuda()
    grid.adi_sweep(direction, MODES[mode_name], P, alpha, t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    exact = orc.adi_sweep(field.copy(), *faces, BCS, direction, orc.MODE_THOMAS, 1, alpha)
    tol = 1e-12 if alpha < 1e-4 else 1e-11
    if mode_name == "ppt":
        assert relerr(out, exact) < tol, (direction, n, P, alpha, relerr(out, exact))
    else:
        dropped = dropped_of(faces, direction, P, alpha)
        got = grid.pdd_dropped_bound(direction, P, alpha)
        assert abs(got - dropped) <= 1e-9 * dropped + 1e-300, (got, dropped)
        ref = orc.adi_sweep(field.copy(), *faces, BCS, direction, orc.MODE_PDD, P, alpha)
        assert relerr(out, ref) < tol, ("pdd vs oracle pdd with the caller's P", direction, n, P, alpha, relerr(out, ref), dropped)
        if dropped <= 1e-11:
            assert relerr(out, exact) < 1e-10
        else:
            assert relerr(out, exact) < 100 * dropped + 1e-10
    grid.close()


# (direction, n, P): 4-, 3-, 2-row and ragged 5/4-row partitions
SHORT_CASES = [(1, 256, 64), (2, 256, 64), (1, 96, 32), (2, 64, 32), (1, 150, 33), (2, 127, 42), (0, 128, 32), (0, 90, 30)]


@pytest.mark.parametrize("direction,n,P", SHORT_CASES)
@pytest.mark.parametrize("alpha", [1e-6, 1e-3])
def test_short_partitions_ppt_merges_them_pdd_keeps_the_callers_map(direction, n, P, alpha):
    """Fewer than 8 rows per partition: PPT (exact for any partitioning) runs with neighbouring partitions
    merged pairwise until a thread has 8 rows -- the launch shows fewer partitions, the result is the exact
    solution; PDD depends on P, keeps the caller's map and equals the oracle's PDD with that P."""
    (nx, ny, nz), faces = grid_for(direction, n, other=(16, 10))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    field = inputs.rhs_uniform((nz, ny, nx), 23 + n + P)
    exact = orc.adi_sweep(field.copy(), *faces, BCS, direction, orc.MODE_THOMAS, 1, alpha)
    tol = 1e-12 if alpha < 1e-4 else 1e-11
    t = torch.from_numpy(field).cuda()
    grid.adi_sweep(direction, tdx.MODE_PPT, P, alpha, t)
    torch.cuda.synchronize()
    assert relerr(t.cpu().numpy(), exact) < tol, (direction, n, P, alpha, relerr(t.cpu().numpy(), exact))
    Pm = P
    while n // Pm < 8 and Pm >= 4:
        Pm = (Pm + 1) // 2
    launch = tdx.last_launch()
    if direction != 0:                                           # strided kernels: block = (lines, partitions)
        assert "block=(" in launch and launch.split("block=(")[1].split(",")[1] == str(Pm), (launch, Pm)
    t = torch.from_numpy(field).cuda()
    grid.adi_sweep(direction, tdx.MODE_PDD, P, alpha, t)
    torch.cuda.synchronize()
    ref = orc.adi_sweep(field.copy(), *faces, BCS, direction, orc.MODE_PDD, P, alpha)
    assert relerr(t.cpu().numpy(), ref) < tol, ("pdd", direction, n, P, alpha, relerr(t.cpu().numpy(), ref))
    if direction != 0 and dropped_of(faces, direction, P, alpha) >= 1e-20:
        launch = tdx.last_launch()
        assert launch.split("block=(")[1].split(",")[1] == str(P), (launch, P)
    grid.close()


def test_long_partition_pdd_is_the_callers_pdd_not_the_sub_partitions():
    """alpha = 1e-3 on 400 uniform rows: PDD with P = 4 (100 rows) deletes couplings of a few 1e-4; PDD with the 16
    sub-partitions the kernel runs would delete O(0.1) ones.  The result must be the former."""
    (nx, ny, nz), faces = grid_for(0, 400)
    alpha = 1e-3
    d4, d16 = dropped_of(faces, 0, 4, alpha), dropped_of(faces, 0, 16, alpha)
    assert 1e-6 < d4 < 1e-2 and d16 > 10 * d4
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    field = inputs.rhs_uniform((nz, ny, nx), 3)
    t = torch.from_numpy(field).cuda()
    grid.adi_sweep(0, tdx.MODE_PDD, 4, alpha, t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    r4 = orc.adi_sweep(field.copy(), *faces, BCS, 0, orc.MODE_PDD, 4, alpha)
    r16 = orc.adi_sweep(field.copy(), *faces, BCS, 0, orc.MODE_PDD, 16, alpha)
    exact = orc.adi_sweep(field.copy(), *faces, BCS, 0, orc.MODE_THOMAS, 1, alpha)
    assert relerr(out, r4) < 1e-11
    assert relerr(out, r16) > 1e-4 and relerr(out, exact) > 1e-7
    grid.close()


@pytest.mark.parametrize("direction,n,P", [(0, 512, 4), (1, 256, 2), (2, 256, 2)])
def test_long_partitions_identity_and_index_encoded_bit_exact(direction, n, P):
    (nx, ny, nz), faces = grid_for(direction, n)
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    field = np.arange(nx * ny * nz, dtype=np.float64).reshape(nz, ny, nx)
    for mode in (tdx.MODE_PPT, tdx.MODE_PDD):
        t = torch.from_numpy(field).cuda()
        grid.adi_sweep(direction, mode, P, 0.0, t)
        torch.cuda.synchronize()
        assert np.array_equal(t.cpu().numpy(), field)
    grid.close()


@pytest.mark.parametrize("P", [2, 3])
@pytest.mark.parametrize("mode_name", ["ppt", "pdd"])
def test_long_partitions_cyclic_user_coefficients(P, mode_name):
    nx, ny, nz = 8, 6, 300
    rng = np.random.default_rng(P)
    a = rng.uniform(-1, -0.1, nz); c = rng.uniform(-1, -0.1, nz); b = 2e-3 - a - c      # weakly dominant: slow spikes
    f8, f6, fz = inputs.faces_uniform(nx, 1.0), inputs.faces_uniform(ny, 1.0), inputs.faces_uniform(nz, 1.0)
    grid = tdx.Grid(nx, ny, nz, f8, f6, fz, bcs=BCS)
    field = inputs.rhs_uniform((nz, ny, nx), 5)
    t = torch.from_numpy(field).cuda()
    grid.cyclic_solve(2, MODES[mode_name], P, a, b, c, t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    if mode_name == "ppt":
        ref = orc.cyclic_solve(field.copy(), 2, orc.MODE_THOMAS, 1, a, b, c)
        assert relerr(out, ref) < 1e-10                                                 # cond(A) ~ 1e4 here
    else:
        ref = orc.cyclic_solve(field.copy(), 2, orc.MODE_PDD, P, a, b, c)
        assert orc.cyclic_pdd_dropped(P, a, b, c) > 1e-9                                # PDD really is approximate here
        assert relerr(out, ref) < 1e-10
    grid.close()


@pytest.mark.parametrize("P", [2, 4])
def test_helmholtz_shared_matrix_long_partitions(P):
    c = configs.get(2)                                           # ny = 128: 64 / 32 rows per partition
    nx, ny, nm = 32, 256, 9                                      # here: 128 / 64 rows
    yf = inputs.faces_tanh_one_sided(ny, 3.0)
    f = inputs.faces_uniform(nx, 1.0); fz = inputs.faces_uniform(16, 1.0)
    grid = tdx.Grid(nx, ny, 16, f, yf, fz, bcs=BCS)
    kz2 = inputs.modified_wavenumbers_z(16, 1.0)
    rhs = inputs.rhs_complex_uniform((nm, ny, nx), 9)
    t = torch.from_numpy(rhs).cuda()
    grid.helmholtz_wavenumber_solve(tdx.MODE_PPT, P, None, kz2, t)
    torch.cuda.synchronize()
    ref = orc.helmholtz_solve(rhs.copy(), yf, None, kz2, orc.MODE_THOMAS, 1)
    out = t.cpu().numpy()
    for m in range(nm):
        assert relerr(out[m], ref[m]) < 1e-11, (m, relerr(out[m], ref[m]))
    assert relerr(out, ref) < 1e-12
    assert np.all(out[0, 0, :] == 0.0)
    grid.close()


@pytest.mark.parametrize("P", [2, 4, 5])
def test_helmholtz_per_line_shift_ppt_long_partitions(P):
    nx, ny, nz = 32, 128, 16                                     # 64 / 32 / 26 rows per partition: more than the 16-row tile
    nm = nz // 2 + 1
    yf = inputs.faces_tanh_one_sided(ny, 3.0)
    f = inputs.faces_uniform(nx, 2.0); fz = inputs.faces_uniform(nz, 1.0)
    grid = tdx.Grid(nx, ny, nz, f, yf, fz, bcs=BCS)
    kz2 = inputs.modified_wavenumbers_z(nz, 1.0)
    kx2 = inputs.modified_wavenumbers_x(nx, 2.0)
    rhs = inputs.rhs_complex_uniform((nm, ny, nx), 11)
    t = torch.from_numpy(rhs).cuda()
    grid.helmholtz_wavenumber_solve(tdx.MODE_PPT, P, kx2, kz2, t)
    torch.cuda.synchronize()
    ref = orc.helmholtz_solve(rhs.copy(), yf, kx2, kz2, orc.MODE_THOMAS, 1)
    out = t.cpu().numpy()
    assert relerr(out, ref) < 1e-12
    assert out[0, 0, 0] == 0.0
    with pytest.raises(tdx.TdxError) as e:                      # PDD is not exact, so its partitions cannot be cut again
        grid.helmholtz_wavenumber_solve(tdx.MODE_PDD, P, kx2, kz2, t)
    assert e.value.status == tdx.ERR_UNSUPPORTED
    grid.close()


def test_per_line_helmholtz_is_stream_ordered_no_host_sync():
    """Two solves enqueued back to back on a side stream, no host synchronisation between them (the header promises
    asynchronous): the second must see the first one's result, i.e. equal solve(solve(rhs))."""
    nx, ny, nz = 64, 64, 32
    nm = nz // 2 + 1
    yf = inputs.faces_tanh_one_sided(ny, 2.0)
    grid = tdx.Grid(nx, ny, nz, inputs.faces_uniform(nx, 2.0), yf, inputs.faces_uniform(nz, 1.0), bcs=BCS)
    kz2 = inputs.modified_wavenumbers_z(nz, 1.0); kx2 = inputs.modified_wavenumbers_x(nx, 2.0)
    rhs = inputs.rhs_complex_uniform((nm, ny, nx), 21)
    st = torch.cuda.Stream()
    t = torch.from_numpy(rhs).cuda()
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        grid.helmholtz_wavenumber_solve(tdx.MODE_PPT, 8, kx2, kz2, t, st.cuda_stream)
        grid.helmholtz_wavenumber_solve(tdx.MODE_PPT, 8, kx2, kz2, t, st.cuda_stream)
    st.synchronize()
    ref = orc.helmholtz_solve(rhs.copy(), yf, kx2, kz2, orc.MODE_THOMAS, 1)
    ref = orc.helmholtz_solve(ref, yf, kx2, kz2, orc.MODE_THOMAS, 1)
    assert relerr(t.cpu().numpy(), ref) < 1e-11
    # the whole Poisson solve as well: two solves on one stream without a host sync in between
    field = inputs.rhs_uniform((nz, ny, nx), 4)
    import transforms as otr
    tf = torch.from_numpy(field).cuda()
    work = torch.empty((nm, ny, nx), dtype=torch.complex128, device="cuda")
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        grid.poisson_solve(tdx.MODE_PPT, 8, None, None, tf, work, st.cuda_stream)
        grid.poisson_solve(tdx.MODE_PPT, 8, None, None, tf, work, st.cuda_stream)
    st.synchronize()
    r1 = otr.poisson_solve(field, yf, 2.0, 1.0)
    r2 = otr.poisson_solve(r1, yf, 2.0, 1.0)
    assert relerr(tf.cpu().numpy(), r2) < 1e-10
    grid.close()


# ---------------------------------------------------------------- strict PDD (TDX_ERR_PDD_BOUND)
def test_strict_pdd_refuses_before_any_launch_and_only_pdd():
    c = configs.get(2)
    faces = c.faces()
    grid = tdx.Grid(c.nx, c.ny, c.nz, *faces, bcs=BCS)
    field = c.rhs_field()
    bound32 = grid.pdd_dropped_bound(1, 32, c.alpha)             # 4 rows per partition on the stretched y grid
    bound4 = grid.pdd_dropped_bound(1, 4, c.alpha)
    assert bound32 > 1e-11 > bound4
    grid.set_pdd_strict(1e-11)
    t = torch.from_numpy(field).cuda()
    n0 = tdx.kernel_launch_count()
    with pytest.raises(tdx.TdxError) as e:
        grid.adi_sweep(1, tdx.MODE_PDD, 32, c.alpha, t)
    assert e.value.status == tdx.ERR_PDD_BOUND and tdx.status_string(e.value.status) == "TDX_ERR_PDD_BOUND"
    assert tdx.kernel_launch_count() == n0                       # plan was cached by the bound queries: nothing launched
    torch.cuda.synchronize()
    assert np.array_equal(t.cpu().numpy(), field)                # nothing written
    with pytest.raises(tdx.TdxError) as e:
        grid.adi_step(tdx.MODE_PDD, 16, 32, 8, c.alpha, 1, None, t)
    assert e.value.status == tdx.ERR_PDD_BOUND
    torch.cuda.synchronize()
    assert np.array_equal(t.cpu().numpy(), field)                # the y plan is checked before the x sweep is launched
    assert grid.pdd_dropped_bound(1, 32, c.alpha) == bound32     # the diagnostic itself is never refused
    grid.adi_sweep(1, tdx.MODE_PDD, 4, c.alpha, t)               # inside the bound: runs
    grid.adi_sweep(1, tdx.MODE_PPT, 32, c.alpha, t)              # PPT is exact: never refused
    grid.adi_sweep(1, tdx.MODE_THOMAS, 32, c.alpha, t)
    # Helmholtz PDD is the paper's counter-example (L172): refused under the strict flag
    h = torch.from_numpy(c.rhs_helmholtz()).cuda()
    with pytest.raises(tdx.TdxError) as e:
        grid.helmholtz_wavenumber_solve(tdx.MODE_PDD, 8, None, c.kz2(), h)
    assert e.value.status == tdx.ERR_PDD_BOUND
    kx2 = inputs.modified_wavenumbers_x(c.nx, c.lx)
    with pytest.raises(tdx.TdxError) as e:
        grid.helmholtz_wavenumber_solve(tdx.MODE_PDD, 8, kx2, c.kz2(), h)
    assert e.value.status == tdx.ERR_PDD_BOUND
    grid.set_pdd_strict(0.0)                                     # off again: runs as asked
    grid.adi_sweep(1, tdx.MODE_PDD, 32, c.alpha, t)
    torch.cuda.synchronize()
    with pytest.raises(tdx.TdxError) as e:
        grid.set_pdd_strict(-1.0)
    assert e.value.status == tdx.ERR_INVALID_ARG
    grid.close()
