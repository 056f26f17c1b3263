"""GPU: bit-exact layout / partition indexing, error paths of the C ABI, cyclic_solve, host entry points."""
import numpy as np
import pytest
import torch

import oracle as orc
from paper_1812_01178_b200 import binding as tdx
from paper_1812_01178_b200 import inputs

pytestmark = pytest.mark.gpu
BCS = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)


def relerr(x, ref):
    return float(np.max(np.abs(x - ref)) / np.max(np.abs(ref)))


@pytest.fixture(scope="module")
def small():
    nx, ny, nz = 64, 36, 30
    faces = (inputs.faces_uniform(nx, 2.0), inputs.faces_tanh_two_sided(ny, 2.0), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    yield (nx, ny, nz), faces, grid
    grid.close()


@pytest.mark.parametrize("direction", [0, 1, 2])
@pytest.mark.parametrize("mode", [tdx.MODE_THOMAS, tdx.MODE_PDD, tdx.MODE_PPT])
@pytest.mark.parametrize("P", [2, 3, 4, 6])
def test_identity_operator_index_encoded_rhs_bit_exact(small, direction, mode, P):
    """alpha = 0: (I - 0*delta2) x = d must return d bit for bit; d = linear index exposes any layout slip."""
    (nx, ny, nz), _, grid = small
    field = np.arange(nx * ny * nz, dtype=np.float64).reshape(nz, ny, nx) + 0.25
    t = torch.from_numpy(field).cuda()
    grid.adi_sweep(direction, mode, P, 0.0, t)
    torch.cuda.synchronize()
    assert np.array_equal(t.cpu().numpy(), field)


@pytest.mark.parametrize("direction", [0, 1, 2])
@pytest.mark.parametrize("mode", [tdx.MODE_THOMAS, tdx.MODE_PDD, tdx.MODE_PPT])
def test_one_hot_changes_only_its_line(small, direction, mode):
    (nx, ny, nz), faces, grid = small
    field = np.zeros((nz, ny, nx)); field[7, 11, 13] = 1.0
    t = torch.from_numpy(field).cuda()
    grid.adi_sweep(direction, mode, 3, 0.02, t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    mask = np.zeros_like(out, dtype=bool)
    if direction == 0: mask[7, 11, :] = True
    if direction == 1: mask[7, :, 13] = True
    if direction == 2: mask[:, 11, 13] = True
    assert np.all(out[~mask] == 0.0) and np.count_nonzero(out[mask]) > 3
    ref = orc.adi_sweep(field.copy(), *faces, BCS, direction, orc.MODE_THOMAS, 1, 0.02)
    if mode != tdx.MODE_PDD:
        assert relerr(out, ref) < 1e-12


def test_error_paths_leave_data_untouched(small):
    (nx, ny, nz), _, grid = small
    field = inputs.rhs_uniform((nz, ny, nx), 1)
    t = torch.from_numpy(field).cuda()
    with pytest.raises(tdx.TdxError) as e:
        grid.adi_sweep(1, tdx.MODE_PPT, 30, 1e-3, t)             # floor(36/30) < 2
    assert e.value.status == tdx.ERR_BAD_PARTITION
    with pytest.raises(tdx.TdxError) as e:
        grid.adi_sweep(0, tdx.MODE_PPT, 0, 1e-3, t)
    assert e.value.status == tdx.ERR_BAD_PARTITION
    with pytest.raises(tdx.TdxError) as e:
        grid.adi_sweep(5, tdx.MODE_PPT, 2, 1e-3, t)
    assert e.value.status == tdx.ERR_INVALID_ARG
    with pytest.raises(tdx.TdxError) as e:
        grid.adi_sweep(0, 7, 2, 1e-3, t)
    assert e.value.status == tdx.ERR_INVALID_ARG
    with pytest.raises(tdx.TdxError) as e:
        grid.adi_sweep(0, tdx.MODE_PPT, 2, 1e-3, 0)              # NULL data pointer
    assert e.value.status == tdx.ERR_INVALID_ARG
    with pytest.raises(tdx.TdxError) as e:
        grid.helmholtz_wavenumber_solve(tdx.MODE_PDD, 2, np.ones(nx), np.ones(3), t)   # per-line shifts, PDD: 18 rows per partition > 16
    assert e.value.status == tdx.ERR_UNSUPPORTED
    torch.cuda.synchronize()
    assert np.array_equal(t.cpu().numpy(), field)


def test_rows_per_partition_has_no_limit():
    """Round 1 refused more than 64 rows per partition; SURVEY 8(b) asks only 1 <= P, floor(n/P) >= 2."""
    nx = 400
    f = inputs.faces_uniform(nx, 1.0); g8 = inputs.faces_uniform(8, 1.0)
    grid = tdx.Grid(nx, 8, 8, f, g8, g8, bcs=BCS)
    field = inputs.rhs_uniform((8, 8, nx), 2)
    ref = orc.adi_sweep(field.copy(), f, g8, g8, BCS, 0, orc.MODE_THOMAS, 1, 1e-5)
    for mode in (tdx.MODE_PPT, tdx.MODE_THOMAS):
        t = torch.from_numpy(field).cuda()
        grid.adi_sweep(0, mode, 4, 1e-5, t)                      # 100 rows per partition
        torch.cuda.synchronize()
        assert np.max(np.abs(t.cpu().numpy() - ref)) / np.max(np.abs(ref)) < 1e-12
    grid.close()


@pytest.mark.parametrize("direction", [0, 1, 2])
@pytest.mark.parametrize("mode,P", [(tdx.MODE_THOMAS, 1), (tdx.MODE_PPT, 3), (tdx.MODE_PDD, 2), (tdx.MODE_PPT, 5), (tdx.MODE_PDD, 5)])
def test_cyclic_solve_user_coefficients(small, direction, mode, P):
    (nx, ny, nz), _, grid = small
    n = (nx, ny, nz)[direction]
    rng = np.random.default_rng(direction * 10 + P)
    a = rng.uniform(-1, -0.1, n); c = rng.uniform(-1, -0.1, n); b = 2.5 - a - c
    field = inputs.rhs_uniform((nz, ny, nx), 5)
    t = torch.from_numpy(field).cuda()
    grid.cyclic_solve(direction, mode, P, a, b, c, t)
    torch.cuda.synchronize()
    ref = orc.cyclic_solve(field.copy(), direction, orc.MODE_THOMAS, 1, a, b, c)
    tol = 1e-12
    if mode == tdx.MODE_PDD:                                 # P interfaces closed cyclically; approximate to O(dropped)
        ref_pdd = orc.cyclic_solve(field.copy(), direction, orc.MODE_PDD, P, a, b, c)
        assert relerr(t.cpu().numpy(), ref_pdd) < 1e-12
        tol = 1e-10 + 50 * orc.cyclic_pdd_dropped(P, a, b, c)
        assert tol < 1e-2                                    # the case must still tell a right answer from a wrong one
    assert relerr(t.cpu().numpy(), ref) < tol


def test_host_entry_points(small):
    (nx, ny, nz), faces, grid = small
    alpha = 1e-3
    field = inputs.rhs_uniform((nz, ny, nx), 8)
    ref = field.copy()
    for d in range(3):
        orc.adi_sweep(ref, *faces, BCS, d, orc.MODE_THOMAS, 1, alpha)
    h = field.copy()
    grid.adi_step_host(tdx.MODE_PPT, 4, 3, 3, alpha, h)
    assert relerr(h, ref) < 1e-12
    h = field.copy()
    grid.adi_sweep_host(1, tdx.MODE_PPT, 3, alpha, h)
    assert relerr(h, orc.adi_sweep(field.copy(), *faces, BCS, 1, orc.MODE_THOMAS, 1, alpha)) < 1e-12
    nm = nz // 2 + 1
    kz2 = inputs.modified_wavenumbers_z(nz)
    rhs = inputs.rhs_complex_uniform((nm, ny, nx), 4)
    hc = rhs.copy()
    grid.helmholtz_wavenumber_solve_host(tdx.MODE_PPT, 4, None, kz2, hc)
    assert relerr(hc, orc.helmholtz_solve(rhs.copy(), faces[1], None, kz2, orc.MODE_THOMAS, 1)) < 1e-12


def test_kernel_launch_counter_counts_this_librarys_kernels(small):
    (nx, ny, nz), _, grid = small
    t = torch.zeros(nx * ny * nz, dtype=torch.float64, device="cuda")
    grid.adi_sweep(1, tdx.MODE_PPT, 3, 1e-3, t)                  # plan cached after this
    n0 = tdx.kernel_launch_count()
    for _ in range(5):
        grid.adi_sweep(1, tdx.MODE_PPT, 3, 1e-3, t)
    assert tdx.kernel_launch_count() - n0 == 5                   # one launch per sweep


def test_pipelined_step_host_equals_device_path_bit_exact():
    """tdx_step_host (slabs over three streams, sub-range launches) must give exactly what the whole-field device calls give."""
    nx, ny, nz = 96, 40, 36
    faces = (inputs.faces_uniform(nx, 2.0), inputs.faces_tanh_two_sided(ny, 2.0), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    field = inputs.rhs_uniform((nz, ny, nx), 41)
    nm = nz // 2 + 1
    helm = inputs.rhs_complex_uniform((nm, ny, nx), 42)
    kz2 = inputs.modified_wavenumbers_z(nz, 1.0)
    alpha = 3e-4
    for mode in (tdx.MODE_PPT, tdx.MODE_PDD, tdx.MODE_THOMAS):
        t = torch.from_numpy(field).cuda(); th = torch.from_numpy(helm).cuda()
        for d, P in ((0, 6), (1, 5), (2, 4)):
            grid.adi_sweep(d, mode, P, alpha, t)
        grid.helmholtz_wavenumber_solve(mode, 4, None, kz2, th)
        torch.cuda.synchronize()
        hf = torch.from_numpy(field.copy()).pin_memory().numpy()
        hh = torch.from_numpy(helm.copy()).pin_memory().numpy()
        grid.step_host(mode, 6, 5, 4, alpha, hf, 4, kz2, hh)
        assert np.array_equal(hf, t.cpu().numpy())
        assert np.array_equal(hh, th.cpu().numpy())
        hf2 = field.copy()                                       # pageable memory and one part only
        grid.step_host(mode, 6, 5, 4, alpha, hf2, 4, None, None)
        assert np.array_equal(hf2, hf)
    with pytest.raises(tdx.TdxError):
        grid.step_host(tdx.MODE_PPT, 6, 5, 999, alpha, hf, 4, kz2, hh)
    grid.close()


def test_step_is_capturable_in_a_cuda_graph_and_replays_bit_exact():
    """Once their plans exist the sweeps are plain stream work (no allocation, no synchronisation): x, y, cyclic z and the
    Helmholtz solve are captured in one CUDA graph on a side stream and the replay gives the bits of the eager calls --
    on new data written into the captured buffers.  Small grids are launch-bound (cfg1: 7 us per sweep); this is how a
    caller removes the launch overhead."""
    nx, ny, nz = 64, 32, 32
    faces = (inputs.faces_uniform(nx, 2.0), inputs.faces_tanh_two_sided(ny, 2.0), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    nm = nz // 2 + 1
    kz2 = inputs.modified_wavenumbers_z(nz, 1.0)
    alpha = 5e-7

    def step(t, th, st):
        for d in range(3):
            grid.adi_sweep(d, tdx.MODE_PPT, 4, alpha, t, st)
        grid.helmholtz_wavenumber_solve(tdx.MODE_PPT, 4, None, kz2, th, st)

    f1, f2 = inputs.rhs_uniform((nz, ny, nx), 1), inputs.rhs_uniform((nz, ny, nx), 2)
    h1, h2 = inputs.rhs_complex_uniform((nm, ny, nx), 3), inputs.rhs_complex_uniform((nm, ny, nx), 4)
    want = []
    for f, h in ((f1, h1), (f2, h2)):                            # eager, default stream: builds the plans too
        t, th = torch.from_numpy(f).cuda(), torch.from_numpy(h).cuda()
        step(t, th, 0)
        torch.cuda.synchronize()
        want.append((t.clone(), th.clone()))
    buf, bufh = torch.from_numpy(f1).cuda(), torch.from_numpy(h1).cuda()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        scratch, scratchh = buf.clone(), bufh.clone()
        step(scratch, scratchh, side.cuda_stream)                # once on this stream outside capture
        side.synchronize()
        n0 = tdx.kernel_launch_count()
        cg = torch.cuda.CUDAGraph()
        with torch.cuda.graph(cg, stream=side):
            step(buf, bufh, side.cuda_stream)
        assert tdx.kernel_launch_count() - n0 == 4               # four kernels recorded, none run yet
    torch.cuda.synchronize()
    assert torch.equal(buf.cpu(), torch.from_numpy(f1))           # capture does not execute
    cg.replay()
    torch.cuda.synchronize()
    assert torch.equal(buf, want[0][0]) and torch.equal(bufh, want[0][1])
    buf.copy_(torch.from_numpy(f2)); bufh.copy_(torch.from_numpy(h2))
    cg.replay()
    torch.cuda.synchronize()
    assert torch.equal(buf, want[1][0]) and torch.equal(bufh, want[1][1])
    del cg
    grid.close()


def test_two_steps_in_flight_equal_the_synchronous_step_bit_exact():
    """tdx_step_host_async: two steps in flight on two slots (different data), then a third on the first slot again, give
    exactly what tdx_step_host gives one at a time; a busy slot is refused; the other host entry points wait for slot 0."""
    nx, ny, nz = 96, 40, 36
    faces = (inputs.faces_uniform(nx, 2.0), inputs.faces_tanh_two_sided(ny, 2.0), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    nm = nz // 2 + 1
    kz2 = inputs.modified_wavenumbers_z(nz, 1.0)
    alpha = 3e-4
    args = (tdx.MODE_PPT, 6, 5, 4, alpha)
    fields = [inputs.rhs_uniform((nz, ny, nx), 50 + k) for k in range(3)]
    helms = [inputs.rhs_complex_uniform((nm, ny, nx), 60 + k) for k in range(3)]
    want = []
    for f, h in zip(fields, helms):
        hf = torch.from_numpy(f.copy()).pin_memory().numpy(); hh = torch.from_numpy(h.copy()).pin_memory().numpy()
        grid.step_host(*args, hf, 4, kz2, hh)
        want.append((hf.copy(), hh.copy()))
    bufs = [(torch.from_numpy(f.copy()).pin_memory().numpy(), torch.from_numpy(h.copy()).pin_memory().numpy()) for f, h in zip(fields, helms)]
    grid.step_host_async(0, *args, bufs[0][0], 4, kz2, bufs[0][1])
    grid.step_host_async(1, *args, bufs[1][0], 4, kz2, bufs[1][1])
    with pytest.raises(tdx.TdxError) as e:                       # slot 1 holds a step
        grid.step_host_async(1, *args, bufs[2][0], 4, kz2, bufs[2][1])
    assert e.value.status == tdx.ERR_INVALID_ARG
    grid.step_host_wait(0)
    grid.step_host_async(0, *args, bufs[2][0], 4, kz2, bufs[2][1])    # slot 0 again while slot 1 is still out
    grid.step_host_wait(1)
    grid.step_host_wait(0)
    grid.step_host_wait(0)                                       # an idle slot: nothing to wait for
    for k in range(3):
        assert np.array_equal(bufs[k][0], want[k][0]), k
        assert np.array_equal(bufs[k][1], want[k][1]), k
    # a step in flight in slot 0, then a synchronous host call that shares its staging: it must wait, both must be right
    b0 = (torch.from_numpy(fields[0].copy()).pin_memory().numpy(), torch.from_numpy(helms[0].copy()).pin_memory().numpy())
    grid.step_host_async(0, *args, b0[0], 4, kz2, b0[1])
    other = fields[1].copy()
    grid.adi_step_host(tdx.MODE_PPT, 6, 5, 4, alpha, other)
    grid.step_host_wait(0)
    assert np.array_equal(b0[0], want[0][0]) and np.array_equal(b0[1], want[0][1])
    assert np.array_equal(other, want[1][0])
    with pytest.raises(tdx.TdxError):
        grid.step_host_wait(2)
    grid.step_host_async(1, *args, b0[0], 4, kz2, b0[1])         # destroyed with a step in flight: must not crash or leak
    grid.close()


def test_plan_cache_is_bounded_and_rebuilds_evicted_plans(small):
    """A caller that keeps changing alpha (variable time step) must not grow the plan cache without bound, and a plan
    that was dropped is rebuilt to the same bits."""
    (nx, ny, nz), faces, grid = small
    field = inputs.rhs_uniform((nz, ny, nx), 77)
    t = torch.from_numpy(field).cuda()
    grid.adi_sweep(1, tdx.MODE_PPT, 4, 1e-3, t)
    torch.cuda.synchronize()
    first = t.clone()
    free0 = torch.cuda.mem_get_info()[0]
    for k in range(200):
        s = torch.from_numpy(field).cuda()
        grid.adi_sweep(1, tdx.MODE_PPT, 4, 1e-3 * (1.0 + 1e-3 * (k + 1)), s)
    torch.cuda.synchronize()
    t2 = torch.from_numpy(field).cuda()
    grid.adi_sweep(1, tdx.MODE_PPT, 4, 1e-3, t2)                 # evicted by now: rebuilt
    torch.cuda.synchronize()
    assert torch.equal(t2, first)
    assert free0 - torch.cuda.mem_get_info()[0] < 64 * 1024 * 1024   # 200 plans of this grid would be far below this anyway; no leak growth


@pytest.mark.parametrize("L,uniform_table", [(3.8, True), (2.1, False)])
@pytest.mark.parametrize("mode", [tdx.MODE_PPT, tdx.MODE_PDD])
def test_uniform_table_switch_at_its_1e_13_boundary(L, uniform_table, mode):
    """A product approximation that is not in the paper: when the partitions' ADI blocks agree row-wise to 1e-13 (uniform
    spacing that is not a binary fraction: the faces L j / N differ by rounding), every block is replaced by one table
    (k_blocks_identical; ||A^-1|| <= 1 for rows with |b| = |a| + |c| + 1, bounds the change by 1e-13).
    Two grids on either side of the switch -- 48 uniform cells, P = 3, alpha = 1e-2 (alpha / h^2 = 1.6 and 5.2: coupled
    partitions): L = 3.8, blocks differ by 0.47e-13 -> one table; L = 2.1, 2.1e-13 -> per-partition tables.  Both must
    meet the 1e-12 gate against the oracle, which always uses the true coefficients."""
    nx, ny, nz, P, alpha = 48, 6, 48, 3, 1e-2
    faces = (inputs.faces_uniform(nx, L), inputs.faces_uniform(ny, 1.0), inputs.faces_uniform(nz, L))
    a, b, c = orc.adi_coeffs(faces[0], orc.BC_DIRICHLET, alpha)
    m = nx // P
    diff = max(abs(b[p * m + jj] - b[jj]) + (abs(a[p * m + jj] - a[jj]) if jj else 0.0) + (abs(c[p * m + jj] - c[jj]) if jj < m - 1 else 0.0)
               for p in range(1, P) for jj in range(m))
    assert (0 < diff < 0.9e-13) if uniform_table else (1.1e-13 < diff < 5e-13)      # the inputs sit where the docstring says
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    field = inputs.rhs_uniform((nz, ny, nx), 8)
    for direction in (0, 2):                                     # x: the TMA kernel; z (periodic): the strided kernel
        t = torch.from_numpy(field).cuda()
        grid.adi_sweep(direction, mode, P, alpha, t)
        torch.cuda.synchronize()
        launch = tdx.last_launch()
        uni = launch.split("<")[1].split(">")[0].split(",")[1 if direction == 0 else 3]
        assert uni == ("1" if uniform_table else "0"), launch
        ref = orc.adi_sweep(field.copy(), *faces, BCS, direction, orc.MODE_THOMAS if mode == tdx.MODE_PPT else orc.MODE_PDD, P, alpha)
        assert relerr(t.cpu().numpy(), ref) < 1e-12, (direction, launch, relerr(t.cpu().numpy(), ref))
    grid.close()
