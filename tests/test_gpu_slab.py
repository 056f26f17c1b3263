"""GPU parity of the slab decomposition (Algorithm 1, L156/L174): every rank is one partition
of PDD / PPT along y (or z).  The box has one GPU, so the ranks' slabs live side by side on it and the phases run one
after the other (all eliminations, then the exchange as tensor copies -- exactly the planes parallel.exchange_* move
between processes, whose pattern tests/test_slab_exchange_gloo.py checks over gloo -- then all corrections); no kernel
waits on another rank.  Compared element by element with the oracle's global sweep."""
import numpy as np
import pytest
import torch

import oracle as orc
from paper_1812_01178_b200 import binding as tdx
from paper_1812_01178_b200 import inputs, parallel

pytestmark = pytest.mark.gpu


def relerr(x, ref):
    return float(np.max(np.abs(x - ref)) / np.max(np.abs(ref)))


def run_slabs(field, faces, bcs, direction, R, alpha, across, local_mode, P_local):
    nz, ny, nx = field.shape
    n = (nx, ny, nz)[direction]
    bounds = parallel.slab_bounds(n, R)
    grids, slabs, parts, ifaces = [], [], [], []
    for r, (s0, s1) in enumerate(bounds):
        f = list(faces)
        f[direction] = faces[direction][s0:s1 + 1]
        dims = [nx, ny, nz]; dims[direction] = s1 - s0
        g = tdx.Grid(dims[0], dims[1], dims[2], *f, bcs=bcs)
        grids.append(g)
        slabs.append(tdx.Slab(g, direction, r, R, faces[direction], bcs[direction], alpha, across, local_mode, P_local))
        sl = field[:, s0:s1, :] if direction == 1 else field[s0:s1]
        parts.append(torch.from_numpy(np.ascontiguousarray(sl)).cuda())
        plane = nx * nz if direction == 1 else nx * ny
        ifaces.append(torch.full((2, plane), float("nan"), dtype=torch.float64, device="cuda"))
    for r in range(R):
        slabs[r].eliminate(parts[r], ifaces[r])
    torch.cuda.synchronize()
    if across == tdx.MODE_PPT:
        nbrs = [torch.stack(ifaces)] * R                         # what the all-gather delivers
    else:
        nbrs = []
        for r in range(R):                                       # what the neighbour send/recv delivers
            nb = torch.full_like(ifaces[r], float("nan"))        # a missing neighbour's plane must never be read
            if r >= 1: nb[0] = ifaces[r - 1][1]
            if r <= R - 2: nb[1] = ifaces[r + 1][0]
            nbrs.append(nb)
    for r in range(R):
        slabs[r].correct(parts[r], ifaces[r], nbrs[r] if R > 1 else None)
    torch.cuda.synchronize()
    out = torch.cat(parts, dim=1 if direction == 1 else 0).cpu().numpy()
    drop = max(s.dropped_bound() for s in slabs)
    for s in slabs: s.close()
    for g in grids: g.close()
    return out, drop


@pytest.mark.parametrize("R", [1, 2, 3, 4, 8])
@pytest.mark.parametrize("local", [(tdx.MODE_THOMAS, 1), (tdx.MODE_PPT, 2)])
def test_y_slabs_ppt_across_ranks_is_exact(R, local):
    nx, ny, nz = 64, 70, 12                                      # 70 rows: ragged slabs for R = 3, 4, 8
    faces = (inputs.faces_uniform(nx, 2.0), inputs.faces_tanh_one_sided(ny, 2.5), inputs.faces_uniform(nz, 1.0))
    bcs = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
    field = inputs.rhs_uniform((nz, ny, nx), 900 + R)
    alpha = 3e-3                                                 # strong coupling: spikes do not decay across a slab
    out, drop = run_slabs(field, faces, bcs, 1, R, alpha, tdx.MODE_PPT, local[0], local[1])
    ref = orc.adi_sweep(field.copy(), *faces, bcs, 1, orc.MODE_THOMAS, 1, alpha)
    assert relerr(out, ref) < 1e-12, (relerr(out, ref), drop)
    if R >= 3:
        assert drop > 1e-6                                       # ... so PDD would not do here (next test)


@pytest.mark.parametrize("R", [2, 4, 5])
def test_y_slabs_pdd_across_ranks_equals_oracle_pdd(R):
    nx, ny, nz = 64, 70, 12
    faces = (inputs.faces_uniform(nx, 2.0), inputs.faces_tanh_one_sided(ny, 2.5), inputs.faces_uniform(nz, 1.0))
    bcs = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
    field = inputs.rhs_uniform((nz, ny, nx), 950 + R)
    for alpha in (3e-3, 1e-6):
        out, drop = run_slabs(field, faces, bcs, 1, R, alpha, tdx.MODE_PDD, tdx.MODE_THOMAS, 1)
        pdd = orc.adi_sweep(field.copy(), *faces, bcs, 1, orc.MODE_PDD, R, alpha)        # the oracle's step-by-step PDD, P = R
        exact = orc.adi_sweep(field.copy(), *faces, bcs, 1, orc.MODE_THOMAS, 1, alpha)
        assert relerr(out, pdd) < 1e-12, (alpha, relerr(out, pdd))
        if R == 2:
            assert relerr(out, exact) < 1e-12                    # one interface: nothing is dropped
        elif drop <= 1e-11:
            assert relerr(out, exact) < 1e-10                    # north_star's PDD gate where the spikes have decayed
        else:
            assert relerr(out, exact) < 100 * drop               # and bounded by what was dropped elsewhere (reading A9)


def test_z_slabs_and_neumann_ends():
    nx, ny, nz = 32, 10, 48
    faces = (inputs.faces_uniform(nx, 1.0), inputs.faces_tanh_two_sided(ny, 2.0), inputs.faces_tanh_two_sided(nz, 1.5))
    bcs = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_NEUMANN)
    field = inputs.rhs_uniform((nz, ny, nx), 990)
    alpha = 2e-3
    ref = orc.adi_sweep(field.copy(), *faces, bcs, 2, orc.MODE_THOMAS, 1, alpha)
    out, _ = run_slabs(field, faces, bcs, 2, 3, alpha, tdx.MODE_PPT, tdx.MODE_PPT, 4)
    assert relerr(out, ref) < 1e-12


def test_cfg2_y_slabs_4_ranks_local_ppt():
    """Config 2 (256x128x128), 4 ranks of 32 rows, local PPT with 4 partitions of 8 rows (the x-TMA / strided kernels)."""
    from paper_1812_01178_b200 import configs
    c = configs.get(2)
    faces = c.faces()
    bcs = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
    field = c.rhs_field()
    ref = orc.adi_sweep(field.copy(), *faces, bcs, 1, orc.MODE_THOMAS, 1, c.alpha)
    for across in (tdx.MODE_PPT, tdx.MODE_PDD):
        out, drop = run_slabs(field, faces, bcs, 1, 4, c.alpha, across, tdx.MODE_PPT, 4)
        tol = 1e-12 if across == tdx.MODE_PPT or drop <= 1e-14 else (1e-10 if drop <= 1e-11 else 100 * drop)
        assert relerr(out, ref) < tol, (across, relerr(out, ref), drop)


def test_slab_error_paths():
    nx, ny, nz = 16, 20, 8
    faces = (inputs.faces_uniform(nx, 1.0), inputs.faces_tanh_one_sided(ny, 2.0), inputs.faces_uniform(nz, 1.0))
    bcs = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
    g = tdx.Grid(nx, 10, nz, faces[0], faces[1][:11], faces[2], bcs=bcs)
    with pytest.raises(tdx.TdxError) as e:                       # x slabs are not offered
        tdx.Slab(g, 0, 0, 2, faces[0], tdx.BC_DIRICHLET, 1e-3, tdx.MODE_PPT, tdx.MODE_THOMAS, 1)
    assert e.value.status == tdx.ERR_UNSUPPORTED
    with pytest.raises(tdx.TdxError) as e:                       # periodic slab direction
        tdx.Slab(g, 1, 0, 2, faces[1], tdx.BC_PERIODIC, 1e-3, tdx.MODE_PPT, tdx.MODE_THOMAS, 1)
    assert e.value.status == tdx.ERR_UNSUPPORTED
    with pytest.raises(tdx.TdxError) as e:                       # 20 rows over 3 ranks: this grid's 10 rows are nobody's share
        tdx.Slab(g, 1, 0, 3, faces[1], tdx.BC_DIRICHLET, 1e-3, tdx.MODE_PPT, tdx.MODE_THOMAS, 1)
    assert e.value.status == tdx.ERR_INVALID_ARG
    with pytest.raises(tdx.TdxError) as e:                       # Thomas is not an across-rank mode
        tdx.Slab(g, 1, 0, 2, faces[1], tdx.BC_DIRICHLET, 1e-3, tdx.MODE_THOMAS, tdx.MODE_THOMAS, 1)
    assert e.value.status == tdx.ERR_INVALID_ARG
    s = tdx.Slab(g, 1, 1, 2, faces[1], tdx.BC_DIRICHLET, 1e-3, tdx.MODE_PDD, tdx.MODE_THOMAS, 1)
    s.close()
    g.close()
