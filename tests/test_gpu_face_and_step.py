"""GPU parity for the face-located ADI operator (tdx_adi_sweep_at) and the multi-component ADI step (tdx_adi_step),
SURVEY 8(f) N1, against the oracle on the same seeded inputs.  Tolerances as in test_gpu_parity.py."""
import numpy as np
import pytest
import torch

import oracle as orc
from paper_1812_01178_b200 import binding as tdx
from paper_1812_01178_b200 import configs, inputs

pytestmark = pytest.mark.gpu

BCS = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
MODES = {"thomas": (tdx.MODE_THOMAS, orc.MODE_THOMAS), "pdd": (tdx.MODE_PDD, orc.MODE_PDD), "ppt": (tdx.MODE_PPT, orc.MODE_PPT)}
STAGGERED = [[1, 0, 0], [0, 1, 0], [0, 0, 1]]                    # u: face in x, v: face in y, w: face in z


def relerr(x, ref):
    return float(np.max(np.abs(x - ref)) / np.max(np.abs(ref)))


@pytest.fixture(scope="module")
def cfg1():
    c = configs.get(1)
    faces = c.faces()
    grid = tdx.Grid(c.nx, c.ny, c.nz, *faces, bcs=BCS)
    yield c, faces, grid, c.rhs_field()
    grid.close()


@pytest.mark.parametrize("direction", [0, 1, 2])
@pytest.mark.parametrize("mode_name", ["thomas", "pdd", "ppt"])
@pytest.mark.parametrize("alpha", [5e-7, 1e-2])
def test_face_sweep_every_element(cfg1, direction, mode_name, alpha):
    c, faces, grid, field = cfg1
    gm, om = MODES[mode_name]
    t = torch.from_numpy(field).cuda()
    grid.adi_sweep_at(direction, tdx.LOC_FACE, gm, 4, alpha, t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    exact = orc.adi_sweep_at(field.copy(), *faces, BCS, direction, 1, orc.MODE_THOMAS, 1, alpha)
    if mode_name == "pdd":
        ref_pdd = orc.adi_sweep_at(field.copy(), *faces, BCS, direction, 1, orc.MODE_PDD, 4, alpha)
        assert relerr(out, ref_pdd) < 1e-12
    else:
        assert relerr(out, exact) < 1e-12, (direction, mode_name, relerr(out, exact))
    if BCS[direction] == tdx.BC_DIRICHLET:                       # wall face: identity row, right-hand side passes through
        wall = {0: out[:, :, -1] == field[:, :, -1], 1: out[:, -1, :] == field[:, -1, :]}[direction]
        assert np.all(wall)


def test_face_center_is_plain_sweep_bit_exact(cfg1):
    c, faces, grid, field = cfg1
    for direction in range(3):
        a = torch.from_numpy(field).cuda(); b = torch.from_numpy(field).cuda()
        grid.adi_sweep_at(direction, tdx.LOC_CENTER, tdx.MODE_PPT, 4, c.alpha, a)
        grid.adi_sweep(direction, tdx.MODE_PPT, 4, c.alpha, b)
        torch.cuda.synchronize()
        assert torch.equal(a, b)


@pytest.mark.parametrize("mode_name", ["ppt", "pdd"])
def test_ragged_stretched_face_sweeps(mode_name):
    nx, ny, nz = 50, 37, 29
    faces = (inputs.faces_tanh_two_sided(nx, 1.2, 2.0), inputs.faces_tanh_one_sided(ny, 2.5), inputs.faces_uniform(nz, 1.0))
    grid = tdx.Grid(nx, ny, nz, *faces, bcs=BCS)
    field = inputs.rhs_gaussian((nz, ny, nx), 78)
    gm, om = MODES[mode_name]
    for direction in range(3):
        for P in (3, 5):
            t = torch.from_numpy(field).cuda()
            grid.adi_sweep_at(direction, tdx.LOC_FACE, gm, P, 3e-4, t)
            torch.cuda.synchronize()
            ref = orc.adi_sweep_at(field.copy(), *faces, BCS, direction, 1, om, P, 3e-4)
            assert relerr(t.cpu().numpy(), ref) < 1e-12, (direction, P)
    grid.close()


@pytest.mark.parametrize("cfg_no,P", [(1, (4, 4, 4)), (2, (16, 8, 8))])
def test_adi_step_three_staggered_components(cfg_no, P):
    c = configs.get(cfg_no)
    faces = c.faces()
    grid = tdx.Grid(c.nx, c.ny, c.nz, *faces, bcs=BCS)
    comps = np.stack([inputs.rhs_uniform((c.nz, c.ny, c.nx), 300 + k) for k in range(3)])
    t = torch.from_numpy(comps).cuda()
    n0 = tdx.kernel_launch_count()
    grid.adi_step(tdx.MODE_PPT, P[0], P[1], P[2], c.alpha, 3, STAGGERED, t)
    torch.cuda.synchronize()
    out = t.cpu().numpy()
    for k in range(3):
        ref = comps[k].copy()
        for d in range(3):
            orc.adi_sweep_at(ref, *faces, BCS, d, STAGGERED[k][d], orc.MODE_THOMAS, 1, c.alpha)
        assert relerr(out[k], ref) < 1e-12, (k, relerr(out[k], ref))
    # all centres: one launch per direction, bit-identical to three separate sweeps per component
    t2 = torch.from_numpy(comps).cuda(); t3 = torch.from_numpy(comps).cuda()
    n1 = tdx.kernel_launch_count()
    grid.adi_step(tdx.MODE_PPT, P[0], P[1], P[2], c.alpha, 3, None, t2)
    assert tdx.kernel_launch_count() - n1 == 3
    for d in range(3):
        for k in range(3):
            grid.adi_sweep(d, tdx.MODE_PPT, P[d], c.alpha, t3[k])
    torch.cuda.synchronize()
    assert torch.equal(t2, t3)
    grid.close()


def test_face_and_step_error_paths():
    nx, ny, nz = 16, 16, 16
    f = inputs.faces_uniform(16, 1.0)
    grid = tdx.Grid(nx, ny, nz, f, f, f, bcs=(tdx.BC_NEUMANN, tdx.BC_DIRICHLET, tdx.BC_PERIODIC))
    t = torch.ones((3, nz, ny, nx), dtype=torch.float64, device="cuda")
    before = t.clone()
    with pytest.raises(tdx.TdxError) as e:
        grid.adi_sweep_at(0, tdx.LOC_FACE, tdx.MODE_PPT, 4, 1e-3, t)          # Neumann ends: face unknowns undefined
    assert e.value.status == tdx.ERR_UNSUPPORTED
    with pytest.raises(tdx.TdxError) as e:
        grid.adi_sweep_at(1, 7, tdx.MODE_PPT, 4, 1e-3, t)
    assert e.value.status == tdx.ERR_INVALID_ARG
    with pytest.raises(tdx.TdxError) as e:
        grid.adi_step(tdx.MODE_PPT, 4, 4, 99, 1e-3, 3, None, t)                # bad Pz: nothing may have been launched
    assert e.value.status == tdx.ERR_BAD_PARTITION
    with pytest.raises(tdx.TdxError):
        grid.adi_step(tdx.MODE_PPT, 4, 4, 4, 1e-3, 0, None, t)
    torch.cuda.synchronize()
    assert torch.equal(t, before)
    grid.close()
