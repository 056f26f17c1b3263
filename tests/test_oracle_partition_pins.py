"""Pins for the oracle's PDD / PPT statement and its 3-D sweeps.  CPU only.
The printed matrices at PAPER.md:L116 / L136 come from tests/golden/Z_n12_p4.txt."""
import os
import re

import numpy as np
import pytest
import scipy.linalg

import oracle as orc
from paper_1812_01178_b200 import configs, inputs

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
rng = np.random.default_rng(4321)


def relerr(x, ref):
    return np.max(np.abs(x - ref)) / np.max(np.abs(ref))


def random_dominant(n, margin=0.5):
    a = rng.uniform(-1, 1, n); c = rng.uniform(-1, 1, n)
    b = (np.abs(a) + np.abs(c) + margin) * rng.choice([-1.0, 1.0], n)
    a[0] = 0.0; c[-1] = 0.0
    return a, b, c


def parse_golden(section):
    rows, on = [], False
    for line in open(os.path.join(GOLD, "Z_n12_p4.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("["):
            on = line == "[%s]" % section
            continue
        if on:
            rows.append(line.split())
    return rows


@pytest.mark.parametrize("section", ["Z", "Zbar"])
def test_Z_structure_as_printed_in_paper(section):
    """n = 12, p = 4, m = 3: every entry of Z (L116) and Z-bar (L136) sits where the paper prints it."""
    n, P, m = 12, 4, 3
    a, b, c = random_dominant(n)
    d = rng.uniform(-1, 1, n)
    _, v, w = orc.local_solves(P, a, b, c, d)
    Z = orc.build_Z(n, P, v, w)
    M = Z if section == "Z" else orc.build_Zbar(Z)
    gold = parse_golden(section)
    assert len(gold) == 6 and all(len(r) == 6 for r in gold)
    for r in range(6):
        for cidx in range(6):
            s = gold[r][cidx]
            if s in (".", "0"):
                assert M[r, cidx] == 0.0, (r, cidx)
            elif s == "1":
                assert M[r, cidx] == 1.0, (r, cidx)
            else:
                kind, pos, part = re.match(r"([vw])([1m])\((\d)\)", s).groups()
                vec = v if kind == "v" else w
                idx = int(part) * m + (0 if pos == "1" else m - 1)
                assert M[r, cidx] == vec[idx] and vec[idx] != 0.0, (r, cidx, s)


def test_Zbar_is_tridiagonal_and_equals_P_plus_EtAinvVP():
    n, P = 24, 6
    a, b, c = random_dominant(n)
    _, v, w = orc.local_solves(P, a, b, c, np.zeros(n))
    Zb = orc.build_Zbar(orc.build_Z(n, P, v, w))
    K = 2 * (P - 1)
    for r in range(K):
        for cidx in range(K):
            if abs(r - cidx) > 1:
                assert Zb[r, cidx] == 0.0
    # independent dense construction of Z = I + E^T A~^{-1} V
    st = orc.partition_bounds(n, P)
    A = orc.dense_from_tridiag(a, b, c)
    At = A.copy(); E = np.zeros((n, K)); V = np.zeros((n, K))
    for i in range(1, P):
        f, l = st[i], st[i] - 1
        At[f, l] = 0.0; At[l, f] = 0.0
        E[l, 2 * i - 2] = 1.0; E[f, 2 * i - 1] = 1.0
        V[f, 2 * i - 2] = a[f]; V[l, 2 * i - 1] = c[l]
    assert np.allclose(At + V @ E.T, A, atol=0)                      # dA = V E^T (L85-91)
    Zd = np.eye(K) + E.T @ np.linalg.solve(At, V)
    assert np.allclose(orc.build_Z(n, P, v, w), Zd, atol=1e-14)
    Pm = np.zeros((K, K))
    for k in range(0, K, 2):
        Pm[k, k + 1] = Pm[k + 1, k] = 1.0
    assert np.allclose(Zb, Pm + E.T @ np.linalg.solve(At, V @ Pm), atol=1e-14)      # Eq. for Z-bar, L136


def test_spikes_and_xt_vs_dense_blocks():
    n, P = 23, 4                                                     # ragged: sizes 6,6,6,5
    a, b, c = random_dominant(n)
    d = rng.uniform(-1, 1, n)
    xt, v, w = orc.local_solves(P, a, b, c, d)
    st = orc.partition_bounds(n, P)
    A = orc.dense_from_tridiag(a, b, c)
    for p in range(P):
        s, e = st[p], st[p + 1]
        Ap = A[s:e, s:e]
        assert relerr(xt[s:e], np.linalg.solve(Ap, d[s:e])) < 1e-14
        e1 = np.zeros(e - s); e1[0] = a[s]
        em = np.zeros(e - s); em[-1] = c[e - 1]
        if p > 0:
            assert np.allclose(v[s:e], np.linalg.solve(Ap, e1), rtol=1e-13, atol=1e-300)
        else:
            assert np.all(v[s:e] == 0)
        if p < P - 1:
            assert np.allclose(w[s:e], np.linalg.solve(Ap, em), rtol=1e-13, atol=1e-300)
        else:
            assert np.all(w[s:e] == 0)


@pytest.mark.parametrize("n,P", [(12, 4), (32, 4), (64, 8), (100, 7), (288, 16), (288, 32)])
def test_ppt_equals_thomas_and_y_are_interface_values(n, P):
    """PPT makes no approximation (L156); y_{2i-1} = x_{last_{i-1}}, y_{2i} = x_{first_i}."""
    a, b, c = random_dominant(n, margin=0.05)
    d = rng.uniform(-1, 1, n)
    x_ref = orc.thomas(a, b, c, d)
    x, y = orc.partitioned_line(P, orc.MODE_PPT, a, b, c, d, return_y=True)
    assert relerr(x, x_ref) < 1e-13
    assert relerr(x, np.linalg.solve(orc.dense_from_tridiag(a, b, c), d)) < 1e-13
    st = orc.partition_bounds(n, P)
    for i in range(1, P):
        assert abs(y[2 * i - 2] - x_ref[st[i] - 1]) < 1e-13 * np.max(np.abs(x_ref))
        assert abs(y[2 * i - 1] - x_ref[st[i]]) < 1e-13 * np.max(np.abs(x_ref))


def test_P1_reduces_to_thomas_bitwise():
    a, b, c = random_dominant(40)
    d = rng.uniform(-1, 1, 40)
    for mode in (orc.MODE_PDD, orc.MODE_PPT):
        assert np.array_equal(orc.partitioned_line(1, mode, a, b, c, d), orc.thomas(a, b, c, d))


def test_pdd_error_bounded_by_dropped_and_exact_when_decayed():
    """L148-154: v_m, w_1 -> 0 when n >> p for strictly dominant systems; then PDD == PPT."""
    n = 256
    for margin, P in [(3.0, 4), (3.0, 8), (0.05, 4), (0.05, 16), (0.002, 8)]:
        a, b, c = random_dominant(n, margin=margin)
        d = rng.uniform(-1, 1, n)
        x_ref = orc.thomas(a, b, c, d)
        dropped = orc.pdd_dropped(P, a, b, c)
        err = relerr(orc.partitioned_line(P, orc.MODE_PDD, a, b, c, d), x_ref)
        assert err <= 50 * dropped + 1e-13, (margin, P, err, dropped)
        if dropped < 1e-30:
            assert err < 1e-13
    # strongly dominant: dropped entries are below the rounding of the 2x2 blocks -> PDD and PPT agree to rounding
    a, b, c = random_dominant(64, margin=50.0)
    d = rng.uniform(-1, 1, 64)
    assert relerr(orc.partitioned_line(4, orc.MODE_PDD, a, b, c, d), orc.partitioned_line(4, orc.MODE_PPT, a, b, c, d)) < 1e-15


def test_pdd_dropped_matches_dense_definition():
    n, P = 48, 6
    a, b, c = random_dominant(n, margin=0.1)
    _, v, w = orc.local_solves(P, a, b, c, np.zeros(n))
    st = orc.partition_bounds(n, P)
    ref = max(max(abs(v[st[i] - 1]) for i in range(2, P)), max(abs(w[st[i]]) for i in range(1, P - 1)))
    assert orc.pdd_dropped(P, a, b, c) == ref
    Zfull = orc.build_Z(n, P, v, w); Zpdd = orc.build_Z(n, P, v, w, pdd=True)
    assert np.max(np.abs(Zfull - Zpdd)) == ref
    for i in range(1, P):                      # PDD Z is block diagonal with 2x2 blocks (L152-154)
        blk = Zpdd[2 * i - 2:2 * i, :].copy(); blk[:, 2 * i - 2:2 * i] = 0
        assert np.all(blk == 0)


def test_paper_claims_pdd_on_adi_and_helmholtz():
    """L164: PDD matches the exact ADI solution to machine accuracy (n >> p); L172: PDD inaccurate on the weakly
    dominant Poisson systems, while PPT stays exact (L156)."""
    cfg = configs.get(2)
    _, yf, _ = cfg.faces()
    d = inputs.uniform_pm1(7, cfg.ny)
    a, b, c = orc.adi_coeffs(yf, orc.BC_DIRICHLET, cfg.alpha)
    assert relerr(orc.partitioned_line(4, orc.MODE_PDD, a, b, c, d), orc.thomas(a, b, c, d)) < 1e-14
    kz2 = cfg.kz2()
    a, b, c, _ = orc.helmholtz_coeffs(yf, kz2[1])
    ref = orc.thomas(a, b, c, d, long_double=True)
    assert relerr(orc.partitioned_line(4, orc.MODE_PDD, a, b, c, d), ref) > 1e-3
    assert relerr(orc.partitioned_line(4, orc.MODE_PPT, a, b, c, d), ref) < 1e-12
    assert relerr(orc.thomas(a, b, c, d), ref) < 1e-12


@pytest.mark.parametrize("mode", [orc.MODE_PDD, orc.MODE_PPT])
def test_cyclic_line_with_partitions(mode):
    n, P = 64, 4
    a = rng.uniform(-1, 0, n); c = rng.uniform(-1, 0, n); b = 1.0 - a - c + 6.0
    d = rng.uniform(-1, 1, n)
    ref = np.linalg.solve(orc.dense_from_tridiag(a, b, c, cyclic=True), d)
    assert relerr(orc.cyclic_line(P, mode, a, b, c, d), ref) < 1e-13
    assert relerr(orc.cyclic_thomas(a, b, c, d), ref) < 1e-14


def cyclic_pdd_dense_reference(P, a, b, c, d):
    """Independent restatement with dense LAPACK algebra: Woodbury (Eq.(3)-(4)) with the wrap corners in dA, the far
    spike ends deleted from Z = I + E^T A~^{-1} V (L148-154), everything else exact."""
    n = b.size
    st = orc.partition_bounds(n, P)
    A = orc.dense_from_tridiag(a, b, c, cyclic=True)
    At = np.zeros_like(A)
    for p in range(P):
        At[st[p]:st[p + 1], st[p]:st[p + 1]] = A[st[p]:st[p + 1], st[p]:st[p + 1]]
    dA = A - At                                              # the 2P corner entries
    cols, V = [], []
    for i in range(P):                                       # interface i: rows last_{i-1}, first_i
        last, first = st[(i - 1) % P + 1] - 1, st[i]
        cols += [last, first]
        ea = np.zeros(n); ea[first] = dA[first, last]; ec = np.zeros(n); ec[last] = dA[last, first]
        V += [ea, ec]                                        # column of V multiplying x_last, then x_first
    E = np.zeros((n, 2 * P)); E[cols, np.arange(2 * P)] = 1.0
    V = np.array(V).T
    assert np.allclose(V @ E.T, dA, atol=0, rtol=0)
    Y = np.linalg.solve(At, V)
    Z = np.eye(2 * P) + E.T @ Y
    Zp = np.zeros_like(Z)
    for i in range(P):                                       # keep only the 2x2 diagonal blocks
        Zp[2 * i:2 * i + 2, 2 * i:2 * i + 2] = Z[2 * i:2 * i + 2, 2 * i:2 * i + 2]
    xt = np.linalg.solve(At, d)
    y = np.linalg.solve(Zp, E.T @ xt)
    return xt - Y @ y, float(np.max(np.abs(Z - Zp)))


@pytest.mark.parametrize("n,P,margin", [(64, 4, 6.0), (60, 2, 0.3), (37, 5, 0.05), (96, 8, 0.01)])
def test_cyclic_pdd_matches_dense_woodbury_with_far_ends_deleted(n, P, margin):
    a = rng.uniform(-1, -0.2, n); c = rng.uniform(-1, -0.2, n); b = margin - a - c
    d = rng.uniform(-1, 1, n)
    ref, dropped = cyclic_pdd_dense_reference(P, a, b, c, d)
    x = orc.cyclic_pdd_line(P, a, b, c, d)
    assert relerr(x, ref) < 1e-12
    assert abs(orc.cyclic_pdd_dropped(P, a, b, c) - dropped) <= 1e-12 * dropped + 1e-300
    assert np.array_equal(orc.cyclic_line(P, orc.MODE_PDD, a, b, c, d), x)
    exact = np.linalg.solve(orc.dense_from_tridiag(a, b, c, cyclic=True), d)
    assert relerr(x, exact) <= 50 * dropped + 1e-13, (relerr(x, exact), dropped)
    if dropped > 1e-6:                                       # and it IS an approximation when the spikes have not decayed
        assert relerr(x, exact) > 1e-3 * dropped


def test_cyclic_pdd_spikes_and_exactness_when_decayed():
    n, P = 48, 4
    a = rng.uniform(-1, 0, n); c = rng.uniform(-1, 0, n); b = 1.0 - a - c + 60.0
    d = rng.uniform(-1, 1, n)
    x, v, w = orc.cyclic_pdd_line(P, a, b, c, d, return_spikes=True)
    st = orc.partition_bounds(n, P)
    for p in range(P):                                       # Eq.(6): A_p v = a_first e_first, A_p w = c_last e_last, every partition
        s, e = st[p], st[p + 1]
        Ap = orc.dense_from_tridiag(a[s:e], b[s:e], c[s:e])
        rv = np.zeros(e - s); rv[0] = a[s]; rw = np.zeros(e - s); rw[-1] = c[e - 1]
        assert np.max(np.abs(Ap @ v[s:e] - rv)) < 1e-13 and np.max(np.abs(Ap @ w[s:e] - rw)) < 1e-13
    assert orc.cyclic_pdd_dropped(P, a, b, c) < 1e-17
    assert relerr(x, orc.cyclic_thomas(a, b, c, d)) < 1e-14
    assert relerr(x, orc.cyclic_line(P, orc.MODE_PPT, a, b, c, d)) < 1e-14
    # identity operator: bit-exact
    z = np.zeros(n)
    assert np.array_equal(orc.cyclic_pdd_line(P, z, np.ones(n), z, d), d)


# ---------------------------------------------------------------- the two definitions of PDD on a periodic line (A16)
def cyclic_pdd_outer_dense_reference(P, a, b, c, d):
    """Independent restatement of the outer-split PDD with LAPACK only: rank-1 split with gamma = -b_0 written out as
    dense matrices, PDD on A' as Woodbury with the far spike ends deleted from Z, q = A'^-1 u by a dense solve."""
    n = b.size
    st = orc.partition_bounds(n, P)
    A = orc.dense_from_tridiag(a, b, c, cyclic=True)
    gamma = -b[0]; g = a[0] / gamma
    u = np.zeros(n); u[0] = gamma; u[-1] = c[-1]
    vt = np.zeros(n); vt[0] = 1.0; vt[-1] = g
    Ap = A - np.outer(u, vt)                                   # plain tridiagonal A'
    assert abs(Ap[0, -1]) < 1e-15 and abs(Ap[-1, 0]) < 1e-15
    Ap[0, -1] = 0.0; Ap[-1, 0] = 0.0
    At = Ap.copy()
    K = 2 * (P - 1)
    V = np.zeros((n, K)); E = np.zeros((n, K))
    for i in range(1, P):
        last, first = st[i] - 1, st[i]
        At[first, last] = 0.0; At[last, first] = 0.0
        E[last, 2 * i - 2] = 1.0; E[first, 2 * i - 1] = 1.0
        V[first, 2 * i - 2] = Ap[first, last]; V[last, 2 * i - 1] = Ap[last, first]
    xt = np.linalg.solve(At, d); Y = np.linalg.solve(At, V)
    Z = np.eye(K) + E.T @ Y
    for i in range(1, P):                                      # PDD: delete v_last^(i-1) (row 2i-2) and w_first^(i) (row 2i-1)
        if i >= 2: Z[2 * i - 2, 2 * i - 4] = 0.0
        if i <= P - 2: Z[2 * i - 1, 2 * i + 1] = 0.0
    y = xt - Y @ np.linalg.solve(Z, E.T @ xt)
    q = np.linalg.solve(Ap, u)
    return y - q * (vt @ y) / (1.0 + vt @ q)


@pytest.mark.parametrize("n,P,margin", [(24, 2, 0.3), (24, 4, 0.3), (30, 5, 1.0), (37, 3, 0.1), (64, 8, 0.5)])
def test_cyclic_pdd_outer_split_matches_dense_restatement(n, P, margin):
    a = rng.uniform(-1, 0, n); c = rng.uniform(-1, 0, n); b = 1.0 - a - c + margin
    d = rng.uniform(-1, 1, n)
    x = orc.cyclic_pdd_outer_line(P, a, b, c, d)
    assert relerr(x, cyclic_pdd_outer_dense_reference(P, a, b, c, d)) < 1e-12
    exact = np.linalg.solve(orc.dense_from_tridiag(a, b, c, cyclic=True), d)
    dropped = orc.cyclic_pdd_outer_dropped(P, a, b, c)
    assert relerr(x, exact) <= 50 * dropped + 1e-13
    # P = 2: ONE interface, nothing to drop -- the outer split is exact there, the cyclic closure is not (reading A16)
    if P == 2:
        assert dropped == 0.0 and relerr(x, exact) < 1e-13
        assert relerr(orc.cyclic_pdd_line(P, a, b, c, d), exact) > 1e-9


def test_cyclic_pdd_outer_P1_is_cyclic_thomas_bitwise():
    n = 19
    a = rng.uniform(-1, 0, n); c = rng.uniform(-1, 0, n); b = 1.5 - a - c
    d = rng.uniform(-1, 1, n)
    assert np.array_equal(orc.cyclic_pdd_outer_line(1, a, b, c, d), orc.cyclic_thomas(a, b, c, d))


@pytest.mark.parametrize("cfg_no", [1, 2, 3, 4, 5, 6])
def test_two_periodic_pdd_definitions_agree_to_dropped_on_config_z_operators(cfg_no):
    """Finding A16 of the round-1 verdict: SURVEY 8(c) C2 gives the oracle the OUTER split, the product computes the
    CYCLIC closure.  Both stay in the oracle; on every config's z operator and every P the configs name (and the bench
    uses) they differ by at most 50 max(dropped) -- and where PDD is inside its regime (dropped <= 1e-11) both equal the
    exact solution to 1e-12, so neither can drift without failing here."""
    c = configs.get(cfg_no)
    a, b, cc = orc.adi_coeffs(c.faces()[2], orc.BC_PERIODIC, c.alpha)
    n = c.nz
    ds = [rng.uniform(-1, 1, n), np.cos(2 * np.pi * 3 * (np.arange(n) + 0.5) / n), np.eye(n)[0]]
    for P in sorted(set([2, 4, 8, 16, 24, 32]) | set(c.P)):
        if n // P < 2:
            continue
        dr_c, dr_o = orc.cyclic_pdd_dropped(P, a, b, cc), orc.cyclic_pdd_outer_dropped(P, a, b, cc)
        for d in ds:
            exact = orc.cyclic_thomas(a, b, cc, d)
            xc, xo = orc.cyclic_pdd_line(P, a, b, cc, d), orc.cyclic_pdd_outer_line(P, a, b, cc, d)
            scale = np.max(np.abs(exact))
            assert np.max(np.abs(xc - xo)) <= (50 * max(dr_c, dr_o) + 1e-13) * scale, (cfg_no, P, dr_c, dr_o)
            assert np.max(np.abs(xc - exact)) <= (50 * dr_c + 1e-13) * scale
            assert np.max(np.abs(xo - exact)) <= (50 * dr_o + 1e-13) * scale
            if max(dr_c, dr_o) <= 1e-11:
                assert np.max(np.abs(xc - exact)) < 1e-12 * scale and np.max(np.abs(xo - exact)) < 1e-12 * scale


def test_two_periodic_pdd_definitions_on_random_weakly_dominant_lines():
    for trial in range(20):
        n = int(rng.integers(12, 80)); P = int(rng.integers(2, max(3, n // 4)))
        if n // P < 2:
            continue
        margin = 10.0 ** rng.uniform(-2, 1)
        a = rng.uniform(-1, 0, n); c = rng.uniform(-1, 0, n); b = 1.0 - a - c + margin
        d = rng.uniform(-1, 1, n)
        exact = np.linalg.solve(orc.dense_from_tridiag(a, b, c, cyclic=True), d)
        dr = max(orc.cyclic_pdd_dropped(P, a, b, c), orc.cyclic_pdd_outer_dropped(P, a, b, c))
        xc, xo = orc.cyclic_pdd_line(P, a, b, c, d), orc.cyclic_pdd_outer_line(P, a, b, c, d)
        assert relerr(xc, xo) <= 50 * dr + 1e-13, (n, P, margin, relerr(xc, xo), dr)
        assert relerr(xc, exact) <= 50 * dr + 1e-13 and relerr(xo, exact) <= 50 * dr + 1e-13


# ---------------------------------------------------------------- 3-D sweeps
def sweep_reference(field, a, b, c, axis, cyclic):
    """independent: move the axis last and solve every line with LAPACK."""
    n = b.size
    A = orc.dense_from_tridiag(a, b, c, cyclic=cyclic)
    moved = np.moveaxis(field, axis, 0).reshape(n, -1)
    sol = np.linalg.solve(A, moved)
    return np.moveaxis(sol.reshape(np.moveaxis(field, axis, 0).shape), 0, axis)


@pytest.mark.parametrize("direction", [0, 1, 2])
@pytest.mark.parametrize("mode,P", [(orc.MODE_THOMAS, 1), (orc.MODE_PPT, 3), (orc.MODE_PDD, 2)])
def test_adi_sweep_every_direction_vs_lapack(direction, mode, P):
    nx, ny, nz = 12, 10, 8
    xf = inputs.faces_uniform(nx, 1.5); yf = inputs.faces_tanh_two_sided(ny, 2.0); zf = inputs.faces_uniform(nz, 1.0)
    bcs = (orc.BC_DIRICHLET, orc.BC_DIRICHLET, orc.BC_PERIODIC)
    alpha = 2e-3
    field = inputs.rhs_uniform((nz, ny, nx), 11)
    f = (xf, yf, zf)[direction]
    a, b, c = orc.adi_coeffs(f, bcs[direction], alpha)
    ref = sweep_reference(field, a, b, c, axis=2 - direction, cyclic=(direction == 2))
    out = orc.adi_sweep(field.copy(), xf, yf, zf, bcs, direction, mode, P, alpha)
    tol = 1e-13
    if mode == orc.MODE_PDD and direction == 2:             # periodic + PDD: P interfaces, an approximation even at P = 2
        tol += 50 * orc.cyclic_pdd_dropped(P, a, b, c)
        assert tol < 1e-2
    assert relerr(out, ref) < tol


def test_sweep_one_hot_touches_only_its_line():
    nx, ny, nz = 8, 6, 5
    xf = inputs.faces_uniform(nx, 1.0); yf = inputs.faces_uniform(ny, 1.0); zf = inputs.faces_uniform(nz, 1.0)
    bcs = (orc.BC_DIRICHLET, orc.BC_DIRICHLET, orc.BC_PERIODIC)
    for direction in range(3):
        field = np.zeros((nz, ny, nx)); field[2, 3, 4] = 1.0
        out = orc.adi_sweep(field, xf, yf, zf, bcs, direction, orc.MODE_THOMAS, 1, 0.05)
        mask = np.zeros_like(out, dtype=bool)
        if direction == 0: mask[2, 3, :] = True
        if direction == 1: mask[2, :, 4] = True
        if direction == 2: mask[:, 3, 4] = True
        assert np.all(out[~mask] == 0.0) and np.all(out[mask] != 0.0)


@pytest.mark.parametrize("mode,P", [(orc.MODE_THOMAS, 1), (orc.MODE_PPT, 4), (orc.MODE_THOMAS_LD, 1)])
def test_helmholtz_solve_residual_and_pin(mode, P):
    nx, ny, nz = 6, 16, 8
    nm = nz // 2 + 1
    yf = inputs.faces_tanh_one_sided(ny, 2.0)
    kz2 = inputs.modified_wavenumbers_z(nz)
    kx2 = inputs.modified_wavenumbers_x(nx, 0.75)
    rhs = inputs.rhs_complex_uniform((nm, ny, nx), 5)
    sol = orc.helmholtz_solve(rhs.copy(), yf, kx2, kz2, mode, P)
    lo, up = orc.metrics(yf, orc.BC_NEUMANN)
    for m in range(nm):
        for i in range(nx):
            lam = kx2[i] + kz2[m]
            L = np.zeros((ny, ny))
            for j in range(ny):                                   # unpinned operator delta2_y - lambda, Neumann ends
                if j > 0: L[j, j - 1] = lo[j]; L[j, j] -= lo[j]
                if j < ny - 1: L[j, j + 1] = up[j]; L[j, j] -= up[j]
                L[j, j] -= lam
            phi = sol[m, :, i]; r = L @ phi - rhs[m, :, i]
            scale = np.max(np.abs(L)) * np.max(np.abs(phi))
            if lam == 0.0:
                assert phi[0] == 0.0                               # pinned point
                assert np.max(np.abs(r[1:])) < 1e-12 * scale
            else:
                assert np.max(np.abs(r)) < 1e-12 * scale
    # kx2 = None means zeros: then the whole m = 0 plane is pinned
    sol0 = orc.helmholtz_solve(rhs.copy(), yf, None, kz2, mode, P)
    assert np.all(sol0[0, 0, :] == 0.0)


def test_cyclic_solve_user_coefficients():
    nx, ny, nz = 5, 4, 12
    a = rng.uniform(-1, 0, nz); c = rng.uniform(-1, 0, nz); b = 2.5 - a - c
    field = inputs.rhs_uniform((nz, ny, nx), 3)
    ref = sweep_reference(field, a, b, c, axis=0, cyclic=True)
    for mode, P in [(orc.MODE_THOMAS, 1), (orc.MODE_PPT, 3), (orc.MODE_PDD, 2)]:
        out = orc.cyclic_solve(field.copy(), 2, mode, P, a, b, c)
        tol = 1e-13 + (50 * orc.cyclic_pdd_dropped(P, a, b, c) if mode == orc.MODE_PDD else 0.0)   # PDD: P interfaces, approximate
        assert relerr(out, ref) < tol < 1e-2
