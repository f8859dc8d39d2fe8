"""GPU parity: libdwf (through its C ABI) against the CPU oracle, element by element on the same
seeded inputs.  Tolerances are BASELINE.json north_star's: relative L2 <= 1e-12 (fp64), <= 1e-5 (fp32)
per operator apply, <= 1e-4 for the fp32 order-64 Chebyshev filter; CG per DESIGN.md R19.
"""
import numpy as np
import pytest

import dwf_inputs as gen
from gpu_util import M5, TOL_APPLY, TOL_CHEB, Rig, rel_l2

pytestmark = pytest.mark.gpu

from paper_2103_05034_b200 import (DWF_DAGGER, DWF_DDW, DWF_DHOP, DWF_DPV, DWF_HDW, DWF_MEE, DWF_MOOINV,  # noqa: E402
                                   DWF_SCHUR_EO)


# ------------------------------------------------------------------ layout round trip (a1)
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("L,Ls,nrhs", [((4, 4, 4, 4), 8, 1), ((6, 4, 8, 4), 4, 3)])
def test_import_export_roundtrip(prec, L, Ls, nrhs):
    rig = Rig(L, Ls, prec)
    psi = rig.spinor(nrhs, 2000)
    assert np.array_equal(rig.canonical(rig.native(psi), nrhs), psi)            # bit exact
    for parity in (0, 1):
        got = rig.canonical(rig.native(psi, parity), nrhs, parity)
        assert np.array_equal(got, gen.keep_parity(psi, L, parity))


# ------------------------------------------------------------------ configs[0]: 4^4 x 8
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("unit", [False, True])
def test_config0_operators(oracle, prec, unit):
    L, Ls, mass = (4, 4, 4, 4), 8, 0.01
    rig = Rig(L, Ls, prec, mass, seed_U=1000, unit_links=unit)
    psi = rig.spinor(1, 2000)
    tol = TOL_APPLY[prec]
    assert rel_l2(rig.apply(DWF_DHOP, psi), oracle.dhop(rig.U, psi)) < tol
    assert rel_l2(rig.apply(DWF_DDW, psi), oracle.ddw(rig.U, psi, M5, mass)) < tol
    assert rel_l2(rig.apply(DWF_HDW, psi), oracle.hdw(rig.U, psi, M5, mass)) < tol
    assert rel_l2(rig.apply(DWF_DPV, psi), oracle.dpv(rig.U, psi, M5)) < tol
    assert rel_l2(rig.apply(DWF_DHOP | DWF_DAGGER, psi), oracle.dhop(rig.U, psi, dagger=True)) < tol
    assert rel_l2(rig.apply(DWF_DDW | DWF_DAGGER, psi), oracle.ddw(rig.U, psi, M5, mass, dagger=True)) < tol
    assert rel_l2(rig.apply(DWF_DPV | DWF_DAGGER, psi), oracle.dpv(rig.U, psi, M5, dagger=True)) < tol
    assert rel_l2(rig.apply(DWF_HDW | DWF_DAGGER, psi), oracle.hdw(rig.U, psi, M5, mass)) < tol


def test_config0_point_source_golden(oracle):
    """The hand-derived worked example (tests/golden/point_source_ddw.txt) straight on the GPU path."""
    from test_oracle_pins import _read_golden
    L, Ls = (4, 4, 4, 4), 8
    rig = Rig(L, Ls, "f64", 0.01, unit_links=True)
    out = rig.apply(DWF_DDW, gen.point_source(L, Ls, (0, 0, 0, 0), 0, 0, 0))[0]
    expect = np.zeros_like(out)
    for src, s, (x, y, z, t), spin, val in _read_golden():
        if src == "A":
            expect[s, t, z, y, x, spin, 0] = val
    assert np.max(np.abs(out - expect)) < 1e-14


# ------------------------------------------------------------------ ragged shapes, several rhs, all Ls
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("L,Ls,nrhs", [((6, 4, 8, 4), 4, 3), ((4, 8, 4, 6), 12, 2), ((8, 4, 4, 4), 24, 1),
                                       ((4, 4, 4, 8), 32, 1), ((4, 4, 6, 4), 6, 5)])
def test_ragged_shapes(oracle, prec, L, Ls, nrhs):
    mass = 0.05
    rig = Rig(L, Ls, prec, mass, seed_U=17)
    psi = rig.spinor(nrhs, 18)
    tol = TOL_APPLY[prec]
    assert rel_l2(rig.apply(DWF_DDW, psi), oracle.ddw(rig.U, psi, M5, mass)) < tol
    assert rel_l2(rig.apply(DWF_HDW, psi), oracle.hdw(rig.U, psi, M5, mass)) < tol
    assert rel_l2(rig.apply(DWF_DDW | DWF_DAGGER, psi), oracle.ddw(rig.U, psi, M5, mass, dagger=True)) < tol
    pe = gen.keep_parity(psi, L, 0)
    assert rel_l2(rig.apply(DWF_MEE, pe, half=True), oracle.mpp(pe, M5, mass, 0)) < tol
    assert rel_l2(rig.apply(DWF_MEE | DWF_DAGGER, pe, half=True), oracle.mpp(pe, M5, mass, 0, dagger=True)) < tol
    if Ls in (4, 8, 12, 16, 24, 32):
        rig.d.set_workspace(nrhs)
        assert rel_l2(rig.apply(DWF_MOOINV, pe, half=True), oracle.mpp_inv(pe, M5, mass, 0)) < tol
        assert rel_l2(rig.apply(DWF_MOOINV | DWF_DAGGER, pe, half=True), oracle.mpp_inv(pe, M5, mass, 0, dagger=True)) < tol
        assert rel_l2(rig.apply(DWF_SCHUR_EO, pe, half=True), oracle.mpc(rig.U, pe, M5, mass)) < tol
        assert rel_l2(rig.apply(DWF_SCHUR_EO | DWF_DAGGER, pe, half=True), oracle.mpc(rig.U, pe, M5, mass, dagger=True)) < tol


# ------------------------------------------------------------------ configs[1]: 8^4 x 16, Schur on 4 RHS + 50 CG iterations
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_config1_schur_and_cg(oracle, prec):
    L, Ls, mass = (8, 8, 8, 8), 16, 0.01
    rig = Rig(L, Ls, prec, mass, seed_U=1001, ws_nrhs=4)
    psi = gen.keep_parity(rig.spinor(4, 2001), L, 0)
    assert rel_l2(rig.apply(DWF_SCHUR_EO, psi, half=True), oracle.mpc(rig.U, psi, M5, mass)) < TOL_APPLY[prec]
    # CG: rhs = vector 0, x0 = 0, 50 iterations (R19 tolerances)
    b = psi[0:1]
    x_or, h_or = oracle.cg_schur(rig.U, b, M5, mass, 50)
    bn = rig.native(b, 0)
    xn = rig.d.field(1, half=True, zero=True)
    hist = np.array(rig.d.cg_schur(bn, xn, 50))
    x = rig.canonical(xn, 1, 0)
    tol_h, tol_x = (1e-9, 1e-10) if prec == "f64" else (1e-4, 1e-5)
    assert np.max(np.abs(hist - h_or) / h_or) < tol_h
    assert rel_l2(x, x_or) < tol_x
    assert hist[50] < 1e-4 * hist[0]                                   # it does converge


# ------------------------------------------------------------------ BLAS-1 (a7)
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("nrhs,half", [(1, False), (3, False), (4, True)])
def test_blas1(oracle, prec, nrhs, half):
    L, Ls = (4, 6, 4, 8), 8
    rig = Rig(L, Ls, prec)
    x, y = rig.spinor(nrhs, 5), rig.spinor(nrhs, 6)
    parity = 0 if half else -1
    if half:
        x, y = gen.keep_parity(x, L, 0), gen.keep_parity(y, L, 0)
    xn, yn = rig.native(x, parity), rig.native(y, parity)
    got = np.array(rig.d.inner(xn, yn, nrhs, half))
    want = oracle.inner(x, y)
    assert np.max(np.abs(got - want) / np.abs(want)) < 1e-13          # fp64 accumulation on both sides
    got = np.array(rig.d.norm2(xn, nrhs, half))
    assert np.max(np.abs(got - oracle.norm2(x)) / oracle.norm2(x)) < 1e-13
    a = [complex(0.3 * (r + 1), -1.1 + 0.2 * r) for r in range(nrhs)]
    rig.d.axpy(a, xn, yn, nrhs, half)
    assert rel_l2(rig.canonical(yn, nrhs, parity), oracle.axpy(a, x, y)) < (1e-15 if prec == "f64" else 2e-7)


# ------------------------------------------------------------------ Chebyshev driver (a8)
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("order", [0, 1, 2, 3, 64])
def test_chebyshev_small(oracle, prec, order):
    L, Ls, mass, nrhs = (4, 4, 4, 8), 8, 0.01, 3
    rig = Rig(L, Ls, prec, mass, seed_U=1000, ws_nrhs=nrhs)
    psi = rig.spinor(nrhs, 2003)
    xn = rig.native(psi)
    out = rig.d.field(nrhs)
    rig.d.chebyshev(order, 0.01, 70.0, xn, out, nrhs)
    want = oracle.chebyshev(rig.U, psi, M5, mass, order, 0.01, 70.0)
    assert rel_l2(rig.canonical(out, nrhs), want) < TOL_CHEB[prec]
    assert np.array_equal(rig.canonical(xn, nrhs), psi)               # input untouched


# ------------------------------------------------------------------ error behaviour of the ABI
def test_abi_errors():
    from paper_2103_05034_b200 import Dwf, DwfError, DWF_F64
    with pytest.raises(DwfError):
        Dwf((4, 4, 4, 5), 8, M5, 0.01, DWF_F64)                        # odd extent
    with pytest.raises(DwfError):
        Dwf((4, 4, 4, 4), 8, 5.0, 0.01, DWF_F64)                       # M5 = 5: M_oo singular
    d = Dwf((4, 4, 4, 4), 8, M5, 0.01, DWF_F64)
    x, y = d.field(1), d.field(1)
    with pytest.raises(DwfError, match="set_gauge"):
        d.apply(DWF_DDW, x, y, 1)                                      # DWF_ENOGAUGE
    with pytest.raises(DwfError, match="in == out"):
        d.apply(DWF_MEE, x, x, 1)
    d2 = Dwf((4, 4, 4, 4), 10, M5, 0.01, DWF_F64)
    with pytest.raises(DwfError, match="instantiated"):
        d2.apply(DWF_MOOINV, d2.field(1, half=True), d2.field(1, half=True), 1)   # Ls = 10 unsupported


# ------------------------------------------------------------------ subspace generation + power method
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_chebyshev_subspace(oracle, prec):
    L, Ls, mass, nrhs = (4, 4, 4, 8), 8, 0.01, 2
    m, lam_lo, lam_max, delta, nvec = 12, 0.5, 60.0, 5, 4           # lam_lo inside the spectrum: the first pass amplifies
    rig = Rig(L, Ls, prec, mass, seed_U=1000, ws_nrhs=nrhs)
    eta = rig.spinor(nrhs, 2005)
    xn = rig.native(eta)
    phi = torch_empty_like_fields(rig, nvec, nrhs)
    rig.d.chebyshev_subspace(m, lam_lo, lam_max, delta, nvec, xn, phi, nrhs)
    want = oracle.chebyshev_subspace(rig.U, eta, M5, mass, m, lam_lo, lam_max, delta, nvec)
    n = xn.numel()
    for k in range(nvec):
        got = rig.canonical(phi[k * n:(k + 1) * n], nrhs)
        assert rel_l2(got, want[k]) < (1e-11 if prec == "f64" else 1e-4), k
    assert np.array_equal(rig.canonical(xn, nrhs), eta)               # input untouched
    # nvec = 1 is the first-pass filter alone
    one = torch_empty_like_fields(rig, 1, nrhs)
    rig.d.chebyshev_subspace(m, lam_lo, lam_max, delta, 1, xn, one, nrhs)
    assert rel_l2(rig.canonical(one, nrhs), want[0]) < (1e-11 if prec == "f64" else 1e-4)


def torch_empty_like_fields(rig, nvec, nrhs):
    import torch
    return torch.empty(nvec * rig.d.field(nrhs).numel(), dtype=rig.d.rdtype, device="cuda")


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_power_lambda_max(oracle, prec):
    L, Ls, mass = (4, 4, 4, 8), 8, 0.01
    rig = Rig(L, Ls, prec, mass, seed_U=1000, ws_nrhs=1)
    v0 = rig.spinor(1, 2006)
    vn = rig.native(v0)
    lam, hist = rig.d.power_lambda_max(30, vn)
    h_or, v_or = oracle.power_lambda_max(rig.U, v0, M5, mass, 30)
    tol = 1e-11 if prec == "f64" else 2e-5
    assert np.max(np.abs(np.array(hist) - np.array(h_or)) / np.array(h_or)) < tol
    assert lam == hist[-1] and 40 < lam < 70                          # random links: lambda_max ~ 48
    assert rel_l2(rig.canonical(vn, 1), v_or) < (1e-9 if prec == "f64" else 1e-3)


# ------------------------------------------------------------------ Chebyshev smoother (eq. 24-25)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_chebyshev_smoother(oracle, prec):
    L, Ls, mass, nrhs = (4, 4, 4, 8), 8, 0.01, 2
    N, a, b = 12, 0.5, 60.0                                           # Table I of the paper: Chebyshev [0.5, 60], order 12
    rig = Rig(L, Ls, prec, mass, seed_U=1000, ws_nrhs=nrhs)
    r = rig.spinor(nrhs, 2008)
    rn = rig.native(r)
    out = rig.d.field(nrhs)
    rig.d.chebyshev_smoother(N, a, b, rn, out, nrhs)
    want = oracle.chebyshev_smoother(rig.U, r, M5, mass, N, a, b)
    assert rel_l2(rig.canonical(out, nrhs), want) < (1e-11 if prec == "f64" else 1e-4)
    assert np.array_equal(rig.canonical(rn, nrhs), r)


# ------------------------------------------------------------------ complete red-black solve
@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
def test_solve_red_black(oracle, prec, tol):
    L, Ls, mass = (4, 4, 4, 8), 8, 0.05
    rig = Rig(L, Ls, prec, mass, seed_U=1000, ws_nrhs=1)
    eta = rig.spinor(1, 2009)
    en = rig.native(eta)
    psi = rig.d.field(1)
    iters, relres = rig.d.solve(en, psi, tol, 2000)
    psi_or, it_or = oracle.solve_rb(rig.U, eta, M5, mass, tol, 2000)
    got = rig.canonical(psi, 1)
    # R25: the oracle stops at the first iteration below tol (tested every iteration), the driver tests every 10
    # iterations: its count is the oracle's rounded up to a multiple of 10 (+- one test period for rounding drift in r_k)
    assert iters < 2000 and iters % 10 == 0
    assert -10 < iters - 10 * ((it_or + 9) // 10) <= 10, (iters, it_or)
    assert relres < 30 * tol                                           # true residual of the original system
    assert rel_l2(oracle.ddw(rig.U, got, M5, mass), eta) < 30 * tol    # ... and the oracle's operator agrees
    assert rel_l2(got, psi_or) < 100 * tol
    assert np.array_equal(rig.canonical(en, 1), eta)


# ------------------------------------------------------------------ Pauli-Villars preconditioned operator
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_mpvdag_m(oracle, prec):
    from paper_2103_05034_b200 import DWF_MPVDAG_M
    L, Ls, mass, nrhs = (4, 4, 6, 8), 8, 0.01, 2
    rig = Rig(L, Ls, prec, mass, seed_U=1000, ws_nrhs=nrhs)
    psi = rig.spinor(nrhs, 2010)
    tol = 2 * TOL_APPLY[prec]                                         # two operator applies
    assert rel_l2(rig.apply(DWF_MPVDAG_M, psi), oracle.mpvdag_m(rig.U, psi, M5, mass)) < tol
    assert rel_l2(rig.apply(DWF_MPVDAG_M | DWF_DAGGER, psi), oracle.mpvdag_m(rig.U, psi, M5, mass, dagger=True)) < tol


# ------------------------------------------------------------------ the other Schur form of Table V (L387; rest of N3)
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("L,Ls", [((8, 8, 4, 4), 16), ((6, 4, 4, 8), 8)])          # tiled (fused M^-1) and generic path
def test_schur_alt(oracle, prec, L, Ls):
    from paper_2103_05034_b200 import DWF_SCHUR_EO_ALT
    mass, nrhs = 0.02, 2
    rig = Rig(L, Ls, prec, mass, seed_U=51, ws_nrhs=nrhs)
    pe = gen.keep_parity(rig.spinor(nrhs, 52), L, 0)
    tol = 2 * TOL_APPLY[prec]
    assert rel_l2(rig.apply(DWF_SCHUR_EO_ALT, pe, half=True), oracle.mpc_alt(rig.U, pe, M5, mass)) < tol
    assert rel_l2(rig.apply(DWF_SCHUR_EO_ALT | DWF_DAGGER, pe, half=True), oracle.mpc_alt(rig.U, pe, M5, mass, dagger=True)) < tol


# ------------------------------------------------------------------ maximum number of right-hand sides (64) through the tiled kernel
def test_max_nrhs(oracle):
    L, Ls, mass, nrhs = (4, 4, 4, 4), 16, 0.01, 64
    rig = Rig(L, Ls, "f32", mass, seed_U=61, ws_nrhs=nrhs)
    psi = rig.spinor(nrhs, 62)
    got = rig.apply(DWF_HDW, psi)
    for r in (0, 31, 63):
        assert rel_l2(got[r:r + 1], oracle.hdw(rig.U, psi[r:r + 1], M5, mass)) < TOL_APPLY["f32"], r
    pe = gen.keep_parity(psi, L, 0)
    gs = rig.apply(DWF_SCHUR_EO, pe, half=True)
    for r in (0, 63):
        assert rel_l2(gs[r:r + 1], oracle.mpc(rig.U, pe[r:r + 1], M5, mass)) < TOL_APPLY["f32"], r
    from paper_2103_05034_b200 import DwfError
    with pytest.raises(DwfError):
        rig.d.apply(DWF_HDW, rig.d.field(1), rig.d.field(1), 65)        # nrhs > 64: DWF_EINVAL


# ------------------------------------------------------------------ multi-RHS CG (rest of SURVEY 8(f) N3): one CG per rhs in lock step
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_cg_multi_rhs(oracle, prec):
    L, Ls, mass, nrhs, iters = (8, 4, 4, 8), 16, 0.01, 3, 25
    rig = Rig(L, Ls, prec, mass, seed_U=71, ws_nrhs=nrhs)
    b = gen.keep_parity(rig.spinor(nrhs, 72), L, 0)
    bn = rig.native(b, 0)
    xn = rig.d.field(nrhs, half=True, zero=True)
    hist = np.array(rig.d.cg_schur_multi(bn, xn, iters, nrhs))          # [iters+1][nrhs]
    x = rig.canonical(xn, nrhs, 0)
    tol_h, tol_x = (1e-9, 1e-10) if prec == "f64" else (1e-4, 1e-5)
    for r in range(nrhs):
        x_or, h_or = oracle.cg_schur(rig.U, b[r:r + 1], M5, mass, iters)
        assert np.max(np.abs(hist[:, r] - h_or) / h_or) < tol_h, r
        assert rel_l2(x[r:r + 1], x_or) < tol_x, r
    # nrhs = 1 through the multi entry point is the single-rhs solver
    x1 = rig.d.field(1, half=True, zero=True)
    h1 = rig.d.cg_schur(rig.native(b[0:1], 0), x1, iters)
    assert np.max(np.abs(np.array(h1) - hist[:, 0]) / hist[:, 0]) < (1e-12 if prec == "f64" else 1e-5)


# ------------------------------------------------------------------ precision conversion + mixed-precision solve (rest of N3)
def test_convert_and_mixed_precision_solve(oracle):
    import torch
    from paper_2103_05034_b200 import Dwf, DWF_F32
    L, Ls, mass = (8, 4, 4, 8), 16, 0.05                               # fp64: 16-site tiles, fp32: 32-site tiles -> different site orders
    r64 = Rig(L, Ls, "f64", mass, seed_U=91, ws_nrhs=1)
    h32 = Dwf(L, Ls, M5, mass, DWF_F32)
    h32.set_gauge(torch.from_numpy(np.ascontiguousarray(r64.U)).to(torch.complex64).cuda())
    h32.set_workspace(1)
    eta = r64.spinor(2, 92)
    # conversion: fp64 native -> fp32 native -> canonical == canonical rounded to fp32 (bit exact), and back
    n64 = r64.native(eta)
    n32 = r64.d.convert_to(h32, n64, 2)
    can32 = h32.export(n32, 2).cpu().numpy()
    assert np.array_equal(can32, eta.astype(np.complex64))
    back = h32.convert_to(r64.d, n32, 2)
    assert np.array_equal(r64.canonical(back, 2), eta.astype(np.complex64).astype(np.complex128))
    # mixed-precision solve to fp64 accuracy
    e1 = r64.native(eta[0:1])
    psi = r64.d.field(1)
    outer, inner, relres = r64.d.solve_mixed(h32, e1, psi, 1e-11, 1e-4, 20, 2000)
    got = r64.canonical(psi, 1)
    assert 2 <= outer <= 8 and relres <= 1e-11
    assert rel_l2(oracle.ddw(r64.U, got, M5, mass), eta[0:1]) < 3e-11   # the oracle's operator agrees with the residual
    psi_or, _ = oracle.solve_rb(r64.U, eta[0:1], M5, mass, 1e-13, 4000)
    assert rel_l2(got, psi_or) < 1e-9


# ------------------------------------------------------------------ unpreconditioned CGNR on M^dag M (Table V)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_cg_normal(oracle, prec):
    L, Ls, mass, nrhs, iters = (4, 4, 4, 8), 16, 0.05, 2, 25
    rig = Rig(L, Ls, prec, mass, seed_U=95, ws_nrhs=nrhs)
    b = rig.spinor(nrhs, 96)
    bn = rig.native(b)
    xn = rig.d.field(nrhs, zero=True)
    hist = np.array(rig.d.cg_normal(bn, xn, iters, nrhs))
    x = rig.canonical(xn, nrhs)
    tol_h, tol_x = (1e-9, 1e-10) if prec == "f64" else (1e-4, 1e-5)
    for r in range(nrhs):
        x_or, h_or = oracle.cg_normal(rig.U, b[r:r + 1], M5, mass, iters)
        assert np.max(np.abs(hist[:, r] - h_or) / h_or) < tol_h, r
        assert rel_l2(x[r:r + 1], x_or) < tol_x, r
