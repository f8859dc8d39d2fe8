"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA code).

Each test names the passage it pins.  A plausible mistake anywhere in oracle/dwf_oracle.c (dropped
term, wrong sign or index, transposed link, wrong projector on a hop direction) fails one of them.
"""
import os

import numpy as np
import pytest

import dwf_inputs as gen

M5, MASS = 1.8, 0.01
L4 = (4, 4, 4, 4)
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


# ---------------------------------------------------------------- gamma algebra (R1, R2)
def test_gamma_algebra(oracle):
    g = [oracle.gamma(mu) for mu in range(4)]
    g5 = oracle.gamma(4)
    for mu in range(4):
        assert np.array_equal(g[mu].conj().T, g[mu])                      # hermitian
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.array_equal(anti, 2.0 * np.eye(4) * (mu == nu))     # Clifford algebra
    assert np.array_equal(g[0] @ g[1] @ g[2] @ g[3], g5)                  # gamma5 = gx gy gz gt
    assert np.array_equal(g5, np.diag([1, 1, -1, -1]).astype(complex))    # chiral: diagonal
    Pp, Pm = 0.5 * (np.eye(4) + g5), 0.5 * (np.eye(4) - g5)
    assert np.array_equal(Pp @ Pp, Pp) and np.array_equal(Pm @ Pm, Pm)
    assert np.array_equal(Pp @ Pm, np.zeros((4, 4))) and np.array_equal(Pp + Pm, np.eye(4))


# ---------------------------------------------------------------- worked example (eq. 2, 4, 5; A.8)
def _read_golden():
    rows = []
    with open(os.path.join(GOLDEN, "point_source_ddw.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            p = line.split()
            rows.append((p[0], int(p[1]), tuple(int(v) for v in p[2:6]), int(p[6]), float(p[7]) + 1j * float(p[8])))
    return rows


def test_worked_example_point_source(oracle):
    U = gen.gauge_unit(L4)
    rows = _read_golden()
    # source A: complete list of non-zero outputs
    out = oracle.ddw(U, gen.point_source(L4, 8, (0, 0, 0, 0), 0, 0, 0), M5, MASS)[0]
    expect = np.zeros_like(out)
    for src, s, (x, y, z, t), spin, val in rows:
        if src == "A":
            expect[s, t, z, y, x, spin, 0] = val
    assert np.count_nonzero(expect) == 18
    assert np.max(np.abs(out - expect)) < 1e-15
    # source B (spin 2): the only s != 0 entry is the m P_- wall at s = Ls-1
    out = oracle.ddw(U, gen.point_source(L4, 8, (0, 0, 0, 0), 0, 2, 0), M5, MASS)[0]
    expect = np.zeros_like(out[1:])
    for src, s, (x, y, z, t), spin, val in rows:
        if src == "B":
            expect[s - 1, t, z, y, x, spin, 0] = val
    assert np.max(np.abs(out[1:] - expect)) < 1e-15


# ---------------------------------------------------------------- free field closed form (L69, A.7)
def _plane_wave(L, Ls, n, chi):
    Lx, Ly, Lz, Lt = L
    p = np.array([2 * np.pi * n[0] / Lx, 2 * np.pi * n[1] / Ly, 2 * np.pi * n[2] / Lz,
                  2 * np.pi * (n[3] + 0.5) / Lt])                   # antiperiodic in t (R3)
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    psi = phase[None, :, :, :, :, None, None] * chi[:, None, None, None, None, :, :]
    return psi[None], p, phase


@pytest.mark.parametrize("L,Ls,n", [((4, 4, 4, 4), 8, (1, 2, 0, 1)), ((4, 6, 4, 8), 4, (3, 1, 2, 5))])
def test_free_field_plane_wave(oracle, L, Ls, n):
    """On unit links a plane wave is mapped to the momentum-space closed form (textbook Wilson
    operator; PAPER.md L69 gives its eigenvalues).  gamma matrices here are built from Pauli
    matrices in the test, not taken from the oracle."""
    sig = [np.array([[0, 1], [1, 0]]), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]])]
    Z, I2 = np.zeros((2, 2)), np.eye(2)
    g = [np.block([[Z, -1j * s], [1j * s, Z]]) for s in sig] + [np.block([[Z, I2], [I2, Z]])]
    Pp, Pm = np.diag([1.0, 1, 0, 0]), np.diag([0.0, 0, 1, 1])
    rng = np.random.default_rng(7)
    chi = rng.standard_normal((Ls, 4, 3)) + 1j * rng.standard_normal((Ls, 4, 3))
    psi, p, phase = _plane_wave(L, Ls, n, chi)
    U = gen.gauge_unit(L)
    # D_hop
    K = sum(2 * np.cos(p[mu]) * np.eye(4) - 2j * np.sin(p[mu]) * g[mu] for mu in range(4))
    want = phase[None, :, :, :, :, None, None] * np.einsum("ab,sbc->sac", K, chi)[:, None, None, None, None]
    assert rel(oracle.dhop(U, psi)[0], want) < 1e-14
    # D_DW
    diag = (5 - M5) * np.eye(4) - 0.5 * K
    o = np.einsum("ab,sbc->sac", diag, chi)
    for s in range(Ls):
        o[s] += (-Pm @ chi[s + 1]) if s + 1 < Ls else (MASS * Pm @ chi[0])
        o[s] += (-Pp @ chi[s - 1]) if s >= 1 else (MASS * Pp @ chi[Ls - 1])
    want = phase[None, :, :, :, :, None, None] * o[:, None, None, None, None]
    assert rel(oracle.ddw(U, psi, M5, MASS)[0], want) < 1e-14
    # D_W(M) = M + 4 - D_hop/2 (eq. 1) on the same wave
    Mw = -M5
    want = phase[None, :, :, :, :, None, None] * np.einsum("ab,sbc->sac", (Mw + 4) * np.eye(4) - 0.5 * K, chi)[:, None, None, None, None]
    assert rel(oracle.dwilson(U, psi, Mw)[0], want) < 1e-14


# ---------------------------------------------------------------- identities on random links
@pytest.fixture(scope="module")
def fields():
    U = gen.gauge_random(L4, 1000)
    x = gen.spinor_gaussian(L4, 8, 2, 2000)
    y = gen.spinor_gaussian(L4, 8, 2, 3000)
    return U, x, y


def test_dpar_is_wilson_plus_one(oracle, fields):
    """eq. 5: D_par = 5 - M5 - D_hop/2 = D_W(-M5) + 1."""
    U, x, _ = fields
    a = (5 - M5) * x - 0.5 * oracle.dhop(U, x)
    assert rel(a, oracle.dwilson(U, x, -M5) + x) < 1e-15


def test_hdw_hermitian(oracle, fields):
    """eq. 6: H_DW = Gamma5 D_DW is hermitian: <x,Hy> = <Hx,y>."""
    U, x, y = fields
    lhs = oracle.inner(x, oracle.hdw(U, y, M5, MASS))
    rhs = oracle.inner(oracle.hdw(U, x, M5, MASS), y)
    assert np.max(np.abs(lhs - rhs) / np.abs(lhs)) < 1e-13


def test_true_adjoint_and_gamma5_hermiticity(oracle, fields):
    """<x, D y> = <D^dag x, y> for the oracle's scatter adjoint; D^dag = Gamma5 D Gamma5 (eq. 12, R12);
    D^dag D = H^2 (eq. 11)."""
    U, x, y = fields
    for op, opd in [(lambda v: oracle.dhop(U, v), lambda v: oracle.dhop(U, v, dagger=True)),
                    (lambda v: oracle.ddw(U, v, M5, MASS), lambda v: oracle.ddw(U, v, M5, MASS, dagger=True)),
                    (lambda v: oracle.mpc(U, gen.keep_parity(v, L4, 0), M5, MASS),
                     lambda v: oracle.mpc(U, gen.keep_parity(v, L4, 0), M5, MASS, dagger=True))]:
        lhs = oracle.inner(x, op(y)); rhs = oracle.inner(opd(x), y)
        assert np.max(np.abs(lhs - rhs) / np.abs(lhs)) < 1e-13
    g5 = oracle.gamma5r5
    assert rel(g5(oracle.ddw(U, g5(x), M5, MASS)), oracle.ddw(U, x, M5, MASS, dagger=True)) < 1e-14
    h2 = oracle.hdw(U, oracle.hdw(U, x, M5, MASS), M5, MASS)
    dd = oracle.ddw(U, oracle.ddw(U, x, M5, MASS), M5, MASS, dagger=True)
    assert rel(h2, dd) < 1e-14
    xe = gen.keep_parity(x, L4, 0)
    assert rel(g5(oracle.mpc(U, g5(xe), M5, MASS)), oracle.mpc(U, xe, M5, MASS, dagger=True)) < 1e-14


def test_dpv_is_unit_mass(oracle, fields):
    """L50: D_PV - D_DW(m) is non-zero only in the two wall blocks and equals (1-m) P+- there."""
    U, x, _ = fields
    d = oracle.dpv(U, x, M5) - oracle.ddw(U, x, M5, MASS)
    Ls = x.shape[1]
    want = np.zeros_like(x)
    want[:, 0, ..., 0:2, :] = (1 - MASS) * x[:, Ls - 1, ..., 0:2, :]      # (0, Ls-1): P_+
    want[:, Ls - 1, ..., 2:4, :] = (1 - MASS) * x[:, 0, ..., 2:4, :]      # (Ls-1, 0): P_-
    assert np.max(np.abs(d - want)) < 1e-13
    assert rel(oracle.dpv(U, x, M5), oracle.ddw(U, x, M5, 1.0)) == 0.0


def _gauge_transform(U, g):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dag ; site axes of the canonical arrays are [t][z][y][x]."""
    Up = np.empty_like(U)
    for mu, axis in enumerate((3, 2, 1, 0)):
        g_fwd = np.roll(g, -1, axis=axis)
        Up[mu] = np.einsum("...ab,...bc,...dc->...ad", g, U[mu], g_fwd.conj())
    return Up


def test_gauge_covariance(oracle, fields):
    """D[U'] (g psi) = g D[U] psi for D_hop, D_DW, H_DW, M_pc and the Chebyshev filter."""
    U, x, _ = fields
    g = gen.su3_site_field(L4, 77)
    Up = _gauge_transform(U, g)
    rot = lambda v: np.einsum("tzyxab,rstzyxcb->rstzyxca", g, v)
    xe = gen.keep_parity(x, L4, 0)
    for op, arg in [(lambda UU, v: oracle.dhop(UU, v), x),
                    (lambda UU, v: oracle.ddw(UU, v, M5, MASS), x),
                    (lambda UU, v: oracle.hdw(UU, v, M5, MASS), x),
                    (lambda UU, v: oracle.mpc(UU, v, M5, MASS), xe),
                    (lambda UU, v: oracle.chebyshev(UU, v, M5, MASS, 5, 0.01, 70.0), x)]:
        assert rel(op(Up, rot(arg)), rot(op(U, arg))) < 1e-13


# ---------------------------------------------------------------- M_oo and its inverse (A.5)
@pytest.mark.parametrize("Ls", [4, 8, 16])
def test_mpp_inverse(oracle, Ls):
    x = gen.spinor_gaussian(L4, Ls, 1, 11)
    for dag in (False, True):
        v = oracle.mpp_inv(x, M5, MASS, 1, dagger=dag)
        back = oracle.mpp(v, M5, MASS, 1, dagger=dag)
        assert rel(back, gen.keep_parity(x, L4, 1)) < 1e-14
    # closed form of SURVEY App. A.5 for the P_+ chirality, written out in the test
    d = 5 - M5; k = 1 / d
    Ainv = np.zeros((Ls, Ls))
    for s in range(Ls):
        for s2 in range(Ls):
            Ainv[s, s2] = k ** (s - s2 + 1) if s >= s2 else -MASS * k ** (Ls + s - s2 + 1)
    Ainv /= (1 + MASS * k ** Ls)
    v = oracle.mpp_inv(x, M5, MASS, 1)
    xo = gen.keep_parity(x, L4, 1)
    want_plus = np.einsum("st,rtabcdef->rsabcdef", Ainv, xo[..., 0:2, :])
    want_minus = np.einsum("ts,rtabcdef->rsabcdef", Ainv, xo[..., 2:4, :])     # A_- = A_+^T
    assert rel(v[..., 0:2, :], want_plus) < 1e-14
    assert rel(v[..., 2:4, :], want_minus) < 1e-14


def test_mpc_composition(oracle, fields):
    """M_pc assembled from the separately-callable pieces; M_eo = -1/2 D_hop_eo."""
    U, x, _ = fields
    xe = gen.keep_parity(x, L4, 0)
    t = -0.5 * oracle.dhop(U, xe, row_parity=1)
    t = oracle.mpp_inv(t, M5, MASS, 1)
    t = -0.5 * oracle.dhop(U, t, row_parity=0)
    want = oracle.mpp(xe, M5, MASS, 0) - t
    got = oracle.mpc(U, xe, M5, MASS)
    assert rel(got, want) < 1e-15
    assert np.max(np.abs(gen.keep_parity(got, L4, 1))) == 0.0               # output lives on even sites


# ---------------------------------------------------------------- BLAS-1
def test_blas1(oracle, fields):
    _, x, y = fields
    a = np.array([0.3 - 1.2j, -2.0 + 0.5j])
    assert rel(oracle.axpy(a, x, y), y + a[:, None, None, None, None, None, None, None] * x) < 1e-15
    want = np.array([np.vdot(x[r], y[r]) for r in range(2)])
    assert np.max(np.abs(oracle.inner(x, y) - want) / np.abs(want)) < 1e-13
    assert np.max(np.abs(oracle.norm2(x) - np.array([np.sum(np.abs(x[r]) ** 2) for r in range(2)]))) < 1e-8


# ---------------------------------------------------------------- site-list mode (used at configs[4])
def _gather(L, U, psi, sites):
    """Neighbourhoods in the layout oracle.ddw_sites expects (harness code: indexing only)."""
    n, Ls = len(sites), psi.shape[1]
    nbr = np.zeros((n, 9, Ls, 4, 3), dtype=complex); links = np.zeros((n, 8, 3, 3), dtype=complex)
    for i, c in enumerate(sites):
        x, y, z, t = c
        nbr[i, 0] = psi[0, :, t, z, y, x]
        for mu in range(4):
            for j, d in enumerate((+1, -1)):
                m = list(c); m[mu] = (m[mu] + d) % L[mu]
                nbr[i, 1 + 2 * mu + j] = psi[0, :, m[3], m[2], m[1], m[0]]
                src = c if d > 0 else m
                links[i, 2 * mu + j] = U[mu, src[3], src[2], src[1], src[0]]
    return nbr, links


def test_site_list_mode(oracle):
    """ddw_sites against (i) the hand-derived golden example and (ii) the pinned full-volume D_DW at every site."""
    L, Ls = (4, 4, 4, 4), 8
    sites = [(x, y, z, t) for t in range(4) for z in range(4) for y in range(4) for x in range(4)]
    U = gen.gauge_unit(L)
    src = gen.point_source(L, Ls, (0, 0, 0, 0), 0, 0, 0)
    nbr, links = _gather(L, U, src, sites)
    got = oracle.ddw_sites(L, Ls, M5, MASS, np.array(sites, dtype=np.int32), nbr, links)
    expect = np.zeros_like(got)
    for s_, s, (x, y, z, t), spin, val in _read_golden():
        if s_ == "A":
            expect[sites.index((x, y, z, t)), s, spin, 0] = val
    assert np.max(np.abs(got - expect)) < 1e-15
    U = gen.gauge_random(L, 1000)
    psi = gen.spinor_gaussian(L, Ls, 1, 2000)
    nbr, links = _gather(L, U, psi, sites)
    got = oracle.ddw_sites(L, Ls, M5, MASS, np.array(sites, dtype=np.int32), nbr, links)
    full = oracle.ddw(U, psi, M5, MASS)[0]
    want = np.stack([full[:, t, z, y, x] for (x, y, z, t) in sites])
    assert rel(got, want) < 1e-15


def _gather2(L, U, psi_e, sites):
    """Two-hop neighbourhoods in the layout oracle.mpc_sites expects (harness code: indexing only)."""
    n, Ls = len(sites), psi_e.shape[1]
    self_ = np.zeros((n, Ls, 4, 3), dtype=complex); nbr2 = np.zeros((n, 8, 8, Ls, 4, 3), dtype=complex)
    links1 = np.zeros((n, 8, 3, 3), dtype=complex); links2 = np.zeros((n, 8, 8, 3, 3), dtype=complex)

    def step(c, mu, d):
        m = list(c); m[mu] = (m[mu] + d) % L[mu]
        return m
    for i, c in enumerate(sites):
        self_[i] = psi_e[0, :, c[3], c[2], c[1], c[0]]
        for mu in range(4):
            for j, d in enumerate((+1, -1)):
                y = step(c, mu, d)
                src = c if d > 0 else y
                links1[i, 2 * mu + j] = U[mu, src[3], src[2], src[1], src[0]]
                for nu in range(4):
                    for k, e in enumerate((+1, -1)):
                        zc = step(y, nu, e)
                        nbr2[i, 2 * mu + j, 2 * nu + k] = psi_e[0, :, zc[3], zc[2], zc[1], zc[0]]
                        src2 = y if e > 0 else zc
                        links2[i, 2 * mu + j, 2 * nu + k] = U[nu, src2[3], src2[2], src2[1], src2[0]]
    return self_, nbr2, links1, links2


@pytest.mark.parametrize("L,Ls", [((4, 4, 4, 4), 8), ((4, 6, 4, 8), 4)])
@pytest.mark.parametrize("dagger", [False, True])
def test_mpc_site_list_mode(oracle, L, Ls, dagger):
    """mpc_sites (configs[4] parity) equals the pinned full-volume M_pc (dense Schur complement pin,
    test_oracle_dense.py) at EVERY even site, seam and corners included; a mass large enough to make the wall terms count."""
    mass = 0.3
    sites = [(x, y, z, t) for t in range(L[3]) for z in range(L[2]) for y in range(L[1]) for x in range(L[0]) if (x + y + z + t) % 2 == 0]
    U = gen.gauge_random(L, 1000)
    psi_e = gen.keep_parity(gen.spinor_gaussian(L, Ls, 1, 2000), L, 0)
    got = oracle.mpc_sites(L, Ls, M5, mass, np.array(sites, dtype=np.int32), *_gather2(L, U, psi_e, sites), dagger=dagger)
    full = oracle.mpc(U, psi_e, M5, mass, dagger=dagger)[0]
    want = np.stack([full[:, t, z, y, x] for (x, y, z, t) in sites])
    assert rel(got, want) < 1e-14
