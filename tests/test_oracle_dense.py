"""Brute force: the C oracle against dense matrices built from the Kronecker deltas of eq. 2 / eq. 4
(oracle/dense.py, independent numpy code), on tiny lattices; plus the drivers (Chebyshev, CG)
against dense eigendecomposition / dense solve, and scalar closed forms of eq. 23 / L173 / Fig. 2.
"""
import numpy as np
import pytest

import dwf_inputs as gen
from oracle import dense

M5, MASS = 1.8, 0.01


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


def test_dense_gammas_match_oracle(oracle):
    g, g5 = dense.gammas()
    for mu in range(4):
        assert np.array_equal(g[mu], oracle.gamma(mu))
    assert np.array_equal(g5, oracle.gamma(4))


def test_dense_wilson_spectrum_free_field():
    """PAPER.md L69 (4D version): eigenvalues of D_W(M) on unit links are
    M + 4 - sum cos p_mu +- i sqrt(sum sin^2 p_mu), each 2 (spin) x 3 (colour) fold. Pins dense.py."""
    L = (4, 2, 2, 4)
    U = gen.gauge_unit(L)
    M = -1.8
    DW = (M + 4) * np.eye(12 * 64) - 0.5 * dense.dhop_4d(U, L)
    ev = np.linalg.eigvals(DW)
    want = []
    for nx in range(L[0]):
        for ny in range(L[1]):
            for nz in range(L[2]):
                for nt in range(L[3]):
                    p = [2 * np.pi * nx / L[0], 2 * np.pi * ny / L[1], 2 * np.pi * nz / L[2],
                         2 * np.pi * (nt + 0.5) / L[3]]
                    # L=2 directions: forward and backward neighbour coincide; the formula still holds
                    re = M + 4 - sum(np.cos(q) for q in p)
                    im = np.sqrt(sum(np.sin(q) ** 2 for q in p))
                    want += [re + 1j * im] * 6 + [re - 1j * im] * 6
    want = np.array(want)
    key = lambda v: np.lexsort((np.round(v.imag, 8), np.round(v.real, 8)))
    assert np.max(np.abs(ev[key(ev)] - want[key(want)])) < 1e-10


CASES = [((3, 3, 3, 3), 4), ((4, 2, 2, 2), 4), ((4, 4, 2, 2), 2)]


@pytest.mark.parametrize("L,Ls", CASES)
def test_oracle_vs_dense(oracle, L, Ls):
    U = gen.gauge_random(L, 5)
    x = gen.spinor_gaussian(L, Ls, 1, 6)
    V4 = L[0] * L[1] * L[2] * L[3]
    xv = x[0].reshape(-1)
    H4 = dense.dhop_4d(U, L)
    D = dense.ddw_5d(U, L, Ls, M5, MASS)
    G5 = dense.gamma5r5_5d(L, Ls)
    # D_hop (every s slice), D_DW, H_DW, D_PV, true adjoints
    want = (x[0].reshape(Ls, V4 * 12) @ H4.T).reshape(-1)
    assert rel(oracle.dhop(U, x)[0].reshape(-1), want) < 1e-14
    want = (x[0].reshape(Ls, V4 * 12) @ H4.conj()).reshape(-1)
    assert rel(oracle.dhop(U, x, dagger=True)[0].reshape(-1), want) < 1e-14
    assert rel(oracle.ddw(U, x, M5, MASS)[0].reshape(-1), D @ xv) < 1e-14
    assert rel(oracle.ddw(U, x, M5, MASS, dagger=True)[0].reshape(-1), D.conj().T @ xv) < 1e-14
    assert rel(oracle.hdw(U, x, M5, MASS)[0].reshape(-1), G5 @ (D @ xv)) < 1e-14
    assert rel(oracle.dpv(U, x, M5)[0].reshape(-1), dense.ddw_5d(U, L, Ls, M5, 1.0) @ xv) < 1e-14
    # dense-level identities: H hermitian (eq. 6), D^dag = Gamma5 D Gamma5 (R12)
    H = G5 @ D
    assert np.max(np.abs(H - H.conj().T)) < 1e-14
    assert np.max(np.abs(G5 @ D @ G5 - D.conj().T)) < 1e-14
    if all(l % 2 == 0 for l in L):
        e = dense.parity_mask_5d(L, Ls, 0)
        Mpc = dense.schur_even(D, L, Ls)
        xe = gen.keep_parity(x, L, 0)
        got = oracle.mpc(U, xe, M5, MASS)[0].reshape(-1)
        assert rel(got[e], Mpc @ xv[e]) < 1e-13
        assert np.max(np.abs(got[~e])) == 0.0
        got = oracle.mpc(U, xe, M5, MASS, dagger=True)[0].reshape(-1)
        assert rel(got[e], Mpc.conj().T @ xv[e]) < 1e-13
        # M_oo^{-1} against numpy's solve
        o = ~e
        xo = gen.keep_parity(x, L, 1)
        got = oracle.mpp_inv(xo, M5, MASS, 1)[0].reshape(-1)
        assert rel(got[o], np.linalg.solve(D[np.ix_(o, o)], xv[o])) < 1e-13


# ---------------------------------------------------------------- Chebyshev (eq. 23, eq. 34)
def test_chebyshev_scalar_closed_forms():
    """T_n(x) = cos(n acos x) (eq. 23), cosh outside; map endpoints (L173); Fig. 2 caption L256:
    order-500 first pass with lambda_lo = 0.02, lambda_max = 60 enhances low modes by ~1e8."""
    def T_rec(n, x):
        t0, t1 = 1.0, x
        if n == 0:
            return t0
        for _ in range(n - 1):
            t0, t1 = t1, 2 * x * t1 - t0
        return t1
    for n in (0, 1, 5, 64):
        for x in (-1.0, -0.3, 0.0, 0.77, 1.0):
            assert abs(T_rec(n, x) - np.cos(n * np.arccos(x))) < 1e-12
    lo, hi = 0.02, 60.0
    mp = lambda y: 2 * (y - lo) / (hi - lo) - 1
    assert mp(lo) == -1.0 and abs(mp(hi) - 1.0) < 1e-15
    val = abs(T_rec(500, mp(0.0)))
    assert abs(val - np.cosh(500 * np.arccosh(-mp(0.0)))) / val < 1e-9
    assert 1e7 < val < 1e8            # 4.3e7: "10^8" to the order of magnitude (reading R10)


@pytest.mark.parametrize("order", [0, 1, 2, 7, 16])
def test_chebyshev_vs_eigendecomposition(oracle, order):
    L, Ls = (4, 2, 2, 2), 4
    U = gen.gauge_random(L, 5)
    x = gen.spinor_gaussian(L, Ls, 2, 6)
    D = dense.ddw_5d(U, L, Ls, M5, MASS)
    lam, V = np.linalg.eigh(D.conj().T @ D)
    lo, hi = 0.01, 70.0
    xm = 2 * (lam - lo) / (hi - lo) - 1
    assert np.all(np.abs(xm) <= 1)
    Tn = np.cos(order * np.arccos(xm))
    got = oracle.chebyshev(U, x, M5, MASS, order, lo, hi)
    for r in range(2):
        want = V @ (Tn * (V.conj().T @ x[r].reshape(-1)))
        assert rel(got[r].reshape(-1), want) < 1e-12


def test_chebyshev_composition_identity(oracle):
    """T_2n(X) eta = 2 T_n(X) T_n(X) eta - eta ;  config-level sanity: ||T_64 eta|| / ||eta|| ~ 1/sqrt 2."""
    L, Ls = (4, 4, 4, 4), 8
    U = gen.gauge_random(L, 1000)
    x = gen.spinor_gaussian(L, Ls, 1, 2000)
    lo, hi = 0.01, 70.0
    t8 = oracle.chebyshev(U, x, M5, MASS, 8, lo, hi)
    t16 = oracle.chebyshev(U, x, M5, MASS, 16, lo, hi)
    assert rel(2 * oracle.chebyshev(U, t8, M5, MASS, 8, lo, hi) - x, t16) < 1e-13
    t64 = oracle.chebyshev(U, x, M5, MASS, 64, lo, hi)
    ratio = np.linalg.norm(t64) / np.linalg.norm(x)
    assert 0.6 < ratio < 0.8


# ---------------------------------------------------------------- subspace generation (eq. 34-37) and power method (L225)
def test_subspace_vs_eigendecomposition(oracle):
    """phi_k = V T_{k Delta}(2 lam/lam_max - 1) T_m(2 (lam - lam_lo)/(lam_max - lam_lo) - 1) V^dag eta  (eq. 37, R10), with
    lam_lo ABOVE the lowest eigenvalues so that the first pass really amplifies them (cosh branch of eq. 23)."""
    L, Ls = (4, 2, 2, 2), 4
    U = gen.gauge_random(L, 5)
    eta = gen.spinor_gaussian(L, Ls, 1, 7)
    D = dense.ddw_5d(U, L, Ls, M5, MASS)
    lam, V = np.linalg.eigh(D.conj().T @ D)
    lam_max, m, delta, nvec = 1.05 * lam[-1], 9, 3, 4
    lam_lo = lam[len(lam) // 8]                       # 1/8 of the spectrum lies below the low-pass value
    cheb = lambda n, x: np.where(np.abs(x) <= 1, np.cos(n * np.arccos(np.clip(x, -1, 1))),
                                 np.sign(x) ** n * np.cosh(n * np.arccosh(np.maximum(np.abs(x), 1))))
    x1 = 2 * (lam - lam_lo) / (lam_max - lam_lo) - 1
    x2 = 2 * lam / lam_max - 1
    assert x1.min() < -1 and np.all(np.abs(x2) <= 1)
    got = oracle.chebyshev_subspace(U, eta, M5, MASS, m, lam_lo, lam_max, delta, nvec)
    c = V.conj().T @ eta[0].reshape(-1)
    for k in range(nvec):
        want = V @ (cheb(k * delta, x2) * cheb(m, x1) * c)
        assert rel(got[k, 0].reshape(-1), want) < 1e-11
    # the first pass enhances the low modes relative to the band (the point of the filter, L225)
    low = np.abs(V[:, :4].conj().T @ got[0, 0].reshape(-1)) / np.abs(c[:4])
    assert np.all(low > 1.0) and np.all(np.abs(cheb(m, x1[len(lam) // 2:])) <= 1 + 1e-12)


def test_chebyshev_smoother_vs_library_interpolant(oracle):
    """eq. 24-25: c_N vanishes identically (cos(N theta_k) = 0), so the smoother polynomial is THE degree N-1 Chebyshev
    interpolant of 1/y at the N first-kind nodes of [a, b] -- numpy's chebinterpolate, evaluated on the dense spectrum.
    And it is what a smoother should be: S M x ~ x with error max |1 - lam p(lam)| over the spectrum."""
    from numpy.polynomial import chebyshev as npcheb
    L, Ls = (4, 2, 2, 2), 4
    U = gen.gauge_random(L, 5)
    r = gen.spinor_gaussian(L, Ls, 2, 9)
    D = dense.ddw_5d(U, L, Ls, M5, MASS)
    lam, V = np.linalg.eigh(D.conj().T @ D)
    a, b, N = 0.9 * lam[0], 1.1 * lam[-1], 24
    coef = npcheb.chebinterpolate(lambda x: 2.0 / ((b - a) * x + (b + a)), N - 1)
    p = npcheb.chebval(2 * (lam - a) / (b - a) - 1, coef)
    got = oracle.chebyshev_smoother(U, r, M5, MASS, N, a, b)
    for q in range(2):
        want = V @ (p * (V.conj().T @ (D.conj().T @ r[q].reshape(-1))))
        assert rel(got[q].reshape(-1), want) < 1e-11
    x = gen.spinor_gaussian(L, Ls, 1, 10)
    sm = oracle.chebyshev_smoother(U, oracle.ddw(U, x, M5, MASS), M5, MASS, N, a, b)
    eps = np.max(np.abs(1 - lam * p))
    assert rel(sm, x) <= eps * (1 + 1e-9) and eps < 0.9


def test_power_method_converges_to_dense_lambda_max(oracle):
    L, Ls = (4, 2, 2, 2), 4
    U = gen.gauge_random(L, 5)
    v0 = gen.spinor_gaussian(L, Ls, 1, 8)
    D = dense.ddw_5d(U, L, Ls, M5, MASS)
    lam = np.linalg.eigvalsh(D.conj().T @ D)
    hist, v = oracle.power_lambda_max(U, v0, M5, MASS, 200)
    assert np.all(np.diff(hist) > -1e-12 * lam[-1])                 # Rayleigh quotients of a power iteration never decrease
    assert hist[-1] <= lam[-1] * (1 + 1e-12) and hist[-1] > 0.999 * lam[-1]
    # first quotient is the plain Rayleigh quotient of the start vector
    x = v0[0].reshape(-1)
    assert abs(hist[0] - (np.vdot(D @ x, D @ x) / np.vdot(x, x)).real) / hist[0] < 1e-12
    assert 0.1 < np.linalg.norm(v) / np.linalg.norm(v0) < 10        # the iterate stays O(1)


# ---------------------------------------------------------------- CG (eq. 9)
def test_cg_against_dense_solve_and_properties(oracle):
    L, Ls = (4, 2, 2, 2), 4
    U = gen.gauge_random(L, 5)
    b = gen.keep_parity(gen.spinor_gaussian(L, Ls, 1, 6), L, 0)
    D = dense.ddw_5d(U, L, Ls, M5, MASS)
    e = dense.parity_mask_5d(L, Ls, 0)
    Mpc = dense.schur_even(D, L, Ls)
    A = Mpc.conj().T @ Mpc
    bv = b[0].reshape(-1)[e]
    x, hist = oracle.cg_schur(U, b, M5, MASS, 150)
    xs = np.linalg.solve(A, bv)
    assert rel(x[0].reshape(-1)[e], xs) < 1e-9                       # converges to the dense solution
    assert abs(hist[0] - np.vdot(bv, bv).real) < 1e-10 * hist[0]     # r_0 = b for x_0 = 0
    # true residual equals recursive residual; A-norm of the error decreases monotonically
    errA = []
    for k in (5, 10, 20, 40):
        xk, hk = oracle.cg_schur(U, b, M5, MASS, k)
        xv = xk[0].reshape(-1)[e]
        true_r = bv - A @ xv
        assert abs(np.vdot(true_r, true_r).real - hk[k]) < 1e-9 * hk[0]
        assert np.allclose(hk, hist[:k + 1], rtol=1e-12, atol=0)
        ev = xv - xs
        errA.append(np.vdot(ev, A @ ev).real)
    assert all(errA[i + 1] < errA[i] for i in range(len(errA) - 1))
    # restart: continuing from x_k reproduces a converging sequence
    x20, _ = oracle.cg_schur(U, b, M5, MASS, 20)
    x20b, h2 = oracle.cg_schur(U, b, M5, MASS, 130, x0=x20)
    assert rel(x20b[0].reshape(-1)[e], xs) < 1e-9


# ---------------------------------------------------------------- complete red-black solve (Table V)
def test_solve_rb_against_dense_solve(oracle):
    """The red-black solve returns THE solution of D_DW psi = eta: dense numpy solve, and the residual through the pinned ddw."""
    L, Ls = (4, 2, 2, 2), 4
    U = gen.gauge_random(L, 5)
    eta = gen.spinor_gaussian(L, Ls, 1, 11)
    D = dense.ddw_5d(U, L, Ls, M5, MASS)
    want = np.linalg.solve(D, eta[0].reshape(-1))
    psi, iters = oracle.solve_rb(U, eta, M5, MASS, 1e-13, 400)
    assert iters < 400
    assert rel(psi[0].reshape(-1), want) < 1e-9
    assert rel(oracle.ddw(U, psi, M5, MASS), eta) < 1e-10
    loose, it2 = oracle.solve_rb(U, eta, M5, MASS, 1e-3, 400)
    assert it2 < iters and 1e-7 < rel(oracle.ddw(U, loose, M5, MASS), eta) < 1e-1     # the tolerance is what stops it


# ---------------------------------------------------------------- Pauli-Villars preconditioned operator (L101-107)
def test_mpvdag_m_dense_and_half_plane(oracle):
    """D_PV^dag D_DW against the dense product; and the property the paper quotes for it (L105): the half-plane condition,
    i.e. the hermitian part of M_PV^dag M_l is positive definite (while D_DW itself is not: its hermitian part is indefinite... for
    the squared operator the spectrum is real, for this one complex with positive real part)."""
    L, Ls = (4, 2, 2, 2), 4
    U = gen.gauge_random(L, 5)
    x = gen.spinor_gaussian(L, Ls, 1, 12)
    D = dense.ddw_5d(U, L, Ls, M5, MASS)
    Dpv = dense.ddw_5d(U, L, Ls, M5, 1.0)
    A = Dpv.conj().T @ D
    assert rel(oracle.mpvdag_m(U, x, M5, MASS)[0].reshape(-1), A @ x[0].reshape(-1)) < 1e-13
    assert rel(oracle.mpvdag_m(U, x, M5, MASS, dagger=True)[0].reshape(-1), A.conj().T @ x[0].reshape(-1)) < 1e-13
    herm = np.linalg.eigvalsh(0.5 * (A + A.conj().T))
    assert herm[0] > 0                                              # half-plane condition
    ev = np.linalg.eigvals(A)
    assert ev.real.min() > 0 and np.abs(ev.imag).max() > 1e-3       # complex spectrum in the right half plane


# ---------------------------------------------------------------- the other Schur form of Table V (L387)
def test_mpc_alt_against_dense(oracle):
    """1 - M_ee^-1 M_eo M_oo^-1 M_oe from the parity-partitioned dense D_DW; equals M_ee^-1 M_pc (the two forms of Table V
    differ by the left factor M_ee^-1); adjoint = dense conjugate transpose."""
    L, Ls = (4, 2, 2, 2), 4
    U = gen.gauge_random(L, 5)
    x = gen.keep_parity(gen.spinor_gaussian(L, Ls, 1, 13), L, 0)
    D = dense.ddw_5d(U, L, Ls, M5, MASS)
    par = np.broadcast_to(gen.site_parity(L)[None, :, :, :, :, None, None], x[0].shape).reshape(-1)
    e, o = np.where(par == 0)[0], np.where(par == 1)[0]
    Mee, Meo, Moe, Moo = D[np.ix_(e, e)], D[np.ix_(e, o)], D[np.ix_(o, e)], D[np.ix_(o, o)]
    A = np.eye(len(e)) - np.linalg.solve(Mee, Meo @ np.linalg.solve(Moo, Moe))
    xe = x[0].reshape(-1)[e]
    got = oracle.mpc_alt(U, x, M5, MASS)[0].reshape(-1)
    assert rel(got[e], A @ xe) < 1e-12 and np.all(got[o] == 0)
    gotd = oracle.mpc_alt(U, x, M5, MASS, dagger=True)[0].reshape(-1)
    assert rel(gotd[e], A.conj().T @ xe) < 1e-12 and np.all(gotd[o] == 0)
    mpc = oracle.mpc(U, x, M5, MASS)
    assert rel(oracle.mpp_inv(mpc, M5, MASS, 0)[0].reshape(-1)[e], A @ xe) < 1e-12


# ---------------------------------------------------------------- unpreconditioned CGNR (Table V)
def test_cg_normal_against_dense(oracle):
    L, Ls = (4, 2, 2, 2), 4
    U = gen.gauge_random(L, 5)
    b = gen.spinor_gaussian(L, Ls, 1, 14)
    D = dense.ddw_5d(U, L, Ls, M5, MASS)
    A = D.conj().T @ D
    want = np.linalg.solve(A, b[0].reshape(-1))
    x, hist = oracle.cg_normal(U, b, M5, MASS, 300)
    assert rel(x[0].reshape(-1), want) < 1e-8 and hist[-1] < 1e-16 * hist[0]
    # true residual = recursive residual; A-norm of the error decreases monotonically (textbook CG)
    xs = [oracle.cg_normal(U, b, M5, MASS, k)[0][0].reshape(-1) for k in (5, 10, 20, 40)]
    errs = [np.vdot(v - want, A @ (v - want)).real for v in xs]
    assert all(e2 < e1 for e1, e2 in zip(errs, errs[1:]))
    x20, h20 = oracle.cg_normal(U, b, M5, MASS, 20)
    rtrue = b[0].reshape(-1) - A @ x20[0].reshape(-1)
    assert abs(np.vdot(rtrue, rtrue).real - h20[-1]) / h20[-1] < 1e-9



# ---------------------------------------------------------------- BiCGSTAB on M_PV^dag M (Table V, ref. [31])
def test_bicgstab_pv_against_dense_solve(oracle):
    """BiCGSTAB on D_PV^dag D_DW converges to THE solution (numpy solve of the dense product), its recursive residual is the
    true residual, and it needs far fewer applications than its dimension (half-plane spectrum, L105)."""
    L, Ls = (4, 2, 2, 2), 4
    U = gen.gauge_random(L, 5)
    b = gen.spinor_gaussian(L, Ls, 1, 12)
    D = dense.ddw_5d(U, L, Ls, M5, MASS)
    Dpv = dense.ddw_5d(U, L, Ls, M5, 1.0)
    A = Dpv.conj().T @ D
    want = np.linalg.solve(A, b[0].reshape(-1))
    x, hist = oracle.bicgstab_pv(U, b, M5, MASS, 100)
    assert hist[-1] < 1e-24 * hist[0]
    assert rel(x[0].reshape(-1), want) < 1e-10
    # recursive residual == true residual while the iteration is still far from rounding level
    x20, h20 = oracle.bicgstab_pv(U, b, M5, MASS, 20)
    rtrue = b - oracle.mpvdag_m(U, x20, M5, MASS)
    assert abs(np.vdot(rtrue, rtrue).real - h20[-1]) < 1e-8 * h20[-1]
    # restart: 10 + 10 iterations from x_10 is a different Krylov process but must also reduce the true residual
    x10, h10 = oracle.bicgstab_pv(U, b, M5, MASS, 10)
    x10b, h10b = oracle.bicgstab_pv(U, b, M5, MASS, 10, x0=x10)
    assert abs(h10b[0] - h10[-1]) < 1e-8 * h10[-1] and h10b[-1] < h10b[0]
    # the two defining conditions of one step, re-derived here: alpha makes s orthogonal to rhat0 (BiCG), omega is the
    # least-squares minimiser of |s - omega t| (the "STAB" step), so r_1 is orthogonal to t
    r0 = b.copy(); v1 = oracle.mpvdag_m(U, r0, M5, MASS)
    alpha = np.vdot(r0, r0) / np.vdot(r0, v1)
    s = r0 - alpha * v1; t = oracle.mpvdag_m(U, s, M5, MASS)
    omega = np.vdot(t, s) / np.vdot(t, t)
    r1 = s - omega * t
    assert abs(np.vdot(r0, s)) < 1e-12 * np.linalg.norm(r0) * np.linalg.norm(s)
    assert abs(np.vdot(t, r1)) < 1e-12 * np.linalg.norm(t) * np.linalg.norm(s)          # r_1 is orthogonal to t
    _, h1 = oracle.bicgstab_pv(U, b, M5, MASS, 1)
    assert abs(h1[1] - np.vdot(r1, r1).real) < 1e-12 * h1[1]
