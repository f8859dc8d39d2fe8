"""ctypes front-end of the CPU oracle (oracle/dwf_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this module.  It never imports the CUDA package.  All arrays are canonical complex128
(DESIGN.md sec. 3): spinor [nrhs][Ls][t][z][y][x][4][3], gauge [4][t][z][y][x][3][3].
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dwf_oracle.c")
_LIB = os.path.join(_HERE, "libdwf_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, OpenMP over the outer site loop only)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fcx-limited-range", "-fopenmp", "-fPIC", "-shared", "-std=c99",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.oracle_mpp_inv.restype = ctypes.c_int
        _lib.oracle_mpc.restype = ctypes.c_int
        _lib.oracle_cg_schur.restype = ctypes.c_int
    return _lib


def _c(a: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.complex128)


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _L(L):
    return (ctypes.c_int * 4)(*[int(v) for v in L])


def _geom(psi):
    nrhs, Ls, Lt, Lz, Ly, Lx = psi.shape[:6]
    return (Lx, Ly, Lz, Lt), Ls, nrhs


def gamma(mu: int) -> np.ndarray:
    """4x4 gamma_mu (mu=0..3) or gamma5 (mu=4) as used by the oracle (R1)."""
    out = np.zeros((4, 4, 2))
    lib().oracle_gamma(ctypes.c_int(mu), _p(out))
    return out[..., 0] + 1j * out[..., 1]


def dhop(U, psi, row_parity: int = -1, dagger: bool = False) -> np.ndarray:
    """D_hop psi (eq. 2)."""
    psi = _c(psi); U = _c(U); L, Ls, nrhs = _geom(psi)
    out = np.empty_like(psi)
    lib().oracle_dhop(_L(L), ctypes.c_int(Ls), _p(U), _p(psi), _p(out), ctypes.c_int(nrhs),
                      ctypes.c_int(row_parity), ctypes.c_int(int(dagger)))
    return out


def dwilson(U, psi, M: float) -> np.ndarray:
    """D_W(M) psi = (M + 4 - D_hop/2) psi (eq. 1), slice by slice."""
    psi = _c(psi); U = _c(U); L, Ls, nrhs = _geom(psi)
    out = np.empty_like(psi)
    lib().oracle_dwilson(_L(L), ctypes.c_int(Ls), ctypes.c_double(M), _p(U), _p(psi), _p(out),
                         ctypes.c_int(nrhs))
    return out


def ddw(U, psi, M5: float, mass: float, dagger: bool = False) -> np.ndarray:
    """D_DW psi (eq. 4, eq. 5); dagger=True is the true adjoint."""
    psi = _c(psi); U = _c(U); L, Ls, nrhs = _geom(psi)
    out = np.empty_like(psi)
    lib().oracle_ddw(_L(L), ctypes.c_int(Ls), ctypes.c_double(M5), ctypes.c_double(mass), _p(U),
                     _p(psi), _p(out), ctypes.c_int(nrhs), ctypes.c_int(int(dagger)))
    return out


def dpv(U, psi, M5: float, dagger: bool = False) -> np.ndarray:
    """D_PV psi = D_DW at unit mass (L50)."""
    psi = _c(psi); U = _c(U); L, Ls, nrhs = _geom(psi)
    out = np.empty_like(psi)
    lib().oracle_dpv(_L(L), ctypes.c_int(Ls), ctypes.c_double(M5), _p(U), _p(psi), _p(out),
                     ctypes.c_int(nrhs), ctypes.c_int(int(dagger)))
    return out


def mpvdag_m(U, psi, M5: float, mass: float, dagger: bool = False) -> np.ndarray:
    """Pauli-Villars preconditioned operator M_PV^dag M_l = D_PV^dag D_DW; dagger: D_DW^dag D_PV."""
    if dagger:
        return ddw(U, dpv(U, psi, M5), M5, mass, dagger=True)
    return dpv(U, ddw(U, psi, M5, mass), M5, dagger=True)


def gamma5r5(psi) -> np.ndarray:
    """Gamma5 psi = gamma5 R5 psi (L46)."""
    psi = _c(psi); L, Ls, nrhs = _geom(psi)
    out = np.empty_like(psi)
    lib().oracle_gamma5r5(_L(L), ctypes.c_int(Ls), _p(psi), _p(out), ctypes.c_int(nrhs))
    return out


def hdw(U, psi, M5: float, mass: float) -> np.ndarray:
    """H_DW psi = Gamma5 D_DW psi (eq. 6)."""
    psi = _c(psi); U = _c(U); L, Ls, nrhs = _geom(psi)
    out = np.empty_like(psi)
    lib().oracle_hdw(_L(L), ctypes.c_int(Ls), ctypes.c_double(M5), ctypes.c_double(mass), _p(U),
                     _p(psi), _p(out), ctypes.c_int(nrhs))
    return out


def mpp(psi, M5: float, mass: float, parity: int, dagger: bool = False) -> np.ndarray:
    """M_pp psi on sites of `parity` (others 0): the 4D-site-diagonal part of eq. 4."""
    psi = _c(psi); L, Ls, nrhs = _geom(psi)
    out = np.empty_like(psi)
    lib().oracle_mpp(_L(L), ctypes.c_int(Ls), ctypes.c_double(M5), ctypes.c_double(mass), _p(psi),
                     _p(out), ctypes.c_int(nrhs), ctypes.c_int(parity), ctypes.c_int(int(dagger)))
    return out


def mpp_inv(psi, M5: float, mass: float, parity: int, dagger: bool = False) -> np.ndarray:
    """M_pp^{-1} psi by generic dense elimination of the Ls x Ls s-matrix."""
    psi = _c(psi); L, Ls, nrhs = _geom(psi)
    out = np.empty_like(psi)
    rc = lib().oracle_mpp_inv(_L(L), ctypes.c_int(Ls), ctypes.c_double(M5), ctypes.c_double(mass),
                              _p(psi), _p(out), ctypes.c_int(nrhs), ctypes.c_int(parity),
                              ctypes.c_int(int(dagger)))
    if rc != 0:
        raise ZeroDivisionError("M_pp is singular")
    return out


def mpc(U, psi_e, M5: float, mass: float, dagger: bool = False) -> np.ndarray:
    """Schur operator M_pc = M_ee - M_eo M_oo^{-1} M_oe on an even half field (Table V)."""
    psi = _c(psi_e); U = _c(U); L, Ls, nrhs = _geom(psi)
    out = np.empty_like(psi)
    rc = lib().oracle_mpc(_L(L), ctypes.c_int(Ls), ctypes.c_double(M5), ctypes.c_double(mass), _p(U),
                          _p(psi), _p(out), ctypes.c_int(nrhs), ctypes.c_int(int(dagger)))
    if rc != 0:
        raise ZeroDivisionError("M_oo is singular")
    return out


def mpc_alt(U, psi_e, M5: float, mass: float, dagger: bool = False) -> np.ndarray:
    """The other Schur form of Table V (L387): 1 - M_ee^-1 M_eo M_oo^-1 M_oe on an even half field, M_eo = M_oe = -1/2 Dhop
    (eq. 4-5); dagger: the adjoint, factors reversed."""
    psi = _c(psi_e)
    if not dagger:
        t = mpp_inv(-0.5 * dhop(U, psi, row_parity=1), M5, mass, 1)
        return psi - mpp_inv(-0.5 * dhop(U, t, row_parity=0), M5, mass, 0)
    # A^dag = 1 - M_oe^dag (M_oo^dag)^-1 M_eo^dag (M_ee^dag)^-1 ; (Dhop restricted to rows p)^dag maps parity p -> 1-p
    t = mpp_inv(psi, M5, mass, 0, dagger=True)
    t = mpp_inv(-0.5 * dhop(U, t, row_parity=0, dagger=True), M5, mass, 1, dagger=True)
    return psi - (-0.5) * dhop(U, t, row_parity=1, dagger=True)


def chebyshev(U, psi, M5: float, mass: float, order: int, lo: float, hi: float) -> np.ndarray:
    """T_order(2(D^dag D - lo)/(hi-lo) - 1) psi (eq. 23, eq. 34)."""
    psi = _c(psi); U = _c(U); L, Ls, nrhs = _geom(psi)
    out = np.empty_like(psi)
    lib().oracle_chebyshev(_L(L), ctypes.c_int(Ls), ctypes.c_double(M5), ctypes.c_double(mass),
                           _p(U), ctypes.c_int(order), ctypes.c_double(lo), ctypes.c_double(hi),
                           _p(psi), _p(out), ctypes.c_int(nrhs))
    return out


def chebyshev_subspace(U, eta, M5: float, mass: float, m: int, lam_lo: float, lam_max: float, delta: int, nvec: int):
    """Setup option 3 of the paper (L221-241): first-pass filter v = T_m(2(M^dag M - lam_lo)/(lam_max - lam_lo) - 1) eta
    (eq. 34, reading R10) and phi_k = T_{k delta}(2 M^dag M/lam_max - 1) v, k = 0..nvec-1 (eq. 35, 37; phi_0 = v, R23).
    Written as the definition: every phi_k is its own polynomial of the pinned `chebyshev` (the shared recurrence that
    makes them "all for the cost of the highest order" is the GPU path's business).  Returns [nvec, *eta.shape]."""
    v = chebyshev(U, eta, M5, mass, m, lam_lo, lam_max)
    return np.stack([chebyshev(U, v, M5, mass, k * delta, 0.0, lam_max) for k in range(nvec)])


def chebyshev_smoother(U, r, M5: float, mass: float, N: int, a: float, b: float) -> np.ndarray:
    """S r = [c_0/2 + sum_{j=1..N} c_j T_j(2(M^dag M - a)/(b-a) - 1)] M^dag r (eq. 24), c_j by eq. 25 with f(y) = 1/y,
    theta_k = pi (k+1/2)/N; y(x) inverts the interval map of L173.  Term by term through the pinned `chebyshev`."""
    th = np.pi * (np.arange(N) + 0.5) / N
    y = 0.5 * ((b - a) * np.cos(th) + (b + a))
    c = [2.0 / N * np.sum(np.cos(j * th) / y) for j in range(N + 1)]
    v = ddw(U, r, M5, mass, dagger=True)
    out = 0.5 * c[0] * v
    for j in range(1, N + 1):
        out = out + c[j] * chebyshev(U, v, M5, mass, j, a, b)
    return out


def cg_normal(U, b, M5: float, mass: float, iters: int, x0=None):
    """Unpreconditioned CGNR (Table V, eq. 9): Hestenes-Stiefel CG [29] on A = M^dag M, M = D_DW, with the true adjoint;
    one right-hand side.  Returns (x_iters, [|r_k|^2 for k = 0..iters])."""
    b = _c(b)
    A = lambda v: ddw(U, ddw(U, v, M5, mass), M5, mass, dagger=True)
    x = np.zeros_like(b) if x0 is None else _c(x0).copy()
    r = b - A(x)
    p = r.copy()
    rr = float(np.vdot(r, r).real)
    hist = [rr]
    for _ in range(iters):
        Ap = A(p)
        alpha = rr / float(np.vdot(p, Ap).real)
        x = x + alpha * p
        r = r - alpha * Ap
        rr_new = float(np.vdot(r, r).real)
        p = r + (rr_new / rr) * p
        rr = rr_new
        hist.append(rr)
    return x, np.array(hist)


def bicgstab_pv(U, b, M5: float, mass: float, iters: int, x0=None):
    """BiCGSTAB (van der Vorst, PAPER.md ref. [31] L671; the paper does not restate it, L120) on the Pauli-Villars preconditioned
    system A x = b, A = M_PV^dag M = D_PV^dag D_DW (L101-107; Table V), one right-hand side, written out step by step in the
    notation of the original algorithm (unpreconditioned form, rhat_0 = r_0, <a,b> = sum conj(a) b):
        rho_i = <rhat0, r_{i-1}>;  beta = (rho_i/rho_{i-1})(alpha/omega_{i-1});  p_i = r_{i-1} + beta (p_{i-1} - omega_{i-1} v_{i-1});
        v_i = A p_i;  alpha = rho_i/<rhat0, v_i>;  s = r_{i-1} - alpha v_i;  t = A s;  omega_i = <t,s>/<t,t>;
        x_i = x_{i-1} + alpha p_i + omega_i s;  r_i = s - omega_i t.
    Returns (x_iters, [|r_i|^2 for i = 0..iters])."""
    b = _c(b)
    A = lambda f: mpvdag_m(U, f, M5, mass)
    x = np.zeros_like(b) if x0 is None else _c(x0).copy()
    r = b - A(x)
    rhat = r.copy()
    rho_old = alpha = omega = 1.0 + 0.0j
    v = np.zeros_like(b); p = np.zeros_like(b)
    hist = [float(np.vdot(r, r).real)]
    for _ in range(iters):
        rho = np.vdot(rhat, r)
        beta = (rho / rho_old) * (alpha / omega)
        p = r + beta * (p - omega * v)
        v = A(p)
        alpha = rho / np.vdot(rhat, v)
        s = r - alpha * v
        t = A(s)
        omega = np.vdot(t, s) / np.vdot(t, t)
        x = x + alpha * p + omega * s
        r = s - omega * t
        rho_old = rho
        hist.append(float(np.vdot(r, r).real))
    return x, np.array(hist)


def _parity_mask(L, parity: int) -> np.ndarray:
    Lx, Ly, Lz, Lt = L
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return (((x + y + z + t) & 1) == parity)[None, None, :, :, :, :, None, None]


def solve_rb(U, eta, M5: float, mass: float, tol: float, max_iters: int):
    """D_DW psi = eta by the complete red-black solve (Table V, eq. 9), nrhs = 1:
    eta'_e = eta_e - M_eo M_oo^-1 eta_o; CGNR on M_pc^dag M_pc psi_e = M_pc^dag eta'_e from 0, stopped at the FIRST iteration
    k with |r_k| <= tol |r_0| (the textbook rule, tested every iteration; reading R25) or at max_iters;
    psi_o = M_oo^-1 (eta_o - M_oe psi_e); M_eo = M_oe = -1/2 Dhop (eq. 4-5).  Returns (psi, iterations)."""
    eta = _c(eta); L, Ls, _ = _geom(eta)
    me, mo = _parity_mask(L, 0), _parity_mask(L, 1)
    eta_e, eta_o = eta * me, eta * mo
    m_eo = lambda f_o: -0.5 * dhop(U, f_o, row_parity=0)            # onto even sites
    m_oe = lambda f_e: -0.5 * dhop(U, f_e, row_parity=1)            # onto odd sites
    src = eta_e - m_eo(mpp_inv(eta_o, M5, mass, 1))
    b = mpc(U, src, M5, mass, dagger=True)
    _, hist = cg_schur(U, b, M5, mass, max_iters)
    iters = max_iters
    for k in range(1, max_iters + 1):
        if hist[k] <= tol * tol * hist[0]:
            iters = k
            break
    psi_e, _ = cg_schur(U, b, M5, mass, iters)
    psi_o = mpp_inv(eta_o - m_oe(psi_e), M5, mass, 1)
    return psi_e * me + psi_o * mo, iters


def power_lambda_max(U, v0, M5: float, mass: float, iters: int):
    """Power method for lambda_max(M^dag M) (L225; reading R24): u = H v, lambda_i = |u|^2/|v|^2, v <- H u / lambda_i.
    Returns (list of the `iters` Rayleigh quotients, last iterate)."""
    v = _c(v0)
    hist = []
    for _ in range(iters):
        u = hdw(U, v, M5, mass)
        lam = float(np.vdot(u, u).real / np.vdot(v, v).real)
        hist.append(lam)
        v = hdw(U, u, M5, mass) / lam
    return hist, v


def cg_schur(U, b_e, M5: float, mass: float, iters: int, x0=None):
    """`iters` iterations of CG on M_pc^dag M_pc x = b (eq. 9). Returns (x, |r_k|^2 history)."""
    b = _c(b_e); U = _c(U); L, Ls, nrhs = _geom(b)
    assert nrhs == 1
    x = np.zeros_like(b) if x0 is None else _c(x0).copy()
    hist = np.zeros(iters + 1)
    rc = lib().oracle_cg_schur(_L(L), ctypes.c_int(Ls), ctypes.c_double(M5), ctypes.c_double(mass),
                               _p(U), _p(b), _p(x), ctypes.c_int(iters), _p(hist))
    if rc != 0:
        raise ZeroDivisionError("M_oo is singular")
    return x, hist


def inner(x, y) -> np.ndarray:
    """<x,y> = sum conj(x) y per rhs."""
    x = _c(x); y = _c(y); nrhs = x.shape[0]
    out = np.zeros(2 * nrhs)
    lib().oracle_inner(ctypes.c_int64(x[0].size), ctypes.c_int(nrhs), _p(x), _p(y), _p(out))
    return out[0::2] + 1j * out[1::2]


def norm2(x) -> np.ndarray:
    return inner(x, x).real


def axpy(a, x, y) -> np.ndarray:
    """y + a x with one complex a per rhs."""
    x = _c(x); y = _c(y).copy(); nrhs = x.shape[0]
    a = np.asarray(a, dtype=np.complex128).reshape(nrhs)
    ab = np.empty(2 * nrhs); ab[0::2] = a.real; ab[1::2] = a.imag
    lib().oracle_axpy(ctypes.c_int64(x[0].size), ctypes.c_int(nrhs), _p(ab), _p(x), _p(y))
    return y


def ddw_sites(L, Ls: int, M5: float, mass: float, coords, nbr, links) -> np.ndarray:
    """Site-list mode: D_DW rows at sampled 4D sites from gathered neighbourhoods (see .c header)."""
    coords = np.ascontiguousarray(coords, dtype=np.int32)
    n = coords.shape[0]
    nbr = _c(nbr); links = _c(links)
    assert nbr.shape == (n, 9, Ls, 4, 3) and links.shape == (n, 8, 3, 3)
    out = np.empty((n, Ls, 4, 3), dtype=np.complex128)
    lib().oracle_ddw_sites(_L(L), ctypes.c_int(Ls), ctypes.c_double(M5), ctypes.c_double(mass),
                           ctypes.c_int64(n), _p(coords), _p(nbr), _p(links), _p(out))
    return out


def mpc_sites(L, Ls: int, M5: float, mass: float, coords, self_, nbr2, links1, links2, dagger: bool = False) -> np.ndarray:
    """Site-list mode: rows of M_pc (Table V) at sampled EVEN 4D sites from gathered neighbourhoods (see .c header)."""
    coords = np.ascontiguousarray(coords, dtype=np.int32)
    n = coords.shape[0]
    self_ = _c(self_); nbr2 = _c(nbr2); links1 = _c(links1); links2 = _c(links2)
    assert self_.shape == (n, Ls, 4, 3) and nbr2.shape == (n, 8, 8, Ls, 4, 3)
    assert links1.shape == (n, 8, 3, 3) and links2.shape == (n, 8, 8, 3, 3)
    assert np.all(coords.sum(axis=1) % 2 == 0), "M_pc lives on even sites (R8)"
    out = np.empty((n, Ls, 4, 3), dtype=np.complex128)
    rc = lib().oracle_mpc_sites(_L(L), ctypes.c_int(Ls), ctypes.c_double(M5), ctypes.c_double(mass), ctypes.c_int64(n),
                                _p(coords), _p(self_), _p(nbr2), _p(links1), _p(links2), _p(out), ctypes.c_int(int(dagger)))
    if rc != 0:
        raise RuntimeError("oracle_mpc_sites: singular M_oo")
    return out
