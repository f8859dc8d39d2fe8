"""Brute-force DENSE matrices of the operators, built from the Kronecker deltas of PAPER.md eq. 2
and eq. 4 with numpy.  TEST INFRASTRUCTURE (tiny lattices only): a second, independent statement
of the same definitions, used by tests/test_oracle_dense.py to pin oracle/dwf_oracle.c.
It shares nothing with the C oracle (own gamma construction from Pauli matrices, own indexing)
and nothing with the CUDA path.

Vector index order = canonical flatten of one field: [s][t][z][y][x][spin][colour].
"""
from __future__ import annotations

import numpy as np

_s0 = np.eye(2, dtype=complex)
_sig = [np.array([[0, 1], [1, 0]], dtype=complex),
        np.array([[0, -1j], [1j, 0]], dtype=complex),
        np.array([[1, 0], [0, -1]], dtype=complex)]
_Z = np.zeros((2, 2), dtype=complex)


def gammas():
    """R1: gamma_k = [[0, -i sigma_k], [i sigma_k, 0]], gamma_t = [[0, 1], [1, 0]]; gamma5 = gx gy gz gt."""
    g = [np.block([[_Z, -1j * s], [1j * s, _Z]]) for s in _sig]
    g.append(np.block([[_Z, _s0], [_s0, _Z]]))
    g5 = g[0] @ g[1] @ g[2] @ g[3]
    return g, g5


def _site(L, c):
    Lx, Ly, Lz, Lt = L
    return c[0] + Lx * (c[1] + Ly * (c[2] + Lz * c[3]))


def dhop_4d(U: np.ndarray, L) -> np.ndarray:
    """(V4*12)^2 dense D_hop (eq. 2); antiperiodic in t (R3)."""
    Lx, Ly, Lz, Lt = L
    V4 = Lx * Ly * Lz * Lt
    g, _ = gammas()
    one = np.eye(4, dtype=complex)
    M = np.zeros((V4 * 12, V4 * 12), dtype=complex)
    for t in range(Lt):
        for z in range(Lz):
            for y in range(Ly):
                for x in range(Lx):
                    c = [x, y, z, t]
                    ix = _site(L, c)
                    for mu in range(4):
                        # forward: delta_{x+mu, y}
                        n = list(c); n[mu] += 1
                        sign = 1.0
                        if n[mu] == L[mu]:
                            n[mu] = 0
                            sign = -1.0 if mu == 3 else 1.0
                        iy = _site(L, n)
                        M[ix * 12:(ix + 1) * 12, iy * 12:(iy + 1) * 12] += sign * np.kron(one - g[mu], U[mu, t, z, y, x])
                        # backward: delta_{x-mu, y}, U_mu^dagger(y)
                        n = list(c); n[mu] -= 1
                        sign = 1.0
                        if n[mu] < 0:
                            n[mu] = L[mu] - 1
                            sign = -1.0 if mu == 3 else 1.0
                        iy = _site(L, n)
                        Uy = U[mu, n[3], n[2], n[1], n[0]]
                        M[ix * 12:(ix + 1) * 12, iy * 12:(iy + 1) * 12] += sign * np.kron(one + g[mu], Uy.conj().T)
    return M


def s_matrices(Ls: int, mass: float):
    """The two Ls x Ls coefficient matrices multiplying P_+ and P_- in eq. 4 (off-diagonal part)."""
    Sp = np.zeros((Ls, Ls)); Sm = np.zeros((Ls, Ls))
    for s in range(Ls):
        if s + 1 < Ls:
            Sm[s, s + 1] += -1.0
        if s - 1 >= 0:
            Sp[s, s - 1] += -1.0
    Sp[0, Ls - 1] += mass
    Sm[Ls - 1, 0] += mass
    return Sp, Sm


def ddw_5d(U: np.ndarray, L, Ls: int, M5: float, mass: float) -> np.ndarray:
    """Dense D_DW (eq. 4, eq. 5)."""
    V4 = L[0] * L[1] * L[2] * L[3]
    _, g5 = gammas()
    Pp = 0.5 * (np.eye(4) + g5); Pm = 0.5 * (np.eye(4) - g5)
    Dpar = (5.0 - M5) * np.eye(V4 * 12) - 0.5 * dhop_4d(U, L)
    Sp, Sm = s_matrices(Ls, mass)
    site_Pp = np.kron(np.eye(V4), np.kron(Pp, np.eye(3)))
    site_Pm = np.kron(np.eye(V4), np.kron(Pm, np.eye(3)))
    return np.kron(np.eye(Ls), Dpar) + np.kron(Sp, site_Pp) + np.kron(Sm, site_Pm)


def gamma5r5_5d(L, Ls: int) -> np.ndarray:
    """Dense Gamma5 = gamma5 R5 (L46)."""
    V4 = L[0] * L[1] * L[2] * L[3]
    _, g5 = gammas()
    R = np.zeros((Ls, Ls))
    for s in range(Ls):
        R[s, Ls - 1 - s] = 1.0
    return np.kron(R, np.kron(np.eye(V4), np.kron(g5, np.eye(3))))


def parity_mask_5d(L, Ls: int, parity: int) -> np.ndarray:
    """Boolean mask over the 5D vector index selecting 4D sites of the given parity."""
    Lx, Ly, Lz, Lt = L
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    par = ((x + y + z + t) & 1).reshape(-1)
    m4 = np.repeat(par == parity, 12)
    return np.tile(m4, Ls)


def schur_even(D: np.ndarray, L, Ls: int) -> np.ndarray:
    """M_pc = M_ee - M_eo M_oo^{-1} M_oe from the parity-partitioned dense D (Table V)."""
    e = parity_mask_5d(L, Ls, 0); o = ~e
    Mee = D[np.ix_(e, e)]; Meo = D[np.ix_(e, o)]; Moe = D[np.ix_(o, e)]; Moo = D[np.ix_(o, o)]
    return Mee - Meo @ np.linalg.solve(Moo, Moe)
