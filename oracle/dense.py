"""Brute-force dense matrix of D (pin P7).  TEST INFRASTRUCTURE, NOT PRODUCT.

A third code path, written from PAPER.md:562 + :123 independently of hisq_oracle.c: pure Python
loops over (site, mu, hop, direction) that write 3x3 blocks into a (3V x 3V) complex matrix.
Row index 3*lex(x) + a, column index 3*lex(y) + b.  `+=` everywhere: on an extent-4 direction the
+3 hop and the -1 hop land on the same site and their blocks add (R19).
Only sensible for tiny lattices (4^4: 768 x 768).
"""
from __future__ import annotations

import itertools

import numpy as np


def dense_D(L, X, W) -> np.ndarray:
    Lx, Ly, Lz, Lt = [int(v) for v in L]
    V = Lx * Ly * Lz * Lt
    ext = (Lx, Ly, Lz, Lt)

    def lex(c):
        return c[0] + Lx * (c[1] + Ly * (c[2] + Lz * c[3]))

    D = np.zeros((3 * V, 3 * V), dtype=np.complex128)
    for t, z, y, x in itertools.product(range(Lt), range(Lz), range(Ly), range(Lx)):
        here = (x, y, z, t)
        i = lex(here)
        for mu in range(4):
            for hop, F in ((1, X), (3, W)):
                # forward: + F_mu(x) phi(x + hop mu)
                fwd = list(here)
                fwd[mu] += hop
                s = 1.0
                if fwd[mu] >= ext[mu]:
                    fwd[mu] -= ext[mu]
                    if mu == 3:
                        s = -1.0          # antiperiodic in time
                j = lex(fwd)
                D[3 * i:3 * i + 3, 3 * j:3 * j + 3] += s * F[i, mu]
                # backward: - F_mu(x - hop mu)^dagger phi(x - hop mu)
                bwd = list(here)
                bwd[mu] -= hop
                s = 1.0
                if bwd[mu] < 0:
                    bwd[mu] += ext[mu]
                    if mu == 3:
                        s = -1.0
                j = lex(bwd)
                D[3 * i:3 * i + 3, 3 * j:3 * j + 3] -= s * F[j, mu].conj().T
    return D


def dense_A_even(L, X, W, mass: float):
    """(A_ee, even_rows): A = m^2 - D_eo D_oe as a dense matrix on the even sites;
    even_rows = row numbers (3*lex + a) of D it refers to, ascending."""
    Lx, Ly, Lz, Lt = [int(v) for v in L]
    V = Lx * Ly * Lz * Lt
    D = dense_D(L, X, W)
    lexs = np.arange(V)
    par = (lexs % Lx + (lexs // Lx) % Ly + (lexs // (Lx * Ly)) % Lz + lexs // (Lx * Ly * Lz)) & 1
    rows_e = np.nonzero(np.repeat(par == 0, 3))[0]
    rows_o = np.nonzero(np.repeat(par == 1, 3))[0]
    D_eo = D[np.ix_(rows_e, rows_o)]
    D_oe = D[np.ix_(rows_o, rows_e)]
    A = mass * mass * np.eye(rows_e.size) - D_eo @ D_oe
    return A, rows_e
