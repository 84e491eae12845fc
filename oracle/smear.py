"""HISQ link smearing: thin links U -> fat links X and Naik links N.  TEST INFRASTRUCTURE, NOT PRODUCT.

The paper only says that "X and W are smeared gauge fields", that the fermion action is the HISQ action
of its Ref. [53] and that "the link variable treatment is given in our documentation on GitHub"
(footnote 3) -- none of which is in the container.  What follows is therefore the published HISQ
construction restated from its definition (reading R26), and every coefficient is pinned by a property
the construction is DEFINED to have (tests/test_oracle_smear_pins.py), not by a remembered table:

    level 1   V_mu = F7[U]_mu              fat7 smearing: removes the couplings to gluons of momentum pi/a in any
                                           transverse direction; linearised, its form factor is
                                           prod_{nu != mu} cos^2(q_nu / 2)                        (pins S1, S2)
    project   W_mu = V_mu (V_mu^+ V_mu)^(-1/2)     back to U(3)                                   (pin S3)
    level 2   X_mu = F7L[W]_mu             fat7 + Lepage term with the one-link weight raised so that level 1 x
                                           level 2 has no O(q^2) error and the free-field weight is 9/8  (pins S4, S5)
              N_mu(x) = W_mu(x) W_mu(x+mu) W_mu(x+2mu)      Naik (three-hop) link, weight -1/24 in the operator:
                                           9/8 sin p - 1/24 sin 3p = p + O(p^5), the improved derivative  (pin S5)

A smeared link is a weighted sum over paths from x to x+mu (explicit enumeration below: 1 + 6 + 24 + 48 + 6 paths):
    c1 U_mu(x) + c3 sum_{+-nu} (nu, mu, -nu) + c5 sum (nu, rho, mu, -rho, -nu) + c7 sum (nu, rho, sigma, mu, -sigma, -rho, -nu)
               + cL sum_{+-nu} (nu, nu, mu, -nu, -nu),          nu, rho, sigma distinct and != mu.
A step +nu from y multiplies by U_nu(y) and moves to y+nu; a step -nu multiplies by U_nu(y-nu)^+ and moves to y-nu.
The gauge field is periodic in all four directions.

Storage: U[lex, mu, a, b] complex128 with lex = x + Lx*(y + Ly*(z + Lz*t)), like the rest of the oracle.
Everything is numpy on whole-lattice arrays; np.linalg.eigh is the library primitive of the projection.

Parity unpinned in one respect: that THIS is the construction the paper's code uses is a reading (R26), the paper prints
no formula for it.  The functions themselves are pinned (S1-S7).
"""
from __future__ import annotations

import itertools

import numpy as np

FAT7 = dict(c1=1.0 / 8.0, c3=1.0 / 16.0, c5=1.0 / 64.0, c7=1.0 / 384.0, cL=0.0)
FAT7_LEPAGE = dict(c1=1.0, c3=1.0 / 16.0, c5=1.0 / 64.0, c7=1.0 / 384.0, cL=-1.0 / 8.0)
NAIK = -1.0 / 24.0


def _grid(L, U):
    Lx, Ly, Lz, Lt = [int(v) for v in L]
    return np.ascontiguousarray(U, dtype=np.complex128).reshape(Lt, Lz, Ly, Lx, 4, 3, 3)


def _shift(A, d, n):
    """B(x) = A(x + n * unit vector d); axes of the grid are (t, z, y, x)."""
    return np.roll(A, -n, axis=3 - d)


def path_product(G, steps):
    """P(x) = ordered product of the links along `steps` (signed directions +-(d+1)) starting at x, for every x.
    G: grid [t,z,y,x,mu,3,3]."""
    shape = G.shape[:4]
    P = np.broadcast_to(np.eye(3, dtype=np.complex128), shape + (3, 3)).copy()
    off = [0, 0, 0, 0]                      # current displacement from x
    for s in steps:
        d = abs(s) - 1
        if s > 0:
            link = G[..., d, :, :]
            for e in range(4):
                link = _shift(link, e, off[e])
            P = P @ link
            off[d] += 1
        else:
            off[d] -= 1
            link = G[..., d, :, :]
            for e in range(4):
                link = _shift(link, e, off[e])
            P = P @ np.conj(np.swapaxes(link, -1, -2))
    return P, off


def smear_paths(mu):
    """The paths of one smeared link in direction mu as (kind, steps); kind in {1, 3, 5, 7, 'L'}."""
    m = mu + 1
    others = [d + 1 for d in range(4) if d != mu]
    paths = [(1, (m,))]
    for nu in others:
        for a in (nu, -nu):
            paths.append((3, (a, m, -a)))
            paths.append(("L", (a, a, m, -a, -a)))
    for nu, rho in itertools.permutations(others, 2):
        for a in (nu, -nu):
            for b in (rho, -rho):
                paths.append((5, (a, b, m, -b, -a)))
    for nu, rho, sig in itertools.permutations(others, 3):
        for a in (nu, -nu):
            for b in (rho, -rho):
                for c in (sig, -sig):
                    paths.append((7, (a, b, c, m, -c, -b, -a)))
    return paths


def smear(L, U, coeff) -> np.ndarray:
    """sum over paths of coeff[kind] * (path product), for all four directions.  Returns [V, 4, 3, 3]."""
    G = _grid(L, U)
    out = np.zeros_like(G)
    w = {1: coeff["c1"], 3: coeff["c3"], 5: coeff["c5"], 7: coeff["c7"], "L": coeff["cL"]}
    for mu in range(4):
        for kind, steps in smear_paths(mu):
            if w[kind] == 0.0:
                continue
            P, off = path_product(G, steps)
            assert off == [1 if d == mu else 0 for d in range(4)]
            out[..., mu, :, :] += w[kind] * P
    return out.reshape(-1, 4, 3, 3)


def project_u3(V) -> np.ndarray:
    """W = V (V^+ V)^(-1/2): the unitary factor of the polar decomposition, link by link."""
    V = np.asarray(V, dtype=np.complex128)
    Q = np.conj(np.swapaxes(V, -1, -2)) @ V
    lam, vec = np.linalg.eigh(Q)
    inv_sqrt = (vec * (lam ** -0.5)[..., None, :]) @ np.conj(np.swapaxes(vec, -1, -2))
    return V @ inv_sqrt


def naik(L, W) -> np.ndarray:
    """N_mu(x) = W_mu(x) W_mu(x+mu) W_mu(x+2mu)."""
    G = _grid(L, W)
    out = np.zeros_like(G)
    for mu in range(4):
        out[..., mu, :, :], _ = path_product(G, (mu + 1, mu + 1, mu + 1))
    return out.reshape(-1, 4, 3, 3)


def eta_phases(L) -> np.ndarray:
    """eta_mu(x), [V, 4]: 1, (-1)^x, (-1)^(x+y), (-1)^(x+y+z)   (R7)."""
    Lx, Ly, Lz, Lt = [int(v) for v in L]
    lex = np.arange(Lx * Ly * Lz * Lt)
    x, y, z = lex % Lx, (lex // Lx) % Ly, (lex // (Lx * Ly)) % Lz
    e = np.ones((lex.size, 4))
    e[:, 1] = 1 - 2 * (x & 1)
    e[:, 2] = 1 - 2 * ((x + y) & 1)
    e[:, 3] = 1 - 2 * ((x + y + z) & 1)
    return e


def hisq_links(L, U, fat_scale: float = 1.0, naik_scale: float = NAIK, fold_phases: bool = True):
    """Thin links -> (X, N) ready for the Dslash: X = fat_scale * eta * F7L[W], N = naik_scale * eta * W W W with
    W = project_u3(F7[U]).  Also returns W."""
    W = project_u3(smear(L, U, FAT7))
    X = fat_scale * smear(L, W, FAT7_LEPAGE)
    N = naik_scale * naik(L, W)
    if fold_phases:
        e = eta_phases(L)[:, :, None, None]
        X, N = X * e, N * e
    return X, N, W
