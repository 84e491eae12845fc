"""Pins of oracle/smear.py (HISQ link smearing) against what DEFINES the construction: path counts and
free-field weights, the fat7 form factor prod cos^2(q_nu/2) (zero at q_nu = pi), unitarity of the projection, the
cancellation of the O(q^2) error between the two levels (fixes the Lepage weight), the Naik-improved derivative
(9/8, -1/24), gauge covariance, and a brute-force site-by-site walker for the path products.  CPU only."""
import itertools

import numpy as np
import pytest
import torch

from oracle import smear
from paper_2306_01098_b200 import inputs


def _haar_links(L, seed):
    s = torch.arange(inputs.volume(L), dtype=torch.int64)
    return (inputs.naik_links(L, seed, s, False).numpy() * (-24.0)).astype(np.complex128)     # undo the -1/24: SU(3)


def _coords(L):
    Lx, Ly, Lz, Lt = L
    lex = np.arange(Lx * Ly * Lz * Lt)
    return np.stack([lex % Lx, (lex // Lx) % Ly, (lex // (Lx * Ly)) % Lz, lex // (Lx * Ly * Lz)], axis=1)


def test_s1_path_counts_and_free_field_weights():
    kinds = [k for k, _ in smear.smear_paths(2)]
    assert [kinds.count(k) for k in (1, 3, 5, 7, "L")] == [1, 6, 24, 48, 6]
    assert len(set(p for _, p in smear.smear_paths(2))) == 85
    L = (4, 4, 4, 4)
    one = np.broadcast_to(np.eye(3), (256, 4, 3, 3)).astype(np.complex128)
    assert np.allclose(smear.smear(L, one, smear.FAT7), one, atol=1e-15)                 # fat7 is normalised to 1
    assert np.allclose(smear.smear(L, one, smear.FAT7_LEPAGE), 9.0 / 8.0 * one, atol=1e-15)
    assert np.allclose(smear.naik(L, one), one)
    X, N, W = smear.hisq_links(L, one, fold_phases=False)
    assert np.allclose(X, 9.0 / 8.0 * one) and np.allclose(N, -one / 24.0) and np.allclose(W, one)
    # 9/8 sin p - 1/24 sin 3p = p + O(p^5): the improved derivative the two weights are chosen for (PAPER.md:562 has
    # exactly these two hop lengths)
    p = np.array([0.05, 0.1])
    err = 9.0 / 8.0 * np.sin(p) - np.sin(3 * p) / 24.0 - p
    assert abs(err[1] / err[0] - 32.0) < 0.5 and abs(err[0]) < 1e-7


def _linear_response(L, coeff_chain, mu0, n):
    """U = exp(i eps A T), A_mu0(x) = cos(q x), abelian T: returns the measured form factor of the chain of smearings."""
    eps = 1e-6
    c = _coords(L)
    q = 2 * np.pi * np.asarray(n) / np.asarray(L)
    A = np.cos(c @ q)
    T = np.diag([1.0, -1.0, 0.0])
    U = np.broadcast_to(np.eye(3), (len(c), 4, 3, 3)).astype(np.complex128).copy()
    U[:, mu0] = np.eye(3) + 1j * eps * A[:, None, None] * T - 0.5 * eps ** 2 * (A ** 2)[:, None, None] * (T @ T)
    one = np.broadcast_to(np.eye(3), U.shape).astype(np.complex128)
    S, S0 = U, one
    for coeff, project in coeff_chain:
        S, S0 = smear.smear(L, S, coeff), smear.smear(L, S0, coeff)
        if project:
            S, S0 = smear.project_u3(S), smear.project_u3(S0)
    resp = (S[:, mu0] - S0[:, mu0]) / (1j * eps)                       # = f(q) A(x) T + O(eps)
    f = np.einsum("xab,ab->x", resp, T).real / 2.0                     # tr(T T) = 2
    k = np.argmax(np.abs(A))
    return f[k] / A[k], np.abs(f - (f[k] / A[k]) * A).max(), q


@pytest.mark.parametrize("n", [(0, 1, 0, 0), (0, 1, 2, 3), (0, 4, 1, 0), (0, 3, 4, 2), (0, 0, 0, 4)])
def test_s2_fat7_form_factor_is_prod_cos2_half_q(n):
    L, mu0 = (4, 8, 8, 8), 0
    f, spread, q = _linear_response(L, [(smear.FAT7, False)], mu0, n)
    expect = np.prod([np.cos(q[nu] / 2) ** 2 for nu in range(4) if nu != mu0])
    assert abs(f - expect) < 2e-6 and spread < 2e-6
    if 4 in n:
        assert abs(f) < 2e-6                                           # no coupling to a gluon with q_nu = pi


def test_s3_projection_is_the_unitary_polar_factor():
    rng = np.random.default_rng(3)
    V = rng.normal(size=(200, 3, 3)) + 1j * rng.normal(size=(200, 3, 3))
    W = smear.project_u3(V)
    I = np.eye(3)
    assert np.abs(np.conj(np.swapaxes(W, -1, -2)) @ W - I).max() < 1e-12
    H = np.conj(np.swapaxes(W, -1, -2)) @ V                            # must be the Hermitian positive factor
    assert np.abs(H - np.conj(np.swapaxes(H, -1, -2))).max() < 1e-11
    assert np.linalg.eigvalsh(H).min() > 0
    U = _haar_links((4, 4, 4, 4), 1)[:50, 0]
    assert np.abs(smear.project_u3(2.5 * U) - U).max() < 1e-13          # unitary x positive scalar -> the unitary


def test_s4_lepage_weight_cancels_the_q2_error_of_the_two_levels():
    """level 1 (fat7, projected) x level 2 (fat7 + Lepage, WITHOUT the 1/8 that belongs to the Naik term) has the form
    factor 1 + O(q^4): doubling q multiplies the deviation by ~16, not 4; with any other Lepage weight it is O(q^2)."""
    L, mu0 = (4, 32, 4, 4), 0
    lvl2 = dict(smear.FAT7_LEPAGE, c1=smear.FAT7_LEPAGE["c1"] - 1.0 / 8.0)
    dev = []
    for ny in (1, 2):
        f, _, q = _linear_response(L, [(smear.FAT7, True), (lvl2, False)], mu0, (0, ny, 0, 0))
        dev.append(f - 1.0)
    assert abs(dev[0]) < 5e-4 and 12.0 < dev[1] / dev[0] < 20.0, dev
    wrong = dict(lvl2, cL=-1.0 / 16.0, c1=lvl2["c1"] - 6.0 / 16.0)     # asqtad's Lepage weight: leaves level 1's q^2
    f, _, q = _linear_response(L, [(smear.FAT7, True), (wrong, False)], mu0, (0, 1, 0, 0))
    assert abs((f - 1.0) + q[1] ** 2 / 4) < 1e-3 and abs(f - 1.0) > 5e-3


def test_s6_gauge_covariance_of_fat_and_naik_links():
    L = (4, 6, 4, 4)
    U = _haar_links(L, 2)
    g = _haar_links(L, 9)[:, 0]                                        # one SU(3) matrix per site
    c = _coords(L)
    Lx, Ly, Lz, Lt = L
    def at(c2):
        c2 = c2 % np.array(L)
        return c2[:, 0] + Lx * (c2[:, 1] + Ly * (c2[:, 2] + Lz * c2[:, 3]))
    gd = np.conj(np.swapaxes(g, -1, -2))
    Ug = np.empty_like(U)
    for mu in range(4):
        e = np.eye(4, dtype=int)[mu]
        Ug[:, mu] = g @ U[:, mu] @ gd[at(c + e)]
    X, N, W = smear.hisq_links(L, U, fold_phases=False)
    Xg, Ng, Wg = smear.hisq_links(L, Ug, fold_phases=False)
    for mu in range(4):
        e = np.eye(4, dtype=int)[mu]
        assert np.abs(Xg[:, mu] - g @ X[:, mu] @ gd[at(c + e)]).max() < 1e-12
        assert np.abs(Wg[:, mu] - g @ W[:, mu] @ gd[at(c + e)]).max() < 1e-12
        assert np.abs(Ng[:, mu] - g @ N[:, mu] @ gd[at(c + 3 * e)]).max() < 1e-12


def test_s7_path_products_against_a_site_by_site_walker():
    L = (4, 4, 6, 4)
    U = _haar_links(L, 4)
    Lx, Ly, Lz, Lt = L
    lex = lambda c: c[0] % Lx + Lx * (c[1] % Ly + Ly * (c[2] % Lz + Lz * (c[3] % Lt)))
    G = smear._grid(L, U)
    rng = np.random.default_rng(0)
    allp = [p for mu in range(4) for _, p in smear.smear_paths(mu)] + [(1, 1, 1), (4, 4, 4)]
    for steps in [allp[i] for i in rng.choice(len(allp), 12, replace=False)] + [(4, 4, 4), (-3, 2, 3, -2)]:
        P, _ = smear.path_product(G, steps)
        P = P.reshape(-1, 3, 3)
        for site in rng.choice(Lx * Ly * Lz * Lt, 5, replace=False):
            c = [site % Lx, (site // Lx) % Ly, (site // (Lx * Ly)) % Lz, site // (Lx * Ly * Lz)]
            M = np.eye(3, dtype=np.complex128)
            for s in steps:
                d = abs(s) - 1
                if s > 0:
                    M = M @ U[lex(c), d]
                    c[d] += 1
                else:
                    c[d] -= 1
                    M = M @ U[lex(c), d].conj().T
            assert np.abs(M - P[site]).max() < 1e-14


def test_phases_and_scales_are_folded_last():
    L = (4, 4, 4, 6)
    U = _haar_links(L, 5)
    X0, N0, _ = smear.hisq_links(L, U, fold_phases=False)
    X1, N1, _ = smear.hisq_links(L, U, fat_scale=0.5, naik_scale=-0.5 / 24.0, fold_phases=True)
    e = smear.eta_phases(L)
    c = _coords(L)
    assert np.array_equal(e[:, 0], np.ones(len(c))) and np.array_equal(e[:, 3], 1 - 2 * ((c[:, 0] + c[:, 1] + c[:, 2]) & 1))
    assert np.allclose(X1, 0.5 * e[:, :, None, None] * X0) and np.allclose(N1, 0.5 * e[:, :, None, None] * N0)
