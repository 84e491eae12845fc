"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path: each one checks it against a
value the paper prints, a closed form, a structural identity, or an independent brute-force build.
"""
import os

import numpy as np
import pytest
import torch

import oracle
from oracle import dense
from paper_2306_01098_b200 import inputs
from tests.helpers import oracle_field, oracle_links, rel_l2

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden_counts():
    vals = {}
    with open(os.path.join(GOLDEN, "paper_counts.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()
            vals[k] = float(v)
    return vals


# ---------------------------------------------------------------- P1: the paper's printed counts
def test_p1_flop_and_word_counts_match_paper():
    g = _golden_counts()
    L = (4, 4, 6, 8)
    X, W = oracle_links(L, 0)
    phi = oracle_field(L, 0, 2)
    flop, lw, vw, ow = oracle.counts_per_site(L, X, W, phi)
    assert flop == g["flop_per_site"]            # 1146
    assert lw == g["link_words_per_site"]        # 288
    assert vw == g["vector_words_per_site"]      # 96
    assert ow == g["output_words_per_site"]      # 6
    # arithmetic intensities printed at PAPER.md:580
    assert abs(flop / ((lw + vw + ow) * 4) - g["ai_fp32"]) < 0.01
    assert abs(flop / ((lw + vw + ow) * 8) - g["ai_fp64"]) < 0.01


# ---------------------------------------------------------------- P10: index maps Eq. (4)/(5)
@pytest.mark.parametrize("L", [(4, 4, 4, 4), (8, 6, 4, 10), (6, 8, 8, 4)])
def test_p10_index_maps_are_bijections_even_first(L):
    V = oracle.volume(L)
    eo = oracle.eo_index(L)
    par = oracle.site_parity(L)
    assert np.array_equal(np.sort(eo), np.arange(V))
    assert eo[par == 0].max() == V // 2 - 1          # "all even sites in the first half" PAPER.md:433
    assert eo[par == 1].min() == V // 2
    # within one parity the order is the lexicographic one (floor(lex/2) is monotone)
    assert np.all(np.diff(eo[par == 0]) > 0) and np.all(np.diff(eo[par == 1]) > 0)
    slot = oracle.link_index(L)
    assert np.array_equal(np.sort(slot.ravel()), np.arange(4 * V))
    assert np.array_equal(slot[:, 2], eo + 2 * V)
    # spot value written out by hand: site (1,0,0,0) is odd, lex = 1 -> index 0 + V/2
    assert eo[1] == V // 2 and eo[0] == 0 and eo[2] == 1


def test_p10_half_full_roundtrip():
    L = (4, 6, 4, 8)
    rng = np.random.default_rng(1)
    half = rng.normal(size=(2, oracle.volume(L) // 2, 3)) + 0j
    for par in (0, 1):
        full = oracle.half_to_full(L, half, par)
        assert np.all(full[:, oracle.site_parity(L) != par] == 0)
        assert np.array_equal(oracle.full_to_half(L, full, par), half)


# ---------------------------------------------------------------- P2: free field closed form
def _free_links(L, c1, c3):
    sites = torch.arange(oracle.volume(L), dtype=torch.int64)
    eta = inputs.staggered_phase(L, sites).numpy()            # [V,4]
    eye = np.eye(3, dtype=np.complex128)
    X = c1 * eta[:, :, None, None] * eye
    W = c3 * eta[:, :, None, None] * eye
    return X, W, eta


def _plane_wave(L, n, v):
    c = oracle.coords(L).astype(np.float64)
    p = np.array([2 * np.pi * n[0] / L[0], 2 * np.pi * n[1] / L[1], 2 * np.pi * n[2] / L[2],
                  (2 * n[3] + 1) * np.pi / L[3]])              # antiperiodic in t
    phase = np.exp(1j * (c @ p))
    return phase[:, None] * np.asarray(v)[None, :], p


@pytest.mark.parametrize("L,n", [((4, 6, 8, 10), (1, 2, 3, 1)), ((8, 8, 8, 8), (3, 0, 5, 2)),
                                 ((4, 4, 4, 4), (1, 1, 0, 3))])
def test_p2_plane_waves_are_eigenvectors(L, n):
    c1, c3 = 0.625, -1.0 / 24.0
    X, W, eta = _free_links(L, c1, c3)
    v = np.array([0.3 - 0.2j, 1.0 + 0.5j, -0.7j])
    phi, p = _plane_wave(L, n, v)
    out = oracle.dslash(L, X, W, phi)[0]
    lam = (eta * (2j * (c1 * np.sin(p) + c3 * np.sin(3 * p)))[None, :]).sum(axis=1)   # [V]
    assert rel_l2(out, lam[:, None] * phi) < 1e-13
    # even-site restriction is an eigenvector of -D_eo D_oe with sum_mu (2 c1 sin p + 2 c3 sin 3p)^2
    par = oracle.site_parity(L)
    phi_e = phi.copy()
    phi_e[par == 1] = 0
    m = 0.37
    Aphi = oracle.apply_A(L, X, W, m, phi_e)[0]
    ev = m * m + ((2 * c1 * np.sin(p) + 2 * c3 * np.sin(3 * p)) ** 2).sum()
    assert rel_l2(Aphi, ev * phi_e) < 1e-13


# ---------------------------------------------------------------- P3: anti-Hermiticity
def test_p3_antihermitian_with_nonunitary_links():
    L = (4, 6, 8, 10)
    X, W = oracle_links(L, 3)
    phi = oracle_field(L, 3, 1)[0]
    psi = oracle_field(L, 4, 1, stream=inputs.STREAM_AUX)[0]
    Dpsi = oracle.dslash(L, X, W, psi)[0]
    Dphi = oracle.dslash(L, X, W, phi)[0]
    a = np.vdot(phi, Dpsi)
    b = -np.vdot(Dphi, psi)
    assert abs(a - b) / abs(a) < 1e-13
    # hence A is Hermitian and >= m^2
    ve = oracle_field(L, 5, 1, parity=0)[0]
    m = 0.05
    Av = oracle.apply_A(L, X, W, m, ve)[0]
    q = np.vdot(ve, Av)
    assert abs(q.imag) / abs(q.real) < 1e-13
    assert q.real >= m * m * np.vdot(ve, ve).real


# ---------------------------------------------------------------- P4: gauge covariance
def test_p4_gauge_covariance():
    L = (4, 6, 8, 10)
    V = oracle.volume(L)
    X, W = oracle_links(L, 7)
    phi = oracle_field(L, 7, 1)[0]
    g = inputs.gauge_transform(L, 7, torch.arange(V)).numpy()         # [V,3,3]
    assert np.abs(g @ g.conj().transpose(0, 2, 1) - np.eye(3)).max() < 1e-14
    assert np.abs(np.linalg.det(g) - 1).max() < 1e-13
    c = oracle.coords(L)

    def shifted(mu, hop):
        cc = c.copy()
        cc[:, mu] = (cc[:, mu] + hop) % L[mu]
        return cc[:, 0] + L[0] * (cc[:, 1] + L[1] * (cc[:, 2] + L[2] * cc[:, 3]))

    Xg, Wg = np.empty_like(X), np.empty_like(W)
    for mu in range(4):
        g1 = g[shifted(mu, 1)].conj().transpose(0, 2, 1)
        g3 = g[shifted(mu, 3)].conj().transpose(0, 2, 1)
        Xg[:, mu] = g @ X[:, mu] @ g1
        Wg[:, mu] = g @ W[:, mu] @ g3
    lhs = oracle.dslash(L, Xg, Wg, np.einsum("xab,xb->xa", g, phi))[0]
    rhs = np.einsum("xab,xb->xa", g, oracle.dslash(L, X, W, phi)[0])
    assert rel_l2(lhs, rhs) < 1e-13


# ---------------------------------------------------------------- P5: parity structure
def test_p5_D_maps_even_to_odd_exactly():
    L = (4, 6, 8, 10)
    X, W = oracle_links(L, 2)
    par = oracle.site_parity(L)
    for p in (0, 1):
        phi = oracle_field(L, 2, 1, parity=p)
        out = oracle.dslash(L, X, W, phi)[0]
        assert np.all(out[par == p] == 0.0)
        assert np.abs(out[par != p]).min() > 0
        # the parity-restricted entry point gives the same rows
        assert np.array_equal(oracle.dslash_parity(L, X, W, phi, 1 - p)[0], out)
        # ... and ignores whatever sits on the output parity of its input
        junk = phi + oracle_field(L, 9, 1, parity=1 - p)
        assert np.array_equal(oracle.dslash_parity(L, X, W, junk, 1 - p)[0], out)


# ---------------------------------------------------------------- P6: boundary sign == folded links
def _roll_D_periodic(L, X, W, phi):
    """Independent numpy implementation with PERIODIC gathers (np.roll on a [t,z,y,x] grid)."""
    Lx, Ly, Lz, Lt = L
    g = lambda a, tail: a.reshape((Lt, Lz, Ly, Lx) + tail)
    ph = g(phi, (3,))
    axis_of = {0: 3, 1: 2, 2: 1, 3: 0}
    out = np.zeros_like(ph)
    for mu in range(4):
        ax = axis_of[mu]
        for hop, F in ((1, X), (3, W)):
            U = g(F[:, mu], (3, 3))
            fwd = np.roll(ph, -hop, axis=ax)                       # phi(x + hop mu)
            out += np.einsum("...ab,...b->...a", U, fwd)
            Ub = np.roll(U, hop, axis=ax)                          # U(x - hop mu)
            bwd = np.roll(ph, hop, axis=ax)                        # phi(x - hop mu)
            out -= np.einsum("...ba,...b->...a", Ub.conj(), bwd)
    return out.reshape(-1, 3)


@pytest.mark.parametrize("L", [(4, 6, 8, 10), (6, 4, 4, 4), (4, 4, 6, 6)])
def test_p6_antiperiodic_sign_equals_sign_folded_into_boundary_links(L):
    X, W = oracle_links(L, 11)
    phi = oracle_field(L, 11, 1)[0]
    t = oracle.coords(L)[:, 3]
    Xf, Wf = X.copy(), W.copy()
    Xf[t == L[3] - 1, 3] *= -1          # the fat t-link leaving the last slice
    Wf[t >= L[3] - 3, 3] *= -1          # the Naik t-links leaving the last three slices
    ref = _roll_D_periodic(L, Xf, Wf, phi)
    out = oracle.dslash(L, X, W, phi)[0]
    assert rel_l2(out, ref) < 1e-14


# ---------------------------------------------------------------- P7 / P14: dense brute force
@pytest.mark.parametrize("L", [(4, 4, 4, 4), (6, 4, 4, 4), (4, 4, 4, 6)])
def test_p7_dense_matrix_matches_matrix_free(L):
    X, W = oracle_links(L, 5)
    D = dense.dense_D(L, X, W)
    assert np.abs(D + D.conj().T).max() < 1e-15                   # anti-Hermitian
    phi = oracle_field(L, 5, 2)
    for k in range(2):
        ref = (D @ phi[k].reshape(-1)).reshape(-1, 3)
        assert rel_l2(oracle.dslash(L, X, W, phi[k])[0], ref) < 1e-14


def test_p7_dense_solve_matches_cg_and_p12_cg_invariants():
    L = (4, 4, 4, 4)
    m, tol = 0.1, 1e-12
    X, W = oracle_links(L, 6)
    A, rows_e = dense.dense_A_even(L, X, W, m)
    assert np.abs(A - A.conj().T).max() < 1e-14
    assert np.linalg.eigvalsh(A).min() >= m * m * (1 - 1e-10)
    b = oracle_field(L, 6, 2, parity=0)
    x, iters, relres, st, hist = oracle.cg(L, X, W, m, tol, b, hist_len=4096)
    assert st == 0 and np.all(relres < 5 * tol)
    kappa = np.linalg.cond(A)
    for k in range(2):
        xd = np.linalg.solve(A, b[k].reshape(-1)[rows_e])
        assert rel_l2(x[k].reshape(-1)[rows_e], xd) < kappa * tol
        assert np.all(x[k][oracle.site_parity(L) == 1] == 0)
    # reported residual history decreases overall and ends under tol (P12)
    h = hist[: iters[0] + 1]
    assert h[0] == 1.0 and h[-1] <= tol and np.all(np.isfinite(h))
    # A-norm of the error decreases monotonically (textbook CG property), checked by re-running
    # with growing iteration caps against the dense solution
    xd = np.linalg.solve(A, b[0].reshape(-1)[rows_e])
    prev = np.inf
    for cap in (1, 2, 4, 8, 16, 32, 64):
        xc = oracle.cg(L, X, W, m, 1e-30, b[:1], max_iter=cap)[0][0].reshape(-1)[rows_e]
        e = xc - xd
        en = np.vdot(e, A @ e).real
        assert en < prev
        prev = en


# ---------------------------------------------------------------- P8: point source
@pytest.mark.parametrize("src_t", [3, 7, 0])
def test_p8_point_source_columns(src_t):
    L = (8, 8, 8, 8)
    V = oracle.volume(L)
    X, W = oracle_links(L, 8)
    y = np.array([2, 5, 1, src_t])
    lex = lambda c: int(c[0] + L[0] * (c[1] + L[1] * (c[2] + L[2] * c[3])))
    col = 1
    phi = np.zeros((V, 3), dtype=np.complex128)
    phi[lex(y), col] = 1.0
    out = oracle.dslash(L, X, W, phi)[0]
    support = set(np.nonzero(np.abs(out).sum(axis=1))[0].tolist())
    expect = {}
    for mu in range(4):
        for hop, F in ((1, X), (3, W)):
            # receiving site x = y - hop mu sees phi(x + hop mu) through F_mu(x): column `col`
            xm = y.copy(); xm[mu] = (y[mu] - hop) % L[mu]
            s = -1.0 if (mu == 3 and xm[3] + hop >= L[3]) else 1.0
            expect[lex(xm)] = s * F[lex(xm), mu][:, col]
            # receiving site x = y + hop mu sees phi(x - hop mu) through -F_mu(y)^dagger:
            # minus the conjugate of ROW `col` of the link stored at the source
            xp = y.copy(); xp[mu] = (y[mu] + hop) % L[mu]
            s = -1.0 if (mu == 3 and xp[3] - hop < 0) else 1.0
            expect[lex(xp)] = -s * F[lex(y), mu][col, :].conj()
    assert len(expect) == 16 and support == set(expect)
    for site, val in expect.items():
        assert np.abs(out[site] - val).max() == 0.0


# ---------------------------------------------------------------- P9 / P13: linearity, fat-only / Naik-only
def test_p9_p13_separation_and_linearity():
    L = (4, 6, 8, 10)
    X, W = oracle_links(L, 12)
    Z = np.zeros_like(X)
    phi = oracle_field(L, 12, 1)[0]
    full = oracle.dslash(L, X, W, phi)[0]
    fat = oracle.dslash(L, X, Z, phi)[0]
    naik = oracle.dslash(L, Z, W, phi)[0]
    assert rel_l2(fat + naik, full) < 1e-15
    # with these distributions the Naik part is ~5.7 % of the norm: 8/576 vs 8*0.54
    ratio = np.linalg.norm(naik) / np.linalg.norm(full)
    assert 0.04 < ratio < 0.08
    # the Naik-only operator pinned separately against the periodic-roll implementation
    t = oracle.coords(L)[:, 3]
    Wf = W.copy(); Wf[t >= L[3] - 3, 3] *= -1
    assert rel_l2(naik, _roll_D_periodic(L, Z, Wf, phi)) < 1e-14
    psi = oracle_field(L, 13, 1, stream=inputs.STREAM_AUX)[0]
    lin = oracle.dslash(L, X, W, 2.0 * phi - 1j * psi)[0]
    assert rel_l2(lin, 2.0 * full - 1j * oracle.dslash(L, X, W, psi)[0]) < 1e-15


# ---------------------------------------------------------------- P11: CG on a free-field plane wave
def test_p11_cg_free_field_one_iteration():
    L = (4, 6, 8, 8)
    c1, c3, m = 0.625, -1.0 / 24.0, 0.2
    X, W, _ = _free_links(L, c1, c3)
    phi, p = _plane_wave(L, (1, 2, 1, 0), np.array([1.0, 0.5j, -0.25]))
    b = phi.copy()
    b[oracle.site_parity(L) == 1] = 0
    x, iters, relres, st, _ = oracle.cg(L, X, W, m, 1e-12, b[None])
    ev = m * m + ((2 * c1 * np.sin(p) + 2 * c3 * np.sin(3 * p)) ** 2).sum()
    assert st == 0 and iters[0] == 1
    assert rel_l2(x[0], b / ev) < 1e-13


# ---------------------------------------------------------------- dslash_at == rows of the full D
def test_dslash_at_is_a_row_subset():
    L = (4, 6, 8, 10)
    X, W = oracle_links(L, 14)
    phi = oracle_field(L, 14, 2)
    sites = np.array([0, 5, 17, oracle.volume(L) - 1, 333])
    assert np.array_equal(oracle.dslash_at(L, X, W, phi, sites), oracle.dslash(L, X, W, phi)[:, sites])


# ---------------------------------------------------------------- input generator sanity (recipe)
def test_inputs_distributions_and_counter_independence():
    L = (4, 6, 8, 10)
    V = inputs.volume(L)
    s = torch.arange(V, dtype=torch.int64)
    X = inputs.fat_links(L, 0, s, fold_phases=False)
    W = inputs.naik_links(L, 0, s, fold_phases=False)
    assert abs(X.real.std().item() - 0.3) < 3e-3 and abs(X.imag.std().item() - 0.3) < 3e-3
    U = W * (-24.0)
    eye = torch.eye(3, dtype=torch.complex128)
    assert (U @ U.conj().transpose(-1, -2) - eye).abs().max() < 1e-13
    assert (torch.linalg.det(U) - 1).abs().max() < 1e-13
    # any subset, any order, gives the same numbers (counter based)
    perm = torch.randperm(V, generator=torch.Generator().manual_seed(0))[:100]
    assert torch.equal(inputs.fat_links(L, 0, perm, fold_phases=False), X[perm])
    assert torch.equal(inputs.naik_links(L, 0, perm), inputs.naik_links(L, 0, s)[perm])
    src = inputs.sources(L, 0, s, 2)
    assert torch.equal(inputs.sources(L, 0, perm, 2), src[:, perm])
    assert abs(src.real.std().item() - 1.0) < 0.02
    # phases: eta_3 = (-1)^(x+y+z)
    eta = inputs.staggered_phase(L, s)
    x, y, z, t = inputs.site_coords(L, s)
    assert torch.equal(eta[:, 3], (1 - 2 * ((x + y + z) & 1)).double()) and torch.all(eta[:, 0] == 1)
    assert inputs.fat_links(L, 1, s[:10]).ne(inputs.fat_links(L, 0, s[:10])).all()


# ---------------------------------------------------------------- gathered evaluation == rows of D
def test_dslash_gathered_matches_full_lattice_rows():
    L = (4, 6, 8, 4)          # Lt = 4: every t-sign case, coinciding hops
    V = oracle.volume(L)
    X, W = oracle_links(L, 21)
    phi = oracle_field(L, 21, 1)[0]
    sites = np.arange(0, V, 7)
    plus, minus, t = oracle.neighbour_sites(L, sites)
    F = np.stack([X, W], axis=1)                                  # [V, 2, 4, 3, 3]
    f_idx = np.arange(2)[None, :, None]
    mu_idx = np.arange(4)[None, None, :]
    Ff = F[sites][:, :, :]                                        # F_mu(x)
    Fb = F[minus, f_idx, mu_idx]                                  # F_mu(x - hop mu)
    out = oracle.dslash_gathered(L[3], t, Ff, Fb, phi[plus], phi[minus])
    assert np.array_equal(out, oracle.dslash(L, X, W, phi)[0][sites])


# ---------------------------------------------------------------- shifted systems (multi-shift CG's targets)
def test_shifted_system_is_a_mass_shift_dense_check():
    """(A + sigma) = (m^2 + sigma) - D_eo D_oe: the oracle CG at mass sqrt(m^2 + sigma) solves the shifted system;
    pinned against a dense solve of A_ee + sigma on 4^4."""
    L, m, sigma = (4, 4, 4, 4), 0.1, 0.37
    X, W = oracle_links(L, 31)
    A, rows_e = dense.dense_A_even(L, X, W, m)
    b = oracle_field(L, 31, 1, parity=0)
    xd = np.linalg.solve(A + sigma * np.eye(A.shape[0]), b[0].reshape(-1)[rows_e])
    x, _, _, st, _ = oracle.cg(L, X, W, float(np.sqrt(m * m + sigma)), 1e-12, b)
    assert st == 0 and rel_l2(x[0].reshape(-1)[rows_e], xd) < 1e-10


# ---------------------------------------------------------------- P15: the full fermion matrix M = D + m
@pytest.mark.parametrize("L", [(4, 4, 4, 4), (4, 4, 4, 6)])
def test_p15_full_matrix_solve_matches_dense_and_schur_identity(L):
    """oracle.solve_M (full-lattice normal-equation CG) against numpy's dense solve of M = D + m built entry by entry
    (oracle/dense.py); and, in dense algebra only, the even-odd identity the GPU path relies on:
    x_e solves (m^2 - D_eo D_oe) x_e = m b_e - D_eo b_o and x_o = (b_o - D_oe x_e) / m."""
    m, tol = 0.25, 1e-12
    X, W = oracle_links(L, 15)
    D = dense.dense_D(L, X, W)
    n = D.shape[0]
    M = D + m * np.eye(n)
    b = oracle_field(L, 15, 2)
    assert rel_l2(oracle.apply_M(L, X, W, m, b)[1], (M @ b[1].reshape(-1)).reshape(-1, 3)) < 1e-14
    x, iters, relres, st = oracle.solve_M(L, X, W, m, tol, b)
    kappa = np.linalg.cond(M)
    assert st == 0 and np.all(relres < kappa * tol)
    par = np.repeat(oracle.site_parity(L), 3)
    e, o = np.nonzero(par == 0)[0], np.nonzero(par == 1)[0]
    Deo, Doe = D[np.ix_(e, o)], D[np.ix_(o, e)]
    assert np.abs(D[np.ix_(e, e)]).max() == 0 and np.abs(D[np.ix_(o, o)]).max() == 0    # P5 again, on the matrix
    for k in range(2):
        bk = b[k].reshape(-1)
        xd = np.linalg.solve(M, bk)
        assert rel_l2(x[k].reshape(-1), xd) < kappa * kappa * tol
        xe = np.linalg.solve(m * m * np.eye(e.size) - Deo @ Doe, m * bk[e] - Deo @ bk[o])
        xo = (bk[o] - Doe @ xe) / m
        assert rel_l2(xe, xd[e]) < 1e-11 and rel_l2(xo, xd[o]) < 1e-11


def test_p15_free_field_inverse_closed_form():
    """Plane waves are eigenvectors of D with eigenvalue i*lambda(x) = sum_mu eta_mu(x) 2i (c1 sin p + c3 sin 3p), but eta
    depends on the site, so M^{-1} is pinned through M^+ M instead: M^+ M phi = (m^2 + sum_mu (...)^2) phi on the whole
    lattice, hence solve_M(M phi) = phi and solve_M(phi) = M^+ phi / (m^2 + sum)."""
    L = (4, 6, 8, 8)
    c1, c3, m = 0.625, -1.0 / 24.0, 0.3
    X, W, _ = _free_links(L, c1, c3)
    phi, p = _plane_wave(L, (1, 2, 1, 0), np.array([1.0, 0.5j, -0.25]))
    ev = m * m + ((2 * c1 * np.sin(p) + 2 * c3 * np.sin(3 * p)) ** 2).sum()
    x, iters, relres, st = oracle.solve_M(L, X, W, m, 1e-13, phi[None])
    Mdag_phi = m * phi - oracle.dslash(L, X, W, phi)[0]
    assert st == 0 and iters[0] <= 2
    assert rel_l2(x[0], Mdag_phi / ev) < 1e-12
    y = oracle.solve_M(L, X, W, m, 1e-13, oracle.apply_M(L, X, W, m, phi[None]))[0]
    assert rel_l2(y[0], phi) < 1e-12
