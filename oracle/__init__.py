"""CPU oracle for the HISQ Dslash / CG hot path.  TEST INFRASTRUCTURE, NOT PRODUCT.

Thin numpy/ctypes front end of `hisq_oracle.c` (the arithmetic) plus `dense.py` (an independent
brute-force matrix builder used to pin the C code).  Only tests/, `__graft_entry__.smoke()` and
bench.py's `cpu_baseline` / `--impl reference` legs may import this package; nothing under
paper_2306_01098_b200/ does, and this package imports nothing from there.

Conventions (see the header of hisq_oracle.c): full lattice, lexicographic site order
lex = x + Lx*(y + Ly*(z + Lz*t)); links  F[lex, mu, a, b] complex128; fields phi[k, lex, c] complex128.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hisq_oracle.c")
_LIBS = {False: os.path.join(_HERE, "liboracle.so"), True: os.path.join(_HERE, "liboracle_count.so")}
_loaded: dict = {}


def build(force: bool = False) -> None:
    """Compile hisq_oracle.c twice: the normal OpenMP build and the counting build (pin P1)."""
    for counting, lib in _LIBS.items():
        if not force and os.path.exists(lib) and os.path.getmtime(lib) >= os.path.getmtime(_SRC):
            continue
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-Wall", "-o", lib + ".tmp", _SRC, "-lm"]
        cmd[1:1] = ["-DORACLE_COUNT"] if counting else ["-fopenmp"]
        subprocess.run(cmd, check=True)
        os.replace(lib + ".tmp", lib)


def _lib(counting: bool = False) -> ctypes.CDLL:
    if counting not in _loaded:
        build()
        _loaded[counting] = ctypes.CDLL(_LIBS[counting])
    return _loaded[counting]


def _L(L: Sequence[int]):
    return (ctypes.c_int * 4)(*[int(v) for v in L])


def _c(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _links(F, V):
    F = np.ascontiguousarray(F, dtype=np.complex128)
    assert F.shape == (V, 4, 3, 3), F.shape
    return F


def _field(phi, V):
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    if phi.ndim == 2:
        phi = phi[None]
    assert phi.shape[1:] == (V, 3), phi.shape
    return phi


def volume(L) -> int:
    return int(L[0]) * int(L[1]) * int(L[2]) * int(L[3])


def threads() -> int:
    return int(_lib().oracle_threads())


def coords(L) -> np.ndarray:
    """[V, 4] coordinates (x, y, z, t) of every lexicographic site."""
    lex = np.arange(volume(L), dtype=np.int64)
    x = lex % L[0]
    y = (lex // L[0]) % L[1]
    z = (lex // (L[0] * L[1])) % L[2]
    t = lex // (L[0] * L[1] * L[2])
    return np.stack([x, y, z, t], axis=1)


def site_parity(L) -> np.ndarray:
    return (coords(L).sum(axis=1) & 1).astype(np.int64)


def eo_index(L) -> np.ndarray:
    """Eq. (4): memory index of every lexicographic site."""
    out = np.empty(volume(L), dtype=np.int64)
    _lib().oracle_eo_index(_L(L), _c(out))
    return out


def link_index(L) -> np.ndarray:
    """Eq. (5): slot of link (lex, mu); shape [V, 4]."""
    out = np.empty((volume(L), 4), dtype=np.int64)
    _lib().oracle_link_index(_L(L), _c(out))
    return out


def dslash(L, X, W, phi, rows: int = 3, counting: bool = False) -> np.ndarray:
    """(D phi) on the rows (sites) whose parity bit is set in `rows` (3 = full lattice)."""
    V = volume(L)
    X, W, phi = _links(X, V), _links(W, V), _field(phi, V)
    out = np.empty_like(phi)
    _lib(counting).oracle_dslash_rows(_L(L), _c(X), _c(W), _c(phi), _c(out), ctypes.c_int(phi.shape[0]),
                                      ctypes.c_int(rows))
    return out


def dslash_parity(L, X, W, phi, parity: int) -> np.ndarray:
    """D_eo (parity = 0: even outputs from odd inputs) or D_oe (parity = 1)."""
    V = volume(L)
    X, W, phi = _links(X, V), _links(W, V), _field(phi, V)
    out = np.empty_like(phi)
    _lib().oracle_dslash_parity(_L(L), _c(X), _c(W), _c(phi), _c(out), ctypes.c_int(phi.shape[0]),
                                ctypes.c_int(parity))
    return out


def dslash_at(L, X, W, phi, sites) -> np.ndarray:
    """(D phi) at the listed lexicographic sites only: [nrhs, len(sites), 3]."""
    V = volume(L)
    X, W, phi = _links(X, V), _links(W, V), _field(phi, V)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((phi.shape[0], sites.size, 3), dtype=np.complex128)
    _lib().oracle_dslash_at(_L(L), _c(X), _c(W), _c(phi), _c(out), ctypes.c_int(phi.shape[0]), _c(sites),
                            ctypes.c_long(sites.size))
    return out


def apply_A(L, X, W, mass: float, v) -> np.ndarray:
    """A v = m^2 v - D_eo D_oe v on even sites (odd sites of the result are zero)."""
    V = volume(L)
    X, W, v = _links(X, V), _links(W, V), _field(v, V)
    out = np.empty_like(v)
    _lib().oracle_apply_A(_L(L), _c(X), _c(W), ctypes.c_double(mass), _c(v), _c(out), ctypes.c_int(v.shape[0]))
    return out


def cg(L, X, W, mass: float, tol: float, b, max_iter: int = 100000, hist_len: int = 0):
    """Textbook CG on A x_k = b_k, x_0 = 0, stop at ||r|| <= tol ||b||.
    Returns (x, iters[nrhs], true_relres[nrhs], status, resid_hist or None)."""
    V = volume(L)
    X, W, b = _links(X, V), _links(W, V), _field(b, V)
    n = b.shape[0]
    x = np.empty_like(b)
    iters = np.zeros(n, dtype=np.int32)
    relres = np.zeros(n, dtype=np.float64)
    hist = np.full(hist_len, np.nan) if hist_len else None
    st = _lib().oracle_cg(_L(L), _c(X), _c(W), ctypes.c_double(mass), ctypes.c_double(tol), ctypes.c_int(max_iter),
                          _c(b), _c(x), ctypes.c_int(n), _c(iters), _c(relres),
                          _c(hist) if hist_len else None, ctypes.c_int(hist_len))
    return x, iters, relres, int(st), hist


def apply_M(L, X, W, mass: float, phi) -> np.ndarray:
    """M phi = (D + m) phi on the whole lattice (Eq. (1))."""
    V = volume(L)
    X, W, phi = _links(X, V), _links(W, V), _field(phi, V)
    out = np.empty_like(phi)
    _lib().oracle_apply_M(_L(L), _c(X), _c(W), ctypes.c_double(mass), _c(phi), _c(out), ctypes.c_int(phi.shape[0]))
    return out


def solve_M(L, X, W, mass: float, tol: float, b, max_iter: int = 100000):
    """Solve M x_k = b_k on the whole lattice by CG on the normal equations with full-lattice operators only.
    Returns (x, iters[nrhs], relres[nrhs] = ||b - M x|| / ||b||, status)."""
    V = volume(L)
    X, W, b = _links(X, V), _links(W, V), _field(b, V)
    n = b.shape[0]
    x = np.empty_like(b)
    iters = np.zeros(n, dtype=np.int32)
    relres = np.zeros(n, dtype=np.float64)
    st = _lib().oracle_solve_M(_L(L), _c(X), _c(W), ctypes.c_double(mass), ctypes.c_double(tol), ctypes.c_int(max_iter),
                               _c(b), _c(x), ctypes.c_int(n), _c(iters), _c(relres))
    return x, iters, relres, int(st)


def counts_per_site(L, X, W, phi):
    """Pin P1: run the counting build on the full lattice, return per-site
    (flops, link words, vector words, output words)."""
    lib = _lib(True)
    lib.oracle_count_reset()
    dslash(L, X, W, phi, rows=3, counting=True)
    c = (ctypes.c_longlong * 4)()
    lib.oracle_count_get(c)
    V = volume(L) * _field(phi, volume(L)).shape[0]
    return tuple(v / V for v in c)


# ---- moving between the oracle's full-lattice fields and half-lattice (one parity) fields ----

def half_to_full(L, half, parity: int) -> np.ndarray:
    """half[k, h, c] in the order of Eq. (4) restricted to one parity (h = eo - parity*V/2)
    -> full[k, lex, c] with zeros on the other parity."""
    V = volume(L)
    half = np.asarray(half)
    if half.ndim == 2:
        half = half[None]
    eo = eo_index(L)
    sel = np.nonzero(site_parity(L) == parity)[0]
    full = np.zeros((half.shape[0], V, 3), dtype=np.complex128)
    full[:, sel, :] = half[:, eo[sel] - parity * (V // 2), :]
    return full


def full_to_half(L, full, parity: int) -> np.ndarray:
    V = volume(L)
    full = _field(full, V)
    eo = eo_index(L)
    sel = np.nonzero(site_parity(L) == parity)[0]
    half = np.empty((full.shape[0], V // 2, 3), dtype=np.complex128)
    half[:, eo[sel] - parity * (V // 2), :] = full[:, sel, :]
    return half


# ---- sampled evaluation on lattices too large for host arrays -------------------------------------------
def neighbour_sites(L, sites):
    """For lexicographic sites [n]: (plus, minus) each [n, 2, 4] = lex of x +- hop*mu, hop = 1 (f=0), 3 (f=1)."""
    sites = np.asarray(sites, dtype=np.int64)
    c = np.stack([sites % L[0], (sites // L[0]) % L[1], (sites // (L[0] * L[1])) % L[2], sites // (L[0] * L[1] * L[2])], axis=1)
    plus = np.empty((sites.size, 2, 4), dtype=np.int64)
    minus = np.empty((sites.size, 2, 4), dtype=np.int64)
    for f, hop in enumerate((1, 3)):
        for mu in range(4):
            for sign, dst in ((+1, plus), (-1, minus)):
                cc = c.copy()
                cc[:, mu] = (cc[:, mu] + sign * hop) % L[mu]
                dst[:, f, mu] = cc[:, 0] + L[0] * (cc[:, 1] + L[1] * (cc[:, 2] + L[2] * cc[:, 3]))
    return plus, minus, c[:, 3].astype(np.int32)


def dslash_gathered(Lt, t, Ff, Fb, vp, vm) -> np.ndarray:
    """(D phi)(x_i) from pre-fetched operands: Ff, Fb [n,2,4,3,3]; vp, vm [n,2,4,3]; t [n] int32."""
    n = len(t)
    Ff = np.ascontiguousarray(Ff, dtype=np.complex128); Fb = np.ascontiguousarray(Fb, dtype=np.complex128)
    vp = np.ascontiguousarray(vp, dtype=np.complex128); vm = np.ascontiguousarray(vm, dtype=np.complex128)
    t = np.ascontiguousarray(t, dtype=np.int32)
    assert Ff.shape == (n, 2, 4, 3, 3) and Fb.shape == Ff.shape and vp.shape == (n, 2, 4, 3) and vm.shape == vp.shape
    out = np.empty((n, 3), dtype=np.complex128)
    _lib().oracle_dslash_gathered(ctypes.c_int(int(Lt)), ctypes.c_long(n), _c(t), _c(Ff), _c(Fb), _c(vp), _c(vm), _c(out))
    return out
