"""Seeded synthetic inputs (BASELINE.json configs).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: no Dslash, no checkerboard index map (Eq. 4/5), no boundary condition.
It only turns (seed, stream, counter) into numbers with the distributions the configs ask for.

Generator: counter based.  Value i of stream s under seed S is

    z = splitmix64_finalizer( key(S, s) + (i + 1) * 0x9E3779B97F4A7C15 )     (mod 2^64)

so any subset of sites can be generated in any order, on the CPU or on a GPU, in chunks, and
always gives the same integers.  Uniforms are ((z >> 11) + 0.5) / 2^53, normals are Box-Muller
of the uniform pair (2i, 2i+1).  (log/cos may differ by an ulp between CPU and CUDA libm, so
parity tests always generate on the CPU and copy.)

Counters (all in terms of the LEXICOGRAPHIC site number lex = x + Lx*(y + Ly*(z + Lz*t)),
PAPER.md:433 "site indexing is done in lexicographic order"):
    links   : ((lex*4 + mu)*9 + e)*2 + ri        e = 3*row + col
    spinors : ((k*V + lex)*3 + c)*2 + ri
    gauge g : (lex*9 + e)*2 + ri
The caller says WHICH sites it wants and in which order (`sites`: int64 lexicographic ids);
the result rows follow that order.  The oracle asks for arange(V); the CUDA binding asks for
its own even-odd order.
"""
from __future__ import annotations

import math
from typing import Sequence

import torch

STREAM_FAT, STREAM_NAIK, STREAM_SOURCE, STREAM_GAUGE, STREAM_AUX = 1, 2, 3, 4, 5

_GOLD = 0x9E3779B97F4A7C15
_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB


def _s64(v: int) -> int:
    """Python int (mod 2^64) -> the signed value torch.int64 stores for it."""
    v &= (1 << 64) - 1
    return v - (1 << 64) if v >= (1 << 63) else v


def _lshr(z: torch.Tensor, s: int) -> torch.Tensor:
    """Logical right shift of an int64 tensor (torch's >> is arithmetic)."""
    return (z >> s) & ((1 << (64 - s)) - 1)


def _mix64(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lshr(z, 30)) * _s64(_M1)
    z = (z ^ _lshr(z, 27)) * _s64(_M2)
    return z ^ _lshr(z, 31)


def _mix64_int(z: int) -> int:
    m = (1 << 64) - 1
    z &= m
    z = ((z ^ (z >> 30)) * _M1) & m
    z = ((z ^ (z >> 27)) * _M2) & m
    return z ^ (z >> 31)


def stream_key(seed: int, stream: int) -> int:
    return _mix64_int(_mix64_int(seed * _GOLD + 0x1234567) + stream * _GOLD)


def raw_u64(seed: int, stream: int, counters: torch.Tensor) -> torch.Tensor:
    """The 64 random bits for each counter, as int64 (two's complement)."""
    key = _s64(stream_key(seed, stream))
    return _mix64((counters + 1) * _s64(_GOLD) + key)


def uniforms(seed: int, stream: int, counters: torch.Tensor) -> torch.Tensor:
    z = _lshr(raw_u64(seed, stream, counters), 11)
    return (z.to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normals(seed: int, stream: int, counters: torch.Tensor) -> torch.Tensor:
    """Standard normal for each counter value (Box-Muller on uniforms 2c and 2c+1)."""
    u1 = uniforms(seed, stream, counters * 2)
    u2 = uniforms(seed, stream, counters * 2 + 1)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)


def volume(L: Sequence[int]) -> int:
    return int(L[0]) * int(L[1]) * int(L[2]) * int(L[3])


def site_coords(L: Sequence[int], sites: torch.Tensor):
    """Lexicographic site id -> (x, y, z, t)."""
    x = sites % L[0]
    r = sites // L[0]
    y = r % L[1]
    r = r // L[1]
    z = r % L[2]
    t = r // L[2]
    return x, y, z, t


def staggered_phase(L: Sequence[int], sites: torch.Tensor) -> torch.Tensor:
    """eta_mu(x), shape [len(sites), 4], values +-1.  Kogut-Susskind convention:
    eta_0 = 1, eta_1 = (-1)^x, eta_2 = (-1)^(x+y), eta_3 = (-1)^(x+y+z)."""
    x, y, z, _ = site_coords(L, sites)
    one = torch.ones_like(x)
    e = torch.stack([one, 1 - 2 * (x & 1), 1 - 2 * ((x + y) & 1), 1 - 2 * ((x + y + z) & 1)], dim=1)
    return e.to(torch.float64)


def _complex_gauss(seed, stream, base: torch.Tensor, n_inner: int) -> torch.Tensor:
    """base: int64 tensor of leading counters; returns complex128 [*base.shape, n_inner] where
    element (.., e) uses counters (base*n_inner + e)*2 + {0: re, 1: im}."""
    e = torch.arange(n_inner, dtype=torch.int64, device=base.device)
    c = (base.unsqueeze(-1) * n_inner + e) * 2
    re = normals(seed, stream, c)
    im = normals(seed, stream, c + 1)
    return torch.complex(re, im)


def _chunks(n: int, chunk: int):
    for s in range(0, n, chunk):
        yield s, min(n, s + chunk)


def _su3_from_gaussian(g: torch.Tensor) -> torch.Tensor:
    """[..., 3, 3] complex Gaussian -> SU(3): rows 0, 1 by classical Gram-Schmidt with positive
    normalisation, row 2 = conj(row0 x row1), so the matrix is unitary with det = 1."""
    r0 = g[..., 0, :]
    r0 = r0 / torch.linalg.vector_norm(r0, dim=-1, keepdim=True)
    r1 = g[..., 1, :]
    r1 = r1 - (r0.conj() * r1).sum(-1, keepdim=True) * r0
    r1 = r1 / torch.linalg.vector_norm(r1, dim=-1, keepdim=True)
    r2 = torch.stack([
        r0[..., 1] * r1[..., 2] - r0[..., 2] * r1[..., 1],
        r0[..., 2] * r1[..., 0] - r0[..., 0] * r1[..., 2],
        r0[..., 0] * r1[..., 1] - r0[..., 1] * r1[..., 0],
    ], dim=-1).conj()
    return torch.stack([r0, r1, r2], dim=-2)


def fat_links(L, seed: int, sites: torch.Tensor, fold_phases: bool = True,
              std: float = 0.3, chunk: int = 1 << 18) -> torch.Tensor:
    """Fat links X_mu(x) for the listed sites: complex128 [len(sites), 4, 3, 3].
    Re and Im of every entry i.i.d. N(0, std^2) (non-unitary, like smeared links),
    times eta_mu(x) when fold_phases (BASELINE.json configs: "staggered phases eta_mu folded in")."""
    out = torch.empty((sites.numel(), 4, 3, 3), dtype=torch.complex128, device=sites.device)
    mu = torch.arange(4, dtype=torch.int64, device=sites.device)
    for a, b in _chunks(sites.numel(), chunk):
        s = sites[a:b]
        base = s.unsqueeze(-1) * 4 + mu
        g = _complex_gauss(seed, STREAM_FAT, base, 9).reshape(b - a, 4, 3, 3) * std
        if fold_phases:
            g = g * staggered_phase(L, s).reshape(b - a, 4, 1, 1)
        out[a:b] = g
    return out


def naik_links(L, seed: int, sites: torch.Tensor, fold_phases: bool = True,
               coeff: float = -1.0 / 24.0, chunk: int = 1 << 18) -> torch.Tensor:
    """Naik links W_mu(x): Haar-random SU(3) (Gaussian + Gram-Schmidt, det = 1) times `coeff`
    (BASELINE.json: -1/24) times eta_mu(x).  complex128 [len(sites), 4, 3, 3]."""
    out = torch.empty((sites.numel(), 4, 3, 3), dtype=torch.complex128, device=sites.device)
    mu = torch.arange(4, dtype=torch.int64, device=sites.device)
    for a, b in _chunks(sites.numel(), chunk):
        s = sites[a:b]
        base = s.unsqueeze(-1) * 4 + mu
        g = _complex_gauss(seed, STREAM_NAIK, base, 9).reshape(b - a, 4, 3, 3)
        u = _su3_from_gaussian(g) * coeff
        if fold_phases:
            u = u * staggered_phase(L, s).reshape(b - a, 4, 1, 1)
        out[a:b] = u
    return out


def thin_links(L, seed: int, sites: torch.Tensor, spread: float = 0.0, chunk: int = 1 << 18) -> torch.Tensor:
    """Thin gauge links U_mu(x) in SU(3) for the smearing (row f4): spread = 0: Haar-random (a "hot" configuration);
    spread > 0: Gram-Schmidt of 1 + spread * (complex Gaussian matrix), i.e. links scattered around the identity like
    those of a thermalised configuration (stand-in: no gauge configurations here).  complex128 [len(sites), 4, 3, 3]."""
    if spread == 0.0:
        return naik_links(L, seed, sites, fold_phases=False, coeff=1.0, chunk=chunk)
    out = torch.empty((sites.numel(), 4, 3, 3), dtype=torch.complex128, device=sites.device)
    mu = torch.arange(4, dtype=torch.int64, device=sites.device)
    eye = torch.eye(3, dtype=torch.complex128, device=sites.device)
    for a, b in _chunks(sites.numel(), chunk):
        base = sites[a:b].unsqueeze(-1) * 4 + mu
        g = _complex_gauss(seed, STREAM_NAIK, base, 9).reshape(b - a, 4, 3, 3)
        out[a:b] = _su3_from_gaussian(eye + spread * g)
    return out


def gauge_transform(L, seed: int, sites: torch.Tensor, chunk: int = 1 << 18) -> torch.Tensor:
    """Random g(x) in SU(3) for gauge-covariance checks: complex128 [len(sites), 3, 3]."""
    out = torch.empty((sites.numel(), 3, 3), dtype=torch.complex128, device=sites.device)
    for a, b in _chunks(sites.numel(), chunk):
        g = _complex_gauss(seed, STREAM_GAUGE, sites[a:b], 9).reshape(b - a, 3, 3)
        out[a:b] = _su3_from_gaussian(g)
    return out


def sources(L, seed: int, sites: torch.Tensor, nrhs: int, stream: int = STREAM_SOURCE,
            chunk: int = 1 << 20) -> torch.Tensor:
    """Gaussian colour vectors (Re, Im ~ N(0,1)) on the listed sites: complex128 [nrhs, len(sites), 3]."""
    V = volume(L)
    out = torch.empty((nrhs, sites.numel(), 3), dtype=torch.complex128, device=sites.device)
    for k in range(nrhs):
        for a, b in _chunks(sites.numel(), chunk):
            base = sites[a:b] + k * V
            out[k, a:b] = _complex_gauss(seed, stream, base, 3)
    return out
