"""Host-side index maps of the product (row a1 of SURVEY.md section 8): Eq. (4)/(5) of the paper
 in torch integer ops.  Used by callers to lay out canonical arrays for
hisq_set_links / hisq_spinor_pack.  (The oracle has its own, independent implementation in C.)"""
from __future__ import annotations

from typing import Sequence

import torch


def volume(L: Sequence[int]) -> int:
    return int(L[0]) * int(L[1]) * int(L[2]) * int(L[3])


def check_extents(L: Sequence[int]) -> None:
    if len(L) != 4 or any(int(v) < 4 or int(v) % 2 for v in L):
        raise ValueError(f"extents must be four even numbers >= 4, got {tuple(L)}")


def lex_of_eo(L: Sequence[int], device="cpu") -> torch.Tensor:
    """For every memory index eo in [0, V) (Eq. 4: even sites first), the lexicographic site number
    lex = x + Lx*(y + Ly*(z + Lz*t)).  Inverse of eo(lex) = lex//2 + (V/2)*parity(lex)."""
    check_extents(L)
    V = volume(L)
    Vh = V // 2
    eo = torch.arange(V, dtype=torch.int64, device=device)
    par = (eo >= Vh).to(torch.int64)
    h = eo - par * Vh
    # the two sites sharing h are lex = 2h and 2h+1 (Lx even => same row); pick the one with the right parity
    lex0 = 2 * h
    r = lex0 // L[0]
    y = r % L[1]
    r = r // L[1]
    z = r % L[2]
    t = r // L[2]
    row_par = (y + z + t) & 1          # parity of the site with even x in this row
    return lex0 + (par ^ row_par)


def eo_of_lex(L: Sequence[int], device="cpu") -> torch.Tensor:
    """Eq. (4): memory index of every lexicographic site."""
    check_extents(L)
    V = volume(L)
    lex = torch.arange(V, dtype=torch.int64, device=device)
    x = lex % L[0]
    r = lex // L[0]
    y = r % L[1]
    r = r // L[1]
    z = r % L[2]
    t = r // L[2]
    return lex // 2 + (V // 2) * ((x + y + z + t) & 1)
