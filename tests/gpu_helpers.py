"""Helpers of the -m gpu parity tests: same seeded inputs to the CUDA path (through the C ABI) and to the oracle."""
import numpy as np
import torch

import oracle
from paper_2306_01098_b200 import binding, inputs, layout
from tests.helpers import oracle_links, rel_l2  # noqa: F401


def make_ctx(L, prec, nrhs_max, seed, fat_only=False, naik_only=False):
    """Returns (ctx, X, W): ctx with links set; X, W the oracle's (lexicographic) copies of the SAME links
    (for fp32: rounded to fp32 and widened, so the comparison isolates arithmetic error)."""
    ctx = binding.Hisq(L, prec, nrhs_max)
    fat, naik = binding.make_links(L, seed, ctx.device, ctx.cdtype)
    X, W = oracle_links(L, seed)
    if fat_only:
        naik.zero_(); W = np.zeros_like(W)
    if naik_only:
        fat.zero_(); X = np.zeros_like(X)
    if prec == "fp32":
        X = X.astype(np.complex64).astype(np.complex128)
        W = W.astype(np.complex64).astype(np.complex128)
    ctx.set_links(fat, naik)
    return ctx, X, W


def make_field(ctx, L, seed, nrhs, parity):
    """(native device tensor, oracle full-lattice array) of the same Gaussian field on one parity."""
    can = binding.make_sources(L, seed, nrhs, parity, ctx.device, ctx.cdtype)
    full = oracle.half_to_full(L, can.cpu().numpy().astype(np.complex128), parity)
    return ctx.pack(can), full


def to_full(ctx, L, native, parity):
    can = ctx.unpack(native).cpu().numpy().astype(np.complex128)
    return oracle.half_to_full(L, can, parity)
