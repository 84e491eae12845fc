"""Shared test helpers: seeded inputs in the ORACLE's layout (full lattice, lexicographic)."""
import numpy as np
import torch

from paper_2306_01098_b200 import inputs


def lex_sites(L):
    return torch.arange(inputs.volume(L), dtype=torch.int64)


def oracle_links(L, seed, fold_phases=True):
    s = lex_sites(L)
    X = inputs.fat_links(L, seed, s, fold_phases).numpy()
    W = inputs.naik_links(L, seed, s, fold_phases).numpy()
    return X, W


def oracle_field(L, seed, nrhs, parity=None, stream=inputs.STREAM_SOURCE):
    """Gaussian field on the full lattice; parity=0/1 keeps only that parity."""
    s = lex_sites(L)
    phi = inputs.sources(L, seed, s, nrhs, stream=stream).numpy()
    if parity is not None:
        x, y, z, t = inputs.site_coords(L, s)
        par = ((x + y + z + t) & 1).numpy()
        phi[:, par != parity, :] = 0.0
    return phi


def rel_l2(a, b):
    a = np.asarray(a)
    b = np.asarray(b)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))
