"""-m gpu: hisq_smear (recursive staples + Newton polar projection on the GPU, canonical layout) against oracle/smear.py
(explicit enumeration of the 85 paths + eigh projection): element by element on the fat links, the projected links and
the Naik links, then end to end -- smear, hisq_set_links, hisq_dslash -- against the oracle operator on the oracle's
smeared links.  SURVEY 8(f) row f4."""
import numpy as np
import pytest
import torch

import oracle
from oracle import smear as osmear
from paper_2306_01098_b200 import binding, inputs, layout
from tests.gpu_helpers import make_field, rel_l2, to_full

pytestmark = pytest.mark.gpu


def _thin(L, seed, spread, ctx):
    thin = binding.make_thin_links(L, seed, ctx.device, ctx.cdtype, spread)
    s = torch.arange(inputs.volume(L), dtype=torch.int64)
    U = inputs.thin_links(L, seed, s, spread).numpy()                   # the oracle's copy: lexicographic [V, 4, 3, 3]
    if ctx.cdtype == torch.complex64:
        U = U.astype(np.complex64).astype(np.complex128)
    return thin, U


def _to_lex(L, canonical):
    """canonical [4, V(eo), 3, 3] device tensor -> oracle order [V(lex), 4, 3, 3]"""
    eo = layout.eo_of_lex(L).numpy()
    return canonical.cpu().numpy().astype(np.complex128)[:, eo].transpose(1, 0, 2, 3)


@pytest.mark.parametrize("L,prec,spread,tol", [
    ((4, 4, 4, 4), "fp64", 0.0, 1e-12),        # hot configuration, smallest lattice: every hop wraps
    ((8, 6, 4, 10), "fp64", 0.3, 1e-13),       # ragged extents, links near the identity
    ((6, 8, 8, 4), "fp64", 0.0, 1e-12),
    ((8, 8, 8, 8), "fp32", 0.3, 2e-5),
])
def test_smear_matches_oracle(L, prec, spread, tol):
    ctx = binding.Hisq(L, prec, 1)
    thin, U = _thin(L, 11, spread, ctx)
    keep = thin.clone()
    fat, naik, W = ctx.smear(thin, fat_scale=0.5, naik_scale=-0.5 / 24.0, fold_phases=True)
    assert torch.equal(thin, keep)
    Xo, No, Wo = osmear.hisq_links(L, U, fat_scale=0.5, naik_scale=-0.5 / 24.0, fold_phases=True)
    for got, ref in ((W, Wo), (fat, Xo), (naik, No)):
        got = _to_lex(L, got)
        assert rel_l2(got, ref) <= tol
        assert np.abs(got - ref).max() <= 50 * tol * np.abs(ref).max()
    # W is unitary (U(3)); the Naik link is a product of three of them
    Wl = _to_lex(L, W)
    eps = 1e-5 if prec == "fp32" else 1e-13
    assert np.abs(np.conj(np.swapaxes(Wl, -1, -2)) @ Wl - np.eye(3)).max() < eps
    ctx.close()


def test_smear_unphased_and_unit_gauge_closed_form():
    L = (4, 6, 4, 8)
    ctx = binding.Hisq(L, "fp64", 1)
    V = inputs.volume(L)
    one = torch.eye(3, dtype=torch.complex128, device=ctx.device).expand(4, V, 3, 3).contiguous()
    fat, naik, W = ctx.smear(one, fat_scale=1.0, naik_scale=-1.0 / 24.0, fold_phases=False)
    assert torch.allclose(fat, 9.0 / 8.0 * one, atol=1e-15, rtol=0) and torch.allclose(naik, -one / 24.0, atol=1e-16, rtol=0)
    assert torch.allclose(W, one, atol=1e-15, rtol=0)
    # a singular level-1 link has no unitary factor: reported, not silently passed on
    zero = torch.zeros_like(one)
    with pytest.raises(binding.HisqError):
        ctx.smear(zero)
    ctx.close()


def test_smear_then_dslash_end_to_end():
    L, seed = (8, 8, 8, 8), 12
    ctx = binding.Hisq(L, "fp64", 2)
    thin, U = _thin(L, seed, 0.3, ctx)
    fat, naik, _ = ctx.smear(thin, fat_scale=0.5, naik_scale=-0.5 / 24.0)
    ctx.set_links(fat, naik)
    Xo, No, _ = osmear.hisq_links(L, U, fat_scale=0.5, naik_scale=-0.5 / 24.0)
    for parity in (0, 1):
        phi_dev, phi_full = make_field(ctx, L, seed, 2, 1 - parity)
        out = to_full(ctx, L, ctx.dslash(phi_dev, parity), parity)
        ref = oracle.dslash_parity(L, Xo, No, phi_full, parity)
        for k in range(2):
            assert rel_l2(out[k], ref[k]) <= 1e-12
    ctx.close()


def test_smear_full_size_lattice_tiled_configuration():
    """C2's lattice (32^3x8, the size bench.py times the smearing on): the thin field is a periodic tiling of a 16x8x4x8
    configuration, so -- smearing being local and the gauge field periodic -- every smeared field must be the same tiling
    of the small lattice's, which the oracle can afford (the whole-lattice oracle takes 9 minutes at this size)."""
    L, tile, seed = (32, 32, 32, 8), (16, 8, 4, 8), 13
    ctx = binding.Hisq(L, "fp64", 1)
    s = torch.arange(inputs.volume(tile), dtype=torch.int64)
    Us = inputs.thin_links(tile, seed, s, 0.3).numpy()                       # [Vs(lex), 4, 3, 3]
    lex_big = layout.lex_of_eo(L).numpy()                                   # eo -> lex on the big lattice
    c = [lex_big % L[0], (lex_big // L[0]) % L[1], (lex_big // (L[0] * L[1])) % L[2], lex_big // (L[0] * L[1] * L[2])]
    small = (c[0] % tile[0]) + tile[0] * ((c[1] % tile[1]) + tile[1] * ((c[2] % tile[2]) + tile[2] * (c[3] % tile[3])))
    thin = torch.from_numpy(np.ascontiguousarray(Us[small].transpose(1, 0, 2, 3))).to(ctx.device)
    fat, naik, W = ctx.smear(thin, fat_scale=0.5, naik_scale=-0.5 / 24.0, fold_phases=True)
    Xo, No, Wo = osmear.hisq_links(tile, Us, fat_scale=0.5, naik_scale=-0.5 / 24.0, fold_phases=True)
    # (the phases are periodic under the tiling too: every tile extent is even)
    for got, ref in ((W, Wo), (fat, Xo), (naik, No)):
        ref_big = ref[small].transpose(1, 0, 2, 3)
        assert rel_l2(got.cpu().numpy(), ref_big) <= 1e-13
    ctx.close()


def test_configuration_file_to_smeared_links(tmp_path):
    """NERSC file -> hisq_nersc_read (host) -> device -> hisq_smear: the same bits as smearing the links directly."""
    L = (4, 6, 4, 8)
    ctx = binding.Hisq(L, "fp64", 1)
    thin = binding.make_thin_links(L, 14, ctx.device, ctx.cdtype, 0.3)
    path = str(tmp_path / "cfg.nersc")
    binding.nersc_write(path, thin, L, rows=3)
    assert binding.nersc_info(path)["L"] == L
    again = binding.nersc_read(path).to(ctx.device)
    assert torch.equal(again, thin)
    a, b = ctx.smear(thin), ctx.smear(again)
    for u, v in zip(a, b):
        assert torch.equal(u, v)
    ctx.close()
