"""-m gpu: row f2, Naik-link compression (14 reals: rows 0, 1 and d = det / |row0 x row1|^2; row 2 = conj(row0 x row1) d
rebuilt in registers).  Same oracle, same tolerances as the uncompressed kernel; exact for c x SU(3) (the BASELINE inputs) and
for c x U(3) (the Naik links of the HISQ smearing); links that are neither must fall back to the full format."""
import numpy as np
import pytest
import torch

import oracle
from paper_2306_01098_b200 import binding
from tests.gpu_helpers import make_field, rel_l2, to_full
from tests.helpers import oracle_links

pytestmark = pytest.mark.gpu
TOL = {"fp64": 1e-14, "fp32": 1e-6}


def _ctx(L, prec, nrhs, seed, naik_from_fat=False):
    ctx = binding.Hisq(L, prec, nrhs)
    ctx.set_option("naik_compress", 1)
    fat, naik = binding.make_links(L, seed, ctx.device, ctx.cdtype)
    X, W = oracle_links(L, seed)
    if naik_from_fat:
        naik = fat.clone() * 0.1
        W = X * 0.1
    if prec == "fp32":
        X = X.astype(np.complex64).astype(np.complex128)
        W = W.astype(np.complex64).astype(np.complex128)
    ctx.set_links(fat, naik)
    return ctx, X, W


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
@pytest.mark.parametrize("L,nrhs", [((8, 8, 8, 8), 1), ((4, 6, 8, 10), 3), ((4, 4, 4, 4), 8), ((12, 6, 10, 8), 2)])
def test_compressed_dslash_matches_oracle(L, nrhs, prec):
    ctx, X, W = _ctx(L, prec, nrhs, 0)
    assert ctx.naik_compressed()
    for parity in (0, 1):
        dev_in, full_in = make_field(ctx, L, 5, nrhs, 1 - parity)
        got = to_full(ctx, L, ctx.dslash(dev_in, parity), parity)
        ref = oracle.dslash_parity(L, X, W, full_in, parity)
        for k in range(nrhs):
            assert rel_l2(got[k], ref[k]) <= TOL[prec]
    ctx.close()


def test_naik_only_compressed():
    """The Naik part is ~6 % of the norm: check the reconstructed links on their own."""
    L = (8, 8, 8, 8)
    ctx = binding.Hisq(L, "fp64", 1)
    ctx.set_option("naik_compress", 1)
    fat, naik = binding.make_links(L, 1, ctx.device)
    X, W = oracle_links(L, 1)
    ctx.set_links(torch.zeros_like(fat), naik)
    assert ctx.naik_compressed()
    dev_in, full_in = make_field(ctx, L, 1, 1, 0)
    got = to_full(ctx, L, ctx.dslash(dev_in, 1), 1)
    assert rel_l2(got, oracle.dslash_parity(L, np.zeros_like(X), W, full_in, 1)) <= 1e-14
    ctx.close()


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_non_unitary_naik_links_fall_back_to_full_format(prec):
    L = (4, 6, 4, 8)
    ctx, X, W = _ctx(L, prec, 2, 2, naik_from_fat=True)
    assert not ctx.naik_compressed()
    dev_in, full_in = make_field(ctx, L, 3, 2, 1)
    got = to_full(ctx, L, ctx.dslash(dev_in, 0), 0)
    assert rel_l2(got, oracle.dslash_parity(L, X, W, full_in, 0)) <= TOL[prec]
    ctx.close()


@pytest.mark.parametrize("prec", ["fp64", "mixed"])
def test_cg_with_compressed_links(prec):
    L, m, tol = (8, 8, 8, 8), 0.1, 1e-10
    ctx, X, W = _ctx(L, prec, 2, 4)
    assert ctx.naik_compressed()
    b_dev, b_full = make_field(ctx, L, 4, 2, 0)
    x_dev, info = ctx.cg(b_dev, m, tol)
    x = to_full(ctx, L, x_dev, 0)
    r = b_full - oracle.apply_A(L, X, W, m, x)
    for k in range(2):
        assert np.linalg.norm(r[k]) / np.linalg.norm(b_full[k]) <= tol
    ctx.close()


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_smeared_u3_naik_links_compress(prec):
    """The Naik links hisq_smear makes are products of U(3)-projected links (det = a phase, not 1): the 14-real format
    holds them exactly; the operator on the compressed links matches the oracle on the oracle's smeared links."""
    from oracle import smear as osmear
    from paper_2306_01098_b200 import inputs
    L, seed = (8, 6, 4, 10), 17
    ctx = binding.Hisq(L, prec, 2)
    thin = binding.make_thin_links(L, seed, ctx.device, ctx.cdtype, 0.3)
    fat, naik, W = ctx.smear(thin, fat_scale=0.5, naik_scale=-0.5 / 24.0)
    dets = torch.linalg.det(W.reshape(-1, 3, 3))
    assert float((dets.abs() - 1).abs().max()) < (1e-4 if prec == "fp32" else 1e-12)
    assert float((dets - 1).abs().max()) > 1e-2                       # genuinely U(3), not SU(3)
    ctx.set_option("naik_compress", 1)
    ctx.set_links(fat, naik)
    assert ctx.naik_compressed()
    U = inputs.thin_links(L, seed, torch.arange(inputs.volume(L), dtype=torch.int64), 0.3).numpy()
    if prec == "fp32":
        U = U.astype(np.complex64).astype(np.complex128)
    Xo, No, _ = osmear.hisq_links(L, U, fat_scale=0.5, naik_scale=-0.5 / 24.0)
    for parity in (0, 1):
        dev_in, full_in = make_field(ctx, L, seed, 2, 1 - parity)
        got = to_full(ctx, L, ctx.dslash(dev_in, parity), parity)
        ref = oracle.dslash_parity(L, Xo, No, full_in, parity)
        for k in range(2):
            assert rel_l2(got[k], ref[k]) <= (2e-5 if prec == "fp32" else 1e-12)
    ctx.close()
