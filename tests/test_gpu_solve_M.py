"""-m gpu: hisq_solve_M, the full staggered system (D + m) x = b on both parities (Eq. (1); SURVEY 8(f) row
f4: odd-site reconstruction x_o = (b_o - D_oe x_e) / m and the full M solve), against the oracle's full-lattice
normal-equation CG, which uses no even-odd decomposition (pinned by a dense solve of M: tests/test_oracle_pins.py P15)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2306_01098_b200 import binding
from tests.gpu_helpers import make_ctx, make_field, rel_l2, to_full

pytestmark = pytest.mark.gpu


def _solve_and_check(L, prec, nrhs, seed, m, tol, slack=0.0):
    ctx, X, W = make_ctx(L, prec, nrhs, seed)
    be_dev, be_full = make_field(ctx, L, seed, nrhs, 0)
    bo_dev, bo_full = make_field(ctx, L, seed, nrhs, 1)
    b_full = be_full + bo_full                       # one Gaussian field on the whole lattice
    be_keep, bo_keep = be_dev.clone(), bo_dev.clone()
    xe_dev, xo_dev, info = ctx.solve_M(be_dev, bo_dev, m, tol)
    assert torch.equal(be_dev, be_keep) and torch.equal(bo_dev, bo_keep)      # inputs untouched
    x = to_full(ctx, L, xe_dev, 0) + to_full(ctx, L, xo_dev, 1)
    # the contract: ||b - M x|| <= tol ||b|| on the whole lattice, judged by the ORACLE's M
    r = b_full - oracle.apply_M(L, X, W, m, x)
    for k in range(nrhs):
        rel = float(np.linalg.norm(r[k]) / np.linalg.norm(b_full[k]))
        assert rel <= tol + slack, (k, rel)
        assert info["true_rel_resid"][k] <= tol
        assert abs(info["true_rel_resid"][k] - rel) <= 0.05 * tol + slack      # the reported ratio IS the full-lattice one
    # the odd residual vanishes by construction (to rounding): everything sits on the even sites
    par = oracle.site_parity(L)
    eps = 1e-6 if prec == "fp32" else 1e-14
    assert np.linalg.norm(r[:, par == 1]) <= 50 * eps * np.linalg.norm(b_full)
    # solution against the oracle's independent solve: sigma_min(M) = m, so ||x - x*|| <= ||r|| / m for both
    xo, it_o, rel_o, st = oracle.solve_M(L, X, W, m, min(tol, 1e-10) * 1e-2, b_full)
    assert st == 0
    for k in range(nrhs):
        bound = (tol + slack + float(rel_o[k])) * np.linalg.norm(b_full[k]) / m
        assert np.linalg.norm(x[k] - xo[k]) <= 1.01 * bound
    ctx.close()
    return info


def test_solve_M_config1_8x8x8x8_fp64():
    info = _solve_and_check((8, 8, 8, 8), "fp64", 1, 0, 0.1, 1e-10)
    assert info["iterations"] > 50


def test_solve_M_ragged_multi_rhs_fp64():
    _solve_and_check((4, 6, 8, 10), "fp64", 3, 4, 0.2, 1e-9)


def test_solve_M_mixed_precision():
    info = _solve_and_check((8, 8, 8, 8), "mixed", 2, 5, 0.05, 1e-9)
    assert info["reliable_updates"] >= 1


def test_solve_M_fp32():
    # an fp32 residual is itself only known to the Dslash tolerance (2e-5 relative, north_star)
    _solve_and_check((8, 8, 8, 8), "fp32", 2, 6, 0.2, 1e-4, slack=2e-5)


def test_solve_M_even_source_reduces_to_cg_and_rejects_bad_arguments():
    L, m, tol = (8, 8, 8, 8), 0.1, 1e-10
    ctx, X, W = make_ctx(L, "fp64", 1, 7)
    be, _ = make_field(ctx, L, 7, 1, 0)
    bo = torch.zeros_like(be)
    xe, xo, _ = ctx.solve_M(be, bo, m, tol)
    xc, _ = ctx.cg(be, m, tol * 0.1)
    # b_o = 0: s_e = m b_e, x_e = m A^{-1} b_e, x_o = -D_oe x_e / m
    assert rel_l2(xe.cpu().numpy(), m * xc.cpu().numpy()) <= 100 * tol
    assert rel_l2(xo.cpu().numpy(), (-ctx.dslash(xe, 1) / m).cpu().numpy()) <= 1e-14
    lib, p = ctx.lib, lambda t: t.data_ptr()
    assert lib.hisq_solve_M(ctx._h, p(xe), p(xo), p(be), p(bo), 0.0, tol, 1) == binding.HISQ_EINVAL      # mass = 0
    assert lib.hisq_solve_M(ctx._h, p(xe), p(xe), p(be), p(bo), m, tol, 1) == binding.HISQ_EINVAL        # x_e aliases x_o
    assert lib.hisq_solve_M(ctx._h, p(xe), p(bo), p(be), p(bo), m, tol, 1) == binding.HISQ_EINVAL        # x_o aliases b_o
    two = [torch.zeros(2, 3, ctx.Vh, dtype=ctx.cdtype, device=ctx.device) for _ in range(4)]
    assert lib.hisq_solve_M(ctx._h, *[p(t) for t in two], m, tol, 2) == binding.HISQ_ENOWORKSPACE        # sized for 1
    ctx.close()


def test_thin_links_to_propagator_pipeline():
    """The whole chain a user runs: thin SU(3) links -> hisq_smear -> hisq_set_links -> hisq_solve_M, judged by the oracle's
    M = D + m built from the ORACLE's smeared links (oracle/smear.py), i.e. two independent implementations end to end."""
    from oracle import smear as osmear
    from paper_2306_01098_b200 import inputs
    L, seed, m, tol = (8, 8, 8, 8), 21, 0.05, 1e-9
    ctx = binding.Hisq(L, "fp64", 2)
    thin = binding.make_thin_links(L, seed, ctx.device, ctx.cdtype, 0.3)
    fat, naik, _ = ctx.smear(thin, fat_scale=0.5, naik_scale=-0.5 / 24.0)
    ctx.set_links(fat, naik)
    U = inputs.thin_links(L, seed, torch.arange(inputs.volume(L), dtype=torch.int64), 0.3).numpy()
    Xo, No, _ = osmear.hisq_links(L, U, fat_scale=0.5, naik_scale=-0.5 / 24.0)
    be_dev, be_full = make_field(ctx, L, seed, 2, 0)
    bo_dev, bo_full = make_field(ctx, L, seed, 2, 1)
    b_full = be_full + bo_full
    xe, xo, info = ctx.solve_M(be_dev, bo_dev, m, tol)
    x = to_full(ctx, L, xe, 0) + to_full(ctx, L, xo, 1)
    r = b_full - oracle.apply_M(L, Xo, No, m, x)
    for k in range(2):
        assert np.linalg.norm(r[k]) <= tol * np.linalg.norm(b_full[k]) * 1.001
    # smeared links are close to unitary x 9/8 * 1/2: the spectrum of D is bounded by ~ 4 (9/8 + 1/24), so the solve is short
    assert 10 < info["iterations"] < 2000
    ctx.close()
