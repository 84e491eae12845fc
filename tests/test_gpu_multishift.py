"""-m gpu: multi-shift CG (row f1) against the oracle: every shifted solution must satisfy its OWN
system (A + sigma_k) x_k = b, judged with the oracle operator, and agree with an independent oracle CG per shift."""
import numpy as np
import pytest
import torch

import oracle
from tests.gpu_helpers import make_ctx, make_field, rel_l2, to_full

pytestmark = pytest.mark.gpu


def _check(L, prec, m, shifts, tol, seed, oracle_solves=True):
    ns = len(shifts)
    ctx, X, W = make_ctx(L, prec, ns, seed)
    b_dev, b_full = make_field(ctx, L, seed, 1, 0)
    x_dev, info = ctx.cg_multishift(b_dev, m, shifts, tol)
    x = to_full(ctx, L, x_dev, 0)
    bn = np.linalg.norm(b_full[0])
    for k, sg in enumerate(shifts):
        r = b_full[0] - (oracle.apply_A(L, X, W, m, x[k])[0] + sg * x[k])
        assert np.linalg.norm(r) / bn <= tol, (k, sg, np.linalg.norm(r) / bn)
        assert abs(info["true_rel_resid"][k] - np.linalg.norm(r) / bn) <= 0.05 * tol
        assert np.all(x[k][oracle.site_parity(L) == 1] == 0)
        if oracle_solves:
            xo, it_o, _, st, _ = oracle.cg(L, X, W, float(np.sqrt(m * m + sg)), tol / 2, b_full)
            assert st == 0 and rel_l2(x[k], xo[0]) <= 10 * tol, (k, rel_l2(x[k], xo[0]))
    ctx.close()
    return info


def test_multishift_fp64_matches_per_shift_oracle_solves():
    shifts = [0.0, 0.01, 0.05, 0.3, 1.0, 4.0]
    info = _check((8, 8, 8, 8), "fp64", 0.1, shifts, 1e-10, seed=0)
    # one operator application per iteration: the count is that of the hardest (smallest) shift alone
    L = (8, 8, 8, 8)
    ctx, X, W = make_ctx(L, "fp64", 1, 0)
    b_dev, _ = make_field(ctx, L, 0, 1, 0)
    _, single = ctx.cg(b_dev, 0.1, 0.5e-10)
    assert abs(info["iterations"] - single["iterations"]) <= 3, (info, single)
    ctx.close()


def test_multishift_unsorted_shifts_and_nonzero_smallest():
    _check((4, 6, 8, 10), "fp64", 0.05, [0.7, 0.02, 2.5, 0.2], 1e-9, seed=1)


def test_multishift_single_shift_equals_plain_cg():
    L, m, tol = (4, 6, 4, 8), 0.1, 1e-10
    ctx, X, W = make_ctx(L, "fp64", 1, 2)
    b_dev, b_full = make_field(ctx, L, 2, 1, 0)
    x1, i1 = ctx.cg_multishift(b_dev, m, [0.0], tol)
    x1 = x1.clone()
    x2, i2 = ctx.cg(b_dev, m, tol / 2)
    assert rel_l2(x1.cpu().numpy(), x2.cpu().numpy()) <= 1e-11
    ctx.close()


def test_multishift_fp32_context():
    _check((8, 8, 8, 8), "fp32", 0.3, [0.0, 0.1, 1.0], 2e-4, seed=3, oracle_solves=False)


def test_multishift_argument_errors():
    from paper_2306_01098_b200 import binding
    L = (4, 4, 4, 4)
    ctx, _, _ = make_ctx(L, "fp64", 2, 0)
    b = ctx.new_field(1)
    with pytest.raises(binding.HisqError) as e:
        ctx.cg_multishift(b, 0.1, [0.0, 0.1, 0.2], 1e-8)      # workspace sized for 2
    assert e.value.code == -3
    with pytest.raises(binding.HisqError) as e:
        ctx.cg_multishift(b, 0.1, [-0.5], 1e-8)               # negative shift
    assert e.value.code == -1
    ctx.close()
    ctxm, _, _ = make_ctx(L, "mixed", 2, 0)
    with pytest.raises(binding.HisqError) as e:
        ctxm.cg_multishift(ctxm.new_field(1), 0.1, [0.0], 1e-8)
    assert e.value.code == -1
    ctxm.close()


def test_multishift_c2_size_rational_like_shifts():
    """32^3 x 8, m = 0.01, 10 shifts spread over 5 decades like a rational approximation's poles."""
    shifts = [0.0] + [float(v) for v in np.geomspace(1e-4, 5.0, 9)]
    info = _check((32, 32, 32, 8), "fp64", 0.01, shifts, 1e-9, seed=0, oracle_solves=False)
    assert 3000 < info["iterations"] < 6500
