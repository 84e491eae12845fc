"""-m gpu, collected LAST: hisq_norm2_noalloc, the entry point that allocates nothing (static device scratch), against the
existing path for the same quantity -- the ||b_k||^2 a solve computes at its start (hisq_cgp_begin -> cg_init_kernel with the
workspace's scratch; read back through hisq_cgp_ptr) -- on two calls in a row that share the scratch, at the tolerance the
fp64 parity tests use (1e-14 relative; the block partition and summation order are the same, so the bits should be too).
Runs alone in a fresh process as well as after every other test (nothing here depends on earlier state: the scratch's
ticket is cleared by every call, its partial sums are rewritten before they are read)."""
import ctypes

import pytest
import torch

from paper_2306_01098_b200 import binding

pytestmark = pytest.mark.gpu


def _existing_path_norm2(ctx, b):
    """LOCAL ||b_k||^2 as the solver computes it (the phase-wise CG's first step on an ordinary context)."""
    n = b.shape[0]
    x = ctx.new_field(n)
    ctx.cgp_begin(x, b, 1e-10)
    torch.cuda.synchronize()
    return ctx.cgp_tensor(2, n).clone()


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_norm2_noalloc_matches_the_solver_norm_twice_in_a_row(prec):
    dev = torch.device("cuda:0")
    L, n = (12, 6, 10, 8), 3                       # 6 * Vh = 17 280 reals per RHS: 5 blocks of 4096 with a ragged tail
    ctx = binding.Hisq(L, prec, n, dev)
    ctx.set_links(*binding.make_links(L, 0, dev, ctx.cdtype))     # the solver's entry points refuse a context without links
    torch.manual_seed(7)
    b1 = ctx.new_field(n)
    b1.copy_(torch.randn_like(b1))
    b2 = ctx.new_field(n)
    b2.copy_(3.0 * torch.randn_like(b2))
    ref1, ref2 = _existing_path_norm2(ctx, b1), _existing_path_norm2(ctx, b2)
    out1 = torch.full((n,), -1.0, dtype=torch.float64, device=dev)
    out2 = torch.full((n,), -1.0, dtype=torch.float64, device=dev)
    before = torch.cuda.memory_allocated(dev)
    binding.norm2_noalloc(b1, out1)                # two calls in a row on one stream: the second reuses the scratch the
    binding.norm2_noalloc(b2, out2)                # first one left behind
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated(dev) == before
    for out, ref, b in ((out1, ref1, b1), (out2, ref2, b2)):
        assert torch.all(torch.abs(out - ref) <= 1e-14 * ref), (out, ref)
        plain = torch.view_as_real(b).double().pow(2).reshape(n, -1).sum(dim=1)        # and the definition
        assert torch.all(torch.abs(out - plain) <= 1e-12 * plain)
    # a third call with fewer right-hand sides and a different length sees the leftovers of a larger call: same answer
    out3 = torch.full((1,), -1.0, dtype=torch.float64, device=dev)
    part = b2[1:2, :, :1000].contiguous()
    binding.norm2_noalloc(part, out3)
    torch.cuda.synchronize()
    want = torch.view_as_real(part).double().pow(2).sum()
    assert abs(out3[0] - want) <= 1e-12 * want
    ctx.close()


def test_norm2_noalloc_rejects_sizes_beyond_its_static_scratch():
    lib = binding.load_library()
    dev = torch.device("cuda:0")
    a = torch.zeros(64, dtype=torch.float64, device=dev)
    out = torch.full((17,), -1.0, dtype=torch.float64, device=dev)
    vp = ctypes.c_void_p
    mx = lib.hisq_norm2_noalloc_max_reals()
    assert mx == 16384 * 4096 >= 6 * 96 * 96 * 96 * 24 // 2           # BASELINE's largest field fits
    # the size is checked before anything is launched or read: a small buffer is enough to ask
    assert lib.hisq_norm2_noalloc(vp(a.data_ptr()), 8, mx + 1, 1, vp(out.data_ptr()), None) == binding.HISQ_ETOOBIG
    assert lib.hisq_norm2_noalloc(vp(a.data_ptr()), 8, 4, 17, vp(out.data_ptr()), None) == binding.HISQ_ETOOBIG
    assert b"static scratch" in lib.hisq_strerror(binding.HISQ_ETOOBIG)
    assert lib.hisq_norm2_noalloc(None, 8, 4, 1, vp(out.data_ptr()), None) == binding.HISQ_EINVAL
    assert lib.hisq_norm2_noalloc(vp(a.data_ptr()), 8, 0, 1, vp(out.data_ptr()), None) == binding.HISQ_EINVAL
    assert lib.hisq_norm2_noalloc(vp(a.data_ptr()), 5, 4, 1, vp(out.data_ptr()), None) == binding.HISQ_EINVAL
    torch.cuda.synchronize()
    assert torch.all(out == -1.0)                                       # refused calls wrote nothing
    with pytest.raises(binding.HisqError) as e:
        binding.norm2_noalloc(torch.zeros((17, 4), dtype=torch.float64, device=dev), out)
    assert e.value.code == binding.HISQ_ETOOBIG
