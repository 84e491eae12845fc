"""-m gpu: parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

Where the oracle can still do the whole field in seconds (C2, C4's operator) it does; on the big lattices
(C3, C5) it evaluates SAMPLED output sites one by one from operands regenerated on the CPU straight from the
counter-based generator (independent of the product's layout code), always including the sites near every
boundary (antiperiodic-t sign, periodic wraps).  CG at sizes where a CPU solve would take hours is checked
through the oracle OPERATOR: ||b - A x_gpu|| / ||b|| <= tol.
"""
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2306_01098_b200 import binding, inputs
from tests.gpu_helpers import make_ctx, make_field, rel_l2, to_full

pytestmark = pytest.mark.gpu


def _sample_sites(L, parity, n_random, n_edge, seed):
    """Lexicographic sites of one parity: random ones plus ones within 3 of a boundary in each direction."""
    rng = np.random.default_rng(seed)
    V = oracle.volume(L)

    def fix_parity(c):
        c = c.copy()
        odd = (c.sum(axis=1) & 1) != parity
        c[odd, 0] ^= 1                      # flip x's low bit (Lx even) to land on the right parity
        return c

    rnd = np.stack([rng.integers(0, L[d], n_random) for d in range(4)], axis=1)
    parts = [rnd]
    for d in range(4):
        e = np.stack([rng.integers(0, L[k], n_edge) for k in range(4)], axis=1)
        edge_vals = np.array([0, 1, 2, L[d] - 3, L[d] - 2, L[d] - 1])
        e[:, d] = edge_vals[rng.integers(0, 6, n_edge)]
        parts.append(e)
    c = fix_parity(np.concatenate(parts))
    lex = c[:, 0] + L[0] * (c[:, 1] + L[1] * (c[:, 2] + L[2] * c[:, 3]))
    assert lex.max() < V
    return np.unique(lex)


def _oracle_at_samples(L, seed_links, seed_src, nrhs, sites, round_to_fp32):
    """(D phi)(x) for the sampled sites, operands regenerated from the counters on the CPU."""
    plus, minus, t = oracle.neighbour_sites(L, sites)
    n = sites.size
    st = torch.from_numpy(sites)
    Ff = np.stack([inputs.fat_links(L, seed_links, st).numpy(), inputs.naik_links(L, seed_links, st).numpy()], axis=1)
    Fb = np.empty_like(Ff)
    for f, gen in enumerate((inputs.fat_links, inputs.naik_links)):
        for mu in range(4):
            Fb[:, f, mu] = gen(L, seed_links, torch.from_numpy(minus[:, f, mu].copy())).numpy()[:, mu]
    vp = inputs.sources(L, seed_src, torch.from_numpy(plus.reshape(-1).copy()), nrhs).numpy().reshape(nrhs, n, 2, 4, 3)
    vm = inputs.sources(L, seed_src, torch.from_numpy(minus.reshape(-1).copy()), nrhs).numpy().reshape(nrhs, n, 2, 4, 3)
    if round_to_fp32:
        Ff, Fb = Ff.astype(np.complex64).astype(np.complex128), Fb.astype(np.complex64).astype(np.complex128)
        vp, vm = vp.astype(np.complex64).astype(np.complex128), vm.astype(np.complex64).astype(np.complex128)
    return np.stack([oracle.dslash_gathered(L[3], t, Ff, Fb, vp[k], vm[k]) for k in range(nrhs)])


def _gpu_sampled_dslash(L, prec, nrhs, parity, seed, n_random=3000, n_edge=400):
    dev = torch.device("cuda:0")
    ctx = binding.Hisq(L, prec, nrhs, dev)
    fat, naik = binding.make_links(L, seed, dev, ctx.cdtype, gen_device=dev)
    ctx.set_links(fat, naik)
    del fat, naik
    torch.cuda.empty_cache()
    src = binding.make_sources(L, seed + 1, nrhs, 1 - parity, dev, ctx.cdtype, gen_device=dev)
    out = ctx.unpack(ctx.dslash(ctx.pack(src), parity))
    sites = _sample_sites(L, parity, n_random, n_edge, seed)
    got = out[:, torch.from_numpy(sites // 2).to(dev), :].cpu().numpy().astype(np.complex128)
    tiles = ctx.tiles(nrhs)
    ctx.close()
    ref = _oracle_at_samples(L, seed, seed + 1, nrhs, sites, prec == "fp32")
    return got, ref, tiles


@pytest.mark.parametrize("parity", [0, 1])
def test_c3_64x64x64x16_fp32_nrhs8_sampled(parity):
    got, ref, tiles = _gpu_sampled_dslash((64, 64, 64, 16), "fp32", 8, parity, seed=0)
    scale = np.sqrt(np.mean(np.abs(ref) ** 2))
    for k in range(8):
        assert rel_l2(got[k], ref[k]) <= 1e-6
        assert np.abs(got[k] - ref[k]).max() / scale <= 2e-5
    assert tiles != (64, 64)            # the nRHS = 8 launch really runs the tiled sweep order


def test_c3_64x64x64x16_fp32_nrhs8_full_field():
    """one oracle application on the WHOLE field for all 8 right-hand sides of the nRHS = 8 launch (the tiled
    launch shape bench.py times), the oracle on the same fp32-rounded inputs widened to double."""
    from paper_2306_01098_b200 import layout
    L, n, parity = (64, 64, 64, 16), 8, 1
    dev = torch.device("cuda:0")
    ctx = binding.Hisq(L, "fp32", n, dev)
    fat, naik = binding.make_links(L, 0, dev, ctx.cdtype, gen_device=dev)
    ctx.set_links(fat, naik)
    eo = layout.eo_of_lex(L)
    X = fat.cpu().permute(1, 0, 2, 3)[eo].contiguous().numpy().astype(np.complex128)     # the fp32 values, widened
    W = naik.cpu().permute(1, 0, 2, 3)[eo].contiguous().numpy().astype(np.complex128)
    del fat, naik
    src = binding.make_sources(L, 2, n, 1 - parity, dev, ctx.cdtype, gen_device=dev)
    out = ctx.unpack(ctx.dslash(ctx.pack(src), parity))
    assert ctx.tiles(n) != (64, 64)
    got = oracle.half_to_full(L, out.cpu().numpy().astype(np.complex128), parity)
    ref = oracle.dslash_parity(L, X, W, oracle.half_to_full(L, src.cpu().numpy().astype(np.complex128), 1 - parity), parity)
    ctx.close()
    for k in range(n):
        assert rel_l2(got[k], ref[k]) <= 1e-6
        scale = np.sqrt(np.mean(np.abs(ref[k]) ** 2)) * np.sqrt(2.0)      # RMS over the output parity (the other half is zero)
        assert np.abs(got[k] - ref[k]).max() / scale <= 2e-5


def test_c5_96x96x96x24_fp64_nrhs8_sampled():
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 130e9:
        pytest.skip(f"needs ~130 GB of device memory, {free / 1e9:.0f} GB free")
    got, ref, tiles = _gpu_sampled_dslash((96, 96, 96, 24), "fp64", 8, 0, seed=0, n_random=2000, n_edge=300)
    scale = np.sqrt(np.mean(np.abs(ref) ** 2))
    for k in range(8):
        # inputs are generated on the GPU here and regenerated on the CPU for the oracle: libm differences of an ulp
        assert rel_l2(got[k], ref[k]) <= 1e-13
        assert np.abs(got[k] - ref[k]).max() / scale <= 1e-12


def test_c2_32x32x32x8_fp64_full_field_and_cg():
    L, m, tol = (32, 32, 32, 8), 0.01, 1e-10
    ctx, X, W = make_ctx(L, "fp64", 1, 0)
    for parity in (0, 1):
        dev_in, full_in = make_field(ctx, L, 7, 1, 1 - parity)
        got = to_full(ctx, L, ctx.dslash(dev_in, parity), parity)
        ref = oracle.dslash_parity(L, X, W, full_in, parity)
        assert rel_l2(got, ref) <= 1e-14
    b_dev, b_full = make_field(ctx, L, 0, 1, 0)
    x_dev, info = ctx.cg(b_dev, m, tol)
    x = to_full(ctx, L, x_dev, 0)
    r = b_full - oracle.apply_A(L, X, W, m, x)
    assert np.linalg.norm(r) / np.linalg.norm(b_full) <= tol
    assert 4000 < info["iterations"] < 6500           # ~49/m for these link distributions
    if os.environ.get("HISQ_SLOW"):
        xo, it_o, _, st, _ = oracle.cg(L, X, W, m, tol, b_full)
        assert st == 0 and rel_l2(x, xo) <= 10 * tol and abs(int(it_o[0]) - info["iterations"]) <= 25
    ctx.close()


def test_c4_48x48x48x12_mixed_nrhs4_cg():
    """Mixed-precision multi-RHS CG at full size: oracle-evaluated true residual <= tol for every RHS and
    agreement with the pure-fp64 GPU solve to 10 tol."""
    L, m, tol, n = (48, 48, 48, 12), 0.002, 1e-9, 4
    ctx, X, W = make_ctx(L, "mixed", n, 0)
    b_dev, b_full = make_field(ctx, L, 0, n, 0)
    x_dev, info = ctx.cg(b_dev, m, tol)
    x = to_full(ctx, L, x_dev, 0)
    r = b_full - oracle.apply_A(L, X, W, m, x)
    for k in range(n):
        assert np.linalg.norm(r[k]) / np.linalg.norm(b_full[k]) <= tol, (k, info)
    assert info["reliable_updates"] >= info["iterations"] // 100
    ctx.close()
    ctx64, _, _ = make_ctx(L, "fp64", n, 0)
    x64_dev, info64 = ctx64.cg(b_dev, m, tol)
    x64 = to_full(ctx64, L, x64_dev, 0)
    for k in range(n):
        assert rel_l2(x[k], x64[k]) <= 10 * tol, (k, rel_l2(x[k], x64[k]))
    assert info["iterations"] <= 1.25 * info64["iterations"] + 100, (info["iterations"], info64["iterations"])
    ctx64.close()


@pytest.fixture(scope="module")
def c5():
    """BASELINE.json configs[4] (96^3 x 24, fp64, nRHS = 8) set up once for the two full-size C5 tests: the context with
    its links, and the same links on the host in the oracle's lexicographic order (24.5 GB)."""
    from paper_2306_01098_b200 import layout
    import gc
    L, n = (96, 96, 96, 24), 8
    gc.collect()
    torch.cuda.empty_cache()                       # what earlier tests left in torch's caching allocator
    free, _ = torch.cuda.mem_get_info()
    if free < 140e9:
        pytest.skip(f"needs ~140 GB of device memory, {free / 1e9:.0f} GB free")
    dev = torch.device("cuda:0")
    ctx = binding.Hisq(L, "fp64", n, dev)
    fat, naik = binding.make_links(L, 0, dev, ctx.cdtype, gen_device=dev)
    ctx.set_links(fat, naik)
    eo = layout.eo_of_lex(L)                                          # lexicographic site -> Eq. (4) slot
    X = fat.cpu().permute(1, 0, 2, 3)[eo].contiguous().numpy()        # [V, 4, 3, 3] in the oracle's order
    del fat
    W = naik.cpu().permute(1, 0, 2, 3)[eo].contiguous().numpy()
    del naik
    torch.cuda.empty_cache()
    yield dict(L=L, n=n, ctx=ctx, X=X, W=W, dev=dev)
    ctx.close()


def test_c5_96x96x96x24_fp64_nrhs8_dslash_full_field(c5):
    """SURVEY 8(d) C5, the final gate: the WHOLE output field of one right-hand side of the nRHS = 8 launch (the tiled
    launch shape bench.py times) against one oracle application, both parities."""
    L, n, ctx, dev = c5["L"], c5["n"], c5["ctx"], c5["dev"]
    for parity in (0, 1):
        src = binding.make_sources(L, 3 + parity, n, 1 - parity, dev, ctx.cdtype, gen_device=dev)
        out = ctx.unpack(ctx.dslash(ctx.pack(src), parity))
        assert ctx.tiles(n) != (96, 96)                       # the tiled sweep order really ran
        k = 5 if parity == 0 else 2                           # one RHS per parity keeps the oracle at ~1 s per application
        full_in = oracle.half_to_full(L, src[k:k + 1].cpu().numpy(), 1 - parity)
        got = oracle.half_to_full(L, out[k:k + 1].cpu().numpy(), parity)
        del src, out
        ref = oracle.dslash_parity(L, c5["X"], c5["W"], full_in, parity)
        assert rel_l2(got, ref) <= 1e-13                      # inputs are generated on the GPU: an ulp of libm in the sources
        scale = np.sqrt(np.mean(np.abs(ref) ** 2)) * np.sqrt(2.0)   # RMS over the sites of the output parity (the other half is zero)
        assert np.abs(got - ref).max() / scale <= 1e-12
        del full_in, got, ref


def test_c5_96x96x96x24_fp64_nrhs8_cg(c5):
    """BASELINE.json configs[4]: 96^3 x 24, fp64, nRHS = 8, CG at m = 0.005 to tol 1e-10, judged by the ORACLE operator
    on the whole field for every right-hand side (a full CPU solve would take hours)."""
    import time
    L, n, ctx, dev = c5["L"], c5["n"], c5["ctx"], c5["dev"]
    m, tol = 0.005, 1e-10
    b_can = binding.make_sources(L, 1, n, 0, dev, ctx.cdtype, gen_device=dev)
    b = ctx.pack(b_can)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    x, info = ctx.cg(b, m, tol)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    print(f"\nC5 CG: {info['iterations']} iterations, {dt:.1f} s, {1e3 * dt / info['iterations']:.2f} ms/iteration, "
          f"true residuals {info['true_rel_resid']}")
    assert 8000 < info["iterations"] < 13000              # ~49/m for these link distributions
    x_can = ctx.unpack(x).cpu().numpy()
    del x, b
    for k in range(n):                                    # one RHS at a time bounds the host memory
        x_full = oracle.half_to_full(L, x_can[k:k + 1], 0)
        b_full = oracle.half_to_full(L, b_can[k:k + 1].cpu().numpy(), 0)
        r = b_full - oracle.apply_A(L, c5["X"], c5["W"], m, x_full)
        rel = np.linalg.norm(r) / np.linalg.norm(b_full)
        print(f"RHS {k}: oracle-evaluated ||b - A x|| / ||b|| = {rel:.3e}")
        assert rel <= tol
