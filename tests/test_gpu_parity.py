"""GPU parity: the CUDA path, called through the C ABI, against the fp64 oracle on the same
seeded inputs.  Tolerances (BASELINE.json:north_star, outer limits): |dlogp|, |dentropy| <= 1e-2;
loss relative error <= 1e-3; gradient relative Frobenius error <= 2e-2; integers bit-exact.
Internal bars are an order tighter and are what the asserts use.
"""
import numpy as np
import pytest
import torch

import oracle as O
from paper_2507_22789_b200 import inputs as I
from tests.helpers import ELEM_BF16, ELEM_F32, elem_excess, make_batch, oracle_run, rel_fro, to_f64

pytestmark = pytest.mark.gpu

# internal bars
TOL_LOGP_BF16 = 1e-4      # fp32 accumulation of exact bf16 products vs fp64
TOL_LOGP_F32 = 2e-5       # fp32 SIMT path (config 0 bar is 1e-5 on logp; entropy a bit looser)
TOL_LOSS_REL = 1e-3
TOL_GRAD_BF16 = 5e-3      # dS rounded to bf16 (1.6e-3) + bf16 dH output rounding (2.3e-3)
TOL_GRAD_F32 = 1e-4


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "these tests need a B200"
    from paper_2507_22789_b200 import binding          # raises if libgcore.so is missing
    return binding


def dev(x, dtype=None):
    t = torch.as_tensor(x)
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


# ------------------------------------------------------------------ tile engine unit tests
@pytest.mark.parametrize("dyn", [False, True])
@pytest.mark.parametrize("cg", [1, 2])
@pytest.mark.parametrize("a_mn,b_mn", [(0, 0), (0, 1), (1, 0), (1, 1)])
@pytest.mark.parametrize("M,N,K", [(128, 256, 64), (392, 520, 200), (1000, 776, 1096)])
def test_engine_gemm(B, dyn, cg, a_mn, b_mn, M, N, K):
    g = torch.Generator(device="cuda").manual_seed(M + N + K)
    A = torch.randn(M, K, device="cuda", generator=g).to(torch.bfloat16)
    Bm = torch.randn(N, K, device="cuda", generator=g).to(torch.bfloat16)
    ref = A.double() @ Bm.double().T
    C = B.gc_debug_gemm_bf16(A.T.contiguous() if a_mn else A, Bm.T.contiguous() if b_mn else Bm,
                             a_mn, b_mn, cta_group=cg, dynamic_schedule=dyn)
    assert (C.double() - ref).abs().max().item() < 1e-3 * K ** 0.5
    C2 = B.gc_debug_gemm_bf16(A.T.contiguous() if a_mn else A, Bm.T.contiguous() if b_mn else Bm,
                              a_mn, b_mn, C_out=C.clone(), accumulate=True, cta_group=cg,
                              dynamic_schedule=dyn)
    assert (C2.double() - 2 * ref).abs().max().item() < 2e-3 * K ** 0.5


@pytest.mark.parametrize("dyn", [False, True])
@pytest.mark.parametrize("a_mn,b_mn", [(0, 0), (0, 1), (1, 0), (1, 1)])
@pytest.mark.parametrize("M,N,K", [(256, 512, 64), (392, 520, 200), (1000, 776, 1096),
                                   (256 * 5 + 8, 256 * 7 + 8, 328)])
def test_engine_gemm_dual_n(B, dyn, a_mn, b_mn, M, N, K):
    """256 x 512 dual-N tiles (the dH kernel's tile), incl. an odd number of 256-wide N tiles."""
    g = torch.Generator(device="cuda").manual_seed(M + N + K + 1)
    A = torch.randn(M, K, device="cuda", generator=g).to(torch.bfloat16)
    Bm = torch.randn(N, K, device="cuda", generator=g).to(torch.bfloat16)
    ref = A.double() @ Bm.double().T
    C = B.gc_debug_gemm_bf16(A.T.contiguous() if a_mn else A, Bm.T.contiguous() if b_mn else Bm,
                             a_mn, b_mn, cta_group=2, dynamic_schedule=dyn, dual_n=True)
    assert (C.double() - ref).abs().max().item() < 1e-3 * K ** 0.5
    C2 = B.gc_debug_gemm_bf16(A.T.contiguous() if a_mn else A, Bm.T.contiguous() if b_mn else Bm,
                              a_mn, b_mn, C_out=C.clone(), accumulate=True, cta_group=2,
                              dynamic_schedule=dyn, dual_n=True)
    assert (C2.double() - 2 * ref).abs().max().item() < 2e-3 * K ** 0.5


@pytest.mark.parametrize("dyn", [False, True])
@pytest.mark.parametrize("dual", [False, True])
@pytest.mark.parametrize("a_mn,b_mn", [(0, 0), (0, 1), (1, 0), (1, 1)])
@pytest.mark.parametrize("M,N,K", [(256, 256, 64), (392, 520, 200), (1000, 776, 1096),
                                   (256 * 5 + 8, 256 * 7 + 8, 328), (256 * 21 + 40, 256 * 9 + 8, 320)])
def test_engine_gemm_cluster4(B, dyn, dual, a_mn, b_mn, M, N, K):
    """Clusters of two CTA pairs: adjacent M tiles, every B stage fetched once and multicast (the
    launch shape of the path's kernels), incl. an odd number of M tiles (phantom tile), both
    schedules, both tile shapes, all operand layouts; reruns bit-identical."""
    g = torch.Generator(device="cuda").manual_seed(M + N + K + 2)
    A = torch.randn(M, K, device="cuda", generator=g).to(torch.bfloat16)
    Bm = torch.randn(N, K, device="cuda", generator=g).to(torch.bfloat16)
    ref = A.double() @ Bm.double().T
    args = (A.T.contiguous() if a_mn else A, Bm.T.contiguous() if b_mn else Bm, a_mn, b_mn)
    kw = dict(cta_group=2, dynamic_schedule=dyn, dual_n=dual, cluster4=True)
    C = B.gc_debug_gemm_bf16(*args, **kw)
    assert (C.double() - ref).abs().max().item() < 1e-3 * K ** 0.5
    C2 = B.gc_debug_gemm_bf16(*args, C_out=C.clone(), accumulate=True, **kw)
    assert (C2.double() - 2 * ref).abs().max().item() < 2e-3 * K ** 0.5
    assert torch.equal(C, B.gc_debug_gemm_bf16(*args, **kw))


@pytest.mark.parametrize("dual", [False, True])
@pytest.mark.parametrize("dyn", [False, True])
def test_engine_gemm_many_tiles(B, dyn, dual):
    """More tiles than CTA pairs (several items per pair, ragged edges), both schedules; the
    dynamic one must also be deterministic (the tile -> pair map does not enter the result).
    dual + static: 22 x 5 = 110 dual tiles = one full wave of 74 + 36 tiles issued as 72 half
    tiles (the dual-N tail)."""
    M, N, K = 256 * 21 + 40, 256 * 9 + 8, 320
    g = torch.Generator(device="cuda").manual_seed(5)
    A = torch.randn(M, K, device="cuda", generator=g).to(torch.bfloat16)
    Bm = torch.randn(N, K, device="cuda", generator=g).to(torch.bfloat16)
    ref = A.float() @ Bm.float().T
    C1 = B.gc_debug_gemm_bf16(A, Bm, dynamic_schedule=dyn, dual_n=dual)
    C2 = B.gc_debug_gemm_bf16(A, Bm, dynamic_schedule=dyn, dual_n=dual)
    assert (C1 - ref).abs().max().item() < 1e-3 * K ** 0.5
    assert torch.equal(C1, C2)


@pytest.mark.parametrize("cg,dual", [(1, False), (2, False), (2, True)])
@pytest.mark.parametrize("a_mn,b_mn", [(0, 1), (1, 0), (1, 1)])
@pytest.mark.parametrize("M,N,K", [(256 * 5 + 64, 256 * 3 + 128, 328), (256 * 21 + 192, 256 * 9 + 64, 200)])
def test_engine_gemm_mn_major_slab_maps(B, cg, dual, a_mn, b_mn, M, N, K):
    """MN-major operands whose extent is a multiple of 64 are fetched through the 3-D slab tensor map
    (one TMA box per operand and stage; tc_gemm.cuh make_slab_tmap_bf16) -- the form the dH and dW
    launches use at every config: several tiles, edge tiles with whole slabs out of bounds
    (zero-filled), K not a multiple of 64, store and accumulate."""
    g = torch.Generator(device="cuda").manual_seed(M + N + K + 3)
    A = torch.randn(M, K, device="cuda", generator=g).to(torch.bfloat16)
    Bm = torch.randn(N, K, device="cuda", generator=g).to(torch.bfloat16)
    ref = A.double() @ Bm.double().T
    args = (A.T.contiguous() if a_mn else A, Bm.T.contiguous() if b_mn else Bm, a_mn, b_mn)
    kw = dict(cta_group=cg, dynamic_schedule=not dual, dual_n=dual)
    C = B.gc_debug_gemm_bf16(*args, C_out=torch.full((M, N), 3.0, device="cuda"), **kw)
    assert (C.double() - ref).abs().max().item() < 1e-3 * K ** 0.5
    C2 = B.gc_debug_gemm_bf16(*args, C_out=C.clone(), accumulate=True, **kw)
    assert (C2.double() - 2 * ref).abs().max().item() < 2e-3 * K ** 0.5


@pytest.mark.parametrize("order", [0, 2])
@pytest.mark.parametrize("cluster4", [False, True])
def test_engine_gemm_dual_n_paced_long_k(B, order, cluster4):
    """The dH launch shape with a K long enough for several K-lockstep progress segments
    (tc_gemm.cuh Sched::lockstep: 16 k-blocks each, here 49 k-blocks = 4 segments, the last one
    short) over two waves: 110 dual tiles = a full wave of 74 + 36 tiles issued as 72 half tiles,
    so two pairs have no tile in the last wave and only keep the progress counts going.  Both tile
    orders; reruns bit-identical."""
    M, N, K = 256 * 21 + 40, 256 * 9 + 8, 64 * 48 + 40
    g = torch.Generator(device="cuda").manual_seed(23)
    A = torch.randn(M, K, device="cuda", generator=g).to(torch.bfloat16)
    Bm = torch.randn(N, K, device="cuda", generator=g).to(torch.bfloat16)
    ref = A.double() @ Bm.double().T
    kw = dict(cta_group=2, dynamic_schedule=False, dual_n=True, c_major=order, cluster4=cluster4)
    C = B.gc_debug_gemm_bf16(A, Bm.T.contiguous(), 0, 1, **kw)
    assert (C.double() - ref).abs().max().item() < 1e-3 * K ** 0.5
    assert torch.equal(C, B.gc_debug_gemm_bf16(A, Bm.T.contiguous(), 0, 1, **kw))


def test_engine_gemm_dual_n_paced_ring_wraps(B):
    """K long enough for 37 progress segments, more than the 32 slots of the counter ring
    (tc_gemm.cuh kLockRing), so every slot is used a second time; 6 dual tiles issued as 12 half
    tiles on 12 of the 74 pairs, the other 62 only keep the counts going."""
    M, N, K = 256 * 3, 512 * 2, 64 * 16 * 36 + 40
    g = torch.Generator(device="cuda").manual_seed(29)
    A = torch.randn(M, K, device="cuda", generator=g).to(torch.bfloat16)
    Bm = torch.randn(N, K, device="cuda", generator=g).to(torch.bfloat16)
    ref = A.double() @ Bm.double().T
    kw = dict(cta_group=2, dynamic_schedule=False, dual_n=True)
    C = B.gc_debug_gemm_bf16(A, Bm.T.contiguous(), 0, 1, **kw)
    assert (C.double() - ref).abs().max().item() < 1e-3 * K ** 0.5
    assert torch.equal(C, B.gc_debug_gemm_bf16(A, Bm.T.contiguous(), 0, 1, **kw))


SCHEDS = {
    "n_band_narrow_last": dict(n_band=4),                       # 10 N tiles -> bands 4, 4, 2
    "n_band_3": dict(n_band=3),                                 # 3, 3, 3, 1
    "m_band_full_plus_rest_k3": dict(c_major=True, m_band=5, chunk_ntiles=3),   # 22 = 4x5 + 2; runs 3,3,3,1
    "m_band_one_band_k4": dict(c_major=True, m_band=0, chunk_ntiles=4),
    "m_band_7_k1": dict(c_major=True, m_band=7, chunk_ntiles=1),
    "n_major": dict(c_major=2),                                 # (N tile, M tile): dH with rows < D
    "n_major_dual": dict(c_major=2, dual_n=True),               # ... on 256 x 512 tiles, half-tile tail
}


@pytest.mark.parametrize("dyn", [False, True])
@pytest.mark.parametrize("a_mn,b_mn", [(0, 0), (1, 1), (0, 1)])
@pytest.mark.parametrize("sched", list(SCHEDS))
def test_engine_gemm_production_item_orders(B, dyn, a_mn, b_mn, sched):
    """The item orders the path's kernels use at full size only (tc_gemm.cuh get_item): the dW
    order with a narrower last N band, and the forward / recompute order with full + remainder M
    bands and runs of k > 1 N tiles with a shorter last run -- here at a size the test can check
    element by element (220 tiles > 74 CTA pairs, ragged M and N), store and accumulate."""
    M, N, K = 256 * 21 + 40, 256 * 9 + 8, 320
    g = torch.Generator(device="cuda").manual_seed(17)
    A = torch.randn(M, K, device="cuda", generator=g).to(torch.bfloat16)
    Bm = torch.randn(N, K, device="cuda", generator=g).to(torch.bfloat16)
    ref = A.double() @ Bm.double().T
    args = (A.T.contiguous() if a_mn else A, Bm.T.contiguous() if b_mn else Bm, a_mn, b_mn)
    kw = dict(cta_group=2, dynamic_schedule=dyn, **SCHEDS[sched])
    C = B.gc_debug_gemm_bf16(*args, C_out=torch.full((M, N), 7.0, device="cuda"), **kw)
    assert (C.double() - ref).abs().max().item() < 1e-3 * K ** 0.5
    C2 = B.gc_debug_gemm_bf16(*args, C_out=C.clone(), accumulate=True, **kw)
    assert (C2.double() - 2 * ref).abs().max().item() < 2e-3 * K ** 0.5
    assert torch.equal(C, B.gc_debug_gemm_bf16(*args, **kw))


# ------------------------------------------------------------------ a6/a7 advantages
@pytest.mark.parametrize("unbiased", [False, True])
@pytest.mark.parametrize("drop", [False, True])
def test_advantages_and_filter(B, unbiased, drop):
    r = np.random.default_rng(3)
    sizes = r.integers(1, 40, 300)
    sizes[5] = 0
    go = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int32)
    rew = (r.random(go[-1]) < 0.5).astype(np.float32)
    rew[go[7]:go[8]] = r.random(sizes[7]).astype(np.float32)
    rew[go[9]:go[10]] = 0.25
    adv, keep = B.gc_grpo_advantages(dev(rew), dev(go), 1e-6, unbiased, drop)
    with np.errstate(invalid="ignore"):
        a_ref, k_ref = O.grpo_advantages(rew, go, 1e-6, unbiased, drop)
    a = adv.cpu().numpy()
    ok = np.isfinite(a_ref)
    assert np.array_equal(keep.cpu().numpy()[sizes > 0], k_ref[sizes > 0])      # bit-exact
    assert np.allclose(a[ok], a_ref[ok].astype(np.float32), rtol=3e-7, atol=1e-9)
    if drop:
        assert np.array_equal(keep.cpu().numpy()[sizes > 0], O.group_filter(rew, go)[sizes > 0])


# ------------------------------------------------------------------ a1 row selection
@pytest.mark.parametrize("T,p", [(1, 1.0), (5000, 0.75), (70001, 0.3), (4096, 0.0), (2_500_003, 0.6)])
def test_compaction_bit_exact(B, T, p):      # the last case: more count blocks than one scan pass takes
    r = np.random.default_rng(T)
    mask = (r.random(T) < p).astype(np.uint8)
    y = r.integers(0, 100, T).astype(np.int32)
    y[r.random(T) < 0.1] = -100
    H = torch.randn(T, 64, device="cuda").to(torch.bfloat16)
    rows, n, Hs = B.gc_compact_rows(H, dev(y), dev(mask))
    ref = np.nonzero((mask != 0) & (y >= 0))[0]
    assert int(n.item()) == len(ref)
    assert np.array_equal(rows.cpu().numpy()[:len(ref)], ref.astype(np.int32))
    assert torch.equal(Hs[:len(ref)], H[torch.from_numpy(ref).cuda()])
    rows2, n2, _ = B.gc_compact_rows(H, dev(y), None, gather=False)
    assert int(n2.item()) == int((y >= 0).sum())


# ------------------------------------------------------------------ a8/a9 loss kernels alone
def _loss_inputs(T, R, seed, old_std=0.3, p_mask=0.75):
    r = np.random.default_rng(seed)
    cuts = np.sort(r.choice(np.arange(1, T), R - 1, replace=False)) if R > 1 else np.zeros(0, int)
    cu = np.concatenate([[0], cuts, [T]]).astype(np.int32)
    logp = (-3.0 * r.random(T)).astype(np.float32)
    old = (logp + r.normal(0, old_std, T)).astype(np.float32)
    ref = (logp + r.normal(0, 0.1, T)).astype(np.float32)
    adv = r.normal(size=R).astype(np.float32)
    mask = (r.random(T) < p_mask).astype(np.uint8)
    y = r.integers(0, 1000, T).astype(np.int32)
    y[r.random(T) < 0.05] = -1
    return logp, old, ref, adv, mask, y, cu


@pytest.mark.parametrize("agg", [O.AGG_TOKEN_MEAN, O.AGG_SEQ_MEAN])
@pytest.mark.parametrize("T,R", [(7, 2), (4099, 37), (200003, 511)])
def test_token_loss_kernels(B, agg, T, R):
    logp, old, ref, adv, mask, y, cu = _loss_inputs(T, R, T + R)
    out5, g = B.gc_grpo_token_loss(dev(logp), dev(old), dev(ref), dev(y), dev(mask), dev(cu),
                                   dev(adv), 0.2, 0.2, 0.04, agg, grad_loss=1.5)
    scored = (mask != 0) & (y >= 0)
    res = O.grpo_loss(logp, old, ref, scored, adv, cu, 0.2, 0.2, 0.04, agg)
    g_ref = O.grpo_loss_grad_logp(logp, old, ref, scored, adv, cu, 0.2, 0.2, 0.04, agg, 1.5)
    o = out5.cpu().numpy().astype(np.float64)
    assert o[4] == res["n_scored"]                                        # integer, exact
    assert abs(o[0] - res["loss"]) <= 1e-5 * max(abs(res["loss"]), 1e-2)
    assert abs(o[1] - res["pg_loss"]) <= 1e-5 * max(abs(res["pg_loss"]), 1e-2)
    assert abs(o[2] - res["kl_mean"]) <= 1e-5 * max(abs(res["kl_mean"]), 1e-3)
    assert (T < 1000 or res["clip_frac"] > 0.05) and abs(o[3] - res["clip_frac"]) <= 2.0 / max(res["n_scored"], 1)
    gg = g.cpu().numpy().astype(np.float64)
    # both sides decide the clip branch from the same fp32 inputs; exclude float near-ties
    resp = O.token_to_response(cu, T)
    rho = np.exp(logp.astype(np.float64) - old)
    near = (np.abs(rho - 1.2) < 1e-5) | (np.abs(rho - 0.8) < 1e-5)
    assert np.all(gg[~scored] == 0.0)
    assert np.allclose(gg[~near], g_ref[~near], rtol=2e-5, atol=2e-6 * np.abs(g_ref).max())
    assert near.sum() < 0.001 * T + 2


@pytest.mark.parametrize("agg", [O.AGG_TOKEN_MEAN, O.AGG_SEQ_MEAN])
def test_token_loss_exact_ties_take_the_unclipped_branch(B, agg):
    """The clip decision AT a tie (reading 7: s1 <= s2 counts as unclipped), on inputs
    where fp32 and fp64 provably agree, so nothing has to be excluded:
      * clip_lo = clip_hi = 0 and logp == old bit for bit: rho = exp(0) = 1 exactly, which is both
        clip bounds at once -- a kernel that treated rho >= 1 + clip_hi (or <= 1 - clip_lo) as
        clipped would zero these gradients and count them in clip_frac;
      * advantage 0 with rho far outside the band: s1 = s2 = 0 whatever rho is -- a kernel that
        decided from rho alone would count these as clipped;
      * rho = exp(+-0.5), far from the bound, both signs of the advantage: the ordinary branches."""
    R, L = 12, 100
    T = R * L
    cu = np.arange(0, T + 1, L, dtype=np.int32)
    adv = np.array([1.0, -1.0, 0.0, 0.5, -2.0, 0.0] * 2, dtype=np.float32)
    r = np.random.default_rng(5)
    logp = (-(1 + r.integers(0, 24, T)) / 8.0).astype(np.float32)        # multiples of 1/8: exact
    shift = r.choice(np.array([0.0, 0.0, 0.5, -0.5], dtype=np.float32), T)
    old = (logp - shift).astype(np.float32)                              # exact in fp32
    assert np.all(old.astype(np.float64) == logp.astype(np.float64) - shift)
    ref = (logp + r.choice(np.array([0.0, 0.25, -0.25], dtype=np.float32), T)).astype(np.float32)
    mask = np.ones(T, np.uint8)
    y = np.zeros(T, np.int32)
    scored = np.ones(T, bool)
    out5, g = B.gc_grpo_token_loss(dev(logp), dev(old), dev(ref), dev(y), dev(mask), dev(cu),
                                   dev(adv), 0.0, 0.0, 0.04, agg, grad_loss=1.0)
    res = O.grpo_loss(logp, old, ref, scored, adv, cu, 0.0, 0.0, 0.04, agg)
    g_ref = O.grpo_loss_grad_logp(logp, old, ref, scored, adv, cu, 0.0, 0.0, 0.04, agg, 1.0)
    adv_t = np.repeat(adv, L)
    tie_rho1 = (shift == 0) & (adv_t != 0)
    tie_adv0 = (adv_t == 0) & (shift != 0)
    assert tie_rho1.sum() > 100 and tie_adv0.sum() > 50
    # the oracle itself: ties are unclipped, so exactly the off-band tokens with A != 0 whose
    # min() picks the clipped term are counted
    n_clipped = int((((shift > 0) & (adv_t > 0)) | ((shift < 0) & (adv_t < 0))).sum())
    assert abs(res["clip_frac"] - n_clipped / T) < 1e-12
    o = out5.cpu().numpy().astype(np.float64)
    assert o[4] == T
    assert abs(o[3] - res["clip_frac"]) <= 1e-6                 # no near-tie allowance here
    assert abs(o[0] - res["loss"]) <= 1e-5 * max(abs(res["loss"]), 1e-2)
    gg = g.cpu().numpy().astype(np.float64)
    assert np.allclose(gg, g_ref, rtol=2e-5, atol=2e-6 * np.abs(g_ref).max())     # every token
    assert np.all(np.abs(gg[tie_rho1]) > 0.1 * np.abs(g_ref[tie_rho1]))           # not zeroed


@pytest.mark.parametrize("agg", [O.AGG_TOKEN_MEAN, O.AGG_SEQ_MEAN])
@pytest.mark.parametrize("R", [5003, 190001])
def test_token_loss_kernel_more_tiles_than_blocks(B, agg, R):
    """T = 3,000,017 tokens = 2930 tiles of 1024 on a persistent grid of at most 1184 blocks: every
    block walks several tiles (double-buffered slices of cu_seqlens / advantages / weights, count
    batches striding the grid) -- the regime of bench.py's 2^26-token stand-ins, which no smaller
    case reaches.  Long responses (~600 tokens) and short ones (~16 tokens), both aggregations,
    element-wise against the oracle."""
    T = 3_000_017
    logp, old, ref, adv, mask, y, cu = _loss_inputs(T, R, 41 + R)
    out5, g = B.gc_grpo_token_loss(dev(logp), dev(old), dev(ref), dev(y), dev(mask), dev(cu),
                                   dev(adv), 0.2, 0.2, 0.04, agg, grad_loss=1.0)
    scored = (mask != 0) & (y >= 0)
    res = O.grpo_loss(logp, old, ref, scored, adv, cu, 0.2, 0.2, 0.04, agg)
    g_ref = O.grpo_loss_grad_logp(logp, old, ref, scored, adv, cu, 0.2, 0.2, 0.04, agg, 1.0)
    o = out5.cpu().numpy().astype(np.float64)
    assert o[4] == res["n_scored"]
    assert abs(o[0] - res["loss"]) <= 1e-5 * max(abs(res["loss"]), 1e-2)
    assert abs(o[1] - res["pg_loss"]) <= 1e-5 * max(abs(res["pg_loss"]), 1e-2)
    assert abs(o[2] - res["kl_mean"]) <= 1e-5 * max(abs(res["kl_mean"]), 1e-3)
    assert abs(o[3] - res["clip_frac"]) <= 5e-6
    gg = g.cpu().numpy().astype(np.float64)
    rho = np.exp(logp.astype(np.float64) - old)
    near = (np.abs(rho - 1.2) < 1e-5) | (np.abs(rho - 0.8) < 1e-5)
    assert np.all(gg[~scored] == 0.0)
    assert np.allclose(gg[~near], g_ref[~near], rtol=2e-5, atol=2e-6 * np.abs(g_ref).max())
    assert near.sum() < 0.001 * T
    out5b, gb = B.gc_grpo_token_loss(dev(logp), dev(old), dev(ref), dev(y), dev(mask), dev(cu),
                                     dev(adv), 0.2, 0.2, 0.04, agg, grad_loss=1.0)
    assert torch.equal(out5, out5b) and torch.equal(g, gb)              # reruns bit-identical


def test_token_loss_edge_cases(B):
    logp, old, ref, adv, mask, y, cu = _loss_inputs(1000, 10, 5)
    # sum m = 0 -> loss 0, g 0 (reading 12)
    out5, g = B.gc_grpo_token_loss(dev(logp), dev(old), dev(ref), dev(y), dev(np.zeros_like(mask)),
                                   dev(cu), dev(adv))
    assert out5.cpu().tolist() == [0.0, 0.0, 0.0, 0.0, 0.0] and float(g.abs().max()) == 0.0
    # beta = 0 with ref = NULL; mask = NULL
    out5, _ = B.gc_grpo_token_loss(dev(logp), dev(old), None, dev(y), None, dev(cu), dev(adv),
                                   beta=0.0)
    res = O.grpo_loss(logp, old, None, y >= 0, adv, cu, beta=0.0)
    assert abs(out5[0].item() - res["loss"]) <= 1e-5 * max(abs(res["loss"]), 1e-2)
    # logp == old, beta = 0: loss = -sum(m A)/sum(m)   (north_star invariant)
    out5, _ = B.gc_grpo_token_loss(dev(logp), dev(logp), dev(ref), dev(y), dev(mask), dev(cu),
                                   dev(adv), beta=0.0)
    scored = (mask != 0) & (y >= 0)
    A = adv[O.token_to_response(cu, 1000)]
    assert abs(out5[0].item() + (A * scored).sum() / scored.sum()) < 1e-6
    assert out5[3].item() == 0.0
    # logp == ref: KL = 0
    out5, _ = B.gc_grpo_token_loss(dev(logp), dev(old), dev(logp), dev(y), dev(mask), dev(cu),
                                   dev(adv))
    assert out5[2].item() == 0.0
    # rerun determinism: bit-identical
    a, ga = B.gc_grpo_token_loss(dev(logp), dev(old), dev(ref), dev(y), dev(mask), dev(cu), dev(adv))
    b, gb = B.gc_grpo_token_loss(dev(logp), dev(old), dev(ref), dev(y), dev(mask), dev(cu), dev(adv))
    assert torch.equal(a, b) and torch.equal(ga, gb)


# ------------------------------------------------------------------ whole path helper
def run_gpu(B, b, agg=0, backward=True, chunk_tokens=0, simt=False, grad_loss=1.0):
    w = b.w
    adv, keep = B.gc_grpo_advantages(b.rewards_t, b.go_t, 1e-6, False, False)
    f = B.gc_grpo_loss_fwd(b.H, b.W, b.y, b.mask_t, w.tau, b.cu_t, adv, b.old_t, b.ref_t,
                           w.clip_lo, w.clip_hi, w.beta, agg, simt=simt)
    out = dict(adv=adv, keep=keep, **f)
    if backward:
        dH, dW = B.gc_grpo_loss_bwd(b.H, b.W, b.y, b.mask_t, w.tau, b.cu_t, adv, b.old_t, b.ref_t,
                                    f["logp"], f["lse"], w.clip_lo, w.clip_hi, w.beta, agg,
                                    grad_loss, chunk_tokens=chunk_tokens, simt=simt)
        # a9 alone on the forward's own logp: the g_t the backward consumed
        _, g = B.gc_grpo_token_loss(f["logp"], b.old_t, b.ref_t, b.y, b.mask_t, b.cu_t, adv,
                                    w.clip_lo, w.clip_hi, w.beta, agg, grad_loss)
        out.update(dH=dH, dW=dW, g=g)
    torch.cuda.synchronize()
    return out


def check_against_oracle(b, got, ref, tol_lp, tol_grad, backward=True):
    lp = got["logp"].cpu().numpy().astype(np.float64)
    en = got["entropy"].cpu().numpy().astype(np.float64)
    ls = got["lse"].cpu().numpy().astype(np.float64)
    s = b.scored_np
    assert np.all(lp[~s] == 0) and np.all(en[~s] == 0) and np.all(ls[~s] == 0)
    assert np.abs(lp - ref["logp"]).max() <= tol_lp
    assert np.abs(en - ref["entropy"]).max() <= tol_lp * 2
    assert np.abs(ls - ref["lse"]).max() <= tol_lp
    o = got["out5"].cpu().numpy().astype(np.float64)
    assert o[4] == ref["n_scored"]
    scale = max(abs(ref["loss"]), 1e-300)
    assert abs(o[0] - ref["loss"]) <= TOL_LOSS_REL * scale, (o[0], ref["loss"])
    assert abs(o[1] - ref["pg_loss"]) <= TOL_LOSS_REL * max(abs(ref["pg_loss"]), 1e-300)
    assert abs(o[2] - ref["kl_mean"]) <= TOL_LOSS_REL * max(abs(ref["kl_mean"]), 1e-300)
    assert abs(o[3] - ref["clip_frac"]) <= 2.0 / max(ref["n_scored"], 1)
    if backward:
        dH = got["dH"].float().cpu().numpy()
        dW = got["dW"].cpu().numpy()
        assert np.all(dH[~s] == 0.0)                                   # masked rows exactly 0
        assert rel_fro(dH, ref["dH"]) <= tol_grad, rel_fro(dH, ref["dH"])
        assert rel_fro(dW, ref["dW"]) <= tol_grad, rel_fro(dW, ref["dW"])
        # per element, scaled per row (a localised error must not hide in the norm)
        el = ELEM_F32 if tol_grad <= TOL_GRAD_F32 else ELEM_BF16
        assert elem_excess(dH, ref["dH"], **el) <= 1.0, elem_excess(dH, ref["dH"], **el)
        assert elem_excess(dW, ref["dW"], **el) <= 1.0, elem_excess(dW, ref["dW"], **el)
        # g_t element by element; both sides decide the clip branch from the same fp32 inputs,
        # float near-ties excluded (reading 19)
        rho = np.exp(ref["logp"] - b.old_np.astype(np.float64))
        w_ = b.w
        near = (np.abs(rho - (1 + w_.clip_hi)) < 2e-5) | (np.abs(rho - (1 - w_.clip_lo)) < 2e-5)
        gg = got["g"].cpu().numpy().astype(np.float64)
        assert np.all(gg[~s] == 0.0)
        gtol = 1e-4 if tol_lp > TOL_LOGP_F32 else 2e-5       # bf16 path: logp itself is off by <= 1e-4
        assert np.allclose(gg[~near], ref["g"][~near], rtol=gtol * 3, atol=gtol * np.abs(ref["g"]).max())


# ------------------------------------------------------------------ config 0 in full (fp32)
@pytest.mark.parametrize("agg", [O.AGG_TOKEN_MEAN, O.AGG_SEQ_MEAN])
def test_config0_full(B, agg):
    b = make_batch(I.CONFIGS[0], seed=0, device="cuda")
    adv_ref, _ = O.grpo_advantages(b.rewards_np, b.lay.group_offsets, 1e-6)
    ref = oracle_run(b, adv_ref, agg)
    got = run_gpu(B, b, agg)
    assert np.allclose(got["adv"].cpu().numpy(), adv_ref.astype(np.float32), rtol=3e-7, atol=1e-9)
    check_against_oracle(b, got, ref, TOL_LOGP_F32, TOL_GRAD_F32)


def test_f32_odd_shapes_masks_temperature(B):
    w = I.reduced(I.CONFIGS[0], D=72, V=1001, groups=3, group_size=3, seq_len=0, tau=0.7,
                  lognormal=(2.5, 0.8, 1, 60), prompt_len=2, old_std=0.3)
    b = make_batch(w, seed=4, device="cuda")
    adv_ref, _ = O.grpo_advantages(b.rewards_np, b.lay.group_offsets, 1e-6)
    for agg in (0, 1):
        check_against_oracle(b, run_gpu(B, b, agg), oracle_run(b, adv_ref, agg), TOL_LOGP_F32,
                             TOL_GRAD_F32)


# ------------------------------------------------------------------ bf16 tcgen05 path, small shapes
BF16_CASES = {
    # spans several 256-row / 256-col tiles with ragged tails; D not a multiple of 64
    "ragged": dict(D=200, V=4097 + 64, groups=3, group_size=4, seq_len=0, lognormal=(3.6, 0.6, 1, 200)),
    "masked": dict(D=512, V=5000, groups=2, group_size=8, seq_len=48, prompt_len=12, old_std=0.3),
    "tau": dict(D=1024, V=8192, groups=1, group_size=8, seq_len=64, tau=0.7),
    "one_token": dict(D=64, V=300, groups=1, group_size=2, seq_len=0, lognormal=(0.0, 0.01, 1, 1)),
}


@pytest.mark.parametrize("name", list(BF16_CASES))
def test_bf16_small_forward_backward(B, name):
    w = I.reduced(I.CONFIGS[2], backward=True, **{"prompt_len": 0, **BF16_CASES[name]})
    b = make_batch(w, seed=7, device="cuda")
    adv_ref, _ = O.grpo_advantages(b.rewards_np, b.lay.group_offsets, 1e-6)
    ref = oracle_run(b, adv_ref)
    got = run_gpu(B, b)
    check_against_oracle(b, got, ref, TOL_LOGP_BF16, TOL_GRAD_BF16)
    # the slow SIMT kernels on the same bf16 operands agree too (on-device cross-check path)
    got2 = run_gpu(B, b, simt=True)
    check_against_oracle(b, got2, ref, TOL_LOGP_BF16, TOL_GRAD_BF16)


def test_bf16_forward_more_rows_than_the_helper_grids(B):
    """T = 400,001 rows: the 1-D helper kernels of the forward (target / lse gathers, zero-fill of
    unscored outputs) run capped grids of 1184 x 256 threads and stride them beyond 303,104 rows --
    past every config (cfg3: 281,898).  Random mask, negative targets; sampled rows against the
    oracle, unscored rows exactly zero, and the masked call equals the dense call on scored rows."""
    T, D, V = 400_001, 64, 512 + 24
    H, W = I.make_hw(T, D, V, "bf16", 21, "cuda")
    y = I.sample_targets(H, W, 1.0, 21)
    mask_np = I.random_mask(T, 0.7, 21)
    y_np = y.cpu().numpy().copy()
    y_np[::13] = -100
    y = torch.from_numpy(y_np).cuda()
    mask = torch.from_numpy(mask_np).cuda()
    lp, en, ls = B.gc_token_logprobs(H, W, y, mask, 1.0)
    lp_d, en_d, ls_d = B.gc_token_logprobs(H, W, y, None, 1.0)
    torch.cuda.synchronize()
    scored = (mask_np != 0) & (y_np >= 0)
    st = torch.from_numpy(scored).cuda()
    assert float(lp[~st].abs().sum()) == 0.0 and float(en[~st].abs().sum()) == 0.0 and float(ls[~st].abs().sum()) == 0.0
    assert torch.equal(lp[st], lp_d[st]) and torch.equal(en[st], en_d[st]) and torch.equal(ls[st], ls_d[st])
    r = np.random.default_rng(3)
    S = np.array(sorted({0, 1, 255, 256, 303_103, 303_104, 303_105, T - 2, T - 1} | {int(x) for x in r.integers(0, T, 300)}))
    St = torch.from_numpy(S).cuda()
    lp_o, en_o, ls_o = O.token_logprobs(to_f64(H[St]), to_f64(W), y_np[S], mask_np[S], 1.0)
    assert np.abs(lp[St].cpu().numpy() - lp_o).max() <= TOL_LOGP_BF16
    assert np.abs(ls[St].cpu().numpy() - ls_o).max() <= TOL_LOGP_BF16
    assert np.abs(en[St].cpu().numpy() - en_o).max() <= 2 * TOL_LOGP_BF16


def test_bf16_random_mask_negative_targets_chunks_accumulate(B):
    w = I.reduced(I.CONFIGS[2], D=256, V=2048 + 8, groups=4, group_size=4, seq_len=40, prompt_len=0,
                  old_std=0.3)
    b0 = make_batch(w, seed=9, device="cpu")
    mask = I.random_mask(b0.T, 0.6, 9)
    b = make_batch(w, seed=9, device="cuda", mask=mask)
    y = b.y_np.copy()
    y[::17] = -100
    b.y_np, b.y = y, torch.from_numpy(y).cuda()
    b.scored_np = (b.mask_np != 0) & (y >= 0)
    adv_ref, _ = O.grpo_advantages(b.rewards_np, b.lay.group_offsets, 1e-6)
    for agg in (0, 1):
        ref = oracle_run(b, adv_ref, agg, grad_loss=0.5)
        for chunk in (0, 256, 512):
            got = run_gpu(B, b, agg, chunk_tokens=chunk, grad_loss=0.5)
            check_against_oracle(b, got, ref, TOL_LOGP_BF16, TOL_GRAD_BF16)
    # dense mode (mask = NULL) with negative targets only
    b.mask_t, b.all_scored = None, True
    b.mask_np = np.ones_like(b.mask_np)
    b.scored_np = y >= 0
    ref = oracle_run(b, adv_ref)
    got = run_gpu(B, b)
    check_against_oracle(b, got, ref, TOL_LOGP_BF16, TOL_GRAD_BF16)
    # accumulate_dW adds to the existing contents; reruns are bit-identical
    dW0 = torch.full_like(got["dW"], 0.25)
    _, dW1 = B.gc_grpo_loss_bwd(b.H, b.W, b.y, None, w.tau, b.cu_t, got["adv"], b.old_t, b.ref_t,
                                got["logp"], got["lse"], dW=dW0.clone(), accumulate_dW=True)
    assert rel_fro((dW1 - 0.25).cpu().numpy(), ref["dW"]) <= TOL_GRAD_BF16
    again = run_gpu(B, b)
    for k in ("logp", "entropy", "lse", "out5", "dH", "dW"):
        assert torch.equal(again[k], got[k]), k


def test_bf16_empty_and_all_masked(B):
    w = I.reduced(I.CONFIGS[2], D=128, V=512, groups=1, group_size=4, seq_len=8, prompt_len=0)
    b = make_batch(w, seed=1, device="cuda", mask=np.zeros(32, np.uint8))
    got = run_gpu(B, b)
    assert float(got["logp"].abs().max()) == 0 and got["out5"].cpu().tolist() == [0.0] * 5
    assert float(got["dH"].float().abs().max()) == 0 and float(got["dW"].abs().max()) == 0
    # T = 0
    H0 = torch.empty(0, 128, dtype=torch.bfloat16, device="cuda")
    lp, en, ls = B.gc_token_logprobs(H0, b.W, torch.empty(0, dtype=torch.int32, device="cuda"))
    assert lp.numel() == 0
    assert B.gc_validate_targets(b.y, None, 512) == 0 and B.gc_validate_targets(b.y, None, 1) > 0


def test_host_buffer_entry_point_matches_device_path(B):
    """gc_token_logprobs_host (the end-to-end entry: pinned host inputs, host outputs) computes
    exactly what gc_token_logprobs computes on device-resident copies, with and without a mask."""
    w = I.reduced(I.CONFIGS[1], D=256, V=2048 + 24, groups=2, group_size=2, seq_len=75)
    b = make_batch(w, seed=4, device="cuda")
    mask_np = I.random_mask(b.T, 0.7, 4)
    for m in (None, mask_np):
        md = None if m is None else torch.from_numpy(m).cuda()
        lp_d, en_d, _ = B.gc_token_logprobs(b.H, b.W, b.y, md, w.tau)
        Hh = b.H.cpu().pin_memory()
        yh = b.y.cpu().pin_memory()
        mh = None if m is None else torch.from_numpy(m).pin_memory()
        lph = torch.empty(b.T, dtype=torch.float32).pin_memory()
        enh = torch.empty(b.T, dtype=torch.float32).pin_memory()
        B.gc_token_logprobs_host(Hh, b.W, yh, mh, w.tau, logp_host=lph, entropy_host=enh)
        torch.cuda.synchronize()
        assert torch.equal(lph, lp_d.cpu()) and torch.equal(enh, en_d.cpu())
    lp_o, en_o, _ = O.token_logprobs(to_f64(b.H), to_f64(b.W), b.y_np, mask_np, w.tau)
    assert np.abs(lph.numpy() - lp_o).max() <= TOL_LOGP_BF16


def test_kernel_timing_counts_the_contraction_launches(B):
    """gc_kernel_timing_*: one record per contraction launch, by kind, positive durations, and off
    again afterwards."""
    w = I.reduced(I.CONFIGS[2], D=256, V=2048, groups=2, group_size=2, seq_len=160, prompt_len=32)
    b = make_batch(w, seed=2, device="cuda")
    B.gc_kernel_timing_begin()
    run_gpu(B, b, chunk_tokens=256)
    k = B.gc_kernel_timing_end()
    n_chunks = -(-b.T // 256)
    assert k["fwd_stats"][1] == 1 and k["recompute_ds"][1] == n_chunks
    assert k["dh"][1] == n_chunks and k["dw"][1] == n_chunks
    assert all(ms > 0 for ms, n in k.values() if n)
    run_gpu(B, b)
    assert all(n == 0 for _, n in B.gc_kernel_timing_end().values())


def test_bf16_padded_leading_dimensions(B):
    """Row strides larger than the row (ldH, ldW, lddH, lddW > D): H, W, dH, dW are views into wider
    buffers; results equal the dense call bit for bit and the padding is never written."""
    w = I.reduced(I.CONFIGS[2], D=256, V=1024 + 40, groups=2, group_size=2, seq_len=90, prompt_len=20)
    b = make_batch(w, seed=6, device="cuda")
    dense = run_gpu(B, b, chunk_tokens=256)

    def widen(t, pad, fill):
        buf = torch.full((t.shape[0], t.shape[1] + pad), fill, dtype=t.dtype, device=t.device)
        buf[:, :t.shape[1]] = t
        return buf, buf[:, :t.shape[1]]
    Hbuf, Hv = widen(b.H, 8, 7.0)
    Wbuf, Wv = widen(b.W, 16, -3.0)
    dHbuf = torch.full((b.T, w.D + 24), 5.0, dtype=torch.bfloat16, device="cuda")
    dWbuf = torch.full((w.V, w.D + 12), 9.0, dtype=torch.float32, device="cuda")
    adv = dense["adv"]
    f = B.gc_grpo_loss_fwd(Hv, Wv, b.y, b.mask_t, w.tau, b.cu_t, adv, b.old_t, b.ref_t,
                           w.clip_lo, w.clip_hi, w.beta)
    dH, dW = B.gc_grpo_loss_bwd(Hv, Wv, b.y, b.mask_t, w.tau, b.cu_t, adv, b.old_t, b.ref_t,
                                f["logp"], f["lse"], w.clip_lo, w.clip_hi, w.beta,
                                dH=dHbuf[:, :w.D], dW=dWbuf[:, :w.D], chunk_tokens=256)
    torch.cuda.synchronize()
    for k in ("logp", "entropy", "lse", "out5"):
        assert torch.equal(f[k], dense[k]), k
    assert torch.equal(dHbuf[:, :w.D], dense["dH"]) and torch.equal(dWbuf[:, :w.D], dense["dW"])
    assert bool((dHbuf[:, w.D:] == 5.0).all()) and bool((dWbuf[:, w.D:] == 9.0).all())
    assert bool((Hbuf[:, w.D:] == 7.0).all()) and bool((Wbuf[:, w.D:] == -3.0).all())


@pytest.mark.parametrize("scale,tau", [(40.0, 1.0), (12.0, 0.05)])
def test_bf16_large_logits_online_softmax_is_stable(B, scale, tau):
    """Logits of magnitude ~1e2 (a peaked policy, or a small temperature): the running-max
    rescaling of the split-V statistics must neither overflow nor lose the tail; near-one-hot rows
    have logp -> 0 and entropy -> 0 (SURVEY.md sec 8(c) pins), and everything matches the oracle."""
    T, D, V = 300, 256, 4096 + 24
    H, W = I.make_hw(T, D, V, "bf16", 11, "cuda")
    W = (W.float() * scale).to(torch.bfloat16)
    y = I.sample_targets(H, W, tau, 11)
    lp, en, ls = B.gc_token_logprobs(H, W, y, None, tau)
    lp_o, en_o, ls_o = O.token_logprobs(to_f64(H), to_f64(W), y.cpu().numpy(), None, tau)
    assert np.isfinite(ls.cpu().numpy()).all() and np.abs(ls_o).max() > 20
    tol = 2e-3
    assert np.abs(lp.cpu().numpy() - lp_o).max() <= tol
    assert np.abs(ls.cpu().numpy() - ls_o).max() <= tol * 2
    assert np.abs(en.cpu().numpy() - en_o).max() <= tol * 2
    peaked = en_o < 1e-3
    if peaked.any():
        assert np.abs(lp.cpu().numpy()[peaked]).max() <= 5e-3


def test_forward_backward_replays_from_a_cuda_graph(B):
    """The calls only enqueue work (no allocation, no sync, no host-side data dependence), so a
    whole forward + backward can be captured once and replayed; replays are bit-identical to the
    eager run (the tile tickets are re-zeroed by a memset node inside the graph)."""
    w = I.reduced(I.CONFIGS[2], D=256, V=2048 + 8, groups=2, group_size=2, seq_len=130, prompt_len=30)
    b = make_batch(w, seed=8, device="cuda")
    eager = run_gpu(B, b, chunk_tokens=256)                 # also sizes the cached workspace
    adv = eager["adv"]
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        run_gpu(B, b, chunk_tokens=256)                     # warm-up on the side stream
    torch.cuda.current_stream().wait_stream(stream)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        f = B.gc_grpo_loss_fwd(b.H, b.W, b.y, b.mask_t, w.tau, b.cu_t, adv, b.old_t, b.ref_t,
                               w.clip_lo, w.clip_hi, w.beta)
        dH, dW = B.gc_grpo_loss_bwd(b.H, b.W, b.y, b.mask_t, w.tau, b.cu_t, adv, b.old_t, b.ref_t,
                                    f["logp"], f["lse"], w.clip_lo, w.clip_hi, w.beta,
                                    chunk_tokens=256)
    for _ in range(2):
        dW.fill_(123.0)
        dH.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(f["logp"], eager["logp"]) and torch.equal(f["out5"], eager["out5"])
        assert torch.equal(dH, eager["dH"]) and torch.equal(dW, eager["dW"])


@pytest.mark.parametrize("seed", range(12))
def test_bf16_randomized_shapes(B, seed):
    """Seeded random small problems (D, V off the tile grid, V below one tile, random masks, both
    aggregations, 1-3 dS chunks, temperature) against the oracle, forward and backward."""
    r = np.random.default_rng(1000 + seed)
    D = int(r.choice([64, 128, 264, 512, 1032]))
    V = int(r.choice([8, 100, 255, 256, 257, 1000, 2048, 4136, 6000]))
    w = I.reduced(I.CONFIGS[2], D=D, V=V, groups=int(r.integers(1, 4)), group_size=int(r.integers(1, 5)),
                  seq_len=int(r.integers(2, 300)), prompt_len=0, old_std=0.3)
    b0 = make_batch(w, seed=seed, device="cpu")
    mask = I.random_mask(b0.T, float(r.uniform(0.2, 1.0)), seed) if r.random() < 0.6 else None
    b = make_batch(w, seed=seed, device="cuda", mask=mask)
    agg = int(r.integers(0, 2))
    adv_ref, _ = O.grpo_advantages(b.rewards_np, b.lay.group_offsets, 1e-6)
    ref = oracle_run(b, adv_ref, agg)
    got = run_gpu(B, b, agg, chunk_tokens=int(r.choice([0, 256, 512])))
    check_against_oracle(b, got, ref, TOL_LOGP_BF16, TOL_GRAD_BF16)


@pytest.mark.parametrize("V", [520, 1096])
@pytest.mark.parametrize("masked", [True, False])
def test_bf16_production_schedules_vs_oracle(B, V, masked):
    """Forward + backward against the DENSE oracle on a problem whose backward chunk is large
    enough (8192 rows x D = 4096: k_rows D > 21 M) for the real kernels to take the schedules that
    the small cases never reach: dW with n_band = 10 < 16 D tiles (a narrower last band), forward /
    recompute with runs of k = 2 (V = 520) or 3 + 2 (V = 1096) vocab tiles and a full + remainder M
    band (34 M tiles = 24 + 10), two dS chunks.  The vocabulary is small so the oracle stays cheap."""
    if masked:      # 8520 scored of 11360 tokens (compaction mode)
        w = I.reduced(I.CONFIGS[2], D=4096, V=V, groups=2, group_size=4, seq_len=1420, prompt_len=355,
                      old_std=0.3)
    else:           # dense mode, 8500 rows
        w = I.reduced(I.CONFIGS[2], D=4096, V=V, groups=1, group_size=4, seq_len=2125, prompt_len=0,
                      old_std=0.3)
    b = make_batch(w, seed=3, device="cuda")
    adv_ref, _ = O.grpo_advantages(b.rewards_np, b.lay.group_offsets, 1e-6)
    ref = oracle_run(b, adv_ref)
    got = run_gpu(B, b, chunk_tokens=8192)
    check_against_oracle(b, got, ref, TOL_LOGP_BF16, TOL_GRAD_BF16)
    again = run_gpu(B, b, chunk_tokens=8192)
    for k in ("logp", "entropy", "lse", "out5", "dH", "dW"):
        assert torch.equal(again[k], got[k]), k


@pytest.mark.parametrize("masked", [True, False])
def test_bf16_backward_more_chunks_than_one_counter_zeroing(B, masked):
    """34 backward chunks of 256 rows: a chunk takes 34 of the 1024 zeroed counter words (two tile
    tickets + the dH progress ring), so the chunk loop re-zeroes the area after 30 chunks -- a
    regime real batches reach beyond 30 x 8192 scored tokens.  Against the dense oracle, and
    bit-identical on a rerun."""
    if masked:
        w = I.reduced(I.CONFIGS[2], D=128, V=520, groups=2, group_size=4, seq_len=1420, prompt_len=355,
                      old_std=0.3)
    else:
        w = I.reduced(I.CONFIGS[2], D=128, V=520, groups=1, group_size=4, seq_len=2125, prompt_len=0,
                      old_std=0.3)
    b = make_batch(w, seed=5, device="cuda")
    assert b.scored_np.sum() > 30 * 256
    adv_ref, _ = O.grpo_advantages(b.rewards_np, b.lay.group_offsets, 1e-6)
    ref = oracle_run(b, adv_ref)
    got = run_gpu(B, b, chunk_tokens=256)
    check_against_oracle(b, got, ref, TOL_LOGP_BF16, TOL_GRAD_BF16)
    again = run_gpu(B, b, chunk_tokens=256)
    for k in ("dH", "dW"):
        assert torch.equal(again[k], got[k]), k


def test_token_loss_offset_mask_and_garbage_at_unscored_positions(B):
    """A mask view at a 4-byte (not 8-byte) offset must take the whole-tile fast path safely, and
    inf / NaN stored at unscored positions of logp / old / ref must not reach the loss (only scored
    tokens matter, gcore.h).  T spans several whole 2048-token tiles and a ragged tail."""
    T, R = 3 * 2048 + 37, 23
    logp, old, ref, adv, mask, y, cu = _loss_inputs(T, R, 77)
    scored = (mask != 0) & (y >= 0)
    res = O.grpo_loss(logp, old, ref, scored, adv, cu, 0.2, 0.2, 0.04)
    g_ref = O.grpo_loss_grad_logp(logp, old, ref, scored, adv, cu, 0.2, 0.2, 0.04)
    for agg in (0, 1):
        res = O.grpo_loss(logp, old, ref, scored, adv, cu, 0.2, 0.2, 0.04, agg)
        buf = torch.zeros(T + 16, dtype=torch.uint8, device="cuda")
        for off in (4, 12, 8):
            mview = buf[off:off + T]
            mview.copy_(dev(mask))
            assert mview.data_ptr() % 8 == off % 8
            bad = [a.copy() for a in (logp, old, ref)]
            fill = [np.nan, -np.inf, np.inf]
            for a, v in zip(bad, fill):
                a[~scored] = v
            out5, g = B.gc_grpo_token_loss(dev(bad[0]), dev(bad[1]), dev(bad[2]), dev(y), mview,
                                           dev(cu), dev(adv), 0.2, 0.2, 0.04, agg)
            o = out5.cpu().numpy().astype(np.float64)
            assert np.isfinite(o).all(), o
            assert abs(o[0] - res["loss"]) <= 1e-5 * max(abs(res["loss"]), 1e-2)
            assert abs(o[2] - res["kl_mean"]) <= 1e-5 * max(abs(res["kl_mean"]), 1e-3)
            gg = g.cpu().numpy()
            assert np.isfinite(gg).all() and np.all(gg[~scored] == 0.0)
            if agg == 0:
                assert np.allclose(gg, g_ref, rtol=3e-5, atol=2e-6 * np.abs(g_ref).max())


def test_token_loss_more_responses_than_tokens(B):
    """Empty responses are legal (repeated cu_seqlens entries), so R is not bounded by T."""
    T, R = 40, 200
    r = np.random.default_rng(5)
    cu = np.sort(np.concatenate([[0, T], r.integers(0, T + 1, R - 1)])).astype(np.int32)
    assert len(cu) == R + 1
    logp, old, ref, _, mask, y, _ = _loss_inputs(T, 2, 9)
    adv = r.normal(size=R).astype(np.float32)
    scored = (mask != 0) & (y >= 0)
    for agg in (0, 1):
        out5, g = B.gc_grpo_token_loss(dev(logp), dev(old), dev(ref), dev(y), dev(mask), dev(cu),
                                       dev(adv), 0.2, 0.2, 0.04, agg)
        res = O.grpo_loss(logp, old, ref, scored, adv, cu, 0.2, 0.2, 0.04, agg)
        g_ref = O.grpo_loss_grad_logp(logp, old, ref, scored, adv, cu, 0.2, 0.2, 0.04, agg)
        assert abs(out5[0].item() - res["loss"]) <= 1e-5 * max(abs(res["loss"]), 1e-2)
        assert np.allclose(g.cpu().numpy(), g_ref, rtol=3e-5, atol=2e-6 * np.abs(g_ref).max())


def test_gather_1d_never_writes_past_max_rows(B):
    x = torch.arange(100, dtype=torch.int32, device="cuda")
    rows = torch.arange(99, -1, -1, dtype=torch.int32, device="cuda")
    n = torch.tensor([100], dtype=torch.int32, device="cuda")       # device count > allocation
    buf = torch.full((64,), -7, dtype=torch.int32, device="cuda")
    import ctypes as C
    B._check(B.lib().gc_gather_1d(C.c_void_p(x.data_ptr()), C.c_void_p(rows.data_ptr()),
                                  C.c_void_p(n.data_ptr()), 40, C.c_void_p(buf.data_ptr()),
                                  C.c_void_p(torch.cuda.current_stream().cuda_stream)))
    torch.cuda.synchronize()
    assert torch.equal(buf[:40], rows[:40]) and bool((buf[40:] == -7).all())


def test_bf16_dw_output_and_forward_state_reuse(B):
    """dW_dtype = bf16 (SURVEY.md sec 8(c) reading 13: accumulated in fp32 across the dS chunks,
    rounded ONCE at the end): equals the fp32 dW rounded to bf16 bit for bit, matches the oracle,
    and accumulate_dW adds with one rounding.  fwd_state: the backward reusing the forward's row
    selection gives bit-identical results to the backward that recomputes it."""
    w = I.reduced(I.CONFIGS[2], D=256, V=2048 + 40, groups=2, group_size=4, seq_len=150, prompt_len=30,
                  old_std=0.3)
    b = make_batch(w, seed=12, device="cuda")
    adv_ref, _ = O.grpo_advantages(b.rewards_np, b.lay.group_offsets, 1e-6)
    ref = oracle_run(b, adv_ref)
    adv, _ = B.gc_grpo_advantages(b.rewards_t, b.go_t)
    f = B.gc_grpo_loss_fwd(b.H, b.W, b.y, b.mask_t, w.tau, b.cu_t, adv, b.old_t, b.ref_t, w.clip_lo,
                           w.clip_hi, w.beta)
    args = (b.H, b.W, b.y, b.mask_t, w.tau, b.cu_t, adv, b.old_t, b.ref_t, f["logp"], f["lse"],
            w.clip_lo, w.clip_hi, w.beta)
    for chunk in (256, 512, 0):
        dH32, dW32 = B.gc_grpo_loss_bwd(*args, chunk_tokens=chunk)
        dH16, dW16 = B.gc_grpo_loss_bwd(*args, chunk_tokens=chunk, dW_dtype=torch.bfloat16)
        assert dW16.dtype == torch.bfloat16
        assert torch.equal(dW16, dW32.to(torch.bfloat16)) and torch.equal(dH16, dH32)
        assert rel_fro(dW16.float().cpu().numpy(), ref["dW"]) <= TOL_GRAD_BF16
        # accumulate: out = bf16(out + sum), one rounding
        base = (torch.randn_like(dW32) * dW32.abs().mean()).to(torch.bfloat16)
        _, acc = B.gc_grpo_loss_bwd(*args, chunk_tokens=chunk, dW=base.clone(), accumulate_dW=True)
        assert torch.equal(acc, (base.float() + dW32).to(torch.bfloat16))
        # a padded bf16 dW view: the padding is never written
        buf = torch.full((w.V, w.D + 8), 3.0, dtype=torch.bfloat16, device="cuda")
        B.gc_grpo_loss_bwd(*args, chunk_tokens=chunk, dW=buf[:, :w.D])
        assert torch.equal(buf[:, :w.D], dW16) and bool((buf[:, w.D:] == 3.0).all())
        # forward-state reuse
        dH_r, dW_r = B.gc_grpo_loss_bwd(*args, chunk_tokens=chunk, fwd_state=f["state"])
        assert torch.equal(dH_r, dH32) and torch.equal(dW_r, dW32)
    # fp32 (SIMT) path with bf16 dW (D not a multiple of 8: element-wise cast)
    w0 = I.reduced(I.CONFIGS[0], D=36, V=300, groups=1, group_size=3, seq_len=9)
    b0 = make_batch(w0, seed=1, device="cuda")
    adv0, _ = B.gc_grpo_advantages(b0.rewards_t, b0.go_t)
    f0 = B.gc_grpo_loss_fwd(b0.H, b0.W, b0.y, None, 1.0, b0.cu_t, adv0, b0.old_t, b0.ref_t)
    a0 = (b0.H, b0.W, b0.y, None, 1.0, b0.cu_t, adv0, b0.old_t, b0.ref_t, f0["logp"], f0["lse"])
    _, d32 = B.gc_grpo_loss_bwd(*a0)
    _, d16 = B.gc_grpo_loss_bwd(*a0, dW_dtype=torch.bfloat16)
    assert torch.equal(d16, d32.to(torch.bfloat16))


def test_stale_forward_state_is_not_used(B):
    """Micro-batches A then B forwarded on the same stream share the cached forward workspace, so
    after B's forward A's state describes B's row selection.  The binding must notice (generation
    counter + shapes + input pointers) and let A's backward recompute its own selection: results
    bit-identical to a backward without any state; B's state, the latest, is still used."""
    def batch(seed, seq_len):
        w = I.reduced(I.CONFIGS[2], D=256, V=2048, groups=2, group_size=4, seq_len=seq_len,
                      prompt_len=40, old_std=0.3)
        b = make_batch(w, seed=seed, device="cuda")
        adv, _ = B.gc_grpo_advantages(b.rewards_t, b.go_t)
        return w, b, adv
    wa, a, adv_a = batch(21, 160)
    wb, bb, adv_b = batch(22, 130)
    fa = B.gc_grpo_loss_fwd(a.H, a.W, a.y, a.mask_t, wa.tau, a.cu_t, adv_a, a.old_t, a.ref_t)
    args_a = (a.H, a.W, a.y, a.mask_t, wa.tau, a.cu_t, adv_a, a.old_t, a.ref_t, fa["logp"], fa["lse"])
    sig_a = B._state_sig(a.H, a.y, a.mask_t, a.T, wa.D, wa.V, B.GC_BF16)
    assert fa["state"].usable_for(sig_a)
    dH_ref, dW_ref = B.gc_grpo_loss_bwd(*args_a)                          # no state: recomputes
    fb = B.gc_grpo_loss_fwd(bb.H, bb.W, bb.y, bb.mask_t, wb.tau, bb.cu_t, adv_b, bb.old_t, bb.ref_t)
    assert not fa["state"].usable_for(sig_a)                              # overwritten by B
    dH_a, dW_a = B.gc_grpo_loss_bwd(*args_a, fwd_state=fa["state"])       # stale: must be ignored
    assert torch.equal(dH_a, dH_ref) and torch.equal(dW_a, dW_ref)
    # a state offered for other inputs than it was made for is ignored as well
    assert not fb["state"].usable_for(sig_a)
    args_b = (bb.H, bb.W, bb.y, bb.mask_t, wb.tau, bb.cu_t, adv_b, bb.old_t, bb.ref_t, fb["logp"],
              fb["lse"])
    dH_b0, dW_b0 = B.gc_grpo_loss_bwd(*args_b)
    dH_b1, dW_b1 = B.gc_grpo_loss_bwd(*args_b, fwd_state=fb["state"])     # latest: used
    assert torch.equal(dH_b0, dH_b1) and torch.equal(dW_b0, dW_b1)
    # the C call refuses a forward state that overlaps its own workspace (a raw tensor bypasses the
    # binding's bookkeeping: here the backward's cached workspace itself)
    nb = int(B.lib().gc_bwd_workspace_bytes(bb.T, wb.D, wb.V, B.GC_BF16, 0, B.GC_F32))
    with pytest.raises(B.GcoreError, match="GC_ERR_ARG"):
        B.gc_grpo_loss_bwd(*args_b, fwd_state=B.workspace(nb, bb.H.device))


def test_host_entry_points_banded_copy_and_training_step(B):
    """The *_host entry points with H long enough to travel in several bands (copy of band b + 1
    overlapped with the scoring of band b on a side stream): log-probs against the oracle, and the
    whole training step from host buffers (gc_grpo_step_host) against the device-resident calls
    and the oracle."""
    w = I.reduced(I.CONFIGS[2], D=64, V=300, groups=4, group_size=4, seq_len=2600, prompt_len=100,
                  old_std=0.3)
    b = make_batch(w, seed=13, device="cuda")
    assert b.T > 2 * 16384                                  # > 2 bands of 64 M tiles
    pin = lambda t: t.cpu().pin_memory()
    Hh, yh, mh = pin(b.H), pin(b.y), pin(b.mask_t)
    lph = torch.empty(b.T, dtype=torch.float32).pin_memory()
    enh = torch.empty(b.T, dtype=torch.float32).pin_memory()
    for _ in range(2):                                      # second call: staging buffers reused
        lph.fill_(7.0)
        B.gc_token_logprobs_host(Hh, b.W, yh, mh, w.tau, logp_host=lph, entropy_host=enh)
        torch.cuda.synchronize()
        lp_o, en_o, _ = O.token_logprobs(to_f64(b.H), to_f64(b.W), b.y_np, b.mask_np, w.tau)
        assert np.abs(lph.numpy() - lp_o).max() <= TOL_LOGP_BF16
        assert np.abs(enh.numpy() - en_o).max() <= 2 * TOL_LOGP_BF16
    # training step from host buffers
    adv_ref, _ = O.grpo_advantages(b.rewards_np, b.lay.group_offsets, 1e-6)
    ref = oracle_run(b, adv_ref)
    dev_run = run_gpu(B, b)
    for dw_dtype in (torch.float32, torch.bfloat16):
        dW = torch.full((w.V, w.D), 5.0, dtype=dw_dtype, device="cuda")
        out5_h, dH_h = B.gc_grpo_step_host(Hh, b.W, yh, mh, w.tau, pin(b.cu_t), pin(b.rewards_t),
                                           pin(b.go_t), pin(b.old_t), pin(b.ref_t), dW,
                                           clip_lo=w.clip_lo, clip_hi=w.clip_hi, beta=w.beta)
        torch.cuda.synchronize()
        o = out5_h.numpy().astype(np.float64)
        assert o[4] == ref["n_scored"]
        assert abs(o[0] - ref["loss"]) <= TOL_LOSS_REL * abs(ref["loss"])
        assert rel_fro(dH_h.float().numpy(), ref["dH"]) <= TOL_GRAD_BF16
        assert rel_fro(dW.float().cpu().numpy(), ref["dW"]) <= TOL_GRAD_BF16 + (3e-3 if dw_dtype == torch.bfloat16 else 0)
        assert np.allclose(o[:4], dev_run["out5"].cpu().numpy()[:4], rtol=2e-5, atol=1e-7)
        assert elem_excess(dH_h.float().numpy(), ref["dH"], **ELEM_BF16) <= 1.0


def test_host_logprobs_at_a_shape_whose_band_needs_more_scratch_than_the_batch(B):
    """T=6144, D=4096, V=50304: the second H band (5376 rows) plans more vocab splits than the whole
    batch does, so its partial statistics need more workspace than the full-T query returns; the
    host entry point used to answer GC_ERR_WORKSPACE here.  Host path against the device path
    (itself oracle-checked) and against the oracle on sampled rows."""
    T, D, V = 6144, 4096, 50304
    g = torch.Generator(device="cuda").manual_seed(77)
    H = (torch.randn(T, D, device="cuda", generator=g)).to(torch.bfloat16)
    W = (torch.randn(V, D, device="cuda", generator=g) / D ** 0.5).to(torch.bfloat16)
    y = torch.randint(0, V, (T,), device="cuda", generator=g, dtype=torch.int32)
    lp_d, en_d, _ = B.gc_token_logprobs(H, W, y, None, 1.0)
    lph = torch.empty(T, dtype=torch.float32).pin_memory()
    enh = torch.empty(T, dtype=torch.float32).pin_memory()
    B.gc_token_logprobs_host(H.cpu().pin_memory(), W, y.cpu().pin_memory(), None, 1.0,
                             logp_host=lph, entropy_host=enh)
    torch.cuda.synchronize()
    assert np.abs(lph.numpy() - lp_d.cpu().numpy()).max() <= TOL_LOGP_BF16
    assert np.abs(enh.numpy() - en_d.cpu().numpy()).max() <= 2 * TOL_LOGP_BF16
    rows = [0, 511, 512, 767, 768, 5000, T - 1]          # both bands, their edges
    lp_o, en_o, _ = O.token_logprobs(to_f64(H[rows]), to_f64(W), y[rows].cpu().numpy(), None, 1.0)
    assert np.abs(lph.numpy()[rows] - lp_o).max() <= TOL_LOGP_BF16
    assert np.abs(enh.numpy()[rows] - en_o).max() <= 2 * TOL_LOGP_BF16
