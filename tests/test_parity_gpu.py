"""GPU parity: the CUDA path, called through the C ABI, against the float64 oracle on the same seeded
inputs, element by element.  Tolerances are BASELINE.json north_star's: per-token log-prob abs err
<= 2e-3, loss rel err <= 1e-3, dHidden / dW rel-L2 <= 1e-2 (bf16 inputs, fp32 accumulation)."""
import numpy as np
import pytest
import torch

from tests.parity_util import (assert_gates, gates, make_ctx, rel_l2, run_cuda,
                               run_oracle, to64)
from workloads.synth import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2606_26997_b200.build import build
    build()


def _check(b, ctx_kw=None, oracle_kw=None, loss_denom=0.0, grad_scale=1.0):
    ctx = make_ctx(b, **(ctx_kw or {}))
    try:
        out = run_cuda(ctx, b, loss_denom=loss_denom, grad_scale=grad_scale)
        assert ctx.grpo_check_errors_sync() == 0
    finally:
        ctx.close()
    okw = dict(oracle_kw or {})
    ref = run_oracle(b, loss_denom=loss_denom if loss_denom > 0 else None, **okw)
    if grad_scale != 1.0:
        ref["dH"] *= grad_scale
        ref["dW"] *= grad_scale
    e = gates(b, out, ref, logit_scale=okw.get("logit_scale", 1.0), grad_scale=grad_scale)
    assert_gates(e)
    return out, ref, e


# ------------------------------------------------------------------ BASELINE config 1 and variants
def test_config1_exact_shape():
    b = make_config(1, device="cuda")
    out, ref, e = _check(b)
    np.testing.assert_allclose(to64(out["metrics"]), ref["metrics"], rtol=1e-4, atol=1e-4)
    assert e["dW_colsum_rel"] < 2e-3


def test_config1b_clip_regions_populated():
    b = make_config(1, device="cuda", variant="1b")
    out, ref, e = _check(b)
    frac = (ref["u"] == 0).mean()
    assert 0.03 < frac < 0.9          # zero-advantage groups and |log rho| < log 1.28 tokens are never clipped
    assert to64(out["metrics"])[3] == ref["metrics"][3]          # same tokens clipped


@pytest.mark.parametrize("kw", [
    dict(mask_frac=0.25), dict(loss_agg=1), dict(loss_agg=1, mask_frac=0.3), dict(bad_target_frac=0.15),
    dict(kl_beta=0.0), dict(kl_beta=0.05), dict(w_std=0.5), dict(w_std=1.5, variant="1b"),
])
def test_config1_variants(kw):
    b = make_config(1, device="cuda", seed=3, variant=kw.pop("variant", "1b"), **kw)
    _check(b, ctx_kw=dict(dhidden_fp32=1))


def test_sample_std_and_temperature():
    b = make_config(1, device="cuda", seed=4, variant="1b", w_std=0.3)
    _check(b, ctx_kw=dict(std_ddof=1, logit_scale=0.7), oracle_kw=dict(std_ddof=1, logit_scale=0.7))
    _check(b, ctx_kw=dict(logit_scale=1.9, dhidden_fp32=1), oracle_kw=dict(logit_scale=1.9), grad_scale=0.25)


def test_explicit_denominator_and_homogeneity():
    b = make_config(1, device="cuda", seed=5, variant="1b")
    out1, _, _ = _check(b, loss_denom=float(b.T))
    out2, _, _ = _check(b, loss_denom=float(b.T) / 4.0)
    np.testing.assert_allclose(out2["loss"].item(), 4 * out1["loss"].item(), rtol=1e-5)
    assert rel_l2(to64(out2["dW"]), 4 * to64(out1["dW"])) < 2e-3


def test_zero_variance_groups_give_exact_zeros():
    b = make_config(1, device="cuda", seed=6, kl_beta=0.0)
    b.rewards = torch.tensor([1.0] * 4 + [0.0] * 4 + [1, 0, 1, 0] + [0.5] * 4, device="cuda")
    out, ref, _ = _check(b)
    zv = out["zero_var"].cpu().numpy()
    np.testing.assert_array_equal(zv, [1, 1, 0, 1])
    cu = b.cu_seqlens.cpu().numpy()
    dH = out["dH"].float().cpu().numpy()
    for g in (0, 1, 3):
        assert np.all(to64(out["adv"])[4 * g:4 * g + 4] == 0.0)
        assert np.all(dH[cu[4 * g]:cu[4 * g + 4]] == 0.0)          # zero advantage, beta = 0 => zero gradient
    assert np.any(dH[cu[8]:cu[12]] != 0.0)


def test_all_masked_gives_zero_loss_and_grads():
    b = make_config(1, device="cuda", seed=7)
    b.mask = torch.zeros(b.T, dtype=torch.uint8, device="cuda")
    ctx = make_ctx(b)
    out = run_cuda(ctx, b)
    ctx.close()
    assert out["loss"].item() == 0.0
    assert torch.all(out["dW"] == 0) and torch.all(out["dH"].float() == 0)


def test_out_of_range_target_sets_error_flag():
    b = make_config(1, device="cuda", seed=8)
    b.targets[5] = b.V + 7
    ctx = make_ctx(b)
    out = run_cuda(ctx, b)
    assert ctx.grpo_check_errors_sync() == 1
    assert ctx.grpo_check_errors_sync() == 0                         # cleared by the read
    ctx.close()
    ref = run_oracle(b)
    assert abs(out["loss"].item() - ref["loss"]) <= 1e-3 * max(abs(ref["loss"]), ref["abs_loss"])


# ------------------------------------------------------------------ several tiles, ragged tails, chunked backward
@pytest.mark.parametrize("d,V,len_div,chunk", [(256, 5000, 20, 0), (72, 1000, 40, 0), (128, 3000, 10, 1024),
                                               (512, 2504, 30, 512)])
def test_config3_shaped_midsize(d, V, len_div, chunk):
    b = make_config(3, device="cuda", d=d, V=V, len_div=len_div, w_std=0.08)
    assert b.zero_var_frac > 0
    kw = dict(bwd_chunk_tokens=chunk) if chunk else {}
    _check(b, ctx_kw=kw)


def test_config4_shaped_large_groups():
    b = make_config(4, device="cuda", d=128, V=4096, len_div=40)
    _check(b)


@pytest.mark.parametrize("cfg_id,kw", [(1, dict(variant="1b")), (3, dict(d=256, V=5000, len_div=20, w_std=0.08))])
def test_single_cta_variant_parity(cfg_id, kw):
    """gemm_cta_group = 1 (cta_group::1, 128x256 tiles) stays a supported A/B reference of the default pair kernel."""
    b = make_config(cfg_id, device="cuda", **kw)
    _check(b, ctx_kw=dict(gemm_cta_group=1))


def test_single_token_and_tiny():
    b = make_config(1, device="cuda", seed=9, n_groups=1, G=2, len_div=100.0)   # every response 1 token
    assert b.T == 2
    _check(b)


# ------------------------------------------------------------------ determinism of the forward, run-to-run
def test_forward_is_deterministic():
    b = make_config(3, device="cuda", d=256, V=5000, len_div=20)
    ctx = make_ctx(b)
    a = run_cuda(ctx, b, want_dw=False, want_dh=False)
    c = run_cuda(ctx, b, want_dw=False, want_dh=False)
    ctx.close()
    assert torch.equal(a["logp"], c["logp"]) and torch.equal(a["coeff"], c["coeff"])


def test_backward_is_deterministic_on_one_stream():
    # every dW element receives exactly one reduce-add per backward chunk and the chunks run in stream order, so on
    # ONE stream the whole step is bit-reproducible (only launches that accumulate CONCURRENTLY into one dW, on
    # several streams, sum in an order the hardware picks: DESIGN.md section 5)
    b = make_config(3, device="cuda", d=256, V=5000, len_div=4)      # T ~ 13k: 50 blocks of A3, 26 chunks
    ctx = make_ctx(b, bwd_chunk_tokens=512)              # several chunks
    a = run_cuda(ctx, b)
    c = run_cuda(ctx, b)
    ctx.close()
    assert torch.equal(a["dH"], c["dH"]) and torch.equal(a["dW"], c["dW"])
    # the scalar loss and the metrics too: A3 sums its blocks in a fixed order (one add per launch and quantity)
    assert torch.equal(a["loss"], c["loss"]) and torch.equal(a["metrics"], c["metrics"])


# ------------------------------------------------------------------ end-to-end over host buffers == device path
def test_step_host_matches_device_path():
    b = make_config(3, device="cuda", d=256, V=5000, len_div=20)
    ctx = make_ctx(b)
    out = run_cuda(ctx, b)
    pin = lambda t: None if t is None else t.cpu().pin_memory()
    dW = torch.zeros_like(out["dW"])
    logp_h = torch.empty(b.T, dtype=torch.float32).pin_memory()
    dh_h = torch.empty(b.T, b.d, dtype=torch.bfloat16).pin_memory()
    loss_h = ctx.grpo_step_host(pin(b.hidden), pin(b.targets), pin(b.cu_seqlens), pin(b.rewards), pin(b.old_logp),
                                b.n_groups, b.G, b.W, dW, ref_logp_h=pin(b.ref_logp), mask_h=pin(b.mask),
                                logp_h=logp_h, dhidden_h=dh_h)
    ctx.close()
    assert torch.equal(logp_h, out["logp"].cpu())
    np.testing.assert_allclose(loss_h.item(), out["loss"].item(), rtol=1e-5)
    assert torch.equal(dh_h, out["dH"].cpu())
    assert rel_l2(to64(dW), to64(out["dW"])) < 1e-5


@pytest.mark.parametrize("d,V", [(72, 1003), (8, 9), (200, 257), (136, 5001)])
@pytest.mark.parametrize("fused", [False, True])
def test_odd_shapes(d, V, fused):
    """Widths that are not multiples of the 64-element K block (only d % 8 == 0 is required) and odd vocabulary
    sizes: K tails, partial 16-byte vectors at the row ends, V smaller than one tile; both backward variants."""
    b = make_config(1, device="cuda", seed=21, variant="1b", d=d, V=V, w_std=0.3)
    ctx = make_ctx(b, dhidden_fp32=1, bwd_chunk_tokens=128)
    try:
        out = run_cuda(ctx, b, fused=fused)
        assert ctx.grpo_check_errors_sync() == 0
    finally:
        ctx.close()
    assert_gates(gates(b, out, run_oracle(b)))


# ------------------------------------------------------------------ no write outside the caller's buffers
@pytest.mark.parametrize("d,V,fp32", [(72, 1003, 1), (8, 9, 0), (200, 257, 0), (136, 5001, 1), (64, 1000, 0)])
@pytest.mark.parametrize("fused", [False, True])
def test_outputs_are_written_inside_their_buffers(d, V, fp32, fused):
    """compute-sanitizer is closed on this GPU pool, so out-of-bounds writes are looked for directly: dHidden and dW
    live inside a pool filled with a sentinel, with guard bands on both sides, for shapes whose tiles, 32-byte store
    vectors and TMA reduce boxes all end ragged (d % 64 != 0, odd V, T not a multiple of the tile); the guard bands
    must come back untouched and the results must be those of ordinary buffers."""
    b = make_config(1, device="cuda", seed=31, variant="1b", d=d, V=V, w_std=0.3, mask_frac=0.2)
    guard = 4096                                                       # elements on each side
    dh_dtype = torch.float32 if fp32 else torch.bfloat16
    pool_h = torch.full((2 * guard + b.T * d,), 7.0, dtype=dh_dtype, device="cuda")
    pool_w = torch.full((2 * guard + V * d,), 7.0, dtype=torch.float32, device="cuda")
    dH = pool_h[guard:guard + b.T * d].view(b.T, d)
    dW = pool_w[guard:guard + V * d].view(V, d)
    dW.zero_()
    ctx = make_ctx(b, dhidden_fp32=fp32, bwd_chunk_tokens=128)
    try:
        adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
        if fused:
            ctx.grpo_fused_logprob_loss_fwd_bwd(b.hidden, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp,
                                                b.mask, dW_accum=dW, dhidden_out=dH)
        else:
            f = ctx.grpo_fused_logprob_loss_fwd(b.hidden, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp,
                                                b.mask)
            ctx.grpo_fused_logprob_loss_bwd(b.hidden, b.W, b.targets, f["lse"], f["coeff"], dW_accum=dW, dhidden_out=dH)
        torch.cuda.synchronize()
        ref = run_cuda(ctx, b, fused=fused)
    finally:
        ctx.close()
    for pool in (pool_h, pool_w):
        assert torch.all(pool[:guard] == 7.0) and torch.all(pool[-guard:] == 7.0)
    assert torch.equal(dH, ref["dH"]) and torch.equal(dW, ref["dW"])


@pytest.mark.parametrize("fused", [False, True])
def test_workspace_is_not_overrun(fused):
    """The library writes nothing beyond the grpo_workspace_bytes(max_T) it asked for: a step at exactly max_T tokens
    in a workspace of exactly that size, sentinel bytes behind it."""
    import ctypes as C
    from paper_2606_26997_b200 import GrpoContext
    b = make_config(3, device="cuda", d=136, V=2500, len_div=30, w_std=0.08, mask_frac=0.2)
    ctx = GrpoContext(b.d, b.V, eps_std=b.eps_std, clip_lo=b.clip_lo, clip_hi=b.clip_hi, kl_beta=b.kl_beta,
                      group_size=b.G, bwd_chunk_tokens=256)
    need = ctx.workspace_bytes(b.T)
    guard = 1 << 16
    pool = torch.full((need + 256 + guard,), 0x5A, dtype=torch.uint8, device="cuda")
    base = (pool.data_ptr() + 255) // 256 * 256
    off = base - pool.data_ptr()
    assert ctx.lib.grpo_set_workspace(ctx.h, C.c_void_p(base), need, b.T, 1) == 0
    ctx.workspace, ctx.max_tokens, ctx.n_slots = pool, b.T, 1          # the binding must not re-allocate
    try:
        out = run_cuda(ctx, b, fused=fused)
        assert ctx.grpo_check_errors_sync() == 0
    finally:
        ctx.close()
    assert torch.all(pool[off + need:] == 0x5A)
    assert_gates(gates(b, out, run_oracle(b)))


# ------------------------------------------------------------------ the step can be captured in a CUDA graph
def test_step_is_cuda_graph_capturable():
    """No call of the direct forward / backward synchronises or allocates (include/grpo.h): a whole step is captured
    into a CUDA graph and replayed with bit-identical results - for small, launch-bound groups the replay saves
    the per-launch host cost (98 -> 76 us per step at config 1's size)."""
    b = make_config(1, device="cuda", variant="1b")
    ctx = make_ctx(b, max_tokens=b.T)
    dW = torch.zeros(b.V, b.d, dtype=torch.float32, device="cuda")
    loss = torch.zeros(1, dtype=torch.float32, device="cuda")
    dH = torch.empty(b.T, b.d, dtype=torch.bfloat16, device="cuda")

    def step():
        adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
        f = ctx.grpo_fused_logprob_loss_fwd(b.hidden, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp,
                                            b.mask, loss_accum=loss)
        ctx.grpo_fused_logprob_loss_bwd(b.hidden, b.W, b.targets, f["lse"], f["coeff"], dW_accum=dW, dhidden_out=dH)
        return f

    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        step()                                                          # warm-up: function attributes, workspace
        torch.cuda.synchronize()
        dW.zero_(); loss.zero_()
        f = step()
    torch.cuda.synchronize()
    ref = (dW.clone(), dH.clone(), loss.clone(), f["logp"].clone())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        f = step()
    for _ in range(2):
        dW.zero_(); loss.zero_(); dH.zero_(); f["logp"].zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(dW, ref[0]) and torch.equal(dH, ref[1]) and torch.equal(loss, ref[2])
        assert torch.equal(f["logp"], ref[3])
    assert ctx.grpo_check_errors_sync() == 0
    ctx.close()


# ------------------------------------------------------------------ wide hidden sizes: L2-bounded unit orders
def test_wide_hidden_size_walks_its_units_in_l2_sized_groups():
    """d = 4352 (17 d tiles: the A5 / A6 units are walked in groups of 8, 8 and 1 tiles; 2.2 MB of hidden state per
    token tile: A2 blocks of 25 and A4 blocks of 17 token tiles, the last ones short) with T ~ 11k tokens (43 token
    tiles): only the ORDER of the units changes with these bounds, so the gates are the usual ones."""
    b = make_config(4, device="cuda", seed=2, d=4352, V=1500, len_div=38.0, w_std=0.05, old_sigma=0.3, mask_frac=0.1)
    assert b.T > 9500
    _check(b)


def test_implicit_token_mean_beyond_2_24_tokens_is_refused():
    """The loss-bearing token count behind an implicit denominator is an fp32 sum on the device: exact only up to
    2^24 tokens.  A larger call without loss_denom is refused (GRPO_ERR_SHAPE) before anything is launched; with an
    explicit denominator the same call runs (W = 0: uniform softmax, logp = -ln V for every token)."""
    from paper_2606_26997_b200 import GrpoContext, GrpoError
    T, d, V = (1 << 24) + 8, 8, 8
    ctx = GrpoContext(d, V, max_tokens=T)
    assert ctx.workspace_bytes(T) < 8 << 30
    z = lambda *shape, dt=torch.float32: torch.zeros(*shape, dtype=dt, device="cuda")
    hidden, W, y = z(T, d, dt=torch.bfloat16), z(V, d, dt=torch.bfloat16), z(T, dt=torch.int32)
    cu = torch.tensor([0, T], dtype=torch.int32, device="cuda")
    adv, old = torch.ones(1, device="cuda"), torch.full((T,), -float(np.log(V)), device="cuda")
    loss = z(1)
    with pytest.raises(GrpoError) as e:
        ctx.grpo_fused_logprob_loss_fwd(hidden, W, y, cu, adv, old, loss_accum=loss)
    assert e.value.status == 2 and "2^24" in str(e.value)
    torch.cuda.synchronize()
    assert loss.item() == 0.0                                          # nothing ran
    f = ctx.grpo_fused_logprob_loss_fwd(hidden, W, y, cu, adv, old, loss_denom=float(T), loss_accum=loss)
    torch.cuda.synchronize()
    assert ctx.grpo_check_errors_sync() == 0
    assert (f["logp"] + float(np.log(V))).abs().max().item() <= 1e-6
    assert abs(loss.item() + 1.0) <= 1e-3                              # rho = 1, A = 1: loss = -mean(rho A) = -1
    ctx.close()
