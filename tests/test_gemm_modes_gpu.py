"""The production tcgen05 kernel as a plain GEMM (test hook grpo_debug_gemm), one case per operand
layout the GRPO step uses, against a float64 matmul of the same bf16 inputs."""
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", params=[(2, 0), (1, 0), (2, 1), (2, -1)],
                ids=["cta_pair", "single_cta", "cta_pair_gate_every_kblock", "cta_pair_gate_off"])
def ctx(request):
    """Both tcgen05 variants of the kernel: cta_group::2 pair tiles (the default) and cta_group::1; the
    drift gate (a performance-only producer throttle) at its default epoch, at the
    tightest epoch (every k block: the gate is exercised on every iteration) and off."""
    from paper_2606_26997_b200 import GrpoContext
    from paper_2606_26997_b200.build import build
    build()
    cg, drift = request.param
    c = GrpoContext(64, 1000, max_tokens=256, gemm_cta_group=cg, gemm_drift_epoch_kb=drift)
    yield c
    c.close()


def _ref(A, B, layout):
    A64, B64 = A.double(), B.double()
    if layout == 0:
        return A64 @ B64.T          # A [M,K], B [N,K]
    if layout == 1:
        return A64 @ B64            # A [M,K], B [K,N]
    return A64.T @ B64              # A [K,M], B [K,N]


# shapes span several 128x256 / 256x256 tiles, ragged M/N tails (including a pair whose second CTA is
# entirely out of range), K tails (not a multiple of 64), tiny K, and more k blocks than ring stages
SHAPES = [(128, 256, 64), (256, 512, 128), (200, 264, 72), (1000, 2048, 320), (136, 64, 1000), (8, 8, 8),
          (384, 1000, 2048), (2048, 136, 4096)]


@pytest.mark.parametrize("layout", [0, 1, 2])
@pytest.mark.parametrize("M,N,K", SHAPES)
def test_gemm_layouts(ctx, layout, M, N, K):
    g = torch.Generator(device="cuda").manual_seed(1000 * layout + M + N + K)
    a_shape = (M, K) if layout < 2 else (K, M)
    b_shape = (N, K) if layout == 0 else (K, N)
    A = torch.randn(a_shape, generator=g, device="cuda").to(torch.bfloat16)
    B = torch.randn(b_shape, generator=g, device="cuda").to(torch.bfloat16)
    C = ctx.grpo_debug_gemm(layout, A, B, M, N, K)
    torch.cuda.synchronize()
    ref = _ref(A, B, layout)
    err = (C.double() - ref).abs().max().item()
    scale = ref.abs().max().item()
    assert err <= 2e-5 * max(scale, 1.0) * max(1.0, (K / 64) ** 0.5), (layout, M, N, K, err, scale)
    # accumulate variant: C += A B
    C2 = ctx.grpo_debug_gemm(layout, A, B, M, N, K, C_out=C.clone(), accumulate=True)
    torch.cuda.synchronize()
    err2 = (C2.double() - 2 * ref).abs().max().item()
    assert err2 <= 4e-5 * max(scale, 1.0) * max(1.0, (K / 64) ** 0.5)
