"""-m gpu: the tcgen05 GEMM kernel against a plain fp32 matmul of the same bf16 operands."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("m,n,k", [(128, 64, 64), (1000, 256, 128), (4096, 1024, 1024), (18944 + 77, 1024, 64), (300, 128, 384), (257, 256, 64), (129, 128, 128), (5000, 1024, 1024),
                                   (1, 64, 64)])
@pytest.mark.parametrize("relu", [True, False])
@pytest.mark.parametrize("pair", [1, 0], ids=["cta_pair", "single_cta"])
def test_gemm_bias_act_matches_fp32_reference(m, n, k, relu, pair):
    import torch
    from paper_2501_05520_b200 import gemm_bf16
    g = torch.Generator(device="cuda").manual_seed(m * 7 + n * 3 + k)
    a = (torch.randn(m, k, device="cuda", generator=g)).to(torch.bfloat16)
    w = (torch.randn(n, k, device="cuda", generator=g) / np.sqrt(k)).to(torch.bfloat16)
    b = torch.randn(n, device="cuda", generator=g)
    out = gemm_bf16(a, w, b, relu=relu, pair=pair)
    torch.cuda.synchronize()
    ref = a.float() @ w.float().t() + b
    if relu:
        ref = torch.relu(ref)
    err = (out.float() - ref).abs().max().item()
    scale = ref.abs().max().item()
    assert err <= 2.0 ** -8 * scale + 1e-3, f"max err {err} (scale {scale})"     # one bf16 rounding of the output
    # exact integers: products and sums representable in fp32 -> result exact after the bf16 output rounding
    ai = torch.randint(-3, 4, (m, k), device="cuda", generator=g).to(torch.bfloat16)
    wi = torch.randint(-2, 3, (n, k), device="cuda", generator=g).to(torch.bfloat16)
    outi = gemm_bf16(ai, wi, torch.zeros(n, device="cuda"), relu=False, pair=pair)
    refi = (ai.float() @ wi.float().t()).to(torch.bfloat16)
    assert torch.equal(outi, refi)
