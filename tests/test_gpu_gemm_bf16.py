"""-m gpu: the tcgen05 BF16 GEMM building block (pnn_gemm_bf16) against an FP64 matmul of the same BF16 operands.
Products of BF16 numbers are exact in FP32 and the accumulation is FP32, so the only error is summation rounding:
|err| <= ~K * 2^-24 * sum|a||w| — the bound used below."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("M,N,K", [(128, 32, 32), (1000, 96, 96), (300, 128, 256), (4133, 384, 128), (2500, 768, 256),
                                   (777, 256, 512), (129, 512, 768), (1, 64, 64),
                                   # >= 8 x 148 tiles: the persistent kernel (double-buffered TMEM accumulator)
                                   (160001, 256, 128), (200003, 96, 64), (90000, 768, 256)])
@pytest.mark.parametrize("act", [0, 1])
def test_gemm_bf16_matches_fp64(M, N, K, act):
    import torch
    import paper_2604_15380_b200 as pnn
    g = torch.Generator(device="cpu").manual_seed(M * 7 + N * 3 + K + act)
    A = torch.randn(M, K, generator=g).to(torch.bfloat16).cuda()
    W = (torch.randn(N, K, generator=g) / K ** 0.5).to(torch.bfloat16).cuda()
    bias = torch.randn(N, generator=g).cuda()
    C = torch.full((M, N), float("nan"), device="cuda")
    Cb = torch.zeros((M, N), dtype=torch.bfloat16, device="cuda")
    pnn.pnn_gemm_bf16(M, N, K, A, K, W, K, bias, act, C, N, Cb, N, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    ref = A.double() @ W.double().T + bias.double()
    bound = (A.double().abs() @ W.double().abs().T + bias.double().abs()) * (K * 2.0 ** -24) + 1e-30
    if act == 1:
        ref = torch.nn.functional.silu(ref)
        bound = bound * 1.2 + 2e-7 * ref.abs()
    err = (C.double() - ref).abs()
    assert torch.isfinite(C).all()
    assert (err <= bound * 2 + 1e-7).all(), float((err / bound).max())
    assert ((Cb.double() - ref).abs() <= ref.abs() * 2.0 ** -8 + bound * 2 + 1e-7).all()
    # the BF16 copy (for large M it leaves through shared memory and a TMA store) is the FP32 output rounded, element by element
    assert torch.equal(Cb, C.to(torch.bfloat16))


def test_gemm_bf16_strided_and_outputs_optional():
    import torch
    import paper_2604_15380_b200 as pnn
    M, N, K, lda = 515, 128, 64, 192
    g = torch.Generator(device="cpu").manual_seed(3)
    Abig = torch.randn(M, lda, generator=g).to(torch.bfloat16).cuda()
    W = torch.randn(N, K, generator=g).to(torch.bfloat16).cuda()
    C = torch.zeros((M, 2 * N), device="cuda")
    pnn.pnn_gemm_bf16(M, N, K, Abig[:, 64:], lda, W, K, None, 0, C[:, N:], 2 * N, None, 0,
                      torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    ref = Abig[:, 64:128].double() @ W.double().T
    assert (C[:, :N] == 0).all()
    assert ((C[:, N:].double() - ref).abs() <= 1e-4 * (1 + ref.abs())).all()


def test_measured_alu_peak_is_near_the_derived_one():
    """the plain-ALU roofs are measured on the box.  Derived: 148 SMs x 128 (64) lanes x 2 x 1.965 GHz =
    74.4 (37.2) TFLOP/s; the packed-FMA micro-benchmark must land within 15 % of it and never above."""
    from paper_2604_15380_b200 import binding as B
    p32 = B.pnn_measure_alu_peak(B.PNN_FP32)
    p64 = B.pnn_measure_alu_peak(B.PNN_FP64)
    assert 0.85 * 74.45 < p32 < 1.02 * 74.45, p32
    assert 0.85 * 37.22 < p64 < 1.02 * 37.22, p64
    with pytest.raises(B.PnnError):
        B.pnn_measure_alu_peak(B.PNN_BF16)


def test_measured_l2_read_bandwidth_is_above_hbm_and_plausible():
    """pnn_measure_l2_peak (context for the gather-bound edge kernels in bench.py): L2-resident reads must be faster than
    the HBM copy peak of MEASURED_PEAKS.json (about 6.5 TB/s on this pool) and below what 148 SMs can take in (64 bytes per
    clock and SM at 1.965 GHz = 18.6 TB/s)."""
    from paper_2604_15380_b200 import binding as B
    v = max(B.pnn_measure_l2_peak() for _ in range(2))
    assert 6500.0 < v < 18600.0, v
