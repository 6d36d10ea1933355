"""GPU parity of the producer-fused quantizers (-m gpu): apex4_rmsnorm_quantize / apex4_silu_mul_quantize against
quantize(rmsnorm(.)) / quantize(silu_mul(.)) of the CPU oracle (readings R17 / R18): the FP16 intermediate, the
INT4 codes and the FP16 scales are all compared bit for bit, then fed through the GEMM."""
import numpy as np
import pytest
import torch

from oracle import apex4_oracle as O
from paper_2606_08761_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def A():
    from paper_2606_08761_b200 import apex4
    apex4.lib()
    assert torch.cuda.is_available()
    return apex4


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def check_quantized(A, q, s, y_gpu, y_ref, g):
    M, K = y_ref.shape
    if y_gpu is not None:
        assert np.array_equal(y_gpu.cpu().numpy().view(np.uint16), y_ref.view(np.uint16))
    qo, so = O.quantize(y_ref, g)
    assert np.array_equal(A.scales_to_natural(s, M, K // g).cpu().numpy().view(np.uint16), so.view(np.uint16))
    assert np.array_equal(A.unpack_codes(q, M, K, A.OPERAND_ACT).cpu().numpy(), qo)
    return qo, so


@pytest.mark.parametrize("M,K,g", [(16, 512, 128), (5, 4096, 128), (130, 1024, 32), (33, 3584, 64), (7, 4096, 4096),
                                   (3, 11008, 128), (2, 28672, 28672), (64, 8192, 1024), (1, 128, 128)])
def test_rmsnorm_quantize_bit_exact(A, M, K, g):
    X = inputs.make_activations(M, K, seed=900 + M, fixed_outliers=(K == 512))
    rng = np.random.default_rng(K + M)
    gamma = (1.0 + 0.2 * rng.standard_normal(K)).astype(np.float16)
    for eps in (1e-5, 1e-6, 0.0):
        y_ref = O.rmsnorm(X, gamma, eps)
        q, s, g_res, y = A.rmsnorm_quantize(dev(X), dev(gamma), eps, g, want_y=True)
        assert g_res == g
        check_quantized(A, q, s, y, y_ref, g)
    # without the optional FP16 copy
    q, s, _ = A.rmsnorm_quantize(dev(X), dev(gamma), 1e-5, g)
    check_quantized(A, q, s, None, O.rmsnorm(X, gamma, 1e-5), g)


def test_rmsnorm_quantize_extreme_rows(A):
    """All-zero rows (ms = 0: inv = 1/sqrt(eps)), huge and tiny magnitudes."""
    K = 1024
    X = np.zeros((6, K), dtype=np.float16)
    X[1] = np.float16(65504)
    X[2] = np.float16(6e-8)
    X[3, ::7] = np.float16(-300)
    X[4] = (np.random.default_rng(3).standard_normal(K) * 1e-3).astype(np.float16)
    X[5, 5] = np.float16(1)
    gamma = np.ones(K, dtype=np.float16)
    for eps in (1e-5, 1e-12):
        y_ref = O.rmsnorm(X, gamma, eps)
        q, s, _, y = A.rmsnorm_quantize(dev(X), dev(gamma), eps, 128, want_y=True)
        check_quantized(A, q, s, y, y_ref, 128)


def test_silu_mul_every_fp16_gate(A):
    """Every finite FP16 gate against several up values: the FP16 product bit for bit (fast path and the FP64 path)."""
    allb = np.arange(0x10000, dtype=np.uint32).astype(np.uint16)
    finite = allb[((allb >> 10) & 0x1F) != 0x1F].view(np.float16)
    K = 4096
    rows = (finite.size + K - 1) // K                     # 16 rows of 4096 gates per up value
    ups = [1.0, -1.0, 0.5, 3.0, 0.0999755859375, 1000.0, 6e-5, -0.33349609375]
    gate = np.zeros((len(ups) * rows, K), dtype=np.float16)
    up = np.zeros_like(gate)
    for i, u in enumerate(ups):
        gate[i * rows:(i + 1) * rows].reshape(-1)[:finite.size] = finite
        up[i * rows:(i + 1) * rows] = np.float16(u)
    y_ref = O.silu_mul(gate, up)
    q, s, _, y = A.silu_mul_quantize(dev(gate), dev(up), 128, want_y=True)
    bad = np.argwhere(y.cpu().numpy().view(np.uint16) != y_ref.view(np.uint16))
    assert bad.size == 0, (bad[:5].tolist(),)
    # codes and scales on the rows whose products stay finite (quantizing Inf is undefined, R16)
    keep = np.isfinite(y_ref.astype(np.float32)).all(axis=1)
    assert keep.sum() >= 5 * rows
    q, s, _, y = A.silu_mul_quantize(dev(gate[keep]), dev(up[keep]), 128, want_y=True)
    check_quantized(A, q, s, y, y_ref[keep], 128)


@pytest.mark.parametrize("M,K,g", [(16, 512, 128), (9, 11008, 128), (130, 1024, 32), (5, 18944, 64), (4, 11008, 11008), (40, 2048, 512)])
def test_silu_mul_quantize_bit_exact(A, M, K, g):
    rng = np.random.default_rng(1000 + M)
    GU = (rng.standard_normal((M, 2 * K)) * 2.5).astype(np.float16)       # a fused gate+up GEMM output [M, 2K]
    gu = dev(GU)
    y_ref = O.silu_mul(GU[:, :K], GU[:, K:])
    q, s, g_res, y = A.silu_mul_quantize(gu[:, :K], gu[:, K:], g, want_y=True)      # strided views, ld = 2K
    assert g_res == g
    check_quantized(A, q, s, y, y_ref, g)
    # separate contiguous tensors
    q, s, _ = A.silu_mul_quantize(dev(GU[:, :K]), dev(GU[:, K:]), g)
    check_quantized(A, q, s, None, y_ref, g)


def test_fused_quantizers_feed_the_gemm(A):
    """rmsnorm_quantize -> GEMM and silu_mul_quantize -> GEMM equal the oracle's linear layer on the oracle's y."""
    from test_gpu_parity import check_output
    M, N, K, g = 48, 264, 1024, 128
    X, W = inputs.make_gemm_inputs(M, N, K, 77)
    gamma = (1.0 + 0.1 * np.random.default_rng(5).standard_normal(K)).astype(np.float16)
    qW, sW, _ = A.pack_weights(dev(W), g)
    y = O.rmsnorm(X, gamma, 1e-5)
    ref = O.w4a4_linear(y, W, g)
    qA, sA, _ = A.rmsnorm_quantize(dev(X), dev(gamma), 1e-5, g)
    Y = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, g).cpu().numpy()
    check_output(Y, ref["Y64"], ref["T"], K // g, True)
    P = A.debug_group_sums(qA, qW, M, N, K, g).cpu().numpy()
    assert np.array_equal(P, O.group_sums(ref["qA"], ref["qW"], g))
    up = inputs.make_activations(M, K, 78, False)
    y2 = O.silu_mul(X, up)
    ref2 = O.w4a4_linear(y2, W, g)
    qA, sA, _ = A.silu_mul_quantize(dev(X), dev(up), g)
    Y = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, g).cpu().numpy()
    check_output(Y, ref2["Y64"], ref2["T"], K // g, True)


def test_quantizer_outputs_do_not_depend_on_buffer_contents(A):
    """The padding rows of the last 128-row blob (which the GEMM kernels bulk-copy) are written as zeros by every
    quantizer call: NaN-poisoned output buffers give the same GEMM result and leave the workspace clean."""
    from test_gpu_parity import check_output
    M, N, K, g = 100, 264, 1024, 128
    X, W = inputs.make_gemm_inputs(M, N, K, 55)
    ref = O.w4a4_linear(X, W, g)
    qW, sW, _ = A.pack_weights(dev(W), g)
    q = torch.full((A.packed_bytes(M, K),), 0xFF, dtype=torch.uint8, device="cuda")
    s = torch.full((A.scale_elems(M, K, g),), float("nan"), dtype=torch.float16, device="cuda")
    A.quantize_act(dev(X), g, q=q, s=s)
    assert not torch.isnan(s).any()
    for o in (None, A.debug_opts(kernel=1, pair_tokens=128, split=1, grid=3)):
        ws = A.make_workspace(M, N, K, g, opts=o)
        Y = A.w4a4_gemm(q, s, qW, sW, M, N, K, g, workspace=ws, opts=o).cpu().numpy()
        check_output(Y, ref["Y64"], ref["T"], K // g, True)
        if ws is not None:
            assert int(ws.count_nonzero()) == 0
    gamma = np.ones(K, dtype=np.float16)
    s.fill_(float("nan")); q.fill_(0xFF)
    A.rmsnorm_quantize(dev(X), dev(gamma), 1e-5, g, q=q, s=s)
    assert not torch.isnan(s).any() and int(A.unpack_codes(q, 128, K, A.OPERAND_ACT)[M:].count_nonzero()) == 0
