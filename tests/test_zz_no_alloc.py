"""apex4_w4a4_gemm_static_ws (-m gpu): the GEMM with its stream-K workspace in the library's static device array,
for callers that cannot call cudaMalloc.  Checked against the existing path (apex4_w4a4_gemm with a caller-owned
workspace) and the oracle, on two calls in a row; collected last (pytest -x stops at the first failure)."""
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


# (M, N, K, g, needs the workspace): stream-K problems of two sizes, a whole-tile problem and a decode problem
CASES = [(200, 520, 1024, 128, True), (256, 2048, 4096, 128, True), (300, 520, 1024, 32, True), (1024, 8192, 4096, 128, True),
         (192, 512, 512, 128, None), (16, 256, 512, 128, False)]


@pytest.mark.parametrize("M,N,K,g,needs_ws", CASES)
@pytest.mark.parametrize("out_dtype", [torch.float16, torch.float32])
def test_static_workspace_gemm_matches_existing_path(A, M, N, K, g, needs_ws, out_dtype):
    X, W = inputs.make_gemm_inputs(M, N, K, seed=900 + M)
    ref = O.w4a4_linear(X, W, g)
    G = K // g
    qA, sA, _ = A.quantize_act(dev(X), g)
    qW, sW, _ = A.pack_weights(dev(W), g)
    need = A.workspace_bytes(M, N, K, g)
    assert need <= A.STATIC_WORKSPACE_BYTES
    if needs_ws is not None:
        assert (need > 0) == needs_ws
    y_old = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, g, out_dtype=out_dtype)          # the existing path, own workspace
    out1 = torch.empty((M, N), dtype=out_dtype, device="cuda")
    out2 = torch.full((M, N), float("nan"), dtype=out_dtype, device="cuda")
    A.w4a4_gemm_static_ws(qA, sA, qW, sW, M, N, K, g, out=out1)                   # first use resolves the array's address
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # two calls in a row on one stream, no host synchronisation between them: the second starts from the first's contents
    A.w4a4_gemm_static_ws(qA, sA, qW, sW, M, N, K, g, out=out1)
    A.w4a4_gemm_static_ws(qA, sA, qW, sW, M, N, K, g, out=out2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0                                  # nothing was allocated on the device
    f16 = out_dtype == torch.float16
    tol = O.output_tolerance(ref["Y64"], ref["T"], G, f16)
    yo = y_old.cpu().numpy().astype(np.float64)
    for y in (out1, out2):
        yn = y.cpu().numpy().astype(np.float64)
        assert np.isfinite(yn).all()
        assert (np.abs(yn - ref["Y64"]) <= tol).all()                             # the oracle, the tests' tolerance
        assert (np.abs(yn - yo) <= tol).all()                                     # the existing path
        if need == 0:
            assert np.array_equal(yn, yo)                                         # same kernel, no reduction order in play


def test_static_workspace_covers_every_baseline_shape(A):
    """The stream-K workspace has one slot per CTA pair (<= 74 x 256 x 192 x 4 B + counters), so the 16 MiB static array
    holds it for every BASELINE.json shape and granularity; apex4_w4a4_gemm_static_ws returns APEX4_ERR_WORKSPACE only
    where apex4_workspace_bytes() exceeds the array (a device with more SMs)."""
    shapes = [(2048, 12288, 4096), (2048, 4096, 4096), (2048, 22016, 4096), (2048, 4096, 11008), (1024, 8192, 8192),
              (4096, 8192, 8192), (8192, 8192, 8192), (256, 10240, 8192), (4096, 57344, 8192), (4096, 8192, 28672)]
    worst = 0
    for M, N, K in shapes:
        for g in (32, 64, 128, K):
            worst = max(worst, A.workspace_bytes(M, N, K, g))
    assert 0 < worst <= A.STATIC_WORKSPACE_BYTES
