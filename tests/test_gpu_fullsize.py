"""GPU parity at BASELINE.json's full sizes (-m gpu), in the launch configuration bench.py times (automatic
dispatch, FP16 output): SURVEY.md 8(d) "Parity coverage at scale".  For every shape of configs 1-4 the
oracle computes (i) a row set -- tile edges plus seeded random rows -- against ALL N columns and (ii) a column
set built the same way against ALL M rows, so every M-tile and every N-tile of the GPU grid is touched;
codes and scales of BOTH operands are compared in full (bit-exact), per-group INT32 sums bit-exactly on
8 x 8 windows at tile corners through apex4_debug_group_sums.  Also here: the headroom pin at the longest
supported row (all-(-8) codes, per-channel K = 28672), the scaled-identity pin (zero weight scales, R4) on
the GPU, and the rho microbenchmark's sanity ranges."""
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


def oracle_quantize_rows(X, g, chunk=1024):
    """O.quantize on row chunks (its float64 temporaries of a whole 57344 x 8192 operand would not fit);
    rows are independent in Eq. 7, so this is the same function call by call."""
    q = np.empty(X.shape, dtype=np.int8)
    s = np.empty((X.shape[0], X.shape[1] // g), dtype=np.float16)
    for r0 in range(0, X.shape[0], chunk):
        q[r0:r0 + chunk], s[r0:r0 + chunk] = O.quantize(X[r0:r0 + chunk], g)
    return q, s


def check_output(Y_gpu, Y64, T, G):
    tol = O.output_tolerance(Y64, T, G, True)
    err = np.abs(Y_gpu.astype(np.float64) - Y64)
    bad = err > tol
    assert not bad.any(), (int(bad.sum()), float((err / np.maximum(tol, 1e-300)).max()), np.argwhere(bad)[:5].tolist())


_W_CACHE = {}


def weights_for(A, N, K, seed, g, gran, layer):
    """(packed weights on the GPU, oracle codes, oracle scales), cached per shape: the M sweeps reuse one W."""
    key = (N, K, seed, g)
    if key not in _W_CACHE:
        _W_CACHE.clear()                              # one big operand at a time
        W = inputs.make_weights(N, K, seed)
        qw, sw = oracle_quantize_rows(W, g)
        qW, sW, g_res = A.pack_weights(dev(W), 128, gran, layer) if gran != A.GRAN_GROUP else A.pack_weights(dev(W), g)
        assert g_res == g
        # a0: codes and scales of the whole operand, bit-exact
        assert np.array_equal(A.unpack_codes(qW, N, K, A.OPERAND_WEIGHT).cpu().numpy(), qw)
        assert np.array_equal(A.scales_to_natural(sW, N, K // g).cpu().numpy().view(np.uint16), sw.view(np.uint16))
        _W_CACHE[key] = (qW, sW, qw, sw)
    return _W_CACHE[key]


def sampled_parity(A, M, N, K, g, seed, fixed_outliers, gran=None, layer=None, X=None):
    gran = A.GRAN_GROUP if gran is None else gran
    layer = A.LAYER_OTHER if layer is None else layer
    gs_arg = g if gran == A.GRAN_GROUP else 128
    assert A.resolve_group_size(K, gs_arg, gran, layer) == g
    G = K // g
    qW, sW, qw, sw = weights_for(A, N, K, seed, g, gran, layer)
    if X is None:
        X = inputs.make_activations(M, K, seed, fixed_outliers)
    qa, sa = oracle_quantize_rows(X, g)
    qA, sA, g_res = A.quantize_act(dev(X), gs_arg, gran, layer)
    assert g_res == g
    # a1: every element of the activation operand
    assert np.array_equal(A.unpack_codes(qA, M, K, A.OPERAND_ACT).cpu().numpy(), qa)
    assert np.array_equal(A.scales_to_natural(sA, M, G).cpu().numpy().view(np.uint16), sa.view(np.uint16))
    ws = A.make_workspace(M, N, K, gs_arg, gran, layer)
    Y = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, gs_arg, gran, layer, workspace=ws).cpu().numpy()
    if ws is not None:
        assert int(ws.count_nonzero()) == 0
    rows = inputs.sample_rows(M, seed + 1)
    cols = inputs.sample_rows(N, seed + 2)
    Y64, T = O.dequant_gemm(qa[rows], sa[rows], qw, sw, g)
    check_output(Y[rows], Y64, T, G)
    Y64, T = O.dequant_gemm(qa, sa, qw[cols], sw[cols], g)
    check_output(Y[:, cols], Y64, T, G)
    # a4: per-group integer sums on windows at tile corners (first / interior / last rows and columns)
    wm = sorted({0, max(0, min(M - 8, 184)), max(0, (M // 2) // 8 * 8 - 8), max(0, M - 8)})
    wn = sorted({0, max(0, min(N - 8, 248)), max(0, (N // 2) // 8 * 8), max(0, N - 8)})
    for m0 in wm:
        for n0 in (wn if m0 in (wm[0], wm[-1]) else wn[:1]):
            m1, n1 = min(M, m0 + 8), min(N, n0 + 8)
            P = A.debug_group_sums(qA, qW, M, N, K, gs_arg, gran, layer, m0=m0, m1=m1, n0=n0, n1=n1).cpu().numpy()
            assert np.array_equal(P, O.group_sums(qa[m0:m1], qw[n0:n1], g)), (m0, n0)


# ------------------------------------------------------------------------------- config 1
@pytest.mark.parametrize("idx,name", list(enumerate(inputs.LLAMA2_7B_SHAPES)))
def test_config1_llama2_7b_layers(A, idx, name):
    """BASELINE.json configs[1]: the four Llama-2-7B linears at M = 2048, g = 128 (what bench.py's step times)."""
    N, K = inputs.LLAMA2_7B_SHAPES[name]
    sampled_parity(A, 2048, N, K, 128, inputs.config_seed(1, idx), True)


# ------------------------------------------------------------------------------- config 2
@pytest.mark.parametrize("M", [64, 256, 1024, 8192])
def test_config2_square_sweep(A, M):
    """BASELINE.json configs[2]: N = K = 8192, g = 128 (M <= 16 is covered in full by test_gpu_parity);
    nested sweep: the first M rows of one draw."""
    seed = inputs.config_seed(2, 0)
    sampled_parity(A, M, 8192, 8192, 128, seed, False)


def test_config2_decode_sizes_full_output(A):
    """M = 1, 4, 16 at N = K = 8192: every output and every window against the oracle."""
    seed = inputs.config_seed(2, 0)
    for M in (1, 4, 16):
        sampled_parity(A, M, 8192, 8192, 128, seed, False)


# ------------------------------------------------------------------------------- config 3
@pytest.mark.parametrize("g", [32, 64, 128, 8192])
def test_config3_granularity_sweep(A, g):
    sampled_parity(A, 4096, 8192, 8192, g, inputs.config_seed(3, 0), False)


@pytest.mark.parametrize("gran_name,layer_name,g", [("GRAN_MIXED", "LAYER_DOWN", 32), ("GRAN_MIXED", "LAYER_O", 8192),
                                                      ("GRAN_MIXED_G128", "LAYER_V", 128), ("GRAN_MIXED_G128", "LAYER_GATE_UP", 8192)])
def test_config3_mixed_policies(A, gran_name, layer_name, g):
    """The paper's mix (fine = 32) and BASELINE.json's wording (fine = 128), g resolved by the library from the
    layer kind (R11)."""
    sampled_parity(A, 4096, 8192, 8192, g, inputs.config_seed(3, 0), False, gran=getattr(A, gran_name),
                   layer=getattr(A, layer_name))


# ------------------------------------------------------------------------------- config 4
@pytest.mark.parametrize("idx,name", list(enumerate(inputs.LLAMA2_70B_SHAPES)))
def test_config4_llama2_70b_layers(A, idx, name):
    """BASELINE.json configs[4]: the four Llama-2-70B linears at M = 16 (decode kernel) and M = 4096 (pair kernel);
    M = 1 and 256 on the two shapes with the extreme N and K."""
    N, K = inputs.LLAMA2_70B_SHAPES[name]
    seed = inputs.config_seed(4, idx)
    X = inputs.make_activations(4096, K, seed, False)
    Ms = (16, 4096) + ((1, 256) if name in ("gate_up", "down") else ())
    for M in Ms:
        sampled_parity(A, M, N, K, 128, seed, False, X=X[:M])


# ------------------------------------------------------------------------------- pins on the GPU
@pytest.mark.parametrize("kernel", [0, 1])
def test_minus8_codes_headroom_per_channel_k28672(A, kernel):
    """R5 / P3 headroom at the longest supported row: all-(-8) codes, per-channel K = 28672, through the CH decode
    kernel (INT32 partial sums across 16 warps, |256 P| = 4.7e8) and the pair kernel (I2F epilogue)."""
    M, N, K = 8, 256, 28672
    qA = A.pack_codes(dev(np.full((M, K), -8, dtype=np.int8)), A.OPERAND_ACT)
    qW = A.pack_codes(dev(np.full((N, K), -8, dtype=np.int8)), A.OPERAND_WEIGHT)
    o = A.debug_opts(kernel=kernel)
    P = A.debug_group_sums(qA, qW, M, N, K, K, opts=o).cpu().numpy()
    assert P.shape == (M, N, 1) and np.all(P == 64 * K) and 64 * K == 1835008
    sA = A.scales_from_natural(dev(np.full((M, 1), 0.5, dtype=np.float16)))
    sW = A.scales_from_natural(dev(np.full((N, 1), 0.25, dtype=np.float16)))
    Y = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, K, out_dtype=torch.float32, opts=o).cpu().numpy()
    assert np.all(Y == 64.0 * K * 0.125)              # 229376, exact in FP32
    # ... and through g = 128 on the same operands: P = 8192 per group
    P = A.debug_group_sums(qA, qW, M, N, K, 128, m1=2, n1=16, opts=o).cpu().numpy()
    assert np.all(P == 8192)


@pytest.mark.parametrize("M,opts", [(16, dict(kernel=0)), (16, dict(kernel=1)), (40, dict(kernel=1, pair_tokens=64)),
                                    (200, dict(kernel=1, pair_tokens=192)), (200, dict(kernel=1, pair_tokens=128, split=1, grid=3))])
@pytest.mark.parametrize("g", [32, 128])
def test_scaled_identity_zero_weight_scales(A, M, opts, g):
    """P4 on the GPU: N = K, W = 0.5 I.  Every weight group but the diagonal's has absmax 0 -> S = 0, codes 0
    (R4); Y[m, n] = sA[m, gamma(n)] qA[m, n] * 0.4998779296875: fails if the kernel pairs sA[m, gamma] with the
    wrong group, and exercises zero scales on the GEMM path."""
    N = K = 1024
    rng = np.random.default_rng(40 + M)
    X = rng.standard_normal((M, K)).astype(np.float16)
    W = (0.5 * np.eye(N)).astype(np.float16)
    ref = O.w4a4_linear(X, W, g)
    assert int((ref["sW"].view(np.uint16) != 0).sum()) == N           # one non-zero scale per row
    o = A.debug_opts(**opts)
    qA, sA, _ = A.quantize_act(dev(X), g)
    qW, sW, _ = A.pack_weights(dev(W), g)
    assert np.array_equal(A.scales_to_natural(sW, N, K // g).cpu().numpy().view(np.uint16), ref["sW"].view(np.uint16))
    Y = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, g, out_dtype=torch.float32, opts=o).cpu().numpy()
    want = ref["sA"].astype(np.float64).repeat(g, axis=1) * ref["qA"].astype(np.float64) * (7 * 0.0714111328125)
    assert np.array_equal(want, ref["Y64"])                          # the closed form, typed out
    # one term per output: the FP32 result is that term rounded once
    assert np.array_equal(Y, want.astype(np.float32))
    P = A.debug_group_sums(qA, qW, M, N, K, g, opts=o).cpu().numpy()
    assert np.array_equal(P, O.group_sums(ref["qA"], ref["qW"], g))


def test_rho_microbenchmark_ranges(A):
    """apex4_measure_rho (Eq. 1-2): B200 per SM and clock -- 8192 INT8 MAC on the tensor pipe,
    128 FP32 FMA lanes, 64 I2F lanes -> rho = 16384 / 256 = 64 nominal."""
    r = A.measure_rho()
    assert 7000 <= r["int8_mac_per_clk_sm"] <= 8300, r
    fma_per_clk_sm = r["fp32_tflops"] * 1e12 / 2 / (r["sm_clock_mhz"] * 1e6) / torch.cuda.get_device_properties(0).multi_processor_count
    assert 100 <= fma_per_clk_sm <= 130, (fma_per_clk_sm, r)
    assert 50 <= r["rho"] <= 70, r
    assert abs(r["rho"] - r["int8_tops"] / r["fp32_tflops"]) < 1e-6 * r["rho"]
    assert 150 <= r["tmem_ld_bytes_per_clk_sm"] <= 1100, r


def test_epilogue_stream_probe_is_ordered(A):
    """apex4_measure_epilogue_stream: adding work to the stream never makes it faster, the FMA-only stream cannot beat
    its FMA-pipe time (2 warps x 96 FFMA2 x 2 clk = 384 clk per sub-partition and group), and the full stream stays
    below the pair kernel's measured group period (~1150 clk)."""
    r = A.measure_epilogue_stream()
    assert r["ld"] < r["ld+st"] < r["ld+st+fma"] <= r["ld+st+lds+fma"] * 1.02, r
    assert r["ld"] < r["ld+fma"] <= r["ld+lds+fma"] * 1.02 and r["ld+lds+fma"] < r["ld+st+lds+fma"], r
    assert 384 <= r["ld+fma"] <= 700 and 500 <= r["ld+st+lds+fma"] <= 1150, r


@pytest.mark.parametrize("encoding", [0, 1])
def test_e4m3_tensor_path_is_exact_on_int4_codes(A, encoding):
    """SURVEY 8(f)4 experiment (measured fact on B200, recorded in DESIGN.md): tcgen05.mma kind::f8f6f4 with the
    codes as E4M3 operands and FP32 accumulation reproduces the kind::i8 sums exactly, up to per-channel K = 32768
    (sums up to 2^21), for random, extreme, cancelling and odd-increment inputs; and the kind::i8 sums of the all-(-8)
    pattern equal the closed form 64 K."""
    for pattern in range(6):
        for K in (128, 4096, 32768):
            r = A.e4m3_exactness(K, pattern, encoding, seed=11 + pattern)
            assert r["compared"] == 128 * 256
            assert r["int8_vs_closed_form_mismatches"] == 0
            assert r["mismatches"] == 0 and r["max_abs_diff"] == 0.0, (pattern, K, r)
            if pattern == 1:
                assert r["max_abs_sum"] == 64 * K
