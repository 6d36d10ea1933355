"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle on the
same seeded inputs.  Bars: bit-exact INT4 codes, FP16 scales and per-group INT32 sums; outputs within
|y - Y64| <= 1e-3 |Y64| + (G+2) 2^-23 T (+ 2^-24 for FP16 output) -- reading R12 of DESIGN.md."""
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


def gpu_quantize(A, X, g, weights=False):
    """-> (q_packed, s_tiled, codes int8 numpy [R,K], scales fp16 numpy [R,G])"""
    R, K = X.shape
    fn = A.pack_weights if weights else A.quantize_act
    q, s, g_res = fn(dev(X), g)
    assert g_res == g
    codes = A.unpack_codes(q, R, K, A.OPERAND_WEIGHT if weights else A.OPERAND_ACT).cpu().numpy()
    scales = A.scales_to_natural(s, R, K // g).cpu().numpy()
    return q, s, codes, scales


def check_output(Y_gpu, Y64, T, G, f16):
    tol = O.output_tolerance(Y64, T, G, f16)
    err = np.abs(Y_gpu.astype(np.float64) - Y64)
    bad = err > tol
    assert not bad.any(), (int(bad.sum()), float((err / np.maximum(tol, 1e-300)).max()),
                           np.argwhere(bad)[:5].tolist())


# ------------------------------------------------------------------------------- quantizer (a0/a1)
@pytest.mark.parametrize("M,K,g", [(16, 512, 128), (16, 512, 32), (16, 512, 64), (16, 512, 256),
                                   (16, 512, 512), (1, 128, 128), (13, 1024, 1024), (130, 384, 128),
                                   (257, 2048, 2048), (5, 11008, 11008), (3, 28672, 28672),
                                   (300, 4096, 128)])
def test_quantizer_bit_exact(A, M, K, g):
    X = inputs.make_activations(M, K, seed=17 + M, fixed_outliers=(K == 512))
    qo, so = O.quantize(X, g)
    _, _, codes, scales = gpu_quantize(A, X, g)
    assert np.array_equal(scales.view(np.uint16), so.view(np.uint16))
    assert np.array_equal(codes, qo)


def test_quantizer_weights_config0(A):
    X, W, g = inputs.config0()
    qo, so = O.quantize(W, g)
    _, _, codes, scales = gpu_quantize(A, W, g, weights=True)
    assert np.array_equal(scales.view(np.uint16), so.view(np.uint16))
    assert np.array_equal(codes, qo)


def test_quantizer_exhaustive_fp16_inputs(A):
    """Every finite FP16 bit pattern through the GPU quantizer, for a set of group scales that
    includes FP16-subnormal scales (R4/R5), compared with the oracle element by element."""
    allb = np.arange(0x10000, dtype=np.uint32).astype(np.uint16)
    finite = allb[((allb >> 10) & 0x1F) != 0x1F].view(np.float16)
    mags = np.abs(finite.astype(np.float64))
    u = 2.0 ** -24
    for amax in (1.0, 7.0, 20.0, 0.0200042724609375, 65504.0, 3 * u, 10 * u, 11 * u, 100 * u, 0.33):
        cand = finite[mags <= amax]
        n = 32768                                   # per-channel rows of the maximum supported K
        per = n - 1
        rows = (cand.size + per - 1) // per
        X = np.zeros((rows, n), dtype=np.float16)
        for r in range(rows):
            part = cand[r * per:(r + 1) * per]
            X[r, :part.size] = part
            X[r, n - 1] = np.float16(amax)          # every row has the same absmax -> the same scale
        qo, so = O.quantize(X, n)
        _, _, codes, scales = gpu_quantize(A, X, n)
        assert np.array_equal(scales.view(np.uint16), so.view(np.uint16)), amax
        assert np.array_equal(codes, qo), amax
    # many groups with different scales in one launch (g = 32): random magnitudes incl. tiny ones
    rng = np.random.default_rng(5)
    X = (rng.standard_normal((64, 1024)) * np.exp2(rng.integers(-26, 12, size=(64, 1024 // 32)).repeat(32, 1))
         ).astype(np.float16)
    qo, so = O.quantize(X, 32)
    _, _, codes, scales = gpu_quantize(A, X, 32)
    assert np.array_equal(scales.view(np.uint16), so.view(np.uint16))
    assert np.array_equal(codes, qo)


def test_pack_unpack_roundtrip_and_scale_layout(A):
    rng = np.random.default_rng(9)
    codes = rng.integers(-8, 8, size=(200, 640)).astype(np.int8)
    for operand in (A.OPERAND_ACT, A.OPERAND_WEIGHT):
        q = A.pack_codes(dev(codes), operand)
        assert q.numel() == A.packed_bytes(200, 640)
        assert np.array_equal(A.unpack_codes(q, 200, 640, operand).cpu().numpy(), codes)
    s = rng.standard_normal((200, 5)).astype(np.float16)
    t = A.scales_from_natural(dev(s))
    assert np.array_equal(A.scales_to_natural(t, 200, 5).cpu().numpy().view(np.uint16), s.view(np.uint16))


# ------------------------------------------------------------------------------- GEMM (a2..a7)
def run_gemm_case(A, M, N, K, g, seed=0, fixed=False, out_f32=False, sums="all", opts=None, XW=None):
    """One problem through quantizer + packer + GEMM (+ the group-sum dump) against the oracle.
    opts: keyword arguments of apex4.debug_opts (kernel / pair_tokens / split / grid / decode_batch)
    passed PER CALL through apex4_w4a4_gemm_ex -- the library has no global dispatch switch."""
    X, W = XW if XW is not None else inputs.make_gemm_inputs(M, N, K, seed, fixed_outliers=fixed)
    ref = O.w4a4_linear(X, W, g)
    G = K // g
    o = A.debug_opts(**opts) if opts else None
    qA, sA, _ = A.quantize_act(dev(X), g)
    qW, sW, _ = A.pack_weights(dev(W), g)
    assert np.array_equal(A.unpack_codes(qA, M, K, A.OPERAND_ACT).cpu().numpy(), ref["qA"])
    assert np.array_equal(A.unpack_codes(qW, N, K, A.OPERAND_WEIGHT).cpu().numpy(), ref["qW"])
    assert np.array_equal(A.scales_to_natural(sA, M, G).cpu().numpy().view(np.uint16), ref["sA"].view(np.uint16))
    assert np.array_equal(A.scales_to_natural(sW, N, G).cpu().numpy().view(np.uint16), ref["sW"].view(np.uint16))
    Y = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, g, out_dtype=torch.float32 if out_f32 else torch.float16, opts=o)
    # a second and third call on one (self-cleaning) workspace must give the same answer
    ws = A.make_workspace(M, N, K, g, opts=o)
    Y2 = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, g, out_dtype=Y.dtype, workspace=ws, opts=o)
    Y3 = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, g, out_dtype=Y.dtype, workspace=ws, opts=o)
    if sums == "all":
        P = A.debug_group_sums(qA, qW, M, N, K, g, opts=o).cpu().numpy()
        assert np.array_equal(P, O.group_sums(ref["qA"], ref["qW"], g))
    elif sums is not None:
        m0, m1, n0, n1 = sums
        P = A.debug_group_sums(qA, qW, M, N, K, g, m0=m0, m1=m1, n0=n0, n1=n1, opts=o).cpu().numpy()
        assert np.array_equal(P, O.group_sums(ref["qA"][m0:m1], ref["qW"][n0:n1], g))
    torch.cuda.synchronize()
    for y in (Y, Y2, Y3):
        check_output(y.cpu().numpy(), ref["Y64"], ref["T"], G, not out_f32)
    if ws is not None:
        assert int(ws.count_nonzero()) == 0      # workspace left zero-filled
    return ref


PAIR, DECODE = 1, 0   # apex4_debug_opts.kernel


def test_gemm_config0(A):
    """BASELINE.json config 0: M=16, N=256, K=512, g=128, seed 0 -- every output, every group sum."""
    X, W, g = inputs.config0()
    assert X.shape == (16, 512) and W.shape == (256, 512)
    run_gemm_case(A, 16, 256, 512, 128, seed=0, fixed=True)


@pytest.mark.parametrize("g", [32, 64, 128, 256, 512])
@pytest.mark.parametrize("opts", [dict(kernel=PAIR), dict(kernel=PAIR, split=1, grid=3), dict(kernel=PAIR, split=1, grid=1),
                                  dict(kernel=PAIR, pair_tokens=128, split=1, grid=2), dict(kernel=PAIR, pair_tokens=192),
                                  dict(kernel=DECODE), dict(kernel=DECODE, grid=3, decode_batch=2)])
def test_gemm_config0_all_dispatches(A, g, opts):
    """Same problem through both kernels, every token-tile width of the pair kernel, whole-tile and
    stream-K work distribution and several grid sizes."""
    if opts["kernel"] == DECODE and g == 256:
        with pytest.raises(A.Apex4Error) as e:      # the decode kernel does not cover 128 < g < K (K = 512 here)
            run_gemm_case(A, 16, 256, 512, g, seed=0, fixed=True, opts=opts)
        assert e.value.status == A.ERR_INVALID_ARG
        return
    run_gemm_case(A, 16, 256, 512, g, seed=0, fixed=True, opts=opts)


@pytest.mark.parametrize("M,N,K,g", [(1, 256, 512, 128), (4, 264, 1024, 128), (17, 136, 384, 32),
                                     (64, 512, 1024, 64), (100, 384, 2048, 2048), (130, 520, 1024, 128),
                                     (257, 768, 1536, 512), (300, 1000, 512, 128), (256, 2048, 4096, 128)])
def test_gemm_ragged_and_multi_tile(A, M, N, K, g):
    run_gemm_case(A, M, N, K, g, seed=100 + M)


@pytest.mark.parametrize("M,N,K", [(1, 8, 128), (16, 136, 1024), (17, 1000, 512), (32, 8192, 256),
                                   (20, 264, 2048), (31, 520, 1024), (5, 64, 28672)])
@pytest.mark.parametrize("grid", [0, 1, 3])
def test_gemm_decode_kernels(A, M, N, K, grid):
    """The decode-regime kernel at g = 128 (one or two m16 token tiles) on ragged N, row ranges that
    straddle 128-row tiles, K from one k-block to the longest supported row, and several grid sizes
    (rows per CTA / batches per CTA)."""
    assert A.debug_get_dispatch(M, N, K, 128)[0] == DECODE      # the automatic choice for M <= 32
    run_gemm_case(A, M, N, K, 128, seed=300 + M, opts=dict(kernel=DECODE, grid=grid))


def test_dispatch_above_decode_range(A):
    """32 < M: CTA pairs (64-token tiles up to M = 64); asking for the decode kernel there is an error."""
    assert A.debug_get_dispatch(33, 264, 2048, 128)[:2] == (PAIR, 64)
    assert A.debug_get_dispatch(64, 8192, 8192, 128)[:2] == (PAIR, 64)
    with pytest.raises(A.Apex4Error):
        A.debug_get_dispatch(33, 264, 2048, 128, opts=A.debug_opts(kernel=DECODE))
    run_gemm_case(A, 33, 264, 2048, 128, seed=333)
    run_gemm_case(A, 64, 456, 1536, 128, seed=364)


@pytest.mark.parametrize("M,N,K", [(1, 8, 256), (16, 136, 1024), (17, 1000, 512), (32, 8192, 256),
                                   (20, 264, 2048), (5, 64, 28672)])
@pytest.mark.parametrize("grid", [0, 1, 3])
def test_gemm_decode_per_channel(A, M, N, K, grid):
    """Per-channel decode (M <= 32, g = K): the decode kernel keeps INT32 partial sums through the k loop
    and the cross-warp reduction, so the group sum is exact and rounded once (R12)."""
    assert A.debug_get_dispatch(M, N, K, K)[0] == DECODE
    run_gemm_case(A, M, N, K, K, seed=700 + M, opts=dict(kernel=DECODE, grid=grid))
    run_gemm_case(A, M, N, K, K, seed=700 + M, opts=dict(kernel=DECODE, grid=grid), out_f32=True, sums=None)


@pytest.mark.parametrize("M,N,K,g", [(1, 8, 256, 32), (16, 136, 1024, 32), (17, 1000, 512, 64), (32, 8192, 256, 32),
                                     (20, 264, 2048, 64), (9, 4096, 11008, 32), (5, 64, 28672, 64)])
@pytest.mark.parametrize("grid", [0, 3])
def test_gemm_decode_fine_groups(A, M, N, K, g, grid):
    """Decode at g = 32 / 64 (M <= 32): every MMA (pair of MMAs) of the decode kernel covers exactly one
    group and is scaled on its own; group sums bit-exact, outputs inside the tolerance, FP16 and FP32."""
    assert A.debug_get_dispatch(M, N, K, g)[0] == DECODE
    run_gemm_case(A, M, N, K, g, seed=800 + M, opts=dict(kernel=DECODE, grid=grid))
    run_gemm_case(A, M, N, K, g, seed=800 + M, opts=dict(kernel=DECODE, grid=grid), out_f32=True, sums=None)


@pytest.mark.parametrize("M,N,K,g", [(40, 264, 512, 128), (64, 520, 1024, 32), (100, 520, 1024, 128),
                                     (130, 304, 1024, 512), (300, 520, 1024, 1024), (200, 264, 2048, 64)])
@pytest.mark.parametrize("opts", [dict(kernel=PAIR, pair_tokens=64, split=0), dict(kernel=PAIR, pair_tokens=128, split=0),
                                  dict(kernel=PAIR, pair_tokens=192, split=0),
                                  dict(kernel=PAIR, pair_tokens=64, split=1, grid=3),
                                  dict(kernel=PAIR, pair_tokens=128, split=1, grid=5),
                                  dict(kernel=PAIR, pair_tokens=192, split=1, grid=2)])
def test_gemm_pair_tile_widths(A, M, N, K, g, opts):
    """The CTA-pair kernel at its three token-tile widths (64 / 128 / 192), whole tiles and stream-K,
    FP16 and FP32 output, on ragged shapes."""
    run_gemm_case(A, M, N, K, g, seed=500 + M, opts=opts)
    run_gemm_case(A, M, N, K, g, seed=500 + M, opts=opts, out_f32=True, sums=None)


@pytest.mark.parametrize("M,N,K,g", [(16, 264, 8192, 256), (16, 264, 8192, 512), (9, 136, 8192, 1024), (32, 264, 8192, 2048),
                                     (20, 136, 4096, 256), (17, 136, 4096, 512), (5, 72, 4096, 1024), (3, 64, 28672, 256),
                                     (16, 264, 2048, 256), (31, 264, 2048, 1024)])
@pytest.mark.parametrize("grid", [0, 3])
def test_gemm_decode_groups_between_128_and_K(A, M, N, K, g, grid):
    """Decode (M <= 32) at 128 < g < K (the paper's granularities 256 / 512 / 1024): a group's INT32 sum
    is completed before it is scaled -- inside a warp when its k range holds whole groups, across warps through
    shared memory when several warps share a group -- so every group is rounded once (R12)."""
    assert A.debug_get_dispatch(M, N, K, g)[0] == DECODE
    run_gemm_case(A, M, N, K, g, seed=850 + M, opts=dict(kernel=DECODE, grid=grid))
    run_gemm_case(A, M, N, K, g, seed=850 + M, opts=dict(kernel=DECODE, grid=grid), out_f32=True, sums=None)
    run_gemm_case(A, M, N, K, g, seed=850 + M, opts=dict(kernel=PAIR), sums=None)       # the pair kernel agrees


def test_gemm_decode_f32_and_large_group_routing(A):
    run_gemm_case(A, 16, 256, 1024, 128, seed=7, out_f32=True, opts=dict(kernel=DECODE))
    # groups larger than a k-block keep one rounding per group: the pair kernel handles them
    assert A.debug_get_dispatch(16, 256, 1024, 256)[:2] == (PAIR, 64)
    run_gemm_case(A, 16, 256, 1024, 256, seed=8)


def test_gemm_f32_output(A):
    run_gemm_case(A, 40, 256, 1024, 128, seed=3, out_f32=True)
    run_gemm_case(A, 200, 512, 1024, 128, seed=4, out_f32=True)


def test_gemm_all_ones_closed_form(A):
    """P3: X = W = 1 -> every code 7, P = 49 g, Y = 49 K (585/4096)^2 for every g."""
    for (M, N, K) in [(16, 256, 512), (150, 384, 4096)]:
        X = np.ones((M, K), dtype=np.float16)
        W = np.ones((N, K), dtype=np.float16)
        for g in (32, 128, K):
            qA, sA, _ = A.quantize_act(dev(X), g)
            qW, sW, _ = A.pack_weights(dev(W), g)
            Y = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, g).cpu().numpy()
            want = np.float16(49.0 * K * (585.0 / 4096.0) ** 2)
            assert np.all(Y == want), (M, N, K, g)
            P = A.debug_group_sums(qA, qW, M, N, K, g, m1=min(M, 8), n1=16).cpu().numpy()
            assert np.all(P == 49 * g)


def test_gemm_minus8_codes_headroom(A):
    """R5: all-(-8) codes injected through apex4_pack_codes: P = 64 g, exact up to per-channel K."""
    M, N, K = 8, 128, 4096
    cA = np.full((M, K), -8, dtype=np.int8)
    cW = np.full((N, K), -8, dtype=np.int8)
    qA, qW = A.pack_codes(dev(cA), A.OPERAND_ACT), A.pack_codes(dev(cW), A.OPERAND_WEIGHT)
    for g in (32, 128, K):
        P = A.debug_group_sums(qA, qW, M, N, K, g).cpu().numpy()
        assert np.all(P == 64 * g)
    g = 128
    sA = A.scales_from_natural(dev(np.full((M, K // g), 0.5, dtype=np.float16)))
    sW = A.scales_from_natural(dev(np.full((N, K // g), 0.25, dtype=np.float16)))
    Y = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, g, out_dtype=torch.float32).cpu().numpy()
    assert np.all(Y == 64.0 * K * 0.125)


def test_gemm_sampled_large(A):
    """A Llama-2-7B shaped layer (config 1, O-proj) at M=2048: sampled rows x all columns and all rows
    x sampled columns against the oracle, group sums bit-exact on a window per tile corner."""
    M, N, K, g = 2048, 4096, 4096, 128
    X, W = inputs.make_gemm_inputs(M, N, K, inputs.config_seed(1, 1), fixed_outliers=True)
    qA, sA, _ = A.quantize_act(dev(X), g)
    qW, sW, _ = A.pack_weights(dev(W), g)
    Y = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, g).cpu().numpy()
    rows = inputs.sample_rows(M, 1)
    cols = inputs.sample_rows(N, 2)
    qa, sa = O.quantize(X, g)
    qw, sw = O.quantize(W, g)
    Y64, T = O.dequant_gemm(qa[rows], sa[rows], qw, sw, g)
    check_output(Y[rows], Y64, T, K // g, True)
    Y64, T = O.dequant_gemm(qa, sa, qw[cols], sw[cols], g)
    check_output(Y[:, cols], Y64, T, K // g, True)
    for (m0, n0) in [(0, 0), (120, 250), (2040, 4088), (1000, 2040)]:
        P = A.debug_group_sums(qA, qW, M, N, K, g, m0=m0, m1=m0 + 8, n0=n0, n1=n0 + 8).cpu().numpy()
        assert np.array_equal(P, O.group_sums(qa[m0:m0 + 8], qw[n0:n0 + 8], g))


@pytest.mark.parametrize("N,K,layer,g_expect", [
    (512, 3584, "LAYER_V", 32),          # Qwen2.5-7B V-proj (4 KV heads x 128), paper mix: fine
    (4096, 3584, "LAYER_Q", 3584),       # fused Q+K, paper mix: per-channel
    (3584, 18944, "LAYER_DOWN", 32),     # down-proj, paper mix: fine, K = 148 k-blocks
])
def test_gemm_qwen_shapes_mixed_policy(A, N, K, layer, g_expect):
    """Qwen2.5-7B linear shapes under the R11 mixed policy (g resolved by the
    library from the layer kind): sampled rows x all columns against the oracle, group sums bit-exact
    on windows."""
    M = 320
    lay = getattr(A, layer)
    g = A.resolve_group_size(K, 128, A.GRAN_MIXED, lay)
    assert g == g_expect
    X, W = inputs.make_gemm_inputs(M, N, K, 7001 + N % 97)
    qA, sA, ga = A.quantize_act(dev(X), 128, A.GRAN_MIXED, lay)
    qW, sW, gw = A.pack_weights(dev(W), 128, A.GRAN_MIXED, lay)
    assert ga == g and gw == g
    Y = A.w4a4_gemm(qA, sA, qW, sW, M, N, K, 128, A.GRAN_MIXED, lay).cpu().numpy()
    rows = inputs.sample_rows(M, 3)
    qa, sa = O.quantize(X, g)
    qw, sw = O.quantize(W, g)
    _, _, codes, _ = gpu_quantize(A, X, g)
    assert np.array_equal(codes, qa)
    Y64, T = O.dequant_gemm(qa[rows], sa[rows], qw, sw, g)
    check_output(Y[rows], Y64, T, K // g, True)
    for (m0, n0) in [(0, 0), (188, N - 8), (M - 8, 250)]:
        P = A.debug_group_sums(qA, qW, M, N, K, 128, A.GRAN_MIXED, lay, m0=m0, m1=m0 + 8, n0=n0, n1=n0 + 8).cpu().numpy()
        assert np.array_equal(P, O.group_sums(qa[m0:m0 + 8], qw[n0:n0 + 8], g))


def test_linear_host_matches_device_path(A):
    M, N, K, g = 16, 256, 512, 128
    X, W, _ = inputs.config0()
    ref = O.w4a4_linear(X, W, g)
    qW, sW, _ = A.pack_weights(dev(W), g)
    xh = torch.from_numpy(X).pin_memory()
    yh = torch.empty((M, N), dtype=torch.float16).pin_memory()
    A.w4a4_linear_host(xh, qW, sW, yh, N, g)
    torch.cuda.synchronize()
    check_output(yh.numpy(), ref["Y64"], ref["T"], K // g, True)


def test_error_codes_on_device(A):
    x = torch.zeros((16, 512), dtype=torch.float16, device="cuda")
    with pytest.raises(A.Apex4Error) as e:
        A.quantize_act(x, 48)
    assert e.value.status == A.ERR_UNSUPPORTED_SHAPE
    q, s, _ = A.quantize_act(x, 128)
    with pytest.raises(A.Apex4Error) as e:     # stream-K dispatch without a workspace
        import ctypes
        o = A.debug_opts(kernel=PAIR, split=1, grid=2)
        st = A.lib().apex4_w4a4_gemm_ex(q.data_ptr(), s.data_ptr(), q.data_ptr(), s.data_ptr(), x.data_ptr(),
                                        0, 16, 512, 512, 128, 0, 0, None, 0, None, ctypes.byref(o))
        A._check(st, "gemm")
    assert e.value.status == A.ERR_WORKSPACE
