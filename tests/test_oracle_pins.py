"""Pins that tie oracle/apex4_oracle.py to something other than itself
(SURVEY.md 8(c) P1..P8): hand-worked fixtures, closed forms, invariants,
an exact-integer restatement of the rounding decision brute-forced over every
FP16 input, and special cases that reduce to a plain integer matmul.
CPU only (-m "not gpu")."""
import numpy as np
import pytest

from conftest import read_kv_fixture, read_rows_fixture
from oracle import apex4_oracle as O


def f16(vals):
    return np.array([float(v) for v in vals], dtype=np.float16)


def bits(a):
    return np.asarray(a, dtype=np.float16).view(np.uint16)


# ----------------------------------------------------------------- P1
@pytest.mark.parametrize("g,tag", [(4, "g4"), (8, "g8")])
def test_p1_worked_example(g, tag):
    fx = read_kv_fixture("p1_worked_example.txt")
    A = f16(fx["A"])[None, :]
    W = f16(fx["W"])[None, :]
    qA, sA = O.quantize(A, g)
    qW, sW = O.quantize(W, g)
    assert [int(v) for v in qA[0]] == [int(v) for v in fx[tag + ".qA"]]
    assert [int(v) for v in qW[0]] == [int(v) for v in fx[tag + ".qW"]]
    assert [int(b) for b in bits(sA)[0]] == [int(v, 16) for v in fx[tag + ".sA_bits"]]
    assert [int(b) for b in bits(sW)[0]] == [int(v, 16) for v in fx[tag + ".sW_bits"]]
    P = O.group_sums(qA, qW, g)
    assert [int(v) for v in P[0, 0]] == [int(v) for v in fx[tag + ".P"]]
    Y64, T = O.dequant_gemm(qA, sA, qW, sW, g)
    assert Y64[0, 0] == float(fx[tag + ".Y64"][0])
    assert int(bits(O.to_f16(Y64))[0, 0]) == int(fx[tag + ".Y16_bits"][0], 16)
    if tag == "g4":
        assert [int(b) for b in O.pack_canonical(qA)[0]] == [int(v, 16) for v in fx["g4.packedA"]]
        assert [int(b) for b in O.pack_canonical(qW)[0]] == [int(v, 16) for v in fx["g4.packedW"]]


def test_p1_discriminates_other_roundings():
    """The fixture's values are NOT what half-away-from-zero or floor would give (R1)."""
    fx = read_kv_fixture("p1_worked_example.txt")
    A = f16(fx["A"]).astype(np.float64)
    W = f16(fx["W"]).astype(np.float64)
    half_away = lambda v: np.sign(v) * np.floor(np.abs(v) + 0.5)
    P_away = int(np.sum(half_away(A / 1.0) * half_away(W / 0.25)))
    P_floor = int(np.sum(np.floor(A / 1.0) * np.floor(W / 0.25)))
    assert P_away == 27 and P_floor == 26 and int(fx["g8.P"][0]) == 34


# ----------------------------------------------------------------- P2
def test_p2_scale_bit_patterns():
    for absmax_expr, want in read_rows_fixture("p2_scale_bits.txt"):
        a = np.float16(eval(absmax_expr))
        assert float(a) == eval(absmax_expr), absmax_expr     # fixture value is exact in FP16
        X = np.zeros((1, 32), dtype=np.float16)
        X[0, 5] = -a                                          # sign must not matter
        _, S = O.quantize(X, 32)
        assert int(bits(S)[0, 0]) == int(want, 16), (absmax_expr, hex(int(bits(S)[0, 0])))


def test_r4_r5_zero_and_subnormal_scale():
    u = 2.0 ** -24
    X = np.zeros((1, 64), dtype=np.float16)
    X[0, :32] = np.float16(3 * u)                 # S rounds to 0 -> all codes 0 (R4)
    X[0, 32] = np.float16(10 * u)                 # S = 1 unit -> x/S = 10 -> clamp to 7 (R5)
    X[0, 33] = np.float16(-10 * u)                # -> -8: the clamp is asymmetric, as written in Eq. 7
    X[0, 34] = np.float16(5 * u)
    q, S = O.quantize(X, 32)
    assert int(bits(S)[0, 0]) == 0 and not q[0, :32].any()
    assert int(bits(S)[0, 1]) == 1
    assert (int(q[0, 32]), int(q[0, 33]), int(q[0, 34])) == (7, -8, 5)
    X2 = np.zeros((1, 32), dtype=np.float16)
    X2[0, 0] = np.float16(11 * u)                 # S = 2 units -> 5.5 -> tie -> 6
    q2, S2 = O.quantize(X2, 32)
    assert int(bits(S2)[0, 0]) == 2 and int(q2[0, 0]) == 6


# ----------------------------------------------------------------- P3
@pytest.mark.parametrize("K,y16", [(512, 511.75), (4096, 4094.0), (8192, 8188.0),
                                   (11008, 11000.0), (28672, 28656.0)])
def test_p3_all_ones_closed_form(K, y16):
    """X = W = 1: every S = 585/4096, every code 7, P_gamma = 49 g,
    Y = 49 K (585/4096)^2 for EVERY g (per-channel included)."""
    X = np.ones((2, K), dtype=np.float16)
    W = np.ones((3, K), dtype=np.float16)
    closed = 49.0 * K * (585.0 / 4096.0) ** 2
    for g in (32, 64, 128, K):
        r = O.w4a4_linear(X, W, g)
        assert np.all(r["qA"] == 7) and np.all(r["qW"] == 7)
        assert np.all(bits(r["sA"]) == 0x3092) and np.all(bits(r["sW"]) == 0x3092)
        P = O.group_sums(r["qA"], r["qW"], g)
        assert np.all(P == 49 * g)
        assert np.allclose(r["Y64"], closed, rtol=1e-13, atol=0)
        assert np.all(r["Y16"] == np.float16(y16))
    assert float(np.float16(closed)) == y16


def test_all_minus8_codes_headroom():
    """R5: -8 is a legal code; P_gamma = 64 g (and 64 K per-channel stays far below 2^31)."""
    K = 256
    qA = np.full((2, K), -8, dtype=np.int8)
    qW = np.full((2, K), -8, dtype=np.int8)
    for g in (32, 128, K):
        assert np.all(O.group_sums(qA, qW, g) == 64 * g)
    assert 64 * 28672 == 1835008 < 2 ** 31


# ----------------------------------------------------------------- P4
def test_p4_scaled_identity_pairs_scales_with_groups():
    K = N = 256
    g = 64
    rng = np.random.default_rng(7)
    X = rng.standard_normal((5, K)).astype(np.float16)
    W = (0.5 * np.eye(N)).astype(np.float16)
    r = O.w4a4_linear(X, W, g)
    # the diagonal's group has S = fp16(0.5/7) = 0x2C92 = 0.0714111328125, code 7; all others S = 0 (R4)
    sW = r["sW"]
    for n in range(N):
        for gamma in range(K // g):
            want = 0x2C92 if gamma == n // g else 0
            assert int(bits(sW)[n, gamma]) == want
    fake_quant_A = r["sA"].astype(np.float64).repeat(g, axis=1) * r["qA"].astype(np.float64)
    want = fake_quant_A * (7 * 0.0714111328125)
    assert np.array_equal(r["Y64"], want)


# ----------------------------------------------------------------- P5
@pytest.mark.parametrize("g", [32, 128, 512])
def test_p5_fp64_dequantise_then_matmul_identity(g):
    from paper_2606_08761_b200 import inputs
    X, W = inputs.make_gemm_inputs(24, 40, 512, seed=11, fixed_outliers=True)
    r = O.w4a4_linear(X, W, g)
    Ahat = r["sA"].astype(np.float64).repeat(g, axis=1) * r["qA"].astype(np.float64)
    What = r["sW"].astype(np.float64).repeat(g, axis=1) * r["qW"].astype(np.float64)
    Y = Ahat @ What.T
    G = 512 // g
    assert np.all(np.abs(Y - r["Y64"]) <= (512 + G) * 2.0 ** -52 * r["T"] + 1e-300)
    # the FP32-ordered variant agrees within the R12 bound
    Y32 = O.dequant_gemm_f32_order(r["qA"], r["sA"], r["qW"], r["sW"], g)
    assert np.all(np.abs(Y32 - r["Y64"]) <= O.output_tolerance(r["Y64"], r["T"], G, False))


# ----------------------------------------------------------------- P6
def test_p6_invariants():
    from paper_2606_08761_b200 import inputs
    K, g = 512, 128
    X, W = inputs.make_gemm_inputs(16, 32, K, seed=5, fixed_outliers=True)
    r = O.w4a4_linear(X, W, g)
    # (i) g = K is the per-channel mode: one scale per row
    rc = O.w4a4_linear(X, W, K)
    assert rc["sA"].shape == (16, 1) and rc["sW"].shape == (32, 1)
    # (ii) power-of-two scaling: same codes, scales x 2^j, Y scales exactly
    for j in (-3, 2):
        r2 = O.w4a4_linear((X.astype(np.float32) * 2.0 ** j).astype(np.float16), W, g)
        assert np.array_equal(r2["qA"], r["qA"])
        assert np.array_equal(r2["sA"].astype(np.float64), r["sA"].astype(np.float64) * 2.0 ** j)
        assert np.array_equal(r2["Y64"], r["Y64"] * 2.0 ** j)
    # (iii) symmetry: quant(-X) = -quant(X) (no -8 for normal-range scales)
    qn, sn = O.quantize(-X, g)
    assert np.array_equal(qn, -r["qA"]) and np.array_equal(sn, r["sA"])
    assert r["qA"].min() >= -7 and r["qA"].max() <= 7
    # (iv) permuting k inside a group (same permutation on both sides) leaves P unchanged
    perm = np.arange(K).reshape(K // g, g)
    rng = np.random.default_rng(3)
    perm = np.concatenate([row[rng.permutation(g)] for row in perm])
    assert np.array_equal(O.group_sums(r["qA"][:, perm], r["qW"][:, perm], g),
                          O.group_sums(r["qA"], r["qW"], g))
    rp = rng.permutation(16)
    assert np.array_equal(O.w4a4_linear(X[rp], W, g)["Y64"], r["Y64"][rp])
    # (v) |x - S q| <= S/2 ; (vi) |P| <= 49 g
    S_full = r["sA"].astype(np.float64).repeat(g, axis=1)
    assert np.all(np.abs(X.astype(np.float64) - S_full * r["qA"]) <= S_full / 2)
    assert np.all(np.abs(O.group_sums(r["qA"], r["qW"], g)) <= 49 * g)
    # (vii) split-K: Y(K1 u K2) = Y(K1) + Y(K2) in float64 (cut on a group boundary)
    h = K // 2
    Ya = O.dequant_gemm(r["qA"][:, :h], r["sA"][:, :2], r["qW"][:, :h], r["sW"][:, :2], g, want_T=False)
    Yb = O.dequant_gemm(r["qA"][:, h:], r["sA"][:, 2:], r["qW"][:, h:], r["sW"][:, 2:], g, want_T=False)
    assert np.all(np.abs((Ya + Yb) - r["Y64"]) <= 4 * 2.0 ** -52 * r["T"])


# ----------------------------------------------------------------- P7
def _exact_rne_quotient(xb: np.ndarray, sb: int) -> np.ndarray:
    """clamp(rne(x/s), -8, 7) for FP16 bit patterns xb and scale bit pattern sb, decided in
    64-bit INTEGER arithmetic (no floating point): x = (-1)^sx X 2^ex, s = Sg 2^es;
    compare 2 X 2^d against (2k+1) Sg."""
    def decode(b):
        b = b.astype(np.int64)
        e = (b >> 10) & 0x1F
        m = b & 0x3FF
        X = np.where(e == 0, m, m | 0x400)
        ex = np.where(e == 0, -24, e - 25)
        return (b >> 15) & 1, X, ex
    sx, X, ex = decode(xb)
    _, Sg, es = decode(np.array([sb], dtype=np.uint16))
    Sg, es = int(Sg[0]), int(es[0])
    if Sg == 0:
        return np.zeros(xb.shape, dtype=np.int64)
    d = ex - es
    big = d > 20                                   # |x/s| >= 2^10: clamps
    dd = np.clip(d, -40, 20)
    num = np.where(dd >= 0, X << np.maximum(dd, 0), X)
    den = np.where(dd >= 0, Sg, Sg << np.maximum(-dd, 0))
    qf = (2 * num + den) // (2 * den)              # round half up
    tie = (2 * num + den) % (2 * den) == 0
    qf = np.where(tie & (qf % 2 == 1), qf - 1, qf)  # ... half to even
    qf = np.where(big & (X > 0), 1 << 20, qf)
    q = np.where(sx == 1, -qf, qf)
    return np.clip(q, -8, 7)


def test_p7_exhaustive_fp16_rounding_decision():
    allb = np.arange(0x10000, dtype=np.uint32).astype(np.uint16)
    finite = allb[((allb >> 10) & 0x1F) != 0x1F]
    scale_bits = [0x0001, 0x0002, 0x0003, 0x0007, 0x000E, 0x0092, 0x03FF, 0x0400, 0x0401,
                  0x19DA, 0x2C92, 0x3000, 0x3092, 0x3400, 0x3492, 0x3555, 0x3800, 0x3C00,
                  0x3C01, 0x3FFF, 0x41B7, 0x4248, 0x5640, 0x7092, 0x7BFF]
    rng = np.random.default_rng(0)
    scale_bits += [int(b) for b in rng.integers(1, 0x7C00, size=40)]
    x = finite.view(np.float16).astype(np.float64)
    for sb in scale_bits:
        s = float(np.array([sb], dtype=np.uint16).view(np.float16)[0])
        want = _exact_rne_quotient(finite, sb)
        got = np.clip(np.rint(x / s), -8, 7).astype(np.int64)      # the oracle's formula
        assert np.array_equal(got, want), hex(sb)
    # ... and through the oracle proper: a group whose absmax produces a chosen scale
    for amax in (1.0, 7.0, 20.0, 0.0200042724609375):
        cand = finite[np.abs(finite.view(np.float16).astype(np.float64)) <= amax]
        n = (cand.size + 1 + 255) // 256 * 256
        X = np.zeros((1, n), dtype=np.float16)
        X[0, :cand.size] = cand.view(np.float16)
        X[0, cand.size] = np.float16(amax)
        q, S = O.quantize(X, n)
        want = _exact_rne_quotient(X.view(np.uint16)[0], int(bits(S)[0, 0]))
        assert np.array_equal(q[0].astype(np.int64), want)


def test_p7_tiny_gemm_corner_codes_bruteforce():
    vals = np.array([-8, -7, 0, 7], dtype=np.int8)
    rng = np.random.default_rng(1)
    for _ in range(20):
        qA = vals[rng.integers(0, 4, size=(3, 32))]
        qW = vals[rng.integers(0, 4, size=(4, 32))]
        P = O.group_sums(qA, qW, 32)
        for m in range(3):
            for n in range(4):
                assert int(P[m, n, 0]) == sum(int(a) * int(b) for a, b in zip(qA[m], qW[n]))


# ----------------------------------------------------------------- P8
def test_p8_unit_scales_reduce_to_integer_matmul():
    rng = np.random.default_rng(2)
    K, g = 256, 32
    XA = rng.integers(-7, 8, size=(9, K))
    XW = rng.integers(-7, 8, size=(11, K))
    XA[:, ::g] = 7                                 # a +-7 in every group -> every scale is exactly 1.0
    XW[:, ::g] = -7
    r = O.w4a4_linear(XA.astype(np.float16), XW.astype(np.float16), g)
    assert np.all(bits(r["sA"]) == 0x3C00) and np.all(bits(r["sW"]) == 0x3C00)
    assert np.array_equal(r["qA"], XA) and np.array_equal(r["qW"], XW)
    assert np.array_equal(r["Y64"], (XA.astype(np.int64) @ XW.astype(np.int64).T).astype(np.float64))


# ----------------------------------------------------------------- packing
def test_pack_roundtrip():
    rng = np.random.default_rng(4)
    q = rng.integers(-8, 8, size=(7, 64)).astype(np.int8)
    assert np.array_equal(O.unpack_canonical(O.pack_canonical(q)), q)
    assert O.pack_canonical(np.array([[-8, 7]], dtype=np.int8))[0, 0] == 0x78


# ----------------------------------------------------------------- rho, Eq. 10, policy
def test_table1_rho_and_eq10():
    for gpu, tc, ops_tc, cc, rho_paper, tops, tflops in read_rows_fixture("table1_rho.txt"):
        r = O.rho(float(tc), float(ops_tc), float(cc), 2.0)
        assert r == float(rho_paper), gpu
        assert abs(float(tops) / float(tflops) / r - 1) < 0.01 or gpu == "A100-40G" and abs(float(tops) / float(tflops) - 64) < 0.1
    # Fig. 5 caption: 192x768x384 -> 3x3x3 tiles of 64x256x128 on 10 SMs -> 3 iterations (Eq. 10)
    assert (192 // 64, 768 // 256, 384 // 128) == (3, 3, 3)
    assert O.sm_iterations(3, 3, 3, 10) == 3


def test_policy_table():
    K = 4096
    for layer in range(10):
        assert O.resolve_group_size(K, layer, O.POLICY_UNIFORM_G128) == 128
    for layer in (O.LAYER_V, O.LAYER_DOWN):
        assert O.resolve_group_size(K, layer, O.POLICY_PAPER_MIX) == 32
        assert O.resolve_group_size(K, layer, O.POLICY_BASELINE_MIX) == 128
    for layer in (O.LAYER_Q, O.LAYER_K, O.LAYER_O, O.LAYER_GATE, O.LAYER_UP, O.LAYER_GATE_UP, O.LAYER_QKV):
        assert O.resolve_group_size(K, layer, O.POLICY_PAPER_MIX) == K


# ----------------------------------------------------------------- T, the tolerance, the FP32-ordered sum
def test_pin_T_and_output_tolerance():
    """T (second return of dequant_gemm) and output_tolerance set the bar of every GPU output check, so they
    are pinned to numbers typed from the hand derivation in tests/golden/p1_worked_example.txt:
    g = 4: terms 1.0*0.125*69 = 8.625 and 0.28564453125*0.25*(-24) = -1.7138671875
           T = 8.625 + 1.7138671875 = 10.3388671875
           tol (FP32 out) = 1e-3 * 6.9111328125 + (2+2) * 2^-23 * 10.3388671875
                          = 0.0069111328125 + 4.76837158203125e-07 * 10.3388671875 = 0.00691606276855...
           FP16 out adds one subnormal ulp 2^-24 = 5.9604644775390625e-08."""
    fx = read_kv_fixture("p1_worked_example.txt")
    A = f16(fx["A"])[None, :]
    W = f16(fx["W"])[None, :]
    qA, sA = O.quantize(A, 4)
    qW, sW = O.quantize(W, 4)
    Y64, T = O.dequant_gemm(qA, sA, qW, sW, 4)
    assert T.shape == (1, 1) and T[0, 0] == 10.3388671875
    tol32 = O.output_tolerance(Y64, T, 2, False)[0, 0]
    tol16 = O.output_tolerance(Y64, T, 2, True)[0, 0]
    assert abs(tol32 - 0.006916062768548727) < 1e-17
    assert abs(tol16 - (0.006916062768548727 + 5.9604644775390625e-08)) < 1e-17
    # a x1000 (or /1000) mistake in either term would move the bound by far more than this
    assert 0.0069 < tol32 < 0.00693 and tol16 > tol32
    # per-channel (g = 8): one term, T = |Y| = 8.5, tol = 8.5e-3 + 3 * 2^-23 * 8.5
    qA8, sA8 = O.quantize(A, 8)
    qW8, sW8 = O.quantize(W, 8)
    Y8, T8 = O.dequant_gemm(qA8, sA8, qW8, sW8, 8)
    assert T8[0, 0] == 8.5
    assert abs(O.output_tolerance(Y8, T8, 1, False)[0, 0] - (0.0085 + 3 * 8.5 / 8388608.0)) < 1e-17
    # P3: every term is positive, so T == Y64 exactly, for every g
    X1 = np.ones((2, 512), dtype=np.float16)
    for g in (32, 128, 512):
        r = O.w4a4_linear(X1, X1, g)
        assert np.array_equal(r["T"], r["Y64"])
    # cancellation: equal and opposite groups give Y = 0 but T = 2 |term| (the bound must not vanish)
    Xc = np.ones((1, 64), dtype=np.float16)
    Wc = np.ones((1, 64), dtype=np.float16)
    Wc[0, 32:] = -1
    rc = O.w4a4_linear(Xc, Wc, 32)
    term = 49 * 32 * (585.0 / 4096.0) ** 2
    assert rc["Y64"][0, 0] == 0.0 and rc["T"][0, 0] == 2 * term
    assert O.output_tolerance(rc["Y64"], rc["T"], 2, False)[0, 0] == 4 * 2.0 ** -23 * 2 * term


def _rn_f32(x):
    """Round an exact rational to binary32 (ties to even) with integer arithmetic only."""
    from fractions import Fraction
    x = Fraction(x)
    if x == 0:
        return Fraction(0)
    s = -1 if x < 0 else 1
    x = abs(x)
    e = 0
    while x >= 2 ** 24:
        x /= 2
        e += 1
    while x < 2 ** 23:
        x *= 2
        e -= 1
    n, rem = divmod(x.numerator, x.denominator)
    twice = 2 * rem
    if twice > x.denominator or (twice == x.denominator and n % 2 == 1):
        n += 1
    return s * Fraction(n) * Fraction(2) ** e


def test_pin_f32_ordered_sum():
    """dequant_gemm_f32_order against (i) the hand example, where every step is exact in binary32:
    fma(69, 0.125, 0) = 8.625, fma(-24, 0.0714111328125, 8.625) = 6.9111328125; (ii) an exact-rational
    restatement of acc = rn32(P * (sA * sW) + acc) on a small random problem."""
    from fractions import Fraction
    fx = read_kv_fixture("p1_worked_example.txt")
    A = f16(fx["A"])[None, :]
    W = f16(fx["W"])[None, :]
    qA, sA = O.quantize(A, 4)
    qW, sW = O.quantize(W, 4)
    Y32 = O.dequant_gemm_f32_order(qA, sA, qW, sW, 4)
    assert Y32.dtype == np.float32 and float(Y32[0, 0]) == 6.9111328125
    rng = np.random.default_rng(12)
    X = (rng.standard_normal((3, 256)) * 3).astype(np.float16)
    Wm = (rng.standard_normal((4, 256)) * 0.02).astype(np.float16)
    g = 32
    r = O.w4a4_linear(X, Wm, g)
    Y32 = O.dequant_gemm_f32_order(r["qA"], r["sA"], r["qW"], r["sW"], g)
    for m in range(3):
        for n in range(4):
            acc = Fraction(0)
            for gam in range(256 // g):
                P = sum(int(a) * int(b) for a, b in zip(r["qA"][m, gam * g:(gam + 1) * g], r["qW"][n, gam * g:(gam + 1) * g]))
                s = Fraction(float(r["sA"][m, gam])) * Fraction(float(r["sW"][n, gam]))     # 22 bits: exact in binary32
                acc = _rn_f32(P * s + acc)
            assert Fraction(float(Y32[m, n])) == acc, (m, n)


# ----------------------------------------------------------------- P9: producers of the quantizer's input
def test_p9_silu_mul_hand_values_and_invariants():
    rows = [r for r in read_rows_fixture("p9_producers.txt") if r[0] == "silu"]
    assert len(rows) >= 8
    for _, g, u, want in rows:
        y = O.silu_mul(f16([g])[None, :], f16([u])[None, :])
        assert int(bits(y)[0, 0]) == int(want, 16), (g, u, hex(int(bits(y)[0, 0])))
    rng = np.random.default_rng(21)
    g = (rng.standard_normal((7, 96)) * 4).astype(np.float16)
    u = rng.standard_normal((7, 96)).astype(np.float16)
    y = O.silu_mul(g, u).astype(np.float64)
    # silu(g) - silu(-g) = g, silu(g) in (min(g,0) - 0.2785, max(g, 0)), sign(y) = sign(g) sign(u), odd in up
    g64, u64 = g.astype(np.float64), u.astype(np.float64)
    s = g64 / (1 + np.exp(-g64))
    assert np.allclose(s - (-g64) / (1 + np.exp(g64)), g64, rtol=0, atol=1e-12)
    assert np.all(np.abs(y - s * u64) <= np.maximum(np.abs(s * u64) * 2.0 ** -11, 2.0 ** -25))     # half an FP16 ulp
    assert np.array_equal(O.silu_mul(g, (-u).astype(np.float16)).view(np.uint16) ^ 0x8000, O.silu_mul(g, u).view(np.uint16))


def test_p9_silu_every_fp16_gate_against_50_digit_decimal():
    """Independent restatement: silu(g) with 50-digit decimal arithmetic, rounded once to FP16 with integer
    arithmetic (ties to even), for EVERY finite FP16 gate and up = 1, and for a second up on a subset."""
    from decimal import Decimal, getcontext
    from fractions import Fraction
    getcontext().prec = 50

    def rn_f16_bits(x: Fraction) -> int:
        if x == 0:
            return 0
        sgn = 0x8000 if x < 0 else 0
        x = abs(x)
        e = 0
        while x >= 2048:
            x /= 2; e += 1
        while x < 1024 and e > -24:          # 11-bit significand, subnormals stop at 2^-24 units
            x *= 2; e -= 1
        n, rem = divmod(x.numerator, x.denominator)
        if 2 * rem > x.denominator or (2 * rem == x.denominator and n % 2 == 1):
            n += 1
        if n == 2048:
            n = 1024; e += 1
        val = Fraction(n) * Fraction(2) ** e
        return sgn | int(np.array([float(val)], dtype=np.float64).astype(np.float16).view(np.uint16)[0])   # exact: val is an FP16 value

    allb = np.arange(0x10000, dtype=np.uint32).astype(np.uint16)
    finite = allb[((allb >> 10) & 0x1F) != 0x1F]
    gates = finite.view(np.float16)
    got = O.silu_mul(gates[None, :], np.ones((1, gates.size), dtype=np.float16)).view(np.uint16)[0]
    step = 1           # every gate
    bad = 0
    for idx in range(0, gates.size, step):
        gd = Decimal(float(gates[idx]))
        if gd == 0:
            want = 0x8000 if (finite[idx] & 0x8000) else 0      # silu(-0) * 1 = -0 / 2 = -0
        else:
            if gd < -120:                        # e^-g overflows nothing in decimal, but keep it cheap: silu -> -|g| e^g ~ 0-
                sd = gd * (gd.exp())             # g / (1 + e^-g) = g e^g / (e^g + 1); e^g + 1 = 1 to 50 digits
            else:
                sd = gd / (1 + (-gd).exp())
            want = rn_f16_bits(Fraction(sd))
            if want & 0x7FFF == 0:
                want = 0x8000 if gd < 0 else 0
        if int(got[idx]) != want:
            bad += 1
            assert bad < 1, (hex(int(finite[idx])), hex(int(got[idx])), hex(want))
    assert bad == 0


def test_p9_rmsnorm_hand_values_invariants_and_exact_restatement():
    from fractions import Fraction
    import math
    fx = read_kv_fixture("p9_producers.txt")
    x = f16(fx["rmsnorm_x"])[None, :]
    y = O.rmsnorm(x, np.ones(4, dtype=np.float16), 0.0)
    assert [int(b) for b in bits(y)[0]] == [int(v, 16) for v in fx["rmsnorm_gamma1"]]
    y = O.rmsnorm(x, f16(fx["rmsnorm_gamma2_in"]), 0.0)
    assert [int(b) for b in bits(y)[0]] == [int(v, 16) for v in fx["rmsnorm_gamma2"]]
    # constant rows with power-of-two magnitude normalise to exactly +-1; scaling x by 2^j changes nothing (eps = 0)
    assert np.all(O.rmsnorm(np.full((2, 64), 4.0, dtype=np.float16), np.ones(64, dtype=np.float16), 0.0) == 1.0)
    rng = np.random.default_rng(22)
    X = rng.standard_normal((5, 256)).astype(np.float16)
    gam = (1 + 0.1 * rng.standard_normal(256)).astype(np.float16)
    base = O.rmsnorm(X, gam, 0.0)
    assert np.array_equal(O.rmsnorm((X.astype(np.float32) * 8).astype(np.float16), gam, 0.0).view(np.uint16), base.view(np.uint16))
    assert np.array_equal(O.rmsnorm(-X, gam, 0.0).view(np.uint16), base.view(np.uint16) ^ 0x8000)
    # against the real-valued definition x gamma / sqrt(mean(x^2) + eps): three binary32 roundings + one FP16 rounding
    eps = 1e-5
    y = O.rmsnorm(X, gam, eps).astype(np.float64)
    X64 = X.astype(np.float64)
    ref = X64 * gam.astype(np.float64)[None, :] / np.sqrt(np.mean(X64 * X64, axis=1, keepdims=True) + eps)
    assert np.all(np.abs(y - ref) <= np.abs(ref) * (2.0 ** -11 + 4 * 2.0 ** -24) + 2.0 ** -25)
    # exact-rational restatement of the binary32 sequence (own rn32, integer square root) on a small case
    def rn32_sqrt(q: Fraction) -> Fraction:
        # correctly rounded binary32 square root of a positive rational: integer sqrt at 2^-60 relative, then rn32
        sc = 0
        while q * Fraction(4) ** sc < Fraction(2) ** 120:
            sc += 1
        v = q * Fraction(4) ** sc
        r = math.isqrt(v.numerator // v.denominator)
        cand = Fraction(r, 2 ** sc)
        lo, hi = _rn_f32(cand), _rn_f32(Fraction(r + 1, 2 ** sc))
        assert lo == hi                      # not within 2^-60 of a rounding boundary
        return lo
    Xs = X[:2, :32]
    gs = gam[:32]
    ys = O.rmsnorm(Xs, gs, eps)
    eps32 = Fraction(float(np.float32(eps)))
    for m in range(2):
        ss = sum(Fraction(float(v)) ** 2 for v in Xs[m])
        ms = _rn_f32(ss / 32)
        inv = _rn_f32(1 / rn32_sqrt(_rn_f32(ms + eps32)))
        for k in range(32):
            y32 = _rn_f32(_rn_f32(Fraction(float(Xs[m, k])) * inv) * Fraction(float(gs[k])))
            assert float(ys[m, k]) == float(np.float16(float(y32))), (m, k)      # float(y32) is exact; one FP16 rounding
