"""APEX4 W4A4 oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

A plain, slow, obviously-correct CPU restatement (numpy, float64 where rounding
is free to vary) of the hot path of APEX4 (arxiv/paper_2606_08761): the
symmetric group quantizer (paper Eq. 7) and the
group-dequantised W4A4 GEMM (paper Eq. 8).

Rules this file lives by
  * It shares no code with the CUDA path (paper_2606_08761_b200/csrc) and
    imports nothing from the package; the package never imports it.
  * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
    `--impl reference` legs may import it.
  * No blocking, fusion or reordering beyond what Eq. 7 / Eq. 8 state.  A
    library matmul (numpy float64 `@` on integer-valued operands, exact because
    every partial sum is < 2**53) serves as the inner-product step of Eq. 8.
  * Readings of silent/garbled points are the ones DESIGN.md lists (R1..R16,
    taken from SURVEY.md 8(c)).

Parity pins (tests/test_oracle_pins.py): hand-worked K=8 example
(tests/golden/p1_worked_example.txt), scale bit patterns, all-ones closed form,
scaled identity, FP64 dequantise-then-matmul identity, invariants, exhaustive
exact-integer restatement of the rounding decision over all FP16 inputs,
integer-matmul special case; T / output_tolerance / dequant_gemm_f32_order on the
hand example and an exact-rational restatement; rmsnorm / silu_mul on hand values,
invariants, an exact-rational (integer sqrt) restatement and a 50-digit decimal
evaluation of every finite FP16 gate.  Every function below has at least one
such pin; nothing here is "parity unpinned".

Natural layouts used here (the C-ABI's device layouts differ; the binding
converts):  X[R,K] float16, codes q[R,K] int8 in [-8,7], scales S[R,G] float16
with G = K // g, P[M,N,G] int32, Y[M,N] float64 / float16.
"""
from __future__ import annotations

import numpy as np

QMAX = 7      # 2**(b-1) - 1, b = 4   (Eq. 7)
QMIN = -8     # -2**(b-1)

# layer kinds / policies of the multi-granularity configuration (paper 3.2.2,
# PAPER.md:162-166, 183).  Numeric values mirror include/apex4.h by intent of
# the boundary, but are typed out here independently.
LAYER_OTHER, LAYER_Q, LAYER_K, LAYER_V, LAYER_QKV, LAYER_O, LAYER_GATE, \
    LAYER_UP, LAYER_GATE_UP, LAYER_DOWN = range(10)
POLICY_UNIFORM_G128 = 0   # "Uniform G=128"
POLICY_PAPER_MIX = 1      # down_proj, v_proj -> G=32; all others per-channel
POLICY_BASELINE_MIX = 2   # BASELINE.json wording: fine layers at g=128, others per-channel


# --------------------------------------------------------------------------
# O1  quantizer  (Eq. 7; FP16 scales PAPER.md:262)
# --------------------------------------------------------------------------
def quantize(X: np.ndarray, g: int):
    """Symmetric INT4 group quantizer along the last axis.

    For every row r and group gamma of g consecutive k:
        a      = max |X[r,k]|                      (exact, FP16)
        S      = fp16_rn( float32(a) / 7.0f )      (R2: IEEE binary32 division, then RN-even to FP16)
        q[r,k] = clamp( rne( X[r,k] / float(S) ), -8, 7 )     (R1: round-half-to-even; R5: clamp kept)
        S == 0  ->  q = 0                          (R4: all-zero or underflowed group)
    The quotient is formed in float64; by SURVEY 8(c) lemma L1 (and the
    exact-integer brute force in the pins) rne() of the float64 quotient equals
    rne() of the true quotient for FP16 x and S.
    Returns (q int8 [R,K], S float16 [R,G]).
    """
    X = np.asarray(X)
    assert X.dtype == np.float16 and X.ndim == 2
    R, K = X.shape
    assert g > 0 and K % g == 0
    G = K // g
    Xg = X.reshape(R, G, g)
    a = np.max(np.abs(Xg), axis=2)                                  # FP16, exact
    s32 = a.astype(np.float32) / np.float32(QMAX)                   # binary32 division
    S = s32.astype(np.float16)                                      # RN-even
    s64 = S.astype(np.float64)[:, :, None]
    x64 = Xg.astype(np.float64)
    with np.errstate(divide="ignore", invalid="ignore"):
        quo = x64 / s64
    r = np.rint(quo)                                                # round-half-to-even
    r = np.clip(r, QMIN, QMAX)
    r = np.where(s64 == 0.0, 0.0, r)
    q = r.astype(np.int8).reshape(R, K)
    return q, S


# --------------------------------------------------------------------------
# O2  canonical packing (byte j of a row holds k=2j in bits 0-3
#     and k=2j+1 in bits 4-7, two's-complement nibbles; PAPER.md:256-260 fixes
#     only "packed along K")
# --------------------------------------------------------------------------
def pack_canonical(q: np.ndarray) -> np.ndarray:
    q = np.asarray(q, dtype=np.int8)
    assert q.shape[-1] % 2 == 0
    u = (q.astype(np.int16) & 0xF).astype(np.uint8)
    return (u[..., 0::2] | (u[..., 1::2] << 4)).astype(np.uint8)


def unpack_canonical(p: np.ndarray) -> np.ndarray:
    p = np.asarray(p, dtype=np.uint8)
    lo = (p & 0xF).astype(np.int16)
    hi = (p >> 4).astype(np.int16)
    lo = np.where(lo >= 8, lo - 16, lo)
    hi = np.where(hi >= 8, hi - 16, hi)
    out = np.empty(p.shape[:-1] + (p.shape[-1] * 2,), dtype=np.int8)
    out[..., 0::2] = lo
    out[..., 1::2] = hi
    return out


# --------------------------------------------------------------------------
# O3  per-group exact integer sums  (Eq. 8 inner product)
# --------------------------------------------------------------------------
def group_sums(qA: np.ndarray, qW: np.ndarray, g: int) -> np.ndarray:
    """P[m,n,gamma] = sum_{k in gamma} qA[m,k] * qW[n,k], exact, int32."""
    qA = np.asarray(qA, dtype=np.int8)
    qW = np.asarray(qW, dtype=np.int8)
    M, K = qA.shape
    N, K2 = qW.shape
    assert K == K2 and K % g == 0
    G = K // g
    P = np.empty((M, N, G), dtype=np.int32)
    for gamma in range(G):
        Ag = qA[:, gamma * g:(gamma + 1) * g].astype(np.float64)
        Wg = qW[:, gamma * g:(gamma + 1) * g].astype(np.float64)
        Pg = Ag @ Wg.T                      # integer-valued, |Pg| <= 64 g < 2**53: exact
        assert np.all(np.abs(Pg) <= 64.0 * g)
        P[:, :, gamma] = Pg.astype(np.int32)
    return P


# --------------------------------------------------------------------------
# O4  group-dequantised GEMM  (Eq. 8)
# --------------------------------------------------------------------------
def dequant_gemm(qA, sA, qW, sW, g: int, want_T: bool = True):
    """Y64[m,n] = sum_gamma sA[m,gamma] * sW[n,gamma] * P[m,n,gamma]  in float64.

    Every term is exact in float64 (11+11 significand bits for the FP16 scales,
    <= 21 bits for P); only the G-1 additions round.  Also returns
    T[m,n] = sum_gamma |term| (the condition number used by the tolerance R12).
    """
    qA = np.asarray(qA, dtype=np.int8)
    qW = np.asarray(qW, dtype=np.int8)
    sA = np.asarray(sA)
    sW = np.asarray(sW)
    assert sA.dtype == np.float16 and sW.dtype == np.float16
    M, K = qA.shape
    N = qW.shape[0]
    assert K % g == 0
    G = K // g
    assert sA.shape == (M, G) and sW.shape == (N, G)
    Y = np.zeros((M, N), dtype=np.float64)
    T = np.zeros((M, N), dtype=np.float64) if want_T else None
    for gamma in range(G):
        Ag = qA[:, gamma * g:(gamma + 1) * g].astype(np.float64)
        Wg = qW[:, gamma * g:(gamma + 1) * g].astype(np.float64)
        Pg = Ag @ Wg.T                                              # exact integers
        scale = sA[:, gamma].astype(np.float64)[:, None] * sW[:, gamma].astype(np.float64)[None, :]
        term = scale * Pg                                           # exact
        Y += term
        if want_T:
            T += np.abs(term)
    return (Y, T) if want_T else Y


def dequant_gemm_f32_order(qA, sA, qW, sW, g: int) -> np.ndarray:
    """One legal FP32 evaluation order of Eq. 8 (debug aid, R7):
    acc = 0; for gamma ascending: acc = fma(float(P), sA*sW, acc) in binary32.
    The fused multiply-add is emulated exactly: float64 product of a <=21-bit
    integer and a 22-bit scale product is exact, the float64 add of a binary32
    acc is then rounded once to binary32 (double rounding can differ from a true
    fma only on float64 ties, which the test tolerance absorbs)."""
    P = group_sums(qA, qW, g)
    M, N, G = P.shape
    acc = np.zeros((M, N), dtype=np.float32)
    for gamma in range(G):
        s = (sA[:, gamma].astype(np.float32)[:, None] * sW[:, gamma].astype(np.float32)[None, :])
        acc = (P[:, :, gamma].astype(np.float64) * s.astype(np.float64) + acc.astype(np.float64)).astype(np.float32)
    return acc


# --------------------------------------------------------------------------
# O5  output cast (R8: FP16 RN-even from the accumulator)
# --------------------------------------------------------------------------
def to_f16(Y: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        return np.asarray(Y).astype(np.float16)


def w4a4_linear(X, W, g: int):
    """The whole path from FP16 operands: quantize both sides (Eq. 7), then Eq. 8.
    g == K is the per-channel mode (R10).  Returns dict with every stage."""
    qA, sA = quantize(X, g)
    qW, sW = quantize(W, g)
    Y64, T = dequant_gemm(qA, sA, qW, sW, g)
    return dict(qA=qA, sA=sA, qW=qW, sW=sW, Y64=Y64, T=T, Y16=to_f16(Y64))


# --------------------------------------------------------------------------
# F1/F2  producers of the quantizer's input ("quantized online", PAPER.md:150, 256 -- the paper
#        does not say what feeds the quantizer; in a Llama / Qwen block it is RMSNorm (QKV, gate/up inputs)
#        and SiLU(gate) * up (down_proj input).  Neither is in the paper's equations: the readings below are
#        DESIGN.md R17 / R18.  The fused CUDA calls apex4_rmsnorm_quantize / apex4_silu_mul_quantize must
#        produce exactly quantize(rmsnorm(...), g) / quantize(silu_mul(...), g).)
# --------------------------------------------------------------------------
def rmsnorm(X: np.ndarray, gamma: np.ndarray, eps: float) -> np.ndarray:
    """R17.  y[m,k] = fp16_rn( (x[m,k] * inv[m]) * gamma[k] ), evaluated in IEEE binary32:
        ss[m]  = sum_k x[m,k]^2                 exact (every square of an FP16 value is exact in binary32 and
                                                 the sum of K <= 32768 of them is exact in binary64, in any order)
        ms[m]  = float32( ss[m] / K )           one rounding
        inv[m] = 1.0f / sqrtf( ms[m] + eps )    IEEE add, sqrt, divide (each correctly rounded)
        y      = fp16_rn( fmul(fmul(x, inv), gamma) )
    X[M,K] float16, gamma[K] float16, eps a binary32 value.  Returns float16 [M,K]."""
    X = np.asarray(X)
    gamma = np.asarray(gamma)
    assert X.dtype == np.float16 and gamma.dtype == np.float16 and X.ndim == 2 and gamma.shape == (X.shape[1],)
    K = X.shape[1]
    assert K <= 32768
    x64 = X.astype(np.float64)
    ss = np.sum(x64 * x64, axis=1)                                   # exact
    ms = (ss / np.float64(K)).astype(np.float32)
    inv = np.float32(1.0) / np.sqrt(ms + np.float32(eps), dtype=np.float32)
    y32 = (X.astype(np.float32) * inv[:, None]) * gamma.astype(np.float32)[None, :]
    assert y32.dtype == np.float32
    with np.errstate(over="ignore"):
        return y32.astype(np.float16)


def silu_mul(gate: np.ndarray, up: np.ndarray) -> np.ndarray:
    """R18.  y = fp16_rn( silu(gate) * up ), silu(g) = g / (1 + exp(-g)): the real-valued product rounded ONCE to
    FP16 (evaluated in binary64, whose 2^-52 error can move an FP16 rounding only within 2^-40 of a tie).
    gate, up float16 of equal shape.  Returns float16."""
    gate = np.asarray(gate)
    up = np.asarray(up)
    assert gate.dtype == np.float16 and up.dtype == np.float16 and gate.shape == up.shape
    g = gate.astype(np.float64)
    with np.errstate(over="ignore"):
        s = g / (1.0 + np.exp(-g))                                   # exp(-g) = inf for g < -709 never happens: |g| <= 65504 -> s = -0.0
        s = np.where(np.isfinite(s), s, 0.0)
        return (s * up.astype(np.float64)).astype(np.float16)


# --------------------------------------------------------------------------
# O6  granularity policy  (paper 3.2.2; reading R11)
# --------------------------------------------------------------------------
def resolve_group_size(K: int, layer: int, policy: int) -> int:
    """Group size a layer runs at.  Uniform: 128 everywhere.  Mixed: the two
    sensitive layer kinds (down_proj, v_proj) get the fine size (32 in the
    paper, 128 under BASELINE.json's wording), every other linear is
    per-channel (g = K).  A fused QKV cannot carry two granularities
    (G_a = G_w): under a mixed policy it resolves as per-channel
    for the Q,K part and the caller runs V on its own (R11)."""
    if policy == POLICY_UNIFORM_G128:
        return 128
    fine = 32 if policy == POLICY_PAPER_MIX else 128
    if layer in (LAYER_V, LAYER_DOWN):
        return fine
    return K


# --------------------------------------------------------------------------
# A5  rho  (Eq. 1-2) and Eq. 10
# --------------------------------------------------------------------------
def rho(n_tc: float, ops_tc: float, n_cc: float, ops_cc: float) -> float:
    """rho = (N_TC * OPs_TC) / (N_CC * OPs_CC); the clock cancels (Eq. 2)."""
    return (n_tc * ops_tc) / (n_cc * ops_cc)


def sm_iterations(m_tiles: int, n_tiles: int, k_tiles: int, n_sms: int) -> int:
    """Eq. 10: ceil(M_tile * N_tile * K_tile / Number_of_SMs)."""
    return -(-(m_tiles * n_tiles * k_tiles) // n_sms)


# --------------------------------------------------------------------------
# tolerance of reading R12 (used by the parity tests, stated once here)
# --------------------------------------------------------------------------
def output_tolerance(Y64: np.ndarray, T: np.ndarray, G: int, out_is_f16: bool) -> np.ndarray:
    """|y - Y64| <= 1e-3 |Y64| + (G+2) 2^-23 T  (+ one FP16 subnormal ulp for FP16 out)."""
    tol = 1e-3 * np.abs(Y64) + (G + 2) * 2.0 ** -23 * T
    if out_is_f16:
        tol = tol + 2.0 ** -24
    return tol
