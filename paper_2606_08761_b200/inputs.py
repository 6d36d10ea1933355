"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests/bench.

This module holds NONE of the method's arithmetic (no quantizer, no GEMM): it
only draws FP16 operands with the shapes and value distributions that
BASELINE.json's configs and SURVEY.md 8(d) prescribe (Gaussian activations with
a few outlier channels x20, weights ~ N(0, 0.02), PAPER.md:35,118 describe the
outlier structure these mimic).  The same bytes go to the oracle and to the GPU.

Recipe:
  W[n,k] = fp16( 0.02 * z ),  z ~ N(0,1) float32 from PCG64([seed, 1])
  X[m,k] = fp16( z * (20 if k in O else 1) ),  z from PCG64([seed, 2]), row-major,
           so the first M rows of any larger draw are identical (nested M sweeps)
  O      = fixed {3, 77, 300, 511} for configs 0/1 (R15), else the first
           round(0.01 K) entries of PCG64([seed, 3]).permutation(K)
  seed   = 0 for config 0, else 1000*config + shape_index
"""
from __future__ import annotations

import numpy as np

FIXED_OUTLIERS = (3, 77, 300, 511)

# BASELINE.json configs -> shapes (M, N, K, g); g = 0 means per-channel (g = K)
LLAMA2_7B_SHAPES = {            # config 1, M = 2048
    "qkv": (12288, 4096), "o": (4096, 4096), "gate_up": (22016, 4096), "down": (4096, 11008),
}
LLAMA2_70B_SHAPES = {           # config 4
    "qkv": (10240, 8192), "o": (8192, 8192), "gate_up": (57344, 8192), "down": (8192, 28672),
}
SQUARE_SWEEP_M = (1, 4, 16, 64, 256, 1024, 4096, 8192)      # config 2, N = K = 8192
GRAN_SWEEP_G = (32, 64, 128, 0)                              # config 3, M = 4096, N = K = 8192
LLAMA70B_M = (1, 16, 256, 4096)


def config_seed(config: int, shape_index: int = 0) -> int:
    return 0 if config == 0 else 1000 * config + shape_index


def outlier_channels(K: int, seed: int, fixed: bool) -> np.ndarray:
    if fixed:
        return np.array([k for k in FIXED_OUTLIERS if k < K], dtype=np.int64)
    n = int(round(0.01 * K))
    perm = np.random.Generator(np.random.PCG64([seed, 3])).permutation(K)
    return np.sort(perm[:n]).astype(np.int64)


def make_weights(N: int, K: int, seed: int) -> np.ndarray:
    rng = np.random.Generator(np.random.PCG64([seed, 1]))
    out = np.empty((N, K), dtype=np.float16)
    step = max(1, (1 << 24) // K)
    for r0 in range(0, N, step):
        r1 = min(N, r0 + step)
        z = rng.standard_normal((r1 - r0, K), dtype=np.float32)
        out[r0:r1] = (np.float32(0.02) * z).astype(np.float16)
    return out


def make_activations(M: int, K: int, seed: int, fixed_outliers: bool) -> np.ndarray:
    rng = np.random.Generator(np.random.PCG64([seed, 2]))
    mult = np.ones(K, dtype=np.float32)
    mult[outlier_channels(K, seed, fixed_outliers)] = 20.0
    out = np.empty((M, K), dtype=np.float16)
    step = max(1, (1 << 24) // K)
    for r0 in range(0, M, step):
        r1 = min(M, r0 + step)
        z = rng.standard_normal((r1 - r0, K), dtype=np.float32)
        out[r0:r1] = (z * mult[None, :]).astype(np.float16)
    return out


def make_gemm_inputs(M: int, N: int, K: int, seed: int, fixed_outliers: bool = False):
    """Returns (X[M,K] fp16, W[N,K] fp16)."""
    return make_activations(M, K, seed, fixed_outliers), make_weights(N, K, seed)


def config0():
    """BASELINE.json config 0: M=16, N=256, K=512, g=128, seed 0, 4 fixed outlier channels."""
    X, W = make_gemm_inputs(16, 256, 512, 0, fixed_outliers=True)
    return X, W, 128


def sample_rows(M: int, seed: int, n_random: int = 21) -> np.ndarray:
    """Row/column subset for parity at scale: tile edges + seeded random rows."""
    fixed = [0, 1, 63, 64, 127, 128, 255, 256, M // 2, M - 2, M - 1]
    rng = np.random.Generator(np.random.PCG64([seed, 4]))
    rnd = rng.integers(0, M, size=n_random).tolist() if M > 0 else []
    rows = sorted({r for r in fixed + rnd if 0 <= r < M})
    return np.array(rows, dtype=np.int64)
