"""K-split (row-parallel) tensor parallelism of the W4A4 linear, SURVEY 8(e)(3) / 8(f)4.

The hot path shards with no exchange along M (replicas) and N (column-parallel).  Along K it shards on GROUP
boundaries only: a rank quantizes its own K-slice of X (the scales of Eq. 7 are per group, so a slice is
self-contained), computes an FP32 partial Y with the same kernels, and the partials are summed -- the one real
exchange step, the multi-GPU form of the paper's inter-SM reduction.  Per-group integer sums
stay bit-exact on every rank; only the FP32 summation order changes (inside the R12 tolerance of DESIGN.md).

This module holds the host logic (the partition) and the NCCL path: local GEMM into FP32, then
torch.distributed all-reduce over NVLink.  The collective is NOT fused into the GEMM epilogue (pushing partial
tiles to peers through NVLink-mapped memory): with one GPU per run in this project that kernel could not be
executed, so it is left out rather than shipped untested; DESIGN.md section 8 says so.
"""
from __future__ import annotations

from typing import Callable, List, Tuple


def k_split(K: int, g: int, world: int) -> List[Tuple[int, int]]:
    """K-ranges [k0, k1) per rank: whole groups (and whole 128-k blocks, the unit of the packed layouts), as even as
    possible, earlier ranks take the remainder.  Ranks beyond the number of units get an empty range."""
    if K <= 0 or g <= 0 or K % g != 0 or world < 1:
        raise ValueError("k_split: K must be a positive multiple of g, world >= 1")
    unit = g if g % 128 == 0 else 128          # g = 32 / 64: a 128-k block holds whole groups
    if K % unit != 0:
        raise ValueError("k_split: K must be a multiple of the 128-k block")
    units = K // unit
    base, rem = divmod(units, world)
    out, k0 = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        out.append((k0, k0 + n * unit))
        k0 += n * unit
    assert k0 == K
    return out


def row_parallel_linear(rank: int, world: int, K: int, g: int, local_partial: Callable[[int, int], "object"], all_reduce) -> "object":
    """Y = sum over ranks of the partial products of their K-slices.  local_partial(k0, k1) returns this rank's FP32
    partial Y[M, N] for columns k0..k1 of X and W (zeros for an empty slice); all_reduce sums it in place over ranks."""
    k0, k1 = k_split(K, g, world)[rank]
    y = local_partial(k0, k1)
    all_reduce(y)
    return y


def cuda_local_partial(x, qW_slices, sW_slices, N: int, g: int):
    """local_partial for the CUDA path: x is this rank's [M, K_r] FP16 slice (device), qW/sW its pre-packed weight
    slice; quantizer + GEMM with FP32 output (no CPU fallback: raises without the library / a GPU)."""
    import torch
    from . import apex4

    def fn(k0: int, k1: int):
        M = x.shape[0]
        if k1 == k0:
            return torch.zeros((M, N), dtype=torch.float32, device=x.device)
        qA, sA, _ = apex4.quantize_act(x, g)
        return apex4.w4a4_gemm(qA, sA, qW_slices, sW_slices, M, N, k1 - k0, g, out_dtype=torch.float32)
    return fn
