"""K-split (row-parallel) tensor parallelism of the W4A4 linear, SURVEY 8(e)(3) / 8(f)4.

The hot path shards with no exchange along M (replicas) and N (column-parallel).  Along K it shards on GROUP
boundaries only: a rank quantizes its own K-slice of X (the scales of Eq. 7 are per group, so a slice is
self-contained), computes an FP32 partial Y with the same kernels, and the partials are summed -- the one real
exchange step, the multi-GPU form of the paper's inter-SM reduction.  Per-group integer sums
stay bit-exact on every rank; only the FP32 summation order changes (inside the R12 tolerance of DESIGN.md).

This module holds the host logic (the partition, the owner map, the buffer exchange) and two forms of the exchange:
  * row_parallel_linear: local GEMM into FP32, then torch.distributed all-reduce (NCCL over NVLink) -- the baseline;
  * row_parallel_linear_push: the reduce-scatter FUSED into the GEMM (apex4_w4a4_gemm_tp_push): every rank owns the
    output columns [N r / R, N (r + 1) / R) in an FP32 buffer, opens its peers' buffers through CUDA IPC (NVLink P2P),
    and the epilogue of its K-slice GEMM adds each finished partial tile straight into the owner's buffer
    (red.global.add.f32, system scope) while the later tiles are still being computed.  Host barriers bracket the
    kernel; no kernel waits on another rank's kernel.
Every run of this project has one GPU: the fused kernel is tested there with the ranks' launches issued one after the
other, and with two PROCESSES sharing the one GPU through CUDA IPC (tests/test_gpu_tp_push.py); NVLink itself is untested.
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


# ---------------------------------------------------------------------------------- fused reduce-scatter (push)
def owner_columns(N: int, world: int) -> List[Tuple[int, int]]:
    """Output columns [n0, n1) owned by each rank for the fused reduce-scatter: equal pieces of whole 8-column units
    (the kernels add 8-column pieces; apex4_w4a4_gemm_tp_push rejects anything else)."""
    if world < 1 or N % world != 0 or (N // world) % 8 != 0:
        raise ValueError("owner_columns: N must split into `world` equal pieces of whole 8-column units")
    c = N // world
    return [(r * c, (r + 1) * c) for r in range(world)]


def share_buffer(t) -> tuple:
    """Picklable CUDA IPC description of a device tensor (its storage), for a peer process to open."""
    return (tuple(t.untyped_storage()._share_cuda_()), t.dtype, tuple(t.shape), t.storage_offset())


def open_buffer(desc):
    """The peer's tensor described by share_buffer(), mapped into this process (NVLink P2P between GPUs)."""
    import torch
    meta, dtype, shape, offset = desc
    st = torch.UntypedStorage._new_shared_cuda(*meta)
    return torch.empty(0, dtype=dtype, device=st.device).set_(st, offset, shape)


class PushGroup:
    """The owners' accumulation buffers of one (M, N) output, exchanged once and reused by every call.
    all_gather_object / barrier: the process group's (torch.distributed with any backend; gloo is enough)."""

    def __init__(self, rank: int, world: int, M: int, N: int, device, all_gather_object, barrier):
        import torch
        self.rank, self.world, self.M, self.N, self.barrier = rank, world, M, N, barrier
        self.cols = owner_columns(N, world)
        self.mine = torch.zeros((M, N // world), dtype=torch.float32, device=device)
        descs = all_gather_object(share_buffer(self.mine)) if world > 1 else [None]
        self.bufs = [self.mine if r == rank else open_buffer(descs[r]) for r in range(world)]
        self.ptrs = [b.data_ptr() for b in self.bufs]


def row_parallel_linear_push(group: "PushGroup", x, qW_slice, sW_slice, K: int, g: int):
    """This rank's part of Y = X W^T with the reduce-scatter fused into the GEMM.  x: the rank's [M, K_r] FP16 slice of
    X (device), qW_slice / sW_slice: its packed weight slice.  Returns the rank's OWN output columns [M, N / world] FP32
    (group.cols[rank]); complete once every rank has returned."""
    import torch
    from . import apex4
    k0, k1 = k_split(K, g, group.world)[group.rank]
    group.mine.zero_()
    torch.cuda.synchronize()
    group.barrier()                      # every owner's buffer is zero before anyone pushes
    if k1 > k0:
        qA, sA, _ = apex4.quantize_act(x, g)
        apex4.w4a4_gemm_tp_push(qA, sA, qW_slice, sW_slice, group.ptrs, group.M, group.N, k1 - k0, g)
    torch.cuda.synchronize()
    group.barrier()                      # every rank's pushes have landed
    return group.mine
