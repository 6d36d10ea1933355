"""Driver for ncu captures (profiles/*.md name the exact command): runs ONE op of the hot path a fixed
number of times on random operands of the right layouts, rotating through operand sets larger than L2.

    python -m paper_2606_08761_b200.profile_driver gemm M,N,K,g [launches]
    python -m paper_2606_08761_b200.profile_driver quant M,K,g [launches]

Timing is bench.py's business; this only produces launches for `ncu -k regex:... -s S -c C`.
"""
from __future__ import annotations

import sys

import torch

from . import apex4

L2_BYTES = 126e6


def run_gemm(M: int, N: int, K: int, g: int, launches: int) -> None:
    dev = torch.device("cuda")
    nsets = int(max(2, min(8, 2 * L2_BYTES // (N * K / 2 + M * K / 2) + 1)))
    sets = []
    for _ in range(nsets):
        sets.append((torch.randint(0, 256, (apex4.packed_bytes(M, K),), dtype=torch.uint8, device=dev),
                     (torch.rand(apex4.scale_elems(M, K, g), device=dev) * 0.1 + 0.01).half(),
                     torch.randint(0, 256, (apex4.packed_bytes(N, K),), dtype=torch.uint8, device=dev),
                     (torch.rand(apex4.scale_elems(N, K, g), device=dev) * 0.01 + 0.001).half()))
    Y = torch.empty((M, N), dtype=torch.float16, device=dev)
    ws = apex4.make_workspace(M, N, K, g, device=dev)
    for i in range(launches):
        qA, sA, qW, sW = sets[i % nsets]
        apex4.w4a4_gemm(qA, sA, qW, sW, M, N, K, g, out=Y, workspace=ws)
    torch.cuda.synchronize()


def run_quant(M: int, K: int, g: int, launches: int) -> None:
    dev = torch.device("cuda")
    nsets = int(max(2, min(8, 2 * L2_BYTES // (2 * M * K) + 1)))
    xs = [torch.randn(M, K, device=dev, dtype=torch.float16) for _ in range(nsets)]
    q = torch.empty(apex4.packed_bytes(M, K), dtype=torch.uint8, device=dev)
    s = torch.empty(apex4.scale_elems(M, K, g), dtype=torch.float16, device=dev)
    for i in range(launches):
        apex4.quantize_act(xs[i % nsets], g, q=q, s=s)
    torch.cuda.synchronize()


def main(argv) -> int:
    if len(argv) < 3 or argv[1] not in ("gemm", "quant"):
        print(__doc__)
        return 2
    dims = [int(v) for v in argv[2].split(",")]
    launches = int(argv[3]) if len(argv) > 3 else 18
    if argv[1] == "gemm":
        run_gemm(*dims, launches)
    else:
        run_quant(*dims, launches)
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv))
