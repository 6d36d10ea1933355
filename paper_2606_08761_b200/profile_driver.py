"""Tool behind the files under profiles/ (each names its exact command): runs ONE op of the hot path a fixed
number of times on random operands of the right layouts, rotating through operand sets larger than L2.

    python -m paper_2606_08761_b200.profile_driver gemm M,N,K,g [launches]      launches for ncu -k regex:... -s S -c C
    python -m paper_2606_08761_b200.profile_driver quant M,K,g [launches]
    python -m paper_2606_08761_b200.profile_driver time M,N,K,g [...]           sweep-protocol time of the GEMM (one JSON line per shape)
    python -m paper_2606_08761_b200.profile_driver timeline M,N,K,g             device timeline of CTA pair 0 (needs a -DAPEX4_TIMELINE build)
    python -m paper_2606_08761_b200.profile_driver pipes                        apex4_measure_epilogue_pipes table
    python -m paper_2606_08761_b200.profile_driver stream                       apex4_measure_epilogue_stream table

Variant libraries (the APEX4_X_* / APEX4_TIMELINE tuning switches) are built with
`python -m paper_2606_08761_b200.build --out /tmp/x.so -DAPEX4_X_NOWIDEN ...` and loaded with APEX4_LIB=/tmp/x.so.
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


TL_EVENTS = {0: "producer issue", 1: "widener: packed stage full", 2: "widener: operand stage empty", 3: "widener: stage published",
             4: "MMA: operands full", 8: "MMA: accumulator empty", 5: "MMA: issued", 6: "epilogue: group begins", 17: "epilogue: chunk 0 in registers",
             16: "epilogue: accumulator released", 7: "epilogue: group ends"}


def run_timeline(M: int, N: int, K: int, g: int) -> None:
    """clock64 stamps of CTA 0 / 1 (rank 0 / 1 of pair 0), group index 8..40, relative to the first."""
    import numpy as np
    dev = torch.device("cuda")
    qA = torch.randint(0, 256, (apex4.packed_bytes(M, K),), dtype=torch.uint8, device=dev)
    qW = torch.randint(0, 256, (apex4.packed_bytes(N, K),), dtype=torch.uint8, device=dev)
    sA = (torch.rand(apex4.scale_elems(M, K, g), device=dev) * 0.1 + 0.01).half()
    sW = (torch.rand(apex4.scale_elems(N, K, g), device=dev) * 0.01 + 0.001).half()
    tl = torch.zeros(64 * 64, dtype=torch.int64, device=dev)
    o = apex4.debug_opts(kernel=apex4.KERNEL_PAIR, timeline=tl.data_ptr())
    for _ in range(3):
        apex4.w4a4_gemm(qA, sA, qW, sW, M, N, K, g, opts=o)
    torch.cuda.synchronize()
    t = tl.cpu().numpy().reshape(64, 64)
    if not t.any():
        raise SystemExit("no stamps: the loaded library was not built with -DAPEX4_TIMELINE")
    base = t[6, 8]
    ev = sorted(TL_EVENTS)
    print("events: " + "; ".join(f"{e} = {TL_EVENTS[e]}" for e in ev))
    print("k    " + " ".join(f"ev{e:<9d}" for e in ev) + "  | rank 1: " + " ".join(f"ev{e:<9d}" for e in (6, 16, 7)))
    for k in range(8, 40):
        print(f"{k:3d}  " + " ".join(f"{int(t[e, k] - base):11d}" for e in ev) + "  |         " + " ".join(f"{int(t[32 + e, k] - base):11d}" for e in (6, 16, 7)))
    print("epilogue period (rank 0) mean", float(np.diff(t[6, 8:56]).mean()), "clk")


def main(argv) -> int:
    if len(argv) >= 2 and argv[1] == "pipes":
        for k, v in apex4.measure_epilogue_pipes().items():
            print(f"{k:12s} TMEM warp {v['tmem_clk_per_16_columns']:7.1f} clk / 16 columns   FFMA2 warp {v['ffma2_clk_per_32']:7.1f} clk / 32 FFMA2")
        return 0
    if len(argv) >= 2 and argv[1] == "stream":
        for k, v in apex4.measure_epilogue_stream().items():
            print(f"{k:24s} {v:7.1f} clk / group (192 columns, 8 warps)")
        return 0
    if len(argv) >= 3 and argv[1] == "time":
        import json
        from . import sweep
        for spec in argv[2:]:
            M, N, K, g = [int(v) for v in spec.split(",")]
            print(json.dumps(sweep.time_shape(M, N, K, g, torch.device("cuda"), cublas=False)))
        return 0
    if len(argv) >= 3 and argv[1] == "timeline":
        run_timeline(*[int(v) for v in argv[2].split(",")])
        return 0
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
