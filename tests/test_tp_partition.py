"""K-split tensor parallelism: the partition on group boundaries and the reduction, on CPU with a
world_size-2 gloo group.  The per-rank compute step is the ORACLE here (this is a test of the host logic and of the
collective plumbing; the CUDA kernels are covered by the -m gpu tests)."""
import os
import subprocess
import sys

import numpy as np
import pytest

from conftest import ROOT


def test_k_split_properties():
    from paper_2606_08761_b200.tp import k_split
    for K, g, world in [(8192, 128, 8), (4096, 32, 2), (11008, 128, 4), (28672, 28672, 2), (1024, 512, 3), (512, 64, 8), (128, 128, 4)]:
        parts = k_split(K, g, world)
        assert len(parts) == world and parts[0][0] == 0 and parts[-1][1] == K
        unit = g if g % 128 == 0 else 128
        sizes = []
        for (a, b), nxt in zip(parts, parts[1:] + [(K, K)]):
            assert b == nxt[0] and (b - a) % unit == 0 and a % g == 0 and b % g == 0      # contiguous, whole groups and k-blocks
            sizes.append((b - a) // unit)
        assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        k_split(4096, 96, 2)
    with pytest.raises(ValueError):
        k_split(4000, 32, 2)


def test_owner_columns_of_the_fused_reduce_scatter():
    from paper_2606_08761_b200.tp import owner_columns
    for N, world in [(8192, 8), (4096, 2), (384, 3), (1024, 1), (57344, 7)]:
        cols = owner_columns(N, world)
        assert len(cols) == world and cols[0][0] == 0 and cols[-1][1] == N
        assert all(b - a == N // world and a % 8 == 0 for a, b in cols)
        assert all(cols[i][1] == cols[i + 1][0] for i in range(world - 1))
    for N, world in [(4096, 3), (8200, 4), (24, 2)]:        # unequal pieces / pieces that are not whole 8-column units
        with pytest.raises(ValueError):
            owner_columns(N, world)


WORKER = r"""
import os, sys
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, {root!r})
from oracle import apex4_oracle as O
from paper_2606_08761_b200 import inputs
from paper_2606_08761_b200.tp import k_split, row_parallel_linear
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank, world = dist.get_rank(), dist.get_world_size()
M, N, K = 24, 40, 1024
for g in (32, 128, 512):
    X, W = inputs.make_gemm_inputs(M, N, K, seed=31 + g, fixed_outliers=True)
    def local(k0, k1):
        r = O.w4a4_linear(X[:, k0:k1], W[:, k0:k1], g)          # the slice quantizes on its own: scales are per group
        return torch.from_numpy(r["Y64"].astype(np.float32))      # FP32 partial, as the CUDA path would return
    y = row_parallel_linear(rank, world, K, g, local, lambda t: dist.all_reduce(t, op=dist.ReduceOp.SUM))
    ref = O.w4a4_linear(X, W, g)
    tol = O.output_tolerance(ref["Y64"], ref["T"], K // g, False)
    assert np.all(np.abs(y.numpy().astype(np.float64) - ref["Y64"]) <= tol), g
    # integer stages are identical on the slice: codes of the slice == slice of the codes
    k0, k1 = k_split(K, g, world)[rank]
    qs, ss = O.quantize(X[:, k0:k1], g)
    assert np.array_equal(qs, ref["qA"][:, k0:k1]) and np.array_equal(ss.view(np.uint16), ref["sA"][:, k0 // g:k1 // g].view(np.uint16))
dist.barrier()
dist.destroy_process_group()
print("rank", rank, "ok")
"""


def test_row_parallel_two_ranks_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT, port=29533))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True,
                              env=dict(os.environ, MASTER_ADDR="127.0.0.1")) for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
        assert "ok" in o
