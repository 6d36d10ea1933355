"""apex4_w4a4_gemm_tp_push (-m gpu): K-split tensor parallelism with the reduce-scatter fused into the GEMM epilogue
(SURVEY 8(e)(3), 8(f)4).  One GPU per run in this project, so (1) the ranks' launches are issued one after the other into
owner buffers that all live on the one device, and (2) two PROCESSES share the one GPU: each opens the other's buffer
through CUDA IPC (the mechanism that maps NVLink peers) and pushes into it; host barriers over gloo.  No kernel waits on
another rank's kernel.  Reference: the oracle's full-K linear, the tests' output tolerance."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch

from conftest import ROOT
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


# (M, N, K, g, world): decode kernel, pair kernel with whole tiles and stream-K, fine and coarse groups, 3 ranks with an
# uneven K split, more ranks than the decode kernel has row blocks per owner
CASES = [(16, 256, 1024, 128, 2), (300, 512, 1024, 128, 2), (200, 528, 2048, 32, 2), (130, 768, 2048, 512, 2),
         (64, 384, 1664, 128, 3), (8, 1024, 4096, 64, 4), (700, 1024, 1024, 128, 2)]


@pytest.mark.parametrize("M,N,K,g,world", CASES)
def test_tp_push_ranks_in_sequence(A, M, N, K, g, world):
    from paper_2606_08761_b200.tp import k_split, owner_columns
    X, W = inputs.make_gemm_inputs(M, N, K, seed=700 + M)
    ref = O.w4a4_linear(X, W, g)
    cols = owner_columns(N, world)
    bufs = [torch.zeros((M, N // world), dtype=torch.float32, device="cuda") for _ in range(world)]
    ptrs = [b.data_ptr() for b in bufs]
    for _ in range(2):                                     # twice: the second round starts from re-zeroed buffers
        for b in bufs:
            b.zero_()
        for r, (k0, k1) in enumerate(k_split(K, g, world)):
            if k1 == k0:
                continue
            qA, sA, _ = A.quantize_act(dev(X[:, k0:k1]), g)
            qW, sW, _ = A.pack_weights(dev(W[:, k0:k1]), g)
            # integer stages of a slice are the slice of the integer stages (groups are self-contained)
            assert np.array_equal(A.unpack_codes(qA, M, k1 - k0, A.OPERAND_ACT).cpu().numpy(), ref["qA"][:, k0:k1])
            A.w4a4_gemm_tp_push(qA, sA, qW, sW, ptrs, M, N, k1 - k0, g)
        torch.cuda.synchronize()
        Y = np.concatenate([b.cpu().numpy() for b in bufs], axis=1).astype(np.float64)
        assert Y.shape == (M, N) and cols[-1][1] == N
        tol = O.output_tolerance(ref["Y64"], ref["T"], K // g, False)
        err = np.abs(Y - ref["Y64"])
        assert (err <= tol).all(), (float((err / tol).max()), np.argwhere(err > tol)[:4].tolist())


def test_tp_push_argument_checks(A):
    t = torch.zeros(4096, dtype=torch.uint8, device="cuda")
    buf = torch.zeros((16, 128), dtype=torch.float32, device="cuda")
    with pytest.raises(A.Apex4Error) as e:                 # N does not split into equal 8-column pieces
        A.w4a4_gemm_tp_push(t, t, t, t, [buf.data_ptr()] * 3, 16, 256, 512, 128)
    assert e.value.status == A.ERR_UNSUPPORTED_SHAPE
    with pytest.raises(A.Apex4Error) as e:                 # more than 8 ranks
        A.w4a4_gemm_tp_push(t, t, t, t, [buf.data_ptr()] * 9, 16, 1152, 512, 128)
    assert e.value.status == A.ERR_INVALID_ARG
    with pytest.raises(A.Apex4Error) as e:                 # a null owner buffer
        A.w4a4_gemm_tp_push(t, t, t, t, [buf.data_ptr(), 0], 16, 256, 512, 128)
    assert e.value.status == A.ERR_INVALID_ARG


WORKER = r"""
import os, sys
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, {root!r}); sys.path.insert(0, os.path.join({root!r}, "tests"))
from oracle import apex4_oracle as O
from paper_2606_08761_b200 import inputs, apex4
from paper_2606_08761_b200.tp import k_split, PushGroup, row_parallel_linear_push
rank = int(sys.argv[1])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=2)
world = dist.get_world_size()
torch.cuda.set_device(0)                                   # both processes on the one GPU; buffers cross through CUDA IPC
def gather(obj):
    out = [None] * world
    dist.all_gather_object(out, obj)
    return out
for (M, N, K, g) in [(16, 512, 2048, 128), (260, 512, 1024, 128), (96, 1024, 2048, 32)]:
    X, W = inputs.make_gemm_inputs(M, N, K, seed=77 + M)
    ref = O.w4a4_linear(X, W, g)
    grp = PushGroup(rank, world, M, N, torch.device("cuda:0"), gather, dist.barrier)
    k0, k1 = k_split(K, g, world)[rank]
    x = torch.from_numpy(np.ascontiguousarray(X[:, k0:k1])).cuda()
    qW, sW, _ = apex4.pack_weights(torch.from_numpy(np.ascontiguousarray(W[:, k0:k1])).cuda(), g)
    for _ in range(2):
        y = row_parallel_linear_push(grp, x, qW, sW, K, g).cpu().numpy().astype(np.float64)
        n0, n1 = grp.cols[rank]
        tol = O.output_tolerance(ref["Y64"], ref["T"], K // g, False)[:, n0:n1]
        err = np.abs(y - ref["Y64"][:, n0:n1])
        assert (err <= tol).all(), (M, N, K, g, float((err / tol).max()))
    dist.barrier()
    del grp
dist.barrier()
dist.destroy_process_group()
print("rank", rank, "ok")
"""


def test_tp_push_two_processes_cuda_ipc(tmp_path):
    """Two processes, one GPU: each owns half of the output columns, opens the other's FP32 buffer through CUDA IPC and
    its GEMM epilogue adds partial tiles into both (tp.PushGroup / row_parallel_linear_push)."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    script = tmp_path / "tp_push_worker.py"
    script.write_text(WORKER.format(root=ROOT, port=port))
    env = dict(os.environ, PYTHONPATH=ROOT)
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
             for r in range(2)]
    outs = []
    for p in procs:
        try:
            out, _ = p.communicate(timeout=420)
        except subprocess.TimeoutExpired:
            for q in procs:
                q.kill()
            raise
        outs.append(out)
    for r, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"rank {r} ok" in out, out[-3000:]
