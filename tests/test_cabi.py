"""CPU-only checks of the boundary: libapex4.so builds/loads, exports every symbol include/apex4.h
declares, and its host-side functions (no CUDA work) agree with the oracle's policy table."""
import ctypes
import os
import re

import pytest

from conftest import ROOT
from oracle import apex4_oracle as O


@pytest.fixture(scope="module")
def L():
    from paper_2606_08761_b200 import build as B
    B.build()
    from paper_2606_08761_b200 import apex4
    return apex4.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "apex4.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(apex4_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(L):
    names = declared_symbols()
    assert "apex4_quantize_act" in names and "apex4_pack_weights" in names and "apex4_w4a4_gemm" in names
    for n in names:
        assert hasattr(L, n), n
    from paper_2606_08761_b200 import apex4
    assert set(apex4.EXPORTS) == set(names)


def test_status_strings(L):
    from paper_2606_08761_b200 import apex4
    assert apex4.status_string(0) == "ok"
    assert "workspace" in apex4.status_string(apex4.ERR_WORKSPACE)
    assert "unknown" in apex4.status_string(99)


def test_policy_table_matches_oracle(L):
    from paper_2606_08761_b200 import apex4
    K = 4096
    for layer in range(10):
        assert apex4.resolve_group_size(K, 128, apex4.GRAN_GROUP, layer) == 128
        assert apex4.resolve_group_size(K, 0, apex4.GRAN_CHANNEL, layer) == K
        assert apex4.resolve_group_size(K, 0, apex4.GRAN_MIXED, layer) == \
            O.resolve_group_size(K, layer, O.POLICY_PAPER_MIX)
        assert apex4.resolve_group_size(K, 0, apex4.GRAN_MIXED_G128, layer) == \
            O.resolve_group_size(K, layer, O.POLICY_BASELINE_MIX)
    assert apex4.resolve_group_size(K, 128, apex4.GRAN_GROUP, apex4.LAYER_DOWN) == \
        O.resolve_group_size(K, O.LAYER_DOWN, O.POLICY_UNIFORM_G128)


def test_argument_validation_without_gpu(L):
    from paper_2606_08761_b200 import apex4
    with pytest.raises(apex4.Apex4Error) as e:
        apex4.resolve_group_size(4096, 48)            # not 32/64/multiple of 128
    assert e.value.status == apex4.ERR_UNSUPPORTED_SHAPE
    with pytest.raises(apex4.Apex4Error):
        apex4.resolve_group_size(4000, 32)            # K % 128 != 0
    with pytest.raises(apex4.Apex4Error):
        apex4.resolve_group_size(4096, 128, 7)        # unknown gran
    with pytest.raises(apex4.Apex4Error):
        apex4.resolve_group_size(4096, 3072)          # does not divide K
    assert apex4.packed_bytes(16, 512) == 4 * 8192    # 1 row tile x 4 k-blocks
    assert apex4.packed_bytes(129, 512) == 8 * 8192
    assert apex4.scale_elems(16, 512, 128) == 128 * 4
    # null pointers are rejected before any CUDA call
    assert L.apex4_w4a4_gemm(None, None, None, None, None, 0, 16, 256, 512, 128, 0, 0, None, 0, None) \
        == apex4.ERR_INVALID_ARG
    assert L.apex4_quantize_act(None, 16, 512, 128, 0, 0, None, None, None) == apex4.ERR_INVALID_ARG


def test_dispatch_table(L):
    """Host-side choice of kernel / token-tile width / work distribution (a6, a8): pure host code, a pure
    function of the problem and the per-call options (no global switch)."""
    from paper_2606_08761_b200 import apex4
    DEC, PAIR = apex4.KERNEL_DECODE, apex4.KERNEL_PAIR
    # decode regime, g = 128: the streaming kernel, 8-row row blocks over all SMs, no workspace
    kern, width, split, grid, upt = apex4.debug_get_dispatch(16, 8192, 8192, 128)
    assert (kern, width, split, upt) == (DEC, 16, 0, 7) and 1 <= grid <= 148
    assert apex4.debug_get_dispatch(32, 8192, 8192, 128)[:2] == (DEC, 32)
    assert apex4.workspace_bytes(16, 8192, 8192, 128) == 0
    # 32 < M <= 64: CTA pairs on 256 x 64 tiles, 32 tiles on <= 74 pairs -> stream-K; the workspace has one slot per
    # CTA pair (2 arrival counters, padded to 256 bytes in total, + a 256 x 64 FP32 tile), whatever M and N are
    kern, width, split, grid, upt = apex4.debug_get_dispatch(64, 8192, 8192, 128)
    assert (kern, width, split, upt) == (PAIR, 64, 1, 64)
    pad256 = lambda n: (n + 255) // 256 * 256
    assert apex4.workspace_bytes(64, 8192, 8192, 128) == pad256(grid * 8) + grid * 256 * 64 * 4
    # M = 256: two 128-token tiles instead of a 192-token tile and a third-full one
    assert apex4.debug_get_dispatch(256, 4096, 4096, 128)[1] == 128
    # tensor-bound regime: CTA pairs on 256 x 192 tiles; 43 x 32 tiles fill the last wave -> whole tiles
    kern, width, split, grid, upt = apex4.debug_get_dispatch(8192, 8192, 8192, 128)
    assert (kern, width, split, upt) == (PAIR, 192, 0, 64) and 1 <= grid <= 74
    assert apex4.workspace_bytes(8192, 8192, 8192, 128) == 0
    # Llama-2-7B O-proj at M = 2048: 11 x 16 tiles on <= 74 pairs -> stream-K with the FP32 workspace
    kern, width, split, grid, upt = apex4.debug_get_dispatch(2048, 4096, 4096, 128)
    assert (kern, width, split, upt) == (PAIR, 192, 1, 32)
    # per CTA pair: 2 counters + a 256 x 192 tile as FP32 in fragment order -- at most ~14.6 MB on 74 pairs
    assert apex4.workspace_bytes(2048, 4096, 4096, 128) == pad256(grid * 8) + grid * 256 * 192 * 4
    assert apex4.workspace_bytes(2048, 4096, 4096, 128) <= 16 << 20
    assert apex4.workspace_bytes(4096, 57344, 8192, 32) <= 16 << 20
    # per-channel decode: the streaming kernel with an exact INT32 cross-warp reduction, no workspace
    assert apex4.debug_get_dispatch(16, 8192, 8192, 0, apex4.GRAN_CHANNEL)[:3] == (DEC, 16, 0)
    assert apex4.workspace_bytes(16, 8192, 8192, 8192) == 0
    # groups between 128 and K at small M: the decode kernel where the groups nest with its 16 warps' k ranges
    # (K / 16 a multiple of g, or g a multiple of K / 16 with K / g dividing 16), CTA pairs on 256 x 64 tiles otherwise
    for g in (256, 512, 1024, 2048, 4096):
        assert apex4.debug_get_dispatch(16, 8192, 8192, g)[0] == DEC
    assert apex4.debug_get_dispatch(16, 8192, 28672, 256)[0] == DEC
    kern, width, split, grid, upt = apex4.debug_get_dispatch(16, 8192, 28672, 1024)      # 224 k-blocks: 14 per warp, 8 per group
    assert (kern, width, upt) == (PAIR, 64, 28)
    assert apex4.debug_get_dispatch(16, 4096, 11008, 256)[0] == PAIR                      # 86 k-blocks do not split over 16 warps
    # per-call options: forcing the pair kernel / a tile width / stream-K changes this call only
    o = apex4.debug_opts(kernel=PAIR, pair_tokens=128, split=1, grid=5)
    assert apex4.debug_get_dispatch(16, 256, 512, 128, opts=o)[:4] == (PAIR, 128, 1, 4)   # 4 units: grid capped
    assert apex4.workspace_bytes(16, 256, 512, 128, opts=o) == 256 + 4 * 256 * 128 * 4           # one slot per pair of the launch
    assert apex4.debug_get_dispatch(16, 256, 512, 128)[0] == DEC                           # ... not the next one
    with pytest.raises(apex4.Apex4Error):            # the decode kernel does not cover M > 32
        apex4.debug_get_dispatch(64, 256, 512, 128, opts=apex4.debug_opts(kernel=DEC))
    with pytest.raises(apex4.Apex4Error):            # ... nor groups that do not nest with its warps' k ranges
        apex4.debug_get_dispatch(16, 256, 1024, 256, opts=apex4.debug_opts(kernel=DEC))
