"""Thin Python binding of the C ABI in include/apex4.h (ctypes; argument marshalling only).

Every step of the path runs in the CUDA kernels of libapex4.so; torch is used for device memory
and streams.  There is no CPU fallback: importing works without the library (so CPU-only tooling
can import the package), but every call fails loudly if libapex4.so is missing or the device is not
sm_100a.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("APEX4_LIB") or os.path.join(_PKG, "libapex4.so")   # APEX4_LIB: load another build

# enums of include/apex4.h
OK, ERR_INVALID_ARG, ERR_UNSUPPORTED_SHAPE, ERR_ALIGNMENT, ERR_WORKSPACE, ERR_CUDA, ERR_ARCH = range(7)
GRAN_GROUP, GRAN_CHANNEL, GRAN_MIXED, GRAN_MIXED_G128 = range(4)
(LAYER_OTHER, LAYER_Q, LAYER_K, LAYER_V, LAYER_QKV, LAYER_O, LAYER_GATE, LAYER_UP, LAYER_GATE_UP,
 LAYER_DOWN) = range(10)
OUT_F16, OUT_F32 = 0, 1
OPERAND_ACT, OPERAND_WEIGHT = 0, 1

EXPORTS = (
    "apex4_resolve_group_size", "apex4_packed_bytes", "apex4_scale_elems", "apex4_workspace_bytes",
    "apex4_workspace_bytes_ex", "apex4_status_string", "apex4_quantize_act", "apex4_pack_weights",
    "apex4_rmsnorm_quantize", "apex4_silu_mul_quantize",
    "apex4_pack_codes", "apex4_scales_from_natural", "apex4_scales_to_natural", "apex4_unpack_codes",
    "apex4_w4a4_gemm", "apex4_w4a4_gemm_ex", "apex4_w4a4_gemm_static_ws", "apex4_w4a4_gemm_tp_push", "apex4_w4a4_linear_host",
    "apex4_linear_host_scratch_bytes",
    "apex4_debug_group_sums", "apex4_debug_get_dispatch", "apex4_measure_rho", "apex4_measure_epilogue_pipes", "apex4_measure_epilogue_stream",
    "apex4_e4m3_exactness",
)


class DebugOpts(ctypes.Structure):
    """apex4_debug_opts of include/apex4.h: per-call kernel / tile / work-distribution overrides."""
    _fields_ = [("kernel", ctypes.c_int), ("pair_tokens", ctypes.c_int), ("split", ctypes.c_int),
                ("grid", ctypes.c_int), ("decode_batch", ctypes.c_int), ("timeline", ctypes.c_void_p)]


KERNEL_DECODE, KERNEL_PAIR = 0, 1


def debug_opts(kernel: int = -1, pair_tokens: int = 0, split: int = -1, grid: int = 0, decode_batch: int = 0,
               timeline: int = 0) -> DebugOpts:
    return DebugOpts(kernel, pair_tokens, split, grid, decode_batch, timeline or None)


def _opts_ref(opts: Optional[DebugOpts]):
    return ctypes.byref(opts) if opts is not None else None


class Apex4Error(RuntimeError):
    def __init__(self, status: int, what: str):
        super().__init__(f"{what}: apex4 status {status} ({status_string(status)})")
        self.status = status


_lib = None


def lib() -> ctypes.CDLL:
    """Loads libapex4.so (built by paper_2606_08761_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(
            f"{LIB_PATH} not found: build it with `python -m paper_2606_08761_b200.build` "
            "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    c_int, c_size_t, c_void_p = ctypes.c_int, ctypes.c_size_t, ctypes.c_void_p
    L.apex4_resolve_group_size.argtypes = [c_int] * 4
    L.apex4_resolve_group_size.restype = c_int
    L.apex4_packed_bytes.argtypes = [c_int, c_int]
    L.apex4_packed_bytes.restype = c_size_t
    L.apex4_scale_elems.argtypes = [c_int, c_int, c_int]
    L.apex4_scale_elems.restype = c_size_t
    L.apex4_workspace_bytes.argtypes = [c_int] * 6
    L.apex4_workspace_bytes.restype = c_size_t
    L.apex4_workspace_bytes_ex.argtypes = [c_int] * 6 + [ctypes.POINTER(DebugOpts)]
    L.apex4_workspace_bytes_ex.restype = c_size_t
    L.apex4_status_string.argtypes = [c_int]
    L.apex4_status_string.restype = ctypes.c_char_p
    for name in ("apex4_quantize_act", "apex4_pack_weights"):
        f = getattr(L, name)
        f.argtypes = [c_void_p, c_int, c_int, c_int, c_int, c_int, c_void_p, c_void_p, c_void_p]
        f.restype = c_int
    L.apex4_rmsnorm_quantize.argtypes = [c_void_p, c_void_p, ctypes.c_float, c_int, c_int, c_int, c_int, c_int, c_void_p, c_void_p,
                                         c_void_p, c_void_p]
    L.apex4_silu_mul_quantize.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_int, c_int, c_int, c_void_p, c_void_p,
                                          c_void_p, c_void_p]
    L.apex4_rmsnorm_quantize.restype = c_int
    L.apex4_silu_mul_quantize.restype = c_int
    L.apex4_pack_codes.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_void_p]
    L.apex4_unpack_codes.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_void_p]
    L.apex4_scales_from_natural.argtypes = [c_void_p, c_int, c_int, c_void_p, c_void_p]
    L.apex4_scales_to_natural.argtypes = [c_void_p, c_int, c_int, c_void_p, c_void_p]
    L.apex4_w4a4_gemm.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_int, c_int,
                                  c_int, c_int, c_int, c_int, c_void_p, c_size_t, c_void_p]
    L.apex4_w4a4_gemm_ex.argtypes = L.apex4_w4a4_gemm.argtypes + [ctypes.POINTER(DebugOpts)]
    L.apex4_w4a4_gemm_static_ws.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_int, c_int,
                                            c_int, c_int, c_int, c_int, c_void_p]
    L.apex4_w4a4_gemm_static_ws.restype = c_int
    L.apex4_w4a4_gemm_tp_push.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, ctypes.POINTER(c_void_p), c_int, c_int, c_int,
                                          c_int, c_int, c_int, c_int, c_void_p, c_size_t, c_void_p]
    L.apex4_w4a4_gemm_tp_push.restype = c_int
    L.apex4_w4a4_linear_host.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_int, c_int, c_int,
                                         c_int, c_int, c_int, c_void_p, c_size_t, c_void_p]
    L.apex4_linear_host_scratch_bytes.argtypes = [c_int] * 6
    L.apex4_linear_host_scratch_bytes.restype = c_size_t
    L.apex4_debug_group_sums.argtypes = [c_void_p, c_void_p] + [c_int] * 10 + [c_void_p, c_void_p,
                                                                              ctypes.POINTER(DebugOpts)]
    L.apex4_measure_rho.argtypes = [ctypes.POINTER(ctypes.c_double), c_void_p]
    L.apex4_measure_epilogue_pipes.argtypes = [ctypes.POINTER(ctypes.c_double), c_void_p]
    L.apex4_measure_epilogue_pipes.restype = c_int
    L.apex4_measure_epilogue_stream.argtypes = [ctypes.POINTER(ctypes.c_double), c_void_p]
    L.apex4_measure_epilogue_stream.restype = c_int
    L.apex4_e4m3_exactness.argtypes = [c_int, c_int, c_int, ctypes.c_uint, ctypes.POINTER(ctypes.c_double), c_void_p]
    L.apex4_e4m3_exactness.restype = c_int
    L.apex4_debug_get_dispatch.argtypes = [c_int] * 6 + [ctypes.POINTER(DebugOpts), ctypes.POINTER(c_int)]
    for name in ("apex4_pack_codes", "apex4_unpack_codes", "apex4_scales_from_natural",
                 "apex4_scales_to_natural", "apex4_w4a4_gemm", "apex4_w4a4_gemm_ex", "apex4_w4a4_linear_host",
                 "apex4_debug_group_sums", "apex4_measure_rho", "apex4_debug_get_dispatch"):
        getattr(L, name).restype = c_int
    _lib = L
    return L


def status_string(status: int) -> str:
    return lib().apex4_status_string(int(status)).decode()


def _check(status: int, what: str) -> None:
    if status != OK:
        raise Apex4Error(status, what)


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _dev(t: torch.Tensor, dtype: torch.dtype, what: str) -> torch.Tensor:
    if not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise ValueError(f"{what}: expected a contiguous CUDA tensor of {dtype}")
    return t


def resolve_group_size(K: int, group_size: int, gran: int = GRAN_GROUP, layer: int = LAYER_OTHER) -> int:
    g = lib().apex4_resolve_group_size(K, group_size, gran, layer)
    if g < 0:
        raise Apex4Error(-g, "apex4_resolve_group_size")
    return g


def packed_bytes(R: int, K: int) -> int:
    return lib().apex4_packed_bytes(R, K)


def scale_elems(R: int, K: int, g: int) -> int:
    return lib().apex4_scale_elems(R, K, g)


def workspace_bytes(M: int, N: int, K: int, group_size: int, gran: int = GRAN_GROUP,
                    layer: int = LAYER_OTHER, opts: Optional[DebugOpts] = None) -> int:
    if opts is None:
        return lib().apex4_workspace_bytes(M, N, K, group_size, gran, layer)
    return lib().apex4_workspace_bytes_ex(M, N, K, group_size, gran, layer, _opts_ref(opts))


def _quantize(fn_name: str, x: torch.Tensor, group_size: int, gran: int, layer: int,
              q: Optional[torch.Tensor], s: Optional[torch.Tensor]):
    _dev(x, torch.float16, fn_name)
    R, K = x.shape
    g = resolve_group_size(K, group_size, gran, layer)
    if q is None:
        q = torch.empty(packed_bytes(R, K), dtype=torch.uint8, device=x.device)
    if s is None:
        s = torch.empty(scale_elems(R, K, g), dtype=torch.float16, device=x.device)
    st = getattr(lib(), fn_name)(x.data_ptr(), R, K, group_size, gran, layer, q.data_ptr(), s.data_ptr(),
                                 _stream())
    _check(st, fn_name)
    return q, s, g


def quantize_act(x, group_size=128, gran=GRAN_GROUP, layer=LAYER_OTHER, q=None, s=None):
    """apex4_quantize_act: X[M,K] fp16 -> (qA PT4 uint8 buffer, sA ST16 fp16 buffer, g)."""
    return _quantize("apex4_quantize_act", x, group_size, gran, layer, q, s)


def pack_weights(w, group_size=128, gran=GRAN_GROUP, layer=LAYER_OTHER, q=None, s=None):
    """apex4_pack_weights: W[N,K] fp16 -> (qW PW4, sW ST16, g)."""
    return _quantize("apex4_pack_weights", w, group_size, gran, layer, q, s)


def _fused_out(M, K, g, device, q, s, want_y):
    if q is None:
        q = torch.empty(packed_bytes(M, K), dtype=torch.uint8, device=device)
    if s is None:
        s = torch.empty(scale_elems(M, K, g), dtype=torch.float16, device=device)
    y = torch.empty((M, K), dtype=torch.float16, device=device) if want_y else None
    return q, s, y


def rmsnorm_quantize(x, gamma, eps: float, group_size=128, gran=GRAN_GROUP, layer=LAYER_OTHER, q=None, s=None, want_y=False):
    """apex4_rmsnorm_quantize: X[M,K], gamma[K] fp16 -> (qA PT4, sA ST16, g[, y fp16 [M,K]])."""
    _dev(x, torch.float16, "apex4_rmsnorm_quantize")
    _dev(gamma, torch.float16, "apex4_rmsnorm_quantize")
    M, K = x.shape
    g = resolve_group_size(K, group_size, gran, layer)
    q, s, y = _fused_out(M, K, g, x.device, q, s, want_y)
    st = lib().apex4_rmsnorm_quantize(x.data_ptr(), gamma.data_ptr(), float(eps), M, K, group_size, gran, layer, q.data_ptr(),
                                      s.data_ptr(), y.data_ptr() if y is not None else None, _stream())
    _check(st, "apex4_rmsnorm_quantize")
    return (q, s, g, y) if want_y else (q, s, g)


def silu_mul_quantize(gate, up, group_size=128, gran=GRAN_GROUP, layer=LAYER_OTHER, q=None, s=None, want_y=False):
    """apex4_silu_mul_quantize: gate, up [M,K] fp16 (views of one [M, 2K] tensor allowed: row stride >= K)
    -> (qA PT4, sA ST16, g[, y fp16 [M,K]])."""
    for t in (gate, up):
        if not t.is_cuda or t.dtype != torch.float16 or t.dim() != 2 or t.stride(1) != 1:
            raise ValueError("apex4_silu_mul_quantize: expected 2-D CUDA float16 tensors with unit column stride")
    if gate.shape != up.shape or gate.stride(0) != up.stride(0):
        raise ValueError("apex4_silu_mul_quantize: gate and up must have the same shape and row stride")
    M, K = gate.shape
    g = resolve_group_size(K, group_size, gran, layer)
    q, s, y = _fused_out(M, K, g, gate.device, q, s, want_y)
    st = lib().apex4_silu_mul_quantize(gate.data_ptr(), up.data_ptr(), gate.stride(0), M, K, group_size, gran, layer, q.data_ptr(),
                                       s.data_ptr(), y.data_ptr() if y is not None else None, _stream())
    _check(st, "apex4_silu_mul_quantize")
    return (q, s, g, y) if want_y else (q, s, g)


def pack_codes(codes: torch.Tensor, operand: int) -> torch.Tensor:
    """apex4_pack_codes: int8 codes [R,K] -> PT4 (OPERAND_ACT) or PW4 (OPERAND_WEIGHT)."""
    _dev(codes, torch.int8, "apex4_pack_codes")
    R, K = codes.shape
    q = torch.empty(packed_bytes(R, K), dtype=torch.uint8, device=codes.device)
    _check(lib().apex4_pack_codes(codes.data_ptr(), R, K, operand, q.data_ptr(), _stream()),
           "apex4_pack_codes")
    return q


def unpack_codes(q: torch.Tensor, R: int, K: int, operand: int) -> torch.Tensor:
    _dev(q, torch.uint8, "apex4_unpack_codes")
    codes = torch.empty((R, K), dtype=torch.int8, device=q.device)
    _check(lib().apex4_unpack_codes(q.data_ptr(), R, K, operand, codes.data_ptr(), _stream()),
           "apex4_unpack_codes")
    return codes


def scales_from_natural(s_nat: torch.Tensor) -> torch.Tensor:
    _dev(s_nat, torch.float16, "apex4_scales_from_natural")
    R, G = s_nat.shape
    out = torch.empty(lib().apex4_scale_elems(R, G, 1), dtype=torch.float16, device=s_nat.device)
    _check(lib().apex4_scales_from_natural(s_nat.data_ptr(), R, G, out.data_ptr(), _stream()),
           "apex4_scales_from_natural")
    return out


def scales_to_natural(s_tiled: torch.Tensor, R: int, G: int) -> torch.Tensor:
    _dev(s_tiled, torch.float16, "apex4_scales_to_natural")
    out = torch.empty((R, G), dtype=torch.float16, device=s_tiled.device)
    _check(lib().apex4_scales_to_natural(s_tiled.data_ptr(), R, G, out.data_ptr(), _stream()),
           "apex4_scales_to_natural")
    return out


def make_workspace(M, N, K, group_size=128, gran=GRAN_GROUP, layer=LAYER_OTHER, device="cuda", opts=None):
    """Zero-filled workspace for apex4_w4a4_gemm (None if the problem needs none)."""
    nbytes = workspace_bytes(M, N, K, group_size, gran, layer, opts)
    if nbytes == 0:
        return None
    return torch.zeros(nbytes, dtype=torch.uint8, device=device)


def w4a4_gemm(qA, sA, qW, sW, M: int, N: int, K: int, group_size=128, gran=GRAN_GROUP,
              layer=LAYER_OTHER, out_dtype=torch.float16, workspace=None, out=None,
              opts: Optional[DebugOpts] = None) -> torch.Tensor:
    """apex4_w4a4_gemm (apex4_w4a4_gemm_ex when `opts` is given): Y[M,N] = sum_g sA sW P_g (Eq. 8)."""
    if out is None:
        out = torch.empty((M, N), dtype=out_dtype, device=qA.device)
    code = OUT_F16 if out.dtype == torch.float16 else OUT_F32
    if workspace is None:
        workspace = make_workspace(M, N, K, group_size, gran, layer, qA.device, opts)
    wp = workspace.data_ptr() if workspace is not None else None
    wb = workspace.numel() if workspace is not None else 0
    args = (qA.data_ptr(), sA.data_ptr(), qW.data_ptr(), sW.data_ptr(), out.data_ptr(), code, M, N, K,
            group_size, gran, layer, wp, wb, _stream())
    if opts is None:
        _check(lib().apex4_w4a4_gemm(*args), "apex4_w4a4_gemm")
    else:
        _check(lib().apex4_w4a4_gemm_ex(*args, _opts_ref(opts)), "apex4_w4a4_gemm_ex")
    return out


def w4a4_gemm_tp_push(qA, sA, qW, sW, owner_ptrs, M: int, N: int, K_local: int, group_size=128, gran=GRAN_GROUP,
                      layer=LAYER_OTHER, workspace=None) -> None:
    """apex4_w4a4_gemm_tp_push: this rank's K-slice GEMM whose epilogue adds the FP32 partial tiles into the owners'
    [M, N / world] buffers (owner_ptrs: device addresses, one per rank; peers' buffers mapped over NVLink)."""
    world = len(owner_ptrs)
    arr = (ctypes.c_void_p * world)(*[int(v) if v else None for v in owner_ptrs])
    if workspace is None:
        workspace = make_workspace(M, N, K_local, group_size, gran, layer, qA.device)
    wp = workspace.data_ptr() if workspace is not None else None
    wb = workspace.numel() if workspace is not None else 0
    _check(lib().apex4_w4a4_gemm_tp_push(qA.data_ptr(), sA.data_ptr(), qW.data_ptr(), sW.data_ptr(), arr, world, M, N, K_local,
                                         group_size, gran, layer, wp, wb, _stream()), "apex4_w4a4_gemm_tp_push")


STATIC_WORKSPACE_BYTES = 16 << 20   # APEX4_STATIC_WORKSPACE_BYTES of include/apex4.h


def w4a4_gemm_static_ws(qA, sA, qW, sW, M: int, N: int, K: int, group_size=128, gran=GRAN_GROUP,
                        layer=LAYER_OTHER, out_dtype=torch.float16, out=None) -> torch.Tensor:
    """apex4_w4a4_gemm_static_ws: apex4_w4a4_gemm with the stream-K workspace taken from the library's static device
    array (no allocation inside the call; pass `out` to keep this wrapper allocation-free too).  Problems that need more
    than STATIC_WORKSPACE_BYTES raise Apex4Error (status APEX4_ERR_WORKSPACE); overlapping calls race on the array."""
    if out is None:
        out = torch.empty((M, N), dtype=out_dtype, device=qA.device)
    code = OUT_F16 if out.dtype == torch.float16 else OUT_F32
    _check(lib().apex4_w4a4_gemm_static_ws(qA.data_ptr(), sA.data_ptr(), qW.data_ptr(), sW.data_ptr(), out.data_ptr(),
                                           code, M, N, K, group_size, gran, layer, _stream()),
           "apex4_w4a4_gemm_static_ws")
    return out


def debug_group_sums(qA, qW, M, N, K, group_size=128, gran=GRAN_GROUP, layer=LAYER_OTHER,
                     m0=0, m1=None, n0=0, n1=None, opts: Optional[DebugOpts] = None) -> torch.Tensor:
    m1 = M if m1 is None else m1
    n1 = N if n1 is None else n1
    g = resolve_group_size(K, group_size, gran, layer)
    P = torch.empty((m1 - m0, n1 - n0, K // g), dtype=torch.int32, device=qA.device)
    st = lib().apex4_debug_group_sums(qA.data_ptr(), qW.data_ptr(), M, N, K, group_size, gran, layer,
                                      m0, m1, n0, n1, P.data_ptr(), _stream(), _opts_ref(opts))
    _check(st, "apex4_debug_group_sums")
    return P


def linear_host_scratch_bytes(M, N, K, group_size=128, gran=GRAN_GROUP, layer=LAYER_OTHER) -> int:
    return lib().apex4_linear_host_scratch_bytes(M, N, K, group_size, gran, layer)


def w4a4_linear_host(x_host: torch.Tensor, qW, sW, y_host: torch.Tensor, N: int, group_size=128,
                     gran=GRAN_GROUP, layer=LAYER_OTHER, scratch: Optional[torch.Tensor] = None):
    """apex4_w4a4_linear_host: HOST X[M,K] fp16 -> HOST Y[M,N] fp16 through quantizer + GEMM, weights
    pre-packed on the device.  The copies run on the current stream; returns after enqueueing."""
    M, K = x_host.shape
    if scratch is None:
        scratch = torch.zeros(linear_host_scratch_bytes(M, N, K, group_size, gran, layer), dtype=torch.uint8,
                              device=qW.device)
    st = lib().apex4_w4a4_linear_host(x_host.data_ptr(), qW.data_ptr(), sW.data_ptr(), y_host.data_ptr(),
                                      M, N, K, group_size, gran, layer, OUT_F16, scratch.data_ptr(),
                                      scratch.numel(), _stream())
    _check(st, "apex4_w4a4_linear_host")
    return scratch


def measure_rho() -> dict:
    out = (ctypes.c_double * 8)()
    _check(lib().apex4_measure_rho(out, _stream()), "apex4_measure_rho")
    keys = ("int8_tops", "fp32_tflops", "i2f_gops", "rho", "tmem_ld_gbs", "sm_clock_mhz",
            "int8_mac_per_clk_sm", "tmem_ld_bytes_per_clk_sm")
    return dict(zip(keys, [float(v) for v in out]))


def measure_epilogue_pipes() -> dict:
    """apex4_measure_epilogue_pipes: clocks per 16 accumulator columns (TMEM warp) / per 32 FFMA2 (FFMA2 warp) with
    tcgen05.ld, tcgen05.st and FFMA2 streams alone and together."""
    out = (ctypes.c_double * 16)()
    _check(lib().apex4_measure_epilogue_pipes(out, _stream()), "apex4_measure_epilogue_pipes")
    names = {1: "ld", 2: "st", 3: "ld+st", 4: "ffma2", 5: "ld|ffma2", 6: "st|ffma2", 7: "ld+st|ffma2"}
    return {names[m]: {"tmem_clk_per_16_columns": float(out[2 * m]), "ffma2_clk_per_32": float(out[2 * m + 1])} for m in range(1, 8)}


def measure_epilogue_stream() -> dict:
    """apex4_measure_epilogue_stream: clocks per 192-column group of the pair kernel's epilogue stream in isolation."""
    out = (ctypes.c_double * 8)()
    _check(lib().apex4_measure_epilogue_stream(out, _stream()), "apex4_measure_epilogue_stream")
    keys = ("ld", "ld+st", "ld+fma", "ld+st+fma", "ld+lds+fma", "ld+st+lds+fma", "16x256b: ld", "16x256b: ld+st+lds+fma")
    return dict(zip(keys, [float(v) for v in out]))


def e4m3_exactness(K: int, pattern: int, encoding: int, seed: int = 0) -> dict:
    """apex4_e4m3_exactness: kind::f8f6f4 (E4M3 operands, FP32 accumulate) against kind::i8 on the same INT4 codes."""
    out = (ctypes.c_double * 5)()
    _check(lib().apex4_e4m3_exactness(K, pattern, encoding, seed, out, _stream()), "apex4_e4m3_exactness")
    keys = ("mismatches", "max_abs_diff", "max_abs_sum", "compared", "int8_vs_closed_form_mismatches")
    return dict(zip(keys, [float(v) for v in out]))


def debug_get_dispatch(M, N, K, group_size=128, gran=GRAN_GROUP, layer=LAYER_OTHER,
                       opts: Optional[DebugOpts] = None) -> Tuple[int, int, int, int, int]:
    """-> (kernel (0 decode, 1 pair), token-tile width, stream-K flag, CTAs / CTA pairs, k units per tile)"""
    out = (ctypes.c_int * 5)()
    _check(lib().apex4_debug_get_dispatch(M, N, K, group_size, gran, layer, _opts_ref(opts), out),
           "apex4_debug_get_dispatch")
    return tuple(int(v) for v in out)
