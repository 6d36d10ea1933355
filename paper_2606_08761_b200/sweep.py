"""Shape sweeps behind `bench.py --sweep`: BASELINE.json config 2 (N = K = 8192, g = 128,
M from decode to prefill), config 3 (granularities at M = 4096, incl. g = 256 / 512 / 1024 and the Fig. 11 g128 / per-channel
ratio over M), config 4 (Llama-2-70B linears at
M = 1, 16, 256, 4096) and whole-block times of Llama-2-7B / Qwen2.5-7B under the granularity
policies.  Per shape: GEMM time, effective TOPS (2MNK/t), the fraction of
the roofline that binds (INT8 tensor peak for M >= 256, HBM copy bandwidth below), and the speed-up
over cuBLAS FP16 (`torch.matmul`) on the same (M, N, K).

Timing protocol: every shape is captured in a CUDA graph of 20 launches that rotate through operand
sets whose total size exceeds L2 (so weights come from HBM), replayed 10 times, median reported;
shapes run in order of increasing work with an idle gap before each (see run_sweeps);
CUDA events on the launching stream.  Operands are random packed codes / scales of the right
layouts (timing does not depend on the values); parity is the business of tests/.
"""
from __future__ import annotations

import time

import torch

from . import apex4

L2_BYTES = 126e6
GRAPH_LAUNCHES = 20


def _graph_time_us(fn, nsets: int) -> float:
    for i in range(max(nsets, 3)):
        fn(i % nsets)
    torch.cuda.synchronize()
    gr = torch.cuda.CUDAGraph()
    with torch.cuda.graph(gr):
        for i in range(GRAPH_LAUNCHES):
            fn(i % nsets)
    ts = []
    for _ in range(10):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        gr.replay()
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1) / GRAPH_LAUNCHES * 1e3)
    ts.sort()
    return ts[len(ts) // 2]


def gemm_bytes(M, N, K, g):
    """Algorithmic bytes of one GEMM: packed codes, FP16 scales, FP16 output."""
    G = K // g
    return N * K / 2 + 2 * N * G + M * K / 2 + 2 * M * G + 2 * M * N


def time_shape(M, N, K, g, dev, cublas=True, with_quant=False):
    """with_quant: also time quantize_act + GEMM captured together (what a W4A4 linear costs next to an FP16
    GEMM, which needs no online quantizer) -> "us_with_quant"."""
    per_set = N * K / 2 + M * K / 2
    nsets = int(max(1, min(8, 2 * L2_BYTES // per_set + 1)))
    sets = []
    for _ in range(nsets):
        qA = torch.randint(0, 256, (apex4.packed_bytes(M, K),), dtype=torch.uint8, device=dev)
        qW = torch.randint(0, 256, (apex4.packed_bytes(N, K),), dtype=torch.uint8, device=dev)
        sA = (torch.rand(apex4.scale_elems(M, K, g), device=dev) * 0.1 + 0.01).half()
        sW = (torch.rand(apex4.scale_elems(N, K, g), device=dev) * 0.01 + 0.001).half()
        sets.append((qA, sA, qW, sW))
    Y = torch.empty((M, N), dtype=torch.float16, device=dev)
    ws = apex4.make_workspace(M, N, K, g, device=dev)

    def run(i):
        qA, sA, qW, sW = sets[i]
        apex4.w4a4_gemm(qA, sA, qW, sW, M, N, K, g, out=Y, workspace=ws)

    us = _graph_time_us(run, nsets)
    out = {"M": M, "N": N, "K": K, "g": g, "us": round(us, 2),
           "tops": round(2.0 * M * N * K / us * 1e-6, 1),
           "gbs": round(gemm_bytes(M, N, K, g) / us * 1e-3, 1),
           "kernel": ("gemv", "pair")[apex4.debug_get_dispatch(M, N, K, g)[0]]}
    if with_quant:
        nx = int(max(2, min(8, 2 * L2_BYTES // (2 * M * K) + 1)))
        xs = [torch.randn(M, K, device=dev, dtype=torch.float16) for _ in range(nx)]
        qa0, sa0 = sets[0][0], sets[0][1]

        def run_q(i):
            apex4.quantize_act(xs[i % nx], g, q=qa0, s=sa0)
            apex4.w4a4_gemm(qa0, sa0, sets[i % nsets][2], sets[i % nsets][3], M, N, K, g, out=Y, workspace=ws)

        out["us_with_quant"] = round(_graph_time_us(run_q, max(nx, nsets)), 2)
        del xs
    del sets
    if cublas:
        nb = int(max(1, min(4, 2 * L2_BYTES // (2 * N * K) + 1)))
        a = torch.randn(M, K, device=dev, dtype=torch.float16)
        bs = [torch.randn(N, K, device=dev, dtype=torch.float16) for _ in range(nb)]
        c = torch.empty((M, N), device=dev, dtype=torch.float16)
        cu = _graph_time_us(lambda i: torch.matmul(a, bs[i].t(), out=c), nb)
        out["cublas_fp16_us"] = round(cu, 2)
        out["speedup_vs_cublas_fp16"] = round(cu / us, 2)                      # GEMM alone
        if with_quant:
            out["speedup_vs_cublas_fp16_with_quant"] = round(cu / out["us_with_quant"], 2)
        del bs
    torch.cuda.empty_cache()
    return out


def time_quant(M, K, g, dev):
    """Activation quantizer (a1) alone, same protocol; rotating inputs larger than L2."""
    nsets = int(max(2, min(8, 2 * L2_BYTES // (2 * M * K) + 1)))
    xs = [torch.randn(M, K, device=dev, dtype=torch.float16) for _ in range(nsets)]
    q = torch.empty(apex4.packed_bytes(M, K), dtype=torch.uint8, device=dev)
    s = torch.empty(apex4.scale_elems(M, K, g), dtype=torch.float16, device=dev)
    us = _graph_time_us(lambda i: apex4.quantize_act(xs[i], g, q=q, s=s), nsets)
    del xs
    torch.cuda.empty_cache()
    return us


# One transformer block's linears, (hidden, kv width, intermediate); shapes from the public model configs,
# weights not needed (PAPER.md:343 evaluates both models end to end).
BLOCK_MODELS = {"llama-2-7b": (4096, 4096, 11008), "qwen2.5-7b": (3584, 512, 18944)}


def block_ops(h, kv, inter, policy):
    """-> (quantizer calls [(K, gran, layer)], GEMMs [(name, N, K, gran, layer)]) of one block under a policy.
    G_a = G_w: an activation is quantized once per distinct granularity its consumers
    use, so the paper's mix (V and DOWN fine, the rest per-channel, R11) splits V off the fused QKV GEMM
    and quantizes the block input twice."""
    A = apex4
    if policy == "uniform_g128":
        gr = A.GRAN_GROUP
        return ([(h, gr, A.LAYER_QKV), (h, gr, A.LAYER_O), (h, gr, A.LAYER_GATE_UP), (inter, gr, A.LAYER_DOWN)],
                [("qkv", h + 2 * kv, h, gr, A.LAYER_QKV), ("o", h, h, gr, A.LAYER_O),
                 ("gate_up", 2 * inter, h, gr, A.LAYER_GATE_UP), ("down", h, inter, gr, A.LAYER_DOWN)])
    if policy == "uniform_channel":
        gr = A.GRAN_CHANNEL
        return ([(h, gr, A.LAYER_QKV), (h, gr, A.LAYER_O), (h, gr, A.LAYER_GATE_UP), (inter, gr, A.LAYER_DOWN)],
                [("qkv", h + 2 * kv, h, gr, A.LAYER_QKV), ("o", h, h, gr, A.LAYER_O),
                 ("gate_up", 2 * inter, h, gr, A.LAYER_GATE_UP), ("down", h, inter, gr, A.LAYER_DOWN)])
    gr = A.GRAN_MIXED if policy == "mixed_fine32" else A.GRAN_MIXED_G128
    return ([(h, gr, A.LAYER_Q), (h, gr, A.LAYER_V), (h, gr, A.LAYER_O), (h, gr, A.LAYER_GATE_UP),
             (inter, gr, A.LAYER_DOWN)],
            [("qk", h + kv, h, gr, A.LAYER_Q), ("v", kv, h, gr, A.LAYER_V), ("o", h, h, gr, A.LAYER_O),
             ("gate_up", 2 * inter, h, gr, A.LAYER_GATE_UP), ("down", h, inter, gr, A.LAYER_DOWN)])


def run_block_policies(dev, M=2048):
    """Whole-block time (every quantizer call + every GEMM of one transformer block, each timed with the
    sweep protocol and summed) per model and granularity policy; g comes from apex4_resolve_group_size."""
    res = []
    cache = {}
    for model, (h, kv, inter) in BLOCK_MODELS.items():
        for policy in ("uniform_g128", "mixed_fine32", "mixed_fine128", "uniform_channel"):
            quants, gemms = block_ops(h, kv, inter, policy)
            ops, total, work = [], 0.0, 0.0
            for (K, gran, layer) in quants:
                g = apex4.resolve_group_size(K, 128, gran, layer)
                key = ("q", M, K, g)
                if key not in cache:
                    time.sleep(0.2)
                    cache[key] = time_quant(M, K, g, dev)
                ops.append({"op": "quantize", "K": K, "g": g, "us": round(cache[key], 2)})
                total += cache[key]
            for (name, N, K, gran, layer) in gemms:
                g = apex4.resolve_group_size(K, 128, gran, layer)
                key = ("g", M, N, K, g)
                if key not in cache:
                    time.sleep(0.2)
                    cache[key] = time_shape(M, N, K, g, dev, cublas=False)["us"]
                ops.append({"op": name, "N": N, "K": K, "g": g, "us": cache[key]})
                total += cache[key]
                work += 2.0 * M * N * K
            res.append({"model": model, "policy": policy, "M": M, "block_us": round(total, 1),
                        "tops": round(work / total * 1e-6, 1), "ops": ops})
    return res


def run_sweeps(dev, peaks=None):
    """-> dict of lists; `peaks` = {"hbm": GB/s, "int8": TOP/s} adds the roofline fractions."""
    res = {"protocol": f"CUDA graph of {GRAPH_LAUNCHES} launches rotating operand sets larger than L2, median of 10 replays"}
    # All shapes are timed in order of increasing work, each after a short idle gap: right after seconds
    # of tensor-bound work the part is still under its power cap, and a shape timed then ran up to 45 %
    # slower (M = 16, N = K = 8192: 16.2 vs 11.2 us; M = 256, N = 8192, K = 28672: 335 vs 180 us).
    shapes70 = ((10240, 8192), (8192, 8192), (57344, 8192), (8192, 28672))
    jobs = [("cfg2", M, 8192, 8192, 128, True) for M in (1, 4, 16, 64, 256, 1024, 4096, 8192)]
    jobs += [("cfg3", 4096, 8192, 8192, g, False) for g in (32, 64, 128, 256, 512, 1024, 8192)]
    # Fig. 11: g = 128 against per-channel over M at N = K = 8192
    jobs += [("fig11", M, 8192, 8192, g, False) for M in (1024, 2048, 4096, 8192, 16384, 32768) for g in (128, 8192)]
    jobs += [("cfg4", M, N, K, 128, True) for M in (1, 16, 256, 4096) for (N, K) in shapes70]
    done = {}
    for i in sorted(range(len(jobs)), key=lambda i: jobs[i][1] * jobs[i][2] * jobs[i][3]):
        tag, M, N, K, g, cub = jobs[i]
        torch.cuda.synchronize()
        time.sleep(0.5)
        done[i] = time_shape(M, N, K, g, dev, cublas=cub)
    cfg2 = [done[i] for i in range(len(jobs)) if jobs[i][0] == "cfg2"]
    cfg3 = [done[i] for i in range(len(jobs)) if jobs[i][0] == "cfg3"]
    cfg4 = [done[i] for i in range(len(jobs)) if jobs[i][0] == "cfg4"]
    if peaks:
        for r in cfg2 + cfg3 + cfg4:
            if r["M"] >= 256:
                r["bound"] = "tensor"
                r["frac_of_int8_peak"] = round(r["tops"] / peaks["int8"], 3)
            else:
                r["bound"] = "hbm"
                r["frac_of_hbm_peak"] = round(r["gbs"] / peaks["hbm"], 3)
    res["config2_square_sweep"] = cfg2
    res["config3_granularity"] = cfg3
    t = {r["g"]: r["us"] for r in cfg3}
    res["config3_mixed"] = {   # R11: 2 fine layers (V, DOWN) + 5 per-channel layers per block, mapped on this shape
        "paper_mix_fine32_us": round((2 * t[32] + 5 * t[8192]) / 7, 2),
        "baseline_mix_fine128_us": round((2 * t[128] + 5 * t[8192]) / 7, 2),
        "uniform_g128_us": t[128]}
    res["config4_llama70b"] = cfg4
    res["block_policies"] = run_block_policies(dev, 2048) + run_block_policies(dev, 16)   # prefill and decode
    f11 = {(jobs[i][1], jobs[i][4]): done[i] for i in range(len(jobs)) if jobs[i][0] == "fig11"}
    res["fig11_g128_over_channel"] = [
        {"M": M, "g128_us": f11[(M, 128)]["us"], "channel_us": f11[(M, 8192)]["us"],
         "g128_tops": f11[(M, 128)]["tops"], "channel_tops": f11[(M, 8192)]["tops"],
         "ratio": round(f11[(M, 128)]["us"] / f11[(M, 8192)]["us"], 3)}
        for M in sorted({k[0] for k in f11})]
    return res


def render_markdown(d: dict, title: str) -> str:
    """bench.py --sweep JSON line (dict) -> the markdown tables committed under profiles/."""
    L = [f"# {title}", ""]
    r = d["roofline"]
    L.append(f"Headline (config 1, M=2048 Llama-2-7B linears, step = quantize + GEMM per layer): **{d['value']:.1f} TOPS**, "
             f"{d['ms_per_step']:.3f} ms/step; GEMM launches alone {r['achieved']:.1f} TOP/s = {r['frac']:.3f} of {r['peak']:.0f} TOP/s "
             f"({r['peak_source']}), {r['frac_of_spec_4500_tops']:.3f} of the 4.5 POPS datasheet figure; e2e {d['e2e']['value']:.1f} TOPS; "
             f"clocks {d['clocks']['sm_mhz']} MHz of {d['clocks']['sm_max_mhz']}, reasons {d['clocks']['reasons']}; "
             f"output check {d.get('check')}; cpu_baseline {d.get('cpu_baseline', {}).get('value', float('nan')):.4f} TOPS on "
             f"{d.get('cpu_baseline', {}).get('cores')} cores.")
    L.append("")
    L.append("Per layer: " + "; ".join(f"{k}: GEMM {v['gemm_ms'] * 1e3:.0f} us = {v['gemm_tops']:.0f} TOPS, quantizer {v['quant_ms'] * 1e3:.1f} us = "
                                       f"{v['quant_gbs']:.0f} GB/s" for k, v in r["per_layer"].items()))
    L.append("")
    if "targets" in r:
        L.append("Target points of BASELINE.json (" + r.get("targets_protocol", "") + "):")
        L.append("")
        L.append("| M | N | K | g | kernel | GEMM us | quant+GEMM us | achieved | bound | frac of measured peak | frac of datasheet | cuBLAS FP16 us | speed-up (GEMM) | speed-up (quant+GEMM) |")
        L.append("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
        for t in r["targets"]:
            L.append(f"| {t['M']} | {t['N']} | {t['K']} | {t['g']} | {t['kernel']} | {t['us']} | {t['us_with_quant']} | {t['achieved']:.1f} {t['unit']} | {t['bound']} | "
                     f"{t['frac']:.3f} | {t['frac_of_spec']:.3f} | {t['cublas_fp16_us']} | {t['speedup_vs_cublas_fp16']} | {t['speedup_vs_cublas_fp16_with_quant']} |")
        L.append("")
        if "rho" in r:
            rh = r["rho"]
            L.append(f"rho microbenchmark in the same run: INT8 {rh['int8_tops']:.0f} TOPS ({rh['int8_mac_per_clk_sm']:.0f} MAC/clk/SM), FP32 {rh['fp32_tflops']:.1f} TFLOP/s, "
                     f"rho = {rh['rho']:.1f}, TMEM read {rh['tmem_ld_bytes_per_clk_sm']:.0f} B/clk/SM, SM clock {rh['sm_clock_mhz']:.0f} MHz.")
            L.append("")
    sw = d.get("sweep")
    if sw:
        L.append("Sweeps: " + sw["protocol"])
        L.append("")
        L.append("| config | M | N | K | g | kernel | us | eff. TOPS | GB/s (algorithmic) | bound | frac of peak | cuBLAS FP16 us | speed-up |")
        L.append("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
        for tag, key in (("2", "config2_square_sweep"), ("3", "config3_granularity"), ("4", "config4_llama70b")):
            for x in sw[key]:
                fr = x.get("frac_of_int8_peak", x.get("frac_of_hbm_peak", ""))
                L.append(f"| {tag} | {x['M']} | {x['N']} | {x['K']} | {x['g']} | {x['kernel']} | {x['us']} | {x['tops']} | {x['gbs']} | {x.get('bound', '')} | {fr} | "
                         f"{x.get('cublas_fp16_us', '')} | {x.get('speedup_vs_cublas_fp16', '')} |")
        L.append("")
        m = sw["config3_mixed"]
        L.append(f"Config 3 mixed granularity (R11, two fine + five per-channel linears per block mapped onto the 4096 x 8192 x 8192 shape): paper mix (fine = 32) "
                 f"{m['paper_mix_fine32_us']} us, BASELINE wording (fine = 128) {m['baseline_mix_fine128_us']} us, uniform g128 {m['uniform_g128_us']} us.")
        L.append("")
        L.append("Fig. 11 (PAPER.md:361-363), N = K = 8192, time of g = 128 over per-channel: " +
                 "; ".join(f"M={x['M']}: {x['g128_us']} / {x['channel_us']} us = {x['ratio']}" for x in sw["fig11_g128_over_channel"]) + ".")
        L.append("")
        L.append("Whole transformer block (every quantizer call + GEMM; G_a = G_w so the paper's mix quantizes the block input twice and splits V off QKV):")
        L.append("")
        L.append("| model | M | policy | block us | eff. TOPS | ops (us) |")
        L.append("|---|---|---|---|---|---|")
        for b in sw["block_policies"]:
            ops = ", ".join(f"{o['op']}@g{o['g']} {o['us']}" for o in b["ops"])
            L.append(f"| {b['model']} | {b['M']} | {b['policy']} | {b['block_us']} | {b['tops']} | {ops} |")
        L.append("")
    return "\n".join(L) + "\n"


if __name__ == "__main__":
    # python -m paper_2606_08761_b200.sweep <bench.json> "<title>"  ->  markdown on stdout
    import json
    import sys
    line = [l for l in open(sys.argv[1]) if l.startswith("{")][-1]
    sys.stdout.write(render_markdown(json.loads(line), sys.argv[2] if len(sys.argv) > 2 else "bench.py --sweep"))
