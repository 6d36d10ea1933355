#!/usr/bin/env python
"""bench.py -- measures the APEX4 W4A4 hot path on B200 (contract: see DESIGN.md "Measurement").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--sweep]

A "step" is one pass of the whole hot path over one batch of BASELINE.json config 1 (the four
Llama-2-7B linear shapes at prefill M=2048, g=128): for each layer the online activation quantizer
(apex4_quantize_act) and the group-dequant GEMM (apex4_w4a4_gemm); weights are packed offline.
`value` = effective TOPS = sum(2 M N K) / time with inputs resident in HBM; `e2e` = the same metric
through apex4_w4a4_linear_host with pinned HOST activations/outputs (copies inside the timed region; the four layers of a
step go out on a stream each so that one layer's H2D copy overlaps another's D2H copy; measured 150 -> 215 TOPS).

BASELINE.json's metric is quoted "vs M" with targets at M = N = K = 8192 (tensor roofline) and M <= 16
(HBM roofline): those points are timed in the same run (rank 0, N = 1), each in a CUDA graph of launches
that rotate through operand sets larger than L2, with cuBLAS FP16 on the same shape beside them, and
reported in `roofline.targets`.  Denominators: a timed region shorter than 1 s at full clock is a burst
and is divided by the burst peak (2 x MEASURED_PEAKS bf16_tflops for the INT8 pipe, nominal 4.5:2.25),
a longer one by the sustained figure; the 4.5 POPS / 8 TB/s datasheet fractions are given alongside.
After the timed region one layer's output is checked against the CPU oracle on sampled rows (`check`).
One JSON line on stdout (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "W4A4-g128 GEMM effective TOPS (2MNK/time) over the Llama-2-7B linear shapes at M=2048"
UNIT = "TOPS"
G = 128
M_PREFILL = 2048


def layers():
    from paper_2606_08761_b200 import inputs
    return [(name, M_PREFILL, n, k) for name, (n, k) in inputs.LLAMA2_7B_SHAPES.items()]


def total_ops(ls):
    return sum(2.0 * m * n * k for _, m, n, k in ls)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], bf16=d["bf16_tflops"], bf16_sus=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    src="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sus=1400.0, src="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region: the sampler is started
    before the warm-up (nvidia-smi takes a few hundred ms to come up), every row is stamped with the
    host clock when it is read, and stop(t0, t1) keeps the rows that fall inside the timed window."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0, period_ms=20):
        self.index, self.rows, self.proc, self.period_ms = index, [], None, period_ms

    def start(self, wait_s=5.0):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", str(self.period_ms)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
            return
        t_end = time.time() + wait_s
        while not self.rows and time.time() < t_end:
            time.sleep(0.01)

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t0=None, t1=None):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(2.5 * self.period_ms * 1e-3)
        self.proc.terminate()
        self.t.join(timeout=2)
        rows = [r for (ts, r) in self.rows if (t0 is None or ts >= t0) and (t1 is None or ts <= t1 + 2e-3 * self.period_ms)]
        window = "timed region"
        if not rows:                      # region shorter than one sampling period: nearest rows after its start
            rows = [r for (ts, r) in self.rows if t0 is None or ts >= t0][:3] or [r for (_, r) in self.rows[-3:]]
            window = "nearest samples (timed region shorter than the sampling period)"
        sm, mx, pw, reasons = [], None, [], set()
        for r in rows:
            try:
                sm.append(float(r[0])); mx = float(r[1]); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "window": window}


CPU_BASELINE_ROWS = 2048     # all token rows of every layer: about 15 s of oracle time on the GPU box (16 cores)


def oracle_sample(sample_rows, chunk=64):
    """The oracle as it stands on a bounded sample of the workload: the first `sample_rows` token rows
    of every config-1 layer (activation quantizer + full-width Eq. 8 against the whole weight), called on
    `chunk` rows at a time (its per-group INT sums of all rows at once would not fit in host memory)."""
    import threadpoolctl
    from oracle import apex4_oracle as O
    from paper_2606_08761_b200 import inputs
    ops, secs = 0.0, 0.0
    for i, (name, m, n, k) in enumerate(layers()):
        seed = inputs.config_seed(1, i)
        X = inputs.make_activations(sample_rows, k, seed, True)
        W = inputs.make_weights(n, k, seed)
        qW, sW = O.quantize(W, G)          # offline (a0): not timed, as on the GPU side
        t0 = time.perf_counter()
        for r0 in range(0, sample_rows, chunk):
            qA, sA = O.quantize(X[r0:r0 + chunk], G)
            Y = O.to_f16(O.dequant_gemm(qA, sA, qW, sW, G, want_T=False))
        secs += time.perf_counter() - t0
        ops += 2.0 * sample_rows * n * k
        del W, qW, sW, Y
    cores = max([p.get("num_threads", 1) for p in threadpoolctl.threadpool_info()] + [1])
    return ops / secs * 1e-12, secs, cores


def run_reference(args):
    """--impl reference: the CPU oracle (numpy, float64) on the same config/metric, bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    rows = 32
    for _ in range(args.warmup if args.warmup < 2 else 1):
        oracle_sample(8)
    vals, tot = [], 0.0
    cores = 1
    for _ in range(args.steps):
        v, s, cores = oracle_sample(rows)
        vals.append(v); tot += s
    v = float(np.mean(vals))
    sample = f"first {rows} of {M_PREFILL} token rows of each of the 4 layers, full N and K, numpy float64 oracle"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": tot / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[1]: Llama-2-7B linears, M=2048, g=128", "sample": sample},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


SPEC_INT8_TOPS = 4500.0      # B200 dense INT8 (datasheet)
SPEC_HBM_GBS = 8000.0        # HBM3e (datasheet)
TARGETS = [                  # (M, N, K, g, bound): the points BASELINE.json's targets are stated on
    (1, 8192, 8192, 128, "hbm"), (16, 8192, 8192, 128, "hbm"), (16, 57344, 8192, 128, "hbm"),
    (8192, 8192, 8192, 128, "tensor"),
]


def time_targets(dev, peaks):
    """The metric's own configuration (config 2 / config 4 points), sweep protocol: CUDA graph of 20 launches
    rotating operand sets larger than L2, median of 10 replays, increasing work, idle gap before each."""
    import torch
    from paper_2606_08761_b200 import sweep
    out = []
    for (M, N, K, g, bound) in TARGETS:
        torch.cuda.synchronize()
        time.sleep(0.5)
        r = sweep.time_shape(M, N, K, g, dev, cublas=True, with_quant=True)
        t = {"M": M, "N": N, "K": K, "g": g, "kernel": r["kernel"], "us": r["us"], "us_with_quant": r["us_with_quant"],
             "cublas_fp16_us": r["cublas_fp16_us"], "speedup_vs_cublas_fp16": r["speedup_vs_cublas_fp16"],
             "speedup_vs_cublas_fp16_with_quant": r["speedup_vs_cublas_fp16_with_quant"], "bound": bound}
        if bound == "tensor":
            t.update(achieved=r["tops"], unit="TOP/s", peak=2.0 * peaks["bf16"], frac=r["tops"] / (2.0 * peaks["bf16"]),
                     peak_kind="burst: 2 x measured bf16_tflops (graph of 20 launches, ~16 ms)",
                     frac_of_spec=r["tops"] / SPEC_INT8_TOPS)
        else:
            t.update(achieved=r["gbs"], unit="GB/s", peak=peaks["hbm"], frac=r["gbs"] / peaks["hbm"],
                     peak_kind="measured copy bandwidth", frac_of_spec=r["gbs"] / SPEC_HBM_GBS)
        out.append(t)
    return out


def check_one_layer(L, rows=12):
    """Cheap output check after the timed region: sampled rows of the O-proj layer against the CPU oracle
    (codes / scales of those rows bit-exact, outputs inside the R12 tolerance).  A stale workspace or a
    mis-dispatch would print a fine number otherwise."""
    import torch
    from oracle import apex4_oracle as O
    from paper_2606_08761_b200 import apex4, inputs
    l = [x for x in L if x["name"] == "o"][0]
    m, n, k = l["m"], l["n"], l["k"]
    seed = inputs.config_seed(1, 1)
    X = l["Xh"].numpy()
    W = inputs.make_weights(n, k, seed)
    cand = inputs.sample_rows(m, 99)
    sel = cand[:: max(1, len(cand) // rows)][:rows]      # tile edges and random rows, spread over M
    qa, sa = O.quantize(X[sel], G)
    qw, sw = O.quantize(W, G)
    Y64, T = O.dequant_gemm(qa, sa, qw, sw, G)
    tol = O.output_tolerance(Y64, T, k // G, True)
    Y = l["Y"].cpu().numpy()[sel].astype("float64")
    codes = apex4.unpack_codes(l["qA"], m, k, apex4.OPERAND_ACT).cpu().numpy()[sel]
    ratio = float((abs(Y - Y64) / tol).max())
    ok = bool(ratio <= 1.0 and (codes == qa).all())
    return {"layer": "o", "rows": int(len(sel)), "max_err_over_tolerance": ratio, "codes_bit_exact": bool((codes == qa).all()), "ok": ok}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="apex4")
    ap.add_argument("--sweep", action="store_true",
                    help="also time the config-2 M sweep, config-3 granularities and config-4 decode shapes + cuBLAS FP16")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-targets", action="store_true", help="skip the roofline.targets points (8192^3, M <= 16 + cuBLAS FP16)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl != "reference":
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2606_08761_b200 import apex4, inputs
    from paper_2606_08761_b200 import build as B
    B.build()
    apex4.lib()                       # fails loudly when the CUDA library is missing
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    ls = layers()

    # ---- resident operands (synthetic, seeded)
    L = []
    for i, (name, m, n, k) in enumerate(ls):
        seed = inputs.config_seed(1, i)
        Xh = torch.from_numpy(inputs.make_activations(m, k, seed, True)).pin_memory()
        Wd = torch.from_numpy(inputs.make_weights(n, k, seed)).to(dev)
        qW, sW, _ = apex4.pack_weights(Wd, G)
        del Wd
        Xd = Xh.to(dev)
        qA = torch.empty(apex4.packed_bytes(m, k), dtype=torch.uint8, device=dev)
        sA = torch.empty(apex4.scale_elems(m, k, G), dtype=torch.float16, device=dev)
        Y = torch.empty((m, n), dtype=torch.float16, device=dev)
        ws = apex4.make_workspace(m, n, k, G, device=dev)
        Yh = torch.empty((m, n), dtype=torch.float16).pin_memory()
        scratch = torch.zeros(apex4.linear_host_scratch_bytes(m, n, k, G), dtype=torch.uint8, device=dev)
        L.append(dict(name=name, m=m, n=n, k=k, Xh=Xh, Xd=Xd, qW=qW, sW=sW, qA=qA, sA=sA, Y=Y, ws=ws, Yh=Yh,
                      scratch=scratch))
    torch.cuda.synchronize()

    def step():
        for l in L:
            apex4.quantize_act(l["Xd"], G, q=l["qA"], s=l["sA"])
            apex4.w4a4_gemm(l["qA"], l["sA"], l["qW"], l["sW"], l["m"], l["n"], l["k"], G, out=l["Y"],
                            workspace=l["ws"])

    # e2e: the layers of a step are independent calls with their own scratch, so each goes out on a stream of its own: the H2D copy
    # of one layer overlaps the D2H copy of another (PCIe is full duplex) and both overlap the kernels; every step joins
    # both streams back into the timed stream.
    side = [torch.cuda.Stream(device=dev) for _ in L]

    def step_e2e():
        cur = torch.cuda.current_stream()
        for sd in side:
            sd.wait_stream(cur)
        for i, l in enumerate(L):
            with torch.cuda.stream(side[i % len(side)]):
                apex4.w4a4_linear_host(l["Xh"], l["qW"], l["sW"], l["Yh"], l["n"], G, scratch=l["scratch"])
        for sd in side:
            cur.wait_stream(sd)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([ms], device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(args.warmup):
        step()
    t0 = time.time()
    ms = timed(step, args.steps)
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    ops = total_ops(ls)
    value = world * ops * args.steps / (ms * 1e-3) * 1e-12

    # ---- e2e: HOST buffers, copies inside the timed region
    for _ in range(3):
        step_e2e()
    e2e_steps = max(3, args.steps // 2)
    ms_e2e = timed(step_e2e, e2e_steps)
    e2e_value = world * ops * e2e_steps / (ms_e2e * 1e-3) * 1e-12
    h2d = sum(2 * l["m"] * l["k"] for l in L)
    d2h = sum(2 * l["m"] * l["n"] for l in L)

    # ---- dominant kernel (the GEMM) timed launch by launch inside the same kind of step
    gemm_ms, quant_ms = [0.0] * len(L), [0.0] * len(L)
    ksteps = max(3, args.steps // 2)
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in L]
    for _ in range(ksteps):
        for l, ev in zip(L, evs):
            ev[0].record()
            apex4.quantize_act(l["Xd"], G, q=l["qA"], s=l["sA"])
            ev[1].record()
            apex4.w4a4_gemm(l["qA"], l["sA"], l["qW"], l["sW"], l["m"], l["n"], l["k"], G, out=l["Y"], workspace=l["ws"])
            ev[2].record()
        torch.cuda.synchronize()
        for i, ev in enumerate(evs):
            quant_ms[i] += ev[0].elapsed_time(ev[1])
            gemm_ms[i] += ev[1].elapsed_time(ev[2])
    gemm_ms = [t / ksteps for t in gemm_ms]
    quant_ms = [t / ksteps for t in quant_ms]
    peaks = measured_peaks()
    # Denominator: the timed region is a burst unless it ran for >= 1 s (then the part is under its power cap
    # and the sustained cuBLAS figure is the like-for-like peak); kind::i8 nominal = 2 x bf16 (4.5 vs 2.25 PFLOP/s).
    sustained = (ms * 1e-3) >= 1.0
    bf16_peak = peaks["bf16_sus"] if sustained else peaks["bf16"]
    int8_peak = 2.0 * bf16_peak
    gemm_tops = ops / (sum(gemm_ms) * 1e-3) * 1e-12
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp):
        traffic = json.load(open(tp)).get("gemm_dram_bytes_per_launch")
    roofline = {
        "kernel": "w4a4_gemm_pair_kernel (tcgen05 cta_group::2 kind::i8, 256x192 tiles)", "bound": "tensor", "achieved": gemm_tops,
        "peak": int8_peak, "unit": "TOP/s", "frac": gemm_tops / int8_peak, "traffic": traffic,
        "traffic_source": "profiles/traffic.json: dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu capture, "
                          "mean over the four layers; not measured in this run",
        "peak_source": f"2 x {bf16_peak} {'sustained' if sustained else 'burst'} bf16 TFLOP/s of {peaks['src']} MEASURED_PEAKS.json "
                       f"(nominal int8:bf16 ratio 4.5:2.25); timed region {ms * 1e-3:.3f} s",
        "frac_of_spec_4500_tops": gemm_tops / SPEC_INT8_TOPS,
        "per_layer": {l["name"]: {"gemm_ms": g_, "quant_ms": q_, "gemm_tops": 2.0 * l["m"] * l["n"] * l["k"] / (g_ * 1e-3) * 1e-12,
                                  "quant_gbs": (2.5 * l["m"] * l["k"] + 2.0 * l["m"] * l["k"] / G) / (q_ * 1e-3) * 1e-9}
                      for l, g_, q_ in zip(L, gemm_ms, quant_ms)},
    }
    check = check_one_layer(L) if rank == 0 else None
    if rank == 0 and world == 1 and not args.no_targets:
        torch.cuda.synchronize()
        time.sleep(1.5)                # let the part leave its power-capped state: rho is a burst figure
        rho = apex4.measure_rho()      # B200's own rho: INT8 tensor ops vs FP32 FMA (Table 1)
        roofline["targets"] = time_targets(dev, peaks)
        roofline["targets_protocol"] = ("CUDA graph of 20 launches rotating operand sets larger than L2, median of 10 replays, CUDA events; "
                                        "us = GEMM alone, us_with_quant = apex4_quantize_act + GEMM; cuBLAS FP16 = torch.matmul, same protocol")
        roofline["rho"] = rho
        for t in roofline["targets"]:
            if t["bound"] == "tensor":
                t["frac_of_measured_int8_burst"] = t["achieved"] / rho["int8_tops"]

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int8 tensor-core MMA (INT4 codes widened), int32 group sums, f32 dequant, f16 out",
        "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[1]: Llama-2-7B linears (QKV 12288x4096, O 4096x4096, "
                               "gate+up 22016x4096, down 4096x11008) at prefill M=2048, g=128; step = quantize_act + "
                               "w4a4_gemm per layer, weights pre-packed",
                   "l2": "inputs larger than L2 (about 0.4 GB touched per step vs 126 MB L2)",
                   "parallelism": f"replicas x{world} (no data-path collective)"},
        "clocks": clocks, "gpu_launches": 2 * len(L) * args.steps,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": ms_e2e / e2e_steps},
        "roofline": roofline, "check": check,
    }
    if clocks is not None and clocks.get("samples", 0) < 10:
        out["clocks"]["note"] = "fewer than 10 nvidia-smi samples inside the timed region: burst measurement"
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, secs, cores = oracle_sample(CPU_BASELINE_ROWS)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": f"first {CPU_BASELINE_ROWS} of {M_PREFILL} token rows of each layer, full N and K "
                                         f"({secs:.1f} s of numpy float64 oracle)"}
    if args.sweep and rank == 0:
        from paper_2606_08761_b200 import sweep
        out["sweep"] = sweep.run_sweeps(dev, {"hbm": peaks["hbm"], "int8": 2.0 * peaks["bf16"]})
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
