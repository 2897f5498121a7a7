#!/usr/bin/env python
"""bench.py — fused rANS-decode GEMM throughput on BASELINE.json config 2 (Qwen-14B-shaped bf16 layer).

One "step" = one pass of the hot path over the layer: anslin_gemm (table residency, compressed tile
fetch, warp-cooperative rANS decode, operand store, X TMA, tcgen05 MMA, epilogue) for the seven
projections q,k,v,o,gate,up,down at batch M (default 75, the paper's Qwen-14B max batch, P:l.378).
Prints ONE JSON line (contract in the task statement).  `--impl reference` times the CPU oracle.
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
sys.path.insert(0, ROOT)

METRIC = "fused_ans_decode_gemm_tflops"
UNIT = "TFLOP/s"
WORKLOAD = "config2: Qwen-14B-shaped decoder layer, bf16, q/k/v/o/gate/up/down, synthetic N(0,0.02^2)+jitter+outliers"


def layer_weights(seed0: int = 1):
    from paper_2606_15789_b200 import inputs
    out = []
    for i, (name, n, k) in enumerate(inputs.QWEN14B_LAYER):
        w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=seed0 + i, jitter=True))
        out.append((name, n, k, w))
    return out


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("bf16_tflops", 1590.0)), "measured"
    return 6650.0, 1590.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
            "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q, "--format=csv,noheader,nounits",
                                          "-lms", "25"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def wait_first(self, timeout=5.0):
        t0 = time.time()
        while self.proc is not None and not self.rows and time.time() - t0 < timeout:
            time.sleep(0.01)

    def mark(self):
        return len(self.rows)

    def stop(self, lo=0, hi=None):
        """Summary over the samples taken between mark() lo and mark() hi (the timed region)."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        rows = self.rows[max(lo - 1, 0):(hi + 1 if hi is not None else None)]
        sm = [float(r[0]) for r in rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm)}


def cpu_oracle_leg(layer, containers, m: int, names=("q", "k", "down")):
    """The oracle as it stands, timed on the host cores over a bounded sample of the workload:
    full container decode (plain C rANS, single thread) + float64 GEMM of the named projections."""
    from oracle import container as oc, gemm as og
    from paper_2606_15789_b200 import inputs
    try:
        from threadpoolctl import threadpool_info
        blas = max([i.get("num_threads", 1) for i in threadpool_info()] or [1])
    except Exception:
        blas = 1
    flops, t0 = 0.0, time.perf_counter()
    for (name, n, k, w), buf in zip(layer, containers):
        if name not in names:
            continue
        _, w_dec, _ = oc.decode(buf)
        x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=7))
        og.gemm_bf16(x, w_dec)
        flops += 2.0 * m * n * k
    dt = time.perf_counter() - t0
    return {"value": flops / dt / 1e12, "unit": UNIT, "cores": int(blas), "kind": "oracle", "seconds": round(dt, 2),
            "sample": "projections %s of the layer at M=%d: oracle container decode (1 thread) + float64 GEMM (%d BLAS threads)"
                      % ("/".join(names), m, blas)}


def run_reference(args):
    from paper_2606_15789_b200 import binding as B, build as libbuild
    libbuild.build()
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    layer = [t for t in layer_weights() if t[0] in ("k",)]       # bounded sample: the k projection (1024x5120)
    containers = [B.anslin_encode_host(B.FMT_BF16, w, n, k, tile_k=64, flags=1)[0] for (_, n, k, w) in layer]
    for _ in range(args.warmup):
        cpu_oracle_leg(layer, containers, args.m, names=("k",))
    t0 = time.perf_counter()
    vals = [cpu_oracle_leg(layer, containers, args.m, names=("k",)) for _ in range(args.steps)]
    dt = time.perf_counter() - t0
    flops = args.steps * 2.0 * args.m * 1024 * 5120
    v = flops / dt / 1e12
    cb = dict(vals[-1]); cb["value"] = v
    cb["sample"] = "each step = oracle decode + float64 GEMM of the k projection (1024x5120) at M=%d" % args.m
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                      "config": {"workload": WORKLOAD, "batch_m": args.m}, "cpu_baseline": cb,
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


# ALU-pipe warp instructions per decoded bf16 symbol in fused_gemm_kernel's hot loop (cuobjdump -sass):
# table slot 1 (LOP3), entry fields 3 (SHF, LOP3, SHF), state shift 1 (SHF), renormalisation test 1 (ISETP),
# symbol + raw byte -> bf16 4 per weight pair... = 3 (PRMT 1.5, SHF 1, LOP3 0.5), per-unit bookkeeping ~1.
ALU_INSTR_PER_SYMBOL = 10.0


def run_other_config(args):
    """--workload c3 | c4 | c5: the other BASELINE.json configs (parity-test cases; DESIGN.md §8 table), one launch of
    the fused kernel per step on the config's largest matrix (c5: all 8 experts of the grouped gate GEMM).  Same JSON
    keys as the headline line; a diagnostic, not the line the driver reads (the default workload stays config 2)."""
    import torch
    from paper_2606_15789_b200 import binding as B, build as libbuild, inputs, runtime as rt
    libbuild.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: anslin has no CPU fallback")
    torch.cuda.set_device(0)
    tile_n, tile_k, lflag = 32, 1024, B.FLAG_LANE_STREAMS
    if args.workload == "c3":
        n, k, m = 13824, 5120, 75
        q, s8 = inputs.quant_sq8_weights(inputs.weights_f32(n, k, seed=5, jitter=True))
        xq, xs = inputs.quant_int8_acts(inputs.acts_f32(m, k, seed=6))
        buf, st = B.anslin_encode_host(B.FMT_INT8, q, n, k, tile_k=tile_k, scales=s8, tile_n=tile_n, flags=lflag)
        copies = [rt.DeviceWeight(buf) for _ in range(6)]          # 6 x 41 MB > L2
        x, xsd = rt.x_to_device(B.FMT_INT8, xq), torch.from_numpy(xs).cuda()
        y = torch.empty((m, n), dtype=torch.float32, device="cuda")
        calls = [(lambda d=d: d.gemm(x, xsd, y)) for d in copies]
        name, dtype, nbytes, nw, flops = "config3: SQ8 int8 gate 13824x5120, M=75", "int8", buf.size, n * k, 2.0 * m * n * k
        x_host, y_rows = torch.from_numpy(xq).pin_memory(), m
    elif args.workload == "c4":
        n, k, m = 28672, 8192, 64
        p4, s4, z4 = inputs.quant_awq4_weights(inputs.weights_f32(n, k, seed=11, outliers=False), 128)
        xh = inputs.acts_f32(m, k, seed=12).astype(np.float16)
        buf, st = B.anslin_encode_host(B.FMT_INT4_AWQ, p4, n, k, tile_k=tile_k, scales=s4, zeros=z4, group_size=128, tile_n=tile_n, flags=lflag)
        copies = [rt.DeviceWeight(buf) for _ in range(3)]          # 3 x 125 MB > L2
        x, y = rt.x_to_device(B.FMT_INT4_AWQ, xh), torch.empty((m, n), dtype=torch.float32, device="cuda")
        calls = [(lambda d=d: d.gemm(x, None, y)) for d in copies]
        name, dtype, nbytes, nw, flops = "config4: AWQ int4 g128 gate 28672x8192, M=64", "f16", buf.size, n * k, 2.0 * m * n * k
        x_host, y_rows = torch.from_numpy(xh).pin_memory(), m
    else:
        n, k, E, tokens = 16384, 6144, 8, 95
        rows, tok = inputs.route_top2(tokens, E, seed=21)
        x8t, xst = inputs.quant_fp8_acts(inputs.acts_f32(tokens, k, seed=22))
        x8, xs = x8t[tok], xst[tok]
        experts, nbytes = [], 0
        for e in range(E):
            f8, sc = inputs.quant_fp8_weights(inputs.weights_f32(n, k, seed=30 + e, std=0.015, outliers=False))
            buf, st = B.anslin_encode_host(B.FMT_FP8_E4M3, f8, n, k, tile_k=tile_k, w_scale=sc, tile_n=tile_n, flags=lflag)
            experts.append(rt.DeviceWeight(buf)); nbytes += buf.size      # 8 x 83 MB > L2
        x, xsd = rt.x_to_device(B.FMT_FP8_E4M3, x8), torch.from_numpy(xs).cuda()
        y = torch.empty((2 * tokens, n), dtype=torch.float32, device="cuda")
        calls = [lambda: rt.gemm_grouped(experts, rows, x, xsd, y)]
        name, dtype, nw, flops = "config5: Mixtral-shaped MoE, 8 experts fp8 gate 16384x6144, 95 tokens top-2", "fp8", E * n * k, 2.0 * 2 * tokens * n * k
        x_host, y_rows = torch.from_numpy(x8).pin_memory(), 2 * tokens
    y_host = torch.empty((y_rows, n), dtype=torch.float32).pin_memory()
    sampler = ClockSampler(0); sampler.start(); sampler.wait_first()
    for i in range(max(args.warmup, 3)):
        calls[i % len(calls)]()
    torch.cuda.synchronize()
    lo = sampler.mark()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches = 0
    e0.record()
    for i in range(args.steps):
        calls[i % len(calls)]()
        launches += B.anslin_last_launch_count()
    e1.record(); torch.cuda.synchronize()
    time.sleep(0.03)
    clocks = sampler.stop(lo, sampler.mark())
    ms = e0.elapsed_time(e1) / args.steps
    t0 = time.perf_counter()
    for i in range(args.steps):                      # e2e: pinned X in, Y out every step
        x.view(torch.uint8).copy_(x_host.view(torch.uint8), non_blocking=True)
        calls[i % len(calls)]()
        y_host.copy_(y, non_blocking=True)
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / args.steps
    hbm_peak, _, kind = peaks()
    algo = nbytes + x.numel() * x.element_size() + y.numel() * 4
    print(json.dumps({"metric": METRIC, "value": flops / (ms * 1e-3) / 1e12, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
                      "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                      "dtype": dtype, "data": "synthetic",
                      "config": {"workload": name, "tile": "%dx%d" % (tile_n, tile_k), "word_layout": "lanes",
                                 "l2_policy": "rotating copies / experts larger than L2"},
                      "clocks": clocks, "gpu_launches": launches,
                      "e2e": {"value": flops / e2e_s / 1e12, "unit": UNIT, "h2d_bytes_per_step": int(x.numel() * x.element_size()),
                              "d2h_bytes_per_step": int(y.numel() * 4)},
                      "roofline": {"bound": "hbm", "achieved": algo / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                                   "frac": algo / (ms * 1e-3) / 1e9 / hbm_peak, "traffic": None, "peak_kind": "of " + kind},
                      "gsym_per_s": nw / (2 if args.workload == "c4" else 1) / (ms * 1e-3) / 1e9,
                      "bits_per_weight": st["bits_per_weight"]}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="anslin")
    ap.add_argument("--m", type=int, default=75)
    ap.add_argument("--no-extras", action="store_true", help="skip per-M table, dense comparator, decode-only and CPU legs")
    ap.add_argument("--tile", default="32x256", help="tile_n x tile_k of the compressed containers (128x64 = BASELINE config 1's shape)")
    ap.add_argument("--layout", default="lanes", choices=["lanes", "interleaved"], help="word layout of the containers: every lane "
                    "its own stream (32-row tiles only) or words interleaved in read order")
    ap.add_argument("--symbols", default="paper", choices=["paper", "pair4"], help="paper = one coded symbol per weight (PAPER.md's "
                    "symbolisation, the headline); pair4 = the variant that codes two K-adjacent bf16 exponents per symbol "
                    "(SURVEY 8(f) NEXT-5, ANSLIN_FMT_BF16_PAIR4; lanes layout only)")
    ap.add_argument("--workload", default="c2", choices=["c2", "c3", "c4", "c5"], help="c2 = the headline (BASELINE config 2); c3 / c4 / c5 = "
                    "diagnostic lines for the other configs (int8, int4, fp8 MoE)")
    ap.add_argument("--group", default="qkv,o,gateup,down", help="launch grouping of the 7 projections: 'each' = 7 launches, or "
                    "comma-separated groups out of qkv / q,k,v / gateup / gate,up / o / down (projections that share an input)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload != "c2":
        return run_other_config(args)

    import torch
    from paper_2606_15789_b200 import binding as B, build as libbuild, inputs, runtime as rt
    libbuild.build()
    from paper_2606_15789_b200.dist import Ranks
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: anslin has no CPU fallback")
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    ranks = Ranks("nccl", torch.device("cuda", local))
    world, rank = ranks.world, ranks.rank

    # ---- offline stage (untimed): synthesize, compress, upload
    layer = layer_weights()
    containers, stats = [], []
    tile_n, tile_k = (int(v) for v in args.tile.split("x"))
    for (_, n, k, w) in layer:
        lflag = B.FLAG_LANE_STREAMS if (args.layout == "lanes" and tile_n == 32) else 0
        buf, st = B.anslin_encode_host(B.FMT_BF16_PAIR4 if args.symbols == "pair4" else B.FMT_BF16, w, n, k, tile_k=tile_k,
                                       flags=B.FLAG_STATE_PAYLOAD | lflag, tile_n=tile_n)
        containers.append(buf); stats.append(st)
    dws = [rt.DeviceWeight(c) for c in containers]
    m = args.m
    # projections that share an input in a decoder layer share the X tensor here too: q/k/v, gate/up
    share = {"k": "q", "v": "q", "up": "gate"}
    names = [t[0] for t in layer]
    x_owner = [names.index(share.get(nm, nm)) for nm in names]
    xs_host = {i: torch.from_numpy(inputs.f32_to_bf16_bits(inputs.acts_f32(m, layer[i][2], seed=ranks.batch_seed(500 + i))).view(np.int16)).pin_memory()
               for i in sorted(set(x_owner))}
    xs_dev = {i: t.cuda().view(torch.bfloat16) for i, t in xs_host.items()}
    xs = [xs_dev[o] for o in x_owner]
    ys = [torch.empty((m, n), dtype=torch.float32, device="cuda") for (_, n, k, _) in layer]
    ys_host = [torch.empty((m, n), dtype=torch.float32).pin_memory() for (_, n, k, _) in layer]
    flops_step = sum(2.0 * m * n * k for (_, n, k, _) in layer)
    comp_bytes = sum(c.size for c in containers)
    n_weights = sum(n * k for (_, n, k, _) in layer)
    # launch groups: each group is ONE anslin_gemm_multi launch (a single projection = anslin_gemm's launch)
    alias = {"qkv": ["q", "k", "v"], "gateup": ["gate", "up"]}
    if args.group == "each":
        groups = [[i] for i in range(len(layer))]
    else:
        groups = [[names.index(nm) for nm in alias.get(g, [g])] for g in args.group.split(",")]
    assert sorted(i for g in groups for i in g) == list(range(len(layer))), "--group must cover every projection once"
    calls = [rt.MultiGemm([dws[i] for i in g], [xs[i] for i in g], None, [ys[i] for i in g]) for g in groups]
    group_names = ["+".join(names[i] for i in g) for g in groups]
    # algorithmic bytes of a launch: its containers + each distinct X once + its Y
    algo_bytes = [sum(containers[i].size + m * layer[i][1] * 4 for i in g) + sum(m * layer[o][2] * 2 for o in {x_owner[i] for i in g})
                  for g in groups]

    def step(record=None):
        launches = 0
        for gi, call in enumerate(calls):
            if record is not None:
                record[gi][0].record()
            call()
            launches += B.anslin_last_launch_count()
            if record is not None:
                record[gi][1].record()
        return launches

    def barrier():
        torch.cuda.synchronize()
        ranks.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local); sampler.start(); sampler.wait_first()
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    mark_lo = sampler.mark()
    # The timed region holds nothing but the step's kernel launches (no events between them: consecutive launches
    # overlap prologue and tail through programmatic dependent launch); CUDA events bracket the K steps.
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches = 0
    e0.record()
    for s in range(args.steps):
        launches += step()
    e1.record()
    barrier()
    time.sleep(0.03)
    clocks = sampler.stop(mark_lo, sampler.mark())
    ms = ranks.max_over_ranks(e0.elapsed_time(e1))
    ms_step = ms / args.steps
    value = world * flops_step / (ms_step * 1e-3) / 1e12
    # diagnostic pass (outside the timed region): one event pair per launch -> per_launch_us
    n_diag = min(args.steps, 20)
    evs = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in calls] for _ in range(n_diag)]
    for s in range(n_diag):
        step(evs[s])
    barrier()
    kern_ms = [[a.elapsed_time(b) for (a, b) in row] for row in evs]
    kern_ms_mean = np.mean(np.array(kern_ms), axis=0)             # per launch group
    hbm_peak, tc_peak, peak_kind = peaks()
    # the fused kernel is the only kernel of a step: its launches' average duration = timed region / launches
    achieved = sum(algo_bytes) / (ms_step * 1e-3) / 1e9
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp):
        traffic = json.load(open(tp)).get("fused_gemm_bytes_per_launch_mean")

    # ---- e2e: the same step through the C ABI with HOST buffers (pinned X in, Y out) inside the timed region
    # Device->host reads of Y run on a copy stream of their own, behind an event per launch group, so that they
    # overlap the next group's kernel; a group's next launch waits for the previous read of its Y buffers.
    copy_stream = torch.cuda.Stream()
    y_ready = [torch.cuda.Event() for _ in groups]
    y_read = [torch.cuda.Event() for _ in groups]

    def step_e2e(calls_=None, ys_=None, ys_host_=None):
        calls_, ys_, ys_host_ = calls_ or calls, ys_ or ys, ys_host_ or ys_host
        main = torch.cuda.current_stream()
        for gi, (g, call) in enumerate(zip(groups, calls_)):
            for o in sorted({x_owner[i] for i in g}):
                xs_dev[o].view(torch.int16).copy_(xs_host[o], non_blocking=True)
            main.wait_event(y_read[gi])
            call()
            y_ready[gi].record(main)
            copy_stream.wait_event(y_ready[gi])
            with torch.cuda.stream(copy_stream):
                for i in g:
                    ys_host_[i].copy_(ys_[i], non_blocking=True)
                y_read[gi].record(copy_stream)
    for _ in range(3):
        step_e2e()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step_e2e()
    barrier()
    e2e_s = ranks.max_over_ranks(time.perf_counter() - t0)
    e2e = {"value": world * flops_step * args.steps / e2e_s / 1e12, "unit": UNIT,
           "h2d_bytes_per_step": int(sum(t.numel() * 2 for t in xs_host.values())),
           "d2h_bytes_per_step": int(sum(m * n * 4 for (_, n, k, _) in layer))}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
           "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
           "data": "synthetic",
           "config": {"workload": WORKLOAD, "batch_m": m, "tile": args.tile, "word_layout": args.layout, "symbols": args.symbols, "streams": 32, "prob_bits": 12,
                      "launch_groups": group_names,
                      "l2_policy": "inputs larger than L2: %.0f MB of compressed weights stream per step" % (comp_bytes / 1e6),
                      "parallelism": "replicas, one batch per GPU" if world > 1 else "1 GPU"},
           "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
           "roofline": {"bound": "hbm", "achieved": achieved, "peak": hbm_peak, "unit": "GB/s", "frac": achieved / hbm_peak,
                        "traffic": traffic, "peak_kind": "of " + peak_kind,
                        "kernel": "fused_gemm_kernel<bf16,payload> (%d launches/step; bytes = containers + X + Y)" % len(calls)},
           # the bound that actually binds (SURVEY §8(d) bound 3): the decoder's integer work on the ALU pipe.
           # peak = SMs x 4 schedulers x 16 lanes/clk (one ALU-pipe warp instruction per 2 clk) x SM clock under load
           #        / ALU-pipe instructions per decoded symbol in the hot loop's SASS
           "decoder_bound": (lambda peak: {"bound": "alu", "achieved": n_weights / (ms_step * 1e-3) / 1e9, "peak": peak,
                                           "unit": "Gsymbol/s", "frac": n_weights / (ms_step * 1e-3) / 1e9 / peak,
                                           "alu_instr_per_symbol": ALU_INSTR_PER_SYMBOL, "sm_mhz": clocks.get("sm_mhz")})(
               148 * 4 * 16 * float(clocks.get("sm_mhz") or 1965.0) * 1e6 / ALU_INSTR_PER_SYMBOL / 1e9),
           "compressed_gbs": world * comp_bytes / (ms_step * 1e-3) / 1e9,
           "decoded_weights_gbs": world * n_weights * 2 / (ms_step * 1e-3) / 1e9,
           "bits_per_weight": 8.0 * comp_bytes / n_weights,
           "h_sym_bits_per_weight": float(np.sum([(s["entropy_bits_per_symbol"] + s["raw_entropy_bits_per_symbol"]) * s["n_weights"]
                                                  for s in stats]) / n_weights),
           "per_launch_us": {nm: round(1e3 * float(t), 2) for nm, t in zip(group_names, kern_ms_mean)}}

    if rank == 0 and not args.no_extras:
        # the same end-to-end step with Y produced in bf16 (anslin_gemm_multi_ex): half the device-to-host bytes
        ys_b = [torch.empty((m, n), dtype=torch.bfloat16, device="cuda") for (_, n, k, _) in layer]
        ys_host_b = [torch.empty((m, n), dtype=torch.bfloat16).pin_memory() for (_, n, k, _) in layer]
        calls_b = [rt.MultiGemm([dws[i] for i in g], [xs[i] for i in g], None, [ys_b[i] for i in g]) for g in groups]
        for _ in range(3):
            step_e2e(calls_b, ys_b, ys_host_b)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            step_e2e(calls_b, ys_b, ys_host_b)
        barrier()
        tb = time.perf_counter() - t0
        out["e2e_y_bf16"] = {"value": flops_step * args.steps / tb / 1e12, "unit": UNIT,
                             "h2d_bytes_per_step": e2e["h2d_bytes_per_step"], "d2h_bytes_per_step": int(sum(m * n * 2 for (_, n, k, _) in layer))}
        # per-M table (BASELINE config 2: M in {1,16,47,75}), dense comparator, decode-only; then the CPU oracle leg
        extra = {}
        for mm in (1, 16, 47, 75):
            xm = [x[:mm].contiguous() for x in xs]
            ym = [torch.empty((mm, n), dtype=torch.float32, device="cuda") for (_, n, k, _) in layer]
            for _ in range(3):
                for i, dw in enumerate(dws):
                    dw.gemm(xm[i], None, ym[i])
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(); a.record()
            for _ in range(5):
                for i, dw in enumerate(dws):
                    dw.gemm(xm[i], None, ym[i])
            b.record(); torch.cuda.synchronize()
            t = a.elapsed_time(b) / 5
            fl = sum(2.0 * mm * n * k for (_, n, k, _) in layer)
            extra["M=%d" % mm] = {"ms": round(t, 4), "tflops": round(fl / (t * 1e-3) / 1e12, 3),
                                  "compressed_gbs": round(comp_bytes / (t * 1e-3) / 1e9, 1)}
        out["per_m"] = extra
        wd = [torch.from_numpy(w.view(np.int16)).cuda() for (_, _, _, w) in layer]
        wsd = [torch.empty(B.anslin_dense_workspace_bytes(n, k, m), dtype=torch.uint8, device="cuda") for (_, n, k, _) in layer]
        for _ in range(3):
            for i in range(len(layer)):
                rt.dense_gemm(B.FMT_BF16, wd[i], xs[i], y=ys[i], ws=wsd[i])
        # the seven launches are replayed from a CUDA graph: at ~25 us each the Python / tensor-map host path, not the GPU,
        # would otherwise set the comparator's time
        def dense_layer():
            for i in range(len(layer)):
                rt.dense_gemm(B.FMT_BF16, wd[i], xs[i], y=ys[i], ws=wsd[i])
        replay, how = dense_layer, "python loop"
        try:
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                dense_layer()
            replay, how = g.replay, "cuda graph replay"
        except Exception:
            torch.cuda.synchronize()
        replay()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); a.record()
        for _ in range(5):
            replay()
        b.record(); torch.cuda.synchronize()
        t = a.elapsed_time(b) / 5
        out["dense_uncompressed"] = {"ms": round(t, 4), "tflops": round(flops_step / (t * 1e-3) / 1e12, 3),
                                     "hbm_gbs": round(n_weights * 2 / (t * 1e-3) / 1e9, 1), "launched_by": how}
        # context only (SURVEY 8(d) "torch.matmul may be printed as extra context"): the same seven GEMMs through cuBLAS
        wt = [t.view(torch.bfloat16) for t in wd]
        for _ in range(3):
            for i in range(len(layer)):
                torch.matmul(xs[i], wt[i].t())
        torch.cuda.synchronize(); a.record()
        for _ in range(5):
            for i in range(len(layer)):
                torch.matmul(xs[i], wt[i].t())
        b.record(); torch.cuda.synchronize()
        t = a.elapsed_time(b) / 5
        out["dense_cublas_context"] = {"ms": round(t, 4), "tflops": round(flops_step / (t * 1e-3) / 1e12, 3),
                                       "hbm_gbs": round(n_weights * 2 / (t * 1e-3) / 1e9, 1), "note": "torch.matmul, bf16 out; context, not the comparator"}
        del wd, wt
        a.record()
        for _ in range(3):
            for dw in dws:
                dw.decode()
        b.record(); torch.cuda.synchronize()
        t = a.elapsed_time(b) / 3
        out["decode_only"] = {"ms": round(t, 4), "decoded_gbs": round(n_weights * 2 / (t * 1e-3) / 1e9, 1),
                              "gsym_per_s": round(n_weights / (t * 1e-3) / 1e9, 1)}
        out["cpu_baseline"] = cpu_oracle_leg(layer, containers, m)
    if rank == 0:
        print(json.dumps(out))
    ranks.close()


if __name__ == "__main__":
    main()
