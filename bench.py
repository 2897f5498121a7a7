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


def _oracle_decode_worker(buf_bytes: bytes) -> int:
    """All-cores leg: one process decodes one container with the oracle (plain C rANS driven from numpy).  Module level so
    that a spawned interpreter can import it; touches nothing but oracle/."""
    from oracle import container as oc
    _, w_dec, _ = oc.decode(np.frombuffer(buf_bytes, dtype=np.uint8))
    return int(w_dec.size)


def cpu_oracle_leg(layer, oracle_containers, m: int, names=("q", "k"), all_cores: bool = True):
    """The oracle as it stands, timed on the host cores over a bounded sample of the workload (containers written by the
    oracle's own encoder): (1) one thread: container decode + float64 GEMM of the named projections; (2) all cores: one
    process per core, each decoding the k projection's container (decode only)."""
    from oracle import container as oc, gemm as og
    from paper_2606_15789_b200 import inputs
    try:
        from threadpoolctl import threadpool_info
        blas = max([i.get("num_threads", 1) for i in threadpool_info()] or [1])
    except Exception:
        blas = 1
    flops, weights, t_dec, t0 = 0.0, 0, 0.0, time.perf_counter()
    for (name, n, k, w) in layer:
        if name not in names:
            continue
        td = time.perf_counter()
        _, w_dec, _ = oc.decode(oracle_containers[name])
        t_dec += time.perf_counter() - td
        x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=7))
        og.gemm_bf16(x, w_dec)
        flops += 2.0 * m * n * k
        weights += n * k
    dt = time.perf_counter() - t0
    out = {"value": flops / dt / 1e12, "unit": UNIT, "cores": int(blas), "kind": "oracle", "seconds": round(dt, 2),
           "decode_weights_per_s": weights / t_dec, "decoded_gbs": 2.0 * weights / t_dec / 1e9,
           "sample": "projections %s of the layer at M=%d: oracle container decode (1 thread) + float64 GEMM (%d BLAS threads)"
                     % ("/".join(names), m, blas)}
    if all_cores:
        import multiprocessing as mp
        ncore = os.cpu_count() or 1
        kbuf = oracle_containers["k"].tobytes()
        kw = next(n * k for (nm, n, k, _) in layer if nm == "k")
        try:
            with mp.get_context("spawn").Pool(ncore) as pool:
                pool.map(_oracle_decode_worker, [kbuf] * ncore)        # warm the workers (imports, library build)
                t1 = time.perf_counter()
                done = pool.map(_oracle_decode_worker, [kbuf] * (2 * ncore))
                ta = time.perf_counter() - t1
            out["all_cores"] = {"cores": ncore, "decode_weights_per_s": sum(done) / ta, "decoded_gbs": 2.0 * sum(done) / ta / 1e9,
                                "seconds": round(ta, 2), "sample": "%d oracle decodes of the k projection (%d weights each), one process per core"
                                                                   % (2 * ncore, kw)}
        except Exception as e:       # a box that cannot spawn processes: say so, keep the single-thread leg
            out["all_cores"] = {"unavailable": repr(e)[:200]}
    return out


def oracle_containers_for(layer, names):
    """Containers of the named projections written by the ORACLE's encoder (the reference arm and the CPU leg load no product code)."""
    from oracle import container as oc
    return {nm: oc.encode(0, w, k, tile_k=256, tile_n=32, flags=3)[0] for (nm, n, k, w) in layer if nm in names}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import codec
    codec.build()
    layer = [t for t in layer_weights() if t[0] in ("k",)]       # bounded sample: the k projection (1024x5120)
    conts = oracle_containers_for(layer, ("k",))
    for _ in range(args.warmup):
        cpu_oracle_leg(layer, conts, args.m, names=("k",), all_cores=False)
    t0 = time.perf_counter()
    vals = [cpu_oracle_leg(layer, conts, args.m, names=("k",), all_cores=False) for _ in range(args.steps)]
    dt = time.perf_counter() - t0
    flops = args.steps * 2.0 * args.m * 1024 * 5120
    v = flops / dt / 1e12
    cb = dict(vals[-1]); cb["value"] = v
    sample = "each step = oracle decode (container from the oracle's encoder) + float64 GEMM of the k projection (1024x5120) at M=%d" % args.m
    cb["sample"] = sample
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                      "config": {"workload": WORKLOAD, "batch_m": args.m, "sample": sample}, "cpu_baseline": cb,
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


# Warp instructions per decoded bf16 symbol in the hot loop of fused_tmem_kernel<bf16> (counted in
# profiles/r2_sass_decode_loop.md): 11 in the rANS step (IMAD.SHL, LOP3, LDS, LEA.HI, SHF x2, IMAD, ISETP, @IMAD, @IMAD.IADD,
# @LDS.U16) and 2.5 in the bf16 merge (PRMT x2, SHF, IMAD.SHL, LOP3 per two weights).
INSTR_PER_SYMBOL = 13.5


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
    launches_per_call = B.anslin_gemm_launches(int(np.count_nonzero(rows)) if args.workload == "c5" else 1)
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
        launches += launches_per_call
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


def config_records(hbm_peak: float, tc_peak: float, sm_mhz: float):
    """one record per (config, matrix, M) for BASELINE configs 3-5 (largest matrix and its `down`, every listed
    M): fused time with the three bounds (compressed bytes over HBM, FLOPs over the tensor peak, rANS steps over the issue
    slots), the dense comparator and the decode-only time.  Inputs larger than L2 by rotating copies; CUDA events."""
    import torch
    from paper_2606_15789_b200 import binding as B, inputs, runtime as rt
    recs = []

    def timed(fns, iters=8):
        for f in fns:
            f()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); a.record()
        for i in range(iters):
            fns[i % len(fns)]()
        b.record(); torch.cuda.synchronize()
        return a.elapsed_time(b) * 1e3 / iters           # us

    def record(cfg, mat, n, k, m, fmt_name, cont_bytes, n_sym, flops, tc_ratio, fused_us, dense_us, decode_us, bits, h):
        hbm_us = cont_bytes / (hbm_peak * 1e9) * 1e6
        tc_us = flops / (tc_peak * tc_ratio * 1e12) * 1e6
        issue_us = n_sym * 11.0 / (148 * 4 * 32 * sm_mhz * 1e6) * 1e6            # 11 warp instructions per rANS step
        recs.append({"config": cfg, "matrix": "%s %dx%d" % (mat, n, k), "m": m, "format": fmt_name, "fused_us": round(fused_us, 1),
                     "tflops": round(flops / fused_us / 1e6, 2), "compressed_gbs": round(cont_bytes / fused_us / 1e3, 1),
                     "bound_hbm_us": round(hbm_us, 1), "bound_tensor_us": round(tc_us, 2), "bound_issue_us": round(issue_us, 1),
                     "frac_of_hbm_roofline": round(hbm_us / fused_us, 3), "dense_us": None if dense_us is None else round(dense_us, 1),
                     "decode_only_us": round(decode_us, 1), "bits_per_weight": round(bits, 3), "h_sym": round(h, 3)})

    def copies_of(buf, min_bytes=140e6):
        return [rt.DeviceWeight(buf) for _ in range(max(2, int(np.ceil(min_bytes / buf.size))))]

    # ---- config 3: SQ8 int8, Qwen-14B gate / down
    for mat, n, k, tk in (("gate", 13824, 5120, 1024), ("down", 5120, 13824, 512)):
        q, s8 = inputs.quant_sq8_weights(inputs.weights_f32(n, k, seed=5 if mat == "gate" else 61, jitter=True))
        buf, st = B.anslin_encode_host(B.FMT_INT8, q, n, k, tile_k=tk, scales=s8, tile_n=32, flags=B.FLAG_LANE_STREAMS)
        dws = copies_of(buf)
        wd = [torch.from_numpy(q).cuda() for _ in range(2)]
        sd = torch.from_numpy(s8.view(np.int16)).cuda()
        dec_us = timed([lambda d=d: d.decode() for d in dws], 4)
        for m in (1, 32, 75):
            xq, xs = inputs.quant_int8_acts(inputs.acts_f32(m, k, seed=6))
            x, xsd = rt.x_to_device(B.FMT_INT8, xq), torch.from_numpy(xs).cuda()
            y = torch.empty((m, n), dtype=torch.float32, device="cuda")
            fused = timed([lambda d=d: d.gemm(x, xsd, y) for d in dws])
            dense = timed([lambda w=w: rt.dense_gemm(B.FMT_INT8, w, x, w_scale_vec=sd, x_scale=xsd, y=y) for w in wd])
            record("c3", mat, n, k, m, "int8", buf.size, n * k, 2.0 * m * n * k, 2.0, fused, dense, dec_us, st["bits_per_weight"], st["entropy_bits_per_symbol"])
        for d in dws:
            d.close()
        del dws, wd
    # ---- config 4: AWQ int4 g128, Llama-70B gate / down
    for mat, n, k in (("gate", 28672, 8192), ("down", 8192, 28672)):
        p4, s4, z4 = inputs.quant_awq4_weights(inputs.weights_f32(n, k, seed=11 if mat == "gate" else 64, outliers=False), 128)
        buf, st = B.anslin_encode_host(B.FMT_INT4_AWQ, p4, n, k, tile_k=1024, scales=s4, zeros=z4, group_size=128, tile_n=32, flags=B.FLAG_LANE_STREAMS)
        dws = copies_of(buf)
        dec_us = timed([lambda d=d: d.decode() for d in dws], 4)
        for m in (1, 16, 64):
            x = rt.x_to_device(B.FMT_INT4_AWQ, inputs.acts_f32(m, k, seed=12).astype(np.float16))
            y = torch.empty((m, n), dtype=torch.float32, device="cuda")
            fused = timed([lambda d=d: d.gemm(x, None, y) for d in dws])
            record("c4", mat, n, k, m, "int4-awq (fp16 MMA)", buf.size, n * k // 2, 2.0 * m * n * k, 1.0, fused, None, dec_us,
                   st["bits_per_weight"], st["entropy_bits_per_symbol"] / 2)
        for d in dws:
            d.close()
        del dws
    # ---- config 5: fp8-e4m3 MoE, 8 Mixtral-shaped experts, top-2 routing, one grouped launch
    for mat, n, k in (("gate", 16384, 6144), ("down", 6144, 16384)):
        experts, nbytes, bits, hs = [], 0, 0.0, 0.0
        for e in range(8):
            f8, sc = inputs.quant_fp8_weights(inputs.weights_f32(n, k, seed=(30 if mat == "gate" else 80) + e, std=0.015, outliers=False))
            buf, st = B.anslin_encode_host(B.FMT_FP8_E4M3, f8, n, k, tile_k=1024, w_scale=sc, tile_n=32, flags=B.FLAG_LANE_STREAMS)
            experts.append(rt.DeviceWeight(buf)); nbytes += buf.size; bits += st["bits_per_weight"] / 8; hs += st["entropy_bits_per_symbol"] / 8
        dec_us = timed([lambda: [d.decode() for d in experts]], 2)
        for tokens in (20, 95):
            rows, tok = inputs.route_top2(tokens, 8, seed=21)
            x8t, xst = inputs.quant_fp8_acts(inputs.acts_f32(tokens, k, seed=22))
            x, xsd = rt.x_to_device(B.FMT_FP8_E4M3, x8t[tok]), torch.from_numpy(xst[tok]).cuda()
            y = torch.empty((2 * tokens, n), dtype=torch.float32, device="cuda")
            fused = timed([lambda: rt.gemm_grouped(experts, rows, x, xsd, y)], 4)
            record("c5", "8 experts x " + mat, n, k, tokens, "fp8-e4m3", nbytes, 8 * n * k, 2.0 * 2 * tokens * n * k, 2.0, fused, None, dec_us, bits, hs)
        for d in experts:
            d.close()
        del experts
    torch.cuda.empty_cache()
    return recs


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="anslin")
    ap.add_argument("--m", type=int, default=75)
    ap.add_argument("--no-extras", action="store_true", help="skip per-M table, dense comparator, decode-only, per-config records and CPU legs")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-(config, matrix, M) records of BASELINE configs 3-5")
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
            launches += B.anslin_gemm_launches(len(groups[gi]))      # one block of <= 256 rows per projection
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
    # dram bytes per launch come from a committed ncu capture: reported only for the configuration that capture was taken on
    traffic, traffic_source = None, None
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp):
        tj = json.load(open(tp))
        if tj.get("config") == {"batch_m": m, "tile": args.tile, "word_layout": args.layout, "symbols": args.symbols, "launch_groups": group_names}:
            traffic, traffic_source = tj.get("fused_gemm_bytes_per_launch_mean"), tj.get("source")

    # ---- e2e: the same step through the C ABI with HOST buffers (pinned X in, Y out) inside the timed region
    # Both directions run on copy streams of their own, as a serving loop would have them: the host->device copy of a launch
    # group's X waits for the group's previous kernel (the last reader of that X buffer) and overlaps the other groups'
    # kernels; the device->host read of its Y runs behind an event per group and overlaps the next group's kernel; a
    # group's next launch waits for its X copy and for the previous read of its Y buffers.  Every step still moves all X in
    # and all Y out inside the timed region.
    copy_stream, h2d_stream = torch.cuda.Stream(), torch.cuda.Stream()
    y_ready = [torch.cuda.Event() for _ in groups]
    y_read = [torch.cuda.Event() for _ in groups]
    x_done = [torch.cuda.Event() for _ in groups]

    def step_e2e(calls_=None, ys_=None, ys_host_=None):
        calls_, ys_, ys_host_ = calls_ or calls, ys_ or ys, ys_host_ or ys_host
        main = torch.cuda.current_stream()
        for gi, (g, call) in enumerate(zip(groups, calls_)):
            h2d_stream.wait_event(y_ready[gi])
            with torch.cuda.stream(h2d_stream):
                for o in sorted({x_owner[i] for i in g}):
                    xs_dev[o].view(torch.int16).copy_(xs_host[o], non_blocking=True)
                x_done[gi].record(h2d_stream)
            main.wait_event(x_done[gi])
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
                        "traffic": traffic, "traffic_source": traffic_source, "peak_kind": "of " + peak_kind,
                        "kernel": "fused_tmem_kernel<bf16,payload> (%d launches/step; bytes = containers + X + Y)" % len(calls)},
           # the bound that actually binds (SURVEY §8(d) bound 3): warp-instruction issue slots of the rANS step.
           # peak = SMs x 4 schedulers x 1 warp instruction (32 lanes) per clk x SM clock under load
           #        / warp instructions per decoded symbol in the hot loop's SASS
           "decoder_bound": (lambda peak: {"bound": "issue", "achieved": n_weights / (ms_step * 1e-3) / 1e9, "peak": peak,
                                           "unit": "Gsymbol/s", "frac": n_weights / (ms_step * 1e-3) / 1e9 / peak,
                                           "instr_per_symbol": INSTR_PER_SYMBOL, "sm_mhz": clocks.get("sm_mhz")})(
               148 * 4 * 32 * float(clocks.get("sm_mhz") or 1965.0) * 1e6 / INSTR_PER_SYMBOL / 1e9),
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
            # the same batch size through the step's four grouped launches (q+k+v, o, gate+up, down)
            calls_m = [rt.MultiGemm([dws[i] for i in g], [xm[x_owner[i]] for i in g], ys=[ym[i] for i in g]) for g in groups]
            for _ in range(3):
                for cm in calls_m:
                    cm()
            torch.cuda.synchronize(); a.record()
            for _ in range(20):
                for cm in calls_m:
                    cm()
            b.record(); torch.cuda.synchronize()
            tg = a.elapsed_time(b) / 20
            extra["M=%d" % mm].update({"grouped_ms": round(tg, 4), "grouped_tflops": round(fl / (tg * 1e-3) / 1e12, 3),
                                       "grouped_compressed_gbs": round(comp_bytes / (tg * 1e-3) / 1e9, 1),
                                       "grouped_frac_of_hbm_roofline": round((comp_bytes + sum(2 * mm * k for (_, n, k, _) in [layer[g[0]] for g in groups]) + sum(4 * mm * n for (_, n, k, _) in layer)) / (tg * 1e-3) / 1e9 / hbm_peak, 4)})
            del calls_m
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
        # decode only (anslin_decode of the seven matrices, one launch each) into preallocated outputs: 550 MB written per pass,
        # so every pass starts with the containers out of L2
        w_outs = [torch.empty((n, k), dtype=torch.int16, device="cuda") for (_, n, k, _) in layer]
        def decode_layer():
            st = torch.cuda.current_stream().cuda_stream
            for dw, o in zip(dws, w_outs):
                B.anslin_decode(dw.weight, o.data_ptr(), o.numel() * 2, st)
        for _ in range(2):
            decode_layer()
        torch.cuda.synchronize()
        a.record()
        for _ in range(5):
            decode_layer()
        b.record(); torch.cuda.synchronize()
        t = a.elapsed_time(b) / 5
        out["decode_only"] = {"ms": round(t, 4), "decoded_gbs": round(n_weights * 2 / (t * 1e-3) / 1e9, 1),
                              "gsym_per_s": round(n_weights / (t * 1e-3) / 1e9, 1)}
        del w_outs
        if not args.no_configs:
            del wsd
            torch.cuda.empty_cache()
            out["configs"] = config_records(hbm_peak, tc_peak, float(clocks.get("sm_mhz") or 1965.0))
        out["cpu_baseline"] = cpu_oracle_leg(layer, oracle_containers_for(layer, ("q", "k")), m)
    if rank == 0:
        print(json.dumps(out))
    ranks.close()


if __name__ == "__main__":
    main()
