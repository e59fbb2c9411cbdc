#!/usr/bin/env python
"""bench.py — BASELINE.json's metric on BASELINE.json's config, through the C ABI.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

A "step" is one pass of the whole hot path over the workload: boa_compress of the full input followed by
boa_decompress of the result (every SURVEY §8(a) row runs, for every byte).  `value` is input MiB per second of
device time over those K steps (the mean of the compress and decompress rates, i.e. 2n/(Tc+Td)), inputs
resident in HBM; `e2e` is the same through the same calls with pinned HOST buffers (copies inside the timing).
The paper's "MB" is MiB, so the unit is MiB/s.

N > 1: chunks are independent — every rank runs the same workload shape on its own seeded input
(weak scaling, no data-path collective); time = max over ranks, value = total bytes / that time.
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
MiB = float(1 << 20)
SM_COUNT = 148
FP32_LANES_PER_SM = 128


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)),
                "bf16_tflops": float(d.get("bf16_tflops_sustained", d.get("bf16_tflops", 1590.0))), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "bf16_tflops": 1400.0, "source": "fallback"}   # B200_PROFILING.md fallback


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "250", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True).start()
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in list(self.lines):
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(cfg, n_streams=64, length=128):
    """The bounded cpu_baseline sample: the first `length` bytes of `n_streams` evenly spaced chunks."""
    data = cfg.data()
    nc = len(data) // cfg.chunk_bytes
    ids = np.linspace(0, nc - 1, n_streams).astype(np.int64)
    buf = np.frombuffer(data, np.uint8)
    return b"".join(buf[i * cfg.chunk_bytes: i * cfg.chunk_bytes + length].tobytes() for i in ids), length


def time_oracle(cfg, n_streams=64, length=128):
    """Oracle (as it stands) compress + decompress of the sample on the host cores.  Returns a dict."""
    from oracle import codec, model as omodel
    try:
        from threadpoolctl import threadpool_info
        cores = max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
    except Exception:
        cores = 1
    w = omodel.load_weights(cfg.weights())
    sample, length = oracle_sample(cfg, n_streams, length)
    t0 = time.perf_counter()
    blob = codec.compress(w, sample, length)
    t1 = time.perf_counter()
    back = codec.decompress(w, blob)
    t2 = time.perf_counter()
    assert back == sample
    n = len(sample)
    return {"value": 2 * n / MiB / (t2 - t0), "unit": "MiB/s", "cores": cores, "kind": "oracle",
            "sample": f"first {length} B of {n_streams} evenly spaced chunks ({n} B), compress+decompress",
            "compress_MiBps": n / MiB / (t1 - t0), "decompress_MiBps": n / MiB / (t2 - t1),
            "seconds": t2 - t0, "bits_per_byte": 8.0 * len(blob) / n}


def workload_name(cfg):
    return (f"{cfg.name}: {cfg.n_bytes / MiB:g} MiB, {cfg.n_bytes // cfg.chunk_bytes} chunks x {cfg.chunk_bytes / 1024:g} KiB, "
            f"{cfg.shape.n_layer}-layer d_model={cfg.shape.d_model} {'bf16' if cfg.weight_dtype else 'fp32'} weights"
            + (f", FFN {cfg.shape.d_ff} + LayerNorm per layer, untied head (the paper's block)" if cfg.shape.d_ff else ""))


def base_line(args, cfg, world):
    return {"metric": "compress+decompress throughput (input bytes), mean of the two directions = 2n/(Tc+Td)",
            "unit": "MiB/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "baseline_config_index": args.config - 1 if args.config <= 5 else None,
                       "streams_per_gpu": cfg.n_bytes // cfg.chunk_bytes, "chunk_bytes": cfg.chunk_bytes,
                       "l2": "inputs larger than L2: the per-step working set is the stream state "
                             f"({cfg.shape.state_bytes_per_stream() * (cfg.n_bytes // cfg.chunk_bytes) / 1e9:.2f} GB) "
                             "vs 126 MB of L2, streamed once per step",
                       "parallelism": f"chunk-sharded x{world}, no collective"}}


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores, same metric/unit/config keys (tier framing (4))."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    line = base_line(args, cfg, args.gpus)
    vals, secs = [], []
    for i in range(args.warmup + args.steps):
        r = time_oracle(cfg, n_streams=16, length=64)
        if i >= args.warmup:
            vals.append(r["value"]); secs.append(r["seconds"])
    v = float(np.mean(vals))
    r.update({"value": v})
    line.update({"impl": "reference", "value": v, "ms_per_step": 1e3 * float(np.mean(secs)), "dtype": "f64",
                 "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
                 "e2e": {"value": v, "unit": "MiB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                 "gpu_launches": 0, "roofline": None, "clocks": None})
    print(json.dumps(line))


# DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) measured by ncu inside the running step, cache
# state left as it is (profiles/r01_insitu_traffic.md): config name -> kernel class -> bytes.
NCU_TRAFFIC = {"cfg2_kinematics_64MiB": {"scan": 145.8e6 + 120.7e6, "inproj": 26.2e6 + 16.7e6, "convx": 12.6e6,
                                         "outproj": 12.6e6, "head": 6.3e6}}


def kernel_work(cfg, B):
    """Algorithmic work of ONE launch of each kernel class for B streams."""
    s = cfg.shape
    D, E, N, R = s.d_model, s.d_inner, s.d_state, s.rank
    # A contraction is computed as `mm` bf16 MMAs per fp32 product (tc_gemm.cuh: 6 for fp32 weights, 3 for bf16
    # weights): its algorithmic tensor work is mm * 2*M*N*K bf16 flops.
    mm = 3 if cfg.weight_dtype else 6
    work = {
        "scan": ("hbm", B * 2 * E * N * 4),                 # h read + written once, fp32
        "convx": ("tensor", mm * 2 * B * E * (R + 2 * N)),  # x_proj
        "inproj": ("tensor", mm * 2 * B * D * 2 * E),
        "outproj": ("tensor", mm * 2 * B * E * D),
        "head": ("tensor", mm * 2 * B * D * 256),
    }
    if s.d_ff:   # the paper's block: two more contractions and a LayerNorm per layer
        work["ffn1"] = ("tensor", mm * 2 * B * D * s.d_ff)
        work["ffn2"] = ("tensor", mm * 2 * B * s.d_ff * D)
        work["lnorm"] = ("hbm", B * D * (4 + 4 + 6))        # v read, u and its image written
    return work


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_2511_11337_b200 import boa, metrics, shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    peaks = load_peaks()

    # weak scaling: every rank gets the full workload shape on its own seeded input
    n, chunk = cfg.n_bytes, cfg.chunk_bytes
    import dataclasses
    rcfg = cfg if rank == 0 else dataclasses.replace(cfg, data_seed=cfg.data_seed + 7919 * rank)
    host = torch.frombuffer(bytearray(rcfg.data()), dtype=torch.uint8)
    m = boa.Model(cfg.weights())
    d_in = host.to(dev)
    d_comp = torch.empty(boa.compress_bound(n, chunk), dtype=torch.uint8, device=dev)
    d_out = torch.empty(n, dtype=torch.uint8, device=dev)
    B = n // chunk

    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]

    def step():
        ev[0].record()
        clen = m.compress_into(d_in, chunk, d_comp)
        pc = m.profile()
        ev[1].record()
        m.decompress_into(d_comp[:clen], d_out)
        pd = m.profile()
        ev[2].record()
        torch.cuda.synchronize()
        return ev[0].elapsed_time(ev[1]), ev[1].elapsed_time(ev[2]), clen, pc, pd

    for i in range(args.warmup):
        _, _, clen, _, _ = step()
        if i == 0 and not torch.equal(d_out, d_in):
            raise SystemExit("bench.py: GPU round trip is not byte-exact")

    m.set_profiling(args.sample_every)
    clocks = ClockSampler(local)
    shard.barrier()
    torch.cuda.synchronize()
    clocks.start()
    tc = td = 0.0
    launches = 0
    samp_ms = {k: 0.0 for k in boa.K_NAMES}
    samp_n = {k: 0 for k in boa.K_NAMES}
    for _ in range(args.steps):
        a, b, clen, pc, pd = step()
        tc += a; td += b
        launches += pc["launches_total"] + pd["launches_total"]
        for p in (pc, pd):
            for k in boa.K_NAMES:
                samp_ms[k] += p["sampled_ms"][k]; samp_n[k] += p["sampled_launches"][k]
    torch.cuda.synchronize()
    shard.barrier()
    clk = clocks.stop()
    m.set_profiling(0)
    if not torch.equal(d_out, d_in):
        raise SystemExit("bench.py: GPU round trip is not byte-exact")

    total_ms, total_bytes = shard.reduce_stats(tc + td, 2.0 * n * args.steps, dev)
    tc_max, _ = shard.reduce_stats(tc, 0.0, dev)
    td_max, _ = shard.reduce_stats(td, 0.0, dev)
    comp_total = shard.reduce_stats(0.0, float(clen), dev)[1]

    # ---- e2e: same calls, pinned HOST buffers, copies inside the timed region
    h_in = host.pin_memory()
    h_comp = torch.empty(boa.compress_bound(n, chunk), dtype=torch.uint8).pin_memory()
    h_out = torch.empty(n, dtype=torch.uint8).pin_memory()
    e2e_steps = max(1, min(args.steps, 2))
    e2e_s = 0.0
    for i in range(1 + e2e_steps):
        shard.barrier(); torch.cuda.synchronize()
        t0 = time.perf_counter()
        hl = m.compress_into(h_in, chunk, h_comp)
        m.decompress_into(h_comp[:hl], h_out)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if i > 0:
            e2e_s += dt
    if not torch.equal(h_out, host):
        raise SystemExit("bench.py: host-buffer round trip is not byte-exact")
    e2e_ms, e2e_bytes = shard.reduce_stats(1e3 * e2e_s, 2.0 * n * e2e_steps, dev)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    line = base_line(args, cfg, world)
    sec = total_ms / 1e3
    line["value"] = total_bytes / MiB / sec
    line["ms_per_step"] = total_ms / args.steps
    line["compress_MiBps"] = world * n * args.steps / MiB / (tc_max / 1e3)
    line["decompress_MiBps"] = world * n * args.steps / MiB / (td_max / 1e3)
    line["bits_per_byte"] = metrics.bits_per_byte(world * n, comp_total)
    line["compression_ratio"] = metrics.compression_ratio(world * n, comp_total)
    line["sigma_ssr_MiBps"] = metrics.sigma_ssr(world * n / MiB, comp_total / MiB, tc_max / 1e3 / args.steps)
    line["clocks"] = clk
    line["e2e"] = {"value": e2e_bytes / MiB / (e2e_ms / 1e3), "unit": "MiB/s",
                   "h2d_bytes_per_step": int(n + hl), "d2h_bytes_per_step": int(hl + n),
                   "note": "timed separately: wall clock around boa_compress + boa_decompress on pinned HOST buffers, the "
                           "copies inside the calls (a few ms of a step of seconds); it runs without the event-bracketed "
                           "eager sample batches that the device-timed steps carry for the roofline, hence value <= e2e"}
    line["gpu_launches"] = int(launches)

    # ---- roofline of the dominant kernel, from the event-bracketed launches inside the timed region
    work = kernel_work(cfg, B)
    alu_peak = SM_COUNT * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12   # TFLOP/s fp32
    tot = sum(samp_ms.values()) or 1.0
    kernels = {}
    for k in boa.K_NAMES:
        if not samp_n[k]:
            continue
        avg_ms = samp_ms[k] / samp_n[k]
        ent = {"share": samp_ms[k] / tot, "avg_us": 1e3 * avg_ms, "launches_sampled": samp_n[k]}
        if k in work:
            bound, amount = work[k]
            if bound == "hbm":
                ent.update({"bound": "hbm", "achieved": amount / 1e9 / (avg_ms / 1e3), "peak": peaks["hbm_gbs"], "unit": "GB/s"})
            elif bound == "tensor":
                ent.update({"bound": "tensor", "achieved": amount / 1e12 / (avg_ms / 1e3), "peak": peaks["bf16_tflops"],
                            "unit": "TFLOP/s", "dtype": "bf16 pieces, fp32 accumulate"})
            else:
                ent.update({"bound": "alu", "achieved": amount / 1e12 / (avg_ms / 1e3), "peak": alu_peak, "unit": "TFLOP/s"})
            ent["frac"] = ent["achieved"] / ent["peak"]
        kernels[k] = ent
    line["kernels"] = kernels
    line["kernels_note"] = ("CUDA events around eagerly launched sample batches of the STEP path (decompression, and the tail of "
                            "compression); compression itself advances 16 steps per pass in time slabs (DESIGN.md 6c) and is "
                            "not sampled per kernel")
    ranked = [k for k in sorted(kernels, key=lambda k: -kernels[k]["share"]) if "bound" in kernels[k]]
    if ranked:
        k = ranked[0]
        e = kernels[k]
        line["roofline"] = {"kernel": k, "bound": e["bound"], "achieved": e["achieved"], "peak": e["peak"], "unit": e["unit"],
                            "frac": e["frac"], "traffic": NCU_TRAFFIC.get(cfg.name, {}).get(k) if B == 4096 else None,
                            "algorithmic": work[k][1], "traffic_unit": "bytes per launch (ncu, in situ)",
                            "peak_source": peaks["source"], "share_of_step": e["share"]}
    else:
        line["roofline"] = None
    s = cfg.shape
    hbm_floor_s = 2.0 * s.state_bytes_per_stream() * n / (peaks["hbm_gbs"] * 1e9)   # per direction, state traffic only
    line["path_roofline"] = {"bound": "hbm", "what": "2 x stream state per input byte (SURVEY 8(d))",
                             "ceiling_MiBps": n / MiB / hbm_floor_s, "frac": line["value"] / (n / MiB / hbm_floor_s) / world}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = time_oracle(cfg)
    else:
        line["cpu_baseline"] = None
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs[] number, 1-based (2 = the metric's config; 6 = the paper's own block on config 2's input, SURVEY 8(f) NEXT-2)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--sample-every", type=int, default=48, help="event-bracket every k-th 32-step batch (roofline)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--streams", type=int, default=0, help="run the config's model with this many chunks (streams per step) ...")
    ap.add_argument("--chunk-bytes", type=int, default=0, help="... of this many bytes each (a sweep point, not the headline workload)")
    args = ap.parse_args()
    from paper_2511_11337_b200 import synth
    cfg = synth.CONFIGS[args.config]
    if args.streams or args.chunk_bytes:
        import dataclasses
        chunk = args.chunk_bytes or cfg.chunk_bytes
        streams = args.streams or cfg.n_bytes // cfg.chunk_bytes
        cfg = dataclasses.replace(cfg, name=f"{cfg.name}[sweep: {streams} streams x {chunk} B]", n_bytes=streams * chunk, chunk_bytes=chunk)
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
