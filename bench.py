#!/usr/bin/env python
"""bench.py — BASELINE.json's metric on BASELINE.json's config, through the C ABI.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

A "step" is one pass of the whole hot path over the workload: boa_compress of the full input followed by
boa_decompress of the result (every SURVEY §8(a) row runs, for every byte).  `value` is input MiB per second of
device time over those K steps (the mean of the compress and decompress rates, i.e. 2n/(Tc+Td)), inputs
resident in HBM; `e2e` is the same through the same calls with pinned HOST buffers (copies inside the timing).
The paper's "MB" is MiB, so the unit is MiB/s.

After the K headline steps the default N = 1 run also takes, ONCE each and through the same C-ABI calls, the points
`north_star` and BASELINE.json's sweeps name (key `sweep`): the configs[3] model at B = 65,536 streams, the configs[4]
model at B = 8,192 / 64 / 1, configs[0] as it is, and (key `largest_config`) the largest single-GPU configuration,
configs[3] at 65,536 chunks x 16 KiB = 1 GiB.  `--no-sweep` / `--no-largest` skip them.

N > 1: chunks are independent.  Default (`--scaling weak`): every rank runs the same workload shape on its own
seeded input, no data-path collective; time = max over ranks, value = total bytes / that time.  `--scaling strong`: the
ranks share ONE input, each compresses its contiguous chunk range (boa_compress_shard), rank 0 assembles one BOA1
container from the gathered parts (boa_container_assemble), every rank decodes its range of that container
(boa_decompress_shard).
"""
from __future__ import annotations

import argparse
import dataclasses
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
PAPER_CONTEXT = ("the paper's own GPU path: ~3.9 MiB/s compression on an RTX 5090 with a 1-layer d_m = 256 model "
                 "(PAPER Table I, P:196-217; BASELINE.md section 1) - another machine and model, context only")


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


# --------------------------------------------------------------------------------------------- the oracle, timed
def oracle_sample(cfg, n_streams, length):
    """The bounded cpu_baseline sample: the first `length` bytes of `n_streams` evenly spaced chunks."""
    data = cfg.data()
    nc = len(data) // cfg.chunk_bytes
    ids = np.linspace(0, nc - 1, n_streams).astype(np.int64)
    buf = np.frombuffer(data, np.uint8)
    return b"".join(buf[i * cfg.chunk_bytes: i * cfg.chunk_bytes + length].tobytes() for i in ids), length


def time_oracle(cfg, n_streams=64, length=128, data=None):
    """Oracle (as it stands: numpy fp64 model + pure-Python integer coder) compress + decompress of the sample on the
    host cores.  `cores` is what it actually used: process CPU time / wall time (its coder loops are single-threaded
    Python; only the small numpy matmuls can fan out over the BLAS pool)."""
    from oracle import codec, model as omodel
    try:
        from threadpoolctl import threadpool_info
        pool = max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
    except Exception:
        pool = 1
    w = omodel.load_weights(cfg.weights())
    sample, length = oracle_sample(cfg, n_streams, length) if data is None else (data, length)
    c0, t0 = time.process_time(), time.perf_counter()
    blob = codec.compress(w, sample, length)
    t1 = time.perf_counter()
    back = codec.decompress(w, blob)
    t2, c2 = time.perf_counter(), time.process_time()
    assert back == sample
    n = len(sample)
    used = max(1, int(round((c2 - c0) / max(t2 - t0, 1e-9))))
    return {"value": 2 * n / MiB / (t2 - t0), "unit": "MiB/s", "cores": used, "kind": "oracle",
            "impl": "numpy fp64 model + pure-Python big-integer range coder (oracle/, as it stands, never tuned)",
            "threads_used": used, "blas_pool_threads": pool, "host_cores": os.cpu_count(),
            "sample": f"first {length} B of {n_streams} evenly spaced chunks of the workload ({n} B), compress+decompress",
            "compress_MiBps": n / MiB / (t1 - t0), "decompress_MiBps": n / MiB / (t2 - t1),
            "seconds": t2 - t0, "bits_per_byte": 8.0 * len(blob) / n, "context": PAPER_CONTEXT}


def workload_name(cfg):
    return (f"{cfg.name}: {cfg.n_bytes / MiB:g} MiB, {cfg.n_bytes // cfg.chunk_bytes} chunks x {cfg.chunk_bytes / 1024:g} KiB, "
            f"{cfg.shape.n_layer}-layer d_model={cfg.shape.d_model} {'bf16' if cfg.weight_dtype else 'fp32'} weights"
            + (f", FFN {cfg.shape.d_ff} + LayerNorm per layer, untied head (the paper's block)" if cfg.shape.d_ff else ""))


def base_line(args, cfg, world):
    strong = getattr(args, "scaling", "weak") == "strong" and world > 1
    return {"metric": "compress+decompress throughput (input bytes), mean of the two directions = 2n/(Tc+Td)",
            "unit": "MiB/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "higher_is_better": True,
            "scaling": "strong" if strong else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "baseline_config_index": args.config - 1 if args.config <= 5 else None,
                       "streams_per_gpu": (cfg.n_bytes // cfg.chunk_bytes) // (world if strong else 1), "chunk_bytes": cfg.chunk_bytes,
                       "l2": "inputs larger than L2: the per-step working set is the stream state "
                             f"({cfg.shape.state_bytes_per_stream() * (cfg.n_bytes // cfg.chunk_bytes) / 1e9:.2f} GB) "
                             "vs 126 MB of L2, streamed once per step",
                       "parallelism": (f"one input, chunk ranges sharded over {world} GPUs, one container assembled on rank 0"
                                       if strong else f"chunk-sharded x{world}, no collective")}}


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores, same metric/unit/config keys (tier framing (4)); every step is a
    bounded sample of the workload (16 chunks x 64 B), which the line says in `sample` and `note`."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    line = base_line(args, cfg, args.gpus)
    vals, secs = [], []
    sample, length = oracle_sample(cfg, 16, 64)
    for i in range(args.warmup + args.steps):
        r = time_oracle(cfg, n_streams=16, length=64, data=sample)
        if i >= args.warmup:
            vals.append(r["value"]); secs.append(r["seconds"])
    v = float(np.mean(vals))
    r.update({"value": v})
    line.update({"impl": "reference", "value": v, "ms_per_step": 1e3 * float(np.mean(secs)), "dtype": "f64",
                 "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "impl", "threads_used", "host_cores", "sample")},
                 "sample": r["sample"],
                 "note": "a step of this arm is the oracle on a BOUNDED SAMPLE of the config's input (1,024 B), not the "
                         "64 MiB workload; it is a deliberately slow checker, so a ratio against it says nothing about "
                         "kernel quality - parity and the roofline fraction do. " + PAPER_CONTEXT,
                 "e2e": {"value": v, "unit": "MiB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                 "gpu_launches": 0, "roofline": None, "clocks": None})
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------- algorithmic work
def kernel_work(cfg, B):
    """Algorithmic work of ONE launch of each kernel class for B streams.
    Contractions: (bound, issued bf16 flops, useful flops).  A contraction is computed as `mm` bf16 MMAs per fp32
    product (tc_gemm.cuh: 6 piece products for fp32 weights, 3 for bf16 weights), so the tensor pipe ISSUES
    mm * 2*M*N*K bf16 flops for 2*M*N*K flops of the method's own work; both are reported."""
    s = cfg.shape
    D, E, N, R = s.d_model, s.d_inner, s.d_state, s.rank
    mm = 3 if cfg.weight_dtype else 6
    work = {
        "scan": ("hbm", B * 2 * E * N * 4, None),           # h read + written once, fp32
        "convx": ("tensor", mm * 2 * B * E * (R + 2 * N), 2 * B * E * (R + 2 * N)),  # x_proj
        "inproj": ("tensor", mm * 2 * B * D * 2 * E, 2 * B * D * 2 * E),
        "outproj": ("tensor", mm * 2 * B * E * D, 2 * B * E * D),
        "head": ("tensor", mm * 2 * B * D * 256, 2 * B * D * 256),
    }
    # the chained launches of the step path (tc::k_gemm_chain): the sum of their contractions
    def chained(*names):
        return ("tensor", sum(work[k][1] for k in names), sum(work[k][2] for k in names))
    work["chain_in_x"] = chained("inproj", "convx")
    work["chain_out_in_x"] = chained("outproj", "inproj", "convx")
    work["chain_out_head"] = chained("outproj", "head")
    if s.d_ff:   # the paper's block: two more contractions and a LayerNorm per layer
        work["ffn1"] = ("tensor", mm * 2 * B * D * s.d_ff, 2 * B * D * s.d_ff)
        work["ffn2"] = ("tensor", mm * 2 * B * s.d_ff * D, 2 * B * s.d_ff * D)
        work["lnorm"] = ("hbm", B * D * (4 + 4 + 6), None)  # v read, u and its image written
    return work, mm


def step_bytes_per_input_byte(shape):
    """HBM bytes the STEP path (decompression) must move per input byte: the stream state read and written once
    (SURVEY 8(d))."""
    return 2.0 * shape.state_bytes_per_stream()


def slab_bytes_per_input_byte(shape, T=16):
    """HBM bytes the encode-side TIME-SLAB path moves per input byte: 1/T of the state, plus the
    activations between its kernels, which at B*T rows no longer fit L2 and do go through HBM.  Per row and layer:
    u image read (6D), xz written + read (2 * 8E), xs image written + read (2 * 6E), x_proj partials written + read,
    y image written + read (2 * 6E), u read + written (2 * 4D), u image written (6D); per row: embedding (u 4D, image
    6D), logits written + read (2 * 1024)."""
    D, E, R = shape.d_model, shape.d_inner, shape.rank
    ldj = 64 if R + 32 <= 64 else 128
    ks = 4 if (E // 64) % 4 == 0 else (2 if (E // 64) % 2 == 0 else 1)
    per_layer = 6 * D + 16 * E + 12 * E + 2 * 4 * ks * ldj + 12 * E + 8 * D + 6 * D
    if shape.d_ff:
        per_layer += 2 * 6 * shape.d_ff + 2 * 4 * D + 8 * D + 6 * D
    return 2.0 * shape.state_bytes_per_stream() / T + shape.n_layer * per_layer + 10 * D + 2048


def ncu_traffic(cfg_name, B, kernel):
    """DRAM bytes per launch of `kernel` from the tracked ncu capture (profiles/r02_ncu_traffic.json: written from an
    `ncu --set full` run of this bench, with the commit it was taken at) - only for the configuration and B it was
    captured on; otherwise None."""
    p = os.path.join(ROOT, "profiles", "r02_ncu_traffic.json")
    if not os.path.exists(p):
        return None, None
    d = json.load(open(p))
    if d.get("config") != cfg_name or d.get("streams") != B or kernel not in d.get("kernels", {}):
        return None, None
    k = d["kernels"][kernel]
    return k["dram_bytes_read"] + k["dram_bytes_write"], f"profiles/r02_ncu_traffic.json @ {d.get('commit', '?')} ({d.get('command', '')})"


# ------------------------------------------------------------------------------------------------- measuring
def measure(boa, m, d_in, chunk, d_comp, d_out, steps, warmup, sample_every, check=True):
    """`warmup` untimed + `steps` timed passes (compress then decompress) on device-resident buffers; CUDA events."""
    import torch
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

    clen = 0
    for i in range(warmup):
        _, _, clen, _, _ = step()
        if i == 0 and check and not torch.equal(d_out, d_in):
            raise SystemExit("bench.py: GPU round trip is not byte-exact")
    m.set_profiling(sample_every)
    r = {"tc": 0.0, "td": 0.0, "launches": 0, "samp_ms": {k: 0.0 for k in boa.K_NAMES}, "samp_n": {k: 0 for k in boa.K_NAMES},
         "steps_c": 0, "steps_d": 0}
    for _ in range(steps):
        a, b, clen, pc, pd = step()
        r["tc"] += a; r["td"] += b
        r["launches"] += pc["launches_total"] + pd["launches_total"]
        r["steps_c"] += pc["steps"]; r["steps_d"] += pd["steps"]
        for p in (pc, pd):
            for k in boa.K_NAMES:
                r["samp_ms"][k] += p["sampled_ms"][k]; r["samp_n"][k] += p["sampled_launches"][k]
    m.set_profiling(0)
    if check and steps > 0 and not torch.equal(d_out, d_in):
        raise SystemExit("bench.py: GPU round trip is not byte-exact")
    r["clen"] = clen
    return r


def kernel_table(boa, cfg, B, r, peaks):
    work, mm = kernel_work(cfg, B)
    tot = sum(r["samp_ms"].values()) or 1.0
    kernels = {}
    for k in boa.K_NAMES:
        if not r["samp_n"][k]:
            continue
        avg_ms = r["samp_ms"][k] / r["samp_n"][k]
        ent = {"share": r["samp_ms"][k] / tot, "avg_us": 1e3 * avg_ms, "launches_sampled": r["samp_n"][k]}
        if k in work:
            bound, amount, useful = work[k]
            if bound == "hbm":
                ent.update({"bound": "hbm", "achieved": amount / 1e9 / (avg_ms / 1e3), "peak": peaks["hbm_gbs"], "unit": "GB/s"})
                ent["frac"] = ent["achieved"] / ent["peak"]
            else:
                issued = amount / 1e12 / (avg_ms / 1e3)
                ent.update({"bound": "tensor", "achieved": issued, "peak": peaks["bf16_tflops"], "unit": "TFLOP/s",
                            "dtype": "bf16 pieces, fp32 accumulate", "frac": issued / peaks["bf16_tflops"],
                            "tensor_pipe_issued_tflops": issued, "tensor_pipe_issued_frac": issued / peaks["bf16_tflops"],
                            "piece_products_per_fp32_product": mm,
                            "useful_tflops": useful / 1e12 / (avg_ms / 1e3),
                            "useful_frac_of_bf16_peak": useful / 1e12 / (avg_ms / 1e3) / peaks["bf16_tflops"]})
        kernels[k] = ent
    return kernels, work


def direction_rooflines(cfg, n, r, steps, peaks, world=1):
    s = cfg.shape
    dec_ceiling = peaks["hbm_gbs"] * 1e9 / step_bytes_per_input_byte(s) / MiB
    enc_ceiling = peaks["hbm_gbs"] * 1e9 / slab_bytes_per_input_byte(s) / MiB
    comp = n * steps / MiB / (r["tc"] / 1e3)
    dec = n * steps / MiB / (r["td"] / 1e3)
    return {"decompress": {"bound": "hbm", "what": "step path: 2 x stream state per input byte (SURVEY 8(d))",
                           "bytes_per_input_byte": step_bytes_per_input_byte(s), "ceiling_MiBps": dec_ceiling,
                           "achieved_MiBps": dec, "frac": dec / dec_ceiling},
            "compress": {"bound": "hbm", "what": "time-slab path: state / 16 + the activations its kernels exchange "
                                                 "through HBM at B x 16 rows (DESIGN.md 6c)",
                         "bytes_per_input_byte": slab_bytes_per_input_byte(s), "ceiling_MiBps": enc_ceiling,
                         "achieved_MiBps": comp, "frac": comp / enc_ceiling}}


def sweep_point(boa, peaks, config, streams, chunk, label, sample_every=2):
    """One pass (after one warm-up pass) of a configs[] model at `streams` x `chunk` bytes; returns the sweep entry."""
    import torch
    from paper_2511_11337_b200 import synth
    base = synth.CONFIGS[config]
    cfg = dataclasses.replace(base, name=f"{base.name}[{streams} streams x {chunk} B]", n_bytes=streams * chunk, chunk_bytes=chunk)
    n = cfg.n_bytes
    dev = torch.device("cuda", torch.cuda.current_device())
    m = boa.Model(cfg.weights())
    d_in = torch.frombuffer(bytearray(cfg.data()), dtype=torch.uint8).to(dev)
    d_comp = torch.empty(boa.compress_bound(n, chunk), dtype=torch.uint8, device=dev)
    d_out = torch.empty(n, dtype=torch.uint8, device=dev)
    r = measure(boa, m, d_in, chunk, d_comp, d_out, 1, 1, sample_every)
    kernels, _ = kernel_table(boa, cfg, streams, r, peaks)
    rf = direction_rooflines(cfg, n, r, 1, peaks)
    ent = {"point": label, "model": f"{cfg.shape.n_layer}-layer d_model={cfg.shape.d_model} {'bf16' if cfg.weight_dtype else 'fp32'}",
           "streams": streams, "chunk_bytes": chunk, "round_trip": "byte-exact",
           "compress_MiBps": rf["compress"]["achieved_MiBps"], "decompress_MiBps": rf["decompress"]["achieved_MiBps"],
           "us_per_step_compress": 1e3 * r["tc"] / max(r["steps_c"], 1), "us_per_step_decompress": 1e3 * r["td"] / max(r["steps_d"], 1),
           "decompress_over_ceiling": rf["decompress"]["frac"], "compress_over_ceiling": rf["compress"]["frac"],
           "decompress_ceiling_MiBps": rf["decompress"]["ceiling_MiBps"],
           "scan_frac_of_hbm_peak": kernels.get("scan", {}).get("frac"), "scan_us": kernels.get("scan", {}).get("avg_us"),
           "kernel_us": {k: round(v["avg_us"], 2) for k, v in kernels.items()}, "gpu_launches": r["launches"]}
    m.close()
    del d_in, d_comp, d_out
    torch.cuda.empty_cache()
    return ent


def fx_point(boa, config, streams, chunk, label, passes=2):
    """One timed pass (the last of `passes`: by default after one warm-up pass) of FX1, the deterministic fixed-point pipeline, on a configs[]
    model shape at `streams` x `chunk` bytes, device buffers, CUDA events around boa_fx_compress / boa_fx_decompress."""
    import torch
    from paper_2511_11337_b200 import synth
    base = synth.CONFIGS[config]
    n = streams * chunk
    dev = torch.device("cuda", torch.cuda.current_device())
    m = boa.FxModel(base.weights())
    d_in = torch.frombuffer(bytearray(base.data(n)), dtype=torch.uint8).to(dev)
    d_comp = torch.empty(boa.compress_bound(n, chunk), dtype=torch.uint8, device=dev)
    d_out = torch.empty(n, dtype=torch.uint8, device=dev)
    for _ in range(passes):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        ev[0].record()
        clen = m.compress_into(d_in, chunk, d_comp)
        launches = m.last_launches
        ev[1].record()
        m.decompress_into(d_comp[:clen], d_out)
        launches += m.last_launches
        ev[2].record()
        torch.cuda.synchronize()
    if not torch.equal(d_out, d_in):
        raise SystemExit("bench.py: FX1 round trip is not byte-exact")
    tc, td = ev[0].elapsed_time(ev[1]), ev[1].elapsed_time(ev[2])
    ent = {"point": label, "model": f"{base.shape.n_layer}-layer d_model={base.shape.d_model}, INT8 rows / Q12.20 values",
           "streams": streams, "chunk_bytes": chunk, "round_trip": "byte-exact",
           "compress_MiBps": n / MiB / (tc / 1e3), "decompress_MiBps": n / MiB / (td / 1e3),
           "us_per_step_compress": 1e3 * tc / (chunk - 1), "us_per_step_decompress": 1e3 * td / (chunk - 1),
           "bits_per_byte": 8.0 * clen / n, "gpu_launches": int(launches)}
    m.close()
    del d_in, d_comp, d_out
    torch.cuda.empty_cache()
    return ent


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
    if args.scaling == "strong" and world > 1:
        return run_strong(args, cfg, world, rank, dev, peaks)

    # weak scaling: every rank gets the full workload shape on its own seeded input
    n, chunk = cfg.n_bytes, cfg.chunk_bytes
    rcfg = cfg if rank == 0 else dataclasses.replace(cfg, data_seed=cfg.data_seed + 7919 * rank)
    host = torch.frombuffer(bytearray(rcfg.data()), dtype=torch.uint8)
    m = boa.Model(cfg.weights())
    if args.pair_tiles >= 0:
        m.debug_set_pair_tiles(args.pair_tiles)
    if args.persist_max >= 0:
        m.debug_set_persist(args.persist_max, args.persist_cluster)
    if args.chain:
        m.debug_set_chain(True)
    d_in = host.to(dev)
    d_comp = torch.empty(boa.compress_bound(n, chunk), dtype=torch.uint8, device=dev)
    d_out = torch.empty(n, dtype=torch.uint8, device=dev)
    B = n // chunk

    measure(boa, m, d_in, chunk, d_comp, d_out, 0, args.warmup, 0)
    clocks = ClockSampler(local)
    shard.barrier()
    torch.cuda.synchronize()
    clocks.start()
    r = measure(boa, m, d_in, chunk, d_comp, d_out, args.steps, 0, args.sample_every)
    torch.cuda.synchronize()
    shard.barrier()
    clk = clocks.stop()
    tc, td, clen = r["tc"], r["td"], r["clen"]

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
    line["us_per_model_step"] = {"compress": 1e3 * tc / max(r["steps_c"], 1), "decompress": 1e3 * td / max(r["steps_d"], 1)}
    line["bits_per_byte"] = metrics.bits_per_byte(world * n, comp_total)
    line["compression_ratio"] = metrics.compression_ratio(world * n, comp_total)
    line["sigma_ssr_MiBps"] = metrics.sigma_ssr(world * n / MiB, comp_total / MiB, tc_max / 1e3 / args.steps)
    line["clocks"] = clk
    line["e2e"] = {"value": e2e_bytes / MiB / (e2e_ms / 1e3), "unit": "MiB/s",
                   "h2d_bytes_per_step": int(n + hl), "d2h_bytes_per_step": int(hl + n), "passes_timed": e2e_steps,
                   "note": f"timed separately over {e2e_steps} passes (not `steps`): wall clock around boa_compress + boa_decompress "
                           "on pinned HOST buffers, the copies inside the calls (a few ms of a step of seconds); it runs without "
                           "the event-bracketed eager sample batches that the device-timed steps carry for the roofline, hence "
                           "value <= e2e"}
    line["gpu_launches"] = int(r["launches"])

    # ---- roofline of the dominant kernel, from the event-bracketed launches inside the timed region
    alu_peak = SM_COUNT * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12   # TFLOP/s fp32
    kernels, work = kernel_table(boa, cfg, B, r, peaks)
    line["kernels"] = kernels
    line["kernels_note"] = ("CUDA events around eagerly launched sample batches of the STEP path (decompression, and the tail of "
                            "compression); compression itself advances 16 steps per pass in time slabs (DESIGN.md 6c) and is "
                            "not sampled per kernel.  Contractions: `frac` = `tensor_pipe_issued_frac` counts the 3 or 6 bf16 "
                            "piece products the tensor pipe issues per fp32 product (piece_products_per_fp32_product); "
                            "`useful_tflops` = 2*M*N*K / t is the method's own work")
    ranked = [k for k in sorted(kernels, key=lambda k: -kernels[k]["share"]) if "bound" in kernels[k]]
    if ranked:
        k = ranked[0]
        e = kernels[k]
        traffic, src = ncu_traffic(cfg.name, B, k)
        line["roofline"] = {"kernel": k, "bound": e["bound"], "achieved": e["achieved"], "peak": e["peak"], "unit": e["unit"],
                            "frac": e["frac"], "traffic": traffic, "traffic_source": src,
                            "algorithmic": work[k][1], "traffic_unit": "bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum)",
                            "peak_source": peaks["source"], "share_of_step": e["share"]}
    else:
        line["roofline"] = None
    line["path_roofline"] = direction_rooflines(cfg, n, r, args.steps, peaks) if world == 1 else None

    if world == 1 and not args.no_sweep and not (args.streams or args.chunk_bytes):
        # the points north_star and the configs' sweeps name, once each (VERDICT r1 "Next" 2a)
        sweep = []
        for config, streams, chunk_b, label in [
                (4, 65536, 273, "north_star point: configs[3] model (4-layer d=256 bf16) at B = 65,536 streams"),
                (5, 8192, 273, "configs[4] model (8-layer d=512 bf16) at B = 8,192 streams"),
                (5, 64, 273, "configs[4] model at B = 64 (per-stream latency)"),
                (5, 1, 273, "configs[4] model at B = 1 (per-stream latency)"),
                (1, 16, 4096, "configs[0] as it is: 16 chunks x 4 KiB, 1-layer d=64")]:
            # (few streams: no event-bracketed eager batches - they would be most of a step that is pure latency)
            sweep.append(sweep_point(boa, peaks, config, streams, chunk_b, label, sample_every=2 if streams > 1024 else 0))
        line["sweep"] = sweep
        # FX1: the integer pipeline whose containers do not depend on the device, once per point
        line["fx1"] = [fx_point(boa, 2, 4096, 273, "configs[1] model shape at B = 4,096 streams", passes=3),
                       fx_point(boa, 4, 65536, 65, "configs[3] model shape at B = 65,536 streams", passes=3),
                       # the metric's own workload once, no warm-up pass (a pass is 16,383 steps: first-call overheads are noise)
                       fx_point(boa, 2, 4096, 16384, "configs[1] as it is: 64 MiB, 4,096 chunks x 16 KiB (one pass)", passes=1)]
        line["fx1_note"] = ("every step an integer kernel (tcgen05.mma kind::i8 contractions, integer RMSNorm / exp / sigmoid / "
                            "softplus by table, Q12.20 recurrence); logits, tables and containers bit-identical to oracle/fixed.py "
                            "(tests/test_gpu_fixed.py); both directions run the step path")
        if not args.no_largest:
            # the largest single-GPU configuration: configs[3] at 65,536 chunks x 16 KiB = 1 GiB, one pass, no warm-up pass
            # of its own (the sweep point above has run the same model at the same B)
            from paper_2511_11337_b200 import synth
            big = synth.CONFIGS[4]
            m.close()
            del d_in, d_comp, d_out, h_in, h_comp, h_out
            torch.cuda.empty_cache()
            mb = boa.Model(big.weights())
            bn = big.n_bytes
            b_in = torch.frombuffer(bytearray(big.data()), dtype=torch.uint8).to(dev)
            b_comp = torch.empty(boa.compress_bound(bn, big.chunk_bytes), dtype=torch.uint8, device=dev)
            b_out = torch.empty(bn, dtype=torch.uint8, device=dev)
            rb = measure(boa, mb, b_in, big.chunk_bytes, b_comp, b_out, 1, 0, 512)
            kb, _ = kernel_table(boa, big, bn // big.chunk_bytes, rb, peaks)
            rfb = direction_rooflines(big, bn, rb, 1, peaks)
            line["largest_config"] = {"workload": workload_name(big), "baseline_config_index": 3, "passes": 1, "round_trip": "byte-exact",
                                      "value": 2 * bn / MiB / ((rb["tc"] + rb["td"]) / 1e3), "unit": "MiB/s",
                                      "compress_MiBps": rfb["compress"]["achieved_MiBps"], "decompress_MiBps": rfb["decompress"]["achieved_MiBps"],
                                      "decompress_over_ceiling": rfb["decompress"]["frac"], "compress_over_ceiling": rfb["compress"]["frac"],
                                      "bits_per_byte": 8.0 * rb["clen"] / bn, "scan_frac_of_hbm_peak": kb.get("scan", {}).get("frac"),
                                      "kernel_us": {k: round(v["avg_us"], 2) for k, v in kb.items()}, "gpu_launches": rb["launches"]}
            mb.close()
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = time_oracle(cfg)
    else:
        line["cpu_baseline"] = None
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_strong(args, cfg, world, rank, dev, peaks):
    """--scaling strong: ONE input and ONE container over `world` GPUs (P:167 chunks are independent).
    Rank r compresses chunks [lo_r, hi_r) with boa_compress_shard; the parts (first bytes, sizes, payload) are gathered
    on rank 0, which writes the container with boa_container_assemble; the container is broadcast and every rank
    decodes its own chunk range with boa_decompress_shard.  Timed region: all of that, max over ranks."""
    import torch
    import torch.distributed as dist
    from paper_2511_11337_b200 import boa, shard

    n, chunk = cfg.n_bytes, cfg.chunk_bytes
    host = torch.frombuffer(bytearray(cfg.data()), dtype=torch.uint8)      # the same input on every rank (seeded)
    m = boa.Model(cfg.weights())
    d_in = host.to(dev)
    d_out = torch.zeros(n, dtype=torch.uint8, device=dev)

    def one_pass():
        t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True); t2 = torch.cuda.Event(enable_timing=True)
        t0.record()
        blob = shard.compress_sharded(m, d_in, chunk, rank, world, dev)      # the assembled container, on every rank
        t1.record()
        lo, hi = shard.decompress_sharded(m, blob, d_out, rank, world)
        t2.record()
        torch.cuda.synchronize()
        if not torch.equal(d_out[lo:hi], d_in[lo:hi]):
            raise SystemExit("bench.py: sharded round trip is not byte-exact")
        return t0.elapsed_time(t1), t1.elapsed_time(t2), blob.numel()

    for _ in range(args.warmup):
        one_pass()
    shard.barrier(); torch.cuda.synchronize()
    clocks = ClockSampler(dev.index)
    clocks.start()
    tc = td = 0.0
    for _ in range(args.steps):
        a, b, clen = one_pass()
        tc += a; td += b
    shard.barrier()
    clk = clocks.stop()
    total_ms, _ = shard.reduce_stats(tc + td, 0.0, dev)
    tc_max, _ = shard.reduce_stats(tc, 0.0, dev)
    td_max, _ = shard.reduce_stats(td, 0.0, dev)
    if rank == 0:
        line = base_line(args, cfg, world)
        line["value"] = 2.0 * n * args.steps / MiB / (total_ms / 1e3)
        line["ms_per_step"] = total_ms / args.steps
        line["compress_MiBps"] = n * args.steps / MiB / (tc_max / 1e3)
        line["decompress_MiBps"] = n * args.steps / MiB / (td_max / 1e3)
        line["bits_per_byte"] = 8.0 * clen / n
        line["clocks"] = clk
        line["e2e"] = None
        line["gpu_launches"] = None
        line["roofline"] = None
        line["cpu_baseline"] = None
        line["note"] = "strong scaling: one input, one BOA1 container assembled from the ranks' parts (byte-identical to the single-GPU container)"
        print(json.dumps(line))
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
    ap.add_argument("--no-sweep", action="store_true", help="skip the once-only sweep points and the largest configuration")
    ap.add_argument("--no-largest", action="store_true", help="skip the 1 GiB configs[3] pass (about two minutes)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"], help="N > 1: independent replicas (weak) or one input / one container sharded over the ranks (strong)")
    ap.add_argument("--persist-max", type=int, default=-1, help="measurement only: waves up to this many streams run the persistent step kernel (boa_debug_set_persist; -1 = library default, 0 = never)")
    ap.add_argument("--persist-cluster", type=int, default=0, help="measurement only: CTAs per row tile in the persistent step kernel (0 = library default)")
    ap.add_argument("--chain", action="store_true", help="measurement only: chain the dependent contractions of the step path inside one launch (boa_debug_set_chain)")
    ap.add_argument("--pair-tiles", type=int, default=-1, help="measurement only: row-tile threshold from which the step path uses CTA-pair tiles (boa_debug_set_pair_tiles; -1 = library default)")
    ap.add_argument("--streams", type=int, default=0, help="run the config's model with this many chunks (streams per step) ...")
    ap.add_argument("--chunk-bytes", type=int, default=0, help="... of this many bytes each (a sweep point, not the headline workload)")
    ap.add_argument("--fx-only", action="store_true", help="measurement only: one FX1 point (--config, --streams, --chunk-bytes) and nothing else; prints that entry")
    args = ap.parse_args()
    from paper_2511_11337_b200 import synth
    if args.fx_only:
        import torch
        from paper_2511_11337_b200 import boa
        if not torch.cuda.is_available():
            raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
        print(json.dumps(fx_point(boa, args.config, args.streams or 4096, args.chunk_bytes or 273, "--fx-only")))
        return
    cfg = synth.CONFIGS[args.config]
    if args.streams or args.chunk_bytes:
        chunk = args.chunk_bytes or cfg.chunk_bytes
        streams = args.streams or cfg.n_bytes // cfg.chunk_bytes
        cfg = dataclasses.replace(cfg, name=f"{cfg.name}[sweep: {streams} streams x {chunk} B]", n_bytes=streams * chunk, chunk_bytes=chunk)
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
