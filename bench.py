"""bench.py — headline measurement of the TurboESM hot path on B200 (contract: DESIGN.md "Measurement").

Workload: BASELINE.json:configs[2] — ESM-2-650M-shaped batched decode: 33 layers x batch 32 x 20 heads,
head_dim 64, 1024 cached tokens, fp16 Student-t(4) activations with 2 outlier channels per head; every
decode step appends one quantised token per head (tq_append) and runs the fused decode attention
(tq_decode_attn) for every layer.  A "step" is one model decode step = 33 x (append + decode).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--layers L]

value     : cached token-heads attended per second (L*B*H*T per step / step time), inputs resident in HBM,
            the 33-layer step replayed as one CUDA graph.
e2e       : same metric through tq_decode_model_step_host with pinned HOST q/k/v/out buffers (copies inside).
roofline  : fused decode kernel, algorithmic packed bytes (62 B per cached token-head) / its average launch
            duration measured live with CUDA events, against MEASURED_PEAKS.json hbm_gbs.
cpu_baseline : the CPU oracle (oracle/, as it stands) timed on this box's host cores on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

from paper_2603_26110_b200 import workloads as W

METRIC = "fused 3-bit decode-attn cached tokens/s"
UNIT = "cached token-heads/s"
FALLBACK_HBM_GBS = 6650.0  # B200_PROFILING.md fallback
NCU_DRAM_BYTES_PER_LAUNCH = 42.63e6  # decode_main_kernel, one ncu --set full capture (profiles/r01b_decode_main_full.md)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def torch_activations(w: W.Workload, layer: int, shape, device, gen):
    """Synthetic K/V of one layer drawn on the device: Student-t(4) = N / sqrt(chi2_4 / 4), per-head outlier
    channels scaled (same recipe as workloads.layer_activations; the numpy version feeds the parity tests)."""
    import torch

    ch = W.outlier_channels(w)[layer]
    scale = np.ones((w.n_heads, w.head_dim), np.float32)
    for h in range(w.n_heads):
        scale[h, ch[h]] = w.outlier_scale
    # [H, d] -> broadcast over [B, H, (T,) d]
    scale = torch.from_numpy(scale).to(device).view((1, w.n_heads) + (1,) * (len(shape) - 3) + (w.head_dim,))
    out = []
    for _ in range(2):
        x = torch.randn(shape, device=device, generator=gen)
        if w.dist == "student_t4":
            chi = torch.randn((4,) + tuple(shape), device=device, generator=gen).square_().sum(0)
            x = x / torch.sqrt(chi / 4.0)
        x = x * scale
        out.append(x.to(torch.float16 if w.dtype == "f16" else torch.float32).contiguous())
    return out


# ------------------------------------------------------------------------------------------ reference arm
def run_reference(args, w: W.Workload):
    """--impl reference: the CPU oracle, as it stands, on this box's host cores.  Each step decodes a bounded
    sample of the workload (a few batch entries of one layer)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import tq_oracle as O
    import math

    O.build()
    sb = 2  # batch entries per sampled step
    ws = w.scaled(n_layers=1, batch=sb)
    pi_k, pi_v = W.rotations(ws)
    S = W.sketch(ws)
    lut = O.lloyd_max_gauss(1.0 / math.sqrt(w.head_dim), 8)[0].astype(np.float32)
    luts = np.tile(lut, (w.n_heads, 1))
    k, v = W.layer_activations(ws, 0)
    t0 = time.perf_counter()
    can = O.quantize_pack(k, v, pi_k[0], pi_v[0], luts, luts, S)
    tq_s = time.perf_counter() - t0
    q = W.queries(ws, 0)
    sl = np.full(sb, w.seq, np.int32)
    for _ in range(args.warmup):
        O.decode_attn(q, sl - 1, sl, pi_k[0], pi_v[0], luts, luts, S, can)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        O.decode_attn(q, sl - 1, sl, pi_k[0], pi_v[0], luts, luts, S, can)
    dt = time.perf_counter() - t0
    th = sb * w.n_heads * w.seq * args.steps
    value = th / dt
    sample = f"decode of {sb} batch entries x {w.n_heads} heads x {w.seq} tokens of one layer per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample,
                         "quantize_pack_vectors_per_s": 2 * sb * w.n_heads * w.seq / tq_s},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------ CPU baseline leg
def cpu_baseline(w: W.Workload):
    """The oracle as it stands on this box's host cores, bounded sample (rank 0, N = 1 only)."""
    from oracle import tq_oracle as O
    import math

    O.build()
    sb = 4
    ws = w.scaled(n_layers=1, batch=sb)
    pi_k, pi_v = W.rotations(ws)
    S = W.sketch(ws)
    lut = O.lloyd_max_gauss(1.0 / math.sqrt(w.head_dim), 8)[0].astype(np.float32)
    luts = np.tile(lut, (w.n_heads, 1))
    k, v = W.layer_activations(ws, 0)
    t0 = time.perf_counter()
    can = O.quantize_pack(k, v, pi_k[0], pi_v[0], luts, luts, S)
    tq_s = time.perf_counter() - t0
    q = W.queries(ws, 0)
    sl = np.full(sb, w.seq, np.int32)
    O.decode_attn(q, sl - 1, sl, pi_k[0], pi_v[0], luts, luts, S, can)
    reps, t0 = 0, time.perf_counter()
    while time.perf_counter() - t0 < 8.0 and reps < 200:
        O.decode_attn(q, sl - 1, sl, pi_k[0], pi_v[0], luts, luts, S, can)
        reps += 1
    dt = time.perf_counter() - t0
    nvec = 2 * sb * w.n_heads * w.seq
    in_bytes = nvec * w.head_dim * 2
    return {
        "value": sb * w.n_heads * w.seq * reps / dt, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
        "sample": f"{reps} decode passes over {sb} batch entries x {w.n_heads} heads x {w.seq} tokens of one layer "
                  f"(fp64, OpenMP over units); quantize/pack of the same {nvec} vectors once",
        "quantize_pack_gbs": (in_bytes + nvec / 2 * 62) / tq_s / 1e9,
        "quantize_pack_s": tq_s,
    }


# ------------------------------------------------------------------------------------------ our arm
def max_over_ranks(values, world: int, device):
    """Element-wise MAX over ranks of a list of per-rank times (the only cross-rank traffic of the bench: the path
    shards by batch with no data-path collective)."""
    import torch
    import torch.distributed as dist

    t = torch.tensor(list(values), device=device, dtype=torch.float64)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_value(tok_heads_per_rank: int, world: int, ms_max: float) -> float:
    """Weak scaling: every rank attends the same number of cached token-heads; the job's rate uses the slowest rank."""
    return world * tok_heads_per_rank / (ms_max * 1e-3)


def run_ours(args, w: W.Workload):
    import torch
    import torch.distributed as dist

    from paper_2603_26110_b200 import binding as tq
    from paper_2603_26110_b200 import build as tqbuild

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        tqbuild.build()
    if world > 1:
        dist.barrier()
    tq.lib()
    dev = torch.device("cuda", local)

    L, B, H, d, T0 = args.layers, w.batch, w.n_heads, w.head_dim, w.seq
    max_seq = T0 + 128
    shape = tq.make_shape(L, B, H, d, max_seq, w.rope_base, 0)
    wl = w.scaled(n_layers=L)
    cal = tq.tq_calibrate_host(shape, 1, seed=w.seed + rank)  # QR-of-Gaussian PI per (layer, head), Lloyd-Max LUT, S
    params = tq.Params(cal, dev)
    cache = tq.Cache(shape, dev)
    ws = tq.Workspace(shape, 1, dev)
    gen = torch.Generator(device=dev)
    gen.manual_seed(w.seed + 1000 * rank)
    dt_code = tq.TQ_F16
    stream = torch.cuda.Stream(dev)

    # ---- prefill: quantize/pack every layer (timed separately: quantize/pack GB/s)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    q_ms = []
    with torch.cuda.stream(stream):
        for layer in range(L):
            k, v = torch_activations(wl, layer, (B, H, T0, d), dev, gen)
            e0, e1 = ev(), ev()
            e0.record(stream)
            tq.tq_quantize_pack(shape, params, cache, layer, k, v, 0, stream)
            e1.record(stream)
            e1.synchronize()
            q_ms.append(e0.elapsed_time(e1))
            del k, v
    q_bytes = 2 * B * H * T0 * d * 2 + B * H * T0 * 62
    quant_gbs = q_bytes / (statistics.median(q_ms) * 1e-3) / 1e9

    # ---- per-step inputs, resident on the device: [L][B][H][d]
    qs, kn, vn = [], [], []
    for layer in range(L):
        a, b_ = torch_activations(wl, layer, (B, H, d), dev, gen)
        c_, _ = torch_activations(wl, layer, (B, H, d), dev, gen)
        qs.append(a), kn.append(b_), vn.append(c_)
    qs, kn, vn = torch.stack(qs), torch.stack(kn), torch.stack(vn)
    outs = torch.empty_like(qs)

    def reset_len():
        cache.seq_len.fill_(T0)

    def one_step():
        for layer in range(L):  # tq_decode_step == tq_append followed by tq_decode_attn, two launches per layer
            tq.tq_decode_step(shape, params, cache, layer, qs[layer], kn[layer], vn[layer], outs[layer], ws, max_seq,
                              stream)

    # ---- capture one model decode step as a CUDA graph (seq_len lives on the device, so it replays)
    with torch.cuda.stream(stream):
        reset_len()
        one_step()  # warm: module load, attribute setting
        stream.synchronize()
        n0 = tq.tq_launch_count()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            one_step()
        launches_per_step = tq.tq_launch_count() - n0
    torch.cuda.synchronize()

    steps_per_fill = 100  # capacity: T0 .. T0+127

    def run_steps(n, timed):
        """n graph replays; seq_len is rewound every 100 steps so the cache never overflows."""
        done, total_ms, tok_heads = 0, 0.0, 0
        while done < n:
            chunk = min(steps_per_fill, n - done)
            with torch.cuda.stream(stream):
                reset_len()
                e0, e1 = ev(), ev()
                e0.record(stream)
                for _ in range(chunk):
                    graph.replay()
                e1.record(stream)
            e1.synchronize()
            total_ms += e0.elapsed_time(e1)
            # step i (0-based) attends T0 + i + 1 tokens
            tok_heads += L * B * H * sum(T0 + i + 1 for i in range(chunk))
            done += chunk
        return total_ms, tok_heads

    run_steps(max(args.warmup, 3), False)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ms, tok_heads = run_steps(args.steps, True)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    assert int(cache.status.item()) == 0, "an append was refused during the timed region"

    # ---- live duration of the decode call (query prep + streaming kernel) measured with CUDA events on
    #      `stream`: one tq_decode_attn per layer over all L layer caches (L x 40.6 MB, larger than L2),
    #      captured as a CUDA graph so that the host's launch cost does not bound the measurement
    with torch.cuda.stream(stream):
        reset_len()

        def decode_all_layers():
            for layer in range(L):
                tq.tq_decode_attn(shape, params, cache, layer, 1, qs[layer:layer + 1], outs[layer:layer + 1], ws, None,
                                  max_seq, stream)

        decode_all_layers()
        stream.synchronize()
        dgraph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(dgraph, stream=stream):
            decode_all_layers()
        dec_ms = []
        for it in range(6):
            e0, e1 = ev(), ev()
            e0.record(stream)
            dgraph.replay()
            e1.record(stream)
            e1.synchronize()
            if it > 0:
                dec_ms.append(e0.elapsed_time(e1) / L)
    dec_bytes = B * H * T0 * 62
    dec_s = statistics.mean(dec_ms) * 1e-3

    # ---- the dominant kernel alone (decode_main_kernel): the same per-layer calls with the library's measurement hook
    #      on (only the streaming kernel is launched, the rotated queries of the calls above are still in the
    #      per-layer workspaces), one launch per layer cache, replayed from a graph between one CUDA event pair
    with torch.cuda.stream(stream):
        wss = [tq.Workspace(shape, 1, dev) for _ in range(L)]  # one workspace per layer keeps every layer's q'' alive

        def decode_all_layers_ws():
            for layer in range(L):
                tq.tq_decode_attn(shape, params, cache, layer, 1, qs[layer:layer + 1], outs[layer:layer + 1], wss[layer],
                                  None, max_seq, stream)

        decode_all_layers_ws()  # ordinary calls: query preparation + streaming kernel
        stream.synchronize()
        tq.tq_profile_decode_main_only(True)
        decode_all_layers_ws()
        stream.synchronize()
        mgraph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(mgraph, stream=stream):
            decode_all_layers_ws()
        tq.tq_profile_decode_main_only(False)
        main_ms = []
        for it in range(6):
            e0, e1 = ev(), ev()
            e0.record(stream)
            mgraph.replay()
            e1.record(stream)
            e1.synchronize()
            if it > 0:
                main_ms.append(e0.elapsed_time(e1) / L)
    main_s = statistics.mean(main_ms) * 1e-3

    # ---- end to end through the host-buffer call: pinned q/k/v in, out back, every layer of every step
    e2e_steps = max(3, min(args.steps, 20))
    staging = torch.zeros(tq.tq_model_step_staging_bytes(shape, dt_code, L) + 256, dtype=torch.uint8, device=dev)
    staging = staging[(-staging.data_ptr()) % 256:]
    qh, kh, vh = qs.cpu().pin_memory(), kn.cpu().pin_memory(), vn.cpu().pin_memory()
    oh = torch.empty_like(qh).pin_memory()

    def e2e_step():  # one model decode step: pinned q/k/v of all L layers in, L x (append + decode), outputs back, sync
        tq.tq_decode_model_step_host(shape, params, cache, 0, L, qh, kh, vh, oh, staging, ws, max_seq, stream)

    with torch.cuda.stream(stream):
        reset_len()
        e2e_step()
        stream.synchronize()
        reset_len()
        stream.synchronize()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
        stream.synchronize()
        e2e_s = time.perf_counter() - t0
    e2e_tok = L * B * H * sum(T0 + i + 1 for i in range(e2e_steps))
    vec_bytes = B * H * d * 2

    # ---- aggregate over ranks (max time)
    ms_max, e2e_max = max_over_ranks([ms, e2e_s], world, dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    peak, peak_src = measured_peaks()
    achieved = dec_bytes / main_s / 1e9
    value = whole_job_value(tok_heads, world, ms_max)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {
            "workload": f"{w.name} (BASELINE.json configs[2]) x {L} layers: batch {B} x {H} heads x d {d}, "
                        f"{T0}+ cached tokens, fp16 Student-t(4) + 2 outlier channels x15, append + decode per layer per step",
            "layers": L, "batch_per_gpu": B, "heads": H, "head_dim": d, "cached_tokens": T0, "io_dtype": "f16",
            "l2": f"inputs larger than L2: {L} layer caches x {B*H*T0*62/1e6:.1f} MB are cycled every step",
            "cuda_graph": True, "bytes_per_token_head": 62,
            "us_per_layer_step": 1e3 * ms_max / args.steps / L,
            "packed_gbs_whole_step": value / world * 62 / 1e9,
            "decode_call_us_live": dec_s * 1e6, "decode_call_packed_gbs": dec_bytes / dec_s / 1e9,
            "decode_main_kernel_us_live": main_s * 1e6,
            "quantize_pack_gbs": quant_gbs, "quantize_pack_ms_per_layer": statistics.median(q_ms),
            "parallelism": f"dp{world} (independent batches, no collective)",
        },
        "clocks": clocks,
        "e2e": {"value": world * e2e_tok / e2e_max, "unit": UNIT, "h2d_bytes_per_step": 3 * L * vec_bytes,
                "d2h_bytes_per_step": L * vec_bytes, "steps": e2e_steps},
        "gpu_launches": int(launches_per_step * args.steps),
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": NCU_DRAM_BYTES_PER_LAUNCH, "kernel": "decode_main_kernel<64, __half>",
                     "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum per launch, profiles/r01b_decode_main_full.md",
                     "peak_source": peak_src, "bytes_per_launch": dec_bytes},
    }
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(w)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--layers", type=int, default=33, help="ESM-2-650M has 33 layers")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    w = W.CONFIGS["cfg2_650m_batch32"]
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
