"""bench.py — headline measurement of the TurboESM hot path on B200 (contract: DESIGN.md "Measurement").

Default workload: BASELINE.json:configs[2] — ESM-2-650M-shaped batched decode: 33 layers x batch 32 x 20 heads,
head_dim 64, 1024 cached tokens, fp16 Student-t(4) activations with 2 outlier channels per head; every decode step
appends one quantised token per head and runs the fused decode attention for every layer.  A "step" is one model
decode step = 33 x (append + decode) through tq_decode_model_step.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--layers L] [--config cfg1|cfg2|cfg3|cfg4]

value     : cached token-heads attended per second (L*B*H*T per step / step time), inputs resident in HBM,
            the step replayed as one CUDA graph.
e2e       : same metric through tq_decode_model_step_host with pinned HOST q/k/v/out buffers (copies inside).
value_sequential : the same step in the order a model must run it (tq_decode_step layer after layer); `value` is the
            run-ahead form, an upper bound a transformer cannot call.
roofline  : fused decode kernel, algorithmic packed bytes (62 B per cached token-head) / its average launch
            duration measured live with CUDA events, against MEASURED_PEAKS.json hbm_gbs; `frac` is taken on zero
            queries (flat softmax: no value work skipped), `frac_peaked_inputs` on the configs[2] queries.
cpu_baseline : the CPU oracle (oracle/, as it stands) timed on this box's host cores on a bounded sample.
--config cfg1|cfg3|cfg4 : the other BASELINE.json configs (prefill quantize/pack GB/s and decode tokens/s), one line each.
"""
from __future__ import annotations

import argparse
import glob
import json
import os
import re
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
V_QJL = 0  # --v-qjl: the V-side residual sketch, +10 / +18 bytes per token-head
CONFIG_NAMES = {"cfg1": "cfg1_650m_step", "cfg2": "cfg2_650m_batch32", "cfg3": "cfg3_long_splitk", "cfg4": "cfg4_15b_heads"}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def kernel_source_sha(name: str = "tq_decode.cu") -> str:
    """sha256 (first 12 hex digits) of a kernel source file as it is now (the GPU box has no .git to ask)."""
    import hashlib

    path = os.path.join(ROOT, "paper_2603_26110_b200", "csrc", name)
    return hashlib.sha256(open(path, "rb").read()).hexdigest()[:12]


def ncu_traffic(kernel_tag: str):
    """DRAM bytes per launch of the dominant kernel from the newest committed `ncu --set full` summary
    (profiles/r*_<kernel_tag>_full.md, line `dram_bytes_per_launch: N`); None when no capture exists.  This is a number
    READ FROM A COMMITTED FILE, not measured by this run: the summary names the source it was captured from
    (`kernel_source_sha256: <12 hex digits of tq_decode.cu>`), and the third element says whether that is still the
    source this run was built from (True / False, None when the summary does not say)."""
    best = None
    for f in sorted(glob.glob(os.path.join(ROOT, "profiles", f"r*_{kernel_tag}_full.md"))):
        text = open(f).read()
        m = re.search(r"dram_bytes_per_launch:\s*([0-9.eE+]+)", text)
        if m:
            sha = re.search(r"kernel_source_sha256:\s*([0-9a-f]{12})", text)
            best = (float(m.group(1)), os.path.relpath(f, ROOT), (sha.group(1) == kernel_source_sha()) if sha else None)
    return best


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
                                          "--format=csv,noheader,nounits", "-lms", "20"],
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


def bytes_per_token_head(d: int) -> int:
    return 62 if d == 64 else 118


# ------------------------------------------------------------------------------------------ oracle legs
def oracle_sample(w: W.Workload, sb: int):
    from oracle import tq_oracle as O
    import math

    O.build()
    ws = w.scaled(n_layers=1, batch=sb)
    pi_k, pi_v = W.rotations(ws)
    S = W.sketch(ws)
    lut = O.lloyd_max_gauss(1.0 / math.sqrt(w.head_dim), 8)[0].astype(np.float32)
    luts = np.tile(lut, (w.n_heads, 1))
    k, v = W.layer_activations(ws, 0)
    q = W.queries(ws, 0)
    return O, ws, pi_k, pi_v, S, luts, k, v, q


def run_reference(args, w: W.Workload):
    """--impl reference: the CPU oracle, as it stands, on this box's host cores.  Each step decodes a bounded
    sample of the workload (a few batch entries of one layer)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    sb = 2  # batch entries per sampled step
    tcap = min(w.seq, 4096)  # bounded sample of long contexts
    O, ws, pi_k, pi_v, S, luts, k, v, q = oracle_sample(w.scaled(seq=tcap), sb)
    t0 = time.perf_counter()
    can = O.quantize_pack(k, v, pi_k[0], pi_v[0], luts, luts, S)
    tq_s = time.perf_counter() - t0
    sl = np.full(sb, tcap, np.int32)
    for _ in range(args.warmup):
        O.decode_attn(q, sl - 1, sl, pi_k[0], pi_v[0], luts, luts, S, can)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        O.decode_attn(q, sl - 1, sl, pi_k[0], pi_v[0], luts, luts, S, can)
    dt = time.perf_counter() - t0
    th = sb * w.n_heads * tcap * args.steps
    value = th / dt
    sample = f"decode of {sb} batch entries x {w.n_heads} heads x {tcap} tokens of one layer per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample,
                         "quantize_pack_vectors_per_s": 2 * sb * w.n_heads * tcap / tq_s},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def cpu_baseline(w: W.Workload):
    """The oracle as it stands on this box's host cores, bounded sample (rank 0, N = 1 only): all cores (OpenMP over
    units) and one thread."""
    sb = 4
    tcap = min(w.seq, 2048)
    O, ws, pi_k, pi_v, S, luts, k, v, q = oracle_sample(w.scaled(seq=tcap), sb)
    t0 = time.perf_counter()
    can = O.quantize_pack(k, v, pi_k[0], pi_v[0], luts, luts, S)
    tq_s = time.perf_counter() - t0
    sl = np.full(sb, tcap, np.int32)
    ncores = O.num_threads()

    def timed(budget_s):
        O.decode_attn(q, sl - 1, sl, pi_k[0], pi_v[0], luts, luts, S, can)
        reps, t0 = 0, time.perf_counter()
        while time.perf_counter() - t0 < budget_s and reps < 200:
            O.decode_attn(q, sl - 1, sl, pi_k[0], pi_v[0], luts, luts, S, can)
            reps += 1
        return sb * w.n_heads * tcap * reps / (time.perf_counter() - t0), reps

    v_all, reps = timed(6.0)
    O.set_num_threads(1)
    try:
        v_one, reps1 = timed(4.0)
    finally:
        O.set_num_threads(ncores)
    nvec = 2 * sb * w.n_heads * tcap
    in_bytes = nvec * w.head_dim * 2
    return {
        "value": v_all, "unit": UNIT, "cores": ncores, "kind": "oracle",
        "sample": f"{reps} decode passes over {sb} batch entries x {w.n_heads} heads x {tcap} tokens of one layer "
                  f"(fp64, OpenMP over units); quantize/pack of the same {nvec} vectors once",
        "single_thread_value": v_one, "single_thread_passes": reps1,
        "quantize_pack_gbs": (in_bytes + nvec / 2 * bytes_per_token_head(w.head_dim)) / tq_s / 1e9,
        "quantize_pack_s": tq_s,
    }


# ------------------------------------------------------------------------------------------ two-step GPU baseline
def two_step_baseline(rig, layer: int, q, out_fused, T: int, reps: int = 6):
    """the paper's comparison system restated on this box ("Standard PyTorch
    implementations dequantize the entire KV cache into FP16 tensors before computing attention, requiring two full
    passes over global memory"; Table 6: 1.19 -> 0.61 ms, 1.96x on its hardware).  Plain PyTorch GPU
    ops on the CANONICAL packed planes of one layer cache (the paper's own vectorised unpack): unpack
    3-bit codes -> LUT gather -> residual-sketch correction -> scale by the stored norms -> fp16 K and V tensors in HBM,
    then torch SDPA with the rotated query, then PI_V^T.  Not part of the product; nothing in libtq.so is on this path
    except the one-off export of the canonical planes (outside the timed region).
    Returns (microseconds per layer call, cosine of its output against the fused kernel's)."""
    import math

    import torch

    tq, dev, B, H, d = rig.tq, rig.dev, rig.B, rig.H, rig.d
    m = d
    with torch.cuda.stream(rig.stream):
        planes = tq.tq_cache_export_canonical(rig.shape, rig.cache, layer, T, stream=rig.stream)
        P = rig.params.t
        pi_k, pi_v = P["pi_k"][layer], P["pi_v"][layer]          # [H, d, d]
        lut_k, lut_v, S = P["lut_k"][layer], P["lut_v"][layer], P["S"]  # [H, 8], [H, 8], [m, d]
        cs = P["rope_cs"][T - 1]                                 # [d/2, 2] (the query sits at the newest position)
        shifts = torch.arange(8, device=dev, dtype=torch.int32) * 3
        bit = torch.arange(8, device=dev, dtype=torch.uint8)
        c_qjl = math.sqrt(math.pi / 2.0) / m
        hidx = torch.arange(H, device=dev).view(1, H, 1, 1)

        def unpack_codes(codes):  # [B, H, T, 3d/8] uint8 -> [B, H, T, d] int64, the paper's snippet on 24-bit groups
            g = codes.view(B, H, T, d // 8, 3).to(torch.int32)
            packed = g[..., 0] | (g[..., 1] << 8) | (g[..., 2] << 16)
            return ((packed.unsqueeze(-1) >> shifts) & 0x7).reshape(B, H, T, d).long()

        def f16_planes(x):  # binary16 bit planes -> float32
            return x.view(torch.float16).float()

        def step():
            # pass 1: dequantise the whole cache to fp16 tensors
            kq = lut_k[hidx.expand(B, H, T, d), unpack_codes(planes["k_codes"])]
            sig = ((planes["k_signs"].unsqueeze(-1) >> bit) & 1).reshape(B, H, T, m).float() * 2.0 - 1.0
            corr = torch.matmul(sig, S) * (c_qjl * f16_planes(planes["k_rnorm"])).unsqueeze(-1)
            k16 = ((kq + corr) * f16_planes(planes["k_norm"]).unsqueeze(-1)).half()
            v16 = (lut_v[hidx.expand(B, H, T, d), unpack_codes(planes["v_codes"])] * f16_planes(planes["v_norm"]).unsqueeze(-1)).half()
            # pass 2: attention over the fp16 tensors with the rotated query, then PI_V^T
            qf = q.float().view(B, H, d // 2, 2)
            qr = torch.stack((qf[..., 0] * cs[:, 0] - qf[..., 1] * cs[:, 1], qf[..., 0] * cs[:, 1] + qf[..., 1] * cs[:, 0]), -1).view(B, H, d)
            qrot = torch.einsum("hik,bhk->bhi", pi_k, qr).half().unsqueeze(2)
            o = torch.nn.functional.scaled_dot_product_attention(qrot, k16, v16).squeeze(2).float()
            return torch.einsum("hki,bhk->bhi", pi_v, o)

        out = step()
        rig.stream.synchronize()
        ts = []
        for _ in range(reps):
            e0, e1 = rig.ev(), rig.ev()
            e0.record(rig.stream)
            out = step()
            e1.record(rig.stream)
            e1.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e3)
        a, b_ = out.reshape(-1, d).double(), out_fused.reshape(-1, d).double()
        cos = float(torch.mean(torch.sum(a * b_, -1) / (a.norm(dim=-1) * b_.norm(dim=-1))))
    return statistics.median(ts), cos


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


class Rig:
    """Device-side state shared by the measurement legs of one workload."""

    def __init__(self, w: W.Workload, L: int, max_seq: int, rank: int, local: int):
        import torch
        from paper_2603_26110_b200 import binding as tq

        self.torch, self.tq, self.w, self.L = torch, tq, w, L
        self.dev = torch.device("cuda", local)
        self.B, self.H, self.d, self.T0 = w.batch, w.n_heads, w.head_dim, w.seq
        self.max_seq = max_seq
        self.shape = tq.make_shape(L, self.B, self.H, self.d, max_seq, w.rope_base, 0, v_qjl=V_QJL)
        self.wl = w.scaled(n_layers=L)
        cal = tq.tq_calibrate_host(self.shape, 1, seed=w.seed + rank)  # QR-of-Gaussian PI per (layer, head), Lloyd-Max LUT, S
        self.params = tq.Params(cal, self.dev)
        self.cache = tq.Cache(self.shape, self.dev)
        self.gen = torch.Generator(device=self.dev)
        self.gen.manual_seed(w.seed + 1000 * rank)
        self.stream = torch.cuda.Stream(self.dev)
        self.bpt = tq.tq_cache_bytes_per_token_head(self.shape)  # 62 | 118; 72 | 136 with the V-side sketch

    def ev(self):
        return self.torch.cuda.Event(enable_timing=True)

    def prefill(self):
        """tq_quantize_pack of T0 tokens into every layer cache, each launch timed; returns (ms list, bytes per layer)."""
        q_ms = []
        with self.torch.cuda.stream(self.stream):
            for layer in range(self.L):
                k, v = torch_activations(self.wl, layer, (self.B, self.H, self.T0, self.d), self.dev, self.gen)
                e0, e1 = self.ev(), self.ev()
                e0.record(self.stream)
                self.tq.tq_quantize_pack(self.shape, self.params, self.cache, layer, k, v, 0, self.stream)
                e1.record(self.stream)
                e1.synchronize()
                q_ms.append(e0.elapsed_time(e1))
                del k, v
        esz = 2 if self.w.dtype == "f16" else 4
        q_bytes = 2 * self.B * self.H * self.T0 * self.d * esz + self.B * self.H * self.T0 * self.bpt
        return q_ms, q_bytes

    def step_inputs(self):
        qs, kn, vn = [], [], []
        for layer in range(self.L):
            a, b_ = torch_activations(self.wl, layer, (self.B, self.H, self.d), self.dev, self.gen)
            c_, _ = torch_activations(self.wl, layer, (self.B, self.H, self.d), self.dev, self.gen)
            qs.append(a), kn.append(b_), vn.append(c_)
        t = self.torch
        return t.stack(qs), t.stack(kn), t.stack(vn)

    def graph_us(self, body, per: int, reps: int = 6, before=None):
        """Capture body() as a CUDA graph on self.stream and return the mean replay time / per, in microseconds."""
        t = self.torch
        with t.cuda.stream(self.stream):
            if before:
                before()
            body()
            self.stream.synchronize()
            g = t.cuda.CUDAGraph()
            with t.cuda.graph(g, stream=self.stream):
                body()
            ts = []
            for it in range(reps):
                if before:
                    before()
                e0, e1 = self.ev(), self.ev()
                e0.record(self.stream)
                g.replay()
                e1.record(self.stream)
                e1.synchronize()
                if it > 0:
                    ts.append(e0.elapsed_time(e1) / per * 1e3)
        return statistics.mean(ts)


def init_dist():
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2603_26110_b200 import binding as tq
    from paper_2603_26110_b200 import build as tqbuild

    if rank == 0:
        tqbuild.build()
    if world > 1:
        dist.barrier()
    tq.lib()
    return rank, world, local


def run_cfg2(args, w: W.Workload):
    import torch
    import torch.distributed as dist

    rank, world, local = init_dist()
    from paper_2603_26110_b200 import binding as tq

    L = args.layers
    rig = Rig(w, L, w.seq + 128, rank, local)
    B, H, d, T0, dev, stream, shape, params, cache = rig.B, rig.H, rig.d, rig.T0, rig.dev, rig.stream, rig.shape, rig.params, rig.cache
    max_seq = rig.max_seq
    dt_code = tq.TQ_F16

    # ---- prefill: quantize/pack every layer (timed separately: quantize/pack GB/s)
    q_ms, q_bytes = rig.prefill()
    q_ms = q_ms[1:] if len(q_ms) > 1 else q_ms  # the first launch also loads the module
    quant_gbs = q_bytes / (statistics.median(q_ms) * 1e-3) / 1e9

    # ---- per-step inputs, resident on the device: [L][B][H][d]
    qs, kn, vn = rig.step_inputs()
    outs = torch.empty_like(qs)
    wsL = tq.Workspace(shape, L, dev)
    ws1 = tq.Workspace(shape, 1, dev)

    def reset_len():
        cache.seq_len.fill_(T0)

    def one_step():  # one model decode step: append + fused decode attention for every layer
        tq.tq_decode_model_step(shape, params, cache, 0, L, qs, kn, vn, outs, wsL, max_seq, stream)

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

    def run_steps(n):
        """n graph replays; seq_len is rewound every 100 steps so the cache never overflows."""
        done, total_ms, tok_heads = 0, 0.0, 0
        while done < n:
            chunk = min(steps_per_fill, n - done)
            with torch.cuda.stream(stream):
                reset_len()
                e0, e1 = rig.ev(), rig.ev()
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

    run_steps(max(args.warmup, 3))
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ms, tok_heads = run_steps(args.steps)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    assert int(cache.status.item()) == 0, "an append was refused during the timed region"

    dec_bytes = B * H * T0 * rig.bpt  # algorithmic packed bytes of one streaming-kernel launch at T0 tokens

    # ---- the same step through the stepper with DEVICE buffers (three-branch graph: the prep kernels of later layer
    #      chunks run beside the streaming chain)
    stepper_dev = tq.HostStepper(shape, params, cache, 0, L, qs, kn, vn, outs, None, wsL, max_seq, args.e2e_chunks)
    with torch.cuda.stream(stream):
        reset_len()
        for _ in range(3):
            stepper_dev.launch(stream)
        reset_len()
        e0, e1 = rig.ev(), rig.ev()
        e0.record(stream)
        n_st = min(args.steps, steps_per_fill)
        for _ in range(n_st):
            stepper_dev.launch(stream)
        e1.record(stream)
        e1.synchronize()
    stepper_ms = e0.elapsed_time(e1) / n_st
    stepper_value = L * B * H * sum(T0 + i + 1 for i in range(n_st)) / n_st / (stepper_ms * 1e-3)
    stepper_dev.close()

    # ---- the same work as a real model must order it: tq_decode_step layer by layer (append + query prep kernel, then the
    #      streaming kernel, each layer waiting for the one before)
    def seq_step():
        for layer in range(L):
            tq.tq_decode_step(shape, params, cache, layer, qs[layer], kn[layer], vn[layer], outs[layer], ws1, max_seq, stream)

    seq_us = rig.graph_us(seq_step, L, before=reset_len)

    # ---- the decode call alone (query prep + streaming kernel), one tq_decode_attn per layer cache
    def decode_all_layers():
        for layer in range(L):
            tq.tq_decode_attn(shape, params, cache, layer, 1, qs[layer:layer + 1], outs[layer:layer + 1], ws1, None, max_seq, stream)

    reset_len()
    call_us = rig.graph_us(decode_all_layers, L)

    # ---- the dominant kernel (decode_main_kernel) with the library's measurement hook on (query operands of the preceding
    #      ordinary call are re-used): (a) as the model step launches it — one launch per layer cache, a run-ahead chain,
    #      plus the one finish kernel; (b) one launch per layer cache, each waiting for the one before (isolated launches)
    with torch.cuda.stream(stream):
        reset_len()
        one_step()
        stream.synchronize()
    reset_len()
    tq.tq_profile_decode_main_only(1)
    try:
        chain_finish_us = rig.graph_us(one_step, L)   # streaming launches + the one finish kernel
        tq.tq_profile_decode_main_only(2)
        chain_us = rig.graph_us(one_step, L)          # the streaming launches alone: the dominant kernel
    finally:
        tq.tq_profile_decode_main_only(0)
    # ---- the same chain with a FLAT softmax (queries = 0: every logit equal, every cached value contributes).  On the
    #      configs[2] inputs the softmax is extremely peaked and the kernel skips the value MMAs of 16-token halves whose
    #      weights underflow to exactly 0; the flat case is the other end: all of the work, every tile
    qz = torch.zeros_like(qs)

    def flat_step():
        tq.tq_decode_model_step(shape, params, cache, 0, L, qz, kn, vn, outs, wsL, max_seq, stream)

    with torch.cuda.stream(stream):
        reset_len()
        flat_step()
        stream.synchronize()
    reset_len()
    tq.tq_profile_decode_main_only(2)
    try:
        chain_flat_us = rig.graph_us(flat_step, L)
    finally:
        tq.tq_profile_decode_main_only(0)
    wss = [tq.Workspace(shape, 1, dev) for _ in range(L)]  # one workspace per layer keeps every layer's operands alive

    def decode_all_layers_ws():
        for layer in range(L):
            tq.tq_decode_attn(shape, params, cache, layer, 1, qs[layer:layer + 1], outs[layer:layer + 1], wss[layer], None,
                              max_seq, stream)

    with torch.cuda.stream(stream):
        decode_all_layers_ws()
        stream.synchronize()
    tq.tq_profile_decode_main_only(True)
    try:
        iso_us = rig.graph_us(decode_all_layers_ws, L)
    finally:
        tq.tq_profile_decode_main_only(False)

    # ---- the paper's comparison system on this box: PyTorch two-step path (dequantise to fp16, then attend) on layer 0
    two_step = None
    if not args.no_two_step and not V_QJL:
        with torch.cuda.stream(stream):
            reset_len()
            tq.tq_decode_attn(shape, params, cache, 0, 1, qs[0:1], outs[0:1], ws1, None, max_seq, stream)
            stream.synchronize()
        two_step = two_step_baseline(rig, 0, qs[0], outs[0], T0)

    # ---- end to end through the host-buffer call: pinned q/k/v in, out back, every layer of every step
    e2e_steps = max(3, min(args.steps, 50))
    staging = torch.zeros(tq.tq_model_step_staging_bytes(shape, dt_code, L) + 256, dtype=torch.uint8, device=dev)
    staging = staging[(-staging.data_ptr()) % 256:]
    qh, kh, vh = qs.cpu().pin_memory(), kn.cpu().pin_memory(), vn.cpu().pin_memory()
    oh = torch.empty_like(qh).pin_memory()

    stepper = tq.HostStepper(shape, params, cache, 0, L, qh, kh, vh, oh, staging, wsL, max_seq, args.e2e_chunks)

    def e2e_step():  # one model decode step: pinned q/k/v of all L layers in, the step, outputs back, sync
        stepper.run(stream)

    def e2e_step_plain():  # the same through tq_decode_model_step_host (no graph: 4 copies + 35 launches from the host)
        tq.tq_decode_model_step_host(shape, params, cache, 0, L, qh, kh, vh, oh, staging, wsL, max_seq, stream)

    def time_e2e(fn):
        with torch.cuda.stream(stream):
            reset_len()
            for _ in range(3):  # warm: graph upload, pinned pages, clocks
                fn()
            stream.synchronize()
            reset_len()
            stream.synchronize()
            t0 = time.perf_counter()
            for _ in range(e2e_steps):
                fn()
            stream.synchronize()
            return time.perf_counter() - t0

    e2e_plain_s = time_e2e(e2e_step_plain)
    e2e_s = time_e2e(e2e_step)
    stepper.close()
    e2e_tok = L * B * H * sum(T0 + i + 1 for i in range(e2e_steps))
    vec_bytes = B * H * d * 2

    # ---- aggregate over ranks (max time)
    ms_max, e2e_max = max_over_ranks([ms, e2e_s], world, dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    peak, peak_src = measured_peaks()
    # roofline.frac is the DATA-INDEPENDENT figure: the chain on zero queries, where no value work can be skipped.  The
    # figure on the configs[2] inputs (peaked softmax, value MMAs of zero-weight halves skipped) is frac_peaked_inputs.
    achieved = dec_bytes / (chain_flat_us * 1e-6) / 1e9
    achieved_peaked = dec_bytes / (chain_us * 1e-6) / 1e9
    value = whole_job_value(tok_heads, world, ms_max)
    traffic = None if V_QJL else ncu_traffic("decode_main")
    us_layer = 1e3 * ms_max / args.steps / L
    # the order a model must run the layers in (layer l + 1's q/k/v come from layer l's output): tq_decode_step per layer
    value_sequential = world * L * B * H * (T0 + 1) / (seq_us * L * 1e-6)
    # what a competent two-pass path must move per layer: read the packed cache, write fp16 K and V, read them back
    two_pass_bytes = dec_bytes + 2 * (2 * B * H * T0 * d * 2)
    two_pass_bound_us = two_pass_bytes / peak / 1e3
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f16", "data": "synthetic",
        # `value` is the run-ahead form (tq_decode_model_step: every layer's q/k/v known before the step) — an upper bound
        # that a transformer cannot call, because layer l + 1's inputs depend on layer l's output.  The form a model can
        # call (tq_decode_step layer after layer, one graph) is value_sequential.
        "value_sequential": value_sequential,
        "value_is": "run-ahead upper bound (all layers' q/k/v before the step); value_sequential is the model-order step",
        "config": {
            "workload": f"{w.name} (BASELINE.json configs[2]) x {L} layers: batch {B} x {H} heads x d {d}, "
                        f"{T0}+ cached tokens, fp16 Student-t(4) + 2 outlier channels x15, append + decode per layer per step",
            "layers": L, "batch_per_gpu": B, "heads": H, "head_dim": d, "cached_tokens": T0, "io_dtype": "f16",
            "arithmetic": "fp16 inputs / outputs and MMA operands (two-term split), fp32 accumulation and softmax",
            "l2": f"inputs larger than L2: {L} layer caches x {B*H*T0*rig.bpt/1e6:.1f} MB are cycled every step",
            "cuda_graph": True, "bytes_per_token_head": rig.bpt, "v_qjl": V_QJL,
            "step_form": "tq_decode_model_step: one append+query-prep launch for all layers, one streaming launch per "
                         "layer cache (run-ahead chain), one finish launch",
            "us_per_layer_step": us_layer,
            "packed_gbs_whole_step": value / world * rig.bpt / 1e9,
            "ms_per_step_stepper_device_buffers": stepper_ms, "value_stepper_device_buffers": stepper_value,
            "us_per_layer_step_sequential": seq_us,
            "value_sequential": value_sequential,
            "decode_call_us_live": call_us, "decode_call_packed_gbs": dec_bytes / call_us / 1e3,
            "two_step_torch_baseline": None if two_step is None else {
                "what": "PAPER.md:221 / Table 6 comparison restated: PyTorch GPU ops dequantise one layer cache to fp16 K, V "
                        "in HBM, then torch SDPA (not the product; context, like the paper's 1.96x on its own hardware)",
                "us_per_layer_call": two_step[0], "fused_call_us": call_us,
                "eager_torch_over_fused": two_step[0] / call_us,
                "note": "eager PyTorch with fp32 gathers: an untuned path, not a yardstick; the ratio that means something is "
                        "against the traffic a two-pass path cannot avoid",
                "two_pass_traffic_bound_us": two_pass_bound_us, "two_pass_bytes_per_layer": two_pass_bytes,
                "two_pass_bound_over_fused_call": two_pass_bound_us / call_us,
                "cosine_vs_fused_output": two_step[1]},
            "decode_main_kernel_us_live": chain_us, "decode_main_kernel_plus_finish_us_live": chain_finish_us,
            "decode_main_kernel_us_isolated_launch": iso_us,
            "quantize_pack_gbs": quant_gbs, "quantize_pack_ms_per_layer": statistics.median(q_ms),
            "quantize_pack_frac_of_hbm": quant_gbs / peak,
            "parallelism": f"dp{world} (independent batches, no collective)",
        },
        "clocks": clocks,
        "e2e": {"value": world * e2e_tok / e2e_max, "unit": UNIT, "h2d_bytes_per_step": 3 * L * vec_bytes,
                "d2h_bytes_per_step": L * vec_bytes, "steps": e2e_steps,
                "how": "tq_host_stepper_run: one captured graph per step (H2D copies of q/k/v, tq_decode_model_step per layer "
                       "chunk, D2H of out; copies overlapped with the chunks), host wall clock incl. the synchronisation",
                "value_uncaptured_host_call": e2e_tok / e2e_plain_s},
        "gpu_launches": int(launches_per_step * args.steps),
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic[0] if traffic else None, "kernel": "decode_main_kernel<64, __half, false, %s>" % ("true" if V_QJL else "false"),
                     "traffic_source": (f"READ FROM A COMMITTED FILE, not measured by this run: dram__bytes_read.sum + "
                                        f"dram__bytes_write.sum per launch, {traffic[1]}" if traffic
                                        else "no ncu capture of the current kernel is committed"),
                     "traffic_capture_matches_this_source": traffic[2] if traffic else None,
                     "peak_source": peak_src, "bytes_per_launch": dec_bytes,
                     "how": f"{L} launches (one per layer cache) as the model step chains them (prep and finish kernels left out "
                            f"through the library's measurement hook), zero queries = flat softmax so that no value work is "
                            f"skipped, CUDA events around the graph, / {L}",
                     "frac_flat_softmax": achieved / peak,
                     "frac_peaked_inputs": achieved_peaked / peak,
                     "peaked_inputs": "the same chain on the configs[2] queries: the softmax is peaked and the kernel skips the "
                                      "value MMAs of 16-token halves whose weights underflow to 0 (data-dependent, so not the headline)",
                     "frac_with_finish_kernel_peaked_inputs": dec_bytes / chain_finish_us / 1e3 / peak,
                     "frac_isolated_launch": dec_bytes / iso_us / 1e3 / peak,
                     "frac_call": dec_bytes / call_us / 1e3 / peak,
                     "frac_step": value / world * rig.bpt / 1e9 / peak,
                     "frac_sequential_step": value_sequential / world * rig.bpt / 1e9 / peak,
                     "sequential_step": "tq_decode_step layer after layer in one graph (append + query prep launch, then the "
                                        "streaming launch, each layer behind the one before): the order a model runs"},
    }
    if world == 1 and not args.no_aux:
        line["config"]["aux"] = aux_legs(args)
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(w)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_aux(args, w: W.Workload, key: str, nested: bool = False):
    """configs[1], [3], [4] (and configs[2] with the V-side sketch): a full prefill tq_quantize_pack of every layer cache
    (GB/s on input + packed bytes), then the fused decode over the cache(s); one JSON line.  nested = True: called from
    the default run on one GPU, which folds the returned line into its own `config.aux` (no print, no clock sampler of
    its own, no process-group work)."""
    import torch
    import torch.distributed as dist

    if nested:
        rank, world, local = 0, 1, int(os.environ.get("LOCAL_RANK", "0"))
    else:
        rank, world, local = init_dist()
    from paper_2603_26110_b200 import binding as tq

    bpt = bytes_per_token_head(w.head_dim) + (0 if not V_QJL else (10 if w.head_dim == 64 else 18))
    cache_mb = w.batch * w.n_heads * w.seq * bpt / 1e6
    # enough layer caches to exceed the 126 MB L2 (configs[1] has its own 33 layers)
    L = w.n_layers if key == "cfg1" else max(2, int(np.ceil(300.0 / cache_mb)))
    if args.layers_aux:
        L = args.layers_aux
    rig = Rig(w, L, w.seq, rank, local)
    B, H, d, T0, dev, stream, shape, params, cache = rig.B, rig.H, rig.d, rig.T0, rig.dev, rig.stream, rig.shape, rig.params, rig.cache
    q_ms, q_bytes = rig.prefill()
    q_ms = q_ms[1:] if len(q_ms) > 1 else q_ms  # the first launch also loads the module
    quant_gbs = q_bytes / (statistics.median(q_ms) * 1e-3) / 1e9
    qs = torch.stack([torch_activations(rig.wl, l, (B, H, d), dev, rig.gen)[0] for l in range(L)])
    outs = torch.empty_like(qs)
    wss = [tq.Workspace(shape, 1, dev) for _ in range(L)]
    wsL = tq.Workspace(shape, L, dev)

    def per_layer():
        for layer in range(L):
            tq.tq_decode_attn(shape, params, cache, layer, 1, qs[layer:layer + 1], outs[layer:layer + 1], wss[layer], None, T0, stream)

    def batched():
        tq.tq_decode_attn(shape, params, cache, 0, L, qs, outs, wsL, None, T0, stream)

    sampler = ClockSampler(local)
    if rank == 0 and not nested:
        sampler.start()
    reps = max(6, min(args.steps, 30))
    call_us = rig.graph_us(per_layer, L, reps=reps)
    batched_us = rig.graph_us(batched, L, reps=reps) if key == "cfg1" else None
    with torch.cuda.stream(stream):
        per_layer()
        stream.synchronize()
    tq.tq_profile_decode_main_only(True)
    try:
        main_us = rig.graph_us(per_layer, L, reps=reps)
    finally:
        tq.tq_profile_decode_main_only(False)
    main_batched_us = None
    if key == "cfg1":  # configs[1] is ONE call over all 33 layers: its streaming kernel is one launch over 660 units
        with torch.cuda.stream(stream):
            batched()
            stream.synchronize()
        tq.tq_profile_decode_main_only(True)
        try:
            main_batched_us = rig.graph_us(batched, 1, reps=reps)
        finally:
            tq.tq_profile_decode_main_only(False)
    clocks = sampler.stop() if rank == 0 and not nested else None
    step_us = (batched_us if batched_us is not None else call_us) * L
    (ms_max,) = max_over_ranks([step_us * 1e-3], world, dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    peak, peak_src = measured_peaks()
    dec_bytes = B * H * T0 * bpt
    value = world * L * B * H * T0 / (ms_max * 1e-3)
    traffic = ncu_traffic(f"decode_main_{key}")
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": reps - 1, "warmup": 3,
        "ms_per_step": ms_max, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f16", "data": "synthetic",
        "config": {
            "workload": f"{w.name} (BASELINE.json configs[{w.index}]): {L} layer cache(s) x batch {B} x {H} heads x d {d}, "
                        f"{T0} cached tokens, {w.dtype} {w.dist}; full prefill tq_quantize_pack, then fused decode over every cache",
            "layers": L, "batch_per_gpu": B, "heads": H, "head_dim": d, "cached_tokens": T0,
            "l2": f"{L} layer caches x {cache_mb:.1f} MB are cycled", "cuda_graph": True, "bytes_per_token_head": bpt,
            "step": "one tq_decode_attn per layer cache" if batched_us is None else "ONE tq_decode_attn call over all 33 layers",
            "decode_call_us_per_layer": call_us, "decode_call_us_per_layer_batched": batched_us,
            "decode_main_kernel_us_live": main_us,
            "quantize_pack_gbs": quant_gbs, "quantize_pack_ms_per_layer": statistics.median(q_ms),
            "quantize_pack_frac_of_hbm": quant_gbs / peak,
            "quantize_pack_roofline": {"bound": "hbm (rotations on tcgen05)", "achieved": quant_gbs, "peak": peak, "unit": "GB/s",
                                       "frac": quant_gbs / peak, "bytes_per_launch": q_bytes},
        },
        "clocks": clocks,
        "e2e": None,
        "gpu_launches": int(tq.tq_launch_count()),
        "roofline": ({"bound": "hbm", "achieved": dec_bytes / main_us / 1e3, "peak": peak, "unit": "GB/s",
                      "frac": dec_bytes / main_us / 1e3 / peak, "traffic": traffic[0] if traffic else None,
                      "kernel": f"decode_main_kernel<{d}, __half, true>", "peak_source": peak_src, "bytes_per_launch": dec_bytes,
                      "frac_call": dec_bytes / call_us / 1e3 / peak} if main_batched_us is None else
                     {"bound": "hbm", "achieved": L * dec_bytes / main_batched_us / 1e3, "peak": peak, "unit": "GB/s",
                      "frac": L * dec_bytes / main_batched_us / 1e3 / peak, "traffic": None,
                      "kernel": f"decode_main_kernel<{d}, __half, true>", "peak_source": peak_src,
                      "bytes_per_launch": L * dec_bytes, "how": "ONE launch over all layers (the call configs[1] describes)",
                      "us_per_launch": main_batched_us, "frac_call": L * dec_bytes / (batched_us * L) / 1e3 / peak,
                      "frac_one_layer_per_launch": dec_bytes / main_us / 1e3 / peak}),
    }
    if nested:
        return line
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def aux_legs(args):
    """The other BASELINE.json configs in the line the driver runs (config.aux): configs[1], [3], [4] and configs[2] with
    the V-side sketch, each the few-second leg `--config cfgN` (`--v-qjl`) runs on its own, boiled down to its numbers."""
    import gc

    import torch

    global V_QJL
    out = {}
    for name, key, vq in (("cfg1", "cfg1", 0), ("cfg3", "cfg3", 0), ("cfg4", "cfg4", 0), ("cfg2_v_qjl", "cfg2", 1)):
        keep, V_QJL = V_QJL, vq
        try:
            line = run_aux(args, W.CONFIGS[CONFIG_NAMES[key]], key, nested=True)
        finally:
            V_QJL = keep
        c, r = line["config"], line["roofline"]
        out[name] = {
            "workload": c["workload"], "layers": c["layers"], "bytes_per_token_head": c["bytes_per_token_head"],
            "value": line["value"], "unit": UNIT, "step": c["step"], "us_per_step": line["ms_per_step"] * 1e3,
            "decode_call_us_per_layer": c["decode_call_us_per_layer"], "decode_main_kernel_us_live": c["decode_main_kernel_us_live"],
            "roofline": {k: r.get(k) for k in ("bound", "achieved", "peak", "unit", "frac", "frac_call", "bytes_per_launch",
                                               "us_per_launch", "frac_one_layer_per_launch", "how") if k in r},
            "inputs": "the workload's own queries (softmax as the inputs make it; no flat-softmax leg here)",
            "quantize_pack_gbs": c["quantize_pack_gbs"], "quantize_pack_ms_per_layer": c["quantize_pack_ms_per_layer"],
            "quantize_pack_frac_of_hbm": c["quantize_pack_frac_of_hbm"],
        }
        gc.collect()
        torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg2", choices=sorted(CONFIG_NAMES))
    ap.add_argument("--layers", type=int, default=33, help="ESM-2-650M has 33 layers (cfg2)")
    ap.add_argument("--layers-aux", type=int, default=0, help="layer caches cycled by cfg3 / cfg4 (0 = enough to exceed L2)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-aux", action="store_true", help="skip the configs[1] / [3] / [4] / v_qjl legs of the default line (config.aux)")
    ap.add_argument("--no-two-step", action="store_true", help="skip the PyTorch two-step GPU baseline (NEXT-4)")
    ap.add_argument("--v-qjl", action="store_true", help="measure with the V-side residual sketch on (tq_shape.v_qjl = 1)")
    ap.add_argument("--e2e-chunks", type=int, default=0, help="layer chunks of the host stepper (0 = the library's choice)")
    args = ap.parse_args()
    w = W.CONFIGS[CONFIG_NAMES[args.config]]
    global V_QJL
    V_QJL = 1 if args.v_qjl else 0
    if args.impl == "reference":
        run_reference(args, w)
        return
    world_env = os.environ.get("WORLD_SIZE")
    if world_env is None and args.gpus > 1:
        # `python bench.py --gpus N`: one process per GPU under torchrun, as the driver launches it
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", os.environ.get("MASTER_PORT", "29533"), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if world_env is not None and int(world_env) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} does not match WORLD_SIZE={world_env}")
    if args.config == "cfg2":
        run_cfg2(args, w)
    else:
        run_aux(args, w, args.config)


if __name__ == "__main__":
    main()
