#!/usr/bin/env python
"""bench.py -- throughput of the Sangam hot path (kv_write -> block_attn) on B200.

One "step" = one pass of the whole hot path over one synthetic batch: sangam_kv_write of the
iteration's fresh K/V rows followed by sangam_block_attn (device-side plan, tcgen05 attention,
split-KV combine), captured once as a CUDA graph and replayed.
Headline workload (N = 1): BASELINE.json configs[1], the LLaDA-8B-like block decode.  Steps
rotate over several independent per-layer pool sets so that consecutive replays never find
their K/V in L2 (cold-L2 rule).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 1..5 | <variant name>] [--all-configs]
  python bench.py --impl reference ...      # times the fp64 CPU oracle on a bounded sample

Besides the headline line it reports, under `all_configs`, every BASELINE.json config (min / median / max over
repetitions, roofline fraction, the oracle timed on the host cores), under `variants` and `fig3_sweep` the shapes of
SURVEY.md 8(f) rank 4 (dKV-Cache-PD refresh, the paper's real response regions, the Fig.-3-shaped batch sweep) and under
`sched_series` the batches Algorithm 1 produces from a simulated arrival trace for tau in {512, 1024, 2048, 16384}
(PAPER.md:327), run through the real kernels.

Multi-GPU: the path does not shard ("replicas only"): under torchrun every rank runs
the same workload on its own GPU, time = max over ranks, value = sum of work / that time.
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import sangam_inputs as si  # noqa: E402

METRIC = "block_attn_tflops"
UNIT = "TFLOP/s"
WORKLOAD_NAMES = {1: "config1_tiny", 2: "config2_llada_block_decode", 3: "config3_dream_gqa_block_decode",
                  4: "config4_kv_refresh_prefill", 5: "config5_hybrid_mixed"}
NSETS = {1: 8, 2: 10, 3: 6, 4: 1, 5: 1}        # independent pool sets rotated per step (>= 8x L2 of distinct data)
BOUND = {1: "hbm", 2: "hbm", 3: "hbm", 4: "tensor", 5: "tensor"}
L2_BYTES = 126e6


def make_workload_batch(key):
    """BASELINE.json config number or a variant name of sangam_inputs.VARIANTS."""
    if isinstance(key, int) or str(key).isdigit():
        return si.CONFIGS[int(key)](), WORKLOAD_NAMES[int(key)], NSETS[int(key)]
    b = si.VARIANTS[key]()
    return b, key, nsets_for(b)


def nsets_for(b):
    """Pool sets to rotate so that consecutive steps touch >= 8x L2 of distinct K/V (one set when a step alone exceeds L2)."""
    by = b.attn_bytes()
    return 1 if by > 2 * L2_BYTES else int(min(12, max(2, np.ceil(8 * L2_BYTES / by))))


def sources_hash():
    from paper_2607_04206_b200.build import sources_hash as h
    return h()


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


def load_traffic():
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f)
    return {}


# ------------------------------------------------------------------------------------------------
# clocks: sampled DURING the timed region
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
           "sw_power_cap": 0x4, "hw_power_brake": 0x80}

    def __init__(self, index=0, period=0.01):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.period, self.stop_evt, self.thread, self.h = period, threading.Event(), None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        while not self.stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for name, bit in self.BAD.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self.stop_evt.wait(self.period)

    def __enter__(self):
        if self.nv is not None:
            self.thread = threading.Thread(target=self._loop, daemon=True)
            self.thread.start()
        return self

    def __exit__(self, *a):
        self.stop_evt.set()
        if self.thread:
            self.thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": int(statistics.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------
# device state
# ------------------------------------------------------------------------------------------------
def _bf16(bits, device):
    import torch
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).to(device).view(torch.bfloat16)


def _i32(a, device):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).to(device)


DISPATCH = 0          # sangam_set_dispatch mode of every engine this run creates (--dispatch; 0 = the library's own choice)


class Workload:
    """A Batch resident in HBM: `nsets` independent (pools, q, k_new, v_new, out) sets + shared metadata."""

    def __init__(self, b: si.Batch, nsets: int, device="cuda"):
        import torch
        import paper_2607_04206_b200 as sg
        self.b, self.nsets, self.device = b, nsets, device
        dev_index = torch.cuda.current_device()             # under torchrun: LOCAL_RANK's GPU (set in dist_setup)
        self.eng = sg.Sangam(num_q_heads=b.num_q_heads, num_kv_heads=b.num_kv_heads, head_dim=b.head_dim,
                             num_pages=b.num_pages, max_batch=b.batch, max_total_q=max(b.total_q, len(b.slot_new), 1),
                             max_pages_per_req=b.max_pages_per_req, device=dev_index)
        if DISPATCH:
            self.eng.set_dispatch(DISPATCH)
        device = f"cuda:{dev_index}"
        self.device = device
        self.block_table, self.cu_q_lens, self.ctx_lens = _i32(b.block_table, device), _i32(b.cu_q_lens, device), _i32(b.ctx_lens, device)
        self.slot_new = _i32(b.slot_new, device)
        k_cache, v_cache, slot_cache = _bf16(b.k_cache, device), _bf16(b.v_cache, device), _i32(b.slot_cache, device)
        q0, kn0, vn0 = _bf16(b.q, device), _bf16(b.k_new, device), _bf16(b.v_new, device)
        self.sets = []
        shape = (b.num_pages, b.num_kv_heads, si.PAGE, b.head_dim)
        for _ in range(nsets):
            kp = torch.zeros(shape, dtype=torch.bfloat16, device=device)
            vp = torch.zeros(shape, dtype=torch.bfloat16, device=device)
            self.eng.kv_write(k_cache, v_cache, slot_cache, kp, vp)          # cache content (setup, untimed)
            self.sets.append({"kp": kp, "vp": vp, "q": q0.clone(), "kn": kn0.clone(), "vn": vn0.clone(),
                              "out": torch.zeros_like(q0)})
        torch.cuda.synchronize()
        del k_cache, v_cache, slot_cache
        self.stream = torch.cuda.Stream()
        self.iter_graphs, self.attn_graphs, self.write_graphs = [], [], []

    def run_iteration(self, s, stream):
        self.eng.kv_write(s["kn"], s["vn"], self.slot_new, s["kp"], s["vp"], stream=stream)
        self.run_attn(s, stream)

    def run_attn(self, s, stream, ctx_lens=None):
        self.eng.block_attn(s["q"], s["kp"], s["vp"], self.block_table, self.cu_q_lens, self.ctx_lens if ctx_lens is None else ctx_lens,
                            float(self.b.scale), s["out"], stream=stream)

    def capture_chain(self, fn):
        """ONE graph holding a step on every pool set back to back, as the layers of a model sit in one captured iteration:
        kernel-to-kernel launch latency inside a graph (programmatic dependent launch) instead of graph-to-graph."""
        import torch
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(self.stream):
            with torch.cuda.graph(g, stream=self.stream):
                for s in self.sets:
                    fn(s, self.stream)
        torch.cuda.synchronize()
        return g

    def capture_plan_miss(self):
        """Attention graphs whose consecutive replays alternate between two metadata sets that differ by one context position
        (the longest request, one token shorter): the two-stream kernel's per-CTA plan cache, keyed by the lengths, misses on
        every launch -- what the first layer of a serving iteration pays.  None when there is nothing to vary."""
        import torch
        c = self.b.ctx_lens.copy()
        r = int(np.argmax(c))
        if c[r] < 2:
            return None
        c[r] -= 1
        alt = _i32(c, self.device)
        graphs = []
        with torch.cuda.stream(self.stream):
            for k in range(2 * self.nsets):
                s, cl = self.sets[k % self.nsets], (alt if k % 2 else self.ctx_lens)
                self.run_attn(s, self.stream, cl)
                self.stream.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=self.stream):
                    self.run_attn(s, self.stream, cl)
                graphs.append(g)
        torch.cuda.synchronize()
        self._alt_ctx = alt
        return graphs

    def capture(self):
        import torch
        with torch.cuda.stream(self.stream):
            for s in self.sets:                       # warm-up outside capture (first-launch work)
                self.run_iteration(s, self.stream)
            self.stream.synchronize()
            for s in self.sets:
                for lst, fn in ((self.iter_graphs, self.run_iteration), (self.attn_graphs, self.run_attn),
                                (self.write_graphs, lambda ss, st: self.eng.kv_write(ss["kn"], ss["vn"], self.slot_new, ss["kp"], ss["vp"], stream=st))):
                    g = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(g, stream=self.stream):
                        fn(s, self.stream)
                    lst.append(g)
        torch.cuda.synchronize()

    def time_graphs(self, graphs, steps, warmup):
        """K replays between two CUDA events on the launching stream; returns total ms."""
        import torch
        n = len(graphs)
        with torch.cuda.stream(self.stream):
            for i in range(warmup):
                graphs[i % n].replay()
            self.stream.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(self.stream)
            for i in range(steps):
                graphs[i % n].replay()
            e1.record(self.stream)
            e1.synchronize()
        return e0.elapsed_time(e1)


def roofline_time_us(b: si.Batch, peaks, which="attn"):
    f = b.flops() / (peaks["bf16_tflops"] * 1e12) * 1e6
    by = (b.attn_bytes() if which == "attn" else b.attn_bytes() + b.write_bytes()) / (peaks["hbm_gbs"] * 1e9) * 1e6
    return max(f, by), f, by


def measure_batch(b: si.Batch, name: str, nsets: int, steps: int, warmup: int, peaks, reps: int = 3, parts=("iteration", "attn", "kv_write")):
    """All figures of one workload: iteration / attention / kv_write time (median, min, max over `reps` repetitions of `steps`
    replays, clocks sampled during the repetitions), TFLOP/s, GB/s and the fraction of the shape's own roofline
    (the slower of flops at the bf16 peak and algorithmic bytes at the HBM peak)."""
    w = Workload(b, nsets)
    w.capture()
    res = {"workload": name, "pool_sets": w.nsets, "steps": steps, "reps": reps}
    graphs = {"iteration": w.iter_graphs, "attn": w.attn_graphs, "kv_write": w.write_graphs}
    import torch
    with ClockSampler(index=torch.cuda.current_device()) as cs:
        for key in parts:
            per = [w.time_graphs(graphs[key], steps, warmup) / steps * 1e3 for _ in range(reps)]   # us per step
            res[key + "_us"] = round(statistics.median(per), 3)
            res[key + "_us_min"] = round(min(per), 3)
            res[key + "_us_max"] = round(max(per), 3)
    res["clocks"] = cs.summary()
    t_roof, t_f, t_b = roofline_time_us(b, peaks)
    a = res["attn_us"]
    res.update({"flops": b.flops(), "attn_bytes": b.attn_bytes(), "write_bytes": b.write_bytes(),
                "attn_tflops": round(b.flops() / a / 1e6, 2), "attn_gbs": round(b.attn_bytes() / a / 1e3, 1),
                "bound": "tensor" if t_f > t_b else "hbm", "t_roof_us": round(t_roof, 2), "roofline_frac": round(t_roof / a, 4),
                "roofline_frac_best": round(t_roof / res["attn_us_min"], 4),
                "device_flags": int(w.eng.device_status())})
    if "kv_write" in parts:
        res["kv_write_gbs"] = round(b.write_bytes() / max(res["kv_write_us"], 1e-9) / 1e3, 1)
    if w.nsets > 1:      # the same steps with the pool sets' launches chained inside one graph (launch gaps of a layer loop)
        for key, fn in (("attn", w.run_attn), ("iteration", w.run_iteration)):
            if key in parts:
                g = w.capture_chain(fn)
                k = max(1, steps // w.nsets)
                per = [w.time_graphs([g], k, max(1, warmup // w.nsets)) / (k * w.nsets) * 1e3 for _ in range(reps)]
                res[key + "_us_chained"] = round(statistics.median(per), 3)
        res["chained"] = f"{w.nsets} consecutive steps (one per pool set) captured in ONE graph and replayed; *_us: one step per graph"
    # The timed replays above repeat one set of lengths, so the two-stream kernel's plan cache (batches of <= 32 requests) hits
    # on every launch; the miss path is timed beside it.  (The decode kernel plans on every launch: no second figure.)
    if w.eng.query(4) == 1 and b.batch <= 32:
        miss = w.capture_plan_miss()
        if miss is not None:
            per = [w.time_graphs(miss, steps, warmup) / steps * 1e3 for _ in range(reps)]
            res["attn_us_plan_miss"] = round(statistics.median(per), 3)
            res["plan_cache"] = "attn_us: every launch hits the per-CTA plan cache; attn_us_plan_miss: every launch misses (lengths alternate)"
    return res, w


def measure_config(cfg: int, steps: int, warmup: int, peaks, reps: int = 3):
    return measure_batch(si.CONFIGS[cfg](), WORKLOAD_NAMES[cfg], NSETS[cfg], steps, warmup, peaks, reps)


# ------------------------------------------------------------------------------------------------
# end to end through the C ABI with HOST buffers (sangam_iteration_host)
# ------------------------------------------------------------------------------------------------
def measure_e2e(w: Workload, steps: int, warmup: int):
    """sangam_iteration_packed: per step ONE host-to-device copy of the packed pinned buffer (q, k, v and all metadata),
    kv_write + block_attn, one device-to-host copy of `out`, stream synchronize."""
    import torch
    b = w.b
    nt = int(b.slot_new.shape[0])
    off = w.eng.packed_layout(b.batch, b.total_q, nt)
    packed = torch.zeros(off[7], dtype=torch.uint8).pin_memory()
    pn = packed.numpy()
    parts = [np.ascontiguousarray(b.q), np.ascontiguousarray(b.k_new), np.ascontiguousarray(b.v_new), b.slot_new.astype(np.int32),
             b.block_table.astype(np.int32), b.cu_q_lens.astype(np.int32), b.ctx_lens.astype(np.int32)]
    for o, a in zip(off, parts):
        raw = a.reshape(-1).view(np.uint8)
        pn[o:o + raw.size] = raw
    out = torch.empty((b.total_q, b.num_q_heads, b.head_dim), dtype=torch.bfloat16).pin_memory()
    h2d = int(off[7])
    d2h = int(out.numel()) * out.element_size()
    n = len(w.sets)

    def step(i):
        s = w.sets[i % n]
        w.eng.iteration_packed(packed, nt, s["kp"], s["vp"], b.batch, b.total_q, float(b.scale), out, stream=w.stream)

    for i in range(warmup):
        step(i)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(steps):
        step(i)                         # each call ends with a stream synchronize (D2H of `out` complete)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    # the copies alone (same buffers, same stream, one synchronize per step): the rest of a step is the kernels
    dev = torch.empty(off[7], dtype=torch.uint8, device=w.device)
    dout = torch.empty_like(out, device=w.device)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    with torch.cuda.stream(w.stream):
        for i in range(steps):
            dev.copy_(packed, non_blocking=True)
            out.copy_(dout, non_blocking=True)
            w.stream.synchronize()
    dc = time.perf_counter() - t1
    return dt / steps, h2d, d2h, dc / steps


# ------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/)
# ------------------------------------------------------------------------------------------------
def oracle_sample(b: si.Batch, rows_per_request: int):
    """Pools as the oracle builds them + the sampled global q rows."""
    import oracle
    kp, vp = si.empty_pools(b, poison=False)
    oracle.kv_write(b.k_cache, b.v_cache, b.slot_cache, kp, vp)
    rows = si.sample_rows(b, per_request=rows_per_request)
    return oracle, kp, vp, rows


def oracle_step(oracle, b, kp, vp, rows):
    oracle.kv_write(b.k_new, b.v_new, b.slot_new, kp, vp)
    oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale, rows=rows)


def sample_flops(b: si.Batch, rows) -> float:
    r_of = np.searchsorted(b.cu_q_lens, rows, side="right") - 1
    return 4.0 * b.num_q_heads * b.head_dim * float(np.sum(b.ctx_lens[r_of].astype(np.int64)))


def cpu_baseline(b: si.Batch, target_s: float = 15.0):
    """The oracle as it stands on the host cores: a bounded row sample of the workload (all heads, full contexts)
    plus its kv_write, repeated until about `target_s` seconds of CPU work have been timed."""
    oracle, kp, vp, rows1 = oracle_sample(b, 1)
    t0 = time.perf_counter()
    oracle_step(oracle, b, kp, vp, rows1)
    t1 = time.perf_counter() - t0
    per = max(1, int(target_s / max(t1, 1e-3)))
    qmax = int(b.q_lens.max())
    per = min(per, qmax)
    rows = si.sample_rows(b, per_request=per)
    reps, dt = 0, 0.0
    t0 = time.perf_counter()
    while True:
        oracle_step(oracle, b, kp, vp, rows)
        reps += 1
        dt = time.perf_counter() - t0
        if dt >= target_s or reps >= 1000:
            break
    f = sample_flops(b, rows) * reps
    return {"value": round(f / dt / 1e12, 6), "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{len(rows)} of {b.total_q} query rows (<= {per} per request, all heads, full contexts) + the kv_write, "
                      f"repeated {reps}x, {dt:.2f} s, fp64 C -O2 -fopenmp",
            "seconds": round(dt, 3), "sample_flops": f}


def cpu_baseline_config(cfg: int, b: si.Batch):
    """SURVEY.md 8(d) / BASELINE.md section 4: the oracle over the WHOLE config for configs 1-3; for the prefill-sized configs a
    stratified row sample (tile-edge + seeded random rows, all heads) with the full-config time extrapolated by the exact
    work ratio sum q_r c_r (all) / sum q_r c_r (evaluated), labelled "extrapolated"."""
    if cfg in (1, 2, 3):
        oracle, kp, vp, _ = oracle_sample(b, 1)
        rows = np.arange(b.total_q, dtype=np.int32)
        label = "full"
    else:
        oracle, kp, vp, rows = oracle_sample(b, 8 if cfg == 4 else 32)     # config 5: its 32-row decodes in full + 32 rows per prefill
        label = "extrapolated"
    t0 = time.perf_counter()
    oracle_step(oracle, b, kp, vp, rows)
    dt = time.perf_counter() - t0
    f = sample_flops(b, rows)
    full_s = dt * b.flops() / max(f, 1.0)
    return {"value": round(f / dt / 1e12, 6), "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{len(rows)} of {b.total_q} query rows, all heads, full contexts + the kv_write, 1 pass, fp64 C -O2 -fopenmp",
            "seconds": round(dt, 3), "full_config_seconds": round(full_s, 3), "full_config": label}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = int(args.workload)
    b = si.CONFIGS[cfg]()
    oracle, kp, vp, rows = oracle_sample(b, 2)
    for _ in range(min(args.warmup, 3)):
        oracle_step(oracle, b, kp, vp, rows)
    steps = min(args.steps, 200)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle_step(oracle, b, kp, vp, rows)
    dt = (time.perf_counter() - t0) / steps
    f = sample_flops(b, rows)
    val = round(f / dt / 1e12, 6)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": min(args.warmup, 3), "ms_per_step": round(dt * 1e3, 4), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAMES[cfg], "sample": f"{len(rows)} of {b.total_q} query rows per step"},
            "cpu_baseline": {"value": val, "unit": UNIT, "kind": "oracle", "cores": oracle.num_threads(),
                             "sample": f"{len(rows)} of {b.total_q} query rows (2 per request, all heads) + kv_write per step"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------
# multi-process plumbing: replicas only, max time over ranks
# ------------------------------------------------------------------------------------------------
def dist_setup():
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world <= 1:
        return 0, 1, None
    import torch
    import torch.distributed as dist
    rank, local = int(os.environ["RANK"]), int(os.environ.get("LOCAL_RANK", "0"))
    backend = "nccl" if torch.cuda.is_available() else "gloo"
    if backend == "nccl":
        torch.cuda.set_device(local)
    dist.init_process_group(backend=backend)
    return rank, world, dist


def max_over_ranks(value: float, dist, device=None) -> float:
    if dist is None:
        return value
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device or ("cuda" if dist.get_backend() == "nccl" else "cpu"))
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier(dist):
    if dist is not None:
        dist.barrier()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20000)
    ap.add_argument("--warmup", type=int, default=200)
    ap.add_argument("--workload", default="2", help="BASELINE.json config 1..5 or a variant name (sangam_inputs.VARIANTS)")
    ap.add_argument("--no-extras", action="store_true", help="skip variants, the Fig.-3 sweep and the scheduler series")
    ap.add_argument("--dispatch", default="auto", choices=["auto", "prefill", "decode", "gqa_pair"],
                    help="attention kernel sangam_block_attn launches (sangam_set_dispatch); auto = the library's own choice")
    ap.add_argument("--impl", default="sangam", choices=["sangam", "reference"])
    ap.add_argument("--all-configs", dest="all_configs", action="store_true", default=None)
    ap.add_argument("--no-all-configs", dest="all_configs", action="store_false")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    global DISPATCH
    DISPATCH = {"auto": 0, "prefill": 1, "decode": 2, "gqa_pair": 3}[args.dispatch]
    rank, world, dist = dist_setup()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the sangam kernels have no CPU fallback)")
    peaks = load_peaks()
    steps, warmup = max(1, args.steps), max(3, args.warmup)
    b, wname, nsets = make_workload_batch(args.workload)
    cfg = int(args.workload) if str(args.workload).isdigit() else None
    w = Workload(b, nsets)
    w.capture()

    # ---- timed region: K steps of the whole hot path, barrier + synchronize on both sides
    barrier(dist)
    torch.cuda.synchronize()
    with ClockSampler(index=torch.cuda.current_device()) as cs:
        ms_total = w.time_graphs(w.iter_graphs, steps, warmup)
    torch.cuda.synchronize()
    barrier(dist)
    ms_total = max_over_ranks(ms_total, dist)
    ms_step = ms_total / steps
    value = world * b.flops() / (ms_step * 1e-3) / 1e12
    # kernels captured in one step's graph: kv_write + the attention kernel(s) the dispatch chose (decode kernel: 1, fused
    # merge; two-stream kernel: attention + combine).  Counted from the library's launch counter over one eager iteration.
    n0 = w.eng.launch_count()
    w.run_iteration(w.sets[0], w.stream)
    torch.cuda.synchronize()
    kernels_per_step = w.eng.launch_count() - n0
    gpu_launches = steps * kernels_per_step

    # ---- dominant kernel (attention), timed alone, L2-cold
    attn_ms = w.time_graphs(w.attn_graphs, steps, warmup) / steps
    attn_ms = max_over_ranks(attn_ms, dist)
    write_ms = w.time_graphs(w.write_graphs, steps, warmup) / steps
    tj = load_traffic()
    traffic = tj.get("workloads", tj).get(wname)
    t_roof, t_f, t_b = roofline_time_us(b, peaks)
    if t_b >= t_f:
        ach = b.attn_bytes() / (attn_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "achieved": round(ach, 1), "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": round(ach / peaks["hbm_gbs"], 4)}
    else:
        ach = b.flops() / (attn_ms * 1e-3) / 1e12
        roof = {"bound": "tensor", "achieved": round(ach, 1), "peak": peaks["bf16_tflops"], "unit": "TFLOP/s",
                "frac": round(ach / peaks["bf16_tflops"], 4)}
    kernel_name = {1: "tc::attn_kernel (two-stream kernel, device-side plan inside) + tc::combine_kernel",
                   2: "dec::decode_kernel (device-side plan, swapped-operand attention, fused split-KV merge)",
                   3: "gqa::gqa_decode_kernel (CTA pairs, K/V tiles multicast, fused split-KV merge)"}.get(w.eng.query(4), "?")
    roof.update({"traffic": traffic, "traffic_sources_hash": tj.get("sources_hash"), "traffic_matches_this_build": tj.get("sources_hash") == sources_hash(),
                 "kernel": kernel_name + ", timed alone over the same rotation",
                 "kernel_us": round(attn_ms * 1e3, 3), "peak_source": peaks["source"] + " (burst)",
                 "algorithmic_bytes": b.attn_bytes(), "algorithmic_flops": b.flops()})

    # ---- end to end from host buffers
    e2e_steps = max(10, min(steps, 300))
    e2e_s, h2d, d2h, copies_s = measure_e2e(w, e2e_steps, 5)
    e2e_s = max_over_ranks(e2e_s, dist)
    e2e = {"value": round(world * b.flops() / e2e_s / 1e12, 4), "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "ms_per_step": round(e2e_s * 1e3, 4), "steps": e2e_steps,
           "split_us": {"copies_and_sync_alone": round(copies_s * 1e6, 1), "kernels_graph_replay": round(ms_step * 1e3, 1)},
           "api": "sangam_iteration_packed (one pinned packed host buffer: 1 H2D copy + kv_write + block_attn + 1 D2H copy + stream sync per step)"}

    line = {"metric": METRIC, "value": round(value, 3), "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": round(ms_step, 6), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16", "data": "synthetic",
            "config": {"workload": wname, "batch": b.batch, "total_q": b.total_q,
                       "sum_ctx": int(b.ctx_lens.sum()), "heads": f"{b.num_q_heads}/{b.num_kv_heads}",
                       "head_dim": b.head_dim, "page": si.PAGE, "parallelism": f"replicas x{world}", "dispatch": args.dispatch,
                       "l2": f"cold: steps rotate over {w.nsets} independent pool sets "
                             f"({w.nsets * b.attn_bytes() / 1e6:.0f} MB distinct per rotation)",
                       "step": "CUDA-graph replay of kv_write + block_attn (device-side plan + tcgen05 attention + split-KV merge)"},
            "us_per_iteration": round(ms_step * 1e3, 3), "attn_us": round(attn_ms * 1e3, 3),
            "kv_write_us": round(write_ms * 1e3, 3),
            "clocks": cs.summary(), "e2e": e2e, "gpu_launches": gpu_launches, "kernels_per_step": kernels_per_step,
            "device_flags": int(w.eng.device_status()), "roofline": roof}

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(b)
    run_all = args.all_configs if args.all_configs is not None else (world == 1)
    if run_all and rank == 0:
        del w
        torch.cuda.empty_cache()
        allc = []
        for c in (1, 2, 3, 4, 5):
            st, reps = {1: (2000, 5), 2: (2000, 5), 3: (1000, 5), 4: (20, 10), 5: (30, 10)}[c]
            r, ww = measure_config(c, st, max(3, st // 10), peaks, reps)
            if not args.no_cpu_baseline:
                r["cpu_baseline"] = cpu_baseline_config(c, ww.b)
            allc.append(r)
            del ww
            torch.cuda.empty_cache()
        line["all_configs"] = allc
        if not args.no_extras:
            line["variants"] = measure_variants(peaks)
            line["fig3_sweep"] = measure_fig3(peaks)
            line["sched_series"] = measure_sched_series()
            line["neighbours"] = measure_neighbours(peaks)
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


# ------------------------------------------------------------------------------------------------
# variant shapes and the Fig.-3-shaped batch sweep (attention only)
# ------------------------------------------------------------------------------------------------
def measure_variants(peaks):
    import torch
    out = []
    for name in si.VARIANTS:
        b = si.VARIANTS[name]()
        st = 300 if b.flops() < 5e10 else 30
        r, w = measure_batch(b, name, nsets_for(b), st, max(3, st // 10), peaks, reps=3, parts=("iteration", "attn"))
        out.append(r)
        del w
        torch.cuda.empty_cache()
    return out


def measure_fig3(peaks):
    """Batch in {1 .. 64} block decodes at sequence length 1024, both head geometries: attention-only us and
    the fraction of the HBM roofline."""
    import torch
    out = []
    for model in ("llada", "dream"):
        for nb in si.FIG3_BATCHES:
            b = si.fig3_point(model, nb)
            r, w = measure_batch(b, b.name, nsets_for(b), 500, 50, peaks, reps=3, parts=("attn",))
            out.append({k: r[k] for k in ("workload", "pool_sets", "attn_us", "attn_us_min", "attn_gbs", "attn_tflops", "bound", "t_roof_us", "roofline_frac", "device_flags")})
            del w
            torch.cuda.empty_cache()
    return out


# ------------------------------------------------------------------------------------------------
# the HBM-bound kernels next to the path, each against its own algorithmic bytes
# ------------------------------------------------------------------------------------------------
def measure_neighbours(peaks):
    """RoPE-fused KV write, confidence sampler (both entry points), KV page gather / scatter: CUDA-event time of `steps`
    back-to-back calls on buffers larger than L2 in total (several buffer sets rotate), algorithmic bytes / time against the
    measured HBM peak.  LLaDA-8B-like geometry (32 kv heads, D 128, vocabulary 126 464)."""
    import torch
    import paper_2607_04206_b200 as sg
    dev = torch.cuda.current_device()
    Hkv, D, V = 32, 128, 126464
    out = []

    def timed(fn, nsets, steps=60, warmup=6):
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            for i in range(warmup):
                fn(i % nsets, st)
            st.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st)
            for i in range(steps):
                fn(i % nsets, st)
            e1.record(st)
            e1.synchronize()
        return e0.elapsed_time(e1) / steps * 1e3          # us per call

    def rec(name, us, nbytes, note):
        out.append({"kernel": name, "us": round(us, 2), "algorithmic_bytes": int(nbytes), "gbs": round(nbytes / us / 1e3, 1),
                    "frac_of_hbm_peak": round(nbytes / us / 1e3 / peaks["hbm_gbs"], 4), "workload": note})

    g = torch.Generator(device="cuda").manual_seed(7)
    # ---- RoPE-fused KV write: a refresh-sized write (8192 rows) and a decode-sized one (16 x 32 rows)
    P = 2048
    eng = sg.Sangam(num_q_heads=Hkv, num_kv_heads=Hkv, head_dim=D, num_pages=P, max_batch=16, max_total_q=8192, max_pages_per_req=512, device=dev)
    table = torch.from_numpy(sg.rope_table(4096, D)).cuda()
    for T, nsets in ((8192, 3), (512, 8)):
        sets = []
        for _ in range(nsets):
            k = torch.randn((T, Hkv, D), device="cuda", generator=g).to(torch.bfloat16); v = torch.randn((T, Hkv, D), device="cuda", generator=g).to(torch.bfloat16)
            kp = torch.zeros((P, Hkv, si.PAGE, D), dtype=torch.bfloat16, device="cuda"); vp = torch.zeros_like(kp)
            sets.append((k, v, kp, vp))
        slots = torch.randperm(P * si.PAGE, device="cuda", generator=g)[:T].to(torch.int32)
        pos = torch.randint(0, 4096, (T,), device="cuda", generator=g, dtype=torch.int32)
        us = timed(lambda i, st: eng.kv_write_rope(sets[i][0], sets[i][1], slots, pos, table, sets[i][2], sets[i][3], stream=st), nsets)
        rec("kv_write_rope", us, 2 * (2 * 2 * T * Hkv * D) + 8 * T + T * D * 4, f"{T} new rows x {Hkv} kv heads x {D}, table rows from L2")
        del sets
    # ---- confidence sampler: one decode iteration's rows (16 requests x 32 rows) at LLaDA's vocabulary
    rows, nsets = 512, 3
    lsets = [(2.0 * torch.randn((rows, V), device="cuda", generator=g)).to(torch.bfloat16) for _ in range(nsets)]
    masked = torch.ones(rows, dtype=torch.int32, device="cuda"); cu = torch.arange(0, rows + 1, 32, dtype=torch.int32, device="cuda")
    tok = torch.empty(rows, dtype=torch.int32, device="cuda"); conf = torch.empty(rows, dtype=torch.float32, device="cuda"); un = torch.empty(rows, dtype=torch.int32, device="cuda")
    nbytes = rows * V * 2 + rows * 16
    us = timed(lambda i, st: eng.confidence_sample(lsets[i], masked, cu, 0.9, tok, conf, un, stream=st), nsets)
    rec("confidence_sample", us, nbytes, f"{rows} rows x vocabulary {V} (bf16 logits read once)")
    us = timed(lambda i, st: sg.confidence_sample_static(lsets[i], masked, cu, 0.9, tok, conf, un, stream=st), nsets)
    rec("confidence_sample_static", us, nbytes, "same, through the entry point that allocates nothing")
    del lsets
    # ---- KV page gather / scatter: one request of 4096 tokens (256 pages)
    npg, nsets = 256, 3
    pools = [(torch.randn((P, Hkv, si.PAGE, D), device="cuda", generator=g).to(torch.bfloat16), torch.randn((P, Hkv, si.PAGE, D), device="cuda", generator=g).to(torch.bfloat16)) for _ in range(nsets)]
    ids = [torch.randperm(P, device="cuda", generator=g)[:npg].to(torch.int32) for _ in range(nsets)]
    ks = torch.empty((npg, Hkv, si.PAGE, D), dtype=torch.bfloat16, device="cuda"); vs = torch.empty_like(ks)
    nbytes = 2 * 2 * npg * Hkv * si.PAGE * D * 2 + 4 * npg
    us = timed(lambda i, st: eng.kv_gather(pools[i][0], pools[i][1], ids[i], ks, vs, stream=st), nsets)
    rec("kv_gather", us, nbytes, f"{npg} pages x {Hkv} kv heads (a 4096-token request), K and V")
    us = timed(lambda i, st: eng.kv_scatter(ks, vs, ids[i], pools[i][0], pools[i][1], stream=st), nsets)
    rec("kv_scatter", us, nbytes, "the same pages back into a pool")
    flags = int(eng.device_status())
    for r in out:
        r["device_flags"] = flags
    del pools
    torch.cuda.empty_cache()
    return out


# ------------------------------------------------------------------------------------------------
# Algorithm 1's batches from a simulated arrival trace, through the real kernels
# ------------------------------------------------------------------------------------------------
def measure_sched_series(taus=(512, 1024, 2048, 16384), iters=250, qps=6.0, n_req=96, iter_time=0.04):
    """LLaDA-8B-like geometry, ShareGPT-like arrivals (Table-1 statistics, +1024 MASK).  The arrival clock advances by a fixed
    nominal model-iteration time so that the batch sequence is deterministic; every produced microbatch runs
    kv_write + block_attn on one persistent pool (metadata copied from the scheduler's pinned arrays) and is timed with
    CUDA events."""
    import torch
    import paper_2607_04206_b200 as sg
    geo = si.GEOMETRY["llada"]
    Hq, Hkv, D = geo["num_q_heads"], geo["num_kv_heads"], geo["head_dim"]
    P, MB, W = 24576, 64, (4096 + 15) // 16
    out = []
    for tau in taus:
        MQ = tau + 4096 + 2048 + MB * 32
        tr = si.sched_trace(21, n_req, qps, "sharegpt_like")
        sch = sg.Scheduler(tau=tau, num_pages=P, max_batch=MB, max_total_q=MQ, max_pages_per_req=W, pinned=True)
        eng = sg.Sangam(num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, num_pages=P, max_batch=MB, max_total_q=MQ,
                        max_pages_per_req=W, device=torch.cuda.current_device())
        g = torch.Generator(device="cuda"); g.manual_seed(5)
        kp = torch.randn(P, Hkv, 16, D, dtype=torch.bfloat16, device="cuda", generator=g)
        vp = torch.randn(P, Hkv, 16, D, dtype=torch.bfloat16, device="cuda", generator=g)
        q = torch.randn(MQ, Hq, D, dtype=torch.bfloat16, device="cuda", generator=g)
        kn = torch.randn(MQ, Hkv, D, dtype=torch.bfloat16, device="cuda", generator=g)
        vn = torch.randn(MQ, Hkv, D, dtype=torch.bfloat16, device="cuda", generator=g)
        o = torch.empty_like(q)
        d_cu = torch.zeros(MB + 1, dtype=torch.int32, device="cuda"); d_cl = torch.zeros(MB, dtype=torch.int32, device="cuda")
        d_bt = torch.zeros(MB, W, dtype=torch.int32, device="cuda"); d_sm = torch.zeros(MQ, dtype=torch.int32, device="cuda")
        stream = torch.cuda.Stream()
        steps_left, nxt, gpu_us, host_us, toks, pre_toks, ndec, hybrid = {}, 0, [], [], [], [], [], 0
        scale = float(1.0 / np.sqrt(D))
        for it in range(iters):
            now = it * iter_time
            t0 = time.perf_counter()
            while nxt < n_req and tr["arrival"][nxt] <= now:
                sch.submit(nxt, float(tr["arrival"][nxt]), int(tr["prompt_len"][nxt]), int(tr["response_len"][nxt]), int(tr["output_len"][nxt]))
                nxt += 1
            bb = sch.next()
            t_host = time.perf_counter() - t0
            R, nd, tq = bb.batch, bb.num_decodes, bb.total_q
            ids = sch.arrays["req_ids"][:R].copy()
            if R > 0:
                with torch.cuda.stream(stream):
                    d_cu[:R + 1].copy_(sch.tensors["cu_q_lens"][:R + 1], non_blocking=True)
                    d_cl[:R].copy_(sch.tensors["ctx_lens"][:R], non_blocking=True)
                    d_bt[:R].copy_(sch.tensors["block_table"][:R], non_blocking=True)
                    d_sm[:tq].copy_(sch.tensors["slot_mapping"][:tq], non_blocking=True)
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(stream)
                    eng.kv_write(kn[:tq], vn[:tq], d_sm[:tq], kp, vp, stream=stream)
                    eng.block_attn(q[:tq], kp, vp, d_bt[:R], d_cu[:R + 1], d_cl[:R], scale, o[:tq], stream=stream)
                    e1.record(stream)
                    e1.synchronize()
                gpu_us.append(e0.elapsed_time(e1) * 1e3)
                toks.append(tq); pre_toks.append(tq - 32 * nd); ndec.append(nd); hybrid += int(nd > 0 and R > nd)
            done = []
            for rid in ids[:nd]:
                # decodes keep their block index in the scheduler; the trace's step counts are consumed in order per request
                key = int(rid)
                cnt = steps_left.setdefault(key, [0, 0])           # [block index, steps taken in it]
                cnt[1] += 1
                fin = cnt[1] >= int(tr["steps"][key, cnt[0]])
                if fin:
                    cnt[0] += 1; cnt[1] = 0
                done.append(1 if fin else 0)
            t1 = time.perf_counter()
            sch.complete(done)
            host_us.append((t_host + time.perf_counter() - t1) * 1e6)
        a = np.asarray(gpu_us)
        out.append({"tau": tau, "iterations": iters, "iterations_with_work": int(len(a)), "requests_submitted": nxt, "qps": qps,
                    "gpu_us_mean": round(float(a.mean()), 1), "gpu_us_p50": round(float(np.percentile(a, 50)), 1),
                    "gpu_us_p99": round(float(np.percentile(a, 99)), 1), "gpu_us_max": round(float(a.max()), 1),
                    "tokens_per_iteration_mean": round(float(np.mean(toks)), 1), "prefill_tokens_per_iteration_mean": round(float(np.mean(pre_toks)), 1),
                    "prefill_tokens_per_iteration_max": int(np.max(pre_toks)), "decodes_per_iteration_mean": round(float(np.mean(ndec)), 2),
                    "hybrid_iterations": hybrid, "scheduler_host_us_mean": round(float(np.mean(host_us)), 2),
                    "device_flags": int(eng.device_status()), "waiting_at_end": sch.query(1), "in_flight_at_end": sch.query(2)})
        del kp, vp, q, kn, vn, o, eng, sch
        torch.cuda.empty_cache()
    return out


if __name__ == "__main__":
    sys.exit(main())
