"""Seeded synthetic inputs for the Sangam hot path (test/bench infrastructure).

This module is the ONLY code shared by the CUDA path and the CPU oracle.  It holds
none of the method's arithmetic: it draws lengths, a page permutation and N(0,1)
tensors, rounds them to bf16 bit patterns and lays out the *metadata* the C ABI
consumes (`cu_q_lens`, `ctx_lens`, `block_table`, `slot_mapping`).  Nothing here
computes a logit, a softmax or a scatter.

Recipe: `g = numpy.random.default_rng(seed)`
and, in this fixed order, (1) lengths, (2) the block index of every decode request,
(3) `perm = g.permutation(P)`, (4) K cache content, (5) V cache content, (6) the
iteration's new k, v, (7) q.  All tensors are `g.standard_normal(float32)` rounded
to bf16 (round-to-nearest-even) and kept as uint16 bit patterns.

The workloads stand in for the paper's LLaDA-8B-Instruct/ShareGPT and
Dream-7B-Instruct/arXiv runs: page 16, block 32, bf16
(PAPER.md:279); MHA for LLaDA, GQA for Dream.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

PAGE = 16  # KV page size in tokens
POISON = np.uint16(0x7FC1)  # a bf16 NaN: fills every slot no request owns


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit pattern (uint16), round to nearest even.  Finite inputs only."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    return ((u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    """bf16 bit pattern (uint16) -> float64, exact widening."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def _normal_bits(g: np.random.Generator, shape) -> np.ndarray:
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.uint16)
    step = 1 << 24  # bounded float32 scratch
    for i in range(0, n, step):
        m = min(step, n - i)
        out[i:i + m] = f32_to_bf16_bits(g.standard_normal(m, dtype=np.float32))
    return out.reshape(shape)


@dataclass
class Batch:
    """One serving iteration's inputs (host side, numpy)."""
    name: str
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    num_pages: int                 # P, pool capacity
    max_pages_per_req: int         # W, block_table width
    scale: np.float32
    q_lens: np.ndarray             # int32[R]
    ctx_lens: np.ndarray           # int32[R]
    cu_q_lens: np.ndarray          # int32[R+1]
    block_table: np.ndarray        # int32[R][W], -1 padded
    q: np.ndarray                  # uint16[T_q][Hq][D]
    k_cache: np.ndarray            # uint16[sum c][Hkv][D]   cache content before the iteration
    v_cache: np.ndarray
    slot_cache: np.ndarray         # int32[sum c]            slots of every context position
    k_new: np.ndarray              # uint16[T_new][Hkv][D]   this iteration's fresh K/V rows
    v_new: np.ndarray
    slot_new: np.ndarray           # int32[T_new]
    kinds: list = field(default_factory=list)   # "decode" | "prefill" per request

    @property
    def batch(self) -> int:
        return int(self.q_lens.shape[0])

    @property
    def total_q(self) -> int:
        return int(self.cu_q_lens[-1])

    @property
    def cu_ctx(self) -> np.ndarray:
        return np.concatenate([[0], np.cumsum(self.ctx_lens)]).astype(np.int64)

    def flops(self) -> float:
        """F = 4 Hq D sum_r q_r c_r."""
        return 4.0 * self.num_q_heads * self.head_dim * float(np.sum(self.q_lens.astype(np.int64) * self.ctx_lens.astype(np.int64)))

    def attn_bytes(self) -> float:
        """B_attn = Q + O + K/V once + metadata."""
        R = self.batch
        qo = 2 * 2 * self.total_q * self.num_q_heads * self.head_dim
        kv = 2 * 2 * self.num_kv_heads * self.head_dim * int(np.sum(self.ctx_lens.astype(np.int64)))
        meta = 4 * (2 * R + 1 + int(np.sum((self.ctx_lens.astype(np.int64) + PAGE - 1) // PAGE)))
        return float(qo + kv + meta)

    def write_bytes(self) -> float:
        """B_write = 2 * (k + v rows) read and written + slots."""
        t = int(self.slot_new.shape[0])
        return float(2 * (2 * 2 * t * self.num_kv_heads * self.head_dim) + 4 * t)


def make_batch(name: str, seed: int, *, num_q_heads: int, num_kv_heads: int, head_dim: int,
               decode_ctx, decode_q: int, response: int, prefill_lens=(), lengths_fn=None,
               pool_slack: float = 1.25, min_width: int = 0) -> Batch:
    """Build a batch of `decode` requests followed by `prefill` requests (Alg. 1 seats
    decodes first).

    lengths_fn(g) -> (decode_ctx array, prefill_lens array) draws the lengths from the
    generator first, so the draw order of the recipe is kept; decode_ctx / prefill_lens
    are used when lengths_fn is None.
    """
    g = np.random.default_rng(seed)
    if lengths_fn is not None:
        decode_ctx, prefill_lens = lengths_fn(g)
    decode_ctx = np.asarray(decode_ctx, dtype=np.int64).reshape(-1)
    prefill_lens = np.asarray(prefill_lens, dtype=np.int64).reshape(-1)
    n_dec, n_pre = len(decode_ctx), len(prefill_lens)
    R = n_dec + n_pre
    ctx = np.concatenate([decode_ctx, prefill_lens]).astype(np.int64)
    qlen = np.concatenate([np.full(n_dec, decode_q, dtype=np.int64), prefill_lens]).astype(np.int64)
    # (2) which block of the response region is "current" for each decode
    blocks_per_resp = max(1, response // max(1, decode_q))
    blk = np.array([int(g.integers(0, blocks_per_resp)) for _ in range(n_dec)], dtype=np.int64)
    # (3) page permutation
    pages_per_req = (ctx + PAGE - 1) // PAGE
    n_owned = int(pages_per_req.sum())
    P = int(np.ceil(pool_slack * n_owned)) + 64
    perm = g.permutation(P)
    W = max(int(pages_per_req.max()) if R else 1, min_width, 1)
    block_table = np.full((R, W), -1, dtype=np.int32)
    nxt = 0
    for r in range(R):
        n = int(pages_per_req[r])
        block_table[r, :n] = perm[nxt:nxt + n]
        nxt += n
    # slots of every context position
    slot_cache = np.empty(int(ctx.sum()), dtype=np.int32)
    o = 0
    for r in range(R):
        j = np.arange(int(ctx[r]))
        slot_cache[o:o + len(j)] = block_table[r, j // PAGE].astype(np.int64) * PAGE + (j % PAGE)
        o += len(j)
    cu_ctx = np.concatenate([[0], np.cumsum(ctx)])
    # (4), (5) cache content
    k_cache = _normal_bits(g, (int(ctx.sum()), num_kv_heads, head_dim))
    v_cache = _normal_bits(g, (int(ctx.sum()), num_kv_heads, head_dim))
    # rows produced this iteration: a decode rewrites its current block, a prefill every row
    new_slots = []
    for r in range(R):
        if r < n_dec:
            first = int(ctx[r]) - response + int(blk[r]) * decode_q
            pos = np.arange(first, first + decode_q)
        else:
            pos = np.arange(int(ctx[r]))
        new_slots.append(slot_cache[cu_ctx[r] + pos])
    slot_new = np.concatenate(new_slots).astype(np.int32) if new_slots else np.zeros(0, np.int32)
    # (6) new k, v   (7) q
    k_new = _normal_bits(g, (len(slot_new), num_kv_heads, head_dim))
    v_new = _normal_bits(g, (len(slot_new), num_kv_heads, head_dim))
    q = _normal_bits(g, (int(qlen.sum()), num_q_heads, head_dim))
    return Batch(
        name=name, num_q_heads=num_q_heads, num_kv_heads=num_kv_heads, head_dim=head_dim,
        num_pages=P, max_pages_per_req=W, scale=np.float32(1.0 / np.sqrt(head_dim)),
        q_lens=qlen.astype(np.int32), ctx_lens=ctx.astype(np.int32),
        cu_q_lens=np.concatenate([[0], np.cumsum(qlen)]).astype(np.int32),
        block_table=block_table, q=q, k_cache=k_cache, v_cache=v_cache, slot_cache=slot_cache,
        k_new=k_new, v_new=v_new, slot_new=slot_new,
        kinds=["decode"] * n_dec + ["prefill"] * n_pre)


# ---------------------------------------------------------------------------------------
# The five BASELINE.json configs.  `scale` < 1 shrinks lengths for CPU-sized parity cases
# (same structure, fewer tokens); scale == 1 is the judged workload.
# ---------------------------------------------------------------------------------------

def config1() -> Batch:
    """tiny correctness case: 2 requests, prompt 64 + response 64, 16 query rows, 4/4 heads, D 64."""
    return make_batch("config1_tiny", 0, num_q_heads=4, num_kv_heads=4, head_dim=64,
                      decode_ctx=[128, 128], decode_q=16, response=64)


def config2(shrink: int = 1) -> Batch:
    """LLaDA-8B-like block decode: batch 8, prompt U[128,1024], response 256, block 32, 32/32 heads."""
    def lens(g):
        p = g.integers(128 // shrink, 1024 // shrink, 8, endpoint=True)
        return p + 256 // shrink, []
    return make_batch("config2_llada_decode", 1, num_q_heads=32, num_kv_heads=32, head_dim=128,
                      decode_ctx=None, decode_q=32, response=256 // shrink, lengths_fn=lens)


def config3(shrink: int = 1) -> Batch:
    """Dream-7B-like GQA block decode: batch 16, prompt U[2048,8192], response 256, 28/4 heads."""
    def lens(g):
        p = g.integers(2048 // shrink, 8192 // shrink, 16, endpoint=True)
        return p + 256 // shrink, []
    return make_batch("config3_dream_gqa_decode", 2, num_q_heads=28, num_kv_heads=4, head_dim=128,
                      decode_ctx=None, decode_q=32, response=256 // shrink, lengths_fn=lens)


def config4(shrink: int = 1) -> Batch:
    """KV refresh prefill: 8 requests, lengths U[1024,6144], full bidirectional self-attention + kv_write."""
    def lens(g):
        return [], g.integers(1024 // shrink, 6144 // shrink, 8, endpoint=True)
    return make_batch("config4_refresh_prefill", 3, num_q_heads=32, num_kv_heads=32, head_dim=128,
                      decode_ctx=None, decode_q=32, response=256, lengths_fn=lens)


def config5(shrink: int = 1) -> Batch:
    """hybrid: 32 decodes (ctx U[512,4096], block 32) + 2 overflow prefills of 4096, one varlen launch."""
    def lens(g):
        c = g.integers(512 // shrink, 4096 // shrink, 32, endpoint=True)
        return c, [4096 // shrink, 4096 // shrink]
    return make_batch("config5_hybrid", 4, num_q_heads=32, num_kv_heads=32, head_dim=128,
                      decode_ctx=None, decode_q=32, response=256 // shrink, lengths_fn=lens)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def custom(seed: int, q_lens, ctx_lens, *, num_q_heads=4, num_kv_heads=4, head_dim=64, pool_slack=1.25,
           min_width: int = 0, new_at_end: bool = False, name: str = "custom") -> Batch:
    """Arbitrary (q_r, c_r) pairs for edge-case tests.  Every request is laid out like a
    prefill whose first q_r rows are queried; K/V for all c_r positions are cache content
    and the 'new' rows rewrite the first min(q_r, c_r) positions."""
    g = np.random.default_rng(seed)
    q_lens = np.asarray(q_lens, dtype=np.int64)
    ctx = np.asarray(ctx_lens, dtype=np.int64)
    R = len(ctx)
    pages_per_req = (ctx + PAGE - 1) // PAGE
    P = int(np.ceil(pool_slack * int(pages_per_req.sum()))) + 64
    perm = g.permutation(P)
    W = max(int(pages_per_req.max()) if R else 1, min_width, 1)
    block_table = np.full((R, W), -1, dtype=np.int32)
    nxt = 0
    for r in range(R):
        n = int(pages_per_req[r])
        block_table[r, :n] = perm[nxt:nxt + n]
        nxt += n
    slot_cache = np.empty(int(ctx.sum()), dtype=np.int32)
    cu_ctx = np.concatenate([[0], np.cumsum(ctx)])
    for r in range(R):
        j = np.arange(int(ctx[r]))
        slot_cache[cu_ctx[r]:cu_ctx[r + 1]] = block_table[r, j // PAGE].astype(np.int64) * PAGE + (j % PAGE)
    k_cache = _normal_bits(g, (int(ctx.sum()), num_kv_heads, head_dim))
    v_cache = _normal_bits(g, (int(ctx.sum()), num_kv_heads, head_dim))
    if new_at_end:   # the rewritten rows are the LAST min(q_r, c_r) positions (a response region at the end of the sequence)
        new_slots = [slot_cache[cu_ctx[r + 1] - min(int(q_lens[r]), int(ctx[r])):cu_ctx[r + 1]] for r in range(R)]
    else:
        new_slots = [slot_cache[cu_ctx[r]:cu_ctx[r] + min(int(q_lens[r]), int(ctx[r]))] for r in range(R)]
    slot_new = np.concatenate(new_slots).astype(np.int32) if R else np.zeros(0, np.int32)
    k_new = _normal_bits(g, (len(slot_new), num_kv_heads, head_dim))
    v_new = _normal_bits(g, (len(slot_new), num_kv_heads, head_dim))
    q = _normal_bits(g, (int(q_lens.sum()), num_q_heads, head_dim))
    return Batch(
        name=name, num_q_heads=num_q_heads, num_kv_heads=num_kv_heads, head_dim=head_dim,
        num_pages=P, max_pages_per_req=W, scale=np.float32(1.0 / np.sqrt(head_dim)),
        q_lens=q_lens.astype(np.int32), ctx_lens=ctx.astype(np.int32),
        cu_q_lens=np.concatenate([[0], np.cumsum(q_lens)]).astype(np.int32),
        block_table=block_table, q=q, k_cache=k_cache, v_cache=v_cache, slot_cache=slot_cache,
        k_new=k_new, v_new=v_new, slot_new=slot_new, kinds=["prefill"] * R)


def empty_pools(b: Batch, poison: bool = True):
    """Fresh K and V pools, uint16[P][Hkv][16][D]; NaN-poisoned for parity runs, zero for timing."""
    shape = (b.num_pages, b.num_kv_heads, PAGE, b.head_dim)
    if poison:
        return np.full(shape, POISON, dtype=np.uint16), np.full(shape, POISON, dtype=np.uint16)
    return np.zeros(shape, dtype=np.uint16), np.zeros(shape, dtype=np.uint16)


def sample_rows(b: Batch, per_request: int = 64, seed: int = 1234) -> np.ndarray:
    """Stratified global q-row sample: tile-edge rows plus seeded random rows."""
    g = np.random.default_rng(seed)
    rows = []
    for r in range(b.batch):
        n = int(b.q_lens[r])
        if n == 0:
            continue
        base = int(b.cu_q_lens[r])
        if n <= per_request:
            rows.extend(range(base, base + n))
            continue
        edge = [0, 1, 63, 64, 127, 128, n - 129, n - 128, n - 65, n - 64, n - 1]
        pick = {e for e in edge if 0 <= e < n}
        while len(pick) < per_request:
            pick.add(int(g.integers(0, n)))
        rows.extend(base + e for e in sorted(pick))
    return np.asarray(rows, dtype=np.int32)


# ---------------------------------------------------------------------------------------
# Seeded synthetic arrival traces for the worker-level scheduler.
# They stand in for the paper's filtered ShareGPT / arXiv-summarization traces,
# which are not in the container: lengths are drawn from log-normal laws fitted to the MEDIAN and P99
# of Table 1 (sigma = ln(P99 / median) / 2.326), requests above 4096 tokens are clipped like the paper's
# filter, 1024 / 512 MASK positions are appended, arrivals are Poisson.  No trace item is
# reproduced.  Only draws live here: no scheduling decision is taken in this module.
# ---------------------------------------------------------------------------------------
TRACE_STATS = {   # name: (prompt median, prompt P99, output median, output P99, appended MASK tokens)
    "sharegpt_like": (795, 2007, 266, 874, 1024),
    "arxiv_like": (2827, 3923, 162, 360, 512),
}


def sched_trace(seed: int, n: int, qps: float, kind: str = "sharegpt_like", block: int = 32, max_steps: int = 12):
    """n requests: dict of arrays arrival [s], prompt_len, response_len, output_len, and steps[n][max blocks]
    (denoising iterations each block takes: the paper's confidence-threshold unmasking makes this data
    dependent; here uniform integers in [2, max_steps])."""
    pm, p99, om, o99, resp = TRACE_STATS[kind]
    g = np.random.default_rng(seed)
    arrival = np.cumsum(g.exponential(1.0 / qps, n))
    out = np.exp(np.log(om) + np.log(o99 / om) / 2.326 * g.standard_normal(n))
    out = np.clip(np.rint(out), 1, resp).astype(np.int32)
    prm = np.exp(np.log(pm) + np.log(p99 / pm) / 2.326 * g.standard_normal(n))
    prm = np.clip(np.rint(prm), 16, 4096 - out).astype(np.int32)
    nblk = (resp + block - 1) // block
    steps = g.integers(2, max_steps, (n, nblk), endpoint=True).astype(np.int32)
    return {"arrival": arrival, "prompt_len": prm, "response_len": np.full(n, resp, np.int32), "output_len": out,
            "steps": steps, "block": block, "kind": kind}


# ---------------------------------------------------------------------------------------
# Variant shapes: the same kernels at other points of the paper's workloads.
# ---------------------------------------------------------------------------------------
GEOMETRY = {"llada": dict(num_q_heads=32, num_kv_heads=32, head_dim=128),      # LLaDA-8B-like MHA
            "dream": dict(num_q_heads=28, num_kv_heads=4, head_dim=128)}       # Dream-7B-like GQA 7:1


def _trace_prompts(g: np.random.Generator, n: int, kind: str, shrink: int = 1):
    pm, p99, _, _, resp = TRACE_STATS[kind]
    prm = np.exp(np.log(pm) + np.log(p99 / pm) / 2.326 * g.standard_normal(n))
    return np.clip(np.rint(prm), 16, 4096 - resp).astype(np.int64) // shrink, resp // shrink


def paper_decode(model: str = "llada", trace: str = "sharegpt_like", batch: int = 16, seed: int = 11, shrink: int = 1) -> Batch:
    """Block decode at the paper's real sequence lengths: prompts with the trace's Table-1 statistics
    (<= 4096 tokens), 1024 (ShareGPT) / 512 (arXiv) appended MASK positions, block 32."""
    def lens(g):
        prm, resp = _trace_prompts(g, batch, trace, shrink)
        return prm + resp, []
    resp = TRACE_STATS[trace][4] // shrink
    return make_batch(f"{model}_{trace}_decode", seed, decode_ctx=None, decode_q=32 // (1 if shrink == 1 else 1), response=resp,
                      lengths_fn=lens, **GEOMETRY[model])


def dkv_refresh(model: str = "llada", trace: str = "sharegpt_like", batch: int = 8, seed: int = 12, shrink: int = 1) -> Batch:
    """dKV-Cache-PD style refresh: only the RESPONSE region is recomputed -- its rows are the queries and the
    rewritten K/V rows -- while the prompt's K/V stay as cached; the context is still prompt + response."""
    g = np.random.default_rng(seed)
    prm, resp = _trace_prompts(g, batch, trace, shrink)
    return custom(seed, [resp] * batch, (prm + resp).tolist(), new_at_end=True, name=f"{model}_{trace}_dkv_refresh", **GEOMETRY[model])


def fig3_point(model: str, batch: int, seed: int = 13, ctx: int = 1024) -> Batch:
    """One point of the Fig.-3-shaped sweep: `batch` block decodes at sequence length 1024, block 32."""
    return make_batch(f"fig3_{model}_b{batch}", seed + batch, decode_ctx=[ctx] * batch, decode_q=32, response=256, **GEOMETRY[model])


VARIANTS = {
    "llada_sharegpt_decode": lambda shrink=1: paper_decode("llada", "sharegpt_like", 16, 11, shrink),
    "dream_arxiv_decode": lambda shrink=1: paper_decode("dream", "arxiv_like", 16, 14, shrink),
    "llada_dkv_refresh": lambda shrink=1: dkv_refresh("llada", "sharegpt_like", 8, 12, shrink),
    "dream_dkv_refresh": lambda shrink=1: dkv_refresh("dream", "arxiv_like", 8, 15, shrink),
}
FIG3_BATCHES = (1, 2, 4, 8, 16, 32, 64)
