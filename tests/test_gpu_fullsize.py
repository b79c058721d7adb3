"""-m gpu parity at BASELINE.json's full sizes, in the launch configuration bench.py times (CUDA-graph replay
of kv_write + block_attn over bench.Workload): KV pools bit-exact against the oracle, attention checked on a
stratified row sample the oracle computes one by one (tile-edge rows + seeded random rows, all heads), and on
every element against the CUDA-core cross-check kernel."""
import numpy as np
import pytest

import sangam_inputs as si
from gpu_harness import MAX_ABS, MEAN_ABS, bits_of, compare

pytestmark = pytest.mark.gpu

# Regression tripwire, tighter than the north-star gate: 5x the healthy error scale of the arithmetic (bf16 P and output,
# fp32 accumulation: max-abs / mean-abs 5.6e-4 / 9.4e-5 at c ~ 900, 2.9e-4 / 4.0e-5 at
# c ~ 5400; configs 4 and 5 mix contexts of 1000 .. 6000).  At c ~ 5400 a dropped 16-token page PASSES 2e-2 / 2e-3, so the
# gate alone would not notice it.
CEILING = {2: (2.8e-3, 4.7e-4), 3: (1.5e-3, 2.0e-4), 4: (2.8e-3, 3.0e-4), 5: (2.8e-3, 3.0e-4)}


@pytest.mark.parametrize("cfg,per_req,kernel", [(2, 32, 0), (3, 32, 0), (3, 32, 3), (4, 24, 0), (5, 16, 0)],
                         ids=["config2", "config3", "config3-gqa_pair_kernel", "config4", "config5"])
def test_full_size_config(oracle, cfg, per_req, kernel, monkeypatch):
    import torch
    import bench
    monkeypatch.setattr(bench, "DISPATCH", kernel)      # 0: the library's choice (what bench.py times); 3: the CTA-pair kernel
    b = si.CONFIGS[cfg]()
    w = bench.Workload(b, 1)
    w.capture()
    s = w.sets[0]
    s["out"].fill_(float("nan"))
    w.iter_graphs[0].replay()
    torch.cuda.synchronize()
    # pages: bit-exact, whole pools (bench pools start zero-filled, so the oracle's do too)
    rows = si.sample_rows(b, per_request=per_req)
    ref, kp, vp = oracle.iteration(b, rows=rows, poison=False)
    assert np.array_equal(bits_of(s["kp"]), kp), "K pool differs"
    assert np.array_equal(bits_of(s["vp"]), vp), "V pool differs"
    del kp, vp
    mx, mean = compare(s["out"], ref, rows=rows)
    print(f"config{cfg} full size, {len(rows)} sampled rows x {b.num_q_heads} heads: max-abs {mx:.3e} mean-abs {mean:.3e}")
    assert mx <= MAX_ABS and mean <= MEAN_ABS
    assert mx <= CEILING[cfg][0] and mean <= CEILING[cfg][1], "more than 5x the healthy error scale of this shape"
    # every element against the CUDA-core kernel (itself oracle-checked on the sample above)
    out_tc = si.bf16_bits_to_f64(bits_of(s["out"]))
    simt = torch.full_like(s["out"], float("nan"))
    w.eng.block_attn(s["q"], s["kp"], s["vp"], w.block_table, w.cu_q_lens, w.ctx_lens, float(b.scale), simt, simt=True)
    torch.cuda.synchronize()
    mx_s, mean_s = compare(simt, ref, rows=rows)
    assert mx_s <= MAX_ABS and mean_s <= MEAN_ABS
    out_simt = si.bf16_bits_to_f64(bits_of(simt))
    assert np.all(np.isfinite(out_tc))
    d = np.abs(out_tc - out_simt)
    print(f"config{cfg} tcgen05 vs simt over all {d.size} elements: max {d.max():.3e} mean {d.mean():.3e}")
    assert d.max() <= MAX_ABS and d.mean() <= MEAN_ABS
    # identical replays are bit-identical
    first = bits_of(s["out"]).copy()
    w.iter_graphs[0].replay()
    torch.cuda.synchronize()
    assert np.array_equal(first, bits_of(s["out"]))
    assert w.eng.device_status() == 0
    # back-to-back replays (kv_write -> attention -> combine with no host sync in between): timing-dependent
    # protocol slips (a regression once showed up only here, in the hybrid config) would raise a device flag
    # or change bits
    for _ in range(3):
        for _ in range(60):
            w.iter_graphs[0].replay()
        torch.cuda.synchronize()
        assert w.eng.device_status() == 0
        assert np.array_equal(first, bits_of(s["out"]))


def test_graph_replay_with_changed_lengths_at_config5_capacities(oracle):
    """One CUDA graph of kv_write -> block_attn captured at the hybrid config's capacities (34 requests, 32/32 heads,
    D 128, contexts up to 4096) and replayed with different lengths, pages and data in the same
    buffers: decode contexts redrawn, the two prefills shortened / swapped, fewer requests than captured.  The
    two-stream kernel's dynamic unit hand-out runs under one capture with changing totals.  Every replay is checked
    against the oracle on a stratified row sample, pools bit-exactly, identical replays bit-identically."""
    import torch
    import paper_2607_04206_b200 as sg
    from gpu_harness import t_bf16, t_i32
    b0 = si.config5()
    Hq, Hkv, D, R = b0.num_q_heads, b0.num_kv_heads, b0.head_dim, b0.batch
    W, P = b0.max_pages_per_req, b0.num_pages + 256
    QCAP = b0.total_q
    eng = sg.Sangam(num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, num_pages=P, max_batch=R, max_total_q=QCAP, max_pages_per_req=W)
    dev = "cuda"
    q = torch.zeros(QCAP, Hq, D, dtype=torch.bfloat16, device=dev)
    out = torch.zeros_like(q)
    kn = torch.zeros(QCAP, Hkv, D, dtype=torch.bfloat16, device=dev)
    vn = torch.zeros_like(kn)
    slot = torch.full((QCAP,), -1, dtype=torch.int32, device=dev)
    bt = torch.zeros(R, W, dtype=torch.int32, device=dev)
    cu = torch.zeros(R + 1, dtype=torch.int32, device=dev)
    cl = torch.zeros(R, dtype=torch.int32, device=dev)
    kp = torch.zeros(P, Hkv, 16, D, dtype=torch.bfloat16, device=dev)
    vp = torch.zeros_like(kp)
    stream = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()

    def batch(seed, n_dec, pre):
        g = np.random.default_rng(seed)
        dec_ctx = g.integers(512, 4096, n_dec, endpoint=True)
        return si.make_batch("replay", seed, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, decode_ctx=dec_ctx, decode_q=32,
                             response=256, prefill_lens=pre, min_width=W)

    def fill(b):
        assert b.num_pages <= P and b.total_q <= QCAP and b.batch <= R and b.max_pages_per_req == W
        kpf = np.zeros((P, Hkv, 16, D), np.uint16); vpf = np.zeros_like(kpf)
        oracle.kv_write(b.k_cache, b.v_cache, b.slot_cache, kpf, vpf)
        kp.copy_(t_bf16(kpf)); vp.copy_(t_bf16(vpf))
        n, t = b.batch, b.total_q
        q.zero_(); q[:t].copy_(t_bf16(b.q))
        kn.zero_(); vn.zero_(); kn[:t].copy_(t_bf16(b.k_new)); vn[:t].copy_(t_bf16(b.v_new))
        slot.fill_(-1); slot[:t].copy_(t_i32(b.slot_new))
        bt.zero_(); bt[:n].copy_(t_i32(b.block_table))
        cuv = np.full(R + 1, t, np.int32); cuv[:n + 1] = b.cu_q_lens; cu.copy_(t_i32(cuv))
        clv = np.zeros(R, np.int32); clv[:n] = b.ctx_lens; cl.copy_(t_i32(clv))
        oracle.kv_write(b.k_new, b.v_new, b.slot_new, kpf, vpf)
        rows = si.sample_rows(b, per_request=12)
        ref = oracle.block_attn(b.q, kpf, vpf, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale, rows=rows)
        return rows, ref, kpf, vpf

    cases = [b0, batch(71, 32, [3000, 4096]), batch(72, 30, [4096, 1500]), batch(73, 32, [4096]), b0]
    fill(cases[0])
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):
        for _ in range(2):
            eng.kv_write(kn, vn, slot, kp, vp, stream=stream)
            eng.block_attn(q, kp, vp, bt, cu, cl, float(b0.scale), out, stream=stream)
        stream.synchronize()
        with torch.cuda.graph(graph, stream=stream):
            eng.kv_write(kn, vn, slot, kp, vp, stream=stream)
            eng.block_attn(q, kp, vp, bt, cu, cl, float(b0.scale), out, stream=stream)
    for i, b in enumerate(cases):
        rows, ref, kpf, vpf = fill(b)
        torch.cuda.synchronize()
        out.fill_(float("nan"))
        graph.replay(); torch.cuda.synchronize()
        mx, mean = compare(out, ref, rows=rows)
        print(f"config-5-capacity replay {i} ({b.batch} requests, {b.total_q} rows): max-abs {mx:.3e} mean-abs {mean:.3e}")
        assert mx <= CEILING[5][0] and mean <= CEILING[5][1]
        assert np.array_equal(bits_of(kp), kpf) and np.array_equal(bits_of(vp), vpf)
        first = bits_of(out[:b.total_q]).copy()
        assert np.all(np.isfinite(si.bf16_bits_to_f64(first)))
        graph.replay(); torch.cuda.synchronize()
        assert np.array_equal(first, bits_of(out[:b.total_q]))
    assert eng.device_status() == 0
