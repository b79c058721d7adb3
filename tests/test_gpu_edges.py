"""-m gpu adversarial and edge-case tests of the tcgen05 path (SURVEY.md 8(c) "GPU-side adversarial tests")."""
import numpy as np
import pytest

import sangam_inputs as si
from gpu_harness import MAX_ABS, MEAN_ABS, DeviceBatch, bits_of, compare, t_bf16, t_i32

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("hq,hkv,d", [(4, 4, 64), (8, 8, 128), (14, 2, 128), (7, 1, 64)])
def test_length_edges(oracle, hq, hkv, d, dispatch):
    q_lens = [0, 1, 16, 32, 33, 127, 128, 129, 5, 3, 2, 40]
    ctx = [5, 1, 15, 16, 17, 127, 128, 129, 255, 256, 257, 0]
    b = si.custom(41, q_lens, ctx, num_q_heads=hq, num_kv_heads=hkv, head_dim=d)
    ref, kp, vp = oracle.iteration(b)
    db = DeviceBatch(b)
    out = db.iteration()
    assert np.array_equal(bits_of(db.k_pages), kp) and np.array_equal(bits_of(db.v_pages), vp)
    mx, mean = compare(out, ref)
    print(f"edges Hq={hq} Hkv={hkv} D={d}: max-abs {mx:.3e} mean-abs {mean:.3e}")
    assert mx <= MAX_ABS and mean <= MEAN_ABS
    # c = 0 rows are exact zeros; c = 1 rows equal v_0 bit-exactly (pin 8 on the GPU)
    got = bits_of(out)
    lo, hi = b.cu_q_lens[11], b.cu_q_lens[12]
    assert np.all(got[lo:hi] == 0)
    G = hq // hkv
    v0 = vp[b.block_table[1, 0], :, 0, :]                     # [Hkv][D]
    assert np.array_equal(got[b.cu_q_lens[1]], np.repeat(v0, G, axis=0))
    assert db.eng.device_status() == 0


@pytest.mark.parametrize("ctx,d,g", [(700, 128, 1), (1500, 128, 7), (300, 64, 1)])
def test_identity_needle_prefill(oracle, ctx, d, g, dispatch):
    """q_t = beta * k_t: row t's logit at j = t dominates, so out[t] == V[t] to 1 bf16 ulp for every t.
    Covers every context position, page mapping and tile boundary in one launch."""
    b = si.custom(42, [ctx], [ctx], num_q_heads=g, num_kv_heads=1, head_dim=d)
    k = si.bf16_bits_to_f64(b.k_cache)[:, 0, :]                        # [c][D]
    q = np.repeat((8.0 * k)[:, None, :], g, axis=1).astype(np.float32)  # exact: power-of-two scaling
    b.q = si.f32_to_bf16_bits(q)
    b.slot_new = b.slot_new[:0]; b.k_new = b.k_new[:0]; b.v_new = b.v_new[:0]
    db = DeviceBatch(b)
    out = db.iteration()
    got = si.bf16_bits_to_f64(bits_of(out))
    v = si.bf16_bits_to_f64(b.v_cache)[:, 0, :]
    err = np.abs(got - v[:, None, :])
    ulp = np.maximum(np.abs(v[:, None, :]) * 2.0 ** -7, 2.0 ** -126)
    assert np.all(err <= ulp + 1e-30), f"needle mismatch: max err {err.max():.3e}"


def test_needle_sweep_decode(oracle, dispatch):
    """Dominant position on the first/last slot of every page and on c-1 (decode shape, split-KV active)."""
    c, d = 1000, 128
    pos = sorted(set([p for pg in range((c + 15) // 16) for p in (16 * pg, min(16 * pg + 15, c - 1))] + [c - 1]))
    b = si.custom(43, [len(pos)], [c], num_q_heads=2, num_kv_heads=2, head_dim=d)
    k = si.bf16_bits_to_f64(b.k_cache)                                  # [c][2][D]
    q = (8.0 * k[pos]).astype(np.float32)                               # row i looks for position pos[i]
    b.q = si.f32_to_bf16_bits(q)
    b.slot_new = b.slot_new[:0]; b.k_new = b.k_new[:0]; b.v_new = b.v_new[:0]
    db = DeviceBatch(b)
    got = si.bf16_bits_to_f64(bits_of(db.iteration()))
    v = si.bf16_bits_to_f64(b.v_cache)[pos]
    assert np.all(np.abs(got - v) <= np.abs(v) * 2.0 ** -7 + 1e-30)


def test_poison_independence_and_bad_block_table_tail(oracle, dispatch):
    b = si.config2(4)
    ref, _, _ = oracle.iteration(b)
    db = DeviceBatch(b, poison=True)
    bt = b.block_table.copy()
    bt[bt < 0] = 2 ** 30                      # entries past ceil(c/16) must never be dereferenced
    db.block_table = t_i32(bt)
    a = bits_of(db.iteration()).copy()
    db2 = DeviceBatch(b, poison=False)
    z = bits_of(db2.iteration())
    assert np.array_equal(a, z), "output depends on poisoned tail slots / unreferenced pages"
    mx, mean = compare(db.out, ref)
    assert mx <= MAX_ABS and mean <= MEAN_ABS
    assert db.eng.device_status() == 0


def test_bitwise_reproducible(oracle, dispatch):
    b = si.config3(8)
    db = DeviceBatch(b)
    a = bits_of(db.iteration()).copy()
    for _ in range(3):
        db.out.fill_(float("nan"))
        db.attend()
        import torch
        torch.cuda.synchronize()
        assert np.array_equal(a, bits_of(db.out))


def test_row_independence_decode_vs_prefill(oracle):
    """A decode whose q rows equal rows of a prefill's Q over the same KV gives the prefill's rows (pin 14)
    within the tolerance (different tilings, same math)."""
    b = si.custom(44, [300], [300], num_q_heads=4, num_kv_heads=4, head_dim=128)
    db = DeviceBatch(b)
    full = si.bf16_bits_to_f64(bits_of(db.iteration())).copy()
    import torch
    sub = slice(100, 132)
    q2 = db.q[sub].contiguous()
    out2 = torch.empty_like(q2)
    db.eng.block_attn(q2, db.k_pages, db.v_pages, db.block_table, t_i32(np.array([0, 32])), db.ctx_lens,
                      float(b.scale), out2)
    torch.cuda.synchronize()
    got = si.bf16_bits_to_f64(bits_of(out2))
    assert np.max(np.abs(got - full[sub])) <= 4e-3


@pytest.mark.parametrize("mode", [0, 1, 2], ids=["auto", "prefill_kernel", "decode_kernel"])
def test_graph_replay_with_changed_lengths(oracle, mode):
    """Capture kv_write -> block_attn once at fixed capacities, replay with different lengths, pages and
    data written into the same buffers; every replay checked against the oracle; identical replays are
    bit-identical (CUDA Graphs: PAPER.md:258)."""
    import torch
    import paper_2607_04206_b200 as sg
    Hq, Hkv, D, R, W, P, QCAP, TNEW = 8, 8, 128, 6, 40, 400, 6 * 64, 6 * 64
    eng = sg.Sangam(num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, num_pages=P, max_batch=R, max_total_q=QCAP,
                    max_pages_per_req=W)
    eng.set_dispatch(mode)
    dev = "cuda"
    q = torch.zeros(QCAP, Hq, D, dtype=torch.bfloat16, device=dev)
    out = torch.zeros_like(q)
    kn = torch.zeros(TNEW, Hkv, D, dtype=torch.bfloat16, device=dev)
    vn = torch.zeros_like(kn)
    slot = torch.full((TNEW,), -1, dtype=torch.int32, device=dev)
    bt = torch.zeros(R, W, dtype=torch.int32, device=dev)
    cu = torch.zeros(R + 1, dtype=torch.int32, device=dev)
    cl = torch.zeros(R, dtype=torch.int32, device=dev)
    kp = torch.zeros(P, Hkv, 16, D, dtype=torch.bfloat16, device=dev)
    vp = torch.zeros_like(kp)
    stream = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()

    def fill(seed, q_lens, ctx):
        b = si.custom(seed, q_lens, ctx, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, min_width=W)
        assert b.num_pages <= P and b.total_q <= QCAP and len(b.slot_new) <= TNEW
        kpn, vpn = si.empty_pools(b)
        kpf = np.full((P, Hkv, 16, D), si.POISON, np.uint16); vpf = kpf.copy()
        oracle.kv_write(b.k_cache, b.v_cache, b.slot_cache, kpf, vpf)          # cache content (setup)
        kp.copy_(t_bf16(kpf)); vp.copy_(t_bf16(vpf))
        n = b.batch
        q.zero_(); q[:b.total_q].copy_(t_bf16(b.q))
        kn.zero_(); kn[:len(b.slot_new)].copy_(t_bf16(b.k_new)); vn.zero_(); vn[:len(b.slot_new)].copy_(t_bf16(b.v_new))
        slot.fill_(-1); slot[:len(b.slot_new)].copy_(t_i32(b.slot_new))
        bt.zero_(); bt[:n].copy_(t_i32(b.block_table[:, :W]))
        cuv = np.full(R + 1, b.total_q, np.int32); cuv[:n + 1] = b.cu_q_lens
        cu.copy_(t_i32(cuv))
        clv = np.zeros(R, np.int32); clv[:n] = b.ctx_lens
        cl.copy_(t_i32(clv))
        oracle.kv_write(b.k_new, b.v_new, b.slot_new, kpf, vpf)
        ref = oracle.block_attn(b.q, kpf, vpf, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
        return b, ref, kpf

    cases = [(51, [32] * 6, [600, 300, 129, 640, 77, 500]), (52, [64, 0, 32, 5], [200, 100, 640, 33]),
             (53, [10, 20, 30, 40, 50, 60], [16, 32, 48, 64, 80, 96]),
             # the per-CTA plan cache is keyed by the lengths: one context longer by one position (a new tile), one
             # query row fewer, the first batch again (each case runs as a miss, then as a hit, bit-identically)
             (54, [32] * 6, [600, 300, 129, 640, 77, 513]), (55, [32] * 5 + [31], [600, 300, 129, 640, 77, 513]),
             (51, [32] * 6, [600, 300, 129, 640, 77, 500])]
    b, ref, _ = fill(*cases[0])
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):
        for _ in range(2):   # warm-up outside capture
            eng.kv_write(kn, vn, slot, kp, vp, stream=stream)
            eng.block_attn(q, kp, vp, bt, cu, cl, float(b.scale), out, stream=stream)
        stream.synchronize()
        with torch.cuda.graph(graph, stream=stream):
            eng.kv_write(kn, vn, slot, kp, vp, stream=stream)
            eng.block_attn(q, kp, vp, bt, cu, cl, float(b.scale), out, stream=stream)
    for case in cases:
        b, ref, kpf = fill(*case)
        torch.cuda.synchronize()
        out.fill_(float("nan"))
        graph.replay(); torch.cuda.synchronize()
        mx, mean = compare(out[:b.total_q], ref)
        print(f"graph replay seed {case[0]}: max-abs {mx:.3e} mean-abs {mean:.3e}")
        assert mx <= MAX_ABS and mean <= MEAN_ABS
        assert np.array_equal(bits_of(kp), kpf)
        first = bits_of(out[:b.total_q]).copy()
        graph.replay(); torch.cuda.synchronize()
        assert np.array_equal(first, bits_of(out[:b.total_q]))
    assert eng.device_status() == 0


@pytest.mark.parametrize("scale", [-0.0883883461356163, 0.0, 0.35])
def test_scale_sign_and_magnitude(oracle, scale, dispatch):
    """The logit scale is a caller-supplied float (reading S5): negative (the kernel flips the sign of S and works
    with |scale|), zero (uniform weights: out = mean of V, oracle pin 7) and large (exercises the lazy rescale:
    logits of up to +-40 in log2 units move the reference maximum many times)."""
    b = si.custom(47, [40, 150, 7], [300, 420, 129], num_q_heads=8, num_kv_heads=2, head_dim=128)
    b.scale = np.float32(scale)
    ref, kp, vp = oracle.iteration(b)
    db = DeviceBatch(b)
    out = db.iteration()
    mx, mean = compare(out, ref)
    print(f"scale {scale}: max-abs {mx:.3e} mean-abs {mean:.3e}")
    assert mx <= MAX_ABS and mean <= MEAN_ABS
    assert db.eng.device_status() == 0


def test_more_than_32_requests(oracle, dispatch):
    """The planner keeps the first 32 requests' metadata in registers and reads the rest from global memory."""
    rng = np.random.default_rng(5)
    R = 45
    q_lens = rng.integers(0, 40, R).tolist()
    ctx = rng.integers(1, 300, R).tolist()
    b = si.custom(48, q_lens, ctx, num_q_heads=4, num_kv_heads=4, head_dim=64)
    ref, kp, vp = oracle.iteration(b)
    db = DeviceBatch(b)
    out = db.iteration()
    assert np.array_equal(bits_of(db.k_pages), kp) and np.array_equal(bits_of(db.v_pages), vp)
    mx, mean = compare(out, ref)
    print(f"45 requests: max-abs {mx:.3e} mean-abs {mean:.3e}")
    assert mx <= MAX_ABS and mean <= MEAN_ABS
    assert db.eng.device_status() == 0


@pytest.mark.parametrize("hq,hkv,d", [(8, 2, 64), (14, 2, 128), (4, 4, 128)])
def test_decode_units_split_into_many_pieces(oracle, hq, hkv, d, dispatch):
    """Few (request, kv head) units with long contexts: the stream-K cut gives every CTA about one kv tile, so a unit is
    merged from tens of partial pieces by combine_kernel (both its row paths, every column slice of the GQA grid)."""
    b = si.custom(49, [32, 32, 5], [3000, 5003, 2049], num_q_heads=hq, num_kv_heads=hkv, head_dim=d)
    ref, kp, vp = oracle.iteration(b)
    db = DeviceBatch(b)
    out = db.iteration()
    assert np.array_equal(bits_of(db.k_pages), kp) and np.array_equal(bits_of(db.v_pages), vp)
    mx, mean = compare(out, ref)
    print(f"many pieces Hq={hq} Hkv={hkv} D={d}: max-abs {mx:.3e} mean-abs {mean:.3e}")
    assert mx <= MAX_ABS and mean <= MEAN_ABS
    first = bits_of(out).copy()
    db.out.fill_(float("nan"))
    db.attend()
    import torch
    torch.cuda.synchronize()
    assert np.array_equal(bits_of(db.out), first), "split-KV merge is not bitwise reproducible"
    assert db.eng.device_status() == 0
