"""-m gpu parity of the two kernels next to the hot path against oracle/neighbours.py, through the C ABI.

RoPE-fused KV write: V pages bit-exact; K pages within 1 bf16 ulp (+ the fp32 rounding of the two products where they
cancel) of the fp64 rotation on every element and identical to its
bf16 rounding on all but a sliver (fp32 arithmetic on an fp32 cos/sin table vs fp64: the results differ by ~1e-7 relative, so
only values that sit on a rounding boundary may round the other way).  Sampler: argmax bit-exact, confidence to 1e-5,
unmask decisions identical wherever the confidence is not within 1e-4 of the threshold (both sides decide in their own
precision: fp32 on the GPU, the kernel's; fp64 in the oracle), fallback row identical."""
import numpy as np
import pytest

import sangam_inputs as si
from gpu_harness import DeviceBatch, bits_of, t_bf16, t_i32
from oracle import neighbours as nb

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("hq,hkv,d", [(8, 8, 128), (28, 4, 128), (4, 4, 64)])
def test_kv_write_rope_matches_the_fp64_rotation(hq, hkv, d):
    import torch
    import paper_2607_04206_b200 as sg
    b = si.custom(81, [40, 7, 300], [700, 90, 300], num_q_heads=hq, num_kv_heads=hkv, head_dim=d)
    db = DeviceBatch(b)
    max_pos = 8192
    table = torch.from_numpy(sg.rope_table(max_pos, d)).cuda()
    g = np.random.default_rng(3)
    pos = g.integers(0, max_pos, len(b.slot_cache)).astype(np.int32)
    pos[:4] = [0, 1, max_pos - 1, 4096]
    slots = b.slot_cache.copy(); slots[[5, 50]] = -1                           # skipped rows stay poisoned
    db.eng.kv_write_rope(db.k_cache, db.v_cache, t_i32(slots), t_i32(pos), table, db.k_pages, db.v_pages)
    torch.cuda.synchronize()
    assert db.eng.device_status() == 0
    P = b.num_pages
    kpf = np.full((P, hkv, 16, d), np.nan); vpb = np.full((P, hkv, 16, d), si.POISON, np.uint16)
    nb.kv_write_rope(b.k_cache, b.v_cache, slots, pos, 10000.0, kpf, vpb)
    assert np.array_equal(bits_of(db.v_pages), vpb), "V pages differ (bit-exact copy required)"
    got_bits = bits_of(db.k_pages)
    written = ~np.isnan(kpf)
    assert np.all(got_bits[~written] == si.POISON), "a slot that was not written changed"
    got = si.bf16_bits_to_f64(got_bits[written]); ref = kpf[written]
    ulp = 2.0 ** (np.floor(np.log2(np.maximum(np.abs(ref), 2.0 ** -126))) - 7)    # one bf16 ulp in the value's binade
    # plus the fp32 rounding of the two products, which matters only where they cancel (|result| << |inputs| ~ 5)
    assert np.all(np.abs(got - ref) <= ulp + 5.0 * 2.0 ** -22), "rotated K is more than 1 bf16 ulp from the fp64 rotation"
    same = got_bits[written] == si.f32_to_bf16_bits(ref.astype(np.float32))
    print(f"rope {hq}/{hkv}/{d}: {written.sum()} elements, {100 * (1 - same.mean()):.4f} % round the other way")
    assert same.mean() > 0.995
    # position 0 rows are copied bit for bit (cos = 1, sin = 0 exactly)
    s0 = int(b.slot_cache[0])
    assert np.array_equal(got_bits[s0 // 16, :, s0 % 16, :], b.k_cache[0])
    # a position outside the table: row skipped, flag raised
    bad = pos.copy(); bad[9] = max_pos
    before = bits_of(db.k_pages).copy()
    db.eng.kv_write_rope(db.k_cache, db.v_cache, t_i32(slots), t_i32(bad), table, db.k_pages, db.v_pages)
    torch.cuda.synchronize()
    assert db.eng.device_status() == 32
    after = bits_of(db.k_pages)
    s9 = int(slots[9])
    assert np.array_equal(after[s9 // 16, :, s9 % 16, :], before[s9 // 16, :, s9 % 16, :])


@pytest.mark.parametrize("vocab,rows_per_req", [(126464, [32, 32, 32, 5]), (151936, [32] * 16), (1000, [3, 1, 32]), (50, [7])])
def test_confidence_sampler_matches_the_oracle(vocab, rows_per_req):
    """Vocabulary sizes of LLaDA-8B (126 464) and Dream-7B (151 936) and small ones with ragged slices."""
    import torch
    import paper_2607_04206_b200 as sg
    g = np.random.default_rng(vocab)
    rows = int(sum(rows_per_req))
    x = 2.0 * g.standard_normal((rows, vocab), dtype=np.float32)
    peak = g.integers(0, vocab, rows)
    boost = g.choice([0.0, 6.0, 12.0, 20.0], rows)                              # from flat to very confident rows
    x[np.arange(rows), peak] += boost
    x[0, vocab - 1] = x[0].max() + 3.0                                          # a maximum at the very last index
    if rows > 2:
        x[2] = np.float32(-1.5)                                                 # all equal: argmax = 0, conf = 1 / V
    logits = si.f32_to_bf16_bits(x)
    masked = (g.random(rows) < 0.7).astype(np.int32)
    cu = np.concatenate([[0], np.cumsum(rows_per_req)]).astype(np.int32)
    thr = 0.9
    tok_ref, conf_ref, un_ref = nb.confidence_sample(logits, masked, cu, thr)
    eng = sg.Sangam(num_q_heads=4, num_kv_heads=4, head_dim=64, num_pages=8, max_batch=len(rows_per_req), max_total_q=max(rows, 1), max_pages_per_req=4)
    d_tok = torch.full((rows,), -1, dtype=torch.int32, device="cuda"); d_conf = torch.zeros(rows, dtype=torch.float32, device="cuda")
    d_un = torch.full((rows,), -1, dtype=torch.int32, device="cuda")
    eng.confidence_sample(t_bf16(logits), t_i32(masked), t_i32(cu), thr, d_tok, d_conf, d_un)
    torch.cuda.synchronize()
    tok, conf, un = d_tok.cpu().numpy(), d_conf.cpu().numpy().astype(np.float64), d_un.cpu().numpy()
    assert np.array_equal(tok, tok_ref), "argmax differs"
    assert np.allclose(conf, conf_ref, rtol=2e-5, atol=1e-9)
    clear = np.abs(conf_ref - thr) > 1e-4
    for r in range(len(rows_per_req)):
        lo, hi = cu[r], cu[r + 1]
        if np.all(clear[lo:hi]):
            assert np.array_equal(un[lo:hi], un_ref[lo:hi]), f"request {r}"
    assert np.all(un[masked == 0] == 0)
    print(f"sampler V={vocab}: {rows} rows, {int(un.sum())} unmasked, conf max rel err {np.max(np.abs(conf - conf_ref) / conf_ref):.2e}")


def test_sampler_fallback_and_exact_threshold_on_the_gpu():
    import torch
    import paper_2607_04206_b200 as sg
    V = 64
    x = np.full((4, V), -200.0, np.float32)
    x[0, 2] = x[0, 5] = 4.0                    # conf = 0.5 exactly (two equal maxima): 0.5 does not exceed 0.5
    x[1, 7] = 4.0                              # conf = 1
    x[2, 1] = x[2, 3] = x[2, 9] = x[2, 11] = 1.0   # conf = 0.25
    x[3, 0] = x[3, 1] = 2.0                    # conf = 0.5
    logits = si.f32_to_bf16_bits(x)
    eng = sg.Sangam(num_q_heads=4, num_kv_heads=4, head_dim=64, num_pages=8, max_batch=2, max_total_q=4, max_pages_per_req=4)
    for masked, cu, thr in (([1, 1, 1, 1], [0, 2, 4], 0.5), ([1, 0, 1, 1], [0, 2, 4], 0.5), ([1, 1, 1, 1], [0, 4], 0.999)):
        ref = nb.confidence_sample(logits, masked, cu, thr)
        d_tok = torch.zeros(4, dtype=torch.int32, device="cuda"); d_conf = torch.zeros(4, dtype=torch.float32, device="cuda")
        d_un = torch.zeros(4, dtype=torch.int32, device="cuda")
        eng.confidence_sample(t_bf16(logits), t_i32(np.array(masked)), t_i32(np.array(cu)), thr, d_tok, d_conf, d_un)
        torch.cuda.synchronize()
        assert np.array_equal(d_tok.cpu().numpy(), ref[0]) and np.array_equal(d_un.cpu().numpy(), ref[2])
        assert np.array_equal(d_conf.cpu().numpy().astype(np.float64), ref[1])          # these confidences are exact in fp32


def test_kv_page_gather_scatter_bit_exact():
    """The single-GPU halves of the KV transfer: gather a request's pages, scatter them into another pool under
    different page ids; the receiver then attends over them and gets the sender's result bit for bit."""
    import torch
    b = si.custom(82, [32, 20], [1000, 333], num_q_heads=8, num_kv_heads=4, head_dim=128)
    src = DeviceBatch(b)
    out_src = bits_of(src.iteration()).copy()
    dst = DeviceBatch(b)                                   # same geometry, empty (poisoned) pools
    g = np.random.default_rng(6)
    new_bt = np.full_like(b.block_table, -1)
    free = g.permutation(b.num_pages)
    used = 0
    for r in range(b.batch):
        n = (int(b.ctx_lens[r]) + 15) // 16
        ids_src = b.block_table[r, :n]
        ids_dst = free[used:used + n].astype(np.int32); used += n
        new_bt[r, :n] = ids_dst
        shape = (n, b.num_kv_heads, 16, b.head_dim)
        ks = torch.zeros(shape, dtype=torch.bfloat16, device="cuda"); vs = torch.zeros_like(ks)
        src.eng.kv_gather(src.k_pages, src.v_pages, t_i32(ids_src), ks, vs)
        kr, vr = nb.kv_gather(bits_of(src.k_pages), bits_of(src.v_pages), ids_src)
        torch.cuda.synchronize()
        assert np.array_equal(bits_of(ks), kr) and np.array_equal(bits_of(vs), vr)
        dst.eng.kv_scatter(ks, vs, t_i32(ids_dst), dst.k_pages, dst.v_pages)
    torch.cuda.synchronize()
    kd = np.full((b.num_pages, b.num_kv_heads, 16, b.head_dim), si.POISON, np.uint16); vd = kd.copy()
    for r in range(b.batch):
        n = (int(b.ctx_lens[r]) + 15) // 16
        nb.kv_scatter(*nb.kv_gather(bits_of(src.k_pages), bits_of(src.v_pages), b.block_table[r, :n]), new_bt[r, :n], kd, vd)
    assert np.array_equal(bits_of(dst.k_pages), kd) and np.array_equal(bits_of(dst.v_pages), vd)
    dst.block_table = t_i32(new_bt)
    dst.attend()
    torch.cuda.synchronize()
    assert np.array_equal(bits_of(dst.out), out_src), "attention over the transferred pages differs from the sender's"
    # a bad page id is skipped and flagged
    ids = t_i32(np.array([0, b.num_pages, 1], np.int32))
    ks = torch.zeros((3, b.num_kv_heads, 16, b.head_dim), dtype=torch.bfloat16, device="cuda"); vs = torch.zeros_like(ks)
    src.eng.kv_gather(src.k_pages, src.v_pages, ids, ks, vs)
    assert src.eng.device_status() == 2
    assert np.all(bits_of(ks)[1] == 0)
