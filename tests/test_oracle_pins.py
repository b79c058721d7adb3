"""Pins for the fp64 oracle (CPU only).  Each test ties oracle/sangam_oracle.c to something
other than itself: a closed form, an invariant, a library routine on a special case, or brute
force on tiny inputs (SURVEY.md 8(c) pins 1-16; north_star's list).  A dropped term, wrong
sign/index or transposed operand in the oracle fails at least one of them."""
import math
import os

import numpy as np
import pytest

import sangam_inputs as si

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _pools(b, oracle, new=True):
    kp, vp = si.empty_pools(b)
    oracle.kv_write(b.k_cache, b.v_cache, b.slot_cache, kp, vp)
    if new:
        oracle.kv_write(b.k_new, b.v_new, b.slot_new, kp, vp)
    return kp, vp


def _gather(b, pool, r):
    """Context rows of request r read back through the block table: float64 [c][Hkv][D]."""
    c = int(b.ctx_lens[r])
    j = np.arange(c)
    pg = b.block_table[r, j // 16]
    return si.bf16_bits_to_f64(pool[pg, :, j % 16, :])


def _dense(b, kp, vp):
    """numpy float64 softmax(scale QK^T)V per (request, head): the textbook routine."""
    G = b.num_q_heads // b.num_kv_heads
    q = si.bf16_bits_to_f64(b.q)
    out = np.zeros(q.shape)
    for r in range(b.batch):
        K, V = _gather(b, kp, r), _gather(b, vp, r)
        lo, hi = int(b.cu_q_lens[r]), int(b.cu_q_lens[r + 1])
        for h in range(b.num_q_heads):
            S = float(b.scale) * (q[lo:hi, h, :] @ K[:, h // G, :].T)
            S -= S.max(axis=1, keepdims=True)
            Pm = np.exp(S)
            Pm /= Pm.sum(axis=1, keepdims=True)
            out[lo:hi, h, :] = Pm @ V[:, h // G, :]
    return out


# -- pin 1: dense library routine on tiny inputs, odd lengths ------------------------------------
@pytest.mark.parametrize("q_lens,ctx_lens,hq,hkv,d", [
    ([16, 16], [128, 128], 4, 4, 64),
    ([1, 3, 5, 2, 7], [1, 15, 16, 17, 33], 4, 2, 8),
    ([4], [40], 14, 2, 16),
])
def test_pin01_dense_numpy(oracle, q_lens, ctx_lens, hq, hkv, d):
    b = si.custom(11, q_lens, ctx_lens, num_q_heads=hq, num_kv_heads=hkv, head_dim=d)
    kp, vp = _pools(b, oracle)
    got = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    assert np.max(np.abs(got - _dense(b, kp, vp))) <= 1e-12


def test_pin01_config1_dense(oracle):
    b = si.config1()
    out, kp, vp = oracle.iteration(b)
    assert np.max(np.abs(out - _dense(b, kp, vp))) <= 1e-12


# -- pin 2: paged == contiguous (two independent addressings) ---------------------------------
def test_pin02_paged_equals_contiguous(oracle):
    b = si.custom(5, [3, 9, 1], [37, 16, 50], num_q_heads=6, num_kv_heads=3, head_dim=16)
    kp, vp = _pools(b, oracle, new=False)
    paged = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    cont = oracle.attn_contiguous(b.q, b.k_cache, b.v_cache, b.cu_ctx, b.cu_q_lens, b.scale)
    assert np.max(np.abs(paged - cont)) <= 1e-13


# -- pin 3: physical page permutation + remapped block table -> bit-identical ------------------
def test_pin03_page_permutation(oracle):
    b = si.custom(6, [5, 4], [45, 70], num_q_heads=4, num_kv_heads=4, head_dim=16)
    kp, vp = _pools(b, oracle)
    ref = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    g = np.random.default_rng(0)
    perm = g.permutation(b.num_pages)            # new_page = perm[old_page]
    kp2, vp2 = np.empty_like(kp), np.empty_like(vp)
    kp2[perm], vp2[perm] = kp, vp
    bt2 = np.where(b.block_table >= 0, perm[np.maximum(b.block_table, 0)], -1).astype(np.int32)
    got = oracle.block_attn(b.q, kp2, vp2, bt2, b.cu_q_lens, b.ctx_lens, b.scale)
    assert np.array_equal(ref, got)


# -- pin 4: softmax rows sum to 1 ---------------------------------------------------------------
def test_pin04_rows_sum_to_one(oracle):
    b = si.custom(7, [4, 4], [100, 33], num_q_heads=4, num_kv_heads=2, head_dim=32)
    kp, vp = _pools(b, oracle)
    _, lse, rs = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale, want_aux=True)
    assert np.max(np.abs(rs - 1.0)) <= 1e-12
    assert np.all(np.isfinite(lse))


# -- pin 5 / 7: identical keys, scale = 0, q = 0  -> mean of V ---------------------------------
def test_pin05_identical_keys_mean_of_v(oracle):
    b = si.custom(8, [3], [29], num_q_heads=4, num_kv_heads=2, head_dim=16)
    b.k_cache[:] = b.k_cache[0:1]
    kp, vp = _pools(b, oracle, new=False)
    got = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    mean_v = _gather(b, vp, 0).mean(axis=0)                   # [Hkv][D]
    for h in range(4):
        assert np.max(np.abs(got[:, h, :] - mean_v[h // 2])) <= 1e-13


def test_pin07_scale_zero_and_q_zero(oracle):
    b = si.custom(9, [2, 2], [20, 31], num_q_heads=2, num_kv_heads=2, head_dim=16)
    kp, vp = _pools(b, oracle)
    a = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, np.float32(0.0))
    z = oracle.block_attn(np.zeros_like(b.q), kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    for r in range(2):
        mv = _gather(b, vp, r).mean(axis=0)
        lo, hi = b.cu_q_lens[r], b.cu_q_lens[r + 1]
        assert np.max(np.abs(a[lo:hi] - mv[None])) <= 1e-13
        assert np.max(np.abs(z[lo:hi] - mv[None])) <= 1e-13


# -- pin 8: c = 1 -> out = v_0 exactly ----------------------------------------------------------
def test_pin08_single_key(oracle):
    b = si.custom(10, [4], [1], num_q_heads=4, num_kv_heads=2, head_dim=16)
    kp, vp = _pools(b, oracle, new=False)
    got = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    v0 = si.bf16_bits_to_f64(b.v_cache[0])
    for h in range(4):
        assert np.array_equal(got[:, h, :], np.broadcast_to(v0[h // 2], (4, 16)))


# -- pin 9: needle -> that V row; also catches a K/V index mismatch ----------------------------
@pytest.mark.parametrize("pos", [0, 15, 16, 31, 40])
def test_pin09_needle(oracle, pos):
    b = si.custom(12, [1], [41], num_q_heads=1, num_kv_heads=1, head_dim=64)
    q = si.bf16_bits_to_f64(b.q)[0, 0]
    b.k_cache[:] = 0
    b.k_cache[pos, 0] = si.f32_to_bf16_bits((q * 64.0).astype(np.float32))   # logit ~ 8*|q|^2*... dominant
    kp, vp = _pools(b, oracle, new=False)
    got = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    assert np.max(np.abs(got[0, 0] - si.bf16_bits_to_f64(b.v_cache[pos, 0]))) <= 1e-9


# -- two keys: weights are the logistic function of the logit gap (closed form, tanh) ----------
def test_two_key_logistic_closed_form(oracle):
    b = si.custom(13, [1], [2], num_q_heads=1, num_kv_heads=1, head_dim=16)
    qv = np.zeros(16, np.float32); qv[3] = 2.0
    k0 = np.zeros(16, np.float32); k0[3] = 1.5
    k1 = np.zeros(16, np.float32); k1[3] = -0.5
    v0 = np.zeros(16, np.float32); v0[0] = 1.0
    v1 = np.zeros(16, np.float32); v1[0] = -1.0; v1[1] = 4.0
    b.q[0, 0] = si.f32_to_bf16_bits(qv)
    b.k_cache[0, 0], b.k_cache[1, 0] = si.f32_to_bf16_bits(k0), si.f32_to_bf16_bits(k1)
    b.v_cache[0, 0], b.v_cache[1, 0] = si.f32_to_bf16_bits(v0), si.f32_to_bf16_bits(v1)
    kp, vp = _pools(b, oracle, new=False)
    got = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, np.float32(0.25))
    gap = 0.25 * (2.0 * 1.5 - 2.0 * -0.5)                 # s0 - s1 = 1.0
    w0 = 0.5 * (1.0 + math.tanh(gap / 2.0))               # sigmoid(gap)
    assert abs(got[0, 0, 0] - (w0 - (1 - w0))) <= 1e-14
    assert abs(got[0, 0, 1] - 4.0 * (1 - w0)) <= 1e-14
    assert np.all(got[0, 0, 2:] == 0.0)


def test_golden_uniform_ramp(oracle):
    """tests/golden/uniform_ramp.txt: with scale 0 every weight is 1/c, so for v_j[d] = j the output
    is (c-1)/2 and for v_j[d] = j^2 it is (c-1)(2c-1)/6 (sums of integers; hand-derived)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "uniform_ramp.txt")) if l.strip() and not l.startswith("#")]
    for c_s, lin_s, sq_s in rows:
        c = int(c_s)
        b = si.custom(14, [1], [c], num_q_heads=1, num_kv_heads=1, head_dim=16)
        v = np.zeros((c, 16), np.float32)
        v[:, 0] = np.arange(c)
        v[:, 1] = np.arange(c) ** 2
        b.v_cache[:, 0] = si.f32_to_bf16_bits(v)     # integers <= 256 are exact in bf16
        kp, vp = _pools(b, oracle, new=False)
        got = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, np.float32(0.0))
        assert abs(got[0, 0, 0] - float(lin_s)) <= 1e-12
        assert abs(got[0, 0, 1] - float(sq_s)) <= 1e-10


# -- pin 6: joint permutation of context positions ---------------------------------------------
def test_pin06_joint_context_permutation(oracle):
    b = si.custom(15, [6], [53], num_q_heads=4, num_kv_heads=2, head_dim=16)
    kp, vp = _pools(b, oracle, new=False)
    ref = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    perm = np.random.default_rng(1).permutation(53)
    b.k_cache, b.v_cache = b.k_cache[perm].copy(), b.v_cache[perm].copy()
    kp2, vp2 = _pools(b, oracle, new=False)
    got = oracle.block_attn(b.q, kp2, vp2, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    assert np.max(np.abs(ref - got)) <= 1e-12


# -- pin 10: adding one vector to every key leaves the output unchanged ------------------------
def test_pin10_key_shift_invariance(oracle):
    b = si.custom(16, [5], [30], num_q_heads=2, num_kv_heads=2, head_dim=16)
    # small-integer keys so k + u stays exactly representable in bf16
    g = np.random.default_rng(2)
    k = g.integers(-3, 4, size=b.k_cache.shape).astype(np.float32)
    b.k_cache = si.f32_to_bf16_bits(k)
    kp, vp = _pools(b, oracle, new=False)
    ref = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    u = g.integers(-2, 3, size=(1, b.num_kv_heads, 16)).astype(np.float32)
    b.k_cache = si.f32_to_bf16_bits(k + u)
    kp2, vp2 = _pools(b, oracle, new=False)
    got = oracle.block_attn(b.q, kp2, vp2, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    assert np.max(np.abs(ref - got)) <= 1e-12


# -- pin 11: convex combination bounds ------------------------------------------------------------
def test_pin11_convex_hull(oracle):
    b = si.custom(17, [8, 3], [64, 19], num_q_heads=4, num_kv_heads=1, head_dim=16)
    kp, vp = _pools(b, oracle)
    got = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    for r in range(2):
        V = _gather(b, vp, r)[:, 0, :]
        lo, hi = b.cu_q_lens[r], b.cu_q_lens[r + 1]
        assert np.all(got[lo:hi] <= V.max(axis=0) + 1e-12) and np.all(got[lo:hi] >= V.min(axis=0) - 1e-12)


# -- pin 12: split-KV merge formula ---------------------------------------------------------------
def test_pin12_split_merge(oracle):
    c, cut = 77, 32          # cut on a page boundary so each half is its own page list
    b = si.custom(18, [3], [c], num_q_heads=2, num_kv_heads=1, head_dim=16)
    kp, vp = _pools(b, oracle, new=False)
    whole = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    oa, la, _ = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, np.array([cut], np.int32), b.scale, want_aux=True)
    bt2 = np.full_like(b.block_table, -1)
    bt2[0, :b.block_table.shape[1] - cut // 16] = b.block_table[0, cut // 16:]
    ob, lb, _ = oracle.block_attn(b.q, kp, vp, bt2, b.cu_q_lens, np.array([c - cut], np.int32), b.scale, want_aux=True)
    for t in range(3):
        for h in range(2):
            # partial i: normalised out_i is the unnormalised sum relative to m_i = lse_i with l_i = 1
            merged = oracle.combine(np.stack([oa[t, h], ob[t, h]]), [la[t, h], lb[t, h]], [1.0, 1.0])
            assert np.max(np.abs(merged - whole[t, h])) <= 1e-12
    # and with genuinely unnormalised partials: O_i = out_i * l_i, m_i = lse_i - log l_i
    l_i = np.array([3.5, 0.25])
    merged = oracle.combine(np.stack([oa[0, 0] * l_i[0], ob[0, 0] * l_i[1]]),
                            [la[0, 0] - math.log(l_i[0]), lb[0, 0] - math.log(l_i[1])], l_i)
    assert np.max(np.abs(merged - whole[0, 0])) <= 1e-12


# -- pin 13: GQA == MHA with repeated kv heads -------------------------------------------------
def test_pin13_gqa_equals_repeated_mha(oracle):
    b = si.custom(19, [4, 2], [35, 18], num_q_heads=6, num_kv_heads=2, head_dim=16)
    kp, vp = _pools(b, oracle, new=False)
    gqa = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    kp6, vp6 = np.repeat(kp, 3, axis=1), np.repeat(vp, 3, axis=1)
    mha = oracle.block_attn(b.q, np.ascontiguousarray(kp6), np.ascontiguousarray(vp6), b.block_table,
                            b.cu_q_lens, b.ctx_lens, b.scale)
    assert np.array_equal(gqa, mha)


# -- pin 14: batch / row independence ---------------------------------------------------------
def test_pin14_batch_and_row_independence(oracle):
    b = si.custom(20, [7, 5, 0, 2], [40, 23, 9, 64], num_q_heads=4, num_kv_heads=2, head_dim=16)
    kp, vp = _pools(b, oracle)
    full = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    for r in range(4):
        lo, hi = int(b.cu_q_lens[r]), int(b.cu_q_lens[r + 1])
        alone = oracle.block_attn(b.q[lo:hi], kp, vp, b.block_table[r:r + 1], np.array([0, hi - lo], np.int32),
                                  b.ctx_lens[r:r + 1], b.scale)
        assert np.array_equal(alone, full[lo:hi])
    # a "decode" whose q rows are rows 2..4 of request 0's "prefill" reproduces those output rows
    dec = oracle.block_attn(b.q[2:5], kp, vp, b.block_table[0:1], np.array([0, 3], np.int32), b.ctx_lens[0:1], b.scale)
    assert np.array_equal(dec, full[2:5])
    # row selection returns the same rows
    sel = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale, rows=[13, 0, 8])
    assert np.array_equal(sel, full[[13, 0, 8]])


# -- pin 15: linear in V -----------------------------------------------------------------------
def test_pin15_linear_in_v(oracle):
    b = si.custom(21, [3], [26], num_q_heads=2, num_kv_heads=2, head_dim=16)
    g = np.random.default_rng(3)
    v1 = g.integers(-4, 5, size=b.v_cache.shape).astype(np.float32)
    v2 = g.integers(-4, 5, size=b.v_cache.shape).astype(np.float32)
    outs = []
    for v in (v1, v2, 2.0 * v1 + v2):
        b.v_cache = si.f32_to_bf16_bits(v)
        kp, vp = _pools(b, oracle, new=False)
        outs.append(oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale))
    assert np.max(np.abs(outs[2] - (2.0 * outs[0] + outs[1]))) <= 1e-12


# -- zero lengths (reading S13) -----------------------------------------------------------------
def test_zero_context_gives_zero_rows(oracle):
    b = si.custom(22, [2, 3], [0, 5], num_q_heads=2, num_kv_heads=1, head_dim=16)
    kp, vp = _pools(b, oracle, new=False)
    out, lse, _ = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale, want_aux=True)
    assert np.all(out[:2] == 0.0) and np.all(np.isneginf(lse[:2])) and np.all(np.isfinite(out[2:]))


# -- poison independence (reading S12) -----------------------------------------------------------
def test_output_ignores_poisoned_tails_and_unowned_pages(oracle):
    b = si.custom(23, [3, 2], [21, 34], num_q_heads=2, num_kv_heads=2, head_dim=16)
    kp, vp = _pools(b, oracle)
    a = oracle.block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale)
    kz, vz = si.empty_pools(b, poison=False)
    oracle.kv_write(b.k_cache, b.v_cache, b.slot_cache, kz, vz)
    oracle.kv_write(b.k_new, b.v_new, b.slot_new, kz, vz)
    bt = b.block_table.copy()
    bt[bt < 0] = 2 ** 30                                    # over-range ids past ceil(c/16) are never read
    z = oracle.block_attn(b.q, kz, vz, bt, b.cu_q_lens, b.ctx_lens, b.scale)
    assert np.all(np.isfinite(a)) and np.array_equal(a, z)


# -- pin 16: kv_write ---------------------------------------------------------------------------
def test_pin16_kv_write_bruteforce_roundtrip(oracle):
    b = si.custom(24, [5, 9], [37, 50], num_q_heads=4, num_kv_heads=3, head_dim=8)
    kp, vp = si.empty_pools(b)
    sentinel_k, sentinel_v = kp.copy(), vp.copy()
    slots = b.slot_cache.copy()
    slots[[3, 40]] = -1                                     # negative slots skipped
    oracle.kv_write(b.k_cache, b.v_cache, slots, kp, vp)
    ek, ev = sentinel_k.copy(), sentinel_v.copy()
    for i, s in enumerate(slots):                           # per-element python loop
        if s < 0:
            continue
        for h in range(3):
            for d in range(8):
                ek[s // 16, h, s % 16, d] = b.k_cache[i, h, d]
                ev[s // 16, h, s % 16, d] = b.v_cache[i, h, d]
    assert np.array_equal(kp, ek) and np.array_equal(vp, ev)
    touched = np.zeros(kp.shape[0] * 16, bool)
    touched[slots[slots >= 0]] = True
    untouched = ~touched.reshape(-1, 16)
    assert np.all(kp.transpose(0, 2, 1, 3)[untouched] == si.POISON)
    # round trip through the block table (ties slot = page*16+off to block_table[r][j/16])
    oracle.kv_write(b.k_cache, b.v_cache, b.slot_cache, kp, vp)
    cu = b.cu_ctx
    for r in range(2):
        c = int(b.ctx_lens[r]); j = np.arange(c)
        back = kp[b.block_table[r, j // 16], :, j % 16, :]
        assert np.array_equal(back, b.k_cache[cu[r]:cu[r + 1]])
