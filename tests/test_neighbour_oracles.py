"""-m "not gpu": pins of oracle/neighbours.py (RoPE before the KV write; the confidence-threshold sampler)."""
import numpy as np

import sangam_inputs as si
from oracle import neighbours as nb


def _bits(x):
    return si.f32_to_bf16_bits(np.asarray(x, np.float32))


def test_rope_position_zero_is_identity_and_norms_are_preserved():
    g = np.random.default_rng(0)
    x = _bits(g.standard_normal((5, 3, 64)))
    pos = np.array([0, 1, 17, 4095, 8191])
    out = nb.rope_rotate(x, pos)
    xf = si.bf16_bits_to_f64(x)
    assert np.array_equal(out[0], xf[0])                          # angle 0: cos = 1, sin = 0 exactly
    half = 32
    n_in = xf[..., :half] ** 2 + xf[..., half:] ** 2               # every (i, i + D/2) pair is rotated in its plane
    n_out = out[..., :half] ** 2 + out[..., half:] ** 2
    assert np.allclose(n_in, n_out, rtol=1e-12, atol=1e-14)


def test_rope_composes_and_depends_on_relative_position_only():
    g = np.random.default_rng(1)
    D = 32
    q = _bits(g.standard_normal((1, 1, D))); k = _bits(g.standard_normal((1, 1, D)))
    a, b = 37, 1000
    # rotating by a then by b == rotating by a + b: the rotation of an exactly-representable intermediate is not available in
    # bf16, so compose on the fp64 result through the definition of a plane rotation
    ra = nb.rope_rotate(q, [a])[0, 0]; rab = nb.rope_rotate(q, [a + b])[0, 0]
    half = D // 2
    comp = np.empty(D)
    for i in range(half):
        th = 10000.0 ** (-2.0 * i / D) * b
        comp[i] = ra[i] * np.cos(th) - ra[i + half] * np.sin(th)
        comp[i + half] = ra[i + half] * np.cos(th) + ra[i] * np.sin(th)
    assert np.allclose(comp, rab, rtol=1e-11, atol=1e-12)
    # <rope(q, m), rope(k, n)> is a function of m - n
    dots = [float(nb.rope_rotate(q, [m])[0, 0] @ nb.rope_rotate(k, [m - 250])[0, 0]) for m in (250, 251, 1000, 5000)]
    assert np.allclose(dots, dots[0], rtol=1e-10, atol=1e-10)
    # hand value: D = 2, pos = 1, base anything: theta_0 = 1 -> (x0 cos1 - x1 sin1, x1 cos1 + x0 sin1)
    x = _bits([[[1.0, 2.0]]])
    out = nb.rope_rotate(x, [1])[0, 0]
    assert np.allclose(out, [np.cos(1) - 2 * np.sin(1), 2 * np.cos(1) + np.sin(1)], rtol=1e-15)


def test_kv_write_rope_scatter_matches_plain_write_for_v_and_slots():
    import oracle
    b = si.custom(5, [6, 3], [40, 20], num_q_heads=4, num_kv_heads=2, head_dim=64)
    P = b.num_pages
    kpf = np.zeros((P, 2, 16, 64)); vpb = np.full((P, 2, 16, 64), si.POISON, np.uint16)
    pos = np.arange(len(b.slot_cache)) % 50
    nb.kv_write_rope(b.k_cache, b.v_cache, b.slot_cache, pos, 10000.0, kpf, vpb)
    kp2, vp2 = si.empty_pools(b)
    oracle.kv_write(b.k_cache, b.v_cache, b.slot_cache, kp2, vp2)
    assert np.array_equal(vpb, vp2)                               # V: the plain scatter, bit for bit
    rot = nb.rope_rotate(b.k_cache, pos)
    for i, s in enumerate(b.slot_cache):
        assert np.array_equal(kpf[s // 16, :, s % 16, :], rot[i])


def test_sampler_top1_against_numpy_softmax_and_threshold_edge():
    g = np.random.default_rng(2)
    logits = _bits(3.0 * g.standard_normal((12, 50)))
    x = si.bf16_bits_to_f64(logits)
    p = np.exp(x - x.max(1, keepdims=True)); p /= p.sum(1, keepdims=True)
    tok, conf, un = nb.confidence_sample(logits, np.ones(12, int), [0, 12], 0.9)
    assert np.array_equal(tok, p.argmax(1)) and np.allclose(conf, p.max(1), rtol=1e-13)
    # strictly "exceeds": two equal maxima and everything else at -inf-like distance give conf = 0.5 exactly
    row = np.full((1, 8), -200.0); row[0, 2] = row[0, 5] = 4.0
    tok, conf, un = nb.confidence_sample(_bits(row), [1], [0, 1], 0.5)
    assert tok[0] == 2 and conf[0] == 0.5 and un[0] == 1          # 0.5 does not exceed 0.5 -> fallback unmasks the only candidate
    row2 = np.concatenate([row, row]); row2[1, 5] = -200.0         # second row: conf = 1.0
    tok, conf, un = nb.confidence_sample(_bits(row2), [1, 1], [0, 2], 0.5)
    assert list(un) == [0, 1]                                      # row 1 passes, so row 0 (conf 0.5, not > 0.5) stays masked


def test_sampler_fallback_and_masks():
    # request 0: nobody passes -> the most confident MASKED row is unmasked; request 1: committed rows are never touched
    V = 6
    x = np.zeros((5, V), np.float32)
    x[0, 1] = 1.0; x[1, 3] = 2.0; x[2, 0] = 1.5          # request 0 rows 0-2: conf ~ 0.35, 0.60, 0.47
    x[3, 2] = 9.0; x[4, 4] = 9.0                          # request 1 rows 3-4: conf ~ 1
    tok, conf, un = nb.confidence_sample(_bits(x), [1, 0, 1, 0, 1], [0, 3, 5], 0.9)
    assert list(tok) == [1, 3, 0, 2, 4]
    assert list(un) == [0, 0, 1, 0, 1]                    # row 1 is the most confident of request 0 but already committed -> row 2
    tok, conf, un = nb.confidence_sample(_bits(x), [0, 0, 0, 0, 0], [0, 3, 5], 0.9)
    assert un.sum() == 0                                  # nothing masked, nothing to do


def test_kv_gather_scatter_oracle_round_trip_and_brute_force():
    g = np.random.default_rng(4)
    P, Hkv, D = 20, 3, 8
    kp = g.integers(0, 65535, (P, Hkv, 16, D)).astype(np.uint16); vp = g.integers(0, 65535, (P, Hkv, 16, D)).astype(np.uint16)
    src_ids = [7, 2, 19, 0]
    ks, vs = nb.kv_gather(kp, vp, src_ids)
    for i, pg in enumerate(src_ids):                       # element by element
        for h in range(Hkv):
            for o in range(16):
                for d in range(D):
                    assert ks[i, h, o, d] == kp[pg, h, o, d] and vs[i, h, o, d] == vp[pg, h, o, d]
    kd = np.zeros_like(kp); vd = np.zeros_like(vp)
    dst_ids = [1, 5, 3, 11]
    nb.kv_scatter(ks, vs, dst_ids, kd, vd)
    for s, t in zip(src_ids, dst_ids):
        assert np.array_equal(kd[t], kp[s]) and np.array_equal(vd[t], vp[s])
    untouched = [p for p in range(P) if p not in dst_ids]
    assert np.all(kd[untouched] == 0) and np.all(vd[untouched] == 0)
