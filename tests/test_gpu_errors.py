"""-m gpu tests of the error contract of include/sangam.h: device-side conditions raise a sticky flag, never fault, and
are handled identically by every kernel (two-stream, decode, CUDA-core); host-side argument errors return a negative
status without launching anything."""
import ctypes

import numpy as np
import pytest

import sangam_inputs as si
from gpu_harness import MAX_ABS, MEAN_ABS, DeviceBatch, bits_of, compare, t_i32

pytestmark = pytest.mark.gpu

BAD_SLOT, BAD_PAGE, CTX_TOO_LONG = 1, 2, 4


KERNEL = {"prefill_kernel": 1, "decode_kernel": 2, "gqa_pair_kernel": 3}      # sangam_set_dispatch modes


def _batch():
    # request 1 is the victim; requests 0 and 2 must be unaffected.  Decode-sized rows so that both kernels are natural.
    return si.custom(61, [32, 32, 20], [200, 333, 97], num_q_heads=8, num_kv_heads=4, head_dim=128)


@pytest.mark.parametrize("bad_id", ["past_the_pool", "negative", "huge"])
@pytest.mark.parametrize("path", ["prefill_kernel", "decode_kernel", "gqa_pair_kernel", "simt"])
def test_bad_page_id_reads_as_zeros_and_raises_the_flag(oracle, path, bad_id):
    """A page id outside [0, num_pages) inside ceil(c/16): SANGAM_DEV_BAD_PAGE, that page's positions read as K = V = 0,
    other requests untouched (sangam.h).  The expectation comes from the oracle run on an equivalent well-formed batch:
    the bad entry redirected to a spare page whose K and V are zeros."""
    b = _batch()
    victim_entry = 5                                     # positions 80..95 of request 1
    bad = {"past_the_pool": b.num_pages, "negative": -7, "huge": 2 ** 30}[bad_id]
    db = DeviceBatch(b)
    if path != "simt":
        db.eng.set_dispatch(KERNEL[path])
    db.load_cache(); db.write_new()
    bt = b.block_table.copy()
    bt[1, victim_entry] = bad
    db.block_table = t_i32(bt)
    db.attend(simt=(path == "simt"))
    import torch
    torch.cuda.synchronize()
    assert db.eng.device_status() & BAD_PAGE
    db.eng.clear_device_status()
    # oracle on the equivalent batch: entry -> a page nobody owns, zero-filled
    kp, vp = si.empty_pools(b)
    oracle.kv_write(b.k_cache, b.v_cache, b.slot_cache, kp, vp)
    oracle.kv_write(b.k_new, b.v_new, b.slot_new, kp, vp)
    owned = set(b.block_table[b.block_table >= 0].tolist())
    spare = next(pg for pg in range(b.num_pages) if pg not in owned)
    kp[spare] = 0; vp[spare] = 0
    bt_ref = b.block_table.copy(); bt_ref[1, victim_entry] = spare
    ref = oracle.block_attn(b.q, kp, vp, bt_ref, b.cu_q_lens, b.ctx_lens, b.scale)
    mx, mean = compare(db.out, ref)
    print(f"bad page ({bad_id}) via {path}: max-abs {mx:.3e} mean-abs {mean:.3e}")
    assert mx <= MAX_ABS and mean <= MEAN_ABS
    # the neighbours are bit-identical to a clean run
    clean = DeviceBatch(b)
    if path != "simt":
        clean.eng.set_dispatch(KERNEL[path])
    c = bits_of(clean.iteration(simt=(path == "simt")))
    got = bits_of(db.out)
    lo, hi = b.cu_q_lens[1], b.cu_q_lens[2]
    assert np.array_equal(got[:lo], c[:lo]) and np.array_equal(got[hi:], c[hi:])
    assert not np.array_equal(got[lo:hi], c[lo:hi])


@pytest.mark.parametrize("path", ["prefill_kernel", "decode_kernel", "gqa_pair_kernel", "simt"])
def test_context_longer_than_the_block_table_gives_zero_rows(oracle, path):
    """ctx_len needing more than max_pages_per_req pages: SANGAM_DEV_CTX_TOO_LONG, that request's rows are zeros, the
    others match the oracle; negative ctx_len is read as 0 (zero rows, no flag)."""
    import torch
    b = _batch()
    ref, _, _ = oracle.iteration(b)
    for new_len, flag in ((b.max_pages_per_req * 16 + 1, CTX_TOO_LONG), (-5, 0)):
        db = DeviceBatch(b)
        if path != "simt":
            db.eng.set_dispatch(KERNEL[path])
        db.load_cache(); db.write_new()
        cl = b.ctx_lens.copy(); cl[1] = new_len
        db.ctx_lens = t_i32(cl)
        db.attend(simt=(path == "simt"))
        torch.cuda.synchronize()
        st = db.eng.device_status()
        assert (st & CTX_TOO_LONG) == flag and (st & ~CTX_TOO_LONG) == 0
        got = bits_of(db.out)
        lo, hi = b.cu_q_lens[1], b.cu_q_lens[2]
        assert np.all(got[lo:hi] == 0)
        keep = np.r_[0:lo, hi:b.total_q]
        mx, mean = compare(db.out[torch.from_numpy(keep).cuda()], ref[keep])
        assert mx <= MAX_ABS and mean <= MEAN_ABS


@pytest.mark.parametrize("path", ["prefill_kernel", "decode_kernel", "gqa_pair_kernel"])
def test_decreasing_cu_q_lens_is_an_empty_request(oracle, path):
    """cu_q_lens[r+1] < cu_q_lens[r] is read as q_r = 0: nothing is written for that request, nothing faults."""
    import torch
    b = _batch()
    db = DeviceBatch(b)
    db.eng.set_dispatch(KERNEL[path])
    db.load_cache(); db.write_new()
    cu = b.cu_q_lens.copy(); cu[3] = cu[2] - 3              # the last request "ends before it starts"
    db.cu_q_lens = t_i32(cu)
    db.out.fill_(float("nan"))
    db.attend()
    torch.cuda.synchronize()
    assert db.eng.device_status() == 0
    got = si.bf16_bits_to_f64(bits_of(db.out))
    assert np.all(np.isfinite(got[:b.cu_q_lens[2]]))        # requests 0 and 1 are computed
    assert np.all(np.isnan(got[b.cu_q_lens[2]:]))           # the malformed request's rows stay untouched


def test_out_of_range_slot_is_skipped_and_flagged(oracle):
    import torch
    b = _batch()
    db = DeviceBatch(b)
    kp, vp = si.empty_pools(b)
    slots = b.slot_cache.copy()
    slots[7] = b.num_pages * 16            # first slot past the pool
    slots[9] = 2 ** 31 - 1
    good = slots.copy(); good[[7, 9]] = -1
    oracle.kv_write(b.k_cache, b.v_cache, good, kp, vp)
    db.slot_cache = t_i32(slots)
    db.load_cache()
    torch.cuda.synchronize()
    assert db.eng.device_status() == BAD_SLOT
    assert np.array_equal(bits_of(db.k_pages), kp) and np.array_equal(bits_of(db.v_pages), vp)


def test_host_argument_errors():
    """Null / misaligned pointers and counts above the ctx maxima return a negative status and a message, launch nothing
    and leave the ctx usable (sangam.h: SANGAM_ERR_INVALID_ARG -1, SANGAM_ERR_WORKSPACE -3)."""
    import torch
    import paper_2607_04206_b200 as sg
    b = _batch()
    db = DeviceBatch(b)
    lib, ctx = db.eng.lib, db.eng.ctx
    stream = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    P = lambda t: ctypes.c_void_p(t.data_ptr())
    n0 = db.eng.launch_count()
    args = lambda **kw: [ctx, kw.get("q", P(db.q)), kw.get("kp", P(db.k_pages)), kw.get("vp", P(db.v_pages)),
                         kw.get("bt", P(db.block_table)), kw.get("cu", P(db.cu_q_lens)), kw.get("cl", P(db.ctx_lens)),
                         kw.get("batch", b.batch), kw.get("total_q", b.total_q), ctypes.c_float(float(b.scale)),
                         kw.get("out", P(db.out)), stream]
    for fn in (lib.sangam_block_attn, lib.sangam_block_attn_simt):
        assert fn(*args(q=ctypes.c_void_p(0))) == -1 and b"null" in lib.sangam_last_error(ctx)
        assert fn(*args(out=ctypes.c_void_p(0))) == -1
        assert fn(*args(bt=ctypes.c_void_p(0))) == -1
        assert fn(*args(q=ctypes.c_void_p(db.q.data_ptr() + 2))) == -1 and b"aligned" in lib.sangam_last_error(ctx)
        assert fn(*args(batch=b.batch + 1)) == -3 and b"max_batch" in lib.sangam_last_error(ctx)
        assert fn(*args(total_q=db.eng.cfg.max_total_q + 1)) == -3
        assert fn(*args(batch=-1)) == -1
        assert fn(*args(batch=0)) == 0 and fn(*args(total_q=0)) == 0          # nothing to do
    assert lib.sangam_block_attn(None, *args()[1:]) == -1
    kw = lambda **k: [ctx, k.get("k", P(db.k_new)), k.get("v", P(db.v_new)), k.get("slot", P(db.slot_new)),
                      k.get("n", int(db.slot_new.numel())), k.get("kp", P(db.k_pages)), k.get("vp", P(db.v_pages)), stream]
    assert lib.sangam_kv_write(*kw(k=ctypes.c_void_p(0))) == -1
    assert lib.sangam_kv_write(*kw(slot=ctypes.c_void_p(0))) == -1
    assert lib.sangam_kv_write(*kw(kp=ctypes.c_void_p(db.k_pages.data_ptr() + 8))) == -1
    assert lib.sangam_kv_write(*kw(n=-1)) == -1
    assert lib.sangam_kv_write(*kw(n=0, k=ctypes.c_void_p(0))) == 0               # empty write: no-op, pointers not looked at
    assert lib.sangam_kv_write(None, *kw()[1:]) == -1
    # iteration_host: null host pointers / counts above the maxima
    hq = db.q.cpu().pin_memory(); hk = db.k_new.cpu().pin_memory(); hv = db.v_new.cpu().pin_memory()
    hs = db.slot_new.cpu().pin_memory(); hbt = db.block_table.cpu().pin_memory(); hcu = db.cu_q_lens.cpu().pin_memory()
    hcl = db.ctx_lens.cpu().pin_memory(); ho = torch.empty_like(hq).pin_memory()
    ih = lambda **k: [ctx, k.get("q", P(hq)), P(hk), P(hv), P(hs), k.get("n", int(hs.numel())), P(db.k_pages), P(db.v_pages),
                      P(hbt), P(hcu), P(hcl), k.get("batch", b.batch), k.get("total_q", b.total_q),
                      ctypes.c_float(float(b.scale)), k.get("out", P(ho)), stream]
    assert lib.sangam_iteration_host(*ih(q=ctypes.c_void_p(0))) == -1
    assert lib.sangam_iteration_host(*ih(out=ctypes.c_void_p(0))) == -1
    assert lib.sangam_iteration_host(*ih(batch=b.batch + 1)) == -3
    assert lib.sangam_iteration_host(*ih(n=db.eng.cfg.max_total_q + 1)) == -3
    assert lib.sangam_set_dispatch(ctx, 7) == -1
    assert db.eng.launch_count() == n0, "a rejected call must not launch"
    # the ctx still works
    db.eng.set_dispatch(sg.DISPATCH_AUTO)
    db.iteration()
    assert db.eng.device_status() == 0


def test_geometry_without_a_decode_kernel():
    """G > 32: the decode kernel does not exist for the geometry; AUTO falls back to the two-stream kernel, DECODE is refused."""
    import paper_2607_04206_b200 as sg
    b = si.custom(62, [3, 2], [70, 33], num_q_heads=64, num_kv_heads=1, head_dim=64)
    db = DeviceBatch(b)
    assert db.eng.query(1) == 0
    with pytest.raises(sg.SangamError):
        db.eng.set_dispatch(sg.DISPATCH_DECODE)
    import oracle as o
    ref, _, _ = o.iteration(b)
    mx, mean = compare(db.iteration(), ref)
    assert mx <= MAX_ABS and mean <= MEAN_ABS


def test_geometry_without_a_pair_kernel():
    """MHA (G = 1): the CTA-pair GQA kernel does not exist for the geometry; GQA_PAIR is refused, AUTO is unaffected."""
    import paper_2607_04206_b200 as sg
    b = si.custom(63, [32, 5], [150, 40], num_q_heads=4, num_kv_heads=4, head_dim=64)
    db = DeviceBatch(b)
    assert db.eng.query(3) == 0
    with pytest.raises(sg.SangamError):
        db.eng.set_dispatch(sg.DISPATCH_GQA_PAIR)
    import oracle as o
    ref, _, _ = o.iteration(b)
    mx, mean = compare(db.iteration(), ref)
    assert mx <= MAX_ABS and mean <= MEAN_ABS
