"""-m gpu parity tests: the CUDA path (through the C ABI) against the fp64 oracle, element by element."""
import numpy as np
import pytest

import sangam_inputs as si
from gpu_harness import MAX_ABS, MEAN_ABS, DeviceBatch, bits_of, compare

pytestmark = pytest.mark.gpu

PATHS = [pytest.param(False, id="tcgen05"), pytest.param(True, id="simt")]


def _check_pages(db, kp_ref, vp_ref):
    assert np.array_equal(bits_of(db.k_pages), kp_ref), "K pool differs (bit-exact required)"
    assert np.array_equal(bits_of(db.v_pages), vp_ref), "V pool differs (bit-exact required)"


@pytest.mark.parametrize("simt", PATHS)
def test_config1_tiny(oracle, simt, dispatch):
    b = si.config1()
    ref, kp, vp = oracle.iteration(b)
    db = DeviceBatch(b)
    if simt and dispatch:
        pytest.skip("the CUDA-core cross-check has no dispatch")
    out = db.iteration(simt=simt)
    _check_pages(db, kp, vp)
    mx, mean = compare(out, ref)
    print(f"config1 simt={simt}: max-abs {mx:.3e} mean-abs {mean:.3e}")
    assert mx <= MAX_ABS and mean <= MEAN_ABS
    assert mx <= 5 * 1.5e-3 * 2, "healthy error scale at c=128, D=64 is ~1.5e-3 (SURVEY 8(c))"
    assert db.eng.device_status() == 0


@pytest.mark.parametrize("simt", PATHS)
@pytest.mark.parametrize("cfg,shrink", [(2, 4), (3, 8), (4, 16), (5, 8)])
def test_configs_shrunk_full_compare(oracle, cfg, shrink, simt, dispatch):
    """Same structure as the BASELINE configs at sizes the oracle finishes in seconds; every element compared."""
    b = si.CONFIGS[cfg](shrink)
    ref, kp, vp = oracle.iteration(b)
    db = DeviceBatch(b)
    if simt and dispatch:
        pytest.skip("the CUDA-core cross-check has no dispatch")
    out = db.iteration(simt=simt)
    _check_pages(db, kp, vp)
    mx, mean = compare(out, ref)
    print(f"config{cfg}/{shrink} simt={simt}: max-abs {mx:.3e} mean-abs {mean:.3e}")
    assert mx <= MAX_ABS and mean <= MEAN_ABS
    assert db.eng.device_status() == 0


def test_kv_write_edge_cases(oracle):
    b = si.custom(31, [5, 9, 40], [37, 50, 129], num_q_heads=8, num_kv_heads=2, head_dim=128)
    import torch
    db = DeviceBatch(b)
    kp, vp = si.empty_pools(b)
    slots = b.slot_cache.copy()
    slots[[0, 17, 100]] = -1
    oracle.kv_write(b.k_cache, b.v_cache, slots, kp, vp)
    db.slot_cache = torch.from_numpy(slots).cuda()
    db.load_cache()
    torch.cuda.synchronize()
    _check_pages(db, kp, vp)                       # untouched (poisoned) slots preserved, negative slots skipped
    # empty write is a no-op
    db.eng.kv_write(db.k_cache[:0], db.v_cache[:0], db.slot_cache[:0], db.k_pages, db.v_pages)
    torch.cuda.synchronize()
    _check_pages(db, kp, vp)
    # out-of-range slot: skipped and flagged, nothing else disturbed
    bad = slots.copy(); bad[5] = b.num_pages * 16 + 3
    db.slot_cache = torch.from_numpy(bad).cuda()
    db.load_cache()
    assert db.eng.device_status() & 1
    db.eng.clear_device_status()
