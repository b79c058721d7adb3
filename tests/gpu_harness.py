"""Shared helpers of the -m gpu parity tests: put a sangam_inputs.Batch on the device, run the
iteration through the C ABI binding, compare with the fp64 oracle."""
from __future__ import annotations

import numpy as np

import sangam_inputs as si

MAX_ABS, MEAN_ABS = 2e-2, 2e-3      # north_star tolerance for bf16-in / fp32-accumulate attention

# which attention kernel sangam_block_attn launches in DeviceBatch (0 auto, 1 two-stream prefill kernel, 2 decode
# kernel, 3 CTA-pair GQA decode kernel); set per test by the `dispatch` fixture of conftest.py so that every parity /
# edge case runs through all of them
DEFAULT_DISPATCH = 0


def t_bf16(bits: np.ndarray, device="cuda"):
    import torch
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).to(device).view(torch.bfloat16)


def t_i32(a: np.ndarray, device="cuda"):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).to(device)


def bits_of(t) -> np.ndarray:
    import torch
    return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


class DeviceBatch:
    def __init__(self, b: si.Batch, poison=True, max_total_q=None, max_batch=None):
        import paper_2607_04206_b200 as sg
        self.b = b
        kp, vp = si.empty_pools(b, poison=poison)
        self.k_pages, self.v_pages = t_bf16(kp), t_bf16(vp)
        self.q = t_bf16(b.q)
        self.k_cache, self.v_cache = t_bf16(b.k_cache), t_bf16(b.v_cache)
        self.k_new, self.v_new = t_bf16(b.k_new), t_bf16(b.v_new)
        self.slot_cache, self.slot_new = t_i32(b.slot_cache), t_i32(b.slot_new)
        self.block_table, self.cu_q_lens, self.ctx_lens = t_i32(b.block_table), t_i32(b.cu_q_lens), t_i32(b.ctx_lens)
        import torch
        self.out = torch.full_like(self.q, float("nan"))
        self.eng = sg.Sangam(num_q_heads=b.num_q_heads, num_kv_heads=b.num_kv_heads, head_dim=b.head_dim,
                             num_pages=b.num_pages, max_batch=max_batch or max(b.batch, 1),
                             max_total_q=max_total_q or max(b.total_q, len(b.slot_cache), 1),
                             max_pages_per_req=b.max_pages_per_req)
        if DEFAULT_DISPATCH:
            if DEFAULT_DISPATCH == sg.DISPATCH_GQA_PAIR and self.eng.query(3) != 1:
                import pytest
                pytest.skip("no CTA-pair kernel for this geometry (it needs 1 < num_q_heads / num_kv_heads <= 128)")
            if DEFAULT_DISPATCH == sg.DISPATCH_DECODE and self.eng.query(1) <= 0:
                import pytest
                pytest.skip("no decode kernel for this geometry (it needs num_q_heads / num_kv_heads <= 32)")
            self.eng.set_dispatch(DEFAULT_DISPATCH)

    def load_cache(self):
        self.eng.kv_write(self.k_cache, self.v_cache, self.slot_cache, self.k_pages, self.v_pages)

    def write_new(self):
        self.eng.kv_write(self.k_new, self.v_new, self.slot_new, self.k_pages, self.v_pages)

    def attend(self, simt=False):
        self.eng.block_attn(self.q, self.k_pages, self.v_pages, self.block_table, self.cu_q_lens, self.ctx_lens,
                            float(self.b.scale), self.out, simt=simt)

    def iteration(self, simt=False):
        self.load_cache()
        self.write_new()
        self.attend(simt=simt)
        import torch
        torch.cuda.synchronize()
        return self.out


def compare(out_gpu, ref: np.ndarray, rows=None):
    """max-abs / mean-abs of bf16 GPU output (widened) against the fp64 oracle."""
    got = si.bf16_bits_to_f64(bits_of(out_gpu))
    if rows is not None:
        got = got[np.asarray(rows)]
    assert got.shape == ref.shape, (got.shape, ref.shape)
    assert np.all(np.isfinite(got)), "NaN/Inf in GPU output"
    err = np.abs(got - ref)
    return float(err.max()) if err.size else 0.0, float(err.mean()) if err.size else 0.0
