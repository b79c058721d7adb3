"""ctypes binding with the same names as include/sangam.h.  torch tensors are used only as
device memory: the binding passes `tensor.data_ptr()` and the current CUDA stream handle."""
from __future__ import annotations

import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libsangam.so")

DECLARED_SYMBOLS = [
    "sangam_create", "sangam_destroy", "sangam_kv_write", "sangam_block_attn", "sangam_block_attn_simt",
    "sangam_iteration_host", "sangam_device_status", "sangam_clear_device_status", "sangam_launch_count",
    "sangam_last_error", "sangam_version", "sangam_set_dispatch", "sangam_query",
    "sangam_sched_create", "sangam_sched_destroy", "sangam_sched_submit", "sangam_sched_next", "sangam_sched_complete",
    "sangam_sched_query", "sangam_packed_layout", "sangam_iteration_packed",
    "sangam_kv_write_rope", "sangam_confidence_sample", "sangam_kv_gather", "sangam_kv_scatter",
    "sangam_confidence_sample_static", "sangam_static_last_error",
]

DISPATCH_AUTO, DISPATCH_PREFILL, DISPATCH_DECODE, DISPATCH_GQA_PAIR = 0, 1, 2, 3


class SangamError(RuntimeError):
    pass


class _Config(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in (
        "num_q_heads", "num_kv_heads", "head_dim", "page_size", "num_pages", "max_batch", "max_total_q",
        "max_pages_per_req", "device")]


class _SchedConfig(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("tau", "block", "page_size", "num_pages", "max_batch", "max_total_q", "max_pages_per_req")]


class _Batch(ctypes.Structure):
    _fields_ = [("batch", ctypes.c_int32), ("num_decodes", ctypes.c_int32), ("total_q", ctypes.c_int32),
                ("num_new_tokens", ctypes.c_int32), ("deficit", ctypes.c_int64),
                ("req_ids", ctypes.c_void_p), ("cu_q_lens", ctypes.c_void_p), ("ctx_lens", ctypes.c_void_p),
                ("block_table", ctypes.c_void_p), ("slot_mapping", ctypes.c_void_p)]


_lib = None


def load_library(build_if_missing: bool = False):
    """dlopen libsangam.so; fails loudly when it is missing (no fallback path exists)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        if build_if_missing:
            from .build import build
            build()
        else:
            raise SangamError(f"{LIB_PATH} not built: run `python -m paper_2607_04206_b200.build`")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, f32 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_float
    lib.sangam_create.argtypes = [ctypes.POINTER(_Config), ctypes.POINTER(vp)]
    lib.sangam_destroy.argtypes = [vp]
    lib.sangam_kv_write.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp]
    lib.sangam_block_attn.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, f32, vp, vp]
    lib.sangam_block_attn_simt.argtypes = lib.sangam_block_attn.argtypes
    lib.sangam_iteration_host.argtypes = [vp, vp, vp, vp, vp, i32, vp, vp, vp, vp, vp, i32, i32, f32, vp, vp]
    lib.sangam_device_status.argtypes = [vp, ctypes.POINTER(ctypes.c_uint32)]
    lib.sangam_clear_device_status.argtypes = [vp]
    lib.sangam_launch_count.argtypes = [vp]
    lib.sangam_launch_count.restype = ctypes.c_int64
    lib.sangam_last_error.argtypes = [vp]
    lib.sangam_last_error.restype = ctypes.c_char_p
    lib.sangam_version.restype = ctypes.c_char_p
    lib.sangam_set_dispatch.argtypes = [vp, i32]
    lib.sangam_query.argtypes = [vp, i32]
    lib.sangam_query.restype = i32
    lib.sangam_packed_layout.argtypes = [vp, i32, i32, i32, ctypes.POINTER(ctypes.c_int64)]
    lib.sangam_iteration_packed.argtypes = [vp, vp, i32, vp, vp, i32, i32, f32, vp, vp]
    lib.sangam_kv_write_rope.argtypes = [vp, vp, vp, vp, vp, vp, i32, i32, vp, vp, vp]
    lib.sangam_confidence_sample.argtypes = [vp, vp, i32, vp, vp, i32, i32, f32, vp, vp, vp, vp]
    lib.sangam_confidence_sample_static.argtypes = [vp, i32, vp, vp, i32, i32, f32, vp, vp, vp, vp]
    lib.sangam_static_last_error.restype = ctypes.c_char_p
    lib.sangam_kv_gather.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp]
    lib.sangam_kv_scatter.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp]
    lib.sangam_sched_create.argtypes = [ctypes.POINTER(_SchedConfig), ctypes.POINTER(vp)]
    lib.sangam_sched_destroy.argtypes = [vp]
    lib.sangam_sched_submit.argtypes = [vp, ctypes.c_int64, ctypes.c_double, i32, i32, i32]
    lib.sangam_sched_next.argtypes = [vp, ctypes.POINTER(_Batch)]
    lib.sangam_sched_complete.argtypes = [vp, vp, i32]
    lib.sangam_sched_query.argtypes = [vp, i32]
    lib.sangam_sched_query.restype = ctypes.c_int64
    _lib = lib
    return lib


def exported_symbols():
    lib = load_library()
    return [s for s in DECLARED_SYMBOLS if hasattr(lib, s)]


def _ptr(t):
    return ctypes.c_void_p(0 if t is None else t.data_ptr())


def _stream(stream):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return ctypes.c_void_p(s.cuda_stream)


STATIC_SAMPLER_MAX_ROWS, STATIC_SAMPLER_MAX_PARTIALS = 4096, 65536      # include/sangam.h


def confidence_sample_static(logits, masked, cu_rows, threshold, token, conf, unmask, stream=None):
    """sangam_confidence_sample_static: the sampler without a ctx and without any allocation (its scratch is a 1 MiB
    static device array inside the library); same arguments and results as Sangam.confidence_sample, on the current
    device, rows <= STATIC_SAMPLER_MAX_ROWS.  Calls that overlap on the GPU race on the shared scratch."""
    lib = load_library()
    rc = lib.sangam_confidence_sample_static(_ptr(logits), int(logits.shape[1]), _ptr(masked), _ptr(cu_rows), int(cu_rows.numel()) - 1,
                                             int(logits.shape[0]), float(threshold), _ptr(token), _ptr(conf), _ptr(unmask), _stream(stream))
    if rc != 0:
        raise SangamError(f"sangam error {rc}: {lib.sangam_static_last_error().decode()}")


def rope_table(max_pos: int, head_dim: int, base: float = 10000.0):
    """Host-side cos/sin cache for sangam_kv_write_rope: float32 numpy [max_pos][head_dim], row p = cos(p theta_j) for j < D/2
    then sin(p theta_j), theta_j = base^(-2j/D), evaluated in float64 (what serving stacks cache once per model)."""
    import numpy as np
    j = np.arange(head_dim // 2, dtype=np.float64)
    ang = np.arange(max_pos, dtype=np.float64)[:, None] * (float(base) ** (-2.0 * j / head_dim))[None, :]
    return np.concatenate([np.cos(ang), np.sin(ang)], axis=1).astype(np.float32)


class Sangam:
    """One sangam_ctx (geometry + library workspace).  Methods mirror the C entry points."""

    def __init__(self, *, num_q_heads, num_kv_heads, head_dim, num_pages, max_batch, max_total_q,
                 max_pages_per_req, page_size=16, device=0):
        import torch
        if not torch.cuda.is_available():
            raise SangamError("no CUDA device: the sangam kernels have no CPU fallback")
        self.lib = load_library()
        self.cfg = _Config(num_q_heads, num_kv_heads, head_dim, page_size, num_pages, max_batch, max_total_q,
                           max_pages_per_req, device)
        self.ctx = ctypes.c_void_p()
        rc = self.lib.sangam_create(ctypes.byref(self.cfg), ctypes.byref(self.ctx))
        if rc != 0:
            raise SangamError(f"sangam_create failed: {rc}")

    def _check(self, rc):
        if rc != 0:
            raise SangamError(f"sangam error {rc}: {self.lib.sangam_last_error(self.ctx).decode()}")

    def close(self):
        if self.ctx:
            self.lib.sangam_destroy(self.ctx)
            self.ctx = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def kv_write(self, k, v, slot_mapping, k_pages, v_pages, stream=None):
        self._check(self.lib.sangam_kv_write(self.ctx, _ptr(k), _ptr(v), _ptr(slot_mapping), int(slot_mapping.numel()),
                                             _ptr(k_pages), _ptr(v_pages), _stream(stream)))

    def kv_write_rope(self, k, v, slot_mapping, positions, cos_sin, k_pages, v_pages, stream=None):
        """cos_sin: device fp32 [max_pos][head_dim] (see rope_table)."""
        self._check(self.lib.sangam_kv_write_rope(self.ctx, _ptr(k), _ptr(v), _ptr(slot_mapping), _ptr(positions), _ptr(cos_sin),
                                                  int(cos_sin.shape[0]), int(slot_mapping.numel()), _ptr(k_pages), _ptr(v_pages), _stream(stream)))

    def confidence_sample(self, logits, masked, cu_rows, threshold, token, conf, unmask, stream=None):
        """logits bf16 [rows][vocab]; masked int32 [rows]; cu_rows int32 [R+1]; outputs token int32, conf fp32, unmask int32."""
        self._check(self.lib.sangam_confidence_sample(self.ctx, _ptr(logits), int(logits.shape[1]), _ptr(masked), _ptr(cu_rows),
                                                      int(cu_rows.numel()) - 1, int(logits.shape[0]), float(threshold), _ptr(token),
                                                      _ptr(conf), _ptr(unmask), _stream(stream)))

    def kv_gather(self, k_pages, v_pages, page_ids, k_stage, v_stage, stream=None):
        self._check(self.lib.sangam_kv_gather(self.ctx, _ptr(k_pages), _ptr(v_pages), _ptr(page_ids), int(page_ids.numel()),
                                              _ptr(k_stage), _ptr(v_stage), _stream(stream)))

    def kv_scatter(self, k_stage, v_stage, page_ids, k_pages, v_pages, stream=None):
        self._check(self.lib.sangam_kv_scatter(self.ctx, _ptr(k_stage), _ptr(v_stage), _ptr(page_ids), int(page_ids.numel()),
                                               _ptr(k_pages), _ptr(v_pages), _stream(stream)))

    def block_attn(self, q, k_pages, v_pages, block_table, cu_q_lens, ctx_lens, scale, out, stream=None, simt=False):
        fn = self.lib.sangam_block_attn_simt if simt else self.lib.sangam_block_attn
        self._check(fn(self.ctx, _ptr(q), _ptr(k_pages), _ptr(v_pages), _ptr(block_table), _ptr(cu_q_lens),
                       _ptr(ctx_lens), int(ctx_lens.numel()), int(q.shape[0]), float(scale), _ptr(out), _stream(stream)))

    def iteration_host(self, q, k, v, slot_mapping, k_pages, v_pages, block_table, cu_q_lens, ctx_lens, scale, out,
                       stream=None):
        """q, k, v, slot_mapping, block_table, cu_q_lens, ctx_lens, out: HOST (pinned) tensors; pools on device."""
        self._check(self.lib.sangam_iteration_host(
            self.ctx, _ptr(q), _ptr(k), _ptr(v), _ptr(slot_mapping), int(slot_mapping.numel()), _ptr(k_pages),
            _ptr(v_pages), _ptr(block_table), _ptr(cu_q_lens), _ptr(ctx_lens), int(ctx_lens.numel()), int(q.shape[0]),
            float(scale), _ptr(out), _stream(stream)))

    def packed_layout(self, batch, total_q, num_tokens):
        """Byte offsets of q, k, v, slot_mapping, block_table, cu_q_lens, ctx_lens in the packed host buffer + total size."""
        off = (ctypes.c_int64 * 8)()
        self._check(self.lib.sangam_packed_layout(self.ctx, int(batch), int(total_q), int(num_tokens), off))
        return list(off)

    def iteration_packed(self, packed, num_tokens, k_pages, v_pages, batch, total_q, scale, out, stream=None):
        """packed, out: HOST (pinned) tensors; one H2D copy, kv_write + block_attn, one D2H copy, stream synchronize."""
        self._check(self.lib.sangam_iteration_packed(self.ctx, _ptr(packed), int(num_tokens), _ptr(k_pages), _ptr(v_pages), int(batch),
                                                     int(total_q), float(scale), _ptr(out), _stream(stream)))

    def set_dispatch(self, mode: int):
        """DISPATCH_AUTO / DISPATCH_PREFILL / DISPATCH_DECODE: which attention kernel sangam_block_attn launches."""
        self._check(self.lib.sangam_set_dispatch(self.ctx, int(mode)))

    def query(self, what: int) -> int:
        """0: SM count, 1: decode-kernel CTAs per SM, 2: dispatch mode, 3: 1 if the CTA-pair GQA kernel exists for the
        geometry, 4: the kernel the last block_attn launched (DISPATCH_PREFILL / DECODE / GQA_PAIR, 0 before the first)."""
        return int(self.lib.sangam_query(self.ctx, int(what)))

    def device_status(self) -> int:
        f = ctypes.c_uint32(0)
        self._check(self.lib.sangam_device_status(self.ctx, ctypes.byref(f)))
        return int(f.value)

    def clear_device_status(self):
        self._check(self.lib.sangam_clear_device_status(self.ctx))

    def launch_count(self) -> int:
        return int(self.lib.sangam_launch_count(self.ctx))


class Scheduler:
    """sangam_sched (Algorithm 1 + batch metadata).  Host only: works without a CUDA device.  The batch arrays are
    torch tensors when `pinned` (pinned host memory, ready for cudaMemcpyAsync), numpy arrays otherwise."""

    def __init__(self, *, tau, num_pages, max_batch, max_total_q, max_pages_per_req, block=32, page_size=16, pinned=False):
        import numpy as np
        self.lib = load_library()
        self.cfg = _SchedConfig(tau, block, page_size, num_pages, max_batch, max_total_q, max_pages_per_req)
        self.s = ctypes.c_void_p()
        rc = self.lib.sangam_sched_create(ctypes.byref(self.cfg), ctypes.byref(self.s))
        if rc != 0:
            raise SangamError(f"sangam_sched_create failed: {rc}")
        shapes = {"req_ids": ((max_batch,), np.int64), "cu_q_lens": ((max_batch + 1,), np.int32), "ctx_lens": ((max_batch,), np.int32),
                  "block_table": ((max_batch, max_pages_per_req), np.int32), "slot_mapping": ((max_total_q,), np.int32)}
        self.tensors = {}
        self.arrays = {}
        for k, (shp, dt) in shapes.items():
            if pinned:
                import torch
                t = torch.zeros(shp, dtype=torch.int64 if dt is np.int64 else torch.int32).pin_memory()
                self.tensors[k] = t
                self.arrays[k] = t.numpy()
            else:
                self.arrays[k] = np.zeros(shp, dtype=dt)
        self.b = _Batch()
        for k, a in self.arrays.items():
            setattr(self.b, k, a.ctypes.data)

    def close(self):
        if self.s:
            self.lib.sangam_sched_destroy(self.s)
            self.s = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def submit(self, req_id, arrival_time, prompt_len, response_len, output_len) -> int:
        return int(self.lib.sangam_sched_submit(self.s, int(req_id), float(arrival_time), int(prompt_len), int(response_len), int(output_len)))

    def next(self):
        """Runs one iteration of Algorithm 1; returns the filled batch header (arrays in self.arrays / self.tensors)."""
        rc = self.lib.sangam_sched_next(self.s, ctypes.byref(self.b))
        if rc != 0:
            raise SangamError(f"sangam_sched_next failed: {rc}")
        return self.b

    def complete(self, block_done):
        import numpy as np
        a = np.ascontiguousarray(block_done, dtype=np.int32)
        rc = self.lib.sangam_sched_complete(self.s, ctypes.c_void_p(a.ctypes.data if len(a) else 0), int(len(a)))
        if rc != 0:
            raise SangamError(f"sangam_sched_complete failed: {rc}")

    def query(self, what: int) -> int:
        return int(self.lib.sangam_sched_query(self.s, int(what)))
