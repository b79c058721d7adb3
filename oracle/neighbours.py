"""Plain fp64 numpy restatements of the two kernels next to the hot path.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  No code is shared with paper_2607_04206_b200/csrc/.

rope_rotate / kv_write_rope -- rotary position embedding applied to the fresh K rows just before they are scattered
  into the paged cache.  The paper does not print the rotation (it serves LLaDA-8B / Dream-7B, Llama- and Qwen-lineage
  models); reading S24 of DESIGN.md: the "rotate-half" convention of those lineages,
      theta_i = base^(-2 i / D),  i < D/2
      out[i]       = x[i] cos(pos theta_i) - x[i + D/2] sin(pos theta_i)
      out[i + D/2] = x[i + D/2] cos(pos theta_i) + x[i] sin(pos theta_i)
  K is rotated, V is copied unchanged; the scatter itself is oracle.kv_write's (slot = page * 16 + offset, slot < 0 skipped).

confidence_sample -- "Confidence-threshold based sampling unmasks every masked position whose top-1 probability exceeds
  a threshold", threshold 0.9.  Per row: p = softmax(logits), token = argmax (lowest index
  on ties), conf = p[token].  Per request (rows cu_rows[r] .. cu_rows[r+1]-1 = its current block): every still-masked
  row with conf > threshold is unmasked.  The paper is silent on a step in which no masked row passes; reading S23
  (Fast-dLLM's rule, which the paper names as the sampler it reuses): the single masked row with the highest
  confidence (lowest index on ties) is unmasked, so that every denoising step commits at least one position.
"""
from __future__ import annotations

import numpy as np


def _bf16_to_f64(b):
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def rope_rotate(x_bits, positions, base=10000.0):
    """x_bits uint16 [T][H][D] (bf16 patterns), positions int [T]  ->  float64 [T][H][D] (not rounded)."""
    x = _bf16_to_f64(x_bits)
    T, H, D = x.shape
    half = D // 2
    out = np.empty_like(x)
    for t in range(T):
        for i in range(half):
            theta = float(base) ** (-2.0 * i / D)
            ang = float(positions[t]) * theta
            c, s = np.cos(ang), np.sin(ang)
            out[t, :, i] = x[t, :, i] * c - x[t, :, i + half] * s
            out[t, :, i + half] = x[t, :, i + half] * c + x[t, :, i] * s
    return out


def kv_write_rope(k_bits, v_bits, slot_mapping, positions, base, k_pages_f64, v_pages_bits):
    """In place: k_pages_f64 float64 [P][Hkv][16][D] receives the rotated rows (exact fp64), v_pages_bits uint16 the copies."""
    kr = rope_rotate(k_bits, positions, base)
    for i, s in enumerate(np.asarray(slot_mapping)):
        if s < 0:
            continue
        page, off = int(s) // 16, int(s) % 16
        k_pages_f64[page, :, off, :] = kr[i]
        v_pages_bits[page, :, off, :] = v_bits[i]


def confidence_sample(logits_bits, masked, cu_rows, threshold):
    """logits_bits uint16 [rows][V]; masked int [rows] (1 = still masked); cu_rows int [R+1].
    Returns token int64 [rows], conf float64 [rows], unmask int32 [rows]."""
    x = _bf16_to_f64(logits_bits)
    rows, V = x.shape
    token = np.zeros(rows, np.int64)
    conf = np.zeros(rows, np.float64)
    for t in range(rows):
        m = x[t].max()
        token[t] = int(np.argmax(x[t]))                  # first index of the maximum
        conf[t] = 1.0 / np.sum(np.exp(x[t] - m))         # p[token] = exp(0) / sum
    unmask = np.zeros(rows, np.int32)
    for r in range(len(cu_rows) - 1):
        lo, hi = int(cu_rows[r]), int(cu_rows[r + 1])
        cand = [t for t in range(lo, hi) if masked[t]]
        if not cand:
            continue
        passed = [t for t in cand if conf[t] > threshold]
        if passed:
            unmask[passed] = 1
        else:
            best = max(cand, key=lambda t: (conf[t], -t))
            unmask[best] = 1
    return token, conf, unmask


def kv_gather(k_pages, v_pages, page_ids):
    """Pools uint16 [P][Hkv][16][D], page_ids int [n]  ->  staging copies [n][Hkv][16][D] (whole-request KV)."""
    ks = np.empty((len(page_ids),) + k_pages.shape[1:], k_pages.dtype)
    vs = np.empty_like(ks)
    for i, pg in enumerate(page_ids):
        ks[i] = k_pages[int(pg)]
        vs[i] = v_pages[int(pg)]
    return ks, vs


def kv_scatter(k_stage, v_stage, page_ids, k_pages, v_pages):
    """In place: the receiver's pages take the staged copies."""
    for i, pg in enumerate(page_ids):
        k_pages[int(pg)] = k_stage[i]
        v_pages[int(pg)] = v_stage[i]
