"""Whole-request KV page transfer between two workers:
the prefill worker gathers the request's pages into a contiguous staging buffer (sangam_kv_gather), the buffer crosses
NVLink with torch.distributed send / recv (NCCL on GPUs; the paper moves whole requests, not layers), the decode-role
worker scatters it into the pages it allocated (sangam_kv_scatter).  A small int64 header announces the request.

Plumbing only: every byte is moved by the library's kernels or by the collective library.  `gather` / `scatter` are the
engine's methods in production; tests on CPU (gloo, world size 2) pass stand-ins to exercise the framing and ordering.
"""
from __future__ import annotations

HEADER_INTS = 4      # request id, context length, number of pages, number of layers


def send_request_kv(dist, dst, req_id, ctx_len, page_ids, layers, gather, new_stage, tag=0):
    """layers: list of (k_pages, v_pages) per layer; page_ids: the request's pages on this worker (int32 tensor);
    gather(k_pages, v_pages, page_ids, k_stage, v_stage) fills the staging pair; new_stage(n_pages) allocates one."""
    import torch
    n = int(page_ids.numel())
    hdr = torch.tensor([int(req_id), int(ctx_len), n, len(layers)], dtype=torch.int64, device=page_ids.device)
    dist.send(hdr, dst=dst, tag=tag)
    for k_pages, v_pages in layers:
        k_stage, v_stage = new_stage(n)
        gather(k_pages, v_pages, page_ids, k_stage, v_stage)
        dist.send(k_stage, dst=dst, tag=tag)
        dist.send(v_stage, dst=dst, tag=tag)


def recv_request_kv(dist, src, layers, alloc_pages, scatter, new_stage, device, tag=0):
    """alloc_pages(n_pages) -> int32 tensor of this worker's page ids for the request.  Returns (req_id, ctx_len, page_ids)."""
    import torch
    hdr = torch.zeros(HEADER_INTS, dtype=torch.int64, device=device)
    dist.recv(hdr, src=src, tag=tag)
    req_id, ctx_len, n, n_layers = (int(x) for x in hdr.tolist())
    if n_layers != len(layers):
        raise ValueError(f"sender has {n_layers} layers, receiver {len(layers)}")
    page_ids = alloc_pages(n)
    for k_pages, v_pages in layers:
        k_stage, v_stage = new_stage(n)
        dist.recv(k_stage, src=src, tag=tag)
        dist.recv(v_stage, src=src, tag=tag)
        scatter(k_stage, v_stage, page_ids, k_pages, v_pages)
    return req_id, ctx_len, page_ids
