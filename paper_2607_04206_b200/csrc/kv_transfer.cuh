// kv_transfer.cuh -- the single-GPU halves of the paper's only GPU-to-GPU data path: a request's KV pages move from a
// prefill worker to a decode-role worker ("transfer KV from the first to the second"; NCCL over NVLink,
// p99 384 ms / 192 ms per request).  SURVEY.md 8(f) rank 3.
//   gather : pool pages listed in page_ids  ->  one contiguous staging buffer [n][Hkv][16][D] (what the sender hands to
//            NCCL send / a peer copy)
//   scatter: staging buffer  ->  the pages the receiver allocated for the request (its own page ids)
// A (page, all heads) is one contiguous Hkv*16*D*2-byte block in the head-major pool, so both directions are block
// copies: 16-byte vectors, fully coalesced on both sides, HBM-bound.  A page id outside [0, P) skips that page and raises
// SANGAM_DEV_BAD_PAGE.  The transfer between the two GPUs itself (torch.distributed send / recv) is in kv_transfer.py.
#pragma once
#include "common.cuh"

template <bool GATHER>
__global__ void __launch_bounds__(256)
kv_pages_copy_kernel(uint4* __restrict__ k_pool, uint4* __restrict__ v_pool, uint4* __restrict__ k_stage, uint4* __restrict__ v_stage,
                     const int32_t* __restrict__ page_ids, int32_t n, int32_t chunks_per_page, int32_t P, uint32_t* flags) {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int64_t total = (int64_t)n * chunks_per_page;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int32_t i = (int32_t)(idx / chunks_per_page);
        const int32_t c = (int32_t)(idx - (int64_t)i * chunks_per_page);
        const int32_t pg = __ldg(page_ids + i);
        if ((unsigned)pg >= (unsigned)P) { if (c == 0) raise_flag(flags, DEV_BAD_PAGE); continue; }
        const int64_t pool = (int64_t)pg * chunks_per_page + c;
        if (GATHER) { k_stage[idx] = __ldcs(k_pool + pool); v_stage[idx] = __ldcs(v_pool + pool); }
        else { k_pool[pool] = __ldcs(k_stage + idx); v_pool[pool] = __ldcs(v_stage + idx); }
    }
}
