// kv_write.cuh -- step a2: scatter fresh K/V rows into head-major bf16 pages.
//   k_pages[s/16][h][s%16][:] = k[i][h][:]  (and v), s = slot_mapping[i], s < 0 skipped.
// PagedAttention with 16-token pages; the refresh rewrites the whole
// cache at a block boundary and every step rewrites the current block.
// Pure data movement, HBM-bound: 16-byte vector loads/stores, one (token, head, 16B chunk) per
// thread-iteration, source fully coalesced, destination contiguous per (token, head) row.
#pragma once
#include "common.cuh"

template <int UNROLL>
__global__ void __launch_bounds__(256)
kv_write_kernel(const uint4* __restrict__ k, const uint4* __restrict__ v,
                const int32_t* __restrict__ slot_mapping, int32_t num_tokens,
                uint4* __restrict__ k_pages, uint4* __restrict__ v_pages,
                int32_t Hkv, int32_t chunks_per_row /* D/8 */, int32_t num_slots_total,
                uint32_t* flags) {
    // programmatic dependent launch: wait for the previous kernel in the stream (it may still read the pages), then let
    // the attention kernel behind this one run its shared-memory / TMEM prologue while the rows are copied
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int64_t chunks_per_token = (int64_t)Hkv * chunks_per_row;
    const int64_t total = (int64_t)num_tokens * chunks_per_token;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; idx < total; idx += stride * UNROLL) {
        uint4 kk[UNROLL], vv[UNROLL];
        int64_t dst[UNROLL];
        // the row data and the slot ids are fetched together (the data address does not depend on the slot): one
        // memory latency per pass instead of two.  Rows that turn out to be skipped (slot < 0) were read for nothing.
        int32_t sl[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            const int64_t e = idx + u * stride;
            sl[u] = -1;
            if (e < total) {
                sl[u] = __ldg(slot_mapping + (int32_t)(e / chunks_per_token));
                kk[u] = __ldcs(k + e);   // streamed once
                vv[u] = __ldcs(v + e);
            }
        }
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            const int64_t e = idx + u * stride;
            dst[u] = -1;
            const int32_t s = sl[u];
            if (e < total && s >= 0) {
                if (s < num_slots_total) {
                    const int32_t i = (int32_t)(e / chunks_per_token);
                    const int32_t rem = (int32_t)(e - (int64_t)i * chunks_per_token);
                    const int32_t h = rem / chunks_per_row, c = rem - h * chunks_per_row;
                    const int32_t page = s >> 4, off = s & 15;
                    dst[u] = (((int64_t)page * Hkv + h) * SANGAM_PAGE + off) * chunks_per_row + c;
                } else {
                    raise_flag(flags, DEV_BAD_SLOT);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < UNROLL; ++u)
            if (dst[u] >= 0) {
                k_pages[dst[u]] = kk[u];
                v_pages[dst[u]] = vv[u];
            }
    }
}
