// common.cuh -- shared declarations of the CUDA library (sm_100a only).
// Nothing here is shared with oracle/ (the CPU oracle has its own, separate source).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#define SANGAM_PAGE 16

// device-side sticky flags; values mirror include/sangam.h
#define DEV_BAD_SLOT 1u
#define DEV_BAD_PAGE 2u
#define DEV_CTX_TOO_LONG 4u
#define DEV_TIMEOUT 8u
#define DEV_BAD_POSITION 32u       // kv_write_rope: position outside the cos/sin table, row skipped
#define DEV_INTERNAL 16u           // an internal bounds guard tripped (library bug; the access was skipped)

struct AttnParams {
    const __nv_bfloat16* q;        // [total_q][Hq][D]
    const __nv_bfloat16* k_pages;  // [P][Hkv][16][D]
    const __nv_bfloat16* v_pages;
    const int32_t* block_table;    // [batch][W]
    const int32_t* cu_q_lens;      // [batch+1]
    const int32_t* ctx_lens;       // [batch]
    __nv_bfloat16* out;            // [total_q][Hq][D]
    int32_t batch, total_q;
    int32_t Hq, Hkv, G, W, P;
    int32_t tpt;                   // query tokens per 128-row q tile = 128 / G
    uint32_t tpt2_magic;           // floor(2^32 / (2 tpt)) + 1: x / (2 tpt) = umulhi(x, magic) for x < 2^24
    float scale;                   // natural-base logit scale
    float scale_log2;              // scale * log2(e)
    // split-KV workspace (library owned)
    float* part_o;                 // [num_slots][256][D]  unnormalised partial sums
    float* part_ml;                // [num_slots][256][2]  (m in log2 units, l)
    int32_t num_slots;
    void* slot_meta;               // [num_ctas] tc::SlotMeta, rewritten by every launch
    uint32_t* flags;               // sticky device flags
    int32_t* sched;                // [0] dynamic work counter (self-resetting), [1] finished-CTA count
    int32_t* plan_cache;           // [num_ctas][PLAN_CACHE_INTS]: each CTA's last plan, keyed by the batch's lengths
};
constexpr int PLAN_CACHE_INTS = 32 * 3 + 16;   // (q0, qn, c) of up to 32 requests + header

__device__ __forceinline__ void raise_flag(uint32_t* flags, uint32_t f) {
    if (flags) atomicOr(flags, f);
}

// All kernels are launched with programmatic stream serialization (they call griddepcontrol.wait before touching
// global memory), also under stream capture: the graph keeps the programmatic edges.
template <typename... KArgs, typename... Args>
static inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, unsigned block, size_t smem, cudaStream_t stream,
                                     Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, args...);
}

#include "trace.cuh"     // debug event trace: every macro is empty unless built with -DSANGAM_TRACE
