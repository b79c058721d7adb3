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
    float scale;                   // natural-base logit scale
    float scale_log2;              // scale * log2(e)
    // split-KV workspace (library owned)
    float* part_o;                 // [num_slots][256][D]  unnormalised partial sums
    float* part_ml;                // [num_slots][256][2]  (m in log2 units, l)
    int32_t num_slots;
    int32_t* unit_count;           // [num_ctas] pieces of a split unit finished so far (self-resetting)
    uint32_t* flags;               // sticky device flags
    int32_t* sched;                // [0] dynamic work counter (self-resetting), [1] finished-CTA count
};

__device__ __forceinline__ void raise_flag(uint32_t* flags, uint32_t f) {
    if (flags) atomicOr(flags, f);
}
