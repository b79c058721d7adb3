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

// Optional event trace of CTA 0 (debug builds with -DSANGAM_TRACE only; compiled out otherwise).
#ifdef SANGAM_TRACE
#define SANGAM_TRACE_CAP 8192            // events per warp
__device__ unsigned long long g_trace[16 * SANGAM_TRACE_CAP];
__device__ unsigned int g_trace_n[16];
__device__ unsigned long long g_cta_times[2 * 512];   // per CTA: %globaltimer at entry / exit
__device__ unsigned int g_trace_cta;     // which CTA records (sangam_trace_set_cta)
__device__ __forceinline__ unsigned int* trace_cnt() {
    __shared__ unsigned int cnt[17];      // [16] = 1 if this CTA records (g_trace_cta read once: a global read per event costs an L2 trip)
    return cnt;
}
__device__ __forceinline__ void trace_ev(unsigned ev) {
    unsigned int* cnt = trace_cnt();
    if (cnt[16] && (threadIdx.x & 31) == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%clock64;" : "=l"(t));
        const unsigned w = threadIdx.x >> 5, i = cnt[w];
        cnt[w] = i + 1;
        if (i < SANGAM_TRACE_CAP) g_trace[w * SANGAM_TRACE_CAP + i] = (t << 16) | ((unsigned long long)w << 8) | ev;
        g_trace_n[w] = i + 1;
    }
}
// same record, but the time stamp is %globaltimer (ns): start/end pair gives the effective SM clock
__device__ __forceinline__ void trace_ns(unsigned ev) {
    unsigned int* cnt = trace_cnt();
    if (cnt[16] && (threadIdx.x & 31) == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        const unsigned w = threadIdx.x >> 5, i = cnt[w];
        cnt[w] = i + 1;
        if (i < SANGAM_TRACE_CAP) g_trace[w * SANGAM_TRACE_CAP + i] = (t << 16) | ((unsigned long long)w << 8) | ev;
        g_trace_n[w] = i + 1;
    }
}
#define TRACE_EV(ev) trace_ev(ev)
#define TRACE_NS(ev) trace_ns(ev)
// bits 63..54 of the entry stamp carry %smid (the timer's high bits are constant over a launch: the host masks them off)
#define TRACE_CTA(which) do { if (threadIdx.x == 0 && blockIdx.x < 512) { unsigned long long t_; unsigned sm_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); asm volatile("mov.u32 %0, %%smid;" : "=r"(sm_)); g_cta_times[2 * blockIdx.x + (which)] = (which) ? t_ : ((t_ & 0x003fffffffffffffull) | ((unsigned long long)sm_ << 54)); } } while (0)
#define TRACE_INIT() do { if (threadIdx.x < 16) trace_cnt()[threadIdx.x] = 0; if (threadIdx.x == 16) trace_cnt()[16] = blockIdx.x == g_trace_cta; __syncthreads(); } while (0)
#else
#define TRACE_EV(ev) ((void)0)
#define TRACE_NS(ev) ((void)0)
#define TRACE_CTA(which) ((void)0)
#define TRACE_INIT() ((void)0)
#endif
