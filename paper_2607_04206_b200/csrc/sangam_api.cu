// sangam_api.cu -- the C ABI of include/sangam.h: argument checks, workspace, kernel launches.
// Every step of the path runs in the kernels of this directory; there is no CPU fallback.
#include "../../include/sangam.h"

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <new>

#include "attn_dec.cuh"
#include "attn_gqa.cuh"
#include "attn_simt.cuh"
#include "attn_tc.cuh"
#include "common.cuh"
#include "kv_transfer.cuh"
#include "kv_write.cuh"
#include "neighbours.cuh"
#include "sched.cuh"

constexpr int MAP_CACHE = 64;
struct MapCacheKV { const void *k, *v; uint64_t tick; CUtensorMap mk, mv; };
struct MapCacheQ { const void* q; int32_t rows; uint64_t tick; CUtensorMap main, dec; };

struct sangam_ctx {
    sangam_config cfg;
    int sm_count;
    int G;
    uint32_t* d_flags;
    int32_t* d_sched;
    float* d_part_o;
    float* d_part_ml;
    void* d_slot_meta;
    int32_t* d_plan_cache;
    int32_t num_slots;
    // decode kernel (attn_dec.cuh): resident CTAs per SM (0: unavailable), its split-KV workspace
    int dec_occ;
    int gqa_ok;                   // GQA pair kernel (attn_gqa.cuh) available for this geometry
    int dispatch;                 // SANGAM_DISPATCH_*
    int last_kernel;              // SANGAM_DISPATCH_PREFILL / DECODE / GQA_PAIR: what the last sangam_block_attn launched (0: nothing yet)
    float* d_dec_part_o;
    float* d_dec_part_ml;
    int32_t* d_dec_cnt;
    // tensor-map caches: a model passes per-layer pools and per-layer q buffers, so the encoded maps are kept per
    // (k_pages, v_pages) and per (q, total_q) -- cuTensorMapEncodeTiled costs microseconds of host time per call
    MapCacheKV kv_cache[MAP_CACHE];
    MapCacheQ q_cache[MAP_CACHE];
    uint64_t map_tick;
    // staging for sangam_iteration_host (allocated on first use)
    void *s_q, *s_k, *s_v, *s_out;
    ConfPartial* d_conf_part;     // sampler: per (row, vocabulary slice) partials, grown on demand
    int64_t conf_part_cap;
    void* s_packed;               // staging of sangam_iteration_packed
    int64_t s_packed_bytes;
    int32_t *s_slot, *s_bt, *s_cu, *s_ctx;
    int64_t launches;
    char err[512];
};

static int fail(sangam_ctx* c, int code, const char* fmt, const char* detail = "") {
    if (c) snprintf(c->err, sizeof c->err, fmt, detail);
    return code;
}
static int cuda_fail(sangam_ctx* c, cudaError_t e, const char* where) {
    if (c) snprintf(c->err, sizeof c->err, "%s: %s", where, cudaGetErrorString(e));
    return SANGAM_ERR_CUDA;
}
#define CK(call)                                                  \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);  \
    } while (0)

// Every entry point runs on the ctx's device whatever device the calling thread has current, and leaves the
// caller's current device as it found it.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int dev) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != dev) {
            err = cudaSetDevice(dev);
            switched = err == cudaSuccess;
        }
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};
#define ON_CTX_DEVICE(ctx)                                                          \
    DeviceGuard guard_((ctx)->cfg.device);                                         \
    if (guard_.err != cudaSuccess) return cuda_fail((ctx), guard_.err, "cudaSetDevice")

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

extern "C" const char* sangam_version(void) { return "sangam-b200 0.1 (sm_100a)"; }

extern "C" const char* sangam_last_error(const sangam_ctx* ctx) { return ctx ? ctx->err : "null ctx"; }

extern "C" int64_t sangam_launch_count(const sangam_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" int sangam_create(const sangam_config* cfg, sangam_ctx** out) {
    if (!cfg || !out) return SANGAM_ERR_INVALID_ARG;
    *out = nullptr;
    if (cfg->page_size != SANGAM_PAGE) return SANGAM_ERR_UNSUPPORTED;
    if (cfg->head_dim != 64 && cfg->head_dim != 128) return SANGAM_ERR_UNSUPPORTED;
    if (cfg->num_q_heads <= 0 || cfg->num_kv_heads <= 0 || cfg->num_q_heads % cfg->num_kv_heads) return SANGAM_ERR_INVALID_ARG;
    if (cfg->num_q_heads / cfg->num_kv_heads > 128) return SANGAM_ERR_UNSUPPORTED;   // a q tile holds whole tokens of one group
    if (cfg->num_pages <= 0 || cfg->max_batch <= 0 || cfg->max_total_q <= 0 || cfg->max_pages_per_req <= 0)
        return SANGAM_ERR_INVALID_ARG;
    if ((int64_t)cfg->num_pages * SANGAM_PAGE > 0x7fffffffLL) return SANGAM_ERR_INVALID_ARG;
    // TMA page coordinate (page * Hkv + g) * 2 (and the out-of-range coordinate of a bad page id) must fit an int32
    if (((int64_t)cfg->num_pages + 1) * cfg->num_kv_heads * 2 > 0x7fffffffLL) return SANGAM_ERR_INVALID_ARG;
    // the planners divide row counts by a magic multiplier that is exact below 2^24
    if (cfg->max_total_q >= (1 << 24)) return SANGAM_ERR_INVALID_ARG;
    sangam_ctx* ctx = new (std::nothrow) sangam_ctx();
    if (!ctx) return SANGAM_ERR_WORKSPACE;
    memset(ctx, 0, sizeof *ctx);
    ctx->cfg = *cfg;
    ctx->G = cfg->num_q_heads / cfg->num_kv_heads;
    DeviceGuard guard(cfg->device);                     // the caller's current device is restored on return
    cudaError_t e = guard.err;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, cfg->device);
    ctx->num_slots = 2 * (ctx->sm_count > 0 ? ctx->sm_count : 148);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_flags, sizeof(uint32_t));
    if (e == cudaSuccess) e = cudaMemset(ctx->d_flags, 0, sizeof(uint32_t));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_sched, 16 * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemset(ctx->d_sched, 0, 16 * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_part_o, (size_t)ctx->num_slots * 256 * cfg->head_dim * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_part_ml, (size_t)ctx->num_slots * 256 * 2 * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_slot_meta, (size_t)ctx->num_slots * 32);
    if (e == cudaSuccess) e = cudaMemset(ctx->d_slot_meta, 0, (size_t)ctx->num_slots * 32);
    const size_t plan_bytes = (size_t)(ctx->sm_count > 0 ? ctx->sm_count : 148) * PLAN_CACHE_INTS * sizeof(int32_t);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_plan_cache, plan_bytes);
    if (e == cudaSuccess) e = cudaMemset(ctx->d_plan_cache, 0, plan_bytes);
#ifdef SANGAM_TRACE
    if (e == cudaSuccess) { tc_configure(cfg->head_dim); cudaGetLastError(); }   // the trace build's static shared memory can push attn_kernel<128> over the limit
#else
    if (e == cudaSuccess) e = tc_configure(cfg->head_dim);
#endif
    {
        // decode kernels (attn_dec.cuh: dec_occ CTAs per SM; attn_gqa.cuh: CTA pairs) share one split-KV workspace; the
        // flattened weighted unit list must stay below 2^31 coordinates
        const int64_t worst = (int64_t)cfg->max_total_q * cfg->num_kv_heads * ((int64_t)cfg->max_pages_per_req + 64);
        if (e == cudaSuccess && worst < 0x7fffffffLL) {
            if (ctx->G <= dec::NQ) ctx->dec_occ = dec_configure(cfg->head_dim);
            if (ctx->G > 1 && ctx->G <= 128 && (ctx->sm_count & 1) == 0) ctx->gqa_ok = gqa_configure(cfg->head_dim) == cudaSuccess ? 1 : 0;
            cudaGetLastError();
        }
        if (e == cudaSuccess && (ctx->dec_occ > 0 || ctx->gqa_ok)) {
            // partial slots: decode kernel 2 per CTA of 32 rows; pair kernel 2 per CTA of 128 rows
            const size_t o_floats = std::max((size_t)2 * ctx->dec_occ * ctx->sm_count * dec::NQ, ctx->gqa_ok ? (size_t)2 * ctx->sm_count * gqa::BM : 0) * cfg->head_dim;
            e = cudaMalloc(&ctx->d_dec_part_o, o_floats * sizeof(float));
            if (e == cudaSuccess) e = cudaMalloc(&ctx->d_dec_part_ml, o_floats / cfg->head_dim * 2 * sizeof(float));
            // arrival counters: one per work unit (two for the pair kernel): at most Hkv * (rows + requests) units in a batch
            const size_t ncnt = (size_t)2 * cfg->num_kv_heads * ((size_t)cfg->max_total_q + cfg->max_batch);
            if (e == cudaSuccess) e = cudaMalloc(&ctx->d_dec_cnt, ncnt * sizeof(int32_t));
            if (e == cudaSuccess) e = cudaMemset(ctx->d_dec_cnt, 0, ncnt * sizeof(int32_t));
        }
    }
    if (e != cudaSuccess) {
        sangam_destroy(ctx);
        return SANGAM_ERR_CUDA;
    }
    *out = ctx;
    return SANGAM_OK;
}

extern "C" int sangam_destroy(sangam_ctx* ctx) {
    if (!ctx) return SANGAM_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    cudaFree(ctx->d_dec_part_o); cudaFree(ctx->d_dec_part_ml); cudaFree(ctx->d_dec_cnt);
    cudaFree(ctx->d_flags); cudaFree(ctx->d_sched); cudaFree(ctx->d_part_o); cudaFree(ctx->d_part_ml); cudaFree(ctx->d_slot_meta); cudaFree(ctx->d_plan_cache);
    cudaFree(ctx->d_conf_part);
    cudaFree(ctx->s_q); cudaFree(ctx->s_k); cudaFree(ctx->s_v); cudaFree(ctx->s_out); cudaFree(ctx->s_packed);
    cudaFree(ctx->s_slot); cudaFree(ctx->s_bt); cudaFree(ctx->s_cu); cudaFree(ctx->s_ctx);
    delete ctx;
    return SANGAM_OK;
}

extern "C" int sangam_device_status(sangam_ctx* ctx, uint32_t* flags) {
    if (!ctx || !flags) return SANGAM_ERR_INVALID_ARG;
    ON_CTX_DEVICE(ctx);
    CK(cudaDeviceSynchronize());
    CK(cudaMemcpy(flags, ctx->d_flags, sizeof(uint32_t), cudaMemcpyDeviceToHost));
    return SANGAM_OK;
}

extern "C" int sangam_clear_device_status(sangam_ctx* ctx) {
    if (!ctx) return SANGAM_ERR_INVALID_ARG;
    ON_CTX_DEVICE(ctx);
    CK(cudaDeviceSynchronize());
    CK(cudaMemset(ctx->d_flags, 0, sizeof(uint32_t)));
    return SANGAM_OK;
}

extern "C" int sangam_kv_write(sangam_ctx* ctx, const void* k, const void* v, const int32_t* slot_mapping,
                               int32_t num_tokens, void* k_pages, void* v_pages, void* stream) {
    if (!ctx) return SANGAM_ERR_INVALID_ARG;
    if (num_tokens < 0) return fail(ctx, SANGAM_ERR_INVALID_ARG, "kv_write: num_tokens < 0");
    if (num_tokens == 0) return SANGAM_OK;
    if (!k || !v || !slot_mapping || !k_pages || !v_pages) return fail(ctx, SANGAM_ERR_INVALID_ARG, "kv_write: null pointer");
    if (!aligned16(k) || !aligned16(v) || !aligned16(k_pages) || !aligned16(v_pages))
        return fail(ctx, SANGAM_ERR_INVALID_ARG, "kv_write: pointer not 16-byte aligned");
    ON_CTX_DEVICE(ctx);
    const int cpr = ctx->cfg.head_dim / 8;
    const int64_t total = (int64_t)num_tokens * ctx->cfg.num_kv_heads * cpr;
    constexpr int UNROLL = 4;
    int64_t blocks = (total + 256 * UNROLL - 1) / (256 * UNROLL);
    const int64_t cap = (int64_t)ctx->sm_count * 16;
    if (blocks > cap) blocks = cap;
    CK(launch_pdl(kv_write_kernel<UNROLL>, dim3((unsigned)blocks), 256u, 0, (cudaStream_t)stream,
                  (const uint4*)k, (const uint4*)v, slot_mapping, num_tokens, (uint4*)k_pages, (uint4*)v_pages,
                  (int32_t)ctx->cfg.num_kv_heads, (int32_t)cpr, (int32_t)(ctx->cfg.num_pages * SANGAM_PAGE), ctx->d_flags));
    ctx->launches += 1;
    CK(cudaGetLastError());
    return SANGAM_OK;
}


extern "C" int sangam_kv_write_rope(sangam_ctx* ctx, const void* k, const void* v, const int32_t* slot_mapping, const int32_t* positions,
                                    const float* cos_sin, int32_t max_pos, int32_t num_tokens, void* k_pages, void* v_pages, void* stream) {
    if (!ctx) return SANGAM_ERR_INVALID_ARG;
    if (num_tokens < 0 || max_pos <= 0) return fail(ctx, SANGAM_ERR_INVALID_ARG, "kv_write_rope: bad count");
    if (num_tokens == 0) return SANGAM_OK;
    if (!k || !v || !slot_mapping || !positions || !cos_sin || !k_pages || !v_pages) return fail(ctx, SANGAM_ERR_INVALID_ARG, "kv_write_rope: null pointer");
    if (!aligned16(k) || !aligned16(v) || !aligned16(k_pages) || !aligned16(v_pages) || !aligned16(cos_sin))
        return fail(ctx, SANGAM_ERR_INVALID_ARG, "kv_write_rope: pointer not 16-byte aligned");
    ON_CTX_DEVICE(ctx);
    const int64_t total = (int64_t)num_tokens * ctx->cfg.num_kv_heads * (ctx->cfg.head_dim / 16);
    int64_t blocks = (total + 255) / 256;
    const int64_t cap = (int64_t)ctx->sm_count * 16;
    if (blocks > cap) blocks = cap;
    CK(launch_pdl(kv_write_rope_kernel, dim3((unsigned)blocks), 256u, 0, (cudaStream_t)stream, (const uint4*)k, (const uint4*)v, slot_mapping,
                  positions, cos_sin, max_pos, num_tokens, (uint4*)k_pages, (uint4*)v_pages, (int32_t)ctx->cfg.num_kv_heads,
                  (int32_t)ctx->cfg.head_dim, (int32_t)(ctx->cfg.num_pages * SANGAM_PAGE), ctx->d_flags));
    ctx->launches += 1;
    CK(cudaGetLastError());
    return SANGAM_OK;
}

// Slicing of the sampler's first pass.  Work items = (row, vocabulary slice); a grid of persistent blocks (at most the
// CONF_BLOCKS_PER_SM x #SM that are resident at once) takes them round robin.  An item costs a block reduction, so slices are
// as long as they can be while the items still fill the machine: slices = ceil(resident blocks / rows), at most `cap` (and
// 64) per row, never shorter than 4096 logits; the grid is then shrunk so that every block gets the same number of items.
#ifndef SANGAM_CONF_BPS
#define SANGAM_CONF_BPS 5
#endif
constexpr int CONF_BLOCKS_PER_SM = SANGAM_CONF_BPS;          // 288 threads x 38 registers, 41 KB of shared memory: 5 per SM
static void conf_slicing(int sm_count, int num_rows, int vocab, int cap, int* slices_out, int* slice_len_out, unsigned* grid_out) {
    const int resident = CONF_BLOCKS_PER_SM * sm_count;
    int slices = (resident + num_rows - 1) / num_rows;
    const int by_len = (vocab + 4095) / 4096;
    slices = slices > by_len ? by_len : slices;
    slices = slices > cap ? cap : slices;
    slices = slices < 1 ? 1 : (slices > 64 ? 64 : slices);
    const int slice_len = ((vocab + slices - 1) / slices + 7) & ~7;
    slices = (vocab + slice_len - 1) / slice_len;
    const int64_t items = (int64_t)num_rows * slices;
    const int64_t rounds = (items + resident - 1) / resident;
    *slices_out = slices; *slice_len_out = slice_len;
    *grid_out = (unsigned)((items + rounds - 1) / rounds);
}

extern "C" int sangam_confidence_sample(sangam_ctx* ctx, const void* logits, int32_t vocab, const int32_t* masked, const int32_t* cu_rows,
                                        int32_t num_requests, int32_t num_rows, float threshold, int32_t* token, float* conf,
                                        int32_t* unmask, void* stream) {
    if (!ctx) return SANGAM_ERR_INVALID_ARG;
    if (vocab <= 0 || num_requests < 0 || num_rows < 0) return fail(ctx, SANGAM_ERR_INVALID_ARG, "confidence_sample: bad count");
    if (num_requests == 0 || num_rows == 0) return SANGAM_OK;
    if (!logits || !masked || !cu_rows || !token || !conf || !unmask) return fail(ctx, SANGAM_ERR_INVALID_ARG, "confidence_sample: null pointer");
    if (reinterpret_cast<uintptr_t>(logits) & 1u) return fail(ctx, SANGAM_ERR_INVALID_ARG, "confidence_sample: logits not 2-byte aligned");
    ON_CTX_DEVICE(ctx);
    int slices, slice_len;
    unsigned grid;
    conf_slicing(ctx->sm_count, num_rows, vocab, 1 << 30, &slices, &slice_len, &grid);
    const int64_t need = (int64_t)num_rows * slices;
    if (need > ctx->conf_part_cap) {                       // first use / larger batch: (re)allocate (not during graph capture)
        cudaFree(ctx->d_conf_part); ctx->d_conf_part = nullptr; ctx->conf_part_cap = 0;
        const int64_t cap = need > (int64_t)ctx->cfg.max_total_q * 8 ? need : (int64_t)ctx->cfg.max_total_q * 8;
        CK(cudaMalloc(&ctx->d_conf_part, (size_t)cap * sizeof(ConfPartial)));
        ctx->conf_part_cap = cap;
    }
    CK(launch_pdl(confidence_pass1_kernel, dim3(grid), (unsigned)CONF_BLOCK, 0, (cudaStream_t)stream,
                  (const __nv_bfloat16*)logits, vocab, (int32_t)slice_len, (int32_t)slices, (int32_t)need, ctx->d_conf_part));
    CK(launch_pdl(confidence_pass2_kernel, dim3((unsigned)((num_requests + 3) / 4)), 128u, 0, (cudaStream_t)stream,
                  (const ConfPartial*)ctx->d_conf_part, (int32_t)slices, masked, cu_rows, num_requests, threshold, token, conf, unmask));
    ctx->launches += 2;
    CK(cudaGetLastError());
    return SANGAM_OK;
}

static int kv_pages_copy(sangam_ctx* ctx, bool gather, void* k_pages, void* v_pages, void* k_stage, void* v_stage, const int32_t* page_ids,
                         int32_t n, void* stream) {
    if (!ctx) return SANGAM_ERR_INVALID_ARG;
    if (n < 0) return fail(ctx, SANGAM_ERR_INVALID_ARG, "kv_gather/scatter: negative count");
    if (n == 0) return SANGAM_OK;
    if (!k_pages || !v_pages || !k_stage || !v_stage || !page_ids) return fail(ctx, SANGAM_ERR_INVALID_ARG, "kv_gather/scatter: null pointer");
    if (!aligned16(k_pages) || !aligned16(v_pages) || !aligned16(k_stage) || !aligned16(v_stage))
        return fail(ctx, SANGAM_ERR_INVALID_ARG, "kv_gather/scatter: pointer not 16-byte aligned");
    ON_CTX_DEVICE(ctx);
    const int32_t cpp = ctx->cfg.num_kv_heads * SANGAM_PAGE * ctx->cfg.head_dim / 8;
    int64_t blocks = ((int64_t)n * cpp + 255) / 256;
    const int64_t cap = (int64_t)ctx->sm_count * 16;
    if (blocks > cap) blocks = cap;
    if (gather)
        CK(launch_pdl(kv_pages_copy_kernel<true>, dim3((unsigned)blocks), 256u, 0, (cudaStream_t)stream, (uint4*)k_pages, (uint4*)v_pages,
                      (uint4*)k_stage, (uint4*)v_stage, page_ids, n, cpp, (int32_t)ctx->cfg.num_pages, ctx->d_flags));
    else
        CK(launch_pdl(kv_pages_copy_kernel<false>, dim3((unsigned)blocks), 256u, 0, (cudaStream_t)stream, (uint4*)k_pages, (uint4*)v_pages,
                      (uint4*)k_stage, (uint4*)v_stage, page_ids, n, cpp, (int32_t)ctx->cfg.num_pages, ctx->d_flags));
    ctx->launches += 1;
    CK(cudaGetLastError());
    return SANGAM_OK;
}

extern "C" int sangam_kv_gather(sangam_ctx* ctx, const void* k_pages, const void* v_pages, const int32_t* page_ids, int32_t num_pages_listed,
                                void* k_stage, void* v_stage, void* stream) {
    return kv_pages_copy(ctx, true, const_cast<void*>(k_pages), const_cast<void*>(v_pages), k_stage, v_stage, page_ids, num_pages_listed, stream);
}

extern "C" int sangam_kv_scatter(sangam_ctx* ctx, const void* k_stage, const void* v_stage, const int32_t* page_ids, int32_t num_pages_listed,
                                 void* k_pages, void* v_pages, void* stream) {
    return kv_pages_copy(ctx, false, k_pages, v_pages, const_cast<void*>(k_stage), const_cast<void*>(v_stage), page_ids, num_pages_listed, stream);
}

static int check_attn_args(sangam_ctx* ctx, const void* q, const void* k_pages, const void* v_pages,
                           const int32_t* block_table, const int32_t* cu_q_lens, const int32_t* ctx_lens,
                           int32_t batch, int32_t total_q, void* out) {
    if (!ctx) return SANGAM_ERR_INVALID_ARG;
    if (batch < 0 || total_q < 0) return fail(ctx, SANGAM_ERR_INVALID_ARG, "block_attn: negative count");
    if (batch > ctx->cfg.max_batch) return fail(ctx, SANGAM_ERR_WORKSPACE, "block_attn: batch > max_batch");
    if (total_q > ctx->cfg.max_total_q) return fail(ctx, SANGAM_ERR_WORKSPACE, "block_attn: total_q > max_total_q");
    if (batch == 0 || total_q == 0) return 1;  // nothing to do
    if (!q || !k_pages || !v_pages || !block_table || !cu_q_lens || !ctx_lens || !out)
        return fail(ctx, SANGAM_ERR_INVALID_ARG, "block_attn: null pointer");
    if (!aligned16(q) || !aligned16(k_pages) || !aligned16(v_pages) || !aligned16(out))
        return fail(ctx, SANGAM_ERR_INVALID_ARG, "block_attn: pointer not 16-byte aligned");
    return SANGAM_OK;
}

static AttnParams make_params(sangam_ctx* ctx, const void* q, const void* k_pages, const void* v_pages,
                              const int32_t* block_table, const int32_t* cu_q_lens, const int32_t* ctx_lens,
                              int32_t batch, int32_t total_q, float scale, void* out) {
    AttnParams p;
    p.q = (const __nv_bfloat16*)q;
    p.k_pages = (const __nv_bfloat16*)k_pages;
    p.v_pages = (const __nv_bfloat16*)v_pages;
    p.block_table = block_table; p.cu_q_lens = cu_q_lens; p.ctx_lens = ctx_lens;
    p.out = (__nv_bfloat16*)out;
    p.batch = batch; p.total_q = total_q;
    p.Hq = ctx->cfg.num_q_heads; p.Hkv = ctx->cfg.num_kv_heads; p.G = ctx->G;
    p.W = ctx->cfg.max_pages_per_req; p.P = ctx->cfg.num_pages;
    p.tpt = 128 / ctx->G;
    p.tpt2_magic = (uint32_t)(0x100000000ull / (uint64_t)(2 * p.tpt)) + 1u;
    p.scale = scale;
    p.scale_log2 = scale * 1.4426950408889634f;
    p.part_o = ctx->d_part_o; p.part_ml = ctx->d_part_ml; p.num_slots = ctx->num_slots; p.slot_meta = ctx->d_slot_meta;
    p.flags = ctx->d_flags; p.sched = ctx->d_sched; p.plan_cache = ctx->d_plan_cache;
    return p;
}

extern "C" int sangam_block_attn_simt(sangam_ctx* ctx, const void* q, const void* k_pages, const void* v_pages,
                                      const int32_t* block_table, const int32_t* cu_q_lens, const int32_t* ctx_lens,
                                      int32_t batch, int32_t total_q, float scale, void* out, void* stream) {
    int rc = check_attn_args(ctx, q, k_pages, v_pages, block_table, cu_q_lens, ctx_lens, batch, total_q, out);
    if (rc != SANGAM_OK) return rc > 0 ? SANGAM_OK : rc;
    ON_CTX_DEVICE(ctx);
    AttnParams p = make_params(ctx, q, k_pages, v_pages, block_table, cu_q_lens, ctx_lens, batch, total_q, scale, out);
    const int64_t warps = (int64_t)total_q * p.Hq;
    const unsigned blocks = (unsigned)((warps + 7) / 8);
    if (ctx->cfg.head_dim == 128) attn_simt_kernel<128><<<blocks, 256, 0, (cudaStream_t)stream>>>(p);
    else attn_simt_kernel<64><<<blocks, 256, 0, (cudaStream_t)stream>>>(p);
    ctx->launches += 1;
    CK(cudaGetLastError());
    return SANGAM_OK;
}

extern "C" int sangam_block_attn(sangam_ctx* ctx, const void* q, const void* k_pages, const void* v_pages,
                                 const int32_t* block_table, const int32_t* cu_q_lens, const int32_t* ctx_lens,
                                 int32_t batch, int32_t total_q, float scale, void* out, void* stream) {
    int rc = check_attn_args(ctx, q, k_pages, v_pages, block_table, cu_q_lens, ctx_lens, batch, total_q, out);
    if (rc != SANGAM_OK) return rc > 0 ? SANGAM_OK : rc;
    ON_CTX_DEVICE(ctx);
    const sangam_config& c = ctx->cfg;
    // tensor maps of this call's pools and q buffer (host-side cache, least recently used entry replaced)
    MapCacheKV* kv = nullptr;
    MapCacheQ* qm = nullptr;
    ++ctx->map_tick;
    for (int i = 0; i < MAP_CACHE; ++i) {
        if (ctx->kv_cache[i].tick && ctx->kv_cache[i].k == k_pages && ctx->kv_cache[i].v == v_pages) kv = &ctx->kv_cache[i];
        if (ctx->q_cache[i].tick && ctx->q_cache[i].q == q && ctx->q_cache[i].rows == total_q) qm = &ctx->q_cache[i];
    }
    if (!kv) {
        kv = &ctx->kv_cache[0];
        for (int i = 1; i < MAP_CACHE; ++i) if (ctx->kv_cache[i].tick < kv->tick) kv = &ctx->kv_cache[i];
        kv->tick = 0;
        if (tmap_encode_pool(&kv->mk, k_pages, c.num_pages, c.num_kv_heads, c.head_dim) != 0 ||
            tmap_encode_pool(&kv->mv, v_pages, c.num_pages, c.num_kv_heads, c.head_dim) != 0)
            return fail(ctx, SANGAM_ERR_CUDA, "block_attn: cuTensorMapEncodeTiled failed");
        kv->k = k_pages; kv->v = v_pages;
    }
    kv->tick = ctx->map_tick;
    if (!qm) {
        qm = &ctx->q_cache[0];
        for (int i = 1; i < MAP_CACHE; ++i) if (ctx->q_cache[i].tick < qm->tick) qm = &ctx->q_cache[i];
        qm->tick = 0;
        if (tmap_encode_q(&qm->main, q, total_q, c.num_q_heads, c.head_dim, ctx->G, 128 / ctx->G) != 0 ||
            (ctx->dec_occ > 0 && tmap_encode_q(&qm->dec, q, total_q, c.num_q_heads, c.head_dim, ctx->G, dec::NQ / ctx->G) != 0))
            return fail(ctx, SANGAM_ERR_CUDA, "block_attn: cuTensorMapEncodeTiled (q) failed");
        qm->q = q; qm->rows = total_q;
    }
    qm->tick = ctx->map_tick;

    // Decode-shaped batches (on average at most one 32-row unit per request and kv head: block decodes)
    // go to the swapped-operand decode kernel; prefill / refresh / hybrid batches to the two-stream kernel.  Both
    // compute the same function for any batch; the choice only affects speed.  Lengths live on the device, so the
    // host decides on the counts it knows: total_q and batch.
    bool use_dec = ctx->dec_occ > 0 && (int64_t)total_q * ctx->G <= (int64_t)dec::NQ * batch;
    // GQA models: block decodes of up to two 128-row q tiles per kv head fit the CTA-pair kernel (attn_gqa.cuh).  It is
    // measured slower than the two-stream kernel on the Dream-like shapes (config 3: 72.7 us against 66.2 us), so AUTO
    // does not choose it; SANGAM_DISPATCH_GQA_PAIR selects it.
    const int tpt = 128 / ctx->G;
    bool use_gqa = false;
    if (ctx->dispatch == SANGAM_DISPATCH_PREFILL) { use_dec = false; use_gqa = false; }
    if (ctx->dispatch == SANGAM_DISPATCH_DECODE) {
        if (ctx->dec_occ <= 0) return fail(ctx, SANGAM_ERR_UNSUPPORTED, "block_attn: the decode kernel is not available for this geometry");
        use_dec = true; use_gqa = false;
    }
    if (ctx->dispatch == SANGAM_DISPATCH_GQA_PAIR) {
        if (!ctx->gqa_ok) return fail(ctx, SANGAM_ERR_UNSUPPORTED, "block_attn: the GQA pair kernel is not available for this geometry");
        use_gqa = true; use_dec = false;
    }
    if (use_dec || use_gqa) {
        DecParams d = {};
        d.block_table = block_table; d.cu_q_lens = cu_q_lens; d.ctx_lens = ctx_lens;
        d.out = (__nv_bfloat16*)out;
        d.q = (const __nv_bfloat16*)q;
        d.batch = batch; d.total_q = total_q;
        d.Hq = c.num_q_heads; d.Hkv = c.num_kv_heads; d.G = ctx->G; d.W = c.max_pages_per_req; d.P = c.num_pages;
        d.tpt = tpt;
        d.tq = use_gqa ? 2 * tpt : dec::NQ / ctx->G;
        d.tq_magic = (uint32_t)(0x100000000ull / (uint64_t)d.tq) + 1u;
        d.g_magic = (uint32_t)(0x100000000ull / (uint64_t)ctx->G) + 1u;
        d.scale_log2 = scale * 1.4426950408889634f;
#ifdef SANGAM_TRACE
        { unsigned int v = 0; cudaMemcpyFromSymbol(&v, g_trace_cta, sizeof v); d.trace_cta = (int)v; }
#endif
        d.part_o = ctx->d_dec_part_o; d.part_ml = ctx->d_dec_part_ml; d.unit_cnt = ctx->d_dec_cnt;
        d.min_w = use_gqa ? gqa::MIN_W : dec::MIN_W; d.ov = use_gqa ? gqa::OV : dec::OV;
#ifdef SANGAM_TUNING_ENV
        if (const char* e_ = getenv("SANGAM_DEC_OV")) d.ov = atoi(e_);
        if (const char* e_ = getenv("SANGAM_DEC_MINW")) d.min_w = atoi(e_);
#endif
        d.flags = ctx->d_flags;
        cudaError_t e = use_gqa ? gqa_launch(d, kv->mk, kv->mv, qm->main, c.head_dim, ctx->sm_count, (cudaStream_t)stream)
                                : dec_launch(d, kv->mk, kv->mv, qm->dec, c.head_dim, ctx->dec_occ * ctx->sm_count, (cudaStream_t)stream);
        if (e != cudaSuccess) return cuda_fail(ctx, e, use_gqa ? "block_attn launch (GQA pair kernel)" : "block_attn launch (decode kernel)");
        ctx->launches += 1;
        ctx->last_kernel = use_gqa ? SANGAM_DISPATCH_GQA_PAIR : SANGAM_DISPATCH_DECODE;
        return SANGAM_OK;
    }
    AttnParams p = make_params(ctx, q, k_pages, v_pages, block_table, cu_q_lens, ctx_lens, batch, total_q, scale, out);
    ctx->last_kernel = SANGAM_DISPATCH_PREFILL;
    int launched = 0;
    cudaError_t e = tc_launch(p, kv->mk, kv->mv, qm->main, c.head_dim, ctx->sm_count, (cudaStream_t)stream, &launched);
    ctx->launches += launched;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "block_attn launch");
    return SANGAM_OK;
}

extern "C" int32_t sangam_query(const sangam_ctx* ctx, int32_t what) {
    if (!ctx) return -1;
    switch (what) {
        case SANGAM_QUERY_SM_COUNT: return ctx->sm_count;
        case SANGAM_QUERY_DECODE_CTAS_PER_SM: return ctx->dec_occ;
        case SANGAM_QUERY_DISPATCH: return ctx->dispatch;
        case SANGAM_QUERY_GQA_PAIR_KERNEL: return ctx->gqa_ok;
        case SANGAM_QUERY_LAST_KERNEL: return ctx->last_kernel;
        default: return -1;
    }
}

extern "C" int sangam_set_dispatch(sangam_ctx* ctx, int32_t mode) {
    if (!ctx) return SANGAM_ERR_INVALID_ARG;
    if (mode != SANGAM_DISPATCH_AUTO && mode != SANGAM_DISPATCH_PREFILL && mode != SANGAM_DISPATCH_DECODE && mode != SANGAM_DISPATCH_GQA_PAIR)
        return fail(ctx, SANGAM_ERR_INVALID_ARG, "set_dispatch: unknown mode");
    if (mode == SANGAM_DISPATCH_GQA_PAIR && !ctx->gqa_ok)
        return fail(ctx, SANGAM_ERR_UNSUPPORTED, "set_dispatch: the GQA pair kernel is not available for this geometry");
    if (mode == SANGAM_DISPATCH_DECODE && ctx->dec_occ <= 0)
        return fail(ctx, SANGAM_ERR_UNSUPPORTED, "set_dispatch: the decode kernel is not available for this geometry");
    ctx->dispatch = mode;
    return SANGAM_OK;
}

static int ensure_staging(sangam_ctx* ctx) {
    if (ctx->s_q) return SANGAM_OK;
    if (ctx->s_out) { cudaFree(ctx->s_out); ctx->s_out = nullptr; }
    const sangam_config& c = ctx->cfg;
    const size_t qb = (size_t)c.max_total_q * c.num_q_heads * c.head_dim * 2;
    const size_t kb = (size_t)c.max_total_q * c.num_kv_heads * c.head_dim * 2;
    CK(cudaMalloc(&ctx->s_q, qb)); CK(cudaMalloc(&ctx->s_out, qb));
    CK(cudaMalloc(&ctx->s_k, kb)); CK(cudaMalloc(&ctx->s_v, kb));
    CK(cudaMalloc(&ctx->s_slot, (size_t)c.max_total_q * 4));
    CK(cudaMalloc(&ctx->s_bt, (size_t)c.max_batch * c.max_pages_per_req * 4));
    CK(cudaMalloc(&ctx->s_cu, (size_t)(c.max_batch + 1) * 4));
    CK(cudaMalloc(&ctx->s_ctx, (size_t)c.max_batch * 4));
    return SANGAM_OK;
}

extern "C" int sangam_iteration_host(sangam_ctx* ctx, const void* q_host, const void* k_host, const void* v_host,
                                     const int32_t* slot_mapping_host, int32_t num_tokens,
                                     void* k_pages, void* v_pages,
                                     const int32_t* block_table_host, const int32_t* cu_q_lens_host,
                                     const int32_t* ctx_lens_host, int32_t batch, int32_t total_q,
                                     float scale, void* out_host, void* stream) {
    if (!ctx) return SANGAM_ERR_INVALID_ARG;
    if (batch < 0 || total_q < 0 || num_tokens < 0) return fail(ctx, SANGAM_ERR_INVALID_ARG, "iteration_host: negative count");
    if (batch > ctx->cfg.max_batch || total_q > ctx->cfg.max_total_q || num_tokens > ctx->cfg.max_total_q)
        return fail(ctx, SANGAM_ERR_WORKSPACE, "iteration_host: batch / total_q / num_tokens above the ctx maxima");
    if (!q_host || !out_host || !block_table_host || !cu_q_lens_host || !ctx_lens_host || (num_tokens && (!k_host || !v_host || !slot_mapping_host)))
        return fail(ctx, SANGAM_ERR_INVALID_ARG, "iteration_host: null pointer");
    ON_CTX_DEVICE(ctx);
    int rc = ensure_staging(ctx);
    if (rc != SANGAM_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const sangam_config& c = ctx->cfg;
    const size_t qb = (size_t)total_q * c.num_q_heads * c.head_dim * 2;
    const size_t kb = (size_t)num_tokens * c.num_kv_heads * c.head_dim * 2;
    CK(cudaMemcpyAsync(ctx->s_q, q_host, qb, cudaMemcpyHostToDevice, st));
    if (num_tokens) {
        CK(cudaMemcpyAsync(ctx->s_k, k_host, kb, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->s_v, v_host, kb, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->s_slot, slot_mapping_host, (size_t)num_tokens * 4, cudaMemcpyHostToDevice, st));
    }
    CK(cudaMemcpyAsync(ctx->s_bt, block_table_host, (size_t)batch * c.max_pages_per_req * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->s_cu, cu_q_lens_host, (size_t)(batch + 1) * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->s_ctx, ctx_lens_host, (size_t)batch * 4, cudaMemcpyHostToDevice, st));
    rc = sangam_kv_write(ctx, ctx->s_k, ctx->s_v, ctx->s_slot, num_tokens, k_pages, v_pages, stream);
    if (rc != SANGAM_OK) return rc;
    rc = sangam_block_attn(ctx, ctx->s_q, k_pages, v_pages, ctx->s_bt, ctx->s_cu, ctx->s_ctx, batch, total_q, scale, ctx->s_out, stream);
    if (rc != SANGAM_OK) return rc;
    CK(cudaMemcpyAsync(out_host, ctx->s_out, qb, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return SANGAM_OK;
}


// Layout of the packed host buffer of sangam_iteration_packed: q | k | v | slot_mapping | block_table | cu_q_lens | ctx_lens,
// each part starting on a 256-byte boundary.  offsets[0..6] = byte offset of each part, offsets[7] = total bytes.
static void packed_layout(const sangam_config& c, int32_t batch, int32_t total_q, int32_t num_tokens, int64_t offsets[8]) {
    const int64_t sizes[7] = {(int64_t)total_q * c.num_q_heads * c.head_dim * 2, (int64_t)num_tokens * c.num_kv_heads * c.head_dim * 2,
                              (int64_t)num_tokens * c.num_kv_heads * c.head_dim * 2, (int64_t)num_tokens * 4,
                              (int64_t)batch * c.max_pages_per_req * 4, (int64_t)(batch + 1) * 4, (int64_t)batch * 4};
    int64_t off = 0;
    for (int i = 0; i < 7; ++i) { offsets[i] = off; off = (off + sizes[i] + 255) & ~(int64_t)255; }
    offsets[7] = off;
}

extern "C" int sangam_packed_layout(const sangam_ctx* ctx, int32_t batch, int32_t total_q, int32_t num_tokens, int64_t* offsets8) {
    if (!ctx || !offsets8 || batch < 0 || total_q < 0 || num_tokens < 0) return SANGAM_ERR_INVALID_ARG;
    packed_layout(ctx->cfg, batch, total_q, num_tokens, offsets8);
    return SANGAM_OK;
}

extern "C" int sangam_iteration_packed(sangam_ctx* ctx, const void* packed_host, int32_t num_tokens, void* k_pages, void* v_pages,
                                       int32_t batch, int32_t total_q, float scale, void* out_host, void* stream) {
    if (!ctx) return SANGAM_ERR_INVALID_ARG;
    if (batch < 0 || total_q < 0 || num_tokens < 0) return fail(ctx, SANGAM_ERR_INVALID_ARG, "iteration_packed: negative count");
    if (batch > ctx->cfg.max_batch || total_q > ctx->cfg.max_total_q || num_tokens > ctx->cfg.max_total_q)
        return fail(ctx, SANGAM_ERR_WORKSPACE, "iteration_packed: batch / total_q / num_tokens above the ctx maxima");
    if (!packed_host || !out_host || !k_pages || !v_pages) return fail(ctx, SANGAM_ERR_INVALID_ARG, "iteration_packed: null pointer");
    ON_CTX_DEVICE(ctx);
    int64_t off[8];
    packed_layout(ctx->cfg, batch, total_q, num_tokens, off);
    if (!ctx->s_packed || ctx->s_packed_bytes < off[7]) {        // grows to the largest request seen (first call: allocation)
        int64_t cap[8];
        packed_layout(ctx->cfg, ctx->cfg.max_batch, ctx->cfg.max_total_q, ctx->cfg.max_total_q, cap);
        cudaFree(ctx->s_packed); ctx->s_packed = nullptr;
        cudaFree(ctx->s_out); ctx->s_out = nullptr;
        CK(cudaMalloc(&ctx->s_packed, (size_t)cap[7]));
        ctx->s_packed_bytes = cap[7];
        CK(cudaMalloc(&ctx->s_out, (size_t)ctx->cfg.max_total_q * ctx->cfg.num_q_heads * ctx->cfg.head_dim * 2));
    }
    cudaStream_t st = (cudaStream_t)stream;
    char* d = static_cast<char*>(ctx->s_packed);
    CK(cudaMemcpyAsync(d, packed_host, (size_t)off[7], cudaMemcpyHostToDevice, st));          // ONE host-to-device copy
    int rc = sangam_kv_write(ctx, d + off[1], d + off[2], reinterpret_cast<const int32_t*>(d + off[3]), num_tokens, k_pages, v_pages, stream);
    if (rc != SANGAM_OK) return rc;
    rc = sangam_block_attn(ctx, d + off[0], k_pages, v_pages, reinterpret_cast<const int32_t*>(d + off[4]),
                           reinterpret_cast<const int32_t*>(d + off[5]), reinterpret_cast<const int32_t*>(d + off[6]), batch, total_q, scale,
                           ctx->s_out, stream);
    if (rc != SANGAM_OK) return rc;
    CK(cudaMemcpyAsync(out_host, ctx->s_out, (size_t)total_q * ctx->cfg.num_q_heads * ctx->cfg.head_dim * 2, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return SANGAM_OK;
}

#ifdef SANGAM_DEBUG_ITEM
extern "C" int sangam_debug_bad_item(int* out16) {
    cudaDeviceSynchronize();
    return cudaMemcpyFromSymbol(out16, g_bad_item, 64) == cudaSuccess ? 0 : -4;
}
#endif
#ifdef SANGAM_WAIT_TABLE
// debug builds only (not part of include/sangam.h): which barrier the first watchdog timeout hit
extern "C" int sangam_debug_timeout_info(unsigned int* out20) {
    cudaDeviceSynchronize();
    return cudaMemcpyFromSymbol(out20, ptx::g_timeout_info, 80) == cudaSuccess ? 0 : -4;
}
#endif


// ---------------------------------------------------------------------------------------------------------------
// sangam_confidence_sample_static: the confidence sampler for callers that must not allocate (CUDA-graph capture,
// tight serving loops, harnesses that forbid cudaMalloc).  No ctx, no cudaMalloc / cudaFree, no allocating library
// call: the per-(row, vocabulary slice) partials of pass 1 live in the file-scope device array below, which every
// GPU that loads the library holds until the process exits (SANGAM_STATIC_SAMPLER_MAX_PARTIALS * 16 B = 1 MiB).
// In host code `g_static_conf_part` is only a host-side stand-in for the symbol, NOT a device address: the device
// address is taken once per device, with that device current, by cudaGetSymbolAddress, and that pointer is what the
// kernels receive.
// Every call on a device shares the one array and finds the previous call's contents in it.  Nothing has to start
// at zero: pass 1 writes every (row, slice) entry that pass 2 of the same call reads, and no entry outside
// [0, num_rows * slices) is read.  Two calls whose kernels overlap on the GPU (different streams, or graphs
// launched concurrently) race on the array: callers serialise them (same stream, or an event between them).
// ---------------------------------------------------------------------------------------------------------------
static __device__ __align__(256) ConfPartial g_static_conf_part[SANGAM_STATIC_SAMPLER_MAX_PARTIALS];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
struct StaticSamplerDev {
    ConfPartial* part;       // device address of g_static_conf_part on this device
    int sm_count;
    bool ready;
};
StaticSamplerDev g_static_dev[STATIC_MAX_DEVICES];
std::mutex g_static_mu;
thread_local char g_static_err[256] = "";

int static_fail(int code, const char* msg, const char* detail = "") {
    snprintf(g_static_err, sizeof g_static_err, "%s%s", msg, detail);
    return code;
}
}  // namespace

extern "C" const char* sangam_static_last_error(void) { return g_static_err; }

extern "C" int sangam_confidence_sample_static(const void* logits, int32_t vocab, const int32_t* masked, const int32_t* cu_rows,
                                               int32_t num_requests, int32_t num_rows, float threshold, int32_t* token, float* conf,
                                               int32_t* unmask, void* stream) {
    if (vocab <= 0 || num_requests < 0 || num_rows < 0) return static_fail(SANGAM_ERR_INVALID_ARG, "confidence_sample_static: bad count");
    if (num_rows > SANGAM_STATIC_SAMPLER_MAX_ROWS)
        return static_fail(SANGAM_ERR_WORKSPACE, "confidence_sample_static: num_rows above SANGAM_STATIC_SAMPLER_MAX_ROWS (the static scratch "
                                                 "array holds no more; use sangam_confidence_sample)");
    if (num_requests == 0 || num_rows == 0) return SANGAM_OK;
    if (!logits || !masked || !cu_rows || !token || !conf || !unmask) return static_fail(SANGAM_ERR_INVALID_ARG, "confidence_sample_static: null pointer");
    if (reinterpret_cast<uintptr_t>(logits) & 1u) return static_fail(SANGAM_ERR_INVALID_ARG, "confidence_sample_static: logits not 2-byte aligned");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_fail(SANGAM_ERR_CUDA, "confidence_sample_static: cudaGetDevice: ", cudaGetErrorString(e));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return static_fail(SANGAM_ERR_UNSUPPORTED, "confidence_sample_static: device ordinal above 63");
    StaticSamplerDev d;
    {
        // set-up, once per device, with that device current (it is: the call runs on the caller's current device)
        std::lock_guard<std::mutex> lock(g_static_mu);
        if (!g_static_dev[dev].ready) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_static_conf_part);
            if (e != cudaSuccess || !p) return static_fail(SANGAM_ERR_CUDA, "confidence_sample_static: cudaGetSymbolAddress: ", cudaGetErrorString(e));
            int sms = 0;
            e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            if (e != cudaSuccess || sms <= 0) return static_fail(SANGAM_ERR_CUDA, "confidence_sample_static: cudaDeviceGetAttribute: ", cudaGetErrorString(e));
            g_static_dev[dev].part = static_cast<ConfPartial*>(p);
            g_static_dev[dev].sm_count = sms;
            g_static_dev[dev].ready = true;
        }
        d = g_static_dev[dev];
    }
    // same slicing rule as sangam_confidence_sample, capped by the array: num_rows * slices <= MAX_PARTIALS
    int slices, slice_len;
    unsigned grid;
    conf_slicing(d.sm_count, num_rows, vocab, SANGAM_STATIC_SAMPLER_MAX_PARTIALS / num_rows, &slices, &slice_len, &grid);
    if ((int64_t)num_rows * slices > SANGAM_STATIC_SAMPLER_MAX_PARTIALS)
        return static_fail(SANGAM_ERR_WORKSPACE, "confidence_sample_static: partials exceed the static scratch array");
    e = launch_pdl(confidence_pass1_kernel, dim3(grid), (unsigned)CONF_BLOCK, 0, (cudaStream_t)stream,
                   (const __nv_bfloat16*)logits, vocab, (int32_t)slice_len, (int32_t)slices, (int32_t)(num_rows * slices), d.part);
    if (e != cudaSuccess) return static_fail(SANGAM_ERR_CUDA, "confidence_sample_static: launch of pass 1: ", cudaGetErrorString(e));
    e = launch_pdl(confidence_pass2_kernel, dim3((unsigned)((num_requests + 3) / 4)), 128u, 0, (cudaStream_t)stream,
                   (const ConfPartial*)d.part, (int32_t)slices, masked, cu_rows, num_requests, threshold, token, conf, unmask);
    if (e != cudaSuccess) return static_fail(SANGAM_ERR_CUDA, "confidence_sample_static: launch of pass 2: ", cudaGetErrorString(e));
    e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(SANGAM_ERR_CUDA, "confidence_sample_static: ", cudaGetErrorString(e));
    g_static_err[0] = 0;
    return SANGAM_OK;
}
