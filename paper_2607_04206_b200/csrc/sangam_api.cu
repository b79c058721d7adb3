// sangam_api.cu -- the C ABI of include/sangam.h: argument checks, workspace, kernel launches.
// Every step of the path runs in the kernels of this directory; there is no CPU fallback.
#include "../../include/sangam.h"

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "attn_simt.cuh"
#include "attn_tc.cuh"
#include "common.cuh"
#include "kv_write.cuh"

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
    // tensor maps for the K / V pools, re-encoded when the pool pointer changes
    TcMaps maps;
    const void* maps_k;
    const void* maps_v;
    const void* maps_q;
    int32_t maps_q_rows;
    // staging for sangam_iteration_host (allocated on first use)
    void *s_q, *s_k, *s_v, *s_out;
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
    sangam_ctx* ctx = new (std::nothrow) sangam_ctx();
    if (!ctx) return SANGAM_ERR_WORKSPACE;
    memset(ctx, 0, sizeof *ctx);
    ctx->cfg = *cfg;
    ctx->G = cfg->num_q_heads / cfg->num_kv_heads;
    cudaError_t e = cudaSetDevice(cfg->device);
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
    if (e == cudaSuccess) e = tc_configure(cfg->head_dim);
    if (e != cudaSuccess) {
        sangam_destroy(ctx);
        return SANGAM_ERR_CUDA;
    }
    *out = ctx;
    return SANGAM_OK;
}

extern "C" int sangam_destroy(sangam_ctx* ctx) {
    if (!ctx) return SANGAM_ERR_INVALID_ARG;
    cudaFree(ctx->d_flags); cudaFree(ctx->d_sched); cudaFree(ctx->d_part_o); cudaFree(ctx->d_part_ml); cudaFree(ctx->d_slot_meta); cudaFree(ctx->d_plan_cache);
    cudaFree(ctx->s_q); cudaFree(ctx->s_k); cudaFree(ctx->s_v); cudaFree(ctx->s_out);
    cudaFree(ctx->s_slot); cudaFree(ctx->s_bt); cudaFree(ctx->s_cu); cudaFree(ctx->s_ctx);
    delete ctx;
    return SANGAM_OK;
}

extern "C" int sangam_device_status(sangam_ctx* ctx, uint32_t* flags) {
    if (!ctx || !flags) return SANGAM_ERR_INVALID_ARG;
    CK(cudaDeviceSynchronize());
    CK(cudaMemcpy(flags, ctx->d_flags, sizeof(uint32_t), cudaMemcpyDeviceToHost));
    return SANGAM_OK;
}

extern "C" int sangam_clear_device_status(sangam_ctx* ctx) {
    if (!ctx) return SANGAM_ERR_INVALID_ARG;
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
    if (ctx->maps_k != k_pages || ctx->maps_v != v_pages) {   // per-layer pools: re-encode on pointer change (host only)
        if (tc_encode_maps(&ctx->maps, k_pages, v_pages, ctx->cfg.num_pages, ctx->cfg.num_kv_heads, ctx->cfg.head_dim) != 0)
            return fail(ctx, SANGAM_ERR_CUDA, "block_attn: cuTensorMapEncodeTiled failed");
        ctx->maps_k = k_pages; ctx->maps_v = v_pages;
    }
    if (ctx->maps_q != q || ctx->maps_q_rows != total_q) {
        if (tc_encode_q(&ctx->maps, q, total_q, ctx->cfg.num_q_heads, ctx->cfg.head_dim, ctx->G, 128 / ctx->G) != 0)
            return fail(ctx, SANGAM_ERR_CUDA, "block_attn: cuTensorMapEncodeTiled (q) failed");
        ctx->maps_q = q; ctx->maps_q_rows = total_q;
    }
    AttnParams p = make_params(ctx, q, k_pages, v_pages, block_table, cu_q_lens, ctx_lens, batch, total_q, scale, out);
    int launched = 0;
    cudaError_t e = tc_launch(p, ctx->maps, ctx->cfg.head_dim, ctx->sm_count, (cudaStream_t)stream, &launched);
    ctx->launches += launched;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "block_attn launch");
    return SANGAM_OK;
}

static int ensure_staging(sangam_ctx* ctx) {
    if (ctx->s_q) return SANGAM_OK;
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

#ifdef SANGAM_DEBUG_ITEM
extern "C" int sangam_debug_bad_item(int* out16) {
    cudaDeviceSynchronize();
    return cudaMemcpyFromSymbol(out16, g_bad_item, 64) == cudaSuccess ? 0 : -4;
}
#endif
// internal diagnostic (not part of include/sangam.h): which barrier the first watchdog timeout hit
extern "C" int sangam_debug_timeout_info(unsigned int* out20) {
    cudaDeviceSynchronize();
    return cudaMemcpyFromSymbol(out20, ptx::g_timeout_info, 80) == cudaSuccess ? 0 : -4;
}

#ifdef SANGAM_TRACE
extern "C" int sangam_trace_cta_times(unsigned long long* host_buf) {
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(host_buf, g_cta_times, sizeof(unsigned long long) * 512);
    return 0;
}
extern "C" int sangam_trace_set_cta(int cta) {
    unsigned int v = (unsigned int)cta, z[16] = {0};
    cudaDeviceSynchronize();
    cudaMemcpyToSymbol(g_trace_cta, &v, sizeof v);
    cudaMemcpyToSymbol(g_trace_n, z, sizeof z);
    return 0;
}
// debug builds only: copy the event trace of the recording CTA (per-warp rings, concatenated) to the host
extern "C" int sangam_trace_read(unsigned long long* host_buf, int cap) {
    unsigned int n[16];
    static unsigned long long tmp[16 * SANGAM_TRACE_CAP];
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(n, g_trace_n, sizeof n);
    cudaMemcpyFromSymbol(tmp, g_trace, sizeof tmp);
    int k = 0;
    for (int w = 0; w < 16; ++w)
        for (unsigned i = 0; i < n[w] && i < SANGAM_TRACE_CAP && k < cap; ++i) host_buf[k++] = tmp[w * SANGAM_TRACE_CAP + i];
    return k;
}
#endif
