/*
 * sangam.h -- C ABI of the B200-native hot path of one cached-dLLM serving iteration
 * (arxiv/paper_2607_04206, "Sangam").  Plain pointers and sizes; no torch types.
 *
 * The two operations follow the paper's statement of the problem:
 *   - sangam_kv_write:  store freshly computed K/V rows into the paged KV cache
 *       (PagedAttention, page size 16: PAPER.md:258; the cache is recomputed at
 *        every block boundary and the current block's K/V change every step: PAPER.md:77).
 *   - sangam_block_attn: batched, varlen, NON-CAUSAL attention of each request's query rows over
 *       that request's paged context ("the causal mask is dropped so tokens attend
 *       bidirectionally over the full prompt-and-response"; a decode "contributes an
 *       entire response block while attending over the prompt and response context", PAPER.md:33;
 *       a prefill is one indivisible pass over prompt+response; a hybrid iteration
 *       mixes decodes and whole prefills in one microbatch, Alg. 1).
 *
 * Layouts (all device memory unless a function says "host"; every pointer 16-byte aligned):
 *   q, out        bf16 [total_q][num_q_heads][head_dim], contiguous, rows of request r are
 *                 cu_q_lens[r] .. cu_q_lens[r+1]-1
 *   k, v          bf16 [num_tokens][num_kv_heads][head_dim], contiguous (token-major)
 *   k_pages,      bf16 [num_pages][num_kv_heads][16][head_dim]  (head-major pages: one
 *   v_pages         (page, kv head) is one contiguous 16*head_dim*2-byte block)
 *   block_table   int32 [batch][max_pages_per_req] row-major; entry i of row r is the page holding
 *                 context positions 16*i .. 16*i+15 of request r.  Entries at or past
 *                 ceil(ctx_lens[r]/16) are never read and may hold anything.
 *   cu_q_lens     int32 [batch+1], prefix sums of query rows, cu_q_lens[0] = 0
 *   ctx_lens      int32 [batch], context length c_r of each request
 *   slot_mapping  int32 [num_tokens]; slot = page*16 + offset; slot < 0 skips the row
 * q head h reads kv head h / (num_q_heads / num_kv_heads).  Slots past ctx_lens[r] inside the last
 * page, and pages no request lists, may hold any bits (NaN included); results never depend on them.
 *
 * Ownership: the caller owns every tensor and the stream.  The library owns only the workspace
 * allocated in sangam_create.  Both calls only enqueue work on `stream`: no host sync, no
 * allocation, no host read of a device array.  All lengths are read on the device, so a captured
 * CUDA graph replays correctly after the caller rewrites q/k/v/metadata in the same buffers;
 * host-side arguments (batch, num_tokens, pointers, scale) are baked into the capture.
 * Padding (q_r = 0, slot = -1) lets a larger capture serve a smaller batch.
 *
 * Errors: every call returns 0 on success or a negative sangam_status; nothing throws or aborts.
 * sangam_last_error gives a message for the last failing call on that ctx.  Conditions only the
 * device can see never fault; each raises a sticky flag, readable with sangam_device_status after
 * a stream sync, and is handled the same way by every kernel of the library:
 *   - a page id outside [0, num_pages) among the first ceil(ctx_len/16) block-table entries
 *     (SANGAM_DEV_BAD_PAGE): that page's 16 positions are read as K = V = 0 (logit 0, value 0);
 *     the request is still computed, other requests are unaffected;
 *   - a context needing more than max_pages_per_req pages (SANGAM_DEV_CTX_TOO_LONG): the request
 *     is treated as ctx_len = 0, i.e. its output rows are zeros;
 *   - a slot >= num_pages*16 in sangam_kv_write (SANGAM_DEV_BAD_SLOT): that row is not written.
 * Negative ctx_lens are read as 0, decreasing cu_q_lens as an empty request (no flag).
 * One ctx per stream; calls on one ctx are not re-entrant.
 */
#ifndef SANGAM_H_
#define SANGAM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sangam_ctx sangam_ctx;

typedef enum {
    SANGAM_OK = 0,
    SANGAM_ERR_INVALID_ARG = -1,      /* null pointer, misalignment, count out of range */
    SANGAM_ERR_UNSUPPORTED = -2,      /* geometry the kernels are not compiled for */
    SANGAM_ERR_WORKSPACE = -3,        /* batch / total_q above what sangam_create sized */
    SANGAM_ERR_CUDA = -4              /* CUDA runtime / driver error; see sangam_last_error */
} sangam_status;

/* sticky device-side flags (sangam_device_status) */
#define SANGAM_DEV_BAD_SLOT   1u      /* kv_write: slot >= num_pages*16, row skipped */
#define SANGAM_DEV_BAD_PAGE   2u      /* block_attn: page id out of [0,num_pages): the page reads as K = V = 0 */
#define SANGAM_DEV_CTX_TOO_LONG 4u    /* block_attn: ctx_len needs more than max_pages_per_req pages: rows are zeros */
#define SANGAM_DEV_TIMEOUT    8u      /* an in-kernel barrier wait gave up (internal error) */
#define SANGAM_DEV_BAD_POSITION 32u   /* kv_write_rope: position outside [0, max_pos), row skipped */
#define SANGAM_DEV_INTERNAL  16u      /* an internal bounds guard tripped; the access was skipped (internal error) */

typedef struct {
    int32_t num_q_heads;        /* Hq */
    int32_t num_kv_heads;       /* Hkv, Hq % Hkv == 0 */
    int32_t head_dim;           /* 64 or 128 */
    int32_t page_size;          /* must be 16 */
    int32_t num_pages;          /* P: capacity of each of the K and V pools */
    int32_t max_batch;          /* largest `batch` of any call */
    int32_t max_total_q;        /* largest total number of query rows of any call */
    int32_t max_pages_per_req;  /* W: row width of block_table */
    int32_t device;             /* CUDA device ordinal */
} sangam_config;

/* Allocates the workspace once (split-KV partials, host staging for the *_host call). */
int sangam_create(const sangam_config* cfg, sangam_ctx** out);
int sangam_destroy(sangam_ctx* ctx);

/*
 * KV write (step a2): for every i < num_tokens with s = slot_mapping[i] >= 0 and every kv head h,
 *   k_pages[s/16][h][s%16][:] = k[i][h][:]   and the same for v.   Bit copies, no arithmetic.
 * Non-negative slots must be unique within one call.  num_tokens = 0 is a no-op.
 */
int sangam_kv_write(sangam_ctx* ctx, const void* k, const void* v, const int32_t* slot_mapping,
                    int32_t num_tokens, void* k_pages, void* v_pages, void* stream);

/*
 * KV write with rotary position embedding fused in (rotate K, then scatter; V is copied): the same contract as
 * sangam_kv_write with  k_pages[s/16][h][s%16][:] = bf16( rope(k[i][h][:], positions[i]) ),  rotate-half convention
 *   out[j] = x[j] cos(a_j) - x[j + D/2] sin(a_j),  out[j + D/2] = x[j + D/2] cos(a_j) + x[j] sin(a_j),  a_j = pos * base^(-2j/D),
 * fp32 arithmetic, round to nearest even.  cos_sin is a device fp32 table [max_pos][head_dim]: row p holds cos(p * theta_j) for
 * j < D/2 followed by sin(p * theta_j); the caller builds it once (any base / scaling).  positions: int32 [num_tokens], device.
 * A position outside [0, max_pos) skips the row and raises SANGAM_DEV_BAD_POSITION.
 */
int sangam_kv_write_rope(sangam_ctx* ctx, const void* k, const void* v, const int32_t* slot_mapping, const int32_t* positions,
                         const float* cos_sin, int32_t max_pos, int32_t num_tokens, void* k_pages, void* v_pages, void* stream);

/*
 * KV page transfer between workers, the two single-GPU halves (a prefill worker
 * hands a request's KV to a decode-role worker).  gather copies the pool pages listed in page_ids (device int32, the
 * request's block-table row) into contiguous staging buffers bf16 [num_pages_listed][Hkv][16][D]; scatter writes such
 * buffers into the pages page_ids names in the destination pools (the receiver's own allocation).  What moves between
 * the GPUs is the staging buffer (NCCL send / recv or a peer copy: paper_2607_04206_b200/kv_transfer.py).  A page id
 * outside [0, num_pages) skips that page and raises SANGAM_DEV_BAD_PAGE.
 */
int sangam_kv_gather(sangam_ctx* ctx, const void* k_pages, const void* v_pages, const int32_t* page_ids, int32_t num_pages_listed,
                     void* k_stage, void* v_stage, void* stream);
int sangam_kv_scatter(sangam_ctx* ctx, const void* k_stage, const void* v_stage, const int32_t* page_ids, int32_t num_pages_listed,
                      void* k_pages, void* v_pages, void* stream);

/*
 * Confidence-threshold sampler over the rows the iteration decoded ("unmasks every masked position whose top-1 probability
 * exceeds a threshold"; threshold 0.9).  logits: bf16 [num_rows][vocab] (device, 2-byte aligned
 * rows); masked: int32 [num_rows], nonzero = still masked; cu_rows: int32 [num_requests + 1], rows of request r (its
 * current block) are cu_rows[r] .. cu_rows[r+1]-1.  Outputs (device): token[t] = argmax_j logits[t][j] (lowest index on
 * ties), conf[t] = softmax(logits[t])[token[t]] (fp32), unmask[t] = 1 for every masked row with conf > threshold; if no
 * masked row of a request passes, its most confident masked row (lowest index on ties) is unmasked instead, so every
 * step commits at least one position per request that still has masked rows.  Two kernels; no host sync.
 */
int sangam_confidence_sample(sangam_ctx* ctx, const void* logits, int32_t vocab, const int32_t* masked, const int32_t* cu_rows,
                             int32_t num_requests, int32_t num_rows, float threshold, int32_t* token, float* conf,
                             int32_t* unmask, void* stream);

/*
 * The same sampler for callers that must not allocate (code under CUDA-graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): no ctx, and the call performs no cudaMalloc / cudaFree and no allocating library routine.
 * sangam_confidence_sample allocates its scratch lazily on first use; here the per-(row, vocabulary slice) partials live
 * in a file-scope device array inside the library, SANGAM_STATIC_SAMPLER_MAX_PARTIALS entries of 16 bytes = 1 MiB,
 * which every GPU that loads the library holds until the process exits.  Same arguments, same results (bit-identical
 * when the slicing coincides, else within fp32 rounding of conf) as sangam_confidence_sample, on the caller's CURRENT
 * device.  Limit: num_rows <= SANGAM_STATIC_SAMPLER_MAX_ROWS, else SANGAM_ERR_WORKSPACE and nothing is launched (use
 * sangam_confidence_sample for larger batches).  Every call on a device shares the one array; nothing in it has to be
 * cleared between calls (each call writes every entry it later reads), but two calls whose kernels overlap on the GPU
 * (different streams without an event between them, concurrently launched graphs) race on it: serialise them.
 * Errors: return code as above; the message of the calling thread's last failure from sangam_static_last_error().
 */
#define SANGAM_STATIC_SAMPLER_MAX_PARTIALS 65536
#define SANGAM_STATIC_SAMPLER_MAX_ROWS     4096
int sangam_confidence_sample_static(const void* logits, int32_t vocab, const int32_t* masked, const int32_t* cu_rows,
                                    int32_t num_requests, int32_t num_rows, float threshold, int32_t* token, float* conf,
                                    int32_t* unmask, void* stream);
const char* sangam_static_last_error(void);

/*
 * Block attention (steps a3-a9): for request r < batch, row t in [cu_q_lens[r], cu_q_lens[r+1]),
 * q head h, kv head g = h / G, context length c = ctx_lens[r]:
 *   s_j = scale * <q[t][h], K_r[j][g]>, j < c;   out[t][h] = sum_j softmax_j(s) V_r[j][g]
 * with K_r[j] = k_pages[block_table[r][j/16]][g][j%16].  No mask among j < c.  c = 0 writes zeros.
 * bf16 inputs, fp32 accumulation, P rounded to bf16 before PV, out = bf16(O / l).
 * Long contexts are split over CTAs and merged by a combine kernel in fixed order; results are bitwise
 * reproducible for fixed inputs.  `total_q` is the host-known number of rows of q/out
 * (an upper bound is fine: rows past cu_q_lens[batch] are not touched).
 */
int sangam_block_attn(sangam_ctx* ctx, const void* q, const void* k_pages, const void* v_pages,
                      const int32_t* block_table, const int32_t* cu_q_lens, const int32_t* ctx_lens,
                      int32_t batch, int32_t total_q, float scale, void* out, void* stream);

/*
 * Kernel choice of sangam_block_attn.  AUTO (default): decode-shaped batches (total_q * G <= 32 * batch, i.e. on
 * average at most one 32-row unit per request and kv head -- block decodes, block 32) run
 * the swapped-operand decode kernel, everything else the two-stream prefill / hybrid kernel.  All kernels compute
 * the same function for every batch they accept; PREFILL / DECODE / GQA_PAIR force one of them (tests, measurements).
 * DECODE returns SANGAM_ERR_UNSUPPORTED for geometries the decode kernel is not built for (num_q_heads /
 * num_kv_heads > 32), GQA_PAIR for MHA (G = 1) and G > 128.  GQA_PAIR is the CTA-pair decode kernel of GQA models
 * (two SMs share every K/V tile through TMA multicast, each computes one 128-row q tile of the request's block); AUTO
 * never picks it: on the Dream-like shapes it is measured slower than the two-stream kernel.
 */
#define SANGAM_DISPATCH_AUTO    0
#define SANGAM_DISPATCH_PREFILL 1
#define SANGAM_DISPATCH_DECODE  2
#define SANGAM_DISPATCH_GQA_PAIR 3
int sangam_set_dispatch(sangam_ctx* ctx, int32_t mode);

/* Read-only facts about a ctx (host side, no device work); -1 for an unknown `what`. */
#define SANGAM_QUERY_SM_COUNT            0   /* SMs of the ctx's device */
#define SANGAM_QUERY_DECODE_CTAS_PER_SM  1   /* resident CTAs per SM of the decode kernel (0: kernel unavailable) */
#define SANGAM_QUERY_DISPATCH            2   /* current SANGAM_DISPATCH_* mode */
#define SANGAM_QUERY_GQA_PAIR_KERNEL     3   /* 1 if the CTA-pair decode kernel exists for the geometry */
#define SANGAM_QUERY_LAST_KERNEL         4   /* SANGAM_DISPATCH_PREFILL / DECODE / GQA_PAIR: the kernel the last sangam_block_attn
                                               launched (what AUTO chose); 0 before the first call */
int32_t sangam_query(const sangam_ctx* ctx, int32_t what);

/*
 * Same contract as sangam_block_attn, computed by a plain CUDA-core (no tensor core) kernel with
 * fp32 arithmetic.  A cross-check for the tcgen05 path on workloads too large for the CPU oracle;
 * never dispatched by sangam_block_attn.
 */
int sangam_block_attn_simt(sangam_ctx* ctx, const void* q, const void* k_pages, const void* v_pages,
                           const int32_t* block_table, const int32_t* cu_q_lens, const int32_t* ctx_lens,
                           int32_t batch, int32_t total_q, float scale, void* out, void* stream);

/*
 * One whole iteration from HOST buffers (the end-to-end entry point): copies q, k, v and the
 * metadata host->device into ctx-owned staging, runs sangam_kv_write then sangam_block_attn on
 * `stream`, copies `out` device->host and synchronises the stream.  *_host pointers are host
 * memory (pinned for full copy speed); k_pages / v_pages are the device pools.
 */
int sangam_iteration_host(sangam_ctx* ctx, const void* q_host, const void* k_host, const void* v_host,
                          const int32_t* slot_mapping_host, int32_t num_tokens,
                          void* k_pages, void* v_pages,
                          const int32_t* block_table_host, const int32_t* cu_q_lens_host,
                          const int32_t* ctx_lens_host, int32_t batch, int32_t total_q,
                          float scale, void* out_host, void* stream);

/*
 * The same iteration from ONE packed host buffer: q | k | v | slot_mapping | block_table | cu_q_lens | ctx_lens, each part
 * on a 256-byte boundary at the offsets sangam_packed_layout returns (offsets8[0..6]; offsets8[7] = total bytes).  One
 * host-to-device copy of the whole buffer, both kernels, one device-to-host copy of `out`, stream synchronize.  Pin the
 * buffers for full copy speed.  The ctx-owned device staging is allocated on the first call.
 */
int sangam_packed_layout(const sangam_ctx* ctx, int32_t batch, int32_t total_q, int32_t num_tokens, int64_t* offsets8);
int sangam_iteration_packed(sangam_ctx* ctx, const void* packed_host, int32_t num_tokens, void* k_pages, void* v_pages,
                            int32_t batch, int32_t total_q, float scale, void* out_host, void* stream);

/* Reads and clears nothing: returns the sticky device flag word (synchronises the ctx's device). */
int sangam_device_status(sangam_ctx* ctx, uint32_t* flags);
int sangam_clear_device_status(sangam_ctx* ctx);

/* Number of kernels this ctx has launched since creation (bench.py's gpu_launches). */
int64_t sangam_launch_count(const sangam_ctx* ctx);

const char* sangam_last_error(const sangam_ctx* ctx);
const char* sangam_version(void);


/* ------------------------------------------------------------------------------------------------------------
 * Worker-level scheduler: Algorithm 1 "Deficit token-budget scheduling" plus the builder of the
 * batch metadata that sangam_kv_write / sangam_block_attn consume.  Host code only (integer logic, no device
 * work, no CUDA calls); every array of sangam_batch is HOST memory owned by the caller.
 *
 * Each iteration has a token budget tau.  sangam_sched_next seats every in-flight decode first (Tokens = one
 * block; decodes are never displaced), then admits waiting prefills -- fresh requests and block-boundary
 * re-prefills, in request ARRIVAL-TIME order -- while Tokens(p) = prompt + response fits
 * budget = tau - Tokens(decodes) + deficit; the first prefill that does not fit stops the scan (prefills cannot
 * be split); the unspent budget max(budget, 0) is carried as the next iteration's deficit; with no prefill
 * waiting the iteration is decode-only and the deficit is cleared.  Idle rule (liveness): while the
 * microbatch is still empty the head prefill is admitted even above the budget.  Over any busy period of W
 * iterations the admitted prefill tokens total at most W tau - sum_t Tokens(decodes_t).
 * Readings where the paper is silent (S20-S22): equal arrival times keep submission order; a head prefill
 * whose KV pages do not fit the free pool, or that would exceed max_batch / max_total_q, "does not fit" (also under
 * the idle rule); pages are taken at a request's first admission and returned when its last block resolves.
 *
 * Life cycle of a request (Fast-dLLM style caching): submit -> prefill (whole prompt +
 * response region) -> decode of block 0, one microbatch per denoising step, until the caller reports the block
 * resolved -> re-prefill queued with the request's original arrival time -> decode of block 1 -> ... for
 * ceil(min(output_len, response_len) / block) blocks, then the request retires.
 * Batch layout: requests in microbatch order, decodes first.  A decode's query rows are its current
 * block, a prefill's the whole sequence; ctx_len = prompt + response for both; slot_mapping lists the slot
 * (page * 16 + offset) of every query row in order: the K/V rows the iteration rewrites.
 */
typedef struct sangam_sched sangam_sched;

typedef struct {
    int32_t tau;                /* per-iteration token budget (PAPER.md:327 evaluates 512 .. 16384) */
    int32_t block;              /* response block = query rows of a decode (32) */
    int32_t page_size;          /* must be 16 */
    int32_t num_pages;          /* KV pool capacity in pages */
    int32_t max_batch;          /* capacities of the sangam_batch arrays (and of the sangam_ctx the batch is run on) */
    int32_t max_total_q;
    int32_t max_pages_per_req;  /* block_table row width W */
} sangam_sched_config;

typedef struct {
    int32_t batch;              /* requests in the microbatch: num_decodes decodes, then batch - num_decodes prefills */
    int32_t num_decodes;
    int32_t total_q;            /* = cu_q_lens[batch] */
    int32_t num_new_tokens;     /* entries of slot_mapping (= total_q) */
    int64_t deficit;            /* carried to the next iteration */
    int64_t* req_ids;           /* [max_batch]                      (any array may be NULL: not filled) */
    int32_t* cu_q_lens;         /* [max_batch + 1] */
    int32_t* ctx_lens;          /* [max_batch] */
    int32_t* block_table;       /* [max_batch][max_pages_per_req], -1 padded */
    int32_t* slot_mapping;      /* [max_total_q] */
} sangam_batch;

int sangam_sched_create(const sangam_sched_config* cfg, sangam_sched** out);
int sangam_sched_destroy(sangam_sched* s);
/* A request arrives.  SANGAM_ERR_WORKSPACE if it could never be scheduled (more pages than the pool or the
 * block-table width, more tokens than max_total_q); SANGAM_ERR_INVALID_ARG for a duplicate id or bad lengths. */
int sangam_sched_submit(sangam_sched* s, int64_t req_id, double arrival_time, int32_t prompt_len, int32_t response_len,
                        int32_t output_len);
/* One iteration of Algorithm 1; fills *out.  Must be followed by sangam_sched_complete before the next call. */
int sangam_sched_next(sangam_sched* s, sangam_batch* out);
/* After the microbatch ran: block_done[i] != 0 says decode i resolved its block (n = num_decodes of the last batch). */
int sangam_sched_complete(sangam_sched* s, const int32_t* block_done, int32_t n);

#define SANGAM_SCHED_DEFICIT        0
#define SANGAM_SCHED_WAITING        1   /* prefills in the queue */
#define SANGAM_SCHED_IN_FLIGHT      2   /* decodes in flight */
#define SANGAM_SCHED_FREE_PAGES     3
#define SANGAM_SCHED_LIVE_REQUESTS  4
int64_t sangam_sched_query(const sangam_sched* s, int32_t what);

#ifdef __cplusplus
}
#endif
#endif /* SANGAM_H_ */
