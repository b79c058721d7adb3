// attn_dec.cuh -- steps a3..a9 for DECODE-shaped batches: paged, varlen, non-causal block attention with
// SWAPPED operands on tcgen05 (sm_100a).
//
// A block decode brings at most a few dozen query rows per (request, kv head) ("a decode contributes an entire
// response block while attending over the prompt and response context"; block = 32) and is
// bound by streaming that request's K/V pages once ("Attention remains memory-bandwidth-bound and scales per request",
// PAPER.md:111).  With the query rows as UMMA M a 32-row block fills a quarter of the tile and one TMEM lane quarter:
// one warp does all softmax work.  Here the kv positions are M instead:
//     S^T[128 kv x 32 rows] = K_tile[128 x D] . Q^T          (A = K tile, K-major;  B = Q, K-major;  N = 32)
//     O^T[D x 32 rows]     += V_tile^T[D x 128] . P^T        (A = V tile, MN-major; B = P^T from shared memory)
// so that thread j of the four softmax warps owns kv position j of the tile (TMEM lane j): all four SM sub-partitions
// share the exponentials, the tensor pipe does N = 32 instead of N = 128 work per tile, and TMEM needs 64 columns.
// Per-row maxima run ACROSS lanes (warp redux + one shared-memory exchange per tile); row sums are kept as per-thread
// partials and reduced once per work item.
//
// Small CTAs, two per SM (256 threads, 113 KB shared memory, 64 TMEM columns): one CTA's fill / drain / epilogue
// overlaps the other's main loop.  Warp roles: 0 = device-side plan (a3) + TMA producer (a4), 1 = MMA issuer
// (a5, a7), 2 = arrival agent of split units, 4..7 = softmax (a6), epilogue (a8) and the fused split-KV merge (a9);
// warp 3 only completes the service warpgroup.  Two CTAs of eight warps put four warps on every SM sub-partition, i.e. 128 registers per
// thread at launch (the register file is split per sub-partition); setmaxnreg then moves the budget from the service
// warpgroup (64) to the softmax warpgroup (192).
// Work unit = (request r, kv head g, chunk of 32/G query tokens); the flattened (unit, page) sequence, each unit
// weighted with a fixed overhead, is cut into #CTA equal contiguous ranges at PAGE granularity (stream-K): at most two
// partial pieces per CTA.  Pieces of a split unit go to the workspace as (O^T fp32, m, l); the CTA that finishes a
// unit's last piece merges all of them in fixed piece order (bitwise reproducible) -- no second kernel.
#pragma once
#include <cuda.h>
#include <stdlib.h>

#include "common.cuh"
#include "ptx.cuh"

struct DecParams {
    const int32_t* block_table;    // [batch][W]
    const int32_t* cu_q_lens;      // [batch+1]
    const int32_t* ctx_lens;       // [batch]
    __nv_bfloat16* out;            // [total_q][Hq][D]
    const __nv_bfloat16* q;        // [total_q][Hq][D] (the GQA pair kernel reads q rows directly; the decode kernel through its tensor map)
    int32_t batch, total_q;
    int32_t Hq, Hkv, G, W, P;
    int32_t tq;                    // query tokens per unit: 32 / G (decode kernel), 2 tpt (GQA pair kernel)
    int32_t tpt;                   // GQA pair kernel: tokens per 128-row q tile = 128 / G
    uint32_t tq_magic;             // floor(2^32 / tq) + 1: x / tq = umulhi(x, magic) for x < 2^24 (unused when tq = 1)
    uint32_t g_magic;              // floor(2^32 / G) + 1 (unused when G = 1)
    float scale_log2;              // scale * log2(e)
    float* part_o;                 // [2 #CTAs][8 row groups][D][4 rows]  unnormalised partial O^T: a warp's 32 output columns of
                                   // one row group are 512 contiguous bytes (coalesced stores and merge loads)
    float* part_ml;                // [2 #CTAs][32][2]  (m in log2 units, l)
    int32_t* unit_cnt;             // [max units] pages of a split unit that have arrived; self-resetting
    int32_t min_w;                 // smallest share of the weighted unit list worth a CTA (coordinates)
    int32_t ov;                    // fixed cost of starting / finishing a unit, in pages (stream-K weight)
    uint32_t* flags;               // sticky device flags
#ifdef SANGAM_TRACE
    int32_t trace_cta;             // debug builds: the CTA that records events
#endif
};

namespace dec {

constexpr int BN = 128;          // kv positions per tile (UMMA M; 8 pages)
constexpr int NQ = 32;           // packed query rows per unit (UMMA N)
constexpr int NSTAGE = 3;        // ring of K / V tiles
constexpr int NTHREADS = 256;
#ifndef SANGAM_DEC_OV
#define SANGAM_DEC_OV 6
#endif
constexpr int OV = SANGAM_DEC_OV;  // fixed cost of starting / finishing a unit, in pages (stream-K weight)
#ifndef SANGAM_DEC_MINW
#define SANGAM_DEC_MINW 8
#endif
constexpr int MIN_W = SANGAM_DEC_MINW;  // smallest share of the weighted unit list given to a CTA (tiny batches use fewer CTAs)
constexpr float LAZY_T = 8.f;    // the reference maximum moves only when a tile exceeds it by 2^8
template <int D> constexpr int KV_ATOM_STRIDE = 1024 * (D / 64);   // page-major stages, see attn_tc.cuh

struct Item {          // one piece of work, published through shared memory (64 bytes)
    int valid;         // 0 = no more work
    int r, g;
    int tok0, ntok;    // first query token (inside the request) and number of tokens of the unit
    int q_start;       // cu_q_lens[r]
    int c;             // context length
    int pg0, pg1;      // page range [pg0, pg1) of the context handled by this piece (pg1 <= ceil(c / 16))
    int part_slot;     // -1: write `out`; else partial slot in the workspace
    int unit;          // split units: global unit index (arrival counter)
    int y0;            // split units: coordinate of the unit's page 0 in the flattened weighted list
    int upages;        // split units: pages of the whole unit
    int b_head, b_last; // split units: CTAs holding the first / last piece (consecutive CTAs hold the pieces in between)
    int pad0;
};
struct OutRef {        // where a unit's rows go
    int q_start, tok0, ntok, g;
};
struct PlanConst {     // published once per CTA by the planner (shared memory): the stream-K cut
    int T, Geff;
};
static_assert(sizeof(Item) == 64, "Item is 64 bytes");

template <int D>
struct Smem {
    static constexpr int KV_BYTES = BN * D * 2;
    static constexpr int Q_BYTES = NQ * D * 2;
    static constexpr int QSLAB = NQ * 128;                 // bytes of one 64-wide swizzled slab of the q tile
    static constexpr int P_BYTES = NQ * BN * 2;            // P^T: two 64-position slabs of 32 rows x 128 bytes
    static constexpr int OFF_KV = 0;
    static constexpr int OFF_Q = NSTAGE * KV_BYTES;
    static constexpr int OFF_P = OFF_Q + Q_BYTES;
    static constexpr int OFF_BAR = OFF_P + P_BYTES;
    static constexpr int B_KV_FULL = 0, B_KV_EMPTY = NSTAGE, B_ITEM_FULL = 2 * NSTAGE, B_ITEM_EMPTY = B_ITEM_FULL + 2,
                         B_Q_FULL = B_ITEM_EMPTY + 2, B_Q_EMPTY = B_Q_FULL + 1, B_S_FULL = B_Q_EMPTY + 1,
                         B_P_FULL = B_S_FULL + 1, B_P_EMPTY = B_P_FULL + 1, B_O_FREE = B_P_EMPTY + 1,
                         B_AGENT_REQ = B_O_FREE + 1, B_AGENT_DONE = B_AGENT_REQ + 1, NBAR = B_AGENT_DONE + 1;
    static constexpr int OFF_ITEMS = OFF_BAR + NBAR * 8;
    static constexpr int OFF_WM = OFF_ITEMS + 2 * (int)sizeof(Item);   // [4 warps][32] floats: per-warp column maxima / sums
    static constexpr int OFF_MREF = OFF_WM + 4 * 32 * 4;               // [32] floats: reference maximum of every row
    // misc block: +0 tmem slot, +8 merge flag, +16 agent_req[2], +32 Deferred[2]; then the abort word (followed, in
    // -DSANGAM_WAIT_TABLE debug builds only, by the per-warp wait table of ptx::mbar_wait)
    static constexpr int OFF_MISC = OFF_MREF + 32 * 4;
    static constexpr int OFF_ABORT = OFF_MISC + 96;
#ifdef SANGAM_WAIT_TABLE
    static constexpr int TOTAL = OFF_ABORT + 80;
#else
    static constexpr int TOTAL = OFF_ABORT + 4;
#endif
};
struct Deferred {      // a unit whose last piece turned out to be one this CTA had already handed to its agent warp
    int valid, unit, b_head, b_last, q_start, tok0, ntok, g;
};
// two CTAs per SM: 2 x (TOTAL + 1 KB reserved) <= 228 KB; the dynamic shared memory base is 1024-byte aligned
// (no static shared memory in this kernel; checked at run time)
#ifndef SANGAM_WAIT_TABLE
static_assert(Smem<128>::TOTAL <= 115712, "two CTAs per SM");
#endif

struct ReqInfo {
    int q0, qn, c, chunks, units, pages, w;
};

__device__ __forceinline__ void load_req(const DecParams& p, int r, int& q0, int& qn, int& c) {
    q0 = __ldg(p.cu_q_lens + r);
    qn = __ldg(p.cu_q_lens + r + 1) - q0;
    if (qn < 0) qn = 0;
    c = __ldg(p.ctx_lens + r);
    if (c < 0) c = 0;
    if ((c + SANGAM_PAGE - 1) / SANGAM_PAGE > p.W) { raise_flag(p.flags, DEV_CTX_TOO_LONG); c = 0; }
}
__device__ __forceinline__ ReqInfo derive(const DecParams& p, int q0, int qn, int c) {
    ReqInfo x;
    x.q0 = q0; x.qn = qn; x.c = c;
    x.chunks = p.tq == 1 ? qn : (int)__umulhi((uint32_t)(qn + p.tq - 1), p.tq_magic);
    x.units = p.Hkv * x.chunks;
    x.pages = (c + SANGAM_PAGE - 1) / SANGAM_PAGE;
    x.w = (x.pages > 0 ? x.pages : 1) + p.ov;                // an empty context still needs one visit (zero rows)
    return x;
}

// floor(n / d) for n < 2^42, 0 < d < 2^31: float estimate, exact correction by multiplication (an integer division is
// ~150 clk of dependent code; the planner sits on the kernel's start-up path and the merge on its tail)
__device__ __forceinline__ int div_floor(uint64_t n, uint32_t d) {
    int q = (int)((float)n * __frcp_rn((float)d));
    int64_t r = (int64_t)n - (int64_t)q * (int64_t)d;
    while (r < 0) { --q; r += d; }
    while (r >= (int64_t)d) { ++q; r -= d; }
    return q;
}
// CTA b of Geff owns the coordinates [cut(b), cut(b + 1)) of the T-long flattened weighted unit list
__device__ __forceinline__ int cut(int b, const PlanConst& pc) {
    if (b >= pc.Geff) return pc.T;
    return div_floor((uint64_t)(uint32_t)b * (uint32_t)pc.T, (uint32_t)pc.Geff);
}
// the CTA whose range holds coordinate y:  ceil((y + 1) Geff / T) - 1
__device__ __forceinline__ int owner(int y, const PlanConst& pc) {
    const int b = div_floor((uint64_t)(uint32_t)(y + 1) * (uint32_t)pc.Geff + (uint32_t)pc.T - 1u, (uint32_t)pc.T) - 1;
    return b < 0 ? 0 : (b > pc.Geff - 1 ? pc.Geff - 1 : b);
}

// ------------------------------------------------------------------------------------------------
// Device-side plan (a3), one warp, all lanes: stream-K cut of the flattened weighted unit list at page granularity.
// `nc` workers (CTAs, or clusters) share the T coordinates equally; worker `b` walks its range with next().
// ------------------------------------------------------------------------------------------------
struct Planner {
    int rq0, rqn, rc;        // request `lane` (< 32) in registers; later look-ups are shuffles
    PlanConst pc;
    int R, b, remaining, r_cur, u_in_r, off, unit_base, unit_gid;
    ReqInfo cur;

    __device__ __forceinline__ ReqInfo get(const DecParams& p, int r) const {             // warp-uniform r
        int a, q, c;
        if (r < 32) { a = __shfl_sync(0xffffffffu, rq0, r); q = __shfl_sync(0xffffffffu, rqn, r); c = __shfl_sync(0xffffffffu, rc, r); }
        else load_req(p, r, a, q, c);
        return derive(p, a, q, c);
    }

    __device__ __forceinline__ void init(const DecParams& p, int lane, int nc, int b_) {
        const unsigned FULL = 0xffffffffu;
        R = p.batch; b = b_;
        rq0 = 0; rqn = 0; rc = 0;
        if (lane < R) load_req(p, lane, rq0, rqn, rc);
        // weighted length and unit count of the first 32 requests, inclusive prefix sums over the lanes
        const ReqInfo mine = derive(p, rq0, rqn, rc);
        const int my_t = lane < R ? mine.units * mine.w : 0, my_u = lane < R ? mine.units : 0;
        int incl_t = my_t, incl_u = my_u;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int vt = __shfl_up_sync(FULL, incl_t, o), vu = __shfl_up_sync(FULL, incl_u, o);
            if (lane >= o) { incl_t += vt; incl_u += vu; }
        }
        int T = __shfl_sync(FULL, incl_t, 31);
        for (int base = 32; base < R; base += 32) {             // batches of more than 32 requests (rare)
            int t = 0;
            if (base + lane < R) { int a, q, c; load_req(p, base + lane, a, q, c); const ReqInfo x = derive(p, a, q, c); t = x.units * x.w; }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(FULL, t, o);
            T += t;
        }
        // Geff workers share the T coordinates equally; a share is never smaller than min_w (tiny batches use fewer
        // workers instead of cutting every unit into slivers)
        pc.T = T;
        int ge = T > 0 ? div_floor((uint64_t)(uint32_t)T, (uint32_t)(p.min_w > 0 ? p.min_w : 1)) : 0;
        ge = ge < 1 ? 1 : ge;
        pc.Geff = T <= 0 ? 0 : (nc < ge ? nc : ge);
        remaining = 0; r_cur = R; u_in_r = 0; off = 0; unit_base = 0; unit_gid = 0;
        cur = mine;
        if (b < pc.Geff) {
            const int x0 = cut(b, pc), x1 = cut(b + 1, pc);
            remaining = x1 - x0;
            // the request holding coordinate x0
            int found = -1, req_base = 0, gid_base = 0;
            const unsigned m = __ballot_sync(FULL, incl_t > x0);
            if (m) {
                found = __ffs(m) - 1;
                req_base = __shfl_sync(FULL, incl_t - my_t, found);
                gid_base = __shfl_sync(FULL, incl_u - my_u, found);
            } else {
                int acc = __shfl_sync(FULL, incl_t, 31), accu = __shfl_sync(FULL, incl_u, 31);
                for (int base = 32; base < R && found < 0; base += 32) {
                    int tl = 0, ul = 0;
                    if (base + lane < R) { int a, q, c; load_req(p, base + lane, a, q, c); const ReqInfo x = derive(p, a, q, c); tl = x.units * x.w; ul = x.units; }
                    int it2 = tl, iu2 = ul;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int vt = __shfl_up_sync(FULL, it2, o), vu = __shfl_up_sync(FULL, iu2, o);
                        if (lane >= o) { it2 += vt; iu2 += vu; }
                    }
                    const unsigned m2 = __ballot_sync(FULL, acc + it2 > x0);
                    if (m2) {
                        const int l = __ffs(m2) - 1;
                        found = base + l;
                        req_base = acc + __shfl_sync(FULL, it2 - tl, l);
                        gid_base = accu + __shfl_sync(FULL, iu2 - ul, l);
                    } else {
                        acc += __shfl_sync(FULL, it2, 31); accu += __shfl_sync(FULL, iu2, 31);
                    }
                }
            }
            if (found >= 0) {
                r_cur = found;
                cur = get(p, r_cur);
                const int pos = x0 - req_base;
                u_in_r = div_floor((uint64_t)(uint32_t)pos, (uint32_t)cur.w);
                off = pos - u_in_r * cur.w;
                unit_base = req_base + u_in_r * cur.w;
                unit_gid = gid_base + u_in_r;
            } else {
                remaining = 0;
            }
        }
    }

    // the next piece of work of this worker (it.valid = 0: none left)
    __device__ __forceinline__ void next(const DecParams& p, Item& it) {
        it.valid = 0; it.r = 0; it.g = 0; it.tok0 = 0; it.ntok = 0; it.q_start = 0; it.c = 0; it.pg0 = 0; it.pg1 = 0;
        it.part_slot = -1; it.unit = 0; it.y0 = 0; it.upages = 0; it.b_head = -1; it.b_last = -1; it.pad0 = 0;
        // this worker owns the weighted coordinates [x0, x1) of the flattened unit list; a unit spans OV + max(pages, 1)
        // of them, coordinate OV + j being its page j.  A range covering only overhead coordinates yields no work there.
        while (remaining > 0 && r_cur < R && !it.valid) {
            const int take = remaining < cur.w - off ? remaining : cur.w - off;
            const int OV = p.ov;
            const int a = off > OV ? off - OV : 0, e = off + take > OV ? off + take - OV : 0;
            if (e > a) {
                const int g = cur.chunks == 1 ? u_in_r : div_floor((uint64_t)(uint32_t)u_in_r, (uint32_t)cur.chunks);
                const int ch = u_in_r - g * cur.chunks;
                it.valid = 1; it.r = r_cur; it.g = g;
                it.tok0 = ch * p.tq;
                const int left = cur.qn - it.tok0;
                it.ntok = left < p.tq ? left : p.tq;
                it.q_start = cur.q0; it.c = cur.c;
                it.pg0 = a; it.pg1 = e < cur.pages ? e : cur.pages;      // empty context: pages = 0 -> no tiles
                if (!(a == 0 && e == cur.w - OV)) {                       // a piece of a unit split across workers
                    it.part_slot = 2 * b + (a == 0 ? 1 : 0);
                    it.unit = unit_gid; it.y0 = unit_base + OV; it.upages = cur.pages;
                    it.b_head = a == 0 ? b : owner(it.y0, pc);
                    it.b_last = e == cur.w - OV ? b : owner(it.y0 + cur.pages - 1, pc);
                }
            }
            remaining -= take;
            off += take;
            if (off == cur.w) {
                off = 0;
                unit_base += cur.w;
                ++unit_gid;
                if (++u_in_r == cur.units) {
                    u_in_r = 0;
                    do {
                        ++r_cur;
                        if (r_cur < R) cur = get(p, r_cur);
                    } while (r_cur < R && cur.units == 0);
                }
            }
        }
    }
};

// ------------------------------------------------------------------------------------------------
// warp 0: device-side plan (a3) + TMA page gather (a4) + Q loads
// ------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void producer_warp(const DecParams& p, const CUtensorMap* mapK, const CUtensorMap* mapV,
                                              const CUtensorMap* mapQ, uint8_t* smem, uint32_t sbase, Item* items,
                                              volatile uint32_t* abort_flag, int lane) {
    using L = Smem<D>;
    const unsigned FULL = 0xffffffffu;
    const int NC = gridDim.x, b = blockIdx.x;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    DT_DECL;
    DT(1);
    Planner plan;
    plan.init(p, lane, NC, b);
    DT(2);

    uint32_t stage = 0, phase = 0, icount = 0, qcount = 0;
    while (true) {
        if (*abort_flag) break;
        Item it;
        plan.next(p, it);
        // publish
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_EMPTY + islot), ((icount >> 1) & 1u) ^ 1u, abort_flag);
        if (lane == 0) {
            items[islot] = it;
            ptx::mbar_arrive(bar(L::B_ITEM_FULL + islot));
        }
        __syncwarp();
        DT(3);
        ++icount;
        if (!it.valid) break;

        const int npg = it.pg1 - it.pg0;
        if (npg > 0) {
            // the piece's page ids, 64 at a time (lane l keeps entries l and 32 + l of the window); the next window is
            // requested while this one is consumed, so no K/V load ever waits on a block-table read except the first
            const int32_t* bt = p.block_table + (int64_t)it.r * p.W + it.pg0;
            int ida = lane < npg ? __ldg(bt + lane) : 0, idb = 32 + lane < npg ? __ldg(bt + 32 + lane) : 0;
            // the unit's query rows: one TMA box (64 columns, G heads, tq tokens) per 64-column slab
            ptx::mbar_wait(bar(L::B_Q_EMPTY), (qcount & 1u) ^ 1u, abort_flag);
            if (lane == 0) ptx::mbar_arrive_expect_tx(bar(L::B_Q_FULL), (uint32_t)(p.G * p.tq * D * 2));
            __syncwarp();
            if (lane < D / 64)
                ptx::tma_load_3d(sbase + (uint32_t)(L::OFF_Q + lane * L::QSLAB), mapQ, bar(L::B_Q_FULL), lane * 64, it.g * p.G,
                                 it.q_start + it.tok0);
            ++qcount;
            // K / V tiles in ring order K(0) V(0) K(1) V(1) ...; one TMA box per page, lanes 0..7 issue
            const int nt = (npg + 7) >> 3;
            int nida = 0, nidb = 0;
            for (int t = 0; t < nt; ++t) {
                const int tw = t & 7;                        // tile inside the 64-page window
                if (tw == 0) {
                    if (t > 0) { ida = nida; idb = nidb; }
                    const int nb = 8 * t + 64;               // first page of the next window
                    nida = nb + lane < npg ? __ldg(bt + nb + lane) : 0;
                    nidb = nb + 32 + lane < npg ? __ldg(bt + nb + 32 + lane) : 0;
                }
                int np = npg - 8 * t;
                np = np > 8 ? 8 : np;
                const int src = (8 * tw + lane) & 31;
                const int pa_ = __shfl_sync(FULL, ida, src), pb_ = __shfl_sync(FULL, idb, src);
                int page = tw < 4 ? pa_ : pb_;
                if (lane < np && (unsigned)page >= (unsigned)p.P) {
                    raise_flag(p.flags, DEV_BAD_PAGE);       // the box falls outside the tensor: TMA fills zeros
                    page = p.P;
                }
                const int coord = (page * p.Hkv + it.g) * 2;
#pragma unroll 1
                for (int kv = 0; kv < 2; ++kv) {
                    ptx::mbar_wait(bar(L::B_KV_EMPTY + stage), phase ^ 1u, abort_flag);
                    if (lane == 0) ptx::mbar_arrive_expect_tx(bar(L::B_KV_FULL + stage), (uint32_t)(np * SANGAM_PAGE * D * 2));
                    __syncwarp();
                    if (lane < np)
                        ptx::tma_load_4d(sbase + (uint32_t)(L::OFF_KV + stage * L::KV_BYTES + lane * (2 * KV_ATOM_STRIDE<D>)),
                                         kv ? mapV : mapK, bar(L::B_KV_FULL + stage), 0, 0, 0, coord);
                    if (++stage == NSTAGE) { stage = 0; phase ^= 1u; }
                    DT(4 + kv);
                }
                if (*abort_flag) break;
            }
        }
    }
    // Tail: every tcgen05.commit aimed at a KV_EMPTY / Q_EMPTY barrier must have landed before this CTA may exit
    // (a late asynchronous arrive would hit the shared memory of whatever CTA runs here next).
    for (int k = 0; k < NSTAGE; ++k) {
        ptx::mbar_wait(bar(L::B_KV_EMPTY + stage), phase ^ 1u, abort_flag);
        if (++stage == NSTAGE) { stage = 0; phase ^= 1u; }
    }
    ptx::mbar_wait(bar(L::B_Q_EMPTY), (qcount & 1u) ^ 1u, abort_flag);
}

// stale rows [nv, ncols) of the last page of a V tile: zero them so that P = 0 meets V = 0, never NaN (reading S12)
template <int D>
__device__ __forceinline__ void zero_v_tail(uint32_t v_addr, int nv, int ncols, int lane) {
    const int nrows = ncols - nv;
    for (int e = lane; e < nrows * 8 * (D / 64); e += 32) {
        const int chunk = e & 7, rr = (e >> 3) % nrows, slab = (e >> 3) / nrows;
        const int row = nv + rr;
        asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(v_addr + (uint32_t)((row >> 3) * KV_ATOM_STRIDE<D> + slab * 1024 + (row & 7) * 128 + chunk * 16)), "r"(0)
                     : "memory");
    }
    ptx::fence_proxy_async_smem();
    __syncwarp();
}

// ------------------------------------------------------------------------------------------------
// warp 1: MMA issuer.  Per kv tile, strictly in ring order:  S^T = K Q^T  ->  (softmax)  ->  O^T += V^T P^T.
// The path is HBM-bound (one tile's chain is ~1 500 clk against ~5 400 clk per tile and CTA at the roofline),
// so nothing is gained by running QK of the next tile ahead.
// ------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void mma_warp(const DecParams& p, uint32_t sbase, uint32_t tmem, const Item* items,
                                         volatile uint32_t* abort_flag, int lane) {
    using L = Smem<D>;
    DT_DECL;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    const uint64_t k_desc0 = ptx::smem_desc_sw128(sbase + L::OFF_KV, 16, KV_ATOM_STRIDE<D>);      // A, K-major (kv rows x d)
    const uint64_t v_desc0 = ptx::smem_desc_sw128(sbase + L::OFF_KV, 1024, KV_ATOM_STRIDE<D>);    // A, MN-major (d x kv)
    const uint64_t q_desc0 = ptx::smem_desc_sw128(sbase + L::OFF_Q, 16, 1024);                    // B, K-major (rows x d)
    const uint64_t p_desc0 = ptx::smem_desc_sw128(sbase + L::OFF_P, 16, 1024);                    // B, K-major (rows x kv)
    constexpr uint32_t IDESC_QK = ptx::idesc_bf16(BN, NQ, 0, 0);
    constexpr uint32_t IDESC_PV = ptx::idesc_bf16(128, NQ, 1, 0);     // M = 128 also for D = 64 (upper lanes unused)
    constexpr uint32_t VSTEP = (uint32_t)(2 * KV_ATOM_STRIDE<D>) >> 4;  // one K-step of PV = 16 kv rows = one page
    const uint32_t s_tmem = tmem, o_tmem = tmem + 32u;
    uint32_t stage = 0, phase = 0, icount = 0, qcount = 0, pcount = 0, ocount = 0;
    while (true) {
        if (*abort_flag) break;
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_FULL + islot), (icount >> 1) & 1u, abort_flag);
        const Item it = items[islot];
        if (!it.valid) break;
        const int npg = it.pg1 - it.pg0, nt = (npg + 7) >> 3;
        if (nt > 0) {
            ptx::mbar_wait(bar(L::B_Q_FULL), qcount & 1u, abort_flag);
            ++qcount;
            const int c_lim = it.c < it.pg1 * SANGAM_PAGE ? it.c : it.pg1 * SANGAM_PAGE;
            for (int t = 0; t < nt; ++t) {
                if (*abort_flag) break;
                int nvt = c_lim - (it.pg0 + 8 * t) * SANGAM_PAGE;
                nvt = nvt > BN ? BN : nvt;
                // ---- S^T = K Q^T
                const uint32_t sk = stage;
                ptx::mbar_wait(bar(L::B_KV_FULL + sk), phase, abort_flag);
                if (++stage == NSTAGE) { stage = 0; phase ^= 1u; }
                ptx::tc_fence_after();
                DT(10);
                if (ptx::elect_one()) {
                    const uint64_t a = k_desc0 + (uint64_t)(sk * (L::KV_BYTES >> 4));
                    ptx::mma_ss_x4(s_tmem, a, q_desc0, IDESC_QK, 0u, 2u);
                    if (D == 128) ptx::mma_ss_x4(s_tmem, a + (1024 >> 4), q_desc0 + (L::QSLAB >> 4), IDESC_QK, 1u, 2u);
                    ptx::mma_commit(bar(L::B_KV_EMPTY + sk));
                    ptx::mma_commit(bar(L::B_S_FULL));
                    if (t == nt - 1) ptx::mma_commit(bar(L::B_Q_EMPTY));
                }
                __syncwarp();
                // ---- O^T += V^T P^T
                const uint32_t sv = stage;
                ptx::mbar_wait(bar(L::B_KV_FULL + sv), phase, abort_flag);
                if (++stage == NSTAGE) { stage = 0; phase ^= 1u; }
                if (nvt & 15) zero_v_tail<D>(sbase + (uint32_t)(L::OFF_KV + sv * L::KV_BYTES), nvt, (nvt + 15) & ~15, lane);
                if (t == 0 && ocount > 0) ptx::mbar_wait(bar(L::B_O_FREE), (ocount - 1u) & 1u, abort_flag);   // previous epilogue has read O^T
                ptx::mbar_wait(bar(L::B_P_FULL), pcount & 1u, abort_flag);
                ++pcount;
                ptx::tc_fence_after();
                DT(11);
                if (ptx::elect_one()) {
                    const uint64_t a = v_desc0 + (uint64_t)(sv * (L::KV_BYTES >> 4));
                    const int ks_n = (nvt + 15) >> 4;
                    if (ks_n == 8) {
                        ptx::mma_ss_x4_ab(o_tmem, a, p_desc0, IDESC_PV, t > 0 ? 1u : 0u, VSTEP, 2u);
                        ptx::mma_ss_x4_ab(o_tmem, a + 4 * VSTEP, p_desc0 + (4096 >> 4), IDESC_PV, 1u, VSTEP, 2u);
                    } else {
                        for (int ks = 0; ks < ks_n; ++ks)
                            ptx::mma_ss(o_tmem, a + (uint64_t)(ks * VSTEP), p_desc0 + (uint64_t)((ks >> 2) * (4096 >> 4) + (ks & 3) * 2),
                                        IDESC_PV, (t > 0 || ks > 0) ? 1u : 0u);
                    }
                    ptx::mma_commit(bar(L::B_KV_EMPTY + sv));
                    ptx::mma_commit(bar(L::B_P_EMPTY));
                }
                __syncwarp();
            }
            ++ocount;
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar(L::B_ITEM_EMPTY + islot));
        ++icount;
    }
}

// ------------------------------------------------------------------------------------------------
// warps 2..5: softmax (a6), epilogue (a8), fused split-KV merge (a9).  Thread jl = (warp % 4) * 32 + lane owns TMEM
// lane jl: kv position jl of the tile in S^T, output column d = jl in O^T.  Column c of either is packed query row c.
// ------------------------------------------------------------------------------------------------
// sum over the warp's lanes of v[c] for every c: lane i returns the sum of column i (31 shuffles, fixed order)
__device__ __forceinline__ float column_sums(float (&v)[32], int lane) {
#pragma unroll
    for (int step = 16; step >= 1; step >>= 1) {
        const bool up = (lane & step) != 0;
#pragma unroll
        for (int k = 0; k < step; ++k) {
            const float send = up ? v[k] : v[k + step];
            const float keep = up ? v[k + step] : v[k];
            v[k] = keep + __shfl_xor_sync(0xffffffffu, send, step);
        }
    }
    return v[0];
}

template <int D>
__device__ __forceinline__ void softmax_warps(const DecParams& p, uint8_t* smem, uint32_t sbase, uint32_t tmem, const Item* items,
                                              volatile uint32_t* abort_flag, int warp, int lane) {
    using L = Smem<D>;
    DT_DECL;
    const unsigned FULL = 0xffffffffu;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    const int qd = warp & 3, jl = qd * 32 + lane;
    const uint32_t lane_base = (uint32_t)(qd * 32) << 16;
    const uint32_t s_taddr = tmem + lane_base, o_taddr = tmem + lane_base + 32u;
    float* wm = reinterpret_cast<float*>(smem + L::OFF_WM);
    float* mref = reinterpret_cast<float*>(smem + L::OFF_MREF);      // reference maximum of every row (log2 units)
    volatile int* merge_flag = reinterpret_cast<volatile int*>(smem + L::OFF_MISC + 8);
    // P^T[row c][kv jl] in the K-major 128B-swizzled B-operand layout: slab = jl / 64, 16-byte chunk (jl % 64) / 8 XOR (c % 8)
    uint32_t pa[8];
#pragma unroll
    for (int k = 0; k < 8; ++k)
        pa[k] = sbase + (uint32_t)(L::OFF_P + (jl >> 6) * 4096 + k * 128 + ((((jl & 63) >> 3) ^ k) << 4) + (jl & 7) * 2);
    const float sc = fabsf(p.scale_log2);
    const uint32_t flip = p.scale_log2 < 0.f ? 0x80000000u : 0u;    // scale < 0: work on -s with |scale|
    volatile int* agent_req = reinterpret_cast<volatile int*>(smem + L::OFF_MISC + 16);
    // Output rows leave through shared memory (the P^T buffer is idle between units): O^T[d][row] is written as bf16
    // [row][d], then every thread moves 16-byte chunks of whole rows to `out` (row c = token c / G, head c % G).
    uint8_t* const obuf = smem + L::OFF_P;
    auto put_rows = [&](const float (&f)[32]) {               // this thread's output column jl of all 32 rows
        if (jl < D) {
#pragma unroll
            for (int c = 0; c < 32; ++c) reinterpret_cast<__nv_bfloat16*>(obuf)[c * D + jl] = __float2bfloat16_rn(f[c]);
        }
    };
    auto flush_rows = [&](const OutRef& r) {
        const int rows = r.ntok * p.G;                        // packed rows (token * G + head) that exist
        const bool tok_ok = r.q_start + r.tok0 >= 0 && r.q_start + r.tok0 + r.ntok <= p.total_q && (unsigned)r.g < (unsigned)p.Hkv;
        if (!tok_ok && lane == 0) raise_flag(p.flags, DEV_INTERNAL | 0x400u);
        ptx::bar_sync(1, 128);
        constexpr int CPR = D / 8;                            // 16-byte chunks per row
        for (int idx = jl; idx < rows * CPR; idx += 128) {
            const int c = idx / CPR, ch = idx - c * CPR;
            const int tl = p.G == 1 ? c : (int)__umulhi((uint32_t)c, p.g_magic), hh = c - tl * p.G;
            const uint4 v = *reinterpret_cast<const uint4*>(obuf + (c * D + ch * 8) * 2);
            if (tok_ok) *reinterpret_cast<uint4*>(p.out + ((int64_t)(r.q_start + r.tok0 + tl) * p.Hq + r.g * p.G + hh) * D + ch * 8) = v;
        }
        ptx::bar_sync(1, 128);                                // the buffer goes back to P^T
    };
    // General merge of a split unit (a9).  Pieces live in consecutive CTAs bh .. bl: slot 2 bh + 1 (head), then 2 (bh + 1),
    // ..., 2 bl; merged in that order whoever merges.  Lane c owns row c's statistics; the weights 2^(m_piece - M) of up
    // to 8 pieces go through this warp's own 1 KB of the idle P^T buffer so that every thread reads them as vectors.
    // Under a saturated memory system every dependent L2 round trip costs a microsecond, so a round requests the
    // statistics of up to 8 pieces and the data of its first three pieces together.
    auto merge_unit = [&](const OutRef& r, int unit, int bh, int bl) {
        const float2* ml = reinterpret_cast<const float2*>(p.part_ml) + lane;
        float* wt = reinterpret_cast<float*>(smem + L::OFF_P + qd * 1024);
        const int dd = jl < D ? jl : 0;
        auto slot_of = [&](int bb) { return bb == bh ? 2 * bh + 1 : 2 * bb; };
        auto load_piece = [&](int bb, float4 (&v)[8]) {        // this thread's column of piece bb, 32 rows
            const float4* so = reinterpret_cast<const float4*>(p.part_o) + (int64_t)slot_of(bb <= bl ? bb : bl) * 8 * D + dd;
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = __ldcg(so + k * D);
        };
        auto add_piece = [&](int k, const float4 (&v)[8], float (&f)[32]) {
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const float4 w4 = reinterpret_cast<const float4*>(wt + k * 32)[q];
                f[4 * q] = fmaf(v[q].x, w4.x, f[4 * q]); f[4 * q + 1] = fmaf(v[q].y, w4.y, f[4 * q + 1]);
                f[4 * q + 2] = fmaf(v[q].z, w4.z, f[4 * q + 2]); f[4 * q + 3] = fmaf(v[q].w, w4.w, f[4 * q + 3]);
            }
        };
        float M = -INFINITY, Lsum = 0.f, f[32];
#pragma unroll
        for (int c = 0; c < 32; ++c) f[c] = 0.f;
        for (int b0 = bh; b0 <= bl; b0 += 8) {
            const int nb = bl - b0 + 1 < 8 ? bl - b0 + 1 : 8;
            float4 va[8], vb[8], vc[8];
            load_piece(b0, va);
            load_piece(b0 + 1, vb);
            load_piece(b0 + 2, vc);
            float2 x[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) x[k] = k < nb ? __ldcg(ml + slot_of(b0 + k) * NQ) : make_float2(-INFINITY, 0.f);
            float Mn = M;
#pragma unroll
            for (int k = 0; k < 8; ++k) Mn = fmaxf(Mn, x[k].x);
            const float alpha = ptx::ex2(M - Mn);              // earlier rounds shrink (0 in the first round)
            M = Mn;
            Lsum *= alpha;
            __syncwarp();
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const float w = ptx::ex2(x[k].x - M);
                Lsum = fmaf(x[k].y, w, Lsum);
                wt[k * 32 + lane] = w;
            }
            if (b0 > bh) {
#pragma unroll
                for (int c = 0; c < 32; ++c) f[c] *= __shfl_sync(FULL, alpha, c);
            }
            __syncwarp();
            add_piece(0, va, f);
            if (nb > 1) add_piece(1, vb, f);
            if (nb > 2) add_piece(2, vc, f);
#pragma unroll 1
            for (int k = 3; k < nb; ++k) {                       // long contexts cut into many pieces
                load_piece(b0 + k, va);
                add_piece(k, va, f);
            }
        }
        const float inv_own = Lsum > 0.f ? 1.f / Lsum : 0.f;
#pragma unroll
        for (int c = 0; c < 32; ++c) f[c] *= __shfl_sync(FULL, inv_own, c);
        ptx::bar_sync(1, 128);           // every warp is done with its weight table before the buffer takes the rows
        put_rows(f);
        flush_rows(r);
        if (qd == 0 && lane == 0) p.unit_cnt[unit] = 0;     // re-arm for the next launch
    };
    uint32_t icount = 0, tcount = 0;       // items seen; kv tiles seen (S_FULL / P_EMPTY phases)
    // The kernel keeps 113 KB of shared memory per CTA, so the L1 holds next to nothing and a register spill is an L2
    // round trip: the row statistics live in shared memory (mref) or one per lane (m_own = row `lane`), S^T is read
    // from TMEM twice (maxima, then exponentials in two halves) instead of being kept, and the epilogue works in halves.
    while (true) {
        if (*abort_flag) break;
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_FULL + islot), (icount >> 1) & 1u, abort_flag);
        const Item it = items[islot];
        if (!it.valid) break;
        const int npg = it.pg1 - it.pg0, nt = (npg + 7) >> 3;
        const int c_lim = it.c < it.pg1 * SANGAM_PAGE ? it.c : it.pg1 * SANGAM_PAGE;
        float lp[32];                          // this thread's share of every row sum
#pragma unroll
        for (int c = 0; c < 32; ++c) lp[c] = 0.f;
        float m_own = -INFINITY;               // reference maximum of row `lane`
        int peek = -1;                         // split units: arrivals seen when this piece's last tile starts (one thread)
        for (int t = 0; t < nt; ++t) {
            if (*abort_flag) break;
            const bool valid = (it.pg0 + 8 * t) * SANGAM_PAGE + jl < c_lim;
            if (t == nt - 1 && it.b_head >= 0 && qd == 0 && lane == 0)      // non-blocking: consumed in the epilogue
                asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(peek) : "l"(p.unit_cnt + it.unit) : "memory");
            ptx::mbar_wait(bar(L::B_S_FULL), tcount & 1u, abort_flag);
            ptx::tc_fence_after();
            DT(20);
            {   // row maxima over the tile's 128 positions: warp redux, then one exchange through shared memory
                uint32_t s[32];
                ptx::tmem_ld32(s_taddr, s);
                ptx::tmem_wait_ld();
                float wx[32];
#pragma unroll
                for (int c = 0; c < 32; ++c) wx[c] = ptx::redux_max(valid ? __uint_as_float(s[c] ^ flip) : -INFINITY);
                if (lane == 0) {
                    float4* dst = reinterpret_cast<float4*>(wm + qd * 32);
#pragma unroll
                    for (int k = 0; k < 8; ++k) dst[k] = make_float4(wx[4 * k], wx[4 * k + 1], wx[4 * k + 2], wx[4 * k + 3]);
                }
            }
            ptx::bar_sync(1, 128);
            DT(21);
            const float cm = fmaxf(fmaxf(wm[lane], wm[32 + lane]), fmaxf(wm[64 + lane], wm[96 + lane])) * sc;
            const bool grow = cm > m_own + LAZY_T;
            bool p_free = false;
            if (__any_sync(FULL, grow)) {       // the same decision in all four warps (same data)
                // the reference maximum of some row moves (always in a unit's first tile, rarely later):
                // l and O^T shrink by alpha = 2^(m_old - m_new) in those rows
                const float m_new = grow ? cm : m_own;
                const float a_own = grow ? ptx::ex2(m_own - m_new) : 1.f;
                m_own = m_new;
                if (qd == 0) mref[lane] = m_new;
#pragma unroll
                for (int c = 0; c < 32; ++c) lp[c] *= __shfl_sync(FULL, a_own, c);
                if (t > 0) {
                    ptx::mbar_wait(bar(L::B_P_EMPTY), (tcount - 1u) & 1u, abort_flag);    // every PV so far has landed in O^T
                    p_free = true;
                    ptx::tc_fence_after();
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        uint32_t o[16];
                        ptx::tmem_ld16(o_taddr + (uint32_t)(16 * h), o);
                        ptx::tmem_wait_ld();
#pragma unroll
                        for (int c = 0; c < 16; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * __shfl_sync(FULL, a_own, 16 * h + c));
                        ptx::tmem_st16(o_taddr + (uint32_t)(16 * h), o);
                    }
                    ptx::tmem_wait_st();
                }
                ptx::bar_sync(1, 128);          // mref is visible to all four warps
            }
            DT(22);
            if (!p_free && tcount > 0) ptx::mbar_wait(bar(L::B_P_EMPTY), (tcount - 1u) & 1u, abort_flag);   // the previous PV has read P^T
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                uint32_t s[16];
                ptx::tmem_ld16(s_taddr + (uint32_t)(16 * h), s);
                float mr[16];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const float4 x = reinterpret_cast<const float4*>(mref)[4 * h + k];
                    mr[4 * k] = x.x; mr[4 * k + 1] = x.y; mr[4 * k + 2] = x.z; mr[4 * k + 3] = x.w;
                }
                ptx::tmem_wait_ld();
#pragma unroll
                for (int c = 0; c < 16; c += 2) {
                    const int cc = 16 * h + c;
                    float p0 = ptx::ex2(fmaf(__uint_as_float(s[c] ^ flip), sc, -mr[c]));
                    float p1 = ptx::ex2(fmaf(__uint_as_float(s[c + 1] ^ flip), sc, -mr[c + 1]));
                    if (!valid) { p0 = 0.f; p1 = 0.f; }            // positions past the context
                    lp[cc] += p0; lp[cc + 1] += p1;
                    ptx::sts_bf16_pair(pa[cc & 7] + (uint32_t)((cc >> 3) * 1024), pa[(cc + 1) & 7] + (uint32_t)((cc >> 3) * 1024),
                                       ptx::pack_bf16(p0, p1));
                }
            }
            ptx::fence_proxy_async_smem();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(L::B_P_FULL));
            DT(23);
            ++tcount;
        }
        // ---------------- epilogue
        // A CTA usually ends on the head piece of a unit whose other pieces were finished long ago by its neighbours (they
        // come first in those CTAs' ranges).  If the counter peeked at the start of the last tile shows that every other piece
        // has arrived, this piece is the last: it skips the partial store and the atomic, requests the other pieces (at most
        // two) now -- the loads fly while the last PV and the O^T read complete -- and merges them with its own registers,
        // accumulating in piece order exactly like the general merge (same bits whoever merges).
        // (the row sums need only this thread's partials, so they are reduced first: their registers are free again when
        // the other pieces are requested)
        const float ls = column_sums(lp, lane);
        wm[qd * 32 + lane] = ls;
        const bool split = nt > 0 && it.part_slot >= 0;
        const int np_u = it.b_last - it.b_head + 1, k_me = (int)blockIdx.x - it.b_head;
        if (split && qd == 0 && lane == 0) {
            int e = (np_u >= 2 && np_u <= 3 && k_me >= 0 && k_me < np_u && peek + npg == it.upages) ? 1 : 0;
            if (e) {
                // acquire the other pieces: an acquire load of the counter (it pairs with the agents' fence + atomic; the value
                // cannot have changed, every other piece had arrived) instead of a gpu-scope fence, which costs ~2 500 clk here
                int v;
                asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p.unit_cnt + it.unit) : "memory");
                e = (v + npg == it.upages) ? 1 : 0;
            }
            *merge_flag = e;
        }
        ptx::bar_sync(1, 128);
        const float l_own = (wm[lane] + wm[32 + lane]) + (wm[64 + lane] + wm[96 + lane]);   // fixed order
        const bool early = split && *merge_flag != 0;
        ptx::bar_sync(1, 128);                  // wm and merge_flag are rewritten later
        DT(24);
        OutRef ref;
        ref.q_start = it.q_start; ref.tok0 = it.tok0; ref.ntok = it.ntok; ref.g = it.g;
        if (early) {
            // self-contained (its registers are live only here): request the other pieces, in piece order, then wait for the
            // last PV, read O^T and merge:  k_me = 0: own a [b];  1: a own [b];  2: a b own
            float4 oa[8], ob[8];
            float2 xb = make_float2(-INFINITY, 0.f);
            const int sa = k_me == 0 ? 2 * (it.b_head + 1) : 2 * it.b_head + 1;
            const int sb = np_u > 2 ? 2 * (it.b_head + (k_me == 2 ? 1 : 2)) : sa;
            const float4* pa_ = reinterpret_cast<const float4*>(p.part_o) + (int64_t)sa * 8 * D + (jl < D ? jl : 0);
            const float4* pb_ = reinterpret_cast<const float4*>(p.part_o) + (int64_t)sb * 8 * D + (jl < D ? jl : 0);
#pragma unroll
            for (int k = 0; k < 8; ++k) { oa[k] = __ldcg(pa_ + k * D); ob[k] = __ldcg(pb_ + k * D); }
            const float2 xa = __ldcg(reinterpret_cast<const float2*>(p.part_ml) + sa * NQ + lane);
            if (np_u > 2) xb = __ldcg(reinterpret_cast<const float2*>(p.part_ml) + sb * NQ + lane);
            ptx::mbar_wait(bar(L::B_P_EMPTY), (tcount - 1u) & 1u, abort_flag);
            ptx::tc_fence_after();
            uint32_t o[32];
            ptx::tmem_ld32(o_taddr, o);
            ptx::tmem_wait_ld();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(L::B_O_FREE));      // the next unit's first PV may overwrite O^T
            DT(25);
            const float M = fmaxf(m_own, fmaxf(xa.x, xb.x));
            const float w_own = ptx::ex2(m_own - M), wa = ptx::ex2(xa.x - M), wb = ptx::ex2(xb.x - M);
            float Lsum = 0.f, f[32];
#pragma unroll
            for (int c = 0; c < 32; ++c) f[c] = 0.f;
            auto add_own = [&]() {
                Lsum = fmaf(l_own, w_own, Lsum);
#pragma unroll
                for (int c = 0; c < 32; ++c) f[c] = fmaf(__uint_as_float(o[c]), __shfl_sync(FULL, w_own, c), f[c]);
            };
            auto add_other = [&](const float4 (&v)[8], float2 x, float w) {
                Lsum = fmaf(x.y, w, Lsum);
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    f[4 * q] = fmaf(v[q].x, __shfl_sync(FULL, w, 4 * q), f[4 * q]);
                    f[4 * q + 1] = fmaf(v[q].y, __shfl_sync(FULL, w, 4 * q + 1), f[4 * q + 1]);
                    f[4 * q + 2] = fmaf(v[q].z, __shfl_sync(FULL, w, 4 * q + 2), f[4 * q + 2]);
                    f[4 * q + 3] = fmaf(v[q].w, __shfl_sync(FULL, w, 4 * q + 3), f[4 * q + 3]);
                }
            };
            if (k_me == 0) add_own();
            add_other(oa, xa, wa);
            if (k_me == 1) add_own();
            if (np_u > 2) add_other(ob, xb, wb);
            if (k_me == 2) add_own();
            const float inv_own = Lsum > 0.f ? 1.f / Lsum : 0.f;
#pragma unroll
            for (int c = 0; c < 32; ++c) f[c] *= __shfl_sync(FULL, inv_own, c);
            put_rows(f);
            flush_rows(ref);
            if (qd == 0 && lane == 0) { p.unit_cnt[it.unit] = 0; agent_req[islot] = 0; }    // re-arm the counter; nothing for the agent
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(L::B_AGENT_REQ));
        } else if (nt == 0) {
            if (it.part_slot < 0) {             // empty context: zero rows (reading S13); never split
                float z[32];
#pragma unroll
                for (int c = 0; c < 32; ++c) z[c] = 0.f;
                put_rows(z);
                flush_rows(ref);
            }
        } else {
            ptx::mbar_wait(bar(L::B_P_EMPTY), (tcount - 1u) & 1u, abort_flag);
            ptx::tc_fence_after();
            uint32_t o[32];
            ptx::tmem_ld32(o_taddr, o);
            ptx::tmem_wait_ld();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(L::B_O_FREE));      // the next unit's first PV may overwrite O^T
            DT(25);
            if (it.part_slot < 0) {
                const float inv_own = l_own > 0.f ? 1.f / l_own : 0.f;
                float f[32];
#pragma unroll
                for (int c = 0; c < 32; ++c) f[c] = __uint_as_float(o[c]) * __shfl_sync(FULL, inv_own, c);
                put_rows(f);
                flush_rows(ref);
            } else {
                // A piece of a split unit: (O^T unnormalised, m, l) go to the workspace and the agent warp is told.  It
                // makes them visible (a gpu-scope fence waits for the loads the producer has in flight: microseconds, so
                // it must not run on these warps) and adds the piece's pages to the unit's arrival counter; these warps
                // go on with the next unit at once.
                const bool slot_ok = it.part_slot < 2 * (int)gridDim.x && it.unit >= 0;
                if (!slot_ok && lane == 0) raise_flag(p.flags, DEV_INTERNAL | 0x100u);
                if (slot_ok) {
                    if (jl < D) {
                        float4* po = reinterpret_cast<float4*>(p.part_o) + (int64_t)it.part_slot * 8 * D + jl;
#pragma unroll
                        for (int k = 0; k < 8; ++k)
                            po[k * D] = make_float4(__uint_as_float(o[4 * k]), __uint_as_float(o[4 * k + 1]), __uint_as_float(o[4 * k + 2]), __uint_as_float(o[4 * k + 3]));
                    }
                    if (qd == 0) reinterpret_cast<float2*>(p.part_ml)[it.part_slot * NQ + lane] = make_float2(m_own, l_own);
                }
                DT(26);
                if (qd == 0 && lane == 0) agent_req[islot] = slot_ok ? 1 : 0;
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(bar(L::B_AGENT_REQ));      // release (cta): the agent's fence covers these stores
            }
        }
        __syncwarp();
        DT(29);
        if (lane == 0) ptx::mbar_arrive(bar(L::B_ITEM_EMPTY + islot));
        ++icount;
    }
    // A piece handed to the agent may have turned out to be its unit's last (the other pieces arrived in between): the
    // agent cannot merge (64 registers), so it leaves a record and the unit is merged here, after everything else.
    ptx::mbar_wait(bar(L::B_AGENT_DONE), 0u, abort_flag);
    const Deferred* defer = reinterpret_cast<const Deferred*>(smem + L::OFF_MISC + 32);
    for (int k = 0; k < 2; ++k) {
        const Deferred dr = defer[k];
        if (dr.valid) {
            OutRef ref;
            ref.q_start = dr.q_start; ref.tok0 = dr.tok0; ref.ntok = dr.ntok; ref.g = dr.g;
            merge_unit(ref, dr.unit, dr.b_head, dr.b_last);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// warp 2: arrival agent.  For every piece of a split unit that the softmax warps stored to the workspace: gpu-scope
// fence (release of the whole CTA's stores, cumulative through the mbarrier), add the piece's pages to the unit's
// counter; if that completes the unit, leave a Deferred record for the softmax warps.
// ------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void agent_warp(const DecParams& p, uint8_t* smem, uint32_t sbase, const Item* items,
                                           volatile uint32_t* abort_flag, int lane) {
    using L = Smem<D>;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    volatile int* agent_req = reinterpret_cast<volatile int*>(smem + L::OFF_MISC + 16);
    Deferred* defer = reinterpret_cast<Deferred*>(smem + L::OFF_MISC + 32);
    uint32_t icount = 0, rcount = 0;
    int ndef = 0;
    while (true) {
        if (*abort_flag) break;
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_FULL + islot), (icount >> 1) & 1u, abort_flag);
        const Item it = items[islot];
        if (!it.valid) break;
        const int npg = it.pg1 - it.pg0;
        if (npg > 0 && it.part_slot >= 0) {
            ptx::mbar_wait(bar(L::B_AGENT_REQ), rcount & 1u, abort_flag);
            ++rcount;
            if (lane == 0 && agent_req[islot] != 0) {
                int old;
                asm volatile("fence.acq_rel.gpu;" ::: "memory");
                asm volatile("atom.relaxed.gpu.global.add.s32 %0, [%1], %2;" : "=r"(old) : "l"(p.unit_cnt + it.unit), "r"(npg) : "memory");
                if (old + npg == it.upages) {
                    asm volatile("fence.acq_rel.gpu;" ::: "memory");
                    if (ndef < 2) {
                        Deferred dr;
                        dr.valid = 1; dr.unit = it.unit; dr.b_head = it.b_head; dr.b_last = it.b_last;
                        dr.q_start = it.q_start; dr.tok0 = it.tok0; dr.ntok = it.ntok; dr.g = it.g;
                        defer[ndef++] = dr;
                    } else {
                        raise_flag(p.flags, DEV_INTERNAL | 0x200u);      // a CTA has at most two split pieces
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar(L::B_ITEM_EMPTY + islot));
        ++icount;
    }
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(bar(L::B_AGENT_DONE));
}

// ------------------------------------------------------------------------------------------------
// kernel entry
// ------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(NTHREADS, 2)
decode_kernel(const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV,
              const __grid_constant__ CUtensorMap mapQ, const DecParams p) {
    using L = Smem<D>;
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = ptx::smem_u32(smem);
    Item* items = reinterpret_cast<Item*>(smem + L::OFF_ITEMS);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::OFF_MISC);
    volatile uint32_t* abort_flag = reinterpret_cast<volatile uint32_t*>(smem + L::OFF_ABORT);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    TRACE_CTA(0);
    if (tid == 0) {
        auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
        for (int s = 0; s < NSTAGE; ++s) { ptx::mbar_init(bar(L::B_KV_FULL + s), 1); ptx::mbar_init(bar(L::B_KV_EMPTY + s), 1); }
        for (int s = 0; s < 2; ++s) { ptx::mbar_init(bar(L::B_ITEM_FULL + s), 1); ptx::mbar_init(bar(L::B_ITEM_EMPTY + s), 6); }   // MMA warp + agent + 4 softmax warps
        ptx::mbar_init(bar(L::B_AGENT_REQ), 4); ptx::mbar_init(bar(L::B_AGENT_DONE), 1);
        ptx::mbar_init(bar(L::B_Q_FULL), 1); ptx::mbar_init(bar(L::B_Q_EMPTY), 1);
        ptx::mbar_init(bar(L::B_S_FULL), 1);
        ptx::mbar_init(bar(L::B_P_FULL), 4); ptx::mbar_init(bar(L::B_P_EMPTY), 1);
        ptx::mbar_init(bar(L::B_O_FREE), 4);
        for (int k = 1; k < (L::TOTAL - L::OFF_MISC) / 4; ++k) tmem_slot[k] = 0u;   // merge flag, agent requests, Deferred records, abort word
        ptx::fence_mbar_init();
        ptx::prefetch_tensormap(&mapK);
        ptx::prefetch_tensormap(&mapV);
        ptx::prefetch_tensormap(&mapQ);
    }
    if (warp == 1) {
        ptx::tmem_alloc(ptx::smem_u32(tmem_slot), 64);
        ptx::tmem_relinquish();
    }
    if (warp >= 4) {
        // rows of the q tile that no TMA box ever writes (G tq < 32) stay zero for the whole kernel
        for (int e = tid - 128; e < L::Q_BYTES / 16; e += 128)
            asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(sbase + (uint32_t)(L::OFF_Q + e * 16)), "r"(0) : "memory");
        ptx::fence_proxy_async_smem();
    }
    // Everything above touches only this CTA's shared memory, TMEM and the kernel parameters: under a programmatic
    // dependent launch it overlaps the tail of the previous kernel, and so does the register hand-over below (the budget
    // moves from the service warpgroup to the softmax warpgroup: 2 CTAs x (4 x 64 + 4 x 192) x 32 = the whole register file;
    // setmaxnreg opens each role's branch so that ptxas allocates the branch against its own budget).
    const bool base_ok = (sbase & 1023u) == 0u;               // the layout relies on a 1024-byte aligned base
    if (!base_ok && tid == 0) raise_flag(p.flags, DEV_INTERNAL | 0x800u);
    auto start = [&]() {                                      // executed by every warp, once, in its own branch
        ptx::pdl_wait();
        ptx::pdl_trigger();
        ptx::tc_fence_before();
        ptx::bar_sync(0, NTHREADS);
        ptx::tc_fence_after();
        return *tmem_slot;
    };
    uint32_t tmem;
    if (warp >= 4) {
        ptx::setmaxnreg_inc<192>();
        tmem = start();
        if (base_ok) softmax_warps<D>(p, smem, sbase, tmem, items, abort_flag, warp, lane);
    } else {
        ptx::setmaxnreg_dec<64>();
        tmem = start();
        if (base_ok && warp == 0) producer_warp<D>(p, &mapK, &mapV, &mapQ, smem, sbase, items, abort_flag, lane);
        else if (base_ok && warp == 1) mma_warp<D>(p, sbase, tmem, items, abort_flag, lane);
        else if (base_ok && warp == 2) agent_warp<D>(p, smem, sbase, items, abort_flag, lane);
    }
    ptx::tc_fence_before();
    __syncthreads();
    TRACE_CTA(1);
    if (tid == 0 && *abort_flag) raise_flag(p.flags, DEV_TIMEOUT);
    if (warp == 1) ptx::tmem_dealloc(tmem, 64);
}

}  // namespace dec

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
// Resident decode CTAs per SM; 0 on error.  Two CTAs fit by construction: 2 x (Smem::TOTAL + 1 KB reserved) <= 228 KB
// (static_assert above), 2 x 256 threads x 128 registers = the register file (checked here against the compiled kernel),
// 2 x 64 TMEM columns.  cudaOccupancyMaxActiveBlocksPerMultiprocessor answers 1 for this kernel (it does not model the
// setmaxnreg hand-over); the in-kernel trace shows both CTAs resident and running on every SM.
template <int D>
static inline int dec_configure_one() {
    cudaFuncAttributes fa;
    if (cudaFuncSetAttribute(dec::decode_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, dec::Smem<D>::TOTAL) != cudaSuccess) return 0;
    if (cudaFuncSetAttribute(dec::decode_kernel<D>, cudaFuncAttributePreferredSharedMemoryCarveout, 100) != cudaSuccess) return 0;
    if (cudaFuncGetAttributes(&fa, dec::decode_kernel<D>) != cudaSuccess) return 0;
    const bool two = fa.numRegs * dec::NTHREADS * 2 <= 65536 && 2 * (dec::Smem<D>::TOTAL + 1024) <= 233472 && fa.sharedSizeBytes == 0;
    return two ? 2 : 1;
}
static inline int dec_configure(int head_dim) {
    const int occ = head_dim == 128 ? dec_configure_one<128>() : dec_configure_one<64>();
#ifdef SANGAM_TUNING_ENV
    if (const char* f = getenv("SANGAM_DEC_OCC")) return atoi(f);
#endif
    return occ;
}

static inline cudaError_t dec_launch(const DecParams& p, const CUtensorMap& mk, const CUtensorMap& mv, const CUtensorMap& mq,
                                     int head_dim, int num_ctas, cudaStream_t stream) {
    cudaError_t e;
    if (head_dim == 128)
        e = launch_pdl(dec::decode_kernel<128>, dim3(num_ctas), dec::NTHREADS, dec::Smem<128>::TOTAL, stream, mk, mv, mq, p);
    else
        e = launch_pdl(dec::decode_kernel<64>, dim3(num_ctas), dec::NTHREADS, dec::Smem<64>::TOTAL, stream, mk, mv, mq, p);
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}
