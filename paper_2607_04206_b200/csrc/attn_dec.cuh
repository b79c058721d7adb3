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
// Small CTAs, two per SM (192 threads, 113 KB shared memory, 64 TMEM columns): one CTA's fill / drain / epilogue
// overlaps the other's main loop.  Warp roles: 0 = device-side plan (a3) + TMA producer (a4), 1 = MMA issuer
// (a5, a7), 2..5 = softmax (a6), epilogue (a8) and the fused split-KV merge (a9).
// Work unit = (request r, kv head g, chunk of 32/G query tokens); the flattened (unit, page) sequence, each unit
// weighted with a fixed overhead, is cut into #CTA equal contiguous ranges at PAGE granularity (stream-K): at most two
// partial pieces per CTA.  Pieces of a split unit go to the workspace as (O^T fp32, m, l); the CTA that finishes a
// unit's last piece merges all of them in fixed piece order (bitwise reproducible) -- no second kernel.
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "ptx.cuh"

struct DecParams {
    const int32_t* block_table;    // [batch][W]
    const int32_t* cu_q_lens;      // [batch+1]
    const int32_t* ctx_lens;       // [batch]
    __nv_bfloat16* out;            // [total_q][Hq][D]
    int32_t batch, total_q;
    int32_t Hq, Hkv, G, W, P;
    int32_t tq;                    // query tokens per unit = 32 / G
    uint32_t tq_magic;             // floor(2^32 / tq) + 1: x / tq = umulhi(x, magic) for x < 2^24
    float scale_log2;              // scale * log2(e)
    float* part_o;                 // [2 #CTAs][32][D]  unnormalised partial O (row-major per piece)
    float* part_ml;                // [2 #CTAs][32][2]  (m in log2 units, l)
    int32_t* piece_cnt;            // [#CTAs] arrivals per split unit, indexed by the CTA of its head piece; self-resetting
    uint32_t* flags;               // sticky device flags
};

namespace dec {

constexpr int BN = 128;          // kv positions per tile (UMMA M; 8 pages)
constexpr int NQ = 32;           // packed query rows per unit (UMMA N)
constexpr int NSTAGE = 3;        // ring of K / V tiles
constexpr int NTHREADS = 192;
#ifndef SANGAM_DEC_OV
#define SANGAM_DEC_OV 12
#endif
constexpr int OV = SANGAM_DEC_OV;  // fixed cost of starting / finishing a unit, in pages (stream-K weight)
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
    int b_head;        // split units: CTA holding the piece that starts at page 0
    int npieces;       // split units: number of CTAs holding a piece
    int pad0, pad1, pad2, pad3;
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
                         B_P_FULL = B_S_FULL + 1, B_P_EMPTY = B_P_FULL + 1, B_O_FREE = B_P_EMPTY + 1, NBAR = B_O_FREE + 1;
    static constexpr int OFF_ITEMS = OFF_BAR + 128;
    static constexpr int OFF_WM = OFF_ITEMS + 2 * (int)sizeof(Item);   // [4 warps][32] floats: per-warp column maxima / sums
    static constexpr int OFF_MISC = OFF_WM + 4 * 32 * 4;               // tmem slot, abort word, merge flag, wait table
    static constexpr int TOTAL = OFF_MISC + 96;
    static_assert(NBAR * 8 <= 128, "barrier block");
};
// two CTAs per SM: 2 x (TOTAL + 1 KB reserved) <= 228 KB; the dynamic shared memory base is 1024-byte aligned
// (no static shared memory in this kernel; checked at run time)
static_assert(Smem<128>::TOTAL <= 115712, "two CTAs per SM");

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
    x.chunks = (int)__umulhi((uint32_t)(qn + p.tq - 1), p.tq_magic);
    x.units = p.Hkv * x.chunks;
    x.pages = (c + SANGAM_PAGE - 1) / SANGAM_PAGE;
    x.w = (x.pages > 0 ? x.pages : 1) + OV;                // an empty context still needs one visit (zero rows)
    return x;
}

// floor(b T / Geff) with T = qT Geff + rT, exactly, in 32-bit arithmetic (b rT < 2^31: Geff <= 2^10 CTAs)
__device__ __forceinline__ int cut(int b, int T, int Geff, int qT, int rT) {
    if (b >= Geff) return T;
    return b * qT + (int)(((uint32_t)b * (uint32_t)rT) / (uint32_t)Geff);
}
// the CTA whose range [cut(b), cut(b+1)) holds coordinate y
__device__ __forceinline__ int owner(int y, int T, int Geff, int qT, int rT) {
    int b = (int)((float)y * (float)Geff / (float)T);
    b = b < 0 ? 0 : (b > Geff - 1 ? Geff - 1 : b);
    while (b > 0 && cut(b, T, Geff, qT, rT) > y) --b;
    while (b < Geff - 1 && cut(b + 1, T, Geff, qT, rT) <= y) ++b;
    return b;
}

// ------------------------------------------------------------------------------------------------
// warp 0: device-side plan (a3) + TMA page gather (a4) + Q loads
// ------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void producer_warp(const DecParams& p, const CUtensorMap* mapK, const CUtensorMap* mapV,
                                              const CUtensorMap* mapQ, uint32_t sbase, Item* items,
                                              volatile uint32_t* abort_flag, int lane) {
    using L = Smem<D>;
    const unsigned FULL = 0xffffffffu;
    const int NC = gridDim.x, b = blockIdx.x, R = p.batch;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };

    // lane r keeps request r (< 32) in registers; later look-ups are shuffles
    int rq0 = 0, rqn = 0, rc = 0;
    if (lane < R) load_req(p, lane, rq0, rqn, rc);
    auto get = [&](int r) {                                  // warp-uniform r
        int a, q, c;
        if (r < 32) { a = __shfl_sync(FULL, rq0, r); q = __shfl_sync(FULL, rqn, r); c = __shfl_sync(FULL, rc, r); }
        else load_req(p, r, a, q, c);
        return derive(p, a, q, c);
    };
    auto get_lane = [&](int base) {                          // per-lane r = base + lane (< R)
        if (base == 0) return derive(p, rq0, rqn, rc);
        int a, q, c;
        load_req(p, base + lane, a, q, c);
        return derive(p, a, q, c);
    };
    int T = 0;
    for (int base = 0; base < R; base += 32)
        if (base + lane < R) { const ReqInfo x = get_lane(base); T += x.units * x.w; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) T += __shfl_xor_sync(FULL, T, o);

    const int Geff = NC < T ? NC : T;
    int qT = 0, rT = 0, remaining = 0, r_cur = R, u_in_r = 0, off = 0, unit_base = 0;
    ReqInfo cur = derive(p, 0, 0, 0);
    if (b < Geff) {
        qT = T / Geff; rT = T - qT * Geff;
        const int x0 = cut(b, T, Geff, qT, rT), x1 = cut(b + 1, T, Geff, qT, rT);
        remaining = x1 - x0;
        // locate the request holding coordinate x0 (chunked warp scan over requests)
        int acc = 0, found = -1, req_base = 0;
        for (int base = 0; base < R && found < 0; base += 32) {
            int tl = 0;
            if (base + lane < R) { const ReqInfo x = get_lane(base); tl = x.units * x.w; }
            int incl = tl;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int v = __shfl_up_sync(FULL, incl, o);
                if (lane >= o) incl += v;
            }
            const unsigned m = __ballot_sync(FULL, acc + incl > x0);
            if (m) {
                const int l = __ffs(m) - 1;
                found = base + l;
                req_base = acc + __shfl_sync(FULL, incl - tl, l);
            } else {
                acc += __shfl_sync(FULL, incl, 31);
            }
        }
        if (found >= 0) {
            r_cur = found;
            cur = get(r_cur);
            const int pos = x0 - req_base;
            u_in_r = pos / cur.w;
            off = pos - u_in_r * cur.w;
            unit_base = req_base + u_in_r * cur.w;
        } else {
            remaining = 0;
        }
    }

    uint32_t stage = 0, phase = 0, icount = 0, qcount = 0;
    while (true) {
        if (*abort_flag) break;
        Item it;
        it.valid = 0; it.r = 0; it.g = 0; it.tok0 = 0; it.ntok = 0; it.q_start = 0; it.c = 0; it.pg0 = 0; it.pg1 = 0;
        it.part_slot = -1; it.b_head = 0; it.npieces = 1; it.pad0 = 0; it.pad1 = 0; it.pad2 = 0; it.pad3 = 0;
        // this CTA owns the weighted coordinates [x0, x1) of the flattened unit list; a unit spans OV + max(pages, 1)
        // of them, coordinate OV + j being its page j.  A range covering only overhead coordinates yields no work there.
        while (remaining > 0 && r_cur < R && !it.valid) {
            const int take = remaining < cur.w - off ? remaining : cur.w - off;
            const int a = off > OV ? off - OV : 0, e = off + take > OV ? off + take - OV : 0;
            if (e > a) {
                const int g = cur.chunks == 1 ? u_in_r : u_in_r / cur.chunks;
                const int ch = u_in_r - g * cur.chunks;
                it.valid = 1; it.r = r_cur; it.g = g;
                it.tok0 = ch * p.tq;
                const int left = cur.qn - it.tok0;
                it.ntok = left < p.tq ? left : p.tq;
                it.q_start = cur.q0; it.c = cur.c;
                it.pg0 = a; it.pg1 = e < cur.pages ? e : cur.pages;      // empty context: pages = 0 -> no tiles
                if (!(a == 0 && e == cur.w - OV)) {                       // a piece of a unit split across CTAs
                    it.part_slot = 2 * b + (a == 0 ? 1 : 0);
                    const int bh = owner(unit_base + OV, T, Geff, qT, rT);
                    const int bl = owner(unit_base + cur.w - 1, T, Geff, qT, rT);
                    it.b_head = bh;
                    it.npieces = bl - bh + 1;
                }
            }
            remaining -= take;
            off += take;
            if (off == cur.w) {
                off = 0;
                unit_base += cur.w;
                if (++u_in_r == cur.units) {
                    u_in_r = 0;
                    do {
                        ++r_cur;
                        if (r_cur < R) cur = get(r_cur);
                    } while (r_cur < R && cur.units == 0);
                }
            }
        }
        // publish
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_EMPTY + islot), ((icount >> 1) & 1u) ^ 1u, abort_flag);
        if (lane == 0) {
            items[islot] = it;
            ptx::mbar_arrive(bar(L::B_ITEM_FULL + islot));
        }
        __syncwarp();
        ++icount;
        if (!it.valid) break;

        const int npg = it.pg1 - it.pg0;
        if (npg > 0) {
            // the unit's query rows: one TMA box (64 columns, G heads, tq tokens) per 64-column slab
            ptx::mbar_wait(bar(L::B_Q_EMPTY), (qcount & 1u) ^ 1u, abort_flag);
            if (lane == 0) ptx::mbar_arrive_expect_tx(bar(L::B_Q_FULL), (uint32_t)(p.G * p.tq * D * 2));
            __syncwarp();
            if (lane < D / 64)
                ptx::tma_load_3d(sbase + (uint32_t)(L::OFF_Q + lane * L::QSLAB), mapQ, bar(L::B_Q_FULL), lane * 64, it.g * p.G,
                                 it.q_start + it.tok0);
            ++qcount;
            // K / V tiles in ring order K(0) V(0) K(1) V(1) ...; one TMA box per page, lanes 0..7 issue;
            // the page ids of the next tile are requested while this tile's boxes are issued
            const int32_t* bt = p.block_table + (int64_t)it.r * p.W + it.pg0;
            const int nt = (npg + 7) >> 3;
            int page = (lane < 8 && lane < npg) ? __ldg(bt + lane) : 0;
            for (int t = 0; t < nt; ++t) {
                int np = npg - 8 * t;
                np = np > 8 ? 8 : np;
                const int nxt = (lane < 8 && 8 * (t + 1) + lane < npg) ? __ldg(bt + 8 * (t + 1) + lane) : 0;
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
                }
                page = nxt;
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
    const unsigned FULL = 0xffffffffu;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    const int qd = warp & 3, jl = qd * 32 + lane;
    const uint32_t lane_base = (uint32_t)(qd * 32) << 16;
    const uint32_t s_taddr = tmem + lane_base, o_taddr = tmem + lane_base + 32u;
    float* wm = reinterpret_cast<float*>(smem + L::OFF_WM);
    volatile int* merge_flag = reinterpret_cast<volatile int*>(smem + L::OFF_MISC + 8);
    // P^T[row c][kv jl] in the K-major 128B-swizzled B-operand layout: slab = jl / 64, 16-byte chunk (jl % 64) / 8 XOR (c % 8)
    uint32_t pa[8];
#pragma unroll
    for (int k = 0; k < 8; ++k)
        pa[k] = sbase + (uint32_t)(L::OFF_P + (jl >> 6) * 4096 + k * 128 + ((((jl & 63) >> 3) ^ k) << 4) + (jl & 7) * 2);
    const float sc = fabsf(p.scale_log2);
    const bool neg = p.scale_log2 < 0.f;
    uint32_t icount = 0, tcount = 0;       // items seen; kv tiles seen (S_FULL / P_EMPTY phases)
    while (true) {
        if (*abort_flag) break;
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_FULL + islot), (icount >> 1) & 1u, abort_flag);
        const Item it = items[islot];
        if (!it.valid) break;
        const int npg = it.pg1 - it.pg0, nt = (npg + 7) >> 3;
        const int c_lim = it.c < it.pg1 * SANGAM_PAGE ? it.c : it.pg1 * SANGAM_PAGE;
        float m_ref[32], lp[32];
#pragma unroll
        for (int c = 0; c < 32; ++c) { m_ref[c] = -INFINITY; lp[c] = 0.f; }
        float m_own = -INFINITY;               // m_ref[lane]
        for (int t = 0; t < nt; ++t) {
            if (*abort_flag) break;
            const bool valid = (it.pg0 + 8 * t) * SANGAM_PAGE + jl < c_lim;
            ptx::mbar_wait(bar(L::B_S_FULL), tcount & 1u, abort_flag);
            ptx::tc_fence_after();
            uint32_t s[32];
            ptx::tmem_ld32(s_taddr, s);
            ptx::tmem_wait_ld();
            if (neg) {                          // rare: scale < 0 -- work on -s with |scale|
#pragma unroll
                for (int c = 0; c < 32; ++c) s[c] ^= 0x80000000u;
            }
            if (!valid) {
#pragma unroll
                for (int c = 0; c < 32; ++c) s[c] = 0xff800000u;    // -inf: positions past the context
            }
            {   // column maxima over the tile's 128 positions: warp redux, then one exchange through shared memory
                float wx[32];
#pragma unroll
                for (int c = 0; c < 32; ++c) wx[c] = ptx::redux_max(__uint_as_float(s[c]));
                if (lane == 0) {
                    float4* dst = reinterpret_cast<float4*>(wm + qd * 32);
#pragma unroll
                    for (int k = 0; k < 8; ++k) dst[k] = make_float4(wx[4 * k], wx[4 * k + 1], wx[4 * k + 2], wx[4 * k + 3]);
                }
            }
            ptx::bar_sync(1, 128);
            const float cm = fmaxf(fmaxf(wm[lane], wm[32 + lane]), fmaxf(wm[64 + lane], wm[96 + lane])) * sc;
            const bool grow = cm > m_own + LAZY_T;
            bool p_free = false;
            if (__any_sync(FULL, grow)) {
                // the reference maximum of some row moves (always in a unit's first tile, rarely later):
                // l and O^T shrink by alpha = 2^(m_old - m_new) in those rows
                const float m_new = grow ? cm : m_own;
                const float a_own = grow ? ptx::ex2(m_own - m_new) : 1.f;
                m_own = m_new;
                float al[32];
#pragma unroll
                for (int c = 0; c < 32; ++c) {
                    m_ref[c] = __shfl_sync(FULL, m_new, c);
                    al[c] = __shfl_sync(FULL, a_own, c);
                    lp[c] *= al[c];
                }
                if (t > 0) {
                    ptx::mbar_wait(bar(L::B_P_EMPTY), (tcount - 1u) & 1u, abort_flag);    // every PV so far has landed in O^T
                    p_free = true;
                    ptx::tc_fence_after();
                    uint32_t o[32];
                    ptx::tmem_ld32(o_taddr, o);
                    ptx::tmem_wait_ld();
#pragma unroll
                    for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * al[c]);
                    ptx::tmem_st32(o_taddr, o);
                    ptx::tmem_wait_st();
                }
            }
            uint32_t pk[16];
#pragma unroll
            for (int c = 0; c < 32; c += 2) {
                float p0 = ptx::ex2(fmaf(__uint_as_float(s[c]), sc, -m_ref[c]));
                float p1 = ptx::ex2(fmaf(__uint_as_float(s[c + 1]), sc, -m_ref[c + 1]));
                if (!valid) { p0 = 0.f; p1 = 0.f; }            // also covers scale = 0 (-inf * 0)
                lp[c] += p0; lp[c + 1] += p1;
                pk[c >> 1] = ptx::pack_bf16(p0, p1);
            }
            if (!p_free && tcount > 0) ptx::mbar_wait(bar(L::B_P_EMPTY), (tcount - 1u) & 1u, abort_flag);   // the previous PV has read P^T
#pragma unroll
            for (int c = 0; c < 32; c += 2)
                ptx::sts_bf16_pair(pa[c & 7] + (uint32_t)((c >> 3) * 1024), pa[(c + 1) & 7] + (uint32_t)((c >> 3) * 1024), pk[c >> 1]);
            ptx::fence_proxy_async_smem();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(L::B_P_FULL));
            ++tcount;
        }
        // ---------------- epilogue
        if (nt > 0) {
            ptx::mbar_wait(bar(L::B_P_EMPTY), (tcount - 1u) & 1u, abort_flag);
            ptx::tc_fence_after();
        }
        const float ls = column_sums(lp, lane);
        wm[qd * 32 + lane] = ls;
        ptx::bar_sync(1, 128);
        const float l_own = (wm[lane] + wm[32 + lane]) + (wm[64 + lane] + wm[96 + lane]);   // fixed order
        ptx::bar_sync(1, 128);                  // wm is rewritten by the next tile / item
        const int rows = it.ntok * p.G;          // packed rows (token * G + head) that exist
        const int64_t out_base = ((int64_t)(it.q_start + it.tok0) * p.Hq + (int64_t)it.g * p.G) * D + jl;
        const bool tok_ok = it.q_start + it.tok0 >= 0 && it.q_start + it.tok0 + it.ntok <= p.total_q && (unsigned)it.g < (unsigned)p.Hkv;
        if (!tok_ok && lane == 0) raise_flag(p.flags, DEV_INTERNAL | 0x400u);
        const bool d_ok = jl < D && tok_ok;
        // row c = token tl * G + head hh  ->  out[(q_start + tok0 + tl)][g G + hh][d]
        auto store_rows = [&](const float (&f)[32]) {
            int tl = 0, hh = 0;
#pragma unroll
            for (int c = 0; c < 32; ++c) {
                if (d_ok && c < rows) p.out[out_base + ((int64_t)tl * p.Hq + hh) * D] = __float2bfloat16_rn(f[c]);
                if (++hh == p.G) { hh = 0; ++tl; }
            }
        };
        if (nt == 0) {
            if (it.part_slot < 0) {             // empty context: zero rows (reading S13); never split
                float z[32];
#pragma unroll
                for (int c = 0; c < 32; ++c) z[c] = 0.f;
                store_rows(z);
            }
        } else {
            uint32_t o[32];
            ptx::tmem_ld32(o_taddr, o);
            ptx::tmem_wait_ld();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(L::B_O_FREE));      // the next unit's first PV may overwrite O^T
            float f[32];
            if (it.part_slot < 0) {
                const float inv_own = l_own > 0.f ? 1.f / l_own : 0.f;
#pragma unroll
                for (int c = 0; c < 32; ++c) f[c] = __uint_as_float(o[c]) * __shfl_sync(FULL, inv_own, c);
                store_rows(f);
            } else {
                // a piece of a split unit: (O^T unnormalised, m, l) to the workspace, then count arrivals; the CTA that
                // brings the last piece merges all of them in piece order
                const bool slot_ok = it.part_slot < 2 * (int)gridDim.x && it.b_head >= 0 && it.b_head + it.npieces <= (int)gridDim.x && it.npieces >= 1;
                if (!slot_ok && lane == 0) raise_flag(p.flags, DEV_INTERNAL | 0x100u);
                if (slot_ok) {
                    float* po = p.part_o + ((int64_t)it.part_slot * NQ) * D + jl;
                    if (jl < D) {
#pragma unroll
                        for (int c = 0; c < 32; ++c) po[c * D] = __uint_as_float(o[c]);
                    }
                    if (qd == 0) reinterpret_cast<float2*>(p.part_ml)[it.part_slot * NQ + lane] = make_float2(m_own, l_own);
                }
                __threadfence();
                ptx::bar_sync(1, 128);
                if (qd == 0 && lane == 0) {
                    int last = 0;
                    if (slot_ok) last = atomicAdd(p.piece_cnt + it.b_head, 1) == it.npieces - 1;
                    *merge_flag = last;
                }
                ptx::bar_sync(1, 128);
                const bool merge = *merge_flag != 0;
                ptx::bar_sync(1, 128);           // merge_flag is rewritten by the next split item
                if (merge) {
                    __threadfence();
                    const float2* ml = reinterpret_cast<const float2*>(p.part_ml);
                    float M[32], Lsum[32];
#pragma unroll
                    for (int c = 0; c < 32; ++c) { M[c] = -INFINITY; Lsum[c] = 0.f; f[c] = 0.f; }
                    for (int pi = 0; pi < it.npieces; ++pi) {
                        const int slot = pi == 0 ? 2 * it.b_head + 1 : 2 * (it.b_head + pi);
                        const float4* src = reinterpret_cast<const float4*>(ml + slot * NQ);
#pragma unroll
                        for (int c2 = 0; c2 < 16; ++c2) {
                            const float4 x = __ldcg(src + c2);
                            M[2 * c2] = fmaxf(M[2 * c2], x.x); M[2 * c2 + 1] = fmaxf(M[2 * c2 + 1], x.z);
                        }
                    }
                    for (int pi = 0; pi < it.npieces; ++pi) {
                        const int slot = pi == 0 ? 2 * it.b_head + 1 : 2 * (it.b_head + pi);
                        const float4* src = reinterpret_cast<const float4*>(ml + slot * NQ);
                        const float* so = p.part_o + ((int64_t)slot * NQ) * D + (jl < D ? jl : 0);
                        float w[32];
#pragma unroll
                        for (int c2 = 0; c2 < 16; ++c2) {
                            const float4 x = __ldcg(src + c2);
                            w[2 * c2] = ptx::ex2(x.x - M[2 * c2]); w[2 * c2 + 1] = ptx::ex2(x.z - M[2 * c2 + 1]);
                            Lsum[2 * c2] = fmaf(x.y, w[2 * c2], Lsum[2 * c2]); Lsum[2 * c2 + 1] = fmaf(x.w, w[2 * c2 + 1], Lsum[2 * c2 + 1]);
                        }
#pragma unroll
                        for (int c = 0; c < 32; ++c) f[c] = fmaf(__ldcg(so + c * D), w[c], f[c]);
                    }
#pragma unroll
                    for (int c = 0; c < 32; ++c) f[c] *= Lsum[c] > 0.f ? 1.f / Lsum[c] : 0.f;
                    store_rows(f);
                    if (qd == 0 && lane == 0) p.piece_cnt[it.b_head] = 0;     // re-arm for the next launch
                }
            }
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar(L::B_ITEM_EMPTY + islot));
        ++icount;
    }
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
    volatile uint32_t* abort_flag = reinterpret_cast<volatile uint32_t*>(smem + L::OFF_MISC + 4);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
        for (int s = 0; s < NSTAGE; ++s) { ptx::mbar_init(bar(L::B_KV_FULL + s), 1); ptx::mbar_init(bar(L::B_KV_EMPTY + s), 1); }
        for (int s = 0; s < 2; ++s) { ptx::mbar_init(bar(L::B_ITEM_FULL + s), 1); ptx::mbar_init(bar(L::B_ITEM_EMPTY + s), 5); }   // MMA warp + 4 softmax warps
        ptx::mbar_init(bar(L::B_Q_FULL), 1); ptx::mbar_init(bar(L::B_Q_EMPTY), 1);
        ptx::mbar_init(bar(L::B_S_FULL), 1);
        ptx::mbar_init(bar(L::B_P_FULL), 4); ptx::mbar_init(bar(L::B_P_EMPTY), 1);
        ptx::mbar_init(bar(L::B_O_FREE), 4);
        for (int k = 1; k < 24; ++k) tmem_slot[k] = 0u;        // abort word, merge flag, wait table
        ptx::fence_mbar_init();
        ptx::prefetch_tensormap(&mapK);
        ptx::prefetch_tensormap(&mapV);
        ptx::prefetch_tensormap(&mapQ);
    }
    if (warp == 1) {
        ptx::tmem_alloc(ptx::smem_u32(tmem_slot), 64);
        ptx::tmem_relinquish();
    }
    if (warp >= 2) {
        // rows of the q tile that no TMA box ever writes (G tq < 32) stay zero for the whole kernel
        for (int e = tid - 64; e < L::Q_BYTES / 16; e += 128)
            asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(sbase + (uint32_t)(L::OFF_Q + e * 16)), "r"(0) : "memory");
        ptx::fence_proxy_async_smem();
    }
    // everything above touches only this CTA's shared memory, TMEM and the kernel parameters (programmatic dependent launch)
    ptx::pdl_wait();
    ptx::pdl_trigger();
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    if ((sbase & 1023u) != 0u) {                              // the layout relies on a 1024-byte aligned base
        if (tid == 0) raise_flag(p.flags, DEV_INTERNAL | 0x800u);
    } else if (warp == 0) {
        producer_warp<D>(p, &mapK, &mapV, &mapQ, sbase, items, abort_flag, lane);
    } else if (warp == 1) {
        mma_warp<D>(p, sbase, tmem, items, abort_flag, lane);
    } else {
        softmax_warps<D>(p, smem, sbase, tmem, items, abort_flag, warp, lane);
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (tid == 0 && *abort_flag) raise_flag(p.flags, DEV_TIMEOUT);
    if (warp == 1) ptx::tmem_dealloc(tmem, 64);
}

}  // namespace dec

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
// resident decode CTAs per SM (2 when shared memory allows); 0 on error
static inline int dec_configure(int head_dim) {
    cudaError_t e;
    int occ = 0;
    if (head_dim == 128) {
        e = cudaFuncSetAttribute(dec::decode_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, dec::Smem<128>::TOTAL);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, dec::decode_kernel<128>, dec::NTHREADS, dec::Smem<128>::TOTAL);
    } else {
        e = cudaFuncSetAttribute(dec::decode_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, dec::Smem<64>::TOTAL);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, dec::decode_kernel<64>, dec::NTHREADS, dec::Smem<64>::TOTAL);
    }
    if (e != cudaSuccess) return 0;
    return occ > 2 ? 2 : occ;
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
