// attn_gqa.cuh -- steps a3..a9 for DECODE-shaped batches of GQA models: paged, varlen, non-causal block attention on
// tcgen05 (sm_100a) with CTA PAIRS sharing every K/V tile through TMA multicast.
//
// A GQA block decode packs (tokens x G heads) query rows per kv head -- 224 rows for a 32-token block at 7:1 (Dream-7B,
// PAPER.md:315) -- i.e. two 128-row q tiles that need the same K/V stream.  One CTA holding both tiles makes
// the SM's tensor pipe, MUFU and shared memory all co-critical with its share of HBM (the shape sits at
// the ridge).  Here a CLUSTER of two CTAs (two SMs) owns a unit: CTA c computes q tile c, and each K/V tile is loaded ONCE
// from L2 -- CTA c fetches half of its pages -- and multicast into both CTAs' shared memory.  Per SM and kv tile that
// leaves one 128x128 QK^T, one PV and 16 K exponentials against 32 KB of HBM traffic: every pipe has slack again and
// HBM is the only bound.
//
// Per CTA: 384 threads; warp 0 = device-side plan (a3) + TMA producer (a4), 1 = MMA issuer (a5, a7), 2 = arrival agent of
// split units, 4..7 and 8..11 = two softmax warpgroups (a6: thread i of a group owns row i of the CTA's q tile).  The kv
// tiles of a unit alternate between the groups (stream b takes the tiles of parity b, with its own S buffer, its own
// running (max, sum) and its own O accumulator in TMEM; the two partial results are merged in the epilogue): one warp
// per SM sub-partition cannot hide the TMEM / MUFU latencies of a tile's 128 exponentials per row, two can.  Group 0
// also runs the epilogue (a8) and the fused split-KV merge (a9).  Work unit = (request, kv head, pair of q tiles); the flattened (unit, page) list is cut into one contiguous range
// per CLUSTER (stream-K, the planner of attn_dec.cuh); both CTAs of a cluster derive the same plan and walk it in
// lockstep (a K/V stage is refilled only after both CTAs released it).  Pieces of split units are merged by the piece
// that arrives last, as in attn_dec.cuh.
#pragma once
#include <cuda.h>

#include "attn_dec.cuh"
#include "common.cuh"
#include "ptx.cuh"

namespace gqa {

using dec::Deferred;
using dec::Item;
using dec::OutRef;
using dec::Planner;

constexpr int BM = 128;          // rows of a q tile (UMMA M)
constexpr int BN = 128;          // kv positions per tile (8 pages)
constexpr int NK = 3;            // stages of the K ring
constexpr int NV = 3;            // stages of the V ring (separate rings with an issuing warp each: a V tile is held until its
                                 // softmax has been multiplied in, much longer than a K tile)
constexpr int NTHREADS = 384;
constexpr float LAZY_T = 8.f;
#ifndef SANGAM_GQA_OV
#define SANGAM_GQA_OV 16
#endif
constexpr int OV = SANGAM_GQA_OV;   // fixed cost of starting / finishing a unit, in pages (stream-K weight)
constexpr int MIN_W = 64;           // smallest share of the weighted unit list given to a cluster
template <int D> constexpr int KV_ATOM_STRIDE = 1024 * (D / 64);
// TMEM columns: Q (bf16 pairs, D / 2 columns) at 0, S[j] at 64 + 128 j (j = 0, 1), O at 320
constexpr uint32_t TM_Q = 0u, TM_S = 64u, TM_O = 320u;

template <int D>
struct Smem {
    static constexpr int KV_BYTES = BN * D * 2;
    static constexpr int OFF_KV = 0;                     // stages 0 .. NK-1: K ring, NK .. NK+NV-1: V ring
    static constexpr int OFF_BAR = (NK + NV) * KV_BYTES;
    static constexpr int B_KV_FULL = 0, B_KV_EMPTY = NK + NV, B_ITEM_FULL = 2 * (NK + NV), B_ITEM_EMPTY = B_ITEM_FULL + 2,
                         B_Q_FULL = B_ITEM_EMPTY + 2, B_Q_EMPTY = B_Q_FULL + 1, B_S_FULL = B_Q_EMPTY + 1 /* [tile parity] */,
                         B_P_FULL = B_S_FULL + 2 /* [tile parity] */, B_PV_DONE = B_P_FULL + 2 /* [tile parity] */, B_O_FREE = B_PV_DONE + 2,
                         B_EPI = B_O_FREE + 1 /* [item slot] */, B_AGENT_REQ = B_EPI + 2, B_AGENT_DONE = B_AGENT_REQ + 1, NBAR = B_AGENT_DONE + 1;
    static constexpr int OFF_ITEMS = OFF_BAR + ((NBAR * 8 + 15) / 16) * 16;
    static constexpr int OFF_ML = OFF_ITEMS + 2 * (int)sizeof(Item);     // [2 item slots][128 rows] row sum of group 1's half
    static constexpr int OFF_MX = OFF_ML + 2 * BM * 4;                   // [2 tile parities][2 groups][128 rows] half-tile row maxima
    // misc block: +0 tmem slot, +8 merge flag, +16 agent_req[2], +32 Deferred[2], +96 abort word (+ wait table in debug builds)
    static constexpr int OFF_MISC = OFF_MX + 4 * BM * 4;
    static constexpr int OFF_ABORT = OFF_MISC + 96;
    static constexpr int TOTAL = OFF_ABORT + 80;
    static constexpr int ALLOC = TOTAL;                  // no alignment slack: the dynamic base is 1024-byte aligned (checked at run time)
};
static_assert(Smem<128>::ALLOC <= 232448, "shared memory budget (227 KB)");

__device__ __forceinline__ uint32_t cluster_rank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// the same shared-memory offset in the peer CTA of the cluster (shared::cluster address)
__device__ __forceinline__ uint32_t peer_addr(uint32_t local, uint32_t peer) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local), "r"(peer));
    return r;
}
// one (page, head) box into BOTH CTAs of the pair: same offset, each CTA's own barrier gets the bytes
__device__ __forceinline__ void tma_load_4d_mc(uint32_t dst_smem, const CUtensorMap* m, uint32_t bar, int32_t c3, uint16_t mask) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%3, %3, %3, %4}], [%2], %5;"
        ::"r"(dst_smem), "l"(reinterpret_cast<uint64_t>(m)), "r"(bar), "r"(0), "r"(c3), "h"(mask)
        : "memory");
}

// ------------------------------------------------------------------------------------------------
// warp 0: plan + TMA (this CTA's half of every tile's pages, multicast to the pair) + its q tile
// ------------------------------------------------------------------------------------------------
// One unit's kv tiles of one ring (K or V), this CTA's half of every tile multicast to both CTAs of the pair.
// Page ids come in 64-page windows, lane l holding entries l and 32 + l; the window after the current one is requested when
// the current one is entered, eight tiles before it is needed: no load waits on a block-table read except the unit's first.
template <int D>
__device__ __forceinline__ void load_tiles(const DecParams& p, const CUtensorMap* map, uint32_t sbase, const Item& it, uint32_t rank, int lane,
                                           uint32_t ring0, uint32_t nstage, uint32_t& st, uint32_t& ph, volatile uint32_t* abort_flag,
                                           [[maybe_unused]] unsigned& dt_i_) {
    using L = Smem<D>;
    const unsigned FULL = 0xffffffffu;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    const int npg = it.pg1 - it.pg0, nt = (npg + 7) >> 3;
    const int32_t* bt = p.block_table + (int64_t)it.r * p.W + it.pg0;
    auto ld_win = [&](int w, int half) { const int e = 64 * w + 32 * half + lane; return e < npg ? __ldg(bt + e) : 0; };
    int clo = ld_win(0, 0), chi = ld_win(0, 1), nlo = ld_win(1, 0), nhi = ld_win(1, 1);
    const bool my_lane = (lane >> 2) == (int)rank && lane < 8;                // pages 0..3 of a tile: CTA 0, pages 4..7: CTA 1
    const uint32_t dst0 = sbase + (uint32_t)(L::OFF_KV + lane * (2 * KV_ATOM_STRIDE<D>));
    for (int t = 0; t < nt; ++t) {
        const int tw = t & 7;
        if (tw == 0 && t > 0) { clo = nlo; chi = nhi; nlo = ld_win((t >> 3) + 1, 0); nhi = ld_win((t >> 3) + 1, 1); }
        const int src = (8 * tw + lane) & 31;
        const int xlo = __shfl_sync(FULL, clo, src), xhi = __shfl_sync(FULL, chi, src);
        int page = tw < 4 ? xlo : xhi;
        int np = npg - 8 * t;
        np = np > 8 ? 8 : np;
        const bool mine = my_lane && lane < np;
        if (mine && (unsigned)page >= (unsigned)p.P) { raise_flag(p.flags, DEV_BAD_PAGE); page = p.P; }
        const uint32_t stage = ring0 + st;
        DT((ring0 ? 200 : 180) + (t & 15));
        ptx::mbar_wait(bar(L::B_KV_EMPTY + stage), ph ^ 1u, abort_flag);      // both CTAs have released the stage
        if (lane == 0) ptx::mbar_arrive_expect_tx(bar(L::B_KV_FULL + stage), (uint32_t)(np * SANGAM_PAGE * D * 2));
        __syncwarp();
        if (mine) tma_load_4d_mc(dst0 + stage * L::KV_BYTES, map, bar(L::B_KV_FULL + stage), (page * p.Hkv + it.g) * 2, (uint16_t)3);
        if (++st == nstage) { st = 0; ph ^= 1u; }
        DT((ring0 ? 120 : 100) + (t & 15));
        if (*abort_flag) break;
    }
}

// warp 0: device-side plan (a3), the K ring
template <int D>
__device__ __forceinline__ void producer_warp(const DecParams& p, const CUtensorMap* mapK, uint32_t sbase, Item* items,
                                              volatile uint32_t* abort_flag, int lane, uint32_t rank) {
    using L = Smem<D>;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    DT_DECL;
    DT(1);
    Planner plan;
    plan.init(p, lane, (int)gridDim.x >> 1, (int)blockIdx.x >> 1);
    DT(2);
    uint32_t kst = 0, kph = 0, icount = 0;
    while (true) {
        if (*abort_flag) break;
        Item it;
        plan.next(p, it);
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_EMPTY + islot), ((icount >> 1) & 1u) ^ 1u, abort_flag);
        if (lane == 0) {
            items[islot] = it;
            ptx::mbar_arrive(bar(L::B_ITEM_FULL + islot));
        }
        __syncwarp();
        ++icount;
        if (!it.valid) break;
        if (it.pg1 - it.pg0 <= 0) continue;
        load_tiles<D>(p, mapK, sbase, it, rank, lane, 0u, (uint32_t)NK, kst, kph, abort_flag, dt_i_);
    }
    for (int k = 0; k < NK; ++k) {          // every commit aimed at this CTA's barriers has landed before it may exit
        ptx::mbar_wait(bar(L::B_KV_EMPTY + kst), kph ^ 1u, abort_flag);
        if (++kst == NK) { kst = 0; kph ^= 1u; }
    }
}

// warp 3: the V ring (a ring and an issuing warp of its own: a V tile is needed a whole softmax later than its K tile, and one
// warp's instruction stream cannot issue both rings at the rate HBM delivers them)
template <int D>
__device__ __forceinline__ void v_producer_warp(const DecParams& p, const CUtensorMap* mapV, uint32_t sbase, const Item* items,
                                                volatile uint32_t* abort_flag, int lane, uint32_t rank) {
    using L = Smem<D>;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    DT_DECL;
    uint32_t vst = 0, vph = 0, icount = 0;
    while (true) {
        if (*abort_flag) break;
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_FULL + islot), (icount >> 1) & 1u, abort_flag);
        const Item it = items[islot];
        if (!it.valid) break;
        if (it.pg1 - it.pg0 > 0) {
            load_tiles<D>(p, mapV, sbase, it, rank, lane, (uint32_t)NK, (uint32_t)NV, vst, vph, abort_flag, dt_i_);
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar(L::B_ITEM_EMPTY + islot));
        ++icount;
    }
    for (int k = 0; k < NV; ++k) {
        ptx::mbar_wait(bar(L::B_KV_EMPTY + NK + vst), vph ^ 1u, abort_flag);
        if (++vst == NV) { vst = 0; vph ^= 1u; }
    }
}

// ------------------------------------------------------------------------------------------------
// warp 1: MMA issuer.  Per kv tile k (global count, score buffer j = k & 1):
//     S[j] = Q K(k)^T    A = Q from TMEM (bf16; the q tile is stored there once per unit by softmax group 1, so a QK reads only
//                        the K tile from shared memory), 128 fp32 columns,
//     O   += P(k) V(k)   A = P from TMEM: bf16, packed over the first 32 columns of each 64-column half of S[j].
// QK(k + 1) is issued before PV(k) is waited for, QK(k + 2) right behind PV(k) (it overwrites the buffer PV(k) reads: the
// tensor pipe executes in order): the scores of the next tile are complete long before the softmax of the current one is.
// TMEM: Q = columns [0, 64), S[0] = [64, 192), S[1] = [192, 320), O = [320, 320 + D).
// ------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void mma_warp(const DecParams& p, uint32_t sbase, uint32_t tmem, const Item* items, volatile uint32_t* abort_flag,
                                         int lane, uint32_t rank) {
    using L = Smem<D>;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    DT_DECL;
    const uint64_t k_desc0 = ptx::smem_desc_sw128(sbase + L::OFF_KV, 16, KV_ATOM_STRIDE<D>);
    const uint64_t v_desc0 = ptx::smem_desc_sw128(sbase + L::OFF_KV, 1024, KV_ATOM_STRIDE<D>);
    constexpr uint32_t VSTEP = (uint32_t)(2 * KV_ATOM_STRIDE<D>) >> 4;       // one page = 16 kv rows, in descriptor units
    constexpr uint32_t IDESC_PV = ptx::idesc_bf16(BM, D, 0, 1);
    const uint32_t peer = rank ^ 1u;
    uint32_t kst = 0, kph = 0, vst = 0, vph = 0, icount = 0, qcount = 0, tcount = 0, ocount = 0;
    auto release = [&](uint32_t s) {         // this CTA is done with stage s: tell both producers of the pair
        ptx::mma_commit(bar(L::B_KV_EMPTY + s));
        ptx::mma_commit(peer_addr(bar(L::B_KV_EMPTY + s), peer));
    };
    while (true) {
        if (*abort_flag) break;
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_FULL + islot), (icount >> 1) & 1u, abort_flag);
        const Item it = items[islot];
        if (!it.valid) break;
        const int npg = it.pg1 - it.pg0, nt = (npg + 7) >> 3;
        const bool active = it.ntok - (int)rank * p.tpt > 0;
        if (nt > 0) {
            const int c_lim = it.c < it.pg1 * SANGAM_PAGE ? it.c : it.pg1 * SANGAM_PAGE;
            auto nv_of = [&](int t) { int nv = c_lim - (it.pg0 + 8 * t) * SANGAM_PAGE; return nv > BN ? BN : nv; };
            if (active) { ptx::mbar_wait(bar(L::B_Q_FULL), qcount & 1u, abort_flag); ++qcount; }
            auto issue_qk = [&](int t) {
                const uint32_t sk = kst;
                ptx::mbar_wait(bar(L::B_KV_FULL + sk), kph, abort_flag);
                if (++kst == NK) { kst = 0; kph ^= 1u; }
                ptx::tc_fence_after();
                DT(140 + (t & 15));
                if (ptx::elect_one()) {
                    if (active) {
                        const uint32_t j = (tcount + (uint32_t)t) & 1u;
                        const int ncol = (nv_of(t) + 15) & ~15;
                        const uint32_t s_tmem = tmem + TM_S + j * 128u;
                        const uint64_t b_desc = k_desc0 + (uint64_t)(sk * (L::KV_BYTES >> 4));
                        const uint32_t idesc = ptx::idesc_bf16(BM, (uint32_t)ncol, 0, 0);
                        ptx::mma_ts_x4(s_tmem, tmem + TM_Q, b_desc, idesc, 0u, 2u);
                        if (D == 128) ptx::mma_ts_x4(s_tmem, tmem + TM_Q + 32u, b_desc + (1024 >> 4), idesc, 1u, 2u);
                    }
                    release(sk);
                    if (active) {
                        ptx::mma_commit(bar(L::B_S_FULL + ((tcount + (uint32_t)t) & 1u)));
                        if (t == nt - 1) ptx::mma_commit(bar(L::B_Q_EMPTY));
                    }
                }
                __syncwarp();
            };
            issue_qk(0);
            if (nt > 1) issue_qk(1);
            for (int t = 0; t < nt; ++t) {
                if (*abort_flag) break;
                const uint32_t sv = NK + vst;
                ptx::mbar_wait(bar(L::B_KV_FULL + sv), vph, abort_flag);
                if (++vst == NV) { vst = 0; vph ^= 1u; }
                DT(160 + (t & 15));
                const int nv = nv_of(t);
                const uint32_t k = tcount + (uint32_t)t, j = k & 1u;
                if (active) {
                    if (nv & 15) dec::zero_v_tail<D>(sbase + (uint32_t)(L::OFF_KV + sv * L::KV_BYTES), nv, (nv + 15) & ~15, lane);
                    // the first PV of a unit overwrites O: the previous unit's epilogue has read it
                    if (t == 0 && ocount > 0) ptx::mbar_wait(bar(L::B_O_FREE), (ocount - 1u) & 1u, abort_flag);
                    ptx::mbar_wait(bar(L::B_P_FULL + j), (k >> 1) & 1u, abort_flag);
                }
                ptx::tc_fence_after();
                DT(11);
                if (ptx::elect_one()) {
                    if (active) {
                        const uint32_t s_tmem = tmem + TM_S + j * 128u, o_tmem = tmem + TM_O;
                        const uint64_t b0 = v_desc0 + (uint64_t)(sv * (L::KV_BYTES >> 4));
                        const int ks_n = (nv + 15) >> 4;                       // one K-step = 16 kv rows = one page
                        if (ks_n == 8) {
                            ptx::mma_ts_x4(o_tmem, s_tmem, b0, IDESC_PV, t > 0 ? 1u : 0u, VSTEP);
                            ptx::mma_ts_x4(o_tmem, s_tmem + 64u, b0 + 4 * VSTEP, IDESC_PV, 1u, VSTEP);
                        } else {
                            for (int ks = 0; ks < ks_n; ++ks)       // P of page ks: half ks / 4, 8 packed columns per page inside the half
                                ptx::mma_ts(o_tmem, s_tmem + (uint32_t)((ks >> 2) * 64 + (ks & 3) * 8), b0 + (uint64_t)(ks * VSTEP), IDESC_PV,
                                            (t > 0 || ks > 0) ? 1u : 0u);
                        }
                    }
                    release(sv);
                    if (active) ptx::mma_commit(bar(L::B_PV_DONE + j));
                }
                __syncwarp();
                if (t + 2 < nt) issue_qk(t + 2);
            }
            if (active) { ++ocount; tcount += (uint32_t)nt; }
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar(L::B_ITEM_EMPTY + islot));
        ++icount;
    }
}

// ------------------------------------------------------------------------------------------------
// warps 4..7 (group 0) and 8..11 (group 1): softmax; thread `row` of a group owns row `row` of the CTA's q tile (TMEM lane
// `row`).  Group h processes kv positions [64 h, 64 h + 64) of every tile (stream h).  Group 0 then merges the two streams and
// runs the epilogue.
// ------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void softmax_warps(const DecParams& p, uint8_t* smem, uint32_t sbase, uint32_t tmem, const Item* items,
                                              volatile uint32_t* abort_flag, int warp, int lane, uint32_t rank) {
    using L = Smem<D>;
    const unsigned FULL = 0xffffffffu;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    DT_DECL;
    const uint32_t wg = (uint32_t)(warp - 4) >> 2;             // stream of this group
    const int qd = warp & 3, row = qd * 32 + lane;
    const uint32_t lane_base = (uint32_t)(qd * 32) << 16;
    const uint32_t s_taddr = tmem + lane_base + TM_S + wg * 64u;    // this group's half of S[0]; S[1] is 128 columns further
    const uint32_t o_taddr = tmem + lane_base + TM_O;               // O
    float* l_x = reinterpret_cast<float*>(smem + L::OFF_ML);        // [item slot][row]: group 1's half of the row sum
    float* mx_x = reinterpret_cast<float*>(smem + L::OFF_MX);       // [tile parity][group][row]: half-tile row maxima
    volatile int* merge_flag = reinterpret_cast<volatile int*>(smem + L::OFF_MISC + 8);
    volatile int* agent_req = reinterpret_cast<volatile int*>(smem + L::OFF_MISC + 16);
    const float sc = fabsf(p.scale_log2);
    const bool flip = p.scale_log2 < 0.f;
    const int NS = 4 * ((int)gridDim.x >> 1);                 // partial slots: 2 per cluster x 2 CTAs
    constexpr int SLOT_F4 = (D / 4) * BM;                      // float4 per partial slot: [D/4 column groups][128 rows]

    // out row of packed row `row` of a unit: token row / G, head row % G
    auto out_ptr = [&](const OutRef& r) {
        const int tl = p.G == 1 ? row : (int)__umulhi((uint32_t)row, p.g_magic), hh = row - tl * p.G;
        const int tok = r.q_start + r.tok0 + (int)rank * p.tpt + tl;
        return p.out + ((int64_t)tok * p.Hq + (int64_t)r.g * p.G + hh) * D;
    };
    auto rows_of = [&](const OutRef& r) { int n = r.ntok - (int)rank * p.tpt; n = n > p.tpt ? p.tpt : n; return n > 0 ? n * p.G : 0; };
    auto ref_ok = [&](const OutRef& r) {
        return r.q_start + r.tok0 >= 0 && r.q_start + r.tok0 + r.ntok <= p.total_q && (unsigned)r.g < (unsigned)p.Hkv;
    };
    // General merge of this CTA's tile of a split unit: pieces in clusters bh .. bl, in that order whoever merges (group 0)
    auto merge_unit = [&](const OutRef& r, int unit, int bh, int bl) {
        const bool ok = row < rows_of(r) && ref_ok(r);
        auto slot_of = [&](int bb) { return (bb == bh ? 2 * bh + 1 : 2 * bb) * 2 + (int)rank; };
        const float2* ml = reinterpret_cast<const float2*>(p.part_ml);
        float M = -INFINITY;
        for (int bb = bh; bb <= bl; ++bb) M = fmaxf(M, __ldcg(ml + (int64_t)slot_of(bb) * BM + row).x);
        float Lsum = 0.f;
        for (int bb = bh; bb <= bl; ++bb) { const float2 x = __ldcg(ml + (int64_t)slot_of(bb) * BM + row); Lsum = fmaf(x.y, ptx::ex2(x.x - M), Lsum); }
        const float inv = Lsum > 0.f ? 1.f / Lsum : 0.f;
        __nv_bfloat16* dst = out_ptr(r);
#pragma unroll 1
        for (int c = 0; c < D / 32; ++c) {
            float f[32];
#pragma unroll
            for (int e = 0; e < 32; ++e) f[e] = 0.f;
            for (int bb = bh; bb <= bl; ++bb) {
                const int slot = slot_of(bb);
                const float w = ptx::ex2(__ldcg(ml + (int64_t)slot * BM + row).x - M);
                const float4* so = reinterpret_cast<const float4*>(p.part_o) + (int64_t)slot * SLOT_F4 + (int64_t)(c * 8) * BM + row;
#pragma unroll
                for (int v = 0; v < 8; ++v) {
                    const float4 o = __ldcg(so + v * BM);
                    f[4 * v] = fmaf(o.x, w, f[4 * v]); f[4 * v + 1] = fmaf(o.y, w, f[4 * v + 1]);
                    f[4 * v + 2] = fmaf(o.z, w, f[4 * v + 2]); f[4 * v + 3] = fmaf(o.w, w, f[4 * v + 3]);
                }
            }
            if (ok) {
#pragma unroll
                for (int v = 0; v < 4; ++v) {
                    uint4 w4;
                    w4.x = ptx::pack_bf16(f[8 * v] * inv, f[8 * v + 1] * inv); w4.y = ptx::pack_bf16(f[8 * v + 2] * inv, f[8 * v + 3] * inv);
                    w4.z = ptx::pack_bf16(f[8 * v + 4] * inv, f[8 * v + 5] * inv); w4.w = ptx::pack_bf16(f[8 * v + 6] * inv, f[8 * v + 7] * inv);
                    reinterpret_cast<uint4*>(dst)[c * 4 + v] = w4;
                }
            }
        }
        ptx::bar_sync(1, 128);
        if (qd == 0 && lane == 0) p.unit_cnt[2 * unit + (int)rank] = 0;       // re-arm for the next launch
    };

    uint32_t icount = 0, tcount = 0;      // items seen; active kv tiles seen (global index)
    uint32_t qcount = 0;                   // units whose Q was stored (group 1)
    // PV of global tile k signals PV_DONE[k & 1] (phase k >> 1); its commit covers every MMA issued before it.  A wait for tile
    // k finds the barrier in phase k >> 1 or one before: the next PV that signals it needs the P of tile k + 2.
    auto wait_pv = [&](uint32_t k) { ptx::mbar_wait(bar(L::B_PV_DONE + (k & 1u)), (k >> 1) & 1u, abort_flag); };
    while (true) {
        if (*abort_flag) break;
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_FULL + islot), (icount >> 1) & 1u, abort_flag);
        const Item it = items[islot];
        if (!it.valid) break;
        OutRef ref;
        ref.q_start = it.q_start; ref.tok0 = it.tok0; ref.ntok = it.ntok; ref.g = it.g;
        const int rows = rows_of(ref);
        const int npg = it.pg1 - it.pg0, nt = rows > 0 ? (npg + 7) >> 3 : 0;
        const int c_lim = it.c < it.pg1 * SANGAM_PAGE ? it.c : it.pg1 * SANGAM_PAGE;
        const bool row_ok = row < rows && ref_ok(ref);
        if (wg == 0 && rows > 0 && !ref_ok(ref) && lane == 0) raise_flag(p.flags, DEV_INTERNAL | 0x400u);
        float m_ref = -INFINITY, l = 0.f;
        int peek = -1;
        uint32_t k_last = 0;                    // global index of the unit's last tile
        if (wg == 1 && nt > 0) {
            // group 1 (it has no epilogue, so it reaches the next unit first) stores the q tile into TMEM as the A operand of
            // QK: row `row` = lane `row`, element pairs in consecutive columns.  Rows past the tile's tokens are zeros.
            const __nv_bfloat16* qrow;
            {
                const int tl = p.G == 1 ? row : (int)__umulhi((uint32_t)row, p.g_magic), hh = row - tl * p.G;
                const int tok = ref.q_start + ref.tok0 + (int)rank * p.tpt + tl;
                qrow = p.q + ((int64_t)tok * p.Hq + (int64_t)ref.g * p.G + hh) * D;
            }
            uint4 qv[D / 8];
#pragma unroll
            for (int c = 0; c < D / 8; ++c) qv[c] = row_ok ? __ldg(reinterpret_cast<const uint4*>(qrow) + c) : make_uint4(0, 0, 0, 0);
            ptx::mbar_wait(bar(L::B_Q_EMPTY), (qcount & 1u) ^ 1u, abort_flag);       // the previous unit's QKs have read theirs
            ptx::tc_fence_after();
#pragma unroll
            for (int c = 0; c < D / 32; ++c) {
                uint32_t w[16];
#pragma unroll
                for (int e = 0; e < 4; ++e) { w[4 * e] = qv[4 * c + e].x; w[4 * e + 1] = qv[4 * c + e].y; w[4 * e + 2] = qv[4 * c + e].z; w[4 * e + 3] = qv[4 * c + e].w; }
                ptx::tmem_st16(tmem + lane_base + TM_Q + (uint32_t)(16 * c), w);
            }
            ptx::tmem_wait_st();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(L::B_Q_FULL));
            ++qcount;
        }
        for (int t = 0; t < nt; ++t) {
            const uint32_t k = tcount + (uint32_t)t;      // (no early exit on abort: the two groups meet at a barrier per tile)
            int nv = c_lim - (it.pg0 + 8 * t) * SANGAM_PAGE;
            nv = nv > BN ? BN : nv;
            if (wg == 0 && t == nt - 1 && it.part_slot >= 0 && qd == 0 && lane == 0)      // the last tile of the unit
                asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(peek) : "l"(p.unit_cnt + 2 * it.unit + (int)rank) : "memory");
            {                                        // this group's half of the tile: kv positions [64 wg, 64 wg + 64) of S[k & 1]
                const uint32_t j = k & 1u;
                const uint32_t sh_taddr = s_taddr + j * 128u;
                const int lim = nv - 64 * (int)wg;   // valid positions of the half (<= 0: the unit's ragged end)
                ptx::mbar_wait(bar(L::B_S_FULL + j), (k >> 1) & 1u, abort_flag);
                ptx::tc_fence_after();
                DT(20);
                uint32_t r0[32], r1[32];
                float mx = -INFINITY;
                if (lim > 0) {
                    ptx::tmem_ld32(sh_taddr, r0);
                    ptx::tmem_ld32(sh_taddr + 32u, r1);
                    ptx::tmem_wait_ld();
                    if (flip) {                                     // rare: scale < 0 -- work on -s with |scale|
#pragma unroll
                        for (int i = 0; i < 32; ++i) { r0[i] ^= 0x80000000u; r1[i] ^= 0x80000000u; }
                    }
                    // the row's maximum over the half (positions >= lim masked); the full path has no per-element tests
                    if (lim >= 64) {
                        float t4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};       // four independent chains
#pragma unroll
                        for (int i = 0; i < 32; ++i) t4[i & 3] = fmaxf(t4[i & 3], fmaxf(__uint_as_float(r0[i]), __uint_as_float(r1[i])));
                        mx = fmaxf(fmaxf(t4[0], t4[1]), fmaxf(t4[2], t4[3]));
                    } else {
#pragma unroll
                        for (int i = 0; i < 32; ++i)
                            mx = fmaxf(mx, fmaxf(i < lim ? __uint_as_float(r0[i]) : -INFINITY, 32 + i < lim ? __uint_as_float(r1[i]) : -INFINITY));
                    }
                    mx *= sc;
                }
                // the two threads of a row (one per group) exchange their halves' maxima: one reference maximum, one accumulator
                // per row.  The exchange buffer alternates with the tile parity: a thread writes tile k + 2's maximum only after
                // the barrier of tile k + 1, which its partner passes after reading tile k's.
                mx_x[(j * 2u + wg) * BM + row] = mx;
                ptx::bar_sync(2, 256);
                mx = fmaxf(mx, mx_x[(j * 2u + (wg ^ 1u)) * BM + row]);
                const bool grow = mx > m_ref + LAZY_T;
                const float m_new = grow ? mx : m_ref;
                const float alpha = grow ? ptx::ex2(m_ref - m_new) : 1.f;
                m_ref = m_new;
                l *= alpha;
                if (wg == 0 && t > 0 && __any_sync(FULL, alpha != 1.f)) {
                    // rare (lazy reference maximum): every PV so far must have landed in O before the rows shrink; group 0 does
                    // it, and the PV of this tile is not issued before group 0 has handed its P
                    wait_pv(k - 1u);
                    ptx::tc_fence_after();
#pragma unroll 1
                    for (int c = 0; c < D / 32; ++c) {
                        uint32_t o[32];
                        ptx::tmem_ld32(o_taddr + (uint32_t)(c * 32), o);
                        ptx::tmem_wait_ld();
#pragma unroll
                        for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * alpha);
                        ptx::tmem_st32(o_taddr + (uint32_t)(c * 32), o);
                    }
                    ptx::tmem_wait_st();
                }
                DT(21);
                if (lim > 0) {
                    // P = 2^(s scale - m_ref) as bf16 pairs over the first 32 columns of the half, row sum into l
                    // (packed fp32x2 arithmetic: one FFMA2 / FADD2 per two columns)
                    const float2 sc2 = make_float2(sc, sc), ng2 = make_float2(-m_ref, -m_ref);
                    float2 sum_a = make_float2(0.f, 0.f), sum_b = make_float2(0.f, 0.f);
                    uint32_t pk[32];
#pragma unroll
                    for (int i = 0; i < 32; i += 2) {
                        const float2 xa = __ffma2_rn(make_float2(__uint_as_float(r0[i]), __uint_as_float(r0[i + 1])), sc2, ng2);
                        const float2 xc = __ffma2_rn(make_float2(__uint_as_float(r1[i]), __uint_as_float(r1[i + 1])), sc2, ng2);
                        float2 pa = make_float2(ptx::ex2(xa.x), ptx::ex2(xa.y)), pc = make_float2(ptx::ex2(xc.x), ptx::ex2(xc.y));
                        if (lim < 64) {
                            if (i >= lim) pa.x = 0.f;
                            if (i + 1 >= lim) pa.y = 0.f;
                            if (32 + i >= lim) pc.x = 0.f;
                            if (33 + i >= lim) pc.y = 0.f;
                        }
                        sum_a = __fadd2_rn(sum_a, pa);
                        sum_b = __fadd2_rn(sum_b, pc);
                        pk[i >> 1] = ptx::pack_bf16(pa.x, pa.y);
                        pk[16 + (i >> 1)] = ptx::pack_bf16(pc.x, pc.y);
                    }
                    ptx::tmem_st16(sh_taddr, pk);
                    ptx::tmem_st16(sh_taddr + 16u, pk + 16);
                    const float2 sum2 = __fadd2_rn(sum_a, sum_b);
                    l += sum2.x + sum2.y;
                    ptx::tmem_wait_st();
                }
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(bar(L::B_P_FULL + j));
                DT(23);
            }
            k_last = k;
        }
        tcount += (uint32_t)nt;
        if (wg == 1) {
            // group 1 hands its half of the row sums to group 0 (double-buffered by item slot: the slot is not reused
            // before group 0 has released the item) and is done with the unit
            // (one EPI barrier per item slot, used for every item: group 1 may run a whole item ahead of group 0, and a
            // parity wait cannot tell phases two apart)
            l_x[islot * BM + row] = l;
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(L::B_EPI + islot));
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(L::B_ITEM_EMPTY + islot));
            ++icount;
            continue;
        }
        // ---------------- epilogue (group 0)
        DT(24);
        ptx::mbar_wait(bar(L::B_EPI + islot), (icount >> 1) & 1u, abort_flag);      // group 1 is done with the unit's tiles
        DT(25);
        const bool split = nt > 0 && it.part_slot >= 0;
        const int np_u = it.b_last - it.b_head + 1, k_me = ((int)blockIdx.x >> 1) - it.b_head;
        bool early = false;
        if (split) {
            if (qd == 0 && lane == 0) {
                if (peek < 0) asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(peek) : "l"(p.unit_cnt + 2 * it.unit + (int)rank) : "memory");
                const int e = (np_u == 2 && (k_me == 0 || k_me == 1) && peek + npg == it.upages) ? 1 : 0;
                if (e) asm volatile("fence.acq_rel.gpu;" ::: "memory");
                *merge_flag = e;
            }
            ptx::bar_sync(1, 128);
            early = *merge_flag != 0;
            ptx::bar_sync(1, 128);
        }
        DT(30 + (early ? 1 : 0) + (split ? 2 : 0));
        __nv_bfloat16* dst = out_ptr(ref);
        if (rows > 0 && nt == 0) {
            if (row_ok && it.part_slot < 0) {                    // empty context: zero rows (reading S13)
#pragma unroll
                for (int c = 0; c < D / 8; ++c) reinterpret_cast<uint4*>(dst)[c] = make_uint4(0, 0, 0, 0);
            }
        } else if (nt > 0) {
            // the other piece of a two-piece unit is requested before the last PVs are awaited (early merge, see attn_dec.cuh)
            const int other = (k_me == 0 ? 2 * (it.b_head + 1) : 2 * it.b_head + 1) * 2 + (int)rank;
            float2 xo = make_float2(-INFINITY, 0.f);
            if (early) xo = __ldcg(reinterpret_cast<const float2*>(p.part_ml) + (int64_t)other * BM + row);
            wait_pv(k_last);                                     // the unit's last PV (its commit covers all before it)
            ptx::tc_fence_after();
            DT(27);
            // own piece: the row's reference maximum is common to the two groups, the row sum is the sum of their halves
            const float m_own = m_ref;
            const float l_own = l + l_x[islot * BM + row];
            const bool partial = split && !early;
            const bool slot_ok = !partial || (it.part_slot * 2 + (int)rank < NS && it.unit >= 0);
            if (!slot_ok && lane == 0) raise_flag(p.flags, DEV_INTERNAL | 0x100u);
            const int slot = it.part_slot * 2 + (int)rank;
            float w_own = 1.f, w_oth = 0.f, inv = l_own > 0.f ? 1.f / l_own : 0.f;
            if (early) {                                         // pieces in order: k_me = 0: own, other;  1: other, own
                const float M = fmaxf(m_own, xo.x);
                w_own = ptx::ex2(m_own - M); w_oth = ptx::ex2(xo.x - M);
                const float Lsum = k_me == 0 ? fmaf(xo.y, w_oth, fmaf(l_own, w_own, 0.f)) : fmaf(l_own, w_own, fmaf(xo.y, w_oth, 0.f));
                inv = Lsum > 0.f ? 1.f / Lsum : 0.f;
            }
#pragma unroll 1
            for (int c = 0; c < D / 32; ++c) {
                float4 ov[8];
                if (early) {
                    const float4* so = reinterpret_cast<const float4*>(p.part_o) + (int64_t)other * SLOT_F4 + (int64_t)(c * 8) * BM + row;
#pragma unroll
                    for (int v = 0; v < 8; ++v) ov[v] = __ldcg(so + v * BM);
                }
                uint32_t oa[32];
                ptx::tmem_ld32(o_taddr + (uint32_t)(c * 32), oa);
                ptx::tmem_wait_ld();
                DT(34);
                float a[32];                                     // this piece's unnormalised row chunk
#pragma unroll
                for (int e = 0; e < 32; ++e) a[e] = __uint_as_float(oa[e]);
                float f[32];
                if (early) {
#pragma unroll
                    for (int v = 0; v < 8; ++v) {
                        const float e0 = ov[v].x, e1 = ov[v].y, e2 = ov[v].z, e3 = ov[v].w;
                        if (k_me == 0) {
                            f[4 * v] = fmaf(e0, w_oth, fmaf(a[4 * v], w_own, 0.f)); f[4 * v + 1] = fmaf(e1, w_oth, fmaf(a[4 * v + 1], w_own, 0.f));
                            f[4 * v + 2] = fmaf(e2, w_oth, fmaf(a[4 * v + 2], w_own, 0.f)); f[4 * v + 3] = fmaf(e3, w_oth, fmaf(a[4 * v + 3], w_own, 0.f));
                        } else {
                            f[4 * v] = fmaf(a[4 * v], w_own, fmaf(e0, w_oth, 0.f)); f[4 * v + 1] = fmaf(a[4 * v + 1], w_own, fmaf(e1, w_oth, 0.f));
                            f[4 * v + 2] = fmaf(a[4 * v + 2], w_own, fmaf(e2, w_oth, 0.f)); f[4 * v + 3] = fmaf(a[4 * v + 3], w_own, fmaf(e3, w_oth, 0.f));
                        }
                    }
                } else {
#pragma unroll
                    for (int e = 0; e < 32; ++e) f[e] = a[e];
                }
                if (partial) {
                    if (slot_ok && row < rows) {
                        float4* po = reinterpret_cast<float4*>(p.part_o) + (int64_t)slot * SLOT_F4 + (int64_t)(c * 8) * BM + row;
#pragma unroll
                        for (int v = 0; v < 8; ++v) po[v * BM] = make_float4(f[4 * v], f[4 * v + 1], f[4 * v + 2], f[4 * v + 3]);
                    }
                } else if (row_ok) {
#pragma unroll
                    for (int v = 0; v < 4; ++v) {
                        uint4 w4;
                        w4.x = ptx::pack_bf16(f[8 * v] * inv, f[8 * v + 1] * inv); w4.y = ptx::pack_bf16(f[8 * v + 2] * inv, f[8 * v + 3] * inv);
                        w4.z = ptx::pack_bf16(f[8 * v + 4] * inv, f[8 * v + 5] * inv); w4.w = ptx::pack_bf16(f[8 * v + 6] * inv, f[8 * v + 7] * inv);
                        reinterpret_cast<uint4*>(dst)[c * 4 + v] = w4;
                    }
                }
            }
            ptx::tc_fence_before();
            __syncwarp();
            DT(28);
            if (lane == 0) {                                     // both accumulators have been read
                ptx::mbar_arrive(bar(L::B_O_FREE));
            }
            if (partial && slot_ok && row < rows) reinterpret_cast<float2*>(p.part_ml)[(int64_t)slot * BM + row] = make_float2(m_own, l_own);
            if (split) {
                if (qd == 0 && lane == 0) {
                    agent_req[islot] = (partial && slot_ok) ? 1 : 0;
                    if (early) p.unit_cnt[2 * it.unit + (int)rank] = 0;        // re-arm the counter
                }
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(bar(L::B_AGENT_REQ));
            }
        }
        __syncwarp();
        DT(29);
        if (lane == 0) ptx::mbar_arrive(bar(L::B_ITEM_EMPTY + islot));
        ++icount;
    }
    if (wg == 1) return;
    ptx::mbar_wait(bar(L::B_AGENT_DONE), 0u, abort_flag);
    const Deferred* defer = reinterpret_cast<const Deferred*>(smem + L::OFF_MISC + 32);
    for (int k = 0; k < 2; ++k) {
        const Deferred dr = defer[k];
        if (dr.valid) {
            OutRef r;
            r.q_start = dr.q_start; r.tok0 = dr.tok0; r.ntok = dr.ntok; r.g = dr.g;
            merge_unit(r, dr.unit, dr.b_head, dr.b_last);
        }
    }
}

// warp 2: arrival agent (attn_dec.cuh): gpu-scope release of a stored piece, arrival count, Deferred record if it was the last
template <int D>
__device__ __forceinline__ void agent_warp(const DecParams& p, uint8_t* smem, uint32_t sbase, const Item* items, volatile uint32_t* abort_flag,
                                           int lane, uint32_t rank) {
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
        const bool active = it.ntok - (int)rank * p.tpt > 0;
        if (npg > 0 && it.part_slot >= 0 && active) {
            ptx::mbar_wait(bar(L::B_AGENT_REQ), rcount & 1u, abort_flag);
            ++rcount;
            if (lane == 0 && agent_req[islot] != 0) {
                int old;
                asm volatile("fence.acq_rel.gpu;" ::: "memory");
                asm volatile("atom.relaxed.gpu.global.add.s32 %0, [%1], %2;" : "=r"(old) : "l"(p.unit_cnt + 2 * it.unit + (int)rank), "r"(npg) : "memory");
                if (old + npg == it.upages) {
                    asm volatile("fence.acq_rel.gpu;" ::: "memory");
                    if (ndef < 2) {
                        Deferred dr;
                        dr.valid = 1; dr.unit = it.unit; dr.b_head = it.b_head; dr.b_last = it.b_last;
                        dr.q_start = it.q_start; dr.tok0 = it.tok0; dr.ntok = it.ntok; dr.g = it.g;
                        defer[ndef++] = dr;
                    } else {
                        raise_flag(p.flags, DEV_INTERNAL | 0x200u);
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

template <int D>
__global__ void __launch_bounds__(NTHREADS, 1)
gqa_decode_kernel(const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV,
                  const __grid_constant__ CUtensorMap /* q map: unused, q rows are read directly */, const DecParams p) {
    using L = Smem<D>;
    // both CTAs of the pair use the same offsets inside their shared-memory windows (a multicast write lands at the issuing
    // CTA's offset in every destination): the dynamic base is the same in every CTA of a launch (no static shared memory)
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = ptx::smem_u32(smem);
    Item* items = reinterpret_cast<Item*>(smem + L::OFF_ITEMS);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::OFF_MISC);
    volatile uint32_t* abort_flag = reinterpret_cast<volatile uint32_t*>(smem + L::OFF_ABORT);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = cluster_rank();
    TRACE_CTA(0);
    if (tid == 0) {
        auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
        for (int s = 0; s < NK + NV; ++s) { ptx::mbar_init(bar(L::B_KV_FULL + s), 1); ptx::mbar_init(bar(L::B_KV_EMPTY + s), 2); }   // both CTAs release
        for (int s = 0; s < 2; ++s) {
            ptx::mbar_init(bar(L::B_ITEM_FULL + s), 1); ptx::mbar_init(bar(L::B_ITEM_EMPTY + s), 11);     // MMA warp + V producer + agent + 8 softmax warps
            ptx::mbar_init(bar(L::B_S_FULL + s), 1); ptx::mbar_init(bar(L::B_P_FULL + s), 8);             // both groups hand their half of P
            ptx::mbar_init(bar(L::B_PV_DONE + s), 1);
        }
        ptx::mbar_init(bar(L::B_O_FREE), 4);
        ptx::mbar_init(bar(L::B_Q_FULL), 4); ptx::mbar_init(bar(L::B_Q_EMPTY), 1);      // group 1's warps store the q tile
        ptx::mbar_init(bar(L::B_EPI), 4); ptx::mbar_init(bar(L::B_EPI + 1), 4);
        ptx::mbar_init(bar(L::B_AGENT_REQ), 4); ptx::mbar_init(bar(L::B_AGENT_DONE), 1);
        for (int k = 1; k < (L::TOTAL - L::OFF_MISC) / 4; ++k) tmem_slot[k] = 0u;
        ptx::fence_mbar_init();
        ptx::prefetch_tensormap(&mapK);
        ptx::prefetch_tensormap(&mapV);
    }
    if (warp == 1) {
        ptx::tmem_alloc(ptx::smem_u32(tmem_slot), 512);
        ptx::tmem_relinquish();
    }
    ptx::pdl_wait();
    ptx::pdl_trigger();
    ptx::tc_fence_before();
    __syncthreads();
    cluster_sync_all();            // the peer's barriers exist before anything is multicast to it or arrives on them
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const bool base_ok = (sbase & 1023u) == 0u;
    if (!base_ok && tid == 0) raise_flag(p.flags, DEV_INTERNAL | 0x800u);
    // 12 warps x 168 registers at launch; the service warpgroup hands its surplus to the two softmax groups
    if (warp >= 4) {
        ptx::setmaxnreg_inc<208>();
        if (base_ok) softmax_warps<D>(p, smem, sbase, tmem, items, abort_flag, warp, lane, rank);
    } else {
        ptx::setmaxnreg_dec<88>();
        if (!base_ok) { }
        else if (warp == 0) producer_warp<D>(p, &mapK, sbase, items, abort_flag, lane, rank);
        else if (warp == 3) v_producer_warp<D>(p, &mapV, sbase, items, abort_flag, lane, rank);
        else if (warp == 1) mma_warp<D>(p, sbase, tmem, items, abort_flag, lane, rank);
        else if (warp == 2) agent_warp<D>(p, smem, sbase, items, abort_flag, lane, rank);
    }
    ptx::tc_fence_before();
    __syncthreads();
    cluster_sync_all();            // neither CTA leaves while the other may still write into it
    TRACE_CTA(1);
    if (tid == 0 && *abort_flag) raise_flag(p.flags, DEV_TIMEOUT);
    if (warp == 1) ptx::tmem_dealloc(tmem, 512);
}

}  // namespace gqa

static inline cudaError_t gqa_configure(int head_dim) {
    cudaError_t e;
    if (head_dim == 128) e = cudaFuncSetAttribute(gqa::gqa_decode_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, gqa::Smem<128>::ALLOC);
    else e = cudaFuncSetAttribute(gqa::gqa_decode_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, gqa::Smem<64>::ALLOC);
    return e;
}

static inline cudaError_t gqa_launch(const DecParams& p, const CUtensorMap& mk, const CUtensorMap& mv, const CUtensorMap& mq, int head_dim,
                                     int num_ctas, cudaStream_t stream) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(num_ctas & ~1); cfg.blockDim = dim3(gqa::NTHREADS); cfg.stream = stream;
    cfg.dynamicSmemBytes = head_dim == 128 ? gqa::Smem<128>::ALLOC : gqa::Smem<64>::ALLOC;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    at[1].id = cudaLaunchAttributeClusterDimension;
    at[1].val.clusterDim.x = 2; at[1].val.clusterDim.y = 1; at[1].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 2;
    cudaError_t e = head_dim == 128 ? cudaLaunchKernelEx(&cfg, gqa::gqa_decode_kernel<128>, mk, mv, mq, p)
                                    : cudaLaunchKernelEx(&cfg, gqa::gqa_decode_kernel<64>, mk, mv, mq, p);
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}
