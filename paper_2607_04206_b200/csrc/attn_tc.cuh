// attn_tc.cuh -- steps a3..a8: paged, varlen, non-causal block attention on tcgen05 (sm_100a).
//
// One persistent CTA per SM, 8 warps, warp-specialised:
//   warp 0      scheduler + TMA producer: plans the work on the device (a3), gathers K/V pages of
//               the current (request, kv head) through the block table with TMA into a ring of
//               128-row, 128B-swizzled shared-memory tiles (a4)
//   warp 1      MMA issuer: S = Q K^T (tcgen05.mma, operands in smem, S in TMEM; a5) and
//               O += P V (P read from TMEM, V from smem, O in TMEM; a7)
//   warp 2      TMEM allocator
//   warps 4-7   softmax warpgroup: thread i owns row i of the tile (TMEM lane i): online softmax
//               in fp32 (a6), P written back to TMEM as bf16, O rescale, epilogue (a8)
// Work unit = (request r, kv head g, 128-row tile of the packed (query row, q head in group) rows):
// the G q heads of a GQA group share every K/V tile.  A unit's kv range may be split across CTAs
// (static stream-K partition for decode-sized batches); partials go to the workspace and are merged
// by combine_kernel (a9).  With many units (prefill / hybrid) whole units are handed out dynamically.
// The attention definition is PAPER.md:67 (no causal mask) over the context of PAPER.md:33.
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "ptx.cuh"

struct TcMaps {
    CUtensorMap k, v;
};

namespace tc {

constexpr int BM = 128;          // rows per q tile  (UMMA M)
constexpr int BN = 128;          // kv positions per tile (8 pages)
constexpr int NSTAGE = 6;        // K/V tile ring depth
constexpr int NTHREADS = 256;
constexpr int SLAB = 128 * 128;  // bytes of one 64-wide swizzled slab of a 128-row tile
constexpr int DYN_UNITS_PER_CTA = 4;   // >= this many units per CTA: whole units, dynamic hand-out

struct Item {          // one piece of work, published through shared memory
    int valid;         // 0 = no more work
    int r, g;
    int row0;          // first packed row of the tile inside the (r, g) unit group
    int rows_valid;    // rows of this tile that exist (<= 128)
    int q_start;       // cu_q_lens[r]
    int c;             // context length
    int kv0, kv1;      // kv tile range [kv0, kv1)
    int part_slot;     // -1: write `out`; else partial slot in the workspace
    int pad0, pad1;
};

struct SlotMeta {      // global, one per partial slot, rewritten by its CTA every launch
    int valid;
    int b_last;        // head slots: last CTA holding a piece of this unit
    int g, row0, rows_valid, q_start;
    int pad0, pad1;
};

template <int D>
struct Smem {
    static constexpr int Q_BYTES = BM * D * 2;
    static constexpr int KV_BYTES = BN * D * 2;
    static constexpr int OFF_Q = 0;
    static constexpr int OFF_KV = Q_BYTES;
    static constexpr int OFF_BAR = OFF_KV + NSTAGE * KV_BYTES;
    // barrier indices
    static constexpr int B_KV_FULL = 0, B_KV_EMPTY = NSTAGE, B_ITEM_FULL = 2 * NSTAGE, B_ITEM_EMPTY = 2 * NSTAGE + 2,
                         B_Q_FULL = 2 * NSTAGE + 4, B_S_FULL = 2 * NSTAGE + 5, B_P_FULL = 2 * NSTAGE + 7,
                         B_PV_DONE = 2 * NSTAGE + 9, NBAR = 2 * NSTAGE + 10;
    static constexpr int OFF_ITEMS = OFF_BAR + ((NBAR * 8 + 15) / 16) * 16;
    static constexpr int OFF_MISC = OFF_ITEMS + 2 * (int)sizeof(Item);
    static constexpr int TOTAL = OFF_MISC + 16;
    static constexpr int ALLOC = TOTAL + 1024;   // slack to align the base to 1024 B (128B swizzle atoms)
};

struct ReqInfo {
    int q0, c, nm, tiles_u, units, rows;
};

__device__ __forceinline__ ReqInfo req_info(const AttnParams& p, int r) {
    ReqInfo x;
    x.q0 = __ldg(p.cu_q_lens + r);
    int qn = __ldg(p.cu_q_lens + r + 1) - x.q0;
    if (qn < 0) qn = 0;
    int c = __ldg(p.ctx_lens + r);
    if (c < 0) c = 0;
    if ((c + SANGAM_PAGE - 1) / SANGAM_PAGE > p.W) { raise_flag(p.flags, DEV_CTX_TOO_LONG); c = 0; }
    x.c = c;
    x.rows = qn * p.G;
    x.nm = (x.rows + BM - 1) / BM;
    const int nkv = (c + BN - 1) / BN;
    x.tiles_u = nkv > 0 ? nkv : 1;
    x.units = p.Hkv * x.nm;
    return x;
}


// ------------------------------------------------------------------------------------------------
// warp 0: device-side plan (a3) + TMA page gather (a4)
// ------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void producer_warp(const AttnParams& p, SlotMeta* meta, const CUtensorMap* mapK,
                                              const CUtensorMap* mapV, uint32_t sbase, Item* items,
                                              volatile uint32_t* abort_flag, int lane) {
    using L = Smem<D>;
    const unsigned FULL = 0xffffffffu;
    const int G_ctas = gridDim.x, b = blockIdx.x, R = p.batch;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };

    // totals over the batch: units U and kv tiles T
    int U = 0, T = 0;
    for (int r = lane; r < R; r += 32) {
        const ReqInfo x = req_info(p, r);
        U += x.units;
        T += x.units * x.tiles_u;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        U += __shfl_xor_sync(FULL, U, o);
        T += __shfl_xor_sync(FULL, T, o);
    }
    const bool dynamic = U >= DYN_UNITS_PER_CTA * G_ctas;
    if (lane < 2) meta[2 * b + lane].valid = 0;
    __syncwarp();

    // walking state
    int r_cur = 0, ubase = 0, u_in_r = 0, kvoff = 0, remaining = 0, tile_base = 0, Geff = 1;
    ReqInfo cur;
    cur.units = 0; cur.tiles_u = 1; cur.nm = 1; cur.c = 0; cur.q0 = 0; cur.rows = 0;
    if (R > 0) cur = req_info(p, 0);
    if (!dynamic && T > 0) {
        Geff = G_ctas < T ? G_ctas : T;
        if (b < Geff) {
            const int t0 = (int)(((int64_t)b * T) / Geff), t1 = (int)(((int64_t)(b + 1) * T) / Geff);
            remaining = t1 - t0;
            // locate the request holding flattened tile t0 (chunked warp scan over requests)
            int acc = 0, found = -1;
            for (int base = 0; base < R && found < 0; base += 32) {
                const int r = base + lane;
                int tl = 0;
                if (r < R) { const ReqInfo x = req_info(p, r); tl = x.units * x.tiles_u; }
                int incl = tl;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int v = __shfl_up_sync(FULL, incl, o);
                    if (lane >= o) incl += v;
                }
                const unsigned m = __ballot_sync(FULL, acc + incl > t0);
                if (m) {
                    const int l = __ffs(m) - 1;
                    found = base + l;
                    tile_base = acc + __shfl_sync(FULL, incl - tl, l);
                } else {
                    acc += __shfl_sync(FULL, incl, 31);
                }
            }
            r_cur = found < 0 ? R : found;
            if (r_cur < R) {
                cur = req_info(p, r_cur);
                const int pos = t0 - tile_base;
                u_in_r = pos / cur.tiles_u;
                kvoff = pos - u_in_r * cur.tiles_u;
            } else {
                remaining = 0;
            }
        }
    }

    uint32_t kvi = 0, icount = 0;
    while (true) {
        if (*abort_flag) break;
        Item it;
        it.valid = 0; it.r = 0; it.g = 0; it.row0 = 0; it.rows_valid = 0; it.q_start = 0; it.c = 0;
        it.kv0 = 0; it.kv1 = 0; it.part_slot = -1; it.pad0 = 0; it.pad1 = 0;
        if (dynamic) {
            int u = 0;
            if (lane == 0) u = atomicAdd(p.sched, 1);
            u = __shfl_sync(FULL, u, 0);
            if (u < U) {
                while (r_cur < R && u >= ubase + cur.units) {
                    ubase += cur.units;
                    ++r_cur;
                    if (r_cur < R) cur = req_info(p, r_cur);
                }
                if (r_cur < R) {
                    const int ul = u - ubase;
                    it.valid = 1; it.r = r_cur; it.g = ul / cur.nm;
                    it.row0 = (ul - it.g * cur.nm) * BM;
                    it.kv0 = 0; it.kv1 = cur.tiles_u;
                }
            }
        } else if (remaining > 0 && r_cur < R) {
            const int take = remaining < cur.tiles_u - kvoff ? remaining : cur.tiles_u - kvoff;
            it.valid = 1; it.r = r_cur; it.g = u_in_r / cur.nm;
            it.row0 = (u_in_r - it.g * cur.nm) * BM;
            it.kv0 = kvoff; it.kv1 = kvoff + take;
            if (!(it.kv0 == 0 && it.kv1 == cur.tiles_u)) {
                const bool head = it.kv0 == 0;
                it.part_slot = 2 * b + (head ? 1 : 0);
                if (lane == 0) {
                    SlotMeta mm;
                    mm.valid = 1; mm.g = it.g; mm.row0 = it.row0;
                    mm.rows_valid = cur.rows - it.row0 < BM ? cur.rows - it.row0 : BM;
                    mm.q_start = cur.q0; mm.pad0 = it.r; mm.pad1 = 0;
                    const int64_t ut1 = (int64_t)tile_base + (int64_t)(u_in_r + 1) * cur.tiles_u;
                    int bl = (int)((ut1 * Geff + T - 1) / T) - 1;
                    mm.b_last = bl > Geff - 1 ? Geff - 1 : bl;
                    meta[it.part_slot] = mm;
                }
            }
            remaining -= take;
            kvoff += take;
            if (kvoff == cur.tiles_u) {
                kvoff = 0;
                if (++u_in_r == cur.units) {
                    u_in_r = 0;
                    do {
                        tile_base += cur.units * cur.tiles_u;
                        ++r_cur;
                        if (r_cur < R) cur = req_info(p, r_cur);
                    } while (r_cur < R && cur.units == 0);
                }
            }
        }
        ReqInfo ri = cur;
        if (it.valid) {
            if (it.r != r_cur) ri = req_info(p, it.r);   // static walk may already have advanced
            it.rows_valid = ri.rows - it.row0 < BM ? ri.rows - it.row0 : BM;
            it.q_start = ri.q0;
            it.c = ri.c;
            if (ri.c == 0) { it.kv0 = 0; it.kv1 = 0; }
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

        // K/V tile loads in the order the MMA warp consumes them: K0, [K1], V0, [K2], V1, ...
        const int n = it.kv1 - it.kv0;
        const int pages_total = (it.c + SANGAM_PAGE - 1) / SANGAM_PAGE;
        const int32_t* bt = p.block_table + (int64_t)it.r * p.W;
        auto load_tile = [&](int tile, bool is_v) {
            const uint32_t stage = kvi % NSTAGE;
            ptx::mbar_wait(bar(L::B_KV_EMPTY + stage), ((kvi / NSTAGE) & 1u) ^ 1u, abort_flag);
            int np = pages_total - tile * 8;
            np = np > 8 ? 8 : np;
            constexpr int BOX_PER_PAGE = D / 64;
            if (lane == 0) ptx::mbar_arrive_expect_tx(bar(L::B_KV_FULL + stage), (uint32_t)(np * SANGAM_PAGE * D * 2));
            __syncwarp();
            if (lane < np * BOX_PER_PAGE) {
                const int pg = lane / BOX_PER_PAGE, slab = lane % BOX_PER_PAGE;
                const int page = __ldg(bt + tile * 8 + pg);
                if ((unsigned)page >= (unsigned)p.P) raise_flag(p.flags, DEV_BAD_PAGE);   // TMA zero-fills out of range
                ptx::tma_load_2d(sbase + (uint32_t)(L::OFF_KV + stage * L::KV_BYTES + slab * SLAB + pg * 2048),
                                 is_v ? mapV : mapK, bar(L::B_KV_FULL + stage), slab * 64,
                                 (page * p.Hkv + it.g) * SANGAM_PAGE);
            }
            ++kvi;
        };
        if (n > 0) {
            load_tile(it.kv0, false);
            for (int j = 0; j < n; ++j) {
                if (*abort_flag) break;
                if (j + 1 < n) load_tile(it.kv0 + j + 1, false);
                load_tile(it.kv0 + j, true);
            }
        }
    }
    if (dynamic && lane == 0) {
        if (atomicAdd(p.sched + 1, 1) == G_ctas - 1) {   // last CTA out re-arms the counters for the next launch
            p.sched[0] = 0;
            p.sched[1] = 0;
            __threadfence();
        }
    }
}


// ------------------------------------------------------------------------------------------------
// warp 1: MMA issuer (a5, a7).  TMEM columns: S0 = [0,128), S1 = [128,256), O = [256,256+D).
// P_b (bf16, two per column) overwrites the first 64 columns of S_b.
// Issue order per item: QK0, [QK1], PV0, [QK2], PV1, ...  -- the next tile's logits are computed
// while the softmax warpgroup works on the current one.
// ------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void mma_warp(const AttnParams& p, uint32_t sbase, uint32_t tmem, const Item* items,
                                         volatile uint32_t* abort_flag, int lane) {
    using L = Smem<D>;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    const uint32_t q_addr = sbase + L::OFF_Q;
    uint32_t kvi = 0, icount = 0, tcount = 0;
    while (true) {
        if (*abort_flag) break;
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_FULL + islot), (icount >> 1) & 1u, abort_flag);
        const Item it = items[islot];
        if (!it.valid) break;
        const int n = it.kv1 - it.kv0;
        ptx::mbar_wait(bar(L::B_Q_FULL), icount & 1u, abort_flag);
        ptx::tc_fence_after();
        auto issue_qk = [&](int j, uint32_t sb) {
            const uint32_t stage = kvi % NSTAGE;
            ptx::mbar_wait(bar(L::B_KV_FULL + stage), (kvi / NSTAGE) & 1u, abort_flag);
            ptx::tc_fence_after();
            int nv = it.c - (it.kv0 + j) * BN;
            nv = nv > BN ? BN : nv;
            const uint32_t ncols = (uint32_t)((nv + 15) & ~15);
            if (lane == 0) {
                const uint32_t k_addr = sbase + (uint32_t)(L::OFF_KV + stage * L::KV_BYTES);
                const uint32_t idesc = ptx::idesc_bf16(BM, ncols, 0, 0);
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks) {
                    const uint32_t off = (uint32_t)((ks >> 2) * SLAB + (ks & 3) * 32);
                    ptx::mma_ss(tmem + sb * 128u, ptx::smem_desc_sw128(q_addr + off, 16, 1024),
                                ptx::smem_desc_sw128(k_addr + off, 16, 1024), idesc, ks > 0);
                }
                ptx::mma_commit(bar(L::B_KV_EMPTY + stage));
                ptx::mma_commit(bar(L::B_S_FULL + sb));
            }
            __syncwarp();
            ++kvi;
        };
        if (n > 0) {
            issue_qk(0, tcount & 1u);
            for (int j = 0; j < n; ++j) {
                if (*abort_flag) break;
                const uint32_t sb = tcount & 1u;
                if (j + 1 < n) issue_qk(j + 1, sb ^ 1u);
                const uint32_t stage = kvi % NSTAGE;
                ptx::mbar_wait(bar(L::B_KV_FULL + stage), (kvi / NSTAGE) & 1u, abort_flag);
                int nv = it.c - (it.kv0 + j) * BN;
                nv = nv > BN ? BN : nv;
                const int ncols = (nv + 15) & ~15;
                const uint32_t v_addr = sbase + (uint32_t)(L::OFF_KV + stage * L::KV_BYTES);
                if (nv < ncols) {
                    // stale rows of the last page: zero them so that P = 0 meets V = 0, never NaN (reading S12)
                    const int nrows = ncols - nv;
                    for (int e = lane; e < nrows * 8 * (D / 64); e += 32) {
                        const int chunk = e & 7, rr = (e >> 3) % nrows, slab = (e >> 3) / nrows;
                        asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(
                                         v_addr + (uint32_t)(slab * SLAB + (nv + rr) * 128 + chunk * 16)),
                                     "r"(0)
                                     : "memory");
                    }
                    ptx::fence_proxy_async_smem();
                    __syncwarp();
                }
                ptx::mbar_wait(bar(L::B_P_FULL + sb), (tcount >> 1) & 1u, abort_flag);
                ptx::tc_fence_after();
                if (lane == 0) {
                    const uint32_t idesc = ptx::idesc_bf16(BM, D, 0, 1);
                    const int nk = ncols / 16;
                    for (int ks = 0; ks < nk; ++ks)
                        ptx::mma_ts(tmem + 256u, tmem + sb * 128u + (uint32_t)(ks * 8),
                                    ptx::smem_desc_sw128(v_addr + (uint32_t)(ks * 2048), SLAB, 1024), idesc,
                                    (j > 0 || ks > 0) ? 1u : 0u);
                    ptx::mma_commit(bar(L::B_KV_EMPTY + stage));
                    ptx::mma_commit(bar(L::B_PV_DONE));
                }
                __syncwarp();
                ++kvi;
                ++tcount;
            }
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar(L::B_ITEM_EMPTY + islot));
        ++icount;
    }
}

// ------------------------------------------------------------------------------------------------
// warps 4-7: softmax warpgroup (a6) + epilogue (a8).  Thread `row` owns TMEM lane `row`.
// ------------------------------------------------------------------------------------------------
template <bool MASK>
__device__ __forceinline__ void softmax_row(uint32_t s_taddr, int nv, float scale_log2, float& m, float& l,
                                            float& alpha, uint32_t (&pk)[64]) {
    uint32_t r[4][32];
#pragma unroll
    for (int c = 0; c < 4; ++c) ptx::tmem_ld32(s_taddr + (uint32_t)(c * 32), r[c]);
    ptx::tmem_wait_ld();
    float mx = -INFINITY;
    if (scale_log2 >= 0.f) {
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int i = 0; i < 32; ++i)
                if (!MASK || c * 32 + i < nv) mx = fmaxf(mx, __uint_as_float(r[c][i]));
    } else {
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int i = 0; i < 32; ++i)
                if (!MASK || c * 32 + i < nv) mx = fmaxf(mx, -__uint_as_float(r[c][i]));
        mx = -mx;
    }
    const float m_new = fmaxf(m, mx * scale_log2);
    alpha = ptx::ex2(m - m_new);
    const float neg = -m_new;
    float sum0 = 0.f, sum1 = 0.f;
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            float p0 = ptx::ex2(fmaf(__uint_as_float(r[c][2 * i]), scale_log2, neg));
            float p1 = ptx::ex2(fmaf(__uint_as_float(r[c][2 * i + 1]), scale_log2, neg));
            if (MASK) {
                if (c * 32 + 2 * i >= nv) p0 = 0.f;
                if (c * 32 + 2 * i + 1 >= nv) p1 = 0.f;
            }
            sum0 += p0;
            sum1 += p1;
            pk[c * 16 + i] = ptx::pack_bf16(p0, p1);
        }
    l = l * alpha + (sum0 + sum1);
    m = m_new;
}

template <int D>
__device__ __forceinline__ void softmax_wg(const AttnParams& p, uint8_t* smem, uint32_t sbase, uint32_t tmem,
                                           const Item* items, volatile uint32_t* abort_flag, int wg_warp, int lane) {
    using L = Smem<D>;
    const unsigned FULL = 0xffffffffu;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    const int row = wg_warp * 32 + lane;
    const int wtid = wg_warp * 32 + lane;   // 0..127
    const uint32_t lane_base = (uint32_t)(wg_warp * 32) << 16;
    const uint32_t o_taddr = tmem + lane_base + 256u;
    uint32_t icount = 0, tcount = 0;
    while (true) {
        if (*abort_flag) break;
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_FULL + islot), (icount >> 1) & 1u, abort_flag);
        const Item it = items[islot];
        if (!it.valid) break;
        // ---- Q tile -> smem, 128B swizzle, zero rows past rows_valid
        {
            constexpr int CPR = D / 8;                 // 16-byte chunks per row
            constexpr int RPP = 128 / CPR;             // rows per pass
            const int chunk = wtid % CPR, rsub = wtid / CPR;
#pragma unroll 4
            for (int i = 0; i < BM / RPP; ++i) {
                const int rr = i * RPP + rsub;
                uint4 v = make_uint4(0, 0, 0, 0);
                if (rr < it.rows_valid) {
                    const int rg = it.row0 + rr;
                    const int tl = rg / p.G, hh = rg - tl * p.G;
                    v = __ldg(reinterpret_cast<const uint4*>(p.q + ((int64_t)(it.q_start + tl) * p.Hq + it.g * p.G + hh) * D) + chunk);
                }
                const int slab = chunk >> 3, c16 = chunk & 7;
                *reinterpret_cast<uint4*>(smem + L::OFF_Q + slab * SLAB + rr * 128 + ((c16 ^ (rr & 7)) << 4)) = v;
            }
            ptx::fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(L::B_Q_FULL));
        }
        const bool warp_active = wg_warp * 32 < it.rows_valid;
        const int n = it.kv1 - it.kv0;
        float m = -INFINITY, l = 0.f;
        for (int j = 0; j < n; ++j) {
            if (*abort_flag) break;
            const uint32_t sb = tcount & 1u;
            ptx::mbar_wait(bar(L::B_S_FULL + sb), (tcount >> 1) & 1u, abort_flag);
            ptx::tc_fence_after();
            int nv = it.c - (it.kv0 + j) * BN;
            nv = nv > BN ? BN : nv;
            float alpha = 1.f;
            const uint32_t s_taddr = tmem + lane_base + sb * 128u;
            if (warp_active) {
                uint32_t pk[64];
                if (nv == BN) softmax_row<false>(s_taddr, nv, p.scale_log2, m, l, alpha, pk);
                else softmax_row<true>(s_taddr, nv, p.scale_log2, m, l, alpha, pk);
                ptx::tmem_st32(s_taddr, *reinterpret_cast<const uint32_t(*)[32]>(&pk[0]));
                ptx::tmem_st32(s_taddr + 32u, *reinterpret_cast<const uint32_t(*)[32]>(&pk[32]));
            }
            if (j > 0) {
                ptx::mbar_wait(bar(L::B_PV_DONE), (tcount - 1u) & 1u, abort_flag);
                ptx::tc_fence_after();
                if (warp_active && __any_sync(FULL, alpha != 1.f)) {
#pragma unroll
                    for (int c = 0; c < D / 32; ++c) {
                        uint32_t o[32];
                        ptx::tmem_ld32(o_taddr + (uint32_t)(c * 32), o);
                        ptx::tmem_wait_ld();
#pragma unroll
                        for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
                        ptx::tmem_st32(o_taddr + (uint32_t)(c * 32), o);
                    }
                }
            }
            ptx::tmem_wait_st();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar(L::B_P_FULL + sb));
            ++tcount;
        }
        if (n > 0) {
            ptx::mbar_wait(bar(L::B_PV_DONE), (tcount - 1u) & 1u, abort_flag);
            ptx::tc_fence_after();
        }
        // ---- epilogue (TMEM loads are warp-collective: predicate only the global stores)
        if (warp_active) {
            const bool row_ok = row < it.rows_valid;
            if (it.part_slot < 0) {
                const float inv = (n > 0 && l > 0.f) ? 1.f / l : 0.f;
                const int rg = it.row0 + row;
                const int tl = rg / p.G, hh = rg - tl * p.G;
                uint4* dst = reinterpret_cast<uint4*>(p.out + ((int64_t)(it.q_start + tl) * p.Hq + it.g * p.G + hh) * D);
#pragma unroll
                for (int c = 0; c < D / 32; ++c) {
                    uint32_t o[32];
                    if (n > 0) {
                        ptx::tmem_ld32(o_taddr + (uint32_t)(c * 32), o);
                        ptx::tmem_wait_ld();
                    } else {
#pragma unroll
                        for (int i = 0; i < 32; ++i) o[i] = 0u;
                    }
                    if (row_ok) {
#pragma unroll
                        for (int v = 0; v < 4; ++v) {
                            uint4 w;
                            w.x = ptx::pack_bf16(__uint_as_float(o[v * 8 + 0]) * inv, __uint_as_float(o[v * 8 + 1]) * inv);
                            w.y = ptx::pack_bf16(__uint_as_float(o[v * 8 + 2]) * inv, __uint_as_float(o[v * 8 + 3]) * inv);
                            w.z = ptx::pack_bf16(__uint_as_float(o[v * 8 + 4]) * inv, __uint_as_float(o[v * 8 + 5]) * inv);
                            w.w = ptx::pack_bf16(__uint_as_float(o[v * 8 + 6]) * inv, __uint_as_float(o[v * 8 + 7]) * inv);
                            dst[c * 4 + v] = w;
                        }
                    }
                }
            } else {
                float* po = p.part_o + ((int64_t)it.part_slot * BM + row) * D;
#pragma unroll
                for (int c = 0; c < D / 32; ++c) {
                    uint32_t o[32];
                    ptx::tmem_ld32(o_taddr + (uint32_t)(c * 32), o);
                    ptx::tmem_wait_ld();
                    if (row_ok) {
#pragma unroll
                        for (int v = 0; v < 8; ++v)
                            reinterpret_cast<uint4*>(po)[c * 8 + v] = make_uint4(o[v * 4], o[v * 4 + 1], o[v * 4 + 2], o[v * 4 + 3]);
                    }
                }
                if (row_ok) reinterpret_cast<float2*>(p.part_ml)[(int64_t)it.part_slot * BM + row] = make_float2(m, l);
            }
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar(L::B_ITEM_EMPTY + islot));
        ++icount;
    }
}


// ------------------------------------------------------------------------------------------------
// kernel entry
// ------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(NTHREADS, 1)
attn_kernel(const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV, const AttnParams p) {
    using L = Smem<D>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    const uint32_t sbase = ptx::smem_u32(smem);
    Item* items = reinterpret_cast<Item*>(smem + L::OFF_ITEMS);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::OFF_MISC);
    volatile uint32_t* abort_flag = reinterpret_cast<volatile uint32_t*>(smem + L::OFF_MISC + 4);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
        for (int s = 0; s < NSTAGE; ++s) { ptx::mbar_init(bar(L::B_KV_FULL + s), 1); ptx::mbar_init(bar(L::B_KV_EMPTY + s), 1); }
        for (int s = 0; s < 2; ++s) {
            ptx::mbar_init(bar(L::B_ITEM_FULL + s), 1);
            ptx::mbar_init(bar(L::B_ITEM_EMPTY + s), 5);   // MMA lane + 4 softmax warps
            ptx::mbar_init(bar(L::B_S_FULL + s), 1);
            ptx::mbar_init(bar(L::B_P_FULL + s), 4);
        }
        ptx::mbar_init(bar(L::B_Q_FULL), 4);
        ptx::mbar_init(bar(L::B_PV_DONE), 1);
        *abort_flag = 0u;
        ptx::fence_mbar_init();
        ptx::prefetch_tensormap(&mapK);
        ptx::prefetch_tensormap(&mapV);
    }
    if (warp == 2) {
        ptx::tmem_alloc(ptx::smem_u32(tmem_slot), 512);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp == 0) {
        producer_warp<D>(p, reinterpret_cast<SlotMeta*>(p.slot_meta), &mapK, &mapV, sbase, items, abort_flag, lane);
    } else if (warp == 1) {
        mma_warp<D>(p, sbase, tmem, items, abort_flag, lane);
    } else if (warp >= 4) {
        softmax_wg<D>(p, smem, sbase, tmem, items, abort_flag, warp - 4, lane);
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (tid == 0 && *abort_flag) raise_flag(p.flags, DEV_TIMEOUT);
    if (warp == 2) ptx::tmem_dealloc(tmem, 512);
}

// ------------------------------------------------------------------------------------------------
// combine (a9): merge the split-KV partials of one unit.  Block b owns the unit whose head piece
// is in slot 2b+1; continuation pieces are slots 2b' of CTAs b' in (b, b_last].  Fixed order, no
// atomics: bitwise reproducible.  m is in log2 units:
//   m* = max m_i;  l* = sum l_i 2^(m_i-m*);  O* = sum O_i 2^(m_i-m*);  out = bf16(O*/l*)
// ------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(256)
combine_kernel(const AttnParams p) {
    const SlotMeta* meta = reinterpret_cast<const SlotMeta*>(p.slot_meta);
    const int b = blockIdx.x;
    const SlotMeta h = meta[2 * b + 1];
    if (!h.valid) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int EPL = D / 32;
    const float2* ml = reinterpret_cast<const float2*>(p.part_ml);
    for (int row = warp; row < h.rows_valid; row += 8) {
        float ms = ml[(int64_t)(2 * b + 1) * BM + row].x;
        for (int bb = b + 1; bb <= h.b_last; ++bb)
            if (meta[2 * bb].valid) ms = fmaxf(ms, ml[(int64_t)(2 * bb) * BM + row].x);
        float acc[EPL];
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] = 0.f;
        float ls = 0.f;
        for (int bb = b; bb <= h.b_last; ++bb) {
            const int slot = bb == b ? 2 * b + 1 : 2 * bb;
            if (bb != b && !meta[slot].valid) continue;
            const float2 x = ml[(int64_t)slot * BM + row];
            const float w = ptx::ex2(x.x - ms);
            ls += x.y * w;
            const float* po = p.part_o + ((int64_t)slot * BM + row) * D + lane * EPL;
#pragma unroll
            for (int e = 0; e < EPL; ++e) acc[e] += po[e] * w;
        }
        const float inv = ls > 0.f ? 1.f / ls : 0.f;
        const int rg = h.row0 + row;
        const int tl = rg / p.G, hh = rg - tl * p.G;
        __nv_bfloat16* dst = p.out + ((int64_t)(h.q_start + tl) * p.Hq + h.g * p.G + hh) * D + lane * EPL;
#pragma unroll
        for (int e = 0; e < EPL; ++e) dst[e] = __float2bfloat16(acc[e] * inv);
    }
}

}  // namespace tc

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
static inline cudaError_t tc_configure(int head_dim) {
    if (head_dim == 128)
        return cudaFuncSetAttribute(tc::attn_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, tc::Smem<128>::ALLOC);
    return cudaFuncSetAttribute(tc::attn_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, tc::Smem<64>::ALLOC);
}

typedef CUresult (*sangam_encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                     const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                     CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// Pool viewed as a 2-D tensor [P*Hkv*16 rows][D] bf16; one box = 16 rows (a page of one head) x 64 columns,
// 128-byte swizzled: exactly one UMMA swizzle slab of a page.
static inline int tc_encode_maps(TcMaps* maps, const void* k_pages, const void* v_pages, int num_pages, int Hkv, int D) {
    static sangam_encode_fn enc = nullptr;
    if (!enc) {
        cudaDriverEntryPointQueryResult q;
        void* fn = nullptr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn) return -1;
        enc = reinterpret_cast<sangam_encode_fn>(fn);
    }
    const cuuint64_t gdim[2] = {(cuuint64_t)D, (cuuint64_t)num_pages * Hkv * SANGAM_PAGE};
    const cuuint64_t gstr[1] = {(cuuint64_t)D * 2};
    const cuuint32_t box[2] = {64, SANGAM_PAGE}, estr[2] = {1, 1};
    const void* ptrs[2] = {k_pages, v_pages};
    CUtensorMap* out[2] = {&maps->k, &maps->v};
    for (int i = 0; i < 2; ++i) {
        CUresult r = enc(out[i], CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptrs[i]), gdim, gstr, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return -1;
    }
    return 0;
}

static inline cudaError_t tc_launch(const AttnParams& p, const TcMaps& maps, int head_dim, int sm_count,
                                    cudaStream_t stream, int* launched) {
    *launched = 0;
    if (head_dim == 128) {
        tc::attn_kernel<128><<<sm_count, tc::NTHREADS, tc::Smem<128>::ALLOC, stream>>>(maps.k, maps.v, p);
        tc::combine_kernel<128><<<sm_count, 256, 0, stream>>>(p);
    } else {
        tc::attn_kernel<64><<<sm_count, tc::NTHREADS, tc::Smem<64>::ALLOC, stream>>>(maps.k, maps.v, p);
        tc::combine_kernel<64><<<sm_count, 256, 0, stream>>>(p);
    }
    *launched = 2;
    return cudaGetLastError();
}
