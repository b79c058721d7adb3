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

}  // namespace tc
