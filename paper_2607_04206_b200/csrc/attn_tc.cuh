// attn_tc.cuh -- steps a3..a9: paged, varlen, non-causal block attention on tcgen05 (sm_100a).
//
// One persistent CTA per SM, 12 warps, warp-specialised, TWO softmax streams per CTA:
//   warp 9      scheduler + TMA producer: plans the work on the device (a3) and gathers K/V pages of
//               the current (request, kv head) through the block table with TMA into a ring of
//               128-row, 128B-swizzled shared-memory tiles (a4)
//   warp 8      Q loader (TMA, 2-slot ring of 128-row q tiles); also owns the TMEM allocation
//   warps 10,11 MMA issuers, one per stream s: S_s = Q_s K^T (tcgen05.mma, operands in smem, S in
//               TMEM; a5) and O_s += P_s V (P read from TMEM, V from smem, O in TMEM; a7)
//   warps 0-3   softmax warpgroup of stream 0;  warps 4-7: stream 1.  Thread i owns row i of the
//               stream's tile (TMEM lane i): online softmax in fp32 with a lazily updated reference
//               maximum (a6), P written back over S as bf16, epilogue (a8), fused split-KV merge (a9)
// Work unit = (request r, kv head g, PAIR of 128-row tiles of the packed rows).  Two modes per unit:
//   SHARED  (more than 128 rows in the pair): stream s owns q tile s, both streams consume the same
//           K/V tile -- the G q heads of a GQA group and the two q tiles share every K/V byte.
//   SPLIT   (at most 128 rows): both streams work on the one q tile, stream s takes the kv tiles
//           kv0 + 2i + s; the two partial results are merged in the epilogue (in-CTA split-KV).
// While one stream's warpgroup runs its softmax the tensor pipe works for the other stream.
// A unit's kv range may also be split across CTAs (static stream-K partition for decode-sized
// batches): pieces go to the workspace as (O fp32, m, l) and the CTA that finishes a unit's last
// piece merges them in fixed slot order (bitwise reproducible).  With many units (prefill / hybrid)
// whole units are handed out dynamically.
// The attention definition is PAPER.md:67 (no causal mask) over the context of PAPER.md:33.
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "ptx.cuh"

#ifdef SANGAM_DEBUG_ITEM
__device__ int g_bad_item[16];
#endif

namespace tc {

constexpr int BM = 128;          // rows per q tile  (UMMA M)
constexpr int BN = 128;          // kv positions per tile (8 pages)
constexpr int PAIR = 2 * BM;     // packed rows per work unit
constexpr int NSTAGE = 5;        // K/V tile ring depth
constexpr int NTHREADS = 384;
constexpr int SLAB = 128 * 128;  // bytes of one 64-wide swizzled slab of a 128-row q tile
// K/V stages are PAGE-major: one TMA box = one whole (page, head) = 16 rows x D, landing as 2 row groups x D/64
// slabs of 8-row x 128-byte swizzle atoms.  Atom (8-row group j, slab t) of a stage sits at j * KV_ATOM_STRIDE + t * 1024,
// so the 8-row groups of one slab are KV_ATOM_STRIDE apart (the descriptors' SBO) and the slabs 1024 bytes (V's LBO).
template <int D> constexpr int KV_ATOM_STRIDE = 1024 * (D / 64);
#ifndef SANGAM_DYN_UNITS
#define SANGAM_DYN_UNITS 4
#endif
constexpr int DYN_UNITS_PER_CTA = SANGAM_DYN_UNITS;   // >= this many units per CTA: whole units, dynamic hand-out
#ifndef SANGAM_UNIT_OV
#define SANGAM_UNIT_OV 1
#endif
constexpr int UNIT_OV = SANGAM_UNIT_OV;  // static partition: fixed cost of starting/finishing a unit, in kv-tile equivalents
constexpr float LAZY_T = 8.f;    // the reference maximum moves only when a tile exceeds it by 2^8

struct Item {          // one piece of work, published through shared memory (64 bytes)
    int valid;         // 0 = no more work
    int r, g;
    int tok0;          // first query token (inside the request) of the pair of q tiles
    int rows0, rows1;  // rows (tokens * G) of q tile 0 / 1 that exist; rows1 > 0 <=> SHARED mode
    int q_start;       // cu_q_lens[r]
    int c;             // context length
    int kv0, kv1;      // kv tile range [kv0, kv1)
    int part_slot;     // -1: write `out`; else partial slot in the workspace
    int b_head;        // split units: CTA holding the piece that starts at kv tile 0
    int npieces;       // split units: number of CTAs holding a piece
    int pad0, pad1, pad2;
};

struct SlotMeta {      // global, one per CTA: the split unit whose head piece (kv tile 0) this CTA computed, if any
    int valid;
    int npieces;       // CTAs b .. b + npieces - 1 hold its pieces: slot 2b+1, then slots 2(b+1), 2(b+2), ..
    int g, tok0, rows0, rows1, q_start;
    int pad0;
};

template <int D>
struct Smem {
    static constexpr int Q_BYTES = BM * D * 2;
    static constexpr int KV_BYTES = BN * D * 2;
    static constexpr int OFF_Q = 0;                       // 2 q-tile slots
    static constexpr int OFF_KV = 2 * Q_BYTES;
    static constexpr int OFF_BAR = OFF_KV + NSTAGE * KV_BYTES;
    // barrier indices
    static constexpr int B_KV_FULL = 0, B_KV_EMPTY = NSTAGE, B_ITEM_FULL = 2 * NSTAGE, B_ITEM_EMPTY = B_ITEM_FULL + 2,
                         B_Q_FULL = B_ITEM_EMPTY + 2, B_Q_EMPTY = B_Q_FULL + 2, B_S_FULL = B_Q_EMPTY + 2,   // [stream][half]
                         B_P_FULL = B_S_FULL + 4, B_PV_DONE = B_P_FULL + 4, B_EPI_A = B_PV_DONE + 4,
                         B_EPI_B = B_EPI_A + 1, B_ZFILL = B_EPI_B + 1, NBAR = B_ZFILL + 1;
    static constexpr int OFF_ITEMS = OFF_BAR + ((NBAR * 8 + 15) / 16) * 16;
    static constexpr int OFF_ML = OFF_ITEMS + 2 * (int)sizeof(Item);    // (m, l) of stream 1, 128 rows
    static constexpr int OFF_MISC = OFF_ML + BM * 8;
    static constexpr int OFF_SEQ = OFF_MISC + 16 + 64;   // tmem slot, abort word, pad; per-warp wait table (diagnostics)
    static constexpr int TOTAL = OFF_SEQ + 32;           // kv_seq[NSTAGE]
#ifdef SANGAM_TRACE
    static constexpr int ALLOC = TOTAL;          // debug trace builds: their static shared memory takes the slack (2 KB static: the base stays aligned)
#else
    static constexpr int ALLOC = TOTAL + 1024;   // slack to align the base to 1024 B (128B swizzle atoms)
#endif
};
static_assert(sizeof(Item) == 64, "Item is 64 bytes");
static_assert(Smem<128>::ALLOC <= 232448, "shared memory budget (227 KB)");

// floor(a * b / d) and ceil(a * b / d) for the static partition.  32-bit arithmetic only (a 64-bit division is some
// 150 instructions of cold code per call site): the static partition is used only while T * #CTAs < 2^31, larger
// batches are handed out dynamically.
__device__ __forceinline__ int mul_div(int a, int b, int d) { return (int)(((uint32_t)a * (uint32_t)b) / (uint32_t)d); }
__device__ __forceinline__ int mul_div_ceil(int a, int b, int d) { return (int)(((uint32_t)a * (uint32_t)b + (uint32_t)d - 1u) / (uint32_t)d); }

struct ReqInfo {
    int q0, qn, c, np, tiles_u, units;
};

// Request metadata of the batch, read once: lane r of the producer warp keeps request r (< 32) in registers
// and every later look-up is a shuffle.  (With 227 KB of shared memory the L1 holds next to nothing, so a
// repeated global read costs an L2 round trip each time.)  Requests >= 32 are read from global memory.
struct ReqCache {
    int q0, qn, c;      // of request `lane`
    __device__ __forceinline__ static void load(const AttnParams& p, int r, int& q0, int& qn, int& c) {
        q0 = __ldg(p.cu_q_lens + r);
        qn = __ldg(p.cu_q_lens + r + 1) - q0;
        if (qn < 0) qn = 0;
        c = __ldg(p.ctx_lens + r);
        if (c < 0) c = 0;
        if ((c + SANGAM_PAGE - 1) / SANGAM_PAGE > p.W) { raise_flag(p.flags, DEV_CTX_TOO_LONG); c = 0; }
    }
    __device__ __forceinline__ void init(const AttnParams& p, int lane) {
        q0 = 0; qn = 0; c = 0;
        if (lane < p.batch) load(p, lane, q0, qn, c);
    }
    __device__ __forceinline__ static ReqInfo derive(const AttnParams& p, int q0_, int qn_, int c_) {
        ReqInfo x;
        x.q0 = q0_; x.qn = qn_; x.c = c_;
        // a q tile holds tpt = 128 / G whole tokens (all G heads of each); ceil(qn / (2 tpt)) by the host's magic
        // multiplier (exact for qn < 2^24): an integer division is ~25 instructions at each of this function's call sites
        x.np = (int)__umulhi((uint32_t)(qn_ + 2 * p.tpt - 1), p.tpt2_magic);
        const int nkv = (c_ + BN - 1) / BN;
        x.tiles_u = nkv > 0 ? nkv : 1;
        x.units = p.Hkv * x.np;
        return x;
    }
    // warp-uniform r: all 32 lanes call
    __device__ __forceinline__ ReqInfo get(const AttnParams& p, int r) const {
        int a, b, d;
        if (r < 32) {
            a = __shfl_sync(0xffffffffu, q0, r); b = __shfl_sync(0xffffffffu, qn, r); d = __shfl_sync(0xffffffffu, c, r);
        } else {
            load(p, r, a, b, d);
        }
        return derive(p, a, b, d);
    }
    // per-lane r = base + lane (r < batch)
    __device__ __forceinline__ ReqInfo get_lane(const AttnParams& p, int base, int lane) const {
        if (base == 0) return derive(p, q0, qn, c);
        int a, b, d;
        load(p, base + lane, a, b, d);
        return derive(p, a, b, d);
    }
};

// Order in which the K/V tiles of one item pass through the shared-memory ring (producer loads, issuers consume):
//   K(0) .. K(lead-1),  then for j = 0, 1, ..:  V(j), K(j + lead)        lead = 1 (SHARED) or 2 (SPLIT)
// SHARED: both issuers read every stage.  SPLIT: tile j belongs to stream j & 1, the other issuer skips it.

// ------------------------------------------------------------------------------------------------
// warp 9: device-side plan (a3) + TMA page gather (a4)
// ------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void producer_warp(const AttnParams& p, const CUtensorMap* mapK, const CUtensorMap* mapV,
                                              uint32_t sbase, Item* items, volatile uint32_t* abort_flag,
                                              volatile uint32_t* kv_seq, int lane) {
    using L = Smem<D>;
    const unsigned FULL = 0xffffffffu;
    const int G_ctas = gridDim.x, b = blockIdx.x, R = p.batch;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    SlotMeta* meta = reinterpret_cast<SlotMeta*>(p.slot_meta);
    if (lane == 0) meta[b].valid = 0;
    TRACE_EV(50);

    // Plan cache: a model runs the same batch metadata through all of its layers, and a captured graph is replayed, so
    // every CTA keeps its last plan in the workspace, keyed by the lengths it was derived from ((q0, qn, c) of up to 32
    // requests, batch size, grid size); private to the CTA, so there is no race inside a launch.  The cached words are
    // requested together with the lengths: a hit replaces ~3 000 clk of serial planning by one compare.
    int32_t* pc = p.plan_cache + (size_t)b * PLAN_CACHE_INTS;
    const bool cacheable = R <= 32;
    bool hit = false;
    int4 h0 = make_int4(0, 0, 0, 0), h1 = h0, h2 = h0;
    int k0 = 0, k1 = 0, k2 = 0;
    if (cacheable) {
        k0 = pc[lane * 3]; k1 = pc[lane * 3 + 1]; k2 = pc[lane * 3 + 2];
        h0 = *reinterpret_cast<const int4*>(pc + 96);      // R + 1 (0: empty), #CTAs, U, T
        h1 = *reinterpret_cast<const int4*>(pc + 100);     // dynamic, r_cur, u_in_r, kvoff
        h2 = *reinterpret_cast<const int4*>(pc + 104);     // remaining, tile_base, Geff, ubase
    }
    ReqCache rc;
    rc.init(p, lane);
    TRACE_EV(59);
    if (cacheable) {
        const bool same = lane >= R || (k0 == rc.q0 && k1 == rc.qn && k2 == rc.c);
        hit = __all_sync(FULL, same) && h0.x == R + 1 && h0.y == G_ctas;
    }
    // totals over the batch: units U and kv tiles T
    int U = 0, T = 0;
    if (hit) {
        U = h0.z; T = h0.w;
    } else {
        for (int base = 0; base < R; base += 32) {
            if (base + lane < R) {
                const ReqInfo x = rc.get_lane(p, base, lane);
                U += x.units;
                T += x.units * (x.tiles_u + UNIT_OV);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            U += __shfl_xor_sync(FULL, U, o);
            T += __shfl_xor_sync(FULL, T, o);
        }
    }
    const bool dynamic = hit ? h1.x != 0 : (U >= DYN_UNITS_PER_CTA * G_ctas || T >= (int)(0x7fffffffu / (uint32_t)(G_ctas + 1)));
    TRACE_EV(51);

    // walking state
    int r_cur = 0, ubase = 0, u_in_r = 0, kvoff = 0, remaining = 0, tile_base = 0, Geff = 1;
    ReqInfo cur = ReqCache::derive(p, 0, 0, 0);
    cur.units = 0;
    if (hit) {
        r_cur = h1.y; u_in_r = h1.z; kvoff = h1.w; remaining = h2.x; tile_base = h2.y; Geff = h2.z; ubase = h2.w;
        if (r_cur < R) cur = rc.get(p, r_cur);
    } else {
    if (R > 0) cur = rc.get(p, 0);
    if (dynamic && R > 0) {                            // dynamic tickets walk downwards from the last request
        r_cur = R - 1;
        cur = rc.get(p, r_cur);
        ubase = U - cur.units;
    }
    TRACE_EV(55);
    if (!dynamic && T > 0) {
        Geff = G_ctas < T ? G_ctas : T;
        if (b < Geff) {
            const int t0 = mul_div(b, T, Geff), t1 = mul_div(b + 1, T, Geff);
            remaining = t1 - t0;
            TRACE_EV(56);
            // locate the request holding flattened tile t0 (chunked warp scan over requests)
            int acc = 0, found = -1;
            for (int base = 0; base < R && found < 0; base += 32) {
                int tl = 0;
                if (base + lane < R) { const ReqInfo x = rc.get_lane(p, base, lane); tl = x.units * (x.tiles_u + UNIT_OV); }
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
            TRACE_EV(57);
            r_cur = found < 0 ? R : found;
            if (r_cur < R) {
                cur = rc.get(p, r_cur);
                const int pos = t0 - tile_base;
                u_in_r = pos / (cur.tiles_u + UNIT_OV);
                kvoff = pos - u_in_r * (cur.tiles_u + UNIT_OV);
            } else {
                remaining = 0;
            }
        }
    }
    if (cacheable) {                                   // remember the plan (this CTA's own entry)
        pc[lane * 3] = rc.q0; pc[lane * 3 + 1] = rc.qn; pc[lane * 3 + 2] = rc.c;
        if (lane == 0) {
            *reinterpret_cast<int4*>(pc + 96) = make_int4(R + 1, G_ctas, U, T);
            *reinterpret_cast<int4*>(pc + 100) = make_int4(dynamic ? 1 : 0, r_cur, u_in_r, kvoff);
            *reinterpret_cast<int4*>(pc + 104) = make_int4(remaining, tile_base, Geff, ubase);
        }
    }
    }
    TRACE_EV(52);

    uint32_t stage = 0, phase = 0, pos = 0, icount = 0;   // next K/V ring position: stage, parity, running index
    while (true) {
        if (*abort_flag) break;
        Item it;
        it.valid = 0; it.r = 0; it.g = 0; it.tok0 = 0; it.rows0 = 0; it.rows1 = 0; it.q_start = 0; it.c = 0;
        it.kv0 = 0; it.kv1 = 0; it.part_slot = -1; it.b_head = 0; it.npieces = 1; it.pad0 = 0; it.pad1 = 0; it.pad2 = 0;
        ReqInfo ri = cur;                               // the request of this item
        if (dynamic) {
            int u = 0;
            if (lane == 0) u = atomicAdd(p.sched, 1);
            u = __shfl_sync(FULL, u, 0);
            if (u < U) {
                // Tickets walk the unit list from the END: Alg. 1 batches seat decodes first and prefills last
                // (PAPER.md:181-190), so the long prefill units start first and the short decode units fill the
                // tail of the launch (longest-first balance).
                const int uu = U - 1 - u;
                while (r_cur > 0 && uu < ubase) {
                    --r_cur;
                    cur = rc.get(p, r_cur);
                    ubase -= cur.units;
                }
                if (r_cur < R) {
                    const int ul = uu - ubase;
                    it.valid = 1; it.r = r_cur; it.g = ul / cur.np;
                    it.tok0 = (ul - it.g * cur.np) * 2 * p.tpt;
                    it.kv0 = 0; it.kv1 = cur.tiles_u;
                    ri = cur;
                }
            }
        } else {
            // static partition: this CTA owns the weighted coordinates [x0, x1) of the flattened unit list; a unit
            // spans UNIT_OV + tiles_u of them, coordinate UNIT_OV + j being its kv tile j.  A range that covers only
            // part of a unit's overhead span yields no work there.
            while (remaining > 0 && r_cur < R && !it.valid) {
                const int wu = cur.tiles_u + UNIT_OV;
                const int take = remaining < wu - kvoff ? remaining : wu - kvoff;
                const int a = kvoff > UNIT_OV ? kvoff - UNIT_OV : 0, e = kvoff + take > UNIT_OV ? kvoff + take - UNIT_OV : 0;
                if (e > a) {
                    it.valid = 1; it.r = r_cur; it.g = u_in_r / cur.np;
                    it.tok0 = (u_in_r - it.g * cur.np) * 2 * p.tpt;
                    it.kv0 = a; it.kv1 = e;
                    ri = cur;
                    if (!(a == 0 && e == cur.tiles_u)) {
                        // a piece of a unit split across CTAs: CTA x owns coordinates [floor(xT/Geff), floor((x+1)T/Geff))
                        it.part_slot = 2 * b + (a == 0 ? 1 : 0);
                        const int ut0 = tile_base + u_in_r * wu + UNIT_OV;           // coordinate of kv tile 0; < T < 2^31
                        const int bh = mul_div_ceil(ut0 + 1, Geff, T) - 1;
                        int bl = mul_div_ceil(ut0 + cur.tiles_u, Geff, T) - 1;
                        bl = bl > Geff - 1 ? Geff - 1 : bl;
                        it.b_head = bh;
                        it.npieces = bl - bh + 1;
                    }
                }
                remaining -= take;
                kvoff += take;
                if (kvoff == wu) {
                    kvoff = 0;
                    if (++u_in_r == cur.units) {
                        u_in_r = 0;
                        do {
                            tile_base += cur.units * wu;
                            ++r_cur;
                            if (r_cur < R) cur = rc.get(p, r_cur);
                        } while (r_cur < R && cur.units == 0);
                    }
                }
            }
        }
        if (it.valid) {
            const int left = ri.qn - it.tok0;
            it.rows0 = (left < p.tpt ? left : p.tpt) * p.G;
            it.rows1 = left > p.tpt ? (left - p.tpt < p.tpt ? left - p.tpt : p.tpt) * p.G : 0;
            it.q_start = ri.q0;
            it.c = ri.c;
            if (ri.c == 0) { it.kv0 = 0; it.kv1 = 0; }
            if (it.part_slot >= 0 && it.kv0 == 0 && lane == 0) {      // head piece: tell combine_kernel what to merge
                SlotMeta mm;
                mm.valid = 1; mm.npieces = it.npieces; mm.g = it.g; mm.tok0 = it.tok0; mm.rows0 = it.rows0; mm.rows1 = it.rows1;
                mm.q_start = it.q_start; mm.pad0 = it.r;
                meta[b] = mm;
            }
        }
        TRACE_EV(58);
        // publish
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_EMPTY + islot), ((icount >> 1) & 1u) ^ 1u, abort_flag);
        if (lane == 0) {
            items[islot] = it;
            ptx::mbar_arrive(bar(L::B_ITEM_FULL + islot));
        }
        __syncwarp();
        TRACE_EV(53);
        ++icount;
        if (!it.valid) break;

        // K/V tile loads in ring order (see above).  The block-table entries of a tile serve its K and its V load
        // and are fetched ahead: lane pg (< 8) keeps page pg of the tiles in flight in the window w0 .. w3.
        const int n = it.kv1 - it.kv0;
        if (n > 0) {
            const int pages_total = (it.c + SANGAM_PAGE - 1) / SANGAM_PAGE;
            const int32_t* bt = p.block_table + (int64_t)it.r * p.W;
            const int pg = lane;                         // one box per page: lanes 0..7 issue
            const int lead = it.rows1 > 0 ? 1 : 2;
            auto ld_page = [&](int j) {                  // page pg of the item's j-th tile (0 if it does not exist)
                const int tile = it.kv0 + j;
                return (j < n && pg < 8 && pg < pages_total - tile * 8) ? __ldg(bt + tile * 8 + pg) : 0;
            };
            // One loop, one copy of the load code (instruction footprint): K runs `lead` tiles ahead of V.  The page
            // ids of the tiles in flight (at most lead + 2) live in a 4-entry register window indexed by tile & 3; the
            // entry of tile kq + 1 is fetched while tile kq's K load is issued, one K step before it is needed.
            int w0 = ld_page(0), w1 = ld_page(1), w2 = 0, w3 = 0;
            int kq = 0, vq = 0;
            while (vq < n) {
                const bool is_v = !(kq < n && kq < vq + lead);
                const int j = is_v ? vq : kq;
                const int sel = j & 3;
                const int page = sel == 0 ? w0 : sel == 1 ? w1 : sel == 2 ? w2 : w3;
                const int tile = it.kv0 + j;
                ptx::mbar_wait(bar(L::B_KV_EMPTY + stage), phase ^ 1u, abort_flag);
                int np = pages_total - tile * 8;
                np = np > 8 ? 8 : np;
                if (lane == 0) {
                    kv_seq[stage] = pos;                     // the issuers check this before trusting the barrier's parity
                    ptx::mbar_arrive_expect_tx(bar(L::B_KV_FULL + stage), (uint32_t)(np * SANGAM_PAGE * D * 2));
                }
                ++pos;
                __syncwarp();
                if (pg < np) {
                    // a page id outside [0, P): flag, and address the first box past the pool -- TMA fills zeros, so the
                    // page's 16 positions read as K = V = 0 (sangam.h; the same in attn_dec.cuh and attn_simt.cuh)
                    const bool bad = (unsigned)page >= (unsigned)p.P;
                    if (bad) raise_flag(p.flags, DEV_BAD_PAGE);
                    ptx::tma_load_4d(sbase + (uint32_t)(L::OFF_KV + stage * L::KV_BYTES + pg * (2 * KV_ATOM_STRIDE<D>)),
                                     is_v ? mapV : mapK, bar(L::B_KV_FULL + stage), 0, 0, 0, ((bad ? p.P : page) * p.Hkv + it.g) * 2);
                }
                TRACE_EV(54);
                if (++stage == NSTAGE) { stage = 0; phase ^= 1u; }
                if (is_v) {
                    ++vq;
                } else {
                    ++kq;
                    const int nx = ld_page(kq + 1), s2 = (kq + 1) & 3;       // prefetch for the K load after the next
                    if (s2 == 0) w0 = nx; else if (s2 == 1) w1 = nx; else if (s2 == 2) w2 = nx; else w3 = nx;
                }
                if (*abort_flag) break;
            }
        }
    }
    // Tail: every tcgen05.commit aimed at a KV_EMPTY barrier must have landed before this CTA may exit -- a late
    // asynchronous arrive would hit the shared memory of whatever CTA runs here next.
    for (int k = 0; k < NSTAGE; ++k) {
        ptx::mbar_wait(bar(L::B_KV_EMPTY + stage), phase ^ 1u, abort_flag);
        if (++stage == NSTAGE) { stage = 0; phase ^= 1u; }
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
// warp 8: Q loader.  q is viewed as a 3-D tensor [total_q][Hq][D]; one TMA box = 64 columns x the G heads
// of the group x tpt tokens lands as rows (token * G + head) of a K-major 128B-swizzled UMMA tile.
// Two q-tile slots form a ring; a slot is refilled as soon as the last QK reading it has completed.
// Rows past the request's last token hold the next request's tokens or TMA zero fill: never stored.
// ------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void qload_warp(const AttnParams& p, const CUtensorMap* mapQ, uint32_t sbase, const Item* items,
                                           volatile uint32_t* abort_flag, int lane) {
    using L = Smem<D>;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    const uint32_t tile_bytes = (uint32_t)(p.tpt * p.G * D * 2);
    uint32_t icount = 0, qcount = 0;
    while (true) {
        if (*abort_flag) break;
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_FULL + islot), (icount >> 1) & 1u, abort_flag);
        const Item it = items[islot];
        if (!it.valid) break;
        const int nq = it.kv1 > it.kv0 ? (it.rows1 > 0 ? 2 : 1) : 0;   // c = 0: no MMA, no q tile
        for (int t = 0; t < nq; ++t) {
            const uint32_t qs = qcount & 1u;
            ptx::mbar_wait(bar(L::B_Q_EMPTY + qs), ((qcount >> 1) & 1u) ^ 1u, abort_flag);
            if (lane == 0) ptx::mbar_arrive_expect_tx(bar(L::B_Q_FULL + qs), tile_bytes);
            __syncwarp();
            if (lane < D / 64)
                ptx::tma_load_3d(sbase + (uint32_t)(L::OFF_Q + qs * L::Q_BYTES + lane * SLAB), mapQ, bar(L::B_Q_FULL + qs),
                                 lane * 64, it.g * p.G, it.q_start + it.tok0 + t * p.tpt);
            ++qcount;
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar(L::B_ITEM_EMPTY + islot));
        ++icount;
    }
    // tail: the commits aimed at the Q_EMPTY barriers must have landed before the CTA exits
    for (int k = 0; k < 2; ++k, ++qcount)
        ptx::mbar_wait(bar(L::B_Q_EMPTY + (qcount & 1u)), ((qcount >> 1) & 1u) ^ 1u, abort_flag);
}

// ------------------------------------------------------------------------------------------------
// warps 10, 11: MMA issuers (a5, a7), one per softmax stream s.
// A 128-column kv tile is processed as two HALVES of 64 columns with their own S/P buffers in TMEM:
//   S_s,h = columns [128 s + 64 h, +64),  P_s,h (bf16, two per column) over the first 32 of them,
//   O_s   = columns [256 + 128 s, +D).
// Per stream the steps alternate A B A B ...; step k waits for P of its half, issues
//   O_s += P_s,h V(tile, half h)   and then   S_s,h = Q K(next tile, half h)^T
// so the softmax warpgroup always has the other half's logits waiting: it never idles on the tensor pipe.
// (Only the last kv tile of a context can lack half B: fewer than 65 valid columns.)
// The two issuers are independent; the in-order tensor pipe interleaves them.  K/V ring stages are consumed
// in the ring order stated above the producer: each issuer walks the whole order, acts on its own tiles and skips the rest.
// KV_EMPTY and Q_EMPTY expect two arrivals: SHARED stages / SPLIT q tiles are read by both issuers (one
// commit each), SPLIT stages / SHARED q tiles by one issuer (which commits twice).
// ------------------------------------------------------------------------------------------------
template <int D>
struct MmaState {
    uint32_t sbase, tmem;
    uint64_t q_desc0, k_desc0, v_desc0;
    uint32_t stage, phase, pos;       // next ring position: stage, parity, running index
    volatile uint32_t* kv_seq;        // [NSTAGE] position being loaded into each stage (written by the producer)
    uint32_t p_par0, p_par1;          // parity of the next P_FULL wait, half A / B
    uint32_t zf_par;                  // parity of the next ZFILL wait (SHARED tail tiles)
    volatile uint32_t* abort_flag;
    __device__ __forceinline__ uint32_t bar(int i) const { return sbase + (uint32_t)(Smem<D>::OFF_BAR + i * 8); }
    // Wait for ring position `pos` (stage = pos % NSTAGE).  In SPLIT mode an issuer does not consume every use
    // of a stage, and an mbarrier parity wait only tells adjacent phases apart (TMA loads complete out of order:
    // the skipped use may still be in flight when the next-but-one is awaited).  So the producer publishes the
    // position it is loading into each stage (kv_seq) and the issuer first waits for ITS position to be the one
    // in flight; from then on the barrier's current phase is exactly that load's.
    // (SHARED mode: both issuers consume every use of every stage, so the check is skipped there)
    __device__ __forceinline__ uint32_t acquire(bool check = true) {
        const uint32_t s0 = stage;
        if (check && kv_seq[s0] != pos) {              // the issuer is ahead of the producer
            uint32_t spins = 0;
            while (kv_seq[s0] != pos)
                if ((++spins & 0x3ffu) == 0 && *abort_flag) break;
        }
        ptx::mbar_wait(bar(Smem<D>::B_KV_FULL + s0), phase, abort_flag);
        skip();
        return s0;
    }
    // a ring position that belongs to the other issuer (SPLIT mode)
    __device__ __forceinline__ void skip() {
        ++pos;
        if (++stage == NSTAGE) { stage = 0; phase ^= 1u; }
    }
};

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

// valid (16-padded) columns of half h of kv tile `tile`; <= 0: the half does not exist
__device__ __forceinline__ int half_cols(int c, int tile, int h) {
    int nv = c - tile * BN;
    nv = nv > BN ? BN : nv;
    const int nc = ((nv + 15) & ~15) - h * 64;
    return nc > 64 ? 64 : nc;
}

// One step of stream s on half h:  [O_s (+)= P_s,h V]  then  [S_s,h = Q K^T].
// pv_cols / qk_cols = padded columns of the half (0: skip that part); rel_* = KV_EMPTY commits after the part
// (0 none, 1 stage shared with the other issuer, 2 sole reader); q_rel = Q_EMPTY commits after the QK.
template <int D>
__device__ __forceinline__ void half_step(MmaState<D>& st, int s, int h, int pv_cols, bool first_pv, uint32_t stage_v, int rel_v,
                                          int qk_cols, uint32_t stage_k, uint32_t qs, int rel_k, int q_rel) {
    using L = Smem<D>;
    TRACE_EV(60 + s);
    if (pv_cols > 0) {
        uint32_t& par = h ? st.p_par1 : st.p_par0;
        ptx::mbar_wait(st.bar(L::B_P_FULL + 2 * s + h), par, st.abort_flag);
        par ^= 1u;
    }
    ptx::tc_fence_after();
    TRACE_EV(62 + s);
    if (ptx::elect_one()) {
        const uint32_t sh_tmem = st.tmem + (uint32_t)(s * 128 + h * 64);          // S_s,h / P_s,h
        if (pv_cols > 0) {
            // K-steps of 16 kv rows = one page = two 8-row groups of V; half h starts 64 rows (8 groups) in
            constexpr uint32_t VSTEP = (uint32_t)(2 * KV_ATOM_STRIDE<D>) >> 4;
            const uint64_t b_desc = st.v_desc0 + (uint64_t)(stage_v * (L::KV_BYTES >> 4) + h * (4 * VSTEP));
            const uint32_t idesc = ptx::idesc_bf16(BM, D, 0, 1);
            const uint32_t d_tmem = st.tmem + 256u + (uint32_t)s * 128u;
            if (pv_cols == 64) {
                ptx::mma_ts_x4(d_tmem, sh_tmem, b_desc, idesc, first_pv ? 0u : 1u, VSTEP);
            } else {
                for (int ks = 0; ks < pv_cols / 16; ++ks)
                    ptx::mma_ts(d_tmem, sh_tmem + (uint32_t)(ks * 8), b_desc + (uint64_t)(ks * VSTEP), idesc, (!first_pv || ks > 0) ? 1u : 0u);
            }
            for (int i = 0; i < rel_v; ++i) ptx::mma_commit(st.bar(L::B_KV_EMPTY + stage_v));
            ptx::mma_commit(st.bar(L::B_PV_DONE + 2 * s + h));
        }
        if (qk_cols > 0) {
            // K-steps of 16 elements = 32 bytes inside a 64-wide slab; second slab SLAB bytes further in the q tile and
            // 1024 bytes further in the page-major K stage; half h of K = rows 64 h .. = 8 row groups in
            const uint64_t a_desc = st.q_desc0 + (uint64_t)(qs * (L::Q_BYTES >> 4));
            const uint64_t b_desc = st.k_desc0 + (uint64_t)(stage_k * (L::KV_BYTES >> 4) + h * ((8 * KV_ATOM_STRIDE<D>) >> 4));
            const uint32_t idesc = ptx::idesc_bf16(BM, (uint32_t)qk_cols, 0, 0);
            ptx::mma_ss_x4(sh_tmem, a_desc, b_desc, idesc, 0u, 2u);
            if (D == 128) ptx::mma_ss_x4(sh_tmem, a_desc + (SLAB >> 4), b_desc + (1024 >> 4), idesc, 1u, 2u);
            for (int i = 0; i < rel_k; ++i) ptx::mma_commit(st.bar(L::B_KV_EMPTY + stage_k));
            ptx::mma_commit(st.bar(L::B_S_FULL + 2 * s + h));
            for (int i = 0; i < q_rel; ++i) ptx::mma_commit(st.bar(L::B_Q_EMPTY + qs));
        }
    }
    __syncwarp();
    TRACE_EV(64 + s);
}

// all steps of stream s on kv tile `tile` (PV) and `next` (QK; next < 0: none).  rel = 1 (SHARED) or 2 (SPLIT);
// q_rel = Q_EMPTY commits owed when `next` is the stream's last tile.
template <int D>
__device__ __forceinline__ void tile_steps(MmaState<D>& st, int s, int c, int tile, bool first, uint32_t sv, int next, uint32_t sk,
                                           uint32_t qs, int rel, int q_rel) {
    const int pa = tile >= 0 ? half_cols(c, tile, 0) : 0, pb = tile >= 0 ? half_cols(c, tile, 1) : 0;
    const int qa = next >= 0 ? half_cols(c, next, 0) : 0, qb = next >= 0 ? half_cols(c, next, 1) : 0;
    half_step<D>(st, s, 0, pa, first, sv, pb > 0 ? 0 : rel, qa, sk, qs, qb > 0 ? 0 : rel, qb > 0 ? 0 : q_rel);
    if (pb > 0 || qb > 0) half_step<D>(st, s, 1, pb > 0 ? pb : 0, false, sv, rel, qb > 0 ? qb : 0, sk, qs, rel, q_rel);
}

struct SharedMode { static constexpr bool value = true; };
struct SplitMode { static constexpr bool value = false; };

template <int D>
__device__ __forceinline__ void mma_warp(const AttnParams& p, uint32_t sbase, uint32_t tmem, const Item* items,
                                         volatile uint32_t* abort_flag, uint32_t* kv_seq_smem, int s, int lane) {
    using L = Smem<D>;
    MmaState<D> st;
    st.sbase = sbase; st.tmem = tmem; st.abort_flag = abort_flag;
    st.q_desc0 = ptx::smem_desc_sw128(sbase + L::OFF_Q, 16, 1024);        // K-major operands (Q, K)
    st.k_desc0 = ptx::smem_desc_sw128(sbase + L::OFF_KV, 16, KV_ATOM_STRIDE<D>);
    st.v_desc0 = ptx::smem_desc_sw128(sbase + L::OFF_KV, 1024, KV_ATOM_STRIDE<D>);     // MN-major operand (V)
    st.stage = 0; st.phase = 0; st.pos = 0; st.kv_seq = reinterpret_cast<volatile uint32_t*>(kv_seq_smem);
    st.p_par0 = 0; st.p_par1 = 0; st.zf_par = 0;
    uint32_t icount = 0, qcount = 0;
    while (true) {
        if (*abort_flag) break;
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(st.bar(L::B_ITEM_FULL + islot), (icount >> 1) & 1u, abort_flag);
        const Item it = items[islot];
        if (!it.valid) break;
        TRACE_EV(1 + s);
        const int n = it.kv1 - it.kv0, c = it.c, kv0 = it.kv0;
        if (n > 0) {
            // One loop serves both modes (a single copy of the issue code: instruction footprint).
            //   SHARED: stream s = q tile s; ring order K_0 | V_0 K_1 | V_1 K_2 ..., every stage read by both issuers.
            //   SPLIT:  one q tile read by both issuers; stream x owns kv tiles kv0 + 2i + x and their stages; ring order
            //           K(0,0) [K(1,0)] | V(0,i) [K(0,i+1)] [V(1,i)] [K(1,i+1)] | ...
            // Round i = -1 is the prologue (first QK only); round i >= 0 issues PV of step i and QK of step i + 1.
            // (instantiated once per mode: the mode tests fold away in the hot SHARED loop of prefill)
            auto rounds = [&](auto shared_c) {
                constexpr bool shared = decltype(shared_c)::value;
                const int n0 = shared ? n : (n + 1) >> 1, n1 = shared ? n : n >> 1, ns = s ? n1 : n0;
                const uint32_t qc = shared ? qcount + (uint32_t)s : qcount, qs = qc & 1u;
                if (shared) {
                    // The other stream's q tile is only observed, and only for items so short that this issuer could
                    // finish them before that tile has landed (same parity-aliasing hazard as for the K/V ring).
                    const uint32_t qo = qcount + (uint32_t)(s ^ 1);
                    if (n <= NSTAGE) ptx::mbar_wait(st.bar(L::B_Q_FULL + (qo & 1u)), (qo >> 1) & 1u, abort_flag);
                }
                ptx::mbar_wait(st.bar(L::B_Q_FULL + qs), (qc >> 1) & 1u, abort_flag);
                TRACE_EV(3 + s);
                if (!shared && ns == 0 && lane == 0) ptx::mbar_arrive(st.bar(L::B_Q_EMPTY + qs));   // nothing to read: release the q tile
                uint32_t sk = 0, sv = 0;
                for (int i = -1; i < n0; ++i) {
                    bool work = false;
                    int tile = -1, next = -1;
    #pragma unroll
                    for (int x = 0; x < 2; ++x) {                // SHARED: one pass (x = s); SPLIT: stream 0's stages, then stream 1's
                        if (shared && x != s) continue;
                        const int nx = x ? n1 : n0;
                        const bool has_v = i >= 0 && i < nx, has_k = i + 1 < nx;
                        if (x != s) {                            // the other issuer's stages (SPLIT)
                            if (has_v) st.skip();
                            if (has_k) st.skip();
                            continue;
                        }
                        if (has_v) {
                            sv = st.acquire(!shared);
                            tile = shared ? kv0 + i : kv0 + 2 * i + x;
                            const int nv = c - tile * BN;
                            if (nv < BN && (nv & 15)) {          // tail tile: stale rows of the last page
                                if (!shared || s == 0) zero_v_tail<D>(sbase + (uint32_t)(L::OFF_KV + sv * L::KV_BYTES), nv, (nv + 15) & ~15, lane);
                                if (shared) {                    // issuer 0 zero-fills, issuer 1 waits for it
                                    if (s == 0) { if (lane == 0) ptx::mbar_arrive(st.bar(L::B_ZFILL)); }
                                    else ptx::mbar_wait(st.bar(L::B_ZFILL), st.zf_par, abort_flag);
                                    st.zf_par ^= 1u;
                                }
                            }
                        }
                        if (has_k) {
                            sk = st.acquire(!shared);
                            next = shared ? kv0 + i + 1 : kv0 + 2 * (i + 1) + x;
                        }
                        work = has_v || has_k;
                    }
                    if (work)
                        tile_steps<D>(st, s, c, tile, i == 0, sv, next, sk, qs, shared ? 1 : 2,
                                      (next >= 0 && i + 2 == ns) ? (shared ? 2 : 1) : 0);
                }
                qcount += shared ? 2u : 1u;
            };
            if (it.rows1 > 0) rounds(SharedMode{}); else rounds(SplitMode{});
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(st.bar(L::B_ITEM_EMPTY + islot));
        ++icount;
    }
}

// ------------------------------------------------------------------------------------------------
// warps 0-7: softmax warpgroups (a6) + epilogue (a8) + fused split-KV merge (a9).
// Thread `row` of stream s owns TMEM lane `row` of S_s / O_s.
// ------------------------------------------------------------------------------------------------
// One 64-column half tile of one row: returns alpha (the factor by which O and l shrink; 1 if the
// reference maximum m_ref stays).  m_ref is in log2 units and is only raised when the half's maximum
// exceeds it by more than LAZY_T, so p = 2^(x - m_ref) <= 2^LAZY_T: exact in range for bf16 / fp32.
// P (bf16 pairs) overwrites the first 32 columns of the half's S buffer.
// `turn`: 0 = none; else the named barrier this warp waits on before its exponentials (the partner warp of the other
// stream on the same sub-partition arrives on it after its own), `turn ^ 1` the one it arrives on after: the two warps
// that share a sub-partition's MUFU alternate instead of contending for it, and each one's loads, maximum, stores and
// hand-over run in the shadow of the other's exponentials (config 4: 1 970 -> 1 810 us; unsynchronised they fall into lock
// step, both in the exponentials, then both outside them).
template <bool MASK>
__device__ __forceinline__ float softmax_half(uint32_t s_taddr, int nv, float scale_log2, float& m_ref, float& l, uint32_t turn = 0) {
    uint32_t r[2][32];
#pragma unroll
    for (int c = 0; c < 2; ++c) ptx::tmem_ld32(s_taddr + (uint32_t)(c * 32), r[c]);
    ptx::tmem_wait_ld();
    if (scale_log2 < 0.f) {                       // rare: max_j(scale * s_j) with scale < 0 -- work on -s with |scale|
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int i = 0; i < 32; ++i) r[c][i] ^= 0x80000000u;
        scale_log2 = -scale_log2;
    }
    float mx4[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        float a = -INFINITY;
#pragma unroll
        for (int i = 0; i < 16; i += 2) {
            const int col = c * 16 + i;
            float v0 = __uint_as_float(r[col >> 5][col & 31]), v1 = __uint_as_float(r[col >> 5][(col & 31) + 1]);
            if (MASK) {
                if (col >= nv) v0 = -INFINITY;
                if (col + 1 >= nv) v1 = -INFINITY;
            }
            a = fmaxf(a, fmaxf(v0, v1));
        }
        mx4[c] = a;
    }
    const float mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * fabsf(scale_log2);
    const bool grow = mx > m_ref + LAZY_T;
    const float m_new = grow ? mx : m_ref;
    const float alpha = grow ? ptx::ex2(m_ref - m_new) : 1.f;
    // packed fp32x2 arithmetic (FFMA2 / FADD2): one instruction per two columns
    const float2 sc2 = make_float2(scale_log2, scale_log2), ng2 = make_float2(-m_new, -m_new);
    float2 sum_a = make_float2(0.f, 0.f), sum_b = make_float2(0.f, 0.f);
    if (turn) asm volatile("bar.sync %0, 64;" ::"r"(turn) : "memory");
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        uint32_t pk[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const float2 x = __ffma2_rn(make_float2(__uint_as_float(r[c][2 * i]), __uint_as_float(r[c][2 * i + 1])), sc2, ng2);
            float2 pp;
            pp.x = ptx::ex2(x.x);
            pp.y = ptx::ex2(x.y);
            if (MASK) {
                if (c * 32 + 2 * i >= nv) pp.x = 0.f;
                if (c * 32 + 2 * i + 1 >= nv) pp.y = 0.f;
            }
            if (i & 1) sum_b = __fadd2_rn(sum_b, pp); else sum_a = __fadd2_rn(sum_a, pp);
            pk[i] = ptx::pack_bf16(pp.x, pp.y);
        }
        ptx::tmem_st16(s_taddr + (uint32_t)(c * 16), pk);
    }
    if (turn) asm volatile("bar.arrive %0, 64;" ::"r"(turn ^ 1u) : "memory");
    const float2 sum2 = __fadd2_rn(sum_a, sum_b);
    const float sum0 = sum2.x, sum1 = sum2.y;
    l = l * alpha + (sum0 + sum1);
    m_ref = m_new;
    return alpha;
}

// One row of the epilogue from TMEM, 32 columns at a time (TMEM loads are warp-collective, stores predicated):
//   final:   out row (bf16)          <- w0 * O0 [+ w1 * O1]      (w's already contain 1 / l)
//   partial: slot row (fp32, unnormalised) <- w0 * O0 [+ w1 * O1];  slot layout [D/4 column groups][256 rows][4 floats]:
//            a warp's 32 rows of one column group are 512 contiguous bytes, so these stores and the merge's loads coalesce.
// One copy of this code serves every mode (`two`, `partial` are warp-uniform run-time flags): the kernel's instruction
// footprint matters more than the few predicated instructions.
template <int D>
__device__ __forceinline__ void store_row(uint32_t o0_taddr, uint32_t o1_taddr, bool two, float w0, float w1, bool row_ok,
                                          bool partial, uint4* dst, float4* po) {
#pragma unroll 1
    for (int c = 0; c < D / 32; ++c) {
        uint32_t o[32], o1[32];
        ptx::tmem_ld32(o0_taddr + (uint32_t)(c * 32), o);
        if (two) ptx::tmem_ld32(o1_taddr + (uint32_t)(c * 32), o1);
        ptx::tmem_wait_ld();
        float f[32];
#pragma unroll
        for (int e = 0; e < 32; ++e) f[e] = __uint_as_float(o[e]) * w0;
        if (two) {
#pragma unroll
            for (int e = 0; e < 32; ++e) f[e] = fmaf(__uint_as_float(o1[e]), w1, f[e]);
        }
        if (row_ok) {
            if (partial) {
#pragma unroll
                for (int v = 0; v < 8; ++v) po[(c * 8 + v) * PAIR] = make_float4(f[v * 4], f[v * 4 + 1], f[v * 4 + 2], f[v * 4 + 3]);
            } else {
#pragma unroll
                for (int v = 0; v < 4; ++v) {
                    uint4 w;
                    w.x = ptx::pack_bf16(f[v * 8 + 0], f[v * 8 + 1]); w.y = ptx::pack_bf16(f[v * 8 + 2], f[v * 8 + 3]);
                    w.z = ptx::pack_bf16(f[v * 8 + 4], f[v * 8 + 5]); w.w = ptx::pack_bf16(f[v * 8 + 6], f[v * 8 + 7]);
                    dst[c * 4 + v] = w;
                }
            }
        }
    }
}

template <int D>
__device__ __forceinline__ void softmax_wg(const AttnParams& p, uint8_t* smem, uint32_t sbase, uint32_t tmem,
                                           const Item* items, volatile uint32_t* abort_flag, int s, int wg_warp, int lane) {
    using L = Smem<D>;
    const unsigned FULL = 0xffffffffu;
    auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
    const int row = wg_warp * 32 + lane;
    const uint32_t lane_base = (uint32_t)(wg_warp * 32) << 16;
    const uint32_t s_taddr = tmem + lane_base + (uint32_t)s * 128u;
    const uint32_t o_taddr = tmem + lane_base + 256u + (uint32_t)s * 128u;     // own accumulator
    const uint32_t o_other = tmem + lane_base + 256u + (uint32_t)(s ^ 1) * 128u;
    float2* ml_x = reinterpret_cast<float2*>(smem + L::OFF_ML);
    uint32_t icount = 0, hpar = 0, pv0 = 0, pv1 = 0, ecount = 0;      // hpar: bit h = parity of the next S_FULL wait of half h
    bool owed = false;               // stream 1: the boundary barrier of its last turn-taking item is still to be waited on
    TRACE_NS(40);
    TRACE_EV(36);
    while (true) {
        if (*abort_flag) break;
        const uint32_t islot = icount & 1u;
        ptx::mbar_wait(bar(L::B_ITEM_FULL + islot), (icount >> 1) & 1u, abort_flag);
        const Item it = items[islot];
        if (!it.valid) break;
        TRACE_EV(30);
        const bool shared = it.rows1 > 0;
        const int n = it.kv1 - it.kv0;
        const int ns = shared ? n : (s == 0 ? (n + 1) / 2 : n / 2);
        const int rows_valid = (shared && s == 1) ? it.rows1 : it.rows0;
        const bool warp_active = wg_warp * 32 < rows_valid;
        float m = -INFINITY, l = 0.f;
        uint32_t steps = 0;                                    // half tiles of this item handed to the issuer
        // SHARED items: warp w of stream 0 and warp w of stream 1 (same sub-partition) take
        // turns at the exponentials; barrier 2 + 2 w = "stream 0 may", 3 + 2 w = "stream 1 may".  Stream 1 primes stream 0's.
        const bool ping = shared && wg_warp * 32 < it.rows0 && wg_warp * 32 < it.rows1;      // both warps of the pair compute
        const uint32_t turn = ping ? (uint32_t)(2 + 2 * wg_warp + s) : 0u;
        if (ping && s == 1) {
            if (owed) { asm volatile("bar.sync %0, 64;" ::"r"(10u + (uint32_t)wg_warp) : "memory"); owed = false; }
            asm volatile("bar.arrive %0, 64;" ::"r"(turn ^ 1u) : "memory");
        }
        for (int i = 0; i < ns; ++i) {
            // (after a watchdog abort every wait returns at once; a warp that takes turns with a partner must still run all
            // of its half steps, or the partner would block for ever on the named barrier)
            if (!ping) { if (*abort_flag) break; }
            const int tile = shared ? it.kv0 + i : it.kv0 + 2 * i + s;
            int nvt = it.c - tile * BN;
            nvt = nvt > BN ? BN : nvt;
#pragma unroll 1
            for (int h = 0; h < 2; ++h) {                     // not unrolled: one copy of the softmax code (instruction cache)
                const int nv = nvt - h * 64 > 64 ? 64 : nvt - h * 64;
                if (nv <= 0) continue;                       // the context's last tile may lack half B
                TRACE_EV(20 + s);
                ptx::mbar_wait(bar(L::B_S_FULL + 2 * s + h), (hpar >> h) & 1u, abort_flag);
                TRACE_EV(22 + s);
                ptx::tc_fence_after();
                hpar ^= 1u << h;
                if (warp_active) {
                    const uint32_t sh = s_taddr + (uint32_t)(h * 64);
                    float alpha;
                    if (nv == 64) alpha = softmax_half<false>(sh, nv, p.scale_log2, m, l, turn);
                    else alpha = softmax_half<true>(sh, nv, p.scale_log2, m, l, turn);
                    if (steps > 0 && __any_sync(FULL, alpha != 1.f)) {
                        // rare (lazy reference maximum): every PV handed over so far must have landed in O first.
                        // Per half at most the latest one is still in flight (the S_FULL just seen was committed
                        // behind the one before), so each parity wait is unambiguous.
                        ptx::mbar_wait(bar(L::B_PV_DONE + 2 * s), (pv0 - 1u) & 1u, abort_flag);
                        ptx::mbar_wait(bar(L::B_PV_DONE + 2 * s + 1), (pv1 - 1u) & 1u, abort_flag);
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
                    }
                    ptx::tmem_wait_st();
                }
                ptx::tc_fence_before();
                __syncwarp();
                TRACE_EV(24 + s);
                if (lane == 0) ptx::mbar_arrive(bar(L::B_P_FULL + 2 * s + h));
                ++steps;
                if (h) ++pv1; else ++pv0;
            }
        }
        if (ping) {
            if (s == 0) {
                asm volatile("bar.sync %0, 64;" ::"r"(turn) : "memory");                  // consume stream 1's last hand-over
                // ... and only then may stream 1 prime its next turn-taking item (it does so after its epilogue; should stream
                // 0 be held up meanwhile -- a late O rescale -- the prime would land in the generation that is still open).
                // Barrier 10 + w: stream 0 arrives here, stream 1 waits on it just before its next prime (`owed`).
                asm volatile("bar.arrive %0, 64;" ::"r"(10u + (uint32_t)wg_warp) : "memory");
            } else {
                owed = true;
            }
        }
        if (steps > 0) {
            ptx::mbar_wait(bar(L::B_PV_DONE + 2 * s), (pv0 - 1u) & 1u, abort_flag);
            ptx::mbar_wait(bar(L::B_PV_DONE + 2 * s + 1), (pv1 - 1u) & 1u, abort_flag);
            ptx::tc_fence_after();
        }
        // ---------------- epilogue
        TRACE_EV(31);
        bool row_ok = row < rows_valid;
        const int tl = row / p.G, hh = row - tl * p.G;                       // row = token * G + head of the group
        const int tok = it.q_start + it.tok0 + ((shared && s == 1) ? p.tpt : 0) + tl;
        if (row_ok && ((unsigned)tok >= (unsigned)p.total_q || (unsigned)it.g >= (unsigned)p.Hkv || it.part_slot >= p.num_slots)) {
            raise_flag(p.flags, DEV_INTERNAL | 0x400u);      // never store through a bad item
#ifdef SANGAM_DEBUG_ITEM
            if (atomicCAS(&ptx::g_timeout_info[0], 0u, 0xdead0000u | (unsigned)s) == 0u) {
                const int* w = reinterpret_cast<const int*>(&it);
                for (int k = 0; k < 13; ++k) g_bad_item[k] = w[k];
                g_bad_item[13] = tok; g_bad_item[14] = row; g_bad_item[15] = (int)icount;
            }
#endif
            row_ok = false;
        }
        uint4* dst = reinterpret_cast<uint4*>(p.out + ((int64_t)tok * p.Hq + it.g * p.G + hh) * D);
        const int prow = ((shared && s == 1) ? BM : 0) + row;                 // row inside the partial slot
        float4* po = reinterpret_cast<float4*>(p.part_o) + (int64_t)(it.part_slot < 0 ? 0 : it.part_slot) * (D / 4) * PAIR + prow;
        float2* pml = reinterpret_cast<float2*>(p.part_ml) + (int64_t)(it.part_slot < 0 ? 0 : it.part_slot) * PAIR + prow;
        const bool partial = it.part_slot >= 0;
        bool do_store = false, two = false;
        float w0 = 1.f, w1 = 0.f, m_out = m, l_out = l;
        if (n == 0) {
            // empty context: zeros (reading S13); never split
            if (row_ok && (shared || s == 0)) {
#pragma unroll
                for (int c = 0; c < D / 8; ++c) dst[c] = make_uint4(0, 0, 0, 0);
            }
        } else if (shared) {
            do_store = warp_active;
        } else {
            // SPLIT: stream 1 hands (m, l) to stream 0, which merges O_0 and O_1
            if (s == 1) {
                ml_x[row] = make_float2(m, l);
                ptx::mbar_arrive(bar(L::B_EPI_A));
            } else {
                ptx::mbar_wait(bar(L::B_EPI_A), ecount & 1u, abort_flag);
                TRACE_EV(37);
                const float2 x = ml_x[row];
                m_out = fmaxf(m, x.x);
                two = n > 1;                                               // stream 1 had tiles
                w0 = ptx::ex2(m - m_out);
                w1 = two ? ptx::ex2(x.x - m_out) : 0.f;
                l_out = l * w0 + x.y * w1;
                do_store = warp_active;
            }
        }
        if (do_store) {
            if (!partial) {
                const float inv = l_out > 0.f ? 1.f / l_out : 0.f;
                w0 *= inv; w1 *= inv;
            }
            store_row<D>(o_taddr, o_other, two, w0, w1, row_ok, partial, dst, po);
            if (partial && row_ok) *pml = make_float2(m_out, l_out);
        }
        if (n > 0 && !shared) {
            if (s == 1) {
                ptx::mbar_wait(bar(L::B_EPI_B), ecount & 1u, abort_flag);       // stream 0 is done reading O_1
            } else {
                ptx::tc_fence_before();
                ptx::mbar_arrive(bar(L::B_EPI_B));
            }
            ++ecount;
        }
        TRACE_EV(32);
        TRACE_EV(34);
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar(L::B_ITEM_EMPTY + islot));
        ++icount;
    }
    if (owed) asm volatile("bar.sync %0, 64;" ::"r"(10u + (uint32_t)wg_warp) : "memory");     // balance stream 0's last arrive
    TRACE_EV(35);
    TRACE_NS(41);
}

// ------------------------------------------------------------------------------------------------
// kernel entry
// ------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(NTHREADS, 1)
attn_kernel(const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV,
            const __grid_constant__ CUtensorMap mapQ, const AttnParams p) {
    using L = Smem<D>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    const uint32_t sbase = ptx::smem_u32(smem);
    Item* items = reinterpret_cast<Item*>(smem + L::OFF_ITEMS);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::OFF_MISC);
    volatile uint32_t* abort_flag = reinterpret_cast<volatile uint32_t*>(smem + L::OFF_MISC + 4);
    uint32_t* kv_seq = reinterpret_cast<uint32_t*>(smem + L::OFF_SEQ);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    TRACE_INIT();
    TRACE_CTA(0);
    if (tid == 0) {
        auto bar = [&](int i) { return sbase + (uint32_t)(L::OFF_BAR + i * 8); };
        for (int s = 0; s < NSTAGE; ++s) { ptx::mbar_init(bar(L::B_KV_FULL + s), 1); ptx::mbar_init(bar(L::B_KV_EMPTY + s), 2); }
        for (int s = 0; s < 2; ++s) {
            ptx::mbar_init(bar(L::B_ITEM_FULL + s), 1);
            ptx::mbar_init(bar(L::B_ITEM_EMPTY + s), 11);  // 2 MMA issuers + loader warp + 8 softmax warps
            ptx::mbar_init(bar(L::B_Q_FULL + s), 1);
            ptx::mbar_init(bar(L::B_Q_EMPTY + s), 2);
            for (int h = 0; h < 2; ++h) {
                ptx::mbar_init(bar(L::B_S_FULL + 2 * s + h), 1);
                ptx::mbar_init(bar(L::B_P_FULL + 2 * s + h), 4);
                ptx::mbar_init(bar(L::B_PV_DONE + 2 * s + h), 1);
            }
        }
        ptx::mbar_init(bar(L::B_EPI_A), 128);
        ptx::mbar_init(bar(L::B_EPI_B), 128);
        ptx::mbar_init(bar(L::B_ZFILL), 1);
        *abort_flag = 0u;
        for (int k = 0; k < 16; ++k) abort_flag[3 + k] = 0u;
        for (int k = 0; k < NSTAGE; ++k) kv_seq[k] = 0xffffffffu;
        ptx::fence_mbar_init();
        ptx::prefetch_tensormap(&mapK);
        ptx::prefetch_tensormap(&mapV);
        ptx::prefetch_tensormap(&mapQ);
    }
    if (warp == 8) {
        ptx::tmem_alloc(ptx::smem_u32(tmem_slot), 512);
        ptx::tmem_relinquish();
    }
    // Everything above touches only this CTA's shared memory, TMEM and the kernel parameters: under a programmatic
    // dependent launch it overlaps the tail of the previous kernel in the stream.  Global memory is read or written
    // only after pdl_wait; the combine kernel behind this one may be scheduled onto SMs as they drain.
    ptx::pdl_wait();
    ptx::pdl_trigger();
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    // Warpgroups 0 and 1 are the softmax streams (TMEM lane quarter = warp % 4); warpgroup 2 holds the
    // service warps.  The MMA issuers are the highest warp ids: the SM sub-partition arbiter favours them
    // over the softmax warps they share a scheduler with, so a tile's MMAs go out the moment P is ready.
    if (warp < 8) {
        ptx::setmaxnreg_inc<208>();   // 8*32*208 + 4*32*80 <= 384*168: the pool is what the CTA got at launch
        softmax_wg<D>(p, smem, sbase, tmem, items, abort_flag, warp >> 2, warp & 3, lane);
    } else {
        ptx::setmaxnreg_dec<80>();
        // the producer sits on sub-partition 1: sub-partition 0 hosts the only active softmax warps of 32-row decodes
        if (warp == 9) producer_warp<D>(p, &mapK, &mapV, sbase, items, abort_flag, kv_seq, lane);
        else if (warp == 8) qload_warp<D>(p, &mapQ, sbase, items, abort_flag, lane);
        else mma_warp<D>(p, sbase, tmem, items, abort_flag, kv_seq, warp - 10, lane);
    }
    ptx::tc_fence_before();
    __syncthreads();
    TRACE_CTA(1);
    if (tid == 0 && *abort_flag) raise_flag(p.flags, DEV_TIMEOUT);
    if (warp == 8) ptx::tmem_dealloc(tmem, 512);
}

// ------------------------------------------------------------------------------------------------
// combine (a9): merge the split-KV pieces of one unit.  Block b owns the unit whose head piece CTA b of
// attn_kernel computed (SlotMeta); pieces in fixed order, no atomics: bitwise reproducible.  m in log2 units:
//   m* = max m_i;  l* = sum l_i 2^(m_i-m*);  O* = sum O_i 2^(m_i-m*);  out = bf16(O*/l*)
// A column group's consecutive rows are contiguous in a slot, so every load coalesces.
// ------------------------------------------------------------------------------------------------
// CS = blocks per unit (grid.y): 4 for GQA models (units of up to 256 rows: the 64 units of a Dream-like decode batch
// keep 256 blocks busy instead of 64), 1 for MHA models (32-row decode units: extra blocks would only add launch cost)
template <int D, int CS>
__global__ void __launch_bounds__(2 * PAIR)
combine_kernel(const AttnParams p) {
    ptx::pdl_wait();       // before any global read, in every block: this grid's completion then implies attn_kernel's
    ptx::pdl_trigger();
    const int b = blockIdx.x;
    const SlotMeta h = reinterpret_cast<const SlotMeta*>(p.slot_meta)[b];
    if (!h.valid) return;
    const int np = h.npieces, R = h.rows0 + h.rows1;
    if (np < 1 || 2 * (b + np - 1) >= p.num_slots || (unsigned)h.g >= (unsigned)p.Hkv) { raise_flag(p.flags, DEV_INTERNAL | 0x100u); return; }
    const float2* ml = reinterpret_cast<const float2*>(p.part_ml);
    if (R > 64) {
        // many rows (GQA decode): one thread per (row, 1/(2 CS) of the columns), D/(8 CS) independent 16-byte loads per
        // piece in flight; the CS blocks (blockIdx.y) of a unit take interleaved column slices
        const int half = (threadIdx.x >> 8) * CS + blockIdx.y, rr = threadIdx.x & (PAIR - 1), s = rr >> 7, row = rr & 127;
        if (row >= (s ? h.rows1 : h.rows0)) return;
        constexpr int HC = D / (2 * CS);                     // columns per thread
        float ms = -INFINITY;
        for (int pi = 0; pi < np; ++pi) ms = fmaxf(ms, ml[(int64_t)(pi == 0 ? 2 * b + 1 : 2 * (b + pi)) * PAIR + rr].x);
        float acc[HC];
#pragma unroll
        for (int e = 0; e < HC; ++e) acc[e] = 0.f;
        float ls = 0.f;
        for (int pi = 0; pi < np; ++pi) {
            const int64_t slot = pi == 0 ? 2 * b + 1 : 2 * (b + pi);
            const float2 x = ml[slot * PAIR + rr];
            const float w = ptx::ex2(x.x - ms);
            ls = fmaf(x.y, w, ls);
            const float4* src = reinterpret_cast<const float4*>(p.part_o) + (slot * (D / 4) + half * (HC / 4)) * PAIR + rr;
#pragma unroll
            for (int c4 = 0; c4 < HC / 4; ++c4) {
                const float4 o = __ldcs(src + c4 * PAIR);
                acc[c4 * 4 + 0] = fmaf(o.x, w, acc[c4 * 4 + 0]); acc[c4 * 4 + 1] = fmaf(o.y, w, acc[c4 * 4 + 1]);
                acc[c4 * 4 + 2] = fmaf(o.z, w, acc[c4 * 4 + 2]); acc[c4 * 4 + 3] = fmaf(o.w, w, acc[c4 * 4 + 3]);
            }
        }
        const float inv = ls > 0.f ? 1.f / ls : 0.f;
        const int tl = row / p.G, hh = row - tl * p.G;
        const int tok = h.q_start + h.tok0 + s * p.tpt + tl;
        if ((unsigned)tok >= (unsigned)p.total_q) { raise_flag(p.flags, DEV_INTERNAL | 0x200u); return; }
        uint4* dst = reinterpret_cast<uint4*>(p.out + ((int64_t)tok * p.Hq + h.g * p.G + hh) * D + half * HC);
#pragma unroll
        for (int c8 = 0; c8 < HC / 8; ++c8) {
            uint4 w4;
            w4.x = ptx::pack_bf16(acc[c8 * 8 + 0] * inv, acc[c8 * 8 + 1] * inv);
            w4.y = ptx::pack_bf16(acc[c8 * 8 + 2] * inv, acc[c8 * 8 + 3] * inv);
            w4.z = ptx::pack_bf16(acc[c8 * 8 + 4] * inv, acc[c8 * 8 + 5] * inv);
            w4.w = ptx::pack_bf16(acc[c8 * 8 + 6] * inv, acc[c8 * 8 + 7] * inv);
            dst[c8] = w4;
        }
        return;
    }
    // few rows (MHA decode): work item = (8-column group cg, row), consecutive threads take consecutive rows of one
    // column group, so a 32-row unit still spreads over all 256 threads
    for (int item = threadIdx.x + blockIdx.y * 2 * PAIR; item < R * (D / 8); item += 2 * PAIR * CS) {
        const int cg = item / R, ri = item - cg * R;
        const int s = ri >= h.rows0, row = ri - (s ? h.rows0 : 0), rr = s * BM + row;      // rr = row inside the slot
        float ms = -INFINITY;
        for (int pi = 0; pi < np; ++pi) ms = fmaxf(ms, ml[(int64_t)(pi == 0 ? 2 * b + 1 : 2 * (b + pi)) * PAIR + rr].x);
        float acc[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) acc[e] = 0.f;
        float ls = 0.f;
#pragma unroll 4
        for (int pi = 0; pi < np; ++pi) {
            const int64_t slot = pi == 0 ? 2 * b + 1 : 2 * (b + pi);
            const float2 x = ml[slot * PAIR + rr];
            const float w = ptx::ex2(x.x - ms);
            ls = fmaf(x.y, w, ls);
            const float4* src = reinterpret_cast<const float4*>(p.part_o) + (slot * (D / 4) + 2 * cg) * PAIR + rr;
            const float4 o0 = __ldcs(src), o1 = __ldcs(src + PAIR);
            acc[0] = fmaf(o0.x, w, acc[0]); acc[1] = fmaf(o0.y, w, acc[1]); acc[2] = fmaf(o0.z, w, acc[2]); acc[3] = fmaf(o0.w, w, acc[3]);
            acc[4] = fmaf(o1.x, w, acc[4]); acc[5] = fmaf(o1.y, w, acc[5]); acc[6] = fmaf(o1.z, w, acc[6]); acc[7] = fmaf(o1.w, w, acc[7]);
        }
        const float inv = ls > 0.f ? 1.f / ls : 0.f;
        const int tl = row / p.G, hh = row - tl * p.G;
        const int tok = h.q_start + h.tok0 + s * p.tpt + tl;
        if ((unsigned)tok >= (unsigned)p.total_q) { raise_flag(p.flags, DEV_INTERNAL | 0x200u); continue; }
        uint4 w4;
        w4.x = ptx::pack_bf16(acc[0] * inv, acc[1] * inv);
        w4.y = ptx::pack_bf16(acc[2] * inv, acc[3] * inv);
        w4.z = ptx::pack_bf16(acc[4] * inv, acc[5] * inv);
        w4.w = ptx::pack_bf16(acc[6] * inv, acc[7] * inv);
        reinterpret_cast<uint4*>(p.out + ((int64_t)tok * p.Hq + h.g * p.G + hh) * D)[cg] = w4;
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

// cuTensorMapEncodeTiled through the runtime's driver entry point (no -lcuda); looked up once
static inline sangam_encode_fn tmap_encode_fn() {
    static sangam_encode_fn enc = nullptr;
    if (!enc) {
        cudaDriverEntryPointQueryResult q;
        void* fn = nullptr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn) return nullptr;
        enc = reinterpret_cast<sangam_encode_fn>(fn);
    }
    return enc;
}

// Pool viewed as a 4-D tensor (64 columns, 8 rows of a row group, D/64 slabs, P*Hkv*2 row groups) of bf16; one box =
// (64, 8, D/64, 2) = a whole page of one head (16 rows x D), 128-byte swizzled: it lands as 2 x D/64 UMMA swizzle atoms.
// One TMA instruction per page instead of one per (page, slab): the gather is bound by TMA instructions, not bytes.
// A box whose last coordinate is >= P*Hkv*2 lies outside the tensor and is filled with zeros (bad page ids).
static inline int tmap_encode_pool(CUtensorMap* out, const void* pages, int num_pages, int Hkv, int D) {
    sangam_encode_fn enc = tmap_encode_fn();
    if (!enc) return -1;
    const cuuint64_t gdim[4] = {64, 8, (cuuint64_t)(D / 64), (cuuint64_t)num_pages * Hkv * (SANGAM_PAGE / 8)};
    const cuuint64_t gstr[3] = {(cuuint64_t)D * 2, 128, (cuuint64_t)D * 2 * 8};
    const cuuint32_t box[4] = {64, 8, (cuuint32_t)(D / 64), SANGAM_PAGE / 8}, estr[4] = {1, 1, 1, 1};
    CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(pages), gdim, gstr, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : -1;
}

// q viewed as [total_q][Hq][D] bf16; one box = `tokens` tokens x G heads x 64 columns, 128-byte swizzled
static inline int tmap_encode_q(CUtensorMap* out, const void* q, int total_q, int Hq, int D, int G, int tokens) {
    sangam_encode_fn enc = tmap_encode_fn();
    if (!enc) return -1;
    const cuuint64_t gdim[3] = {(cuuint64_t)D, (cuuint64_t)Hq, (cuuint64_t)total_q};
    const cuuint64_t gstr[2] = {(cuuint64_t)D * 2, (cuuint64_t)Hq * D * 2};
    const cuuint32_t box[3] = {64, (cuuint32_t)G, (cuuint32_t)tokens}, estr[3] = {1, 1, 1};
    CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(q), gdim, gstr, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : -1;
}

static inline cudaError_t tc_launch(const AttnParams& p, const CUtensorMap& mk, const CUtensorMap& mv, const CUtensorMap& mq,
                                    int head_dim, int sm_count, cudaStream_t stream, int* launched) {
    cudaError_t e;
    *launched = 0;
    if (head_dim == 128) {
        e = launch_pdl(tc::attn_kernel<128>, dim3(sm_count), tc::NTHREADS, tc::Smem<128>::ALLOC, stream, mk, mv, mq, p);
        if (e != cudaSuccess) return e;
        *launched = 1;
        e = p.G > 1 ? launch_pdl(tc::combine_kernel<128, 4>, dim3(sm_count, 4), 2 * tc::PAIR, 0, stream, p)
                    : launch_pdl(tc::combine_kernel<128, 1>, dim3(sm_count, 1), 2 * tc::PAIR, 0, stream, p);
    } else {
        e = launch_pdl(tc::attn_kernel<64>, dim3(sm_count), tc::NTHREADS, tc::Smem<64>::ALLOC, stream, mk, mv, mq, p);
        if (e != cudaSuccess) return e;
        *launched = 1;
        e = p.G > 1 ? launch_pdl(tc::combine_kernel<64, 4>, dim3(sm_count, 4), 2 * tc::PAIR, 0, stream, p)
                    : launch_pdl(tc::combine_kernel<64, 1>, dim3(sm_count, 1), 2 * tc::PAIR, 0, stream, p);
    }
    if (e != cudaSuccess) return e;
    *launched = 2;
    return cudaGetLastError();
}
