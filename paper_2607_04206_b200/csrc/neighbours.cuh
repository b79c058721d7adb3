// neighbours.cuh -- the two per-iteration kernels next to the hot path, both HBM-bound:
//
//  kv_write_rope_kernel   rotary position embedding applied to the fresh K rows on their way into the paged cache
//      (rotate, then scatter: one pass over K instead of a rotation kernel plus sangam_kv_write); V is copied.
//      Convention (reading S24, the Llama / Qwen lineage of the models the paper serves): rotate-half,
//          out[i] = x[i] cos - x[i + D/2] sin,   out[i + D/2] = x[i + D/2] cos + x[i] sin,   angle = pos * base^(-2i/D).
//      cos / sin come from a caller-provided fp32 table [max_pos][D] (first D/2 entries of a row: cos, last D/2: sin), as
//      serving stacks cache them; arithmetic in fp32, result rounded to bf16 (RNE).
//
//  confidence kernels     "Confidence-threshold based sampling unmasks every masked position whose top-1 probability
//      exceeds a threshold" (0.9).  Per row of bf16 logits: token = argmax (lowest index on ties),
//      conf = softmax(logits)[token] = 1 / sum exp(x - max).  Per request (its current block of rows): unmask every
//      still-masked row with conf > threshold; if none passes, the most confident masked row (reading S23).
//      Pass 1 streams the logits once (grid = rows x vocabulary slices, online max / sum / argmax per slice);
//      pass 2 merges the slices per row and takes the per-request decision.
#pragma once
#include "common.cuh"
#include "ptx.cuh"

// one thread-iteration = one 16-byte chunk (8 bf16) of a K row's LOWER half and the matching chunk of its upper half
__global__ void __launch_bounds__(256)
kv_write_rope_kernel(const uint4* __restrict__ k, const uint4* __restrict__ v, const int32_t* __restrict__ slot_mapping,
                     const int32_t* __restrict__ positions, const float* __restrict__ cos_sin, int32_t max_pos,
                     int32_t num_tokens, uint4* __restrict__ k_pages, uint4* __restrict__ v_pages, int32_t Hkv, int32_t D,
                     int32_t num_slots_total, uint32_t* flags) {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int32_t cpr = D / 8, hc = cpr / 2;                       // chunks per row, per half row
    const int64_t per_token = (int64_t)Hkv * hc;
    const int64_t total = (int64_t)num_tokens * per_token;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int32_t i = (int32_t)(idx / per_token);
        const int32_t rem = (int32_t)(idx - (int64_t)i * per_token);
        const int32_t h = rem / hc, c = rem - h * hc;
        const int32_t s = __ldg(slot_mapping + i);
        if (s < 0) continue;
        if (s >= num_slots_total) { raise_flag(flags, DEV_BAD_SLOT); continue; }
        int32_t pos = __ldg(positions + i);
        if (pos < 0 || pos >= max_pos) { raise_flag(flags, DEV_BAD_POSITION); continue; }
        const int64_t src = ((int64_t)i * Hkv + h) * cpr + c;
        const uint4 lo = __ldcs(k + src), hi = __ldcs(k + src + hc);
        const uint4 vlo = __ldcs(v + src), vhi = __ldcs(v + src + hc);
        const float4* cs = reinterpret_cast<const float4*>(cos_sin + (int64_t)pos * D + c * 8);
        const float4 c0 = __ldg(cs), c1 = __ldg(cs + 1);
        const float4 s0 = __ldg(cs + D / 8), s1 = __ldg(cs + D / 8 + 1);          // sin: D/2 floats further
        const float cosv[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
        const float sinv[8] = {s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w};
        const uint32_t lw[4] = {lo.x, lo.y, lo.z, lo.w}, hw[4] = {hi.x, hi.y, hi.z, hi.w};
        uint32_t ol[4], oh[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float a0 = __uint_as_float(lw[j] << 16), a1 = __uint_as_float(lw[j] & 0xffff0000u);     // elements 2j, 2j+1 (lower half)
            const float b0 = __uint_as_float(hw[j] << 16), b1 = __uint_as_float(hw[j] & 0xffff0000u);     // same, upper half
            const float r0 = a0 * cosv[2 * j] - b0 * sinv[2 * j], r1 = a1 * cosv[2 * j + 1] - b1 * sinv[2 * j + 1];
            const float t0 = b0 * cosv[2 * j] + a0 * sinv[2 * j], t1 = b1 * cosv[2 * j + 1] + a1 * sinv[2 * j + 1];
            __nv_bfloat162 pl = __floats2bfloat162_rn(r0, r1), ph = __floats2bfloat162_rn(t0, t1);
            ol[j] = *reinterpret_cast<uint32_t*>(&pl);
            oh[j] = *reinterpret_cast<uint32_t*>(&ph);
        }
        const int64_t dst = (((int64_t)(s >> 4) * Hkv + h) * SANGAM_PAGE + (s & 15)) * cpr + c;
        k_pages[dst] = make_uint4(ol[0], ol[1], ol[2], ol[3]);
        k_pages[dst + hc] = make_uint4(oh[0], oh[1], oh[2], oh[3]);
        v_pages[dst] = vlo;
        v_pages[dst + hc] = vhi;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// confidence-threshold sampler
// ---------------------------------------------------------------------------------------------------------------
struct ConfPartial {          // one vocabulary slice of one row
    float m, sum;             // max and sum exp(x - m) over the slice
    int32_t arg;              // index of the (first) maximum
    int32_t pad;
};

__device__ __forceinline__ void conf_merge(float& m, float& sum, int32_t& arg, float m2, float sum2, int32_t arg2) {
    // an empty holder has sum = 0; ties keep the lower index
    if (sum2 == 0.f) return;
    if (sum == 0.f) { m = m2; sum = sum2; arg = arg2; return; }
    if (m2 == m) { sum += sum2; arg = arg2 < arg ? arg2 : arg; return; }
    if (m2 > m) {
        sum = sum * __expf(m - m2) + sum2;
        m = m2; arg = arg2;
    } else {
        sum = sum + sum2 * __expf(m2 - m);
    }
}

constexpr int CONF_THREADS = 256;
// Persistent blocks (the grid fills the machine once): block b takes the work items b, b + gridDim.x, ...; item = (row t, slice
// sl) scans logits[t][sl * slice_len .. + slice_len).  Consecutive items are consecutive slices of a row, so neighbouring
// blocks stream neighbouring memory.
// The logits are streamed through a shared-memory ring by 1-D bulk copies (cp.async.bulk + mbarrier): thread 0 keeps
// CONF_NST chunks of CONF_CHUNK bytes in flight per block, across item boundaries, so the bytes in flight per SM (3 - 4 blocks x
// 40 KB) cover the HBM latency whatever the exponentials cost; with plain loads 4 x 16 B per thread the kernel ran at half
// the bandwidth (memory latency and MUFU time in series).
constexpr int CONF_CHUNK = 8192;                      // bytes per stage = 2 vectors of 8 logits per consumer thread
constexpr int CONF_NST = 5;
constexpr int CONF_BLOCK = CONF_THREADS + 32;         // 8 consumer warps + 1 producer warp
__global__ void __launch_bounds__(CONF_BLOCK)
confidence_pass1_kernel(const __nv_bfloat16* __restrict__ logits, int32_t V, int32_t slice_len, int32_t slices, int32_t num_items,
                        ConfPartial* __restrict__ part) {
    __shared__ __align__(128) uint8_t ring[CONF_NST * CONF_CHUNK];
    __shared__ __align__(8) unsigned long long full[CONF_NST], empty[CONF_NST];
    __shared__ float sm[CONF_THREADS / 32], ss[CONF_THREADS / 32];
    __shared__ int32_t sa[CONF_THREADS / 32];
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int s_ = 0; s_ < CONF_NST; ++s_) { ptx::mbar_init(ptx::smem_u32(&full[s_]), 1); ptx::mbar_init(ptx::smem_u32(&empty[s_]), CONF_THREADS); }
        ptx::fence_mbar_init();
    }
    __syncthreads();
    // geometry of an item: [lo, hi) of its row, `head` scalar elements up to the first 16-byte boundary, nvec whole vectors
    auto geom = [&](int32_t item, int32_t& t, int32_t& lo, int32_t& hi, int32_t& head, int32_t& nvec) {
        t = item / slices;
        const int32_t sl = item - t * slices;
        lo = sl * slice_len; hi = min(V, lo + slice_len);
        const uintptr_t a0 = reinterpret_cast<uintptr_t>(logits + (int64_t)t * V + lo);
        head = min((int32_t)(((16 - (a0 & 15)) & 15) / 2), hi - lo);
        nvec = (hi - lo - head) / 8;
    };
    auto wait = [&](unsigned long long* b_, uint32_t ph) {
        const uint32_t bar = ptx::smem_u32(b_);
        uint32_t spins = 0;
        while (!ptx::mbar_try_wait_hint(bar, ph, 10000u))
            if (++spins > (1u << 20)) break;                        // (never in a correct run: no hang, wrong numbers instead)
    };
    if (tid >= CONF_THREADS) {
        // ---- producer warp (one lane): the block's flattened chunk stream, CONF_NST chunks ahead of the consumers
        if (tid == CONF_THREADS) {
            uint32_t issued = 0;
            for (int32_t item = blockIdx.x; item < num_items; item += gridDim.x) {
                int32_t t, lo, hi, head, nvec;
                geom(item, t, lo, hi, head, nvec);
                const uint8_t* src = reinterpret_cast<const uint8_t*>(logits + (int64_t)t * V + lo + head);
                for (int32_t left = nvec * 16; left > 0; left -= CONF_CHUNK, src += CONF_CHUNK, ++issued) {
                    const uint32_t st = issued % CONF_NST, use = issued / CONF_NST;
                    if (use > 0) wait(&empty[st], (use - 1u) & 1u);            // every consumer thread has the previous use in registers
                    const uint32_t bytes = (uint32_t)(left < CONF_CHUNK ? left : CONF_CHUNK);
                    ptx::mbar_arrive_expect_tx(ptx::smem_u32(&full[st]), bytes);
                    ptx::bulk_load(ptx::smem_u32(ring + st * CONF_CHUNK), src, bytes, ptx::smem_u32(&full[st]));
                }
            }
        }
        return;
    }
    // ---- consumer warps
    const float LOG2E = 1.4426950408889634f;
    uint32_t cons = 0;                          // chunks consumed so far
    for (int32_t item = blockIdx.x; item < num_items; item += gridDim.x) {
        int32_t t, lo, hi, head, nvec;
        geom(item, t, lo, hi, head, nvec);
        const __nv_bfloat16* row = logits + (int64_t)t * V;
        float m = -INFINITY, sum = 0.f;
        int32_t arg = 0x7fffffff;
        auto visit = [&](float x, int32_t j) {
            if (x > m) { sum = sum * __expf(m - x) + 1.f; m = x; arg = j; }
            else if (x == m) { sum += 1.f; arg = j < arg ? j : arg; }
            else sum += __expf(x - m);
        };
        for (int32_t j = lo + tid; j < lo + head; j += CONF_THREADS) visit(__bfloat162float(row[j]), j);
        // A thread meets its indices in increasing order, so only a strictly larger value moves (m, arg) (an equal one keeps
        // the earlier index).  The maximum of a chunk's 16 logits is taken first, so that test is made once per chunk, and
        // the rest is branch-free: exp(x - m) =
        // ex2(x log2e - m log2e), one packed FFMA per two logits and one MUFU each.  A vector past the slice's end reads as
        // eight -inf (exp = 0).
        auto unpack = [](const uint4& w, float (&x)[8]) {
            x[0] = __uint_as_float(w.x << 16); x[1] = __uint_as_float(w.x & 0xffff0000u);
            x[2] = __uint_as_float(w.y << 16); x[3] = __uint_as_float(w.y & 0xffff0000u);
            x[4] = __uint_as_float(w.z << 16); x[5] = __uint_as_float(w.z & 0xffff0000u);
            x[6] = __uint_as_float(w.w << 16); x[7] = __uint_as_float(w.w & 0xffff0000u);
        };
        auto max8 = [](const float (&x)[8]) {
            return fmaxf(fmaxf(fmaxf(x[0], x[1]), fmaxf(x[2], x[3])), fmaxf(fmaxf(x[4], x[5]), fmaxf(x[6], x[7])));
        };
        auto first_of = [](const float (&x)[8], float mx) {         // lowest e with x[e] == mx, 8 if none
            int32_t k = 8;
#pragma unroll
            for (int e = 7; e >= 0; --e) k = x[e] == mx ? e : k;
            return k;
        };
        auto sum8 = [&](const float (&x)[8], float2 nm2) {          // sum of ex2(x log2e + nm2)
            const float2 sc2 = make_float2(LOG2E, LOG2E);
            float2 acc = make_float2(0.f, 0.f);
#pragma unroll
            for (int e = 0; e < 8; e += 2) {
                const float2 y = __ffma2_rn(make_float2(x[e], x[e + 1]), sc2, nm2);
                acc = __fadd2_rn(acc, make_float2(ptx::ex2(y.x), ptx::ex2(y.y)));
            }
            return acc.x + acc.y;
        };
        const uint4 NEG = make_uint4(0xff80ff80u, 0xff80ff80u, 0xff80ff80u, 0xff80ff80u);       // bf16 -inf x 8
        const int32_t nchunks = (nvec * 16 + CONF_CHUNK - 1) / CONF_CHUNK;
        int32_t cbest = -1;                                        // chunk in which this thread's maximum was last raised
        uint4 wb0 = NEG, wb1 = NEG;                                // ... and the thread's two vectors of that chunk
        for (int32_t c = 0; c < nchunks; ++c, ++cons) {
            const uint32_t st = cons % CONF_NST;
            wait(&full[st], (cons / CONF_NST) & 1u);
            const int32_t v0 = c * (CONF_CHUNK / 16) + tid, v1 = v0 + CONF_THREADS;      // vector indices inside the slice
            const uint4* stage = reinterpret_cast<const uint4*>(ring + st * CONF_CHUNK);
            const uint4 w0 = v0 < nvec ? stage[tid] : NEG, w1 = v1 < nvec ? stage[tid + CONF_THREADS] : NEG;
            float x0[8], x1[8];
            unpack(w0, x0); unpack(w1, x1);
            const float mx = fmaxf(max8(x0), max8(x1));
            // Release the stage only when the 32 bytes are in registers: the arrive takes `mx` (which depends on every loaded
            // word) as an operand, so it issues after the loads have returned.  An arrive right behind the LDS instructions
            // let the producer's next bulk copy overwrite the stage under loads still queued in the shared-memory pipe.
            {
                // (the barrier address is made to depend on mx: a value with nonzero low mantissa bits cannot come out of bf16
                // logits, so the offset is always 0, but neither compiler can know that and drop the dependency)
                const uint32_t off = __float_as_uint(mx) == 0x7fc00001u ? 8u : 0u;
                ptx::mbar_arrive(ptx::smem_u32(&empty[st]) + off);                        // every consumer thread arrives
            }
            if (mx > m) {                                          // new maximum: keep the chunk's vectors, find the index later
                sum *= __expf(m - mx);                             // (m = -inf, sum = 0: 0 * 0)
                m = mx; cbest = c; wb0 = w0; wb1 = w1;
            }
            const float nm = -fmaxf(m, -1.0e30f) * LOG2E;          // (nothing but -inf so far: ex2(-inf + 1.4e30) = 0, not NaN)
            const float2 nm2 = make_float2(nm, nm);
            sum += sum8(x0, nm2) + sum8(x1, nm2);
        }
        if (cbest >= 0) {
            // the index of the maximum, once per item, from the kept copy of the two vectors that raised it last (8 registers)
            // instead of 32 compare / select instructions in every chunk
            float x0[8], x1[8];
            unpack(wb0, x0); unpack(wb1, x1);
            const int32_t k0 = first_of(x0, m), k1 = first_of(x1, m);
            const int32_t jb = lo + head + (cbest * (CONF_CHUNK / 16) + tid) * 8;
            arg = k0 < 8 ? jb + k0 : jb + CONF_THREADS * 8 + k1;
        }
        for (int32_t j = lo + head + nvec * 8 + tid; j < hi; j += CONF_THREADS) visit(__bfloat162float(row[j]), j);
        // block reduction (the 256 consumer threads: named barrier 1)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float m2 = __shfl_xor_sync(0xffffffffu, m, o), s2 = __shfl_xor_sync(0xffffffffu, sum, o);
            const int32_t a2 = __shfl_xor_sync(0xffffffffu, arg, o);
            conf_merge(m, sum, arg, m2, s2, a2);
        }
        const int w = tid >> 5, l = tid & 31;
        if (l == 0) { sm[w] = m; ss[w] = sum; sa[w] = arg; }
        asm volatile("bar.sync 1, %0;" ::"n"(CONF_THREADS) : "memory");
        if (tid == 0) {
            for (int k = 1; k < CONF_THREADS / 32; ++k) conf_merge(m, sum, arg, sm[k], ss[k], sa[k]);
            ConfPartial p;
            p.m = m; p.sum = sum; p.arg = arg; p.pad = 0;
            part[item] = p;                                        // = [t][sl]
        }
        asm volatile("bar.sync 1, %0;" ::"n"(CONF_THREADS) : "memory");       // the staging arrays are reused by the next item
    }
}

// one warp per request: merge the slices of each of its rows, then decide which masked rows are unmasked
__global__ void __launch_bounds__(128)
confidence_pass2_kernel(const ConfPartial* __restrict__ part, int32_t slices, const int32_t* __restrict__ masked,
                        const int32_t* __restrict__ cu_rows, int32_t num_requests, float threshold,
                        int32_t* __restrict__ token, float* __restrict__ conf, int32_t* __restrict__ unmask) {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int r = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (r >= num_requests) return;
    const int32_t lo = __ldg(cu_rows + r), hi = __ldg(cu_rows + r + 1);
    float best = -1.f;
    int32_t best_row = 0x7fffffff;
    bool any_pass = false;
    for (int32_t t0 = lo; t0 < hi; t0 += 32) {
        const int32_t t = t0 + lane;
        float cf = 0.f;
        bool msk = false;
        if (t < hi) {
            ConfPartial a = part[(int64_t)t * slices];
            for (int32_t s = 1; s < slices; ++s) { const ConfPartial b = part[(int64_t)t * slices + s]; conf_merge(a.m, a.sum, a.arg, b.m, b.sum, b.arg); }
            cf = 1.f / a.sum;
            token[t] = a.arg;
            conf[t] = cf;
            msk = __ldg(masked + t) != 0;
            unmask[t] = (msk && cf > threshold) ? 1 : 0;
            if (msk && (cf > best || (cf == best && t < best_row))) { best = cf; best_row = t; }
        }
        any_pass |= __any_sync(0xffffffffu, msk && cf > threshold);
    }
    // fallback: nobody passed -> the most confident masked row (lowest index on ties)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float b2 = __shfl_xor_sync(0xffffffffu, best, o);
        const int32_t r2 = __shfl_xor_sync(0xffffffffu, best_row, o);
        if (b2 > best || (b2 == best && r2 < best_row)) { best = b2; best_row = r2; }
    }
    if (!any_pass && lane == 0 && best_row != 0x7fffffff) unmask[best_row] = 1;
}
