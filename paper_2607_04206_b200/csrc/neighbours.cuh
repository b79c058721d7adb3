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
// grid = (slices, rows): block (s, t) scans logits[t][s * slice_len .. +slice_len)
__global__ void __launch_bounds__(CONF_THREADS)
confidence_pass1_kernel(const __nv_bfloat16* __restrict__ logits, int32_t V, int32_t slice_len, ConfPartial* __restrict__ part) {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int32_t t = blockIdx.y, sl = blockIdx.x;
    const int32_t lo = sl * slice_len, hi = min(V, lo + slice_len);
    const __nv_bfloat16* row = logits + (int64_t)t * V;
    float m = -INFINITY, sum = 0.f;
    int32_t arg = 0x7fffffff;
    // 16-byte vector loads over the aligned middle of the slice, scalar loads at its ragged ends
    const uintptr_t a0 = reinterpret_cast<uintptr_t>(row + lo);
    int32_t head = (int32_t)(((16 - (a0 & 15)) & 15) / 2);
    head = min(head, hi - lo);
    auto visit = [&](float x, int32_t j) {
        if (x > m) { sum = sum * __expf(m - x) + 1.f; m = x; arg = j; }
        else if (x == m) { sum += 1.f; arg = j < arg ? j : arg; }
        else sum += __expf(x - m);
    };
    for (int32_t j = lo + threadIdx.x; j < lo + head; j += CONF_THREADS) visit(__bfloat162float(row[j]), j);
    const int32_t nvec = (hi - lo - head) / 8;
    const uint4* vec = reinterpret_cast<const uint4*>(row + lo + head);
    for (int32_t q = threadIdx.x; q < nvec; q += CONF_THREADS) {
        const uint4 w = __ldcs(vec + q);
        const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
        const int32_t j0 = lo + head + q * 8;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            visit(__uint_as_float(ww[e] << 16), j0 + 2 * e);
            visit(__uint_as_float(ww[e] & 0xffff0000u), j0 + 2 * e + 1);
        }
    }
    for (int32_t j = lo + head + nvec * 8 + threadIdx.x; j < hi; j += CONF_THREADS) visit(__bfloat162float(row[j]), j);
    // block reduction
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float m2 = __shfl_xor_sync(0xffffffffu, m, o), s2 = __shfl_xor_sync(0xffffffffu, sum, o);
        const int32_t a2 = __shfl_xor_sync(0xffffffffu, arg, o);
        conf_merge(m, sum, arg, m2, s2, a2);
    }
    __shared__ float sm[CONF_THREADS / 32], ss[CONF_THREADS / 32];
    __shared__ int32_t sa[CONF_THREADS / 32];
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { sm[w] = m; ss[w] = sum; sa[w] = arg; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < CONF_THREADS / 32; ++k) conf_merge(m, sum, arg, sm[k], ss[k], sa[k]);
        ConfPartial p;
        p.m = m; p.sum = sum; p.arg = arg; p.pad = 0;
        part[(int64_t)t * gridDim.x + sl] = p;
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
