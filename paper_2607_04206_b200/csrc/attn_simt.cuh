// attn_simt.cuh -- CUDA-core cross-check of the attention contract (sangam_block_attn_simt).
// One warp per (query row, q head); lanes split head_dim; fp32 online softmax, one key at a time.
// Slow by design: it exists to check the tcgen05 kernel on workloads too big for the CPU oracle
// and is never dispatched by sangam_block_attn.  Definition: PAPER.md:67 (no causal mask),
// PAPER.md:33 (block over prompt+response context); readings S4, S12, S13 of DESIGN.md.
#pragma once
#include "common.cuh"

template <int D>
__global__ void __launch_bounds__(256)
attn_simt_kernel(AttnParams p) {
    constexpr int EPL = D / 32;  // elements per lane
    const int lane = threadIdx.x & 31;
    const int64_t warp_global = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int32_t total_rows = __ldg(p.cu_q_lens + p.batch);
    if (warp_global >= (int64_t)total_rows * p.Hq) return;
    const int32_t t = (int32_t)(warp_global / p.Hq), h = (int32_t)(warp_global % p.Hq);
    int32_t r = 0;
    while (r < p.batch && !(__ldg(p.cu_q_lens + r) <= t && t < __ldg(p.cu_q_lens + r + 1))) ++r;
    if (r >= p.batch) return;
    const int32_t c = __ldg(p.ctx_lens + r);
    const int32_t g = h / p.G;
    __nv_bfloat16* o = p.out + ((int64_t)t * p.Hq + h) * D + lane * EPL;
    if (c <= 0 || (c + SANGAM_PAGE - 1) / SANGAM_PAGE > p.W) {
        if (c > 0) raise_flag(p.flags, DEV_CTX_TOO_LONG);
#pragma unroll
        for (int e = 0; e < EPL; ++e) o[e] = __float2bfloat16(0.f);
        return;
    }
    float qv[EPL], acc[EPL];
    const __nv_bfloat16* qp = p.q + ((int64_t)t * p.Hq + h) * D + lane * EPL;
#pragma unroll
    for (int e = 0; e < EPL; ++e) { qv[e] = __bfloat162float(qp[e]); acc[e] = 0.f; }
    float m = -INFINITY, l = 0.f;
    const int32_t* bt = p.block_table + (int64_t)r * p.W;
    for (int32_t j = 0; j < c; ++j) {
        const int32_t page = __ldg(bt + (j >> 4));
        const bool bad = page < 0 || page >= p.P;         // flagged; the page's positions read as K = V = 0 (sangam.h)
        if (bad) raise_flag(p.flags, DEV_BAD_PAGE);
        const int64_t row = (((int64_t)(bad ? 0 : page) * p.Hkv + g) * SANGAM_PAGE + (j & 15)) * D + lane * EPL;
        float dot = 0.f;
#pragma unroll
        for (int e = 0; e < EPL; ++e) dot += bad ? 0.f : qv[e] * __bfloat162float(p.k_pages[row + e]);
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, s);
        const float sj = dot * p.scale;
        const float mn = fmaxf(m, sj);
        const float corr = expf(m - mn), pj = expf(sj - mn);
        l = l * corr + pj;
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] = acc[e] * corr + (bad ? 0.f : pj * __bfloat162float(p.v_pages[row + e]));
        m = mn;
    }
    const float inv = l > 0.f ? 1.f / l : 0.f;
#pragma unroll
    for (int e = 0; e < EPL; ++e) o[e] = __float2bfloat16(acc[e] * inv);
}
