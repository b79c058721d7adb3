// trace.cuh -- debug scaffolding, not part of the product: in-kernel event traces (%clock64 / %globaltimer stamps per warp of one
// chosen CTA, entry / exit time and %smid of every CTA) and the host calls that read them back.  Everything here exists only in
// builds with -DSANGAM_TRACE; in the library build.py makes, every macro below is empty and no symbol is defined.
#pragma once
#ifdef SANGAM_TRACE
#define SANGAM_TRACE_CAP 8192            // events per warp
__device__ unsigned long long g_trace[16 * SANGAM_TRACE_CAP];
__device__ unsigned int g_trace_n[16];
__device__ unsigned long long g_cta_times[2 * 512];   // per CTA: %globaltimer at entry / exit
__device__ unsigned int g_trace_cta;     // which CTA records (sangam_trace_set_cta)
__device__ __forceinline__ unsigned int* trace_cnt() {
    __shared__ unsigned int cnt[17];      // [16] = 1 if this CTA records (g_trace_cta read once: a global read per event costs an L2 trip)
    return cnt;
}
__device__ __forceinline__ void trace_ev(unsigned ev) {
    unsigned int* cnt = trace_cnt();
    if (cnt[16] && (threadIdx.x & 31) == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%clock64;" : "=l"(t));
        const unsigned w = threadIdx.x >> 5, i = cnt[w];
        cnt[w] = i + 1;
        if (i < SANGAM_TRACE_CAP) g_trace[w * SANGAM_TRACE_CAP + i] = (t << 16) | ((unsigned long long)w << 8) | ev;
        g_trace_n[w] = i + 1;
    }
}
// same record, but the time stamp is %globaltimer (ns): start/end pair gives the effective SM clock
__device__ __forceinline__ void trace_ns(unsigned ev) {
    unsigned int* cnt = trace_cnt();
    if (cnt[16] && (threadIdx.x & 31) == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        const unsigned w = threadIdx.x >> 5, i = cnt[w];
        cnt[w] = i + 1;
        if (i < SANGAM_TRACE_CAP) g_trace[w * SANGAM_TRACE_CAP + i] = (t << 16) | ((unsigned long long)w << 8) | ev;
        g_trace_n[w] = i + 1;
    }
}
#define TRACE_EV(ev) trace_ev(ev)
#define TRACE_NS(ev) trace_ns(ev)
// bits 63..54 of the entry stamp carry %smid (the timer's high bits are constant over a launch: the host masks them off)
#define TRACE_CTA(which) do { if (threadIdx.x == 0 && blockIdx.x < 512) { unsigned long long t_; unsigned sm_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); asm volatile("mov.u32 %0, %%smid;" : "=r"(sm_)); g_cta_times[2 * blockIdx.x + (which)] = (which) ? t_ : ((t_ & 0x003fffffffffffffull) | ((unsigned long long)sm_ << 54)); } } while (0)
#define TRACE_INIT() do { if (threadIdx.x < 16) trace_cnt()[threadIdx.x] = 0; if (threadIdx.x == 16) trace_cnt()[16] = blockIdx.x == g_trace_cta; __syncthreads(); } while (0)
#else
#define TRACE_EV(ev) ((void)0)
#define TRACE_NS(ev) ((void)0)
#define TRACE_CTA(which) ((void)0)
#define TRACE_INIT() ((void)0)
#endif

// decode kernels (attn_dec.cuh, attn_gqa.cuh): events of the CTA DecParams::trace_cta names
#ifdef SANGAM_TRACE
// debug builds: per-warp event trace of one CTA; the event index lives in a register of the role function (DT_DECL), so an
// event costs one clock read and one store
__device__ __forceinline__ void dtrace(int trace_cta, unsigned ev, unsigned& i) {
    if ((int)blockIdx.x == trace_cta && (threadIdx.x & 31) == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%clock64;" : "=l"(t));
        const unsigned w = threadIdx.x >> 5;
        if (i < SANGAM_TRACE_CAP) g_trace[w * SANGAM_TRACE_CAP + i] = (t << 16) | ((unsigned long long)w << 8) | ev;
        ++i;
        g_trace_n[w] = i;
    }
}
#define DT_DECL unsigned dt_i_ = 0
#define DT(ev) dtrace(p.trace_cta, ev, dt_i_)
#else
#define DT_DECL [[maybe_unused]] unsigned dt_i_ = 0
#define DT(ev) ((void)0)
#endif

// host side of the trace (debug builds only)
#ifdef SANGAM_TRACE
extern "C" int sangam_trace_cta_times(unsigned long long* host_buf) {
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(host_buf, g_cta_times, sizeof(unsigned long long) * 1024);
    return 0;
}
extern "C" int sangam_trace_set_cta(int cta) {
    unsigned int v = (unsigned int)cta, z[16] = {0};
    cudaDeviceSynchronize();
    cudaMemcpyToSymbol(g_trace_cta, &v, sizeof v);
    cudaMemcpyToSymbol(g_trace_n, z, sizeof z);
    return 0;
}
// debug builds only: copy the event trace of the recording CTA (per-warp rings, concatenated) to the host
extern "C" int sangam_trace_read(unsigned long long* host_buf, int cap) {
    unsigned int n[16];
    static unsigned long long tmp[16 * SANGAM_TRACE_CAP];
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(n, g_trace_n, sizeof n);
    cudaMemcpyFromSymbol(tmp, g_trace, sizeof tmp);
    int k = 0;
    for (int w = 0; w < 16; ++w)
        for (unsigned i = 0; i < n[w] && i < SANGAM_TRACE_CAP && k < cap; ++i) host_buf[k++] = tmp[w * SANGAM_TRACE_CAP + i];
    return k;
}
#endif
