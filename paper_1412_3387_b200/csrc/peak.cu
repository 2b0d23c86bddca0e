// peak.cu -- md_debug_peak: measured issue rate of the non-tensor pipes the hot path runs on ("measure
// the non-tensor FP64/FP32 peaks with a microbenchmark rather than trust these estimates").  One kernel per pipe: every
// thread runs 8 independent dependency chains of the instruction for `iters` trips, enough CTAs to fill every SM with 32
// warps; the rate is lane-instructions per second from CUDA events on the context's stream (best of 3 launches).
// bench.py calls it before the timed region and reports the pair-force kernel's algorithmic instruction rate against it
// (`roofline_alu`).  No arithmetic of the method lives here.
#include "md_device.cuh"

namespace {

constexpr int PEAK_ILP = 8;
constexpr int PEAK_BLOCK = 256;

template <int PIPE>
__global__ void __launch_bounds__(PEAK_BLOCK) k_peak(int iters, double seed, double *sink)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (PIPE == MD_PEAK_FP32_FMA) {
        float a[PEAK_ILP];
        const float m = 1.0f + (float)seed * 1e-9f, c = (float)seed * 1e-7f;
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) a[k] = (float)(t + k);
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int k = 0; k < PEAK_ILP; ++k) a[k] = fmaf(a[k], m, c);
        }
        float s = 0.f;
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) s += a[k];
        if (s == 12345.678f) sink[0] = s;
    } else if (PIPE == MD_PEAK_FP32_FMA2) {
        unsigned long long a[PEAK_ILP];
        const float m = 1.0f + (float)seed * 1e-9f, c = (float)seed * 1e-7f;
        unsigned long long mm, cc;
        asm("mov.b64 %0, {%1, %1};" : "=l"(mm) : "f"(m));
        asm("mov.b64 %0, {%1, %1};" : "=l"(cc) : "f"(c));
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) asm("mov.b64 %0, {%1, %1};" : "=l"(a[k]) : "f"((float)(t + k)));
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int k = 0; k < PEAK_ILP; ++k) asm("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a[k]) : "l"(mm), "l"(cc));
        }
        unsigned long long s = 0;
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) s ^= a[k];
        if (s == 0x123456789abcdefull) sink[0] = (double)s;
    } else if (PIPE == MD_PEAK_FP64_FMA) {
        double a[PEAK_ILP];
        const double m = 1.0 + seed * 1e-12, c = seed * 1e-9;
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) a[k] = (double)(t + k);
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int k = 0; k < PEAK_ILP; ++k) a[k] = fma(a[k], m, c);
        }
        double s = 0.0;
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) s += a[k];
        if (s == 12345.678) sink[0] = s;
    } else if (PIPE == MD_PEAK_INT32_MAD) {
        uint32_t a[PEAK_ILP];
        const uint32_t m = 0xD2511F53u + (uint32_t)seed, c = 0x9E3779B9u;
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) a[k] = (uint32_t)(t + k);
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int k = 0; k < PEAK_ILP; ++k) a[k] = a[k] * m + c;
        }
        uint32_t s = 0;
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) s ^= a[k];
        if (s == 0x12345678u && seed == 77.0) sink[0] = (double)s;
    } else if (PIPE == MD_PEAK_INT32_MULHI) {
        uint32_t a[PEAK_ILP];
        const uint32_t m = 0xCD9E8D57u + (uint32_t)seed;
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) a[k] = 0x80000000u + (uint32_t)(t + k);
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int k = 0; k < PEAK_ILP; ++k) a[k] = __umulhi(a[k], m) | 0x80000000u;
        }
        uint32_t s = 0;
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) s ^= a[k];
        if (s == 0x12345678u && seed == 77.0) sink[0] = (double)s;
    } else if (PIPE == MD_PEAK_CVT_F32_F64) {
        float a[PEAK_ILP];
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) a[k] = (float)(t + k) + (float)seed;
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int k = 0; k < PEAK_ILP; ++k) {  // one widening and one narrowing conversion per trip
                double d;
                asm volatile("cvt.f64.f32 %0, %1;" : "=d"(d) : "f"(a[k]));
                asm volatile("cvt.rn.f32.f64 %0, %1;" : "=f"(a[k]) : "d"(d));
            }
        }
        float s = 0.f;
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) s += a[k];
        if (s == 12345.678f) sink[0] = s;
    } else if (PIPE == MD_PEAK_RCP_F32) {
        float a[PEAK_ILP];
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) a[k] = 1.5f + (float)(t + k) * 1e-6f + (float)seed * 1e-9f;
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int k = 0; k < PEAK_ILP; ++k) asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(a[k]));
        }
        float s = 0.f;
#pragma unroll
        for (int k = 0; k < PEAK_ILP; ++k) s += a[k];
        if (s == 12345.678f) sink[0] = s;
    } else if (PIPE == MD_PEAK_LDS128) {
        __shared__ float4 buf[PEAK_BLOCK * 2];
        buf[threadIdx.x] = make_float4((float)t, 1.f, 2.f, 3.f);
        buf[threadIdx.x + PEAK_BLOCK] = make_float4(0.f, 1.f, 2.f, (float)seed);
        __syncthreads();
        float s = 0.f;
        uint32_t j = threadIdx.x;
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int k = 0; k < PEAK_ILP; ++k) {  // conflict-free: consecutive lanes, consecutive 16-byte records
                const float4 v = buf[(j + 32u * k) & (2 * PEAK_BLOCK - 1)];
                s += v.x + v.w;
            }
            j += 7u * 32u;
        }
        if (s == 12345.678f) sink[0] = s;
    }
}

template <int PIPE>
int run_peak(md_ctx *c, double *out)
{
    int dev = 0, sms = 0;
    MD_CUDA_CHECK(c, cudaGetDevice(&dev));
    MD_CUDA_CHECK(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double *sink = nullptr;
    MD_TRY(md_alloc(c, (void **)&sink, 64));
    const int grid = sms * 8, iters = 4096;
    cudaEvent_t e0, e1;
    MD_CUDA_CHECK(c, cudaEventCreate(&e0));
    MD_CUDA_CHECK(c, cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {  // the first launch warms up
        cudaEventRecord(e0, c->stream);
        k_peak<PIPE><<<grid, PEAK_BLOCK, 0, c->stream>>>(iters, 1.0, sink);
        cudaEventRecord(e1, c->stream);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    c->stats.launches += 4;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    md_free(c, sink);
    MD_CUDA_CHECK(c, cudaGetLastError());
    const double per_trip = PIPE == MD_PEAK_CVT_F32_F64 ? 2.0 : 1.0;  // instructions of the pipe per chain and trip
    *out = (double)grid * PEAK_BLOCK * (double)iters * PEAK_ILP * per_trip / (best * 1e-3) * 1e-9;
    return MD_OK;
}

}  // namespace

extern "C" int md_debug_peak(md_ctx *c, int pipe, double *giga_per_s)
{
    if (!c || !giga_per_s) return MD_EINVAL;
    switch (pipe) {
    case MD_PEAK_FP32_FMA: return run_peak<MD_PEAK_FP32_FMA>(c, giga_per_s);
    case MD_PEAK_FP32_FMA2: return run_peak<MD_PEAK_FP32_FMA2>(c, giga_per_s);
    case MD_PEAK_FP64_FMA: return run_peak<MD_PEAK_FP64_FMA>(c, giga_per_s);
    case MD_PEAK_INT32_MAD: return run_peak<MD_PEAK_INT32_MAD>(c, giga_per_s);
    case MD_PEAK_INT32_MULHI: return run_peak<MD_PEAK_INT32_MULHI>(c, giga_per_s);
    case MD_PEAK_CVT_F32_F64: return run_peak<MD_PEAK_CVT_F32_F64>(c, giga_per_s);
    case MD_PEAK_RCP_F32: return run_peak<MD_PEAK_RCP_F32>(c, giga_per_s);
    case MD_PEAK_LDS128: return run_peak<MD_PEAK_LDS128>(c, giga_per_s);
    default: c->err = "md_debug_peak: unknown pipe"; return MD_EINVAL;
    }
}
