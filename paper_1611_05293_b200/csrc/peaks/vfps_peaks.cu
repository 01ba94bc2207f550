// vfps_peaks.cu -- measurement harness, NOT part of libvfps.so: micro-benchmarks for the roofline
// denominators that MEASURED_PEAKS.json does not carry: the
// shared-memory bandwidth of an SM, the bandwidth of an L2-resident copy, and the fp32 FMA-pipe
// rate (FFMA and packed FFMA2), plus how many thread-block clusters of each size the device keeps
// resident.  Built into libvfps_peaks.so by build.py; called by `bench.py --peaks`.
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

namespace {

constexpr int PK_THREADS = 1024;

// ---- shared memory: every thread streams 128-bit loads (and stores) over a 64 KB window
template <bool WRITE>
__global__ void __launch_bounds__(PK_THREADS, 1) k_smem_stream(float *sink, int iters, long long *cyc)
{
    extern __shared__ __align__(16) float4 sm4[];
    constexpr int NV = 65536 / 16;                    // 4096 float4
    for (int i = threadIdx.x; i < NV; i += PK_THREADS) sm4[i] = make_float4((float)i, 1.0f, 2.0f, 3.0f);
    __syncthreads();
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(sm4) + threadIdx.x * 16u;
    float4 acc = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {                 // 4 x 16 KB slabs: conflict-free 128-bit accesses
            const uint32_t a = base + (uint32_t)k * 16384u;
            float4 v;
            asm volatile("ld.volatile.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
            if (WRITE) {
                v.x += 1.0f;
                asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
            } else {
                acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
            }
        }
    }
    const long long t1 = clock64();
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
    if (acc.x + acc.y + acc.z + acc.w == -1.0f) sink[0] = acc.x;
}

// ---- FMA pipe: 16 independent accumulators per thread, three distinct register operands
__global__ void __launch_bounds__(PK_THREADS, 1) k_ffma(float *sink, float a, float b, int iters, long long *cyc)
{
    float x[16], y[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) { x[i] = threadIdx.x * 1e-3f + (float)i; y[i] = a + 1e-3f * (float)i; }
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], y[i], y[(i + 5) & 15]);
    }
    const long long t1 = clock64();
    float s = b;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == -1.0f) sink[0] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

// the same with two operands common to all accumulators (no register-bank conflicts possible)
__global__ void __launch_bounds__(PK_THREADS, 1) k_ffma_ab(float *sink, float a, float b, int iters, long long *cyc)
{
    float x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = threadIdx.x * 1e-3f + (float)i;
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], a, b);
    }
    const long long t1 = clock64();
    float s = b;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == -1.0f) sink[0] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

__global__ void __launch_bounds__(PK_THREADS, 1) k_ffma2(float *sink, float a, float b, int iters, long long *cyc)
{
    float2 x[8], y[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        x[i] = make_float2(threadIdx.x * 1e-3f + (float)i, (float)i);
        y[i] = make_float2(a + 1e-3f * (float)i, a - 1e-3f * (float)i);
    }
    const long long t0 = clock64();
#pragma unroll 8
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = __ffma2_rn(x[i], y[i], y[(i + 3) & 7]);
    }
    const long long t1 = clock64();
    float s = b;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i].x + x[i].y;
    if (s == -1.0f) sink[0] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

// FFMA interleaved with 128-bit shared loads in the ratio of the rotation pass (about 8 : 1)
__global__ void __launch_bounds__(PK_THREADS, 1) k_ffma_lds(float *sink, float a, float b, int iters, long long *cyc)
{
    extern __shared__ __align__(16) float4 sm4[];
    for (int i = threadIdx.x; i < 4096; i += PK_THREADS) sm4[i] = make_float4(1e-3f * (float)i, 1.0f, 2.0f, 3.0f);
    __syncthreads();
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(sm4) + threadIdx.x * 16u;
    float x[16], y[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) { x[i] = threadIdx.x * 1e-3f + (float)i; y[i] = a + 1e-3f * (float)i; }
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        float4 v0, v1;
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v0.x), "=f"(v0.y), "=f"(v0.z), "=f"(v0.w) : "r"(base + (uint32_t)(it & 3) * 16384u));
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v1.x), "=f"(v1.y), "=f"(v1.z), "=f"(v1.w) : "r"(base + (uint32_t)((it + 1) & 3) * 16384u));
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], y[i], (i & 1) ? v0.x : v1.y);
    }
    const long long t1 = clock64();
    float s = b;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == -1.0f) sink[0] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

// ---- L2-resident copy: grid-stride float4 copy, repeated by the host
__global__ void __launch_bounds__(256) k_copy(const float4 *__restrict__ src, float4 *__restrict__ dst, size_t n)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        dst[i] = src[i];
}

__global__ void k_dummy_cluster(float *p) { if (p) p[0] = 0.0f; }

struct Timer {
    cudaEvent_t a, b;
    Timer() { cudaEventCreate(&a); cudaEventCreate(&b); }
    ~Timer() { cudaEventDestroy(a); cudaEventDestroy(b); }
    void start() { cudaEventRecord(a); }
    float stop() { cudaEventRecord(b); cudaEventSynchronize(b); float ms = 0; cudaEventElapsedTime(&ms, a, b); return ms; }
};

double median_cycles(long long *d_cyc, int n)
{
    long long h[1024];
    if (n > 1024) n = 1024;
    cudaMemcpy(h, d_cyc, n * sizeof(long long), cudaMemcpyDeviceToHost);
    for (int i = 1; i < n; ++i) { long long v = h[i]; int j = i - 1; while (j >= 0 && h[j] > v) { h[j + 1] = h[j]; --j; } h[j + 1] = v; }
    return (double)h[n / 2];
}

}  // namespace

extern "C" {

// out[0]  SMs
// out[1]  shared-memory read,        B / clk / SM            out[2]  GB/s over all SMs
// out[3]  shared-memory read+write,  B / clk / SM            out[4]  GB/s over all SMs
// out[5]  FFMA  lanes / clk / SM                             out[6]  G FMA / s over all SMs
// out[7]  FFMA2 lanes / clk / SM (2 per instruction-lane)    out[8]  G FMA / s
// out[9]  FFMA with 1 LDS.128 per 8 FFMA: FFMA lanes / clk / SM
// out[10] L2-resident copy 16 MB: GB/s (read + write bytes)  out[11] the same, 32 MB
// out[12] L2-resident copy 64 MB                             out[13] HBM copy 1 GB (read + write bytes)
// out[14] effective SM clock during the FFMA run, MHz
// out[15] FFMA lanes / clk / SM with two operands common to all accumulators (x = x * a + b)
// out[16 + k] max resident clusters of size k+1 (k = 0..15) with 200 KB dynamic shared memory per CTA
// Returns 0, or the cudaError_t that stopped it.
int vfps_peaks_measure(double *out, int n_out)
{
    if (!out || n_out < 32) return -1;
    memset(out, 0, sizeof(double) * n_out);
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    out[0] = sms;
    float *sink = nullptr; long long *cyc = nullptr;
    cudaMalloc(&sink, 64); cudaMalloc(&cyc, 1024 * sizeof(long long));
    cudaFuncSetAttribute(k_smem_stream<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
    cudaFuncSetAttribute(k_smem_stream<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
    cudaFuncSetAttribute(k_ffma_lds, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
    Timer T;
    const int iters = 20000;
    for (int rep = 0; rep < 2; ++rep) {              // first pass warms up
        k_smem_stream<false><<<sms, PK_THREADS, 65536>>>(sink, iters, cyc);
        T.start(); k_smem_stream<false><<<sms, PK_THREADS, 65536>>>(sink, iters, cyc); float ms = T.stop();
        double bytes = (double)iters * 4 * 16 * PK_THREADS;
        out[1] = bytes / median_cycles(cyc, sms); out[2] = bytes * sms / (ms * 1e-3) / 1e9;
        T.start(); k_smem_stream<true><<<sms, PK_THREADS, 65536>>>(sink, iters, cyc); ms = T.stop();
        out[3] = 2 * bytes / median_cycles(cyc, sms); out[4] = 2 * bytes * sms / (ms * 1e-3) / 1e9;
        T.start(); k_ffma<<<sms, PK_THREADS>>>(sink, 0.999f, 0.5f, iters, cyc); ms = T.stop();
        double fmas = (double)iters * 16 * PK_THREADS;
        const double c1 = median_cycles(cyc, sms);
        out[5] = fmas / c1; out[6] = fmas * sms / (ms * 1e-3) / 1e9;
        out[14] = c1 / (ms * 1e-3) / 1e6;
        T.start(); k_ffma_ab<<<sms, PK_THREADS>>>(sink, 0.999f, 0.5f, iters, cyc); ms = T.stop();
        out[15] = fmas / median_cycles(cyc, sms);
        T.start(); k_ffma2<<<sms, PK_THREADS>>>(sink, 0.999f, 0.5f, iters, cyc); ms = T.stop();
        out[7] = fmas / median_cycles(cyc, sms); out[8] = fmas * sms / (ms * 1e-3) / 1e9;
        T.start(); k_ffma_lds<<<sms, PK_THREADS, 65536>>>(sink, 0.999f, 0.5f, iters, cyc); ms = T.stop();
        out[9] = fmas / median_cycles(cyc, sms);
    }
    // L2-resident and HBM copies
    const size_t sizes[4] = {16u << 20, 32u << 20, 64u << 20, 512u << 20};
    for (int s = 0; s < 4; ++s) {
        float4 *a = nullptr, *b = nullptr;
        if (cudaMalloc(&a, sizes[s]) != cudaSuccess || cudaMalloc(&b, sizes[s]) != cudaSuccess) { cudaGetLastError(); if (a) cudaFree(a); continue; }
        cudaMemset(a, 1, sizes[s]); cudaMemset(b, 0, sizes[s]);
        const size_t n = sizes[s] / 16;
        const int reps = s < 3 ? 50 : 10;
        for (int w = 0; w < 3; ++w) k_copy<<<sms * 8, 256>>>(a, b, n);
        T.start();
        for (int r = 0; r < reps; ++r) k_copy<<<sms * 8, 256>>>(a, b, n);
        const float ms = T.stop();
        out[10 + s] = 2.0 * (double)sizes[s] * reps / (ms * 1e-3) / 1e9;
        cudaFree(a); cudaFree(b);
    }
    // resident clusters per size
    cudaFuncSetAttribute(k_dummy_cluster, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_dummy_cluster, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    for (int S = 1; S <= 16; ++S) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(S * 148)); cfg.blockDim = dim3(512); cfg.dynamicSmemBytes = 200 * 1024;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = (unsigned)S; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        int mc = 0;
        if (cudaOccupancyMaxActiveClusters(&mc, k_dummy_cluster, &cfg) != cudaSuccess) { cudaGetLastError(); mc = -1; }
        out[16 + S - 1] = mc;
    }
    cudaFree(sink); cudaFree(cyc);
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaGetLastError();
    return (int)e;
}

}  // extern "C"
