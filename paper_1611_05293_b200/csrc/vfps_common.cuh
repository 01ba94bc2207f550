// vfps_common.cuh -- what every device translation unit shares (sm_100a): the per-handle grid
// constants, the Lagrange weights of Eq. 13 and warp sums.  No kernels here.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

// Per-phase clock stamps of the persistent kernels: compiled in only with -DVFPS_PHASE_CLOCKS
// (build.py: environment VFPS_PHASE_CLOCKS=1); release builds carry no instrumentation.
// dbg: [CTA][64 steps][8] clock64 values, written by thread 0 of every CTA.
#ifdef VFPS_PHASE_CLOCKS
#define VFPS_STAMP(dbg, step, k)                                                                            \
    do {                                                                                                    \
        if ((dbg) != nullptr && threadIdx.x == 0 && (step) < 64)                                            \
            (dbg)[((size_t)blockIdx.x * 64 + (step)) * 8 + (k)] = clock64();                                \
    } while (0)
#else
#define VFPS_STAMP(dbg, step, k) do { } while (0)
#endif

namespace vfps {

constexpr int ROT_MAX_H = 8;      // largest supported halo (source displacement + stencil reach)

struct GridConst {
    int N;             // grid points per axis
    int order;         // Lagrange points per axis
    float a;           // cos(dphi) - 1
    float b;           // -sin(dphi) * dp/dq      : dx = a*X + b*Y   (cells)
    float d;           // +sin(dphi) * dq/dp      : dy = d*X + a*Y   (cells)
    float x0c, y0c;    // q_min/dq, p_min/dp      : X = x + x0c, Y = y + y0c
    float dq, dp;
    float kick_c;      // dphi/dp                 : kick shift in cells = kick_c * V_x
    float fp_b;        // beta/steps_per_period
    float p_min;
    float q_min;
    int H;             // rotation halo
    float mh_q;        // Manhattan drift:   shift along q in cells = mh_q * Y,  mh_q = -dphi * dp/dq
    float mh_p;        // Manhattan RF kick: shift along p in cells = mh_p * X,  mh_p = +dphi * dq/dp
    int renorm;
};

// ---------------------------------------------------------------- Lagrange weights (Eq. 13)
// nodes o_k = k - floor((ORDER-1)/2); t in [0,1)
template <int ORDER>
__device__ __forceinline__ void lagrange(float t, float (&l)[ORDER]);

template <>
__device__ __forceinline__ void lagrange<2>(float t, float (&l)[2])
{
    l[0] = 1.0f - t;
    l[1] = t;
}
template <>
__device__ __forceinline__ void lagrange<3>(float t, float (&l)[3])
{
    // nodes -1, 0, 1
    const float h = 0.5f * t;
    l[0] = h * (t - 1.0f);
    l[1] = fmaf(-t, t, 1.0f);
    l[2] = h * (t + 1.0f);
}
template <>
__device__ __forceinline__ void lagrange<4>(float t, float (&l)[4])
{
    // nodes -1, 0, 1, 2.  With A = t(t-1)/6 and B = (t+1)(t-2)/2 = 3A - 1:
    //   l0 = -A (t-2), l1 = B (t-1), l2 = -B t, l3 = A (t+1)
    const float u = fmaf(t, t, -t);          // t(t-1)
    const float A = u * (1.0f / 6.0f);
    const float B = fmaf(u, 0.5f, -1.0f);
    l[0] = A * (2.0f - t);
    l[1] = fmaf(B, t, -B);
    l[2] = -B * t;
    l[3] = fmaf(A, t, A);
}

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
// Transposed warp reduction of NV (power of two <= 8) per-lane values: afterwards every lane holds
// the warp total of value index  idx = lane >> (5 - log2 NV)  (the top bits of the lane number).
// NV/2 + NV/4 + ... + 1 + (5 - log2 NV) shuffles instead of 5 NV.
template <int NV>
__device__ __forceinline__ float warp_reduce_transposed(float (&v)[NV], int lane)
{
    constexpr unsigned FULL = 0xffffffffu;
    if constexpr (NV == 1) {
        return warp_sum(v[0]);
    } else {
        // level with xor offset 16, 8, 4: keep the half of the values selected by that lane bit
        float u[NV / 2];
        const bool hi = (lane & 16) != 0;
#pragma unroll
        for (int i = 0; i < NV / 2; ++i) {
            const float keep = hi ? v[NV / 2 + i] : v[i];
            const float send = hi ? v[i] : v[NV / 2 + i];
            u[i] = keep + __shfl_xor_sync(FULL, send, 16);
        }
        if constexpr (NV == 2) {
            float r = u[0];
#pragma unroll
            for (int o = 8; o > 0; o >>= 1) r += __shfl_xor_sync(FULL, r, o);
            return r;
        } else {
            float w[NV / 4];
            const bool hi2 = (lane & 8) != 0;
#pragma unroll
            for (int i = 0; i < NV / 4; ++i) {
                const float keep = hi2 ? u[NV / 4 + i] : u[i];
                const float send = hi2 ? u[i] : u[NV / 4 + i];
                w[i] = keep + __shfl_xor_sync(FULL, send, 8);
            }
            float r;
            if constexpr (NV == 4) {
                r = w[0];
                r += __shfl_xor_sync(FULL, r, 4);
            } else {
                const bool hi3 = (lane & 4) != 0;
                const float keep = hi3 ? w[1] : w[0];
                const float send = hi3 ? w[0] : w[1];
                r = keep + __shfl_xor_sync(FULL, send, 4);
            }
            r += __shfl_xor_sync(FULL, r, 2);
            r += __shfl_xor_sync(FULL, r, 1);
            return r;
        }
    }
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace vfps
