// vfps_kernels.cuh -- device code of the streaming engine (sm_100a).
//
// One split step = three launches:
//   k_rotate      a1 rotation + a2 projection (per-tile partial row sums)
//   k_wake_fft    a2 finish (sum partials) + a3 wake by shared-memory FFT + q-moments + CSR power
//   k_kick_fp     a4 kick + a5 Fokker-Planck + a6 charge / p-moments; the last CTA of each member
//                 finalises the diagnostics row and the renormalisation scalar
// psi is stored UN-normalised together with a per-member scalar `scale` = 1/C of the previous
// step; k_rotate applies it (the rotation is linear), so renormalisation costs no extra pass.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace vfps {

constexpr int ROT_TX = 16;        // target rows per rotation tile
constexpr int ROT_TY = 128;       // target columns per rotation tile (4 warps x 32 lanes)
constexpr int ROT_THREADS = 256;
constexpr int ROT_MAX_H = 8;      // largest supported halo (source displacement + stencil reach)
constexpr int KFP_THREADS = 256;
constexpr int KFP_WARPS = KFP_THREADS / 32;
constexpr int KFP_PADL = 4;       // zero floats before a staged row
constexpr int KFP_PADR = 8;       // zero floats after a staged row

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
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---------------------------------------------------------------- a1 + a2: rotation + projection
// grid = (tiles_x * tiles_y, members), block = 256.  Tile = ROT_TX rows x ROT_TY columns; the
// source tile with halo H (zero outside the grid) is staged in shared memory, so every tap is an
// unchecked shared-memory read.  Warp w handles 8 consecutive rows x 32 columns (lane = column:
// stores are 128-byte coalesced, shared reads are conflict-free).
// rho_part[m][x][tile_y] = dp * scale * sum over the tile's columns of psi'(x, .)
template <int ORDER>
__global__ void __launch_bounds__(ROT_THREADS)
k_rotate(GridConst G, const float *__restrict__ psi_in, float *__restrict__ psi_out,
         const float *__restrict__ scale, float *__restrict__ rho_part, int tiles_y)
{
    extern __shared__ float tile[];
    __shared__ float red[ROT_TX][4];
    const int N = G.N, H = G.H;
    const int m = blockIdx.y;
    const int tx0 = (blockIdx.x / tiles_y) * ROT_TX;
    const int ty0 = (blockIdx.x % tiles_y) * ROT_TY;
    const int pitch = ROT_TY + 2 * H, rows = ROT_TX + 2 * H;
    const float *src = psi_in + (size_t)m * N * N;
    float *dst = psi_out + (size_t)m * N * N;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    for (int r = warp; r < rows; r += ROT_THREADS / 32) {
        const int gx = tx0 - H + r;
        const bool rok = (gx >= 0) && (gx < N);
        for (int c = lane; c < pitch; c += 32) {
            const int gy = ty0 - H + c;
            float v = 0.0f;
            if (rok && gy >= 0 && gy < N) v = __ldg(src + (size_t)gx * N + gy);
            tile[r * pitch + c] = v;
        }
    }
    __syncthreads();

    const float sc = G.renorm ? __ldg(scale + m) : 1.0f;
    const int wy = warp & 3, wx = warp >> 2;
    const int y = ty0 + wy * 32 + lane;
    // lanes / rows beyond the grid (partial tiles) compute with the last valid coordinate so that
    // their taps stay inside the staged tile; their results are never stored
    const float Y = (float)min(y, N - 1) + G.y0c;
    const float bY = G.b * Y, aY = G.a * Y;
    constexpr int O0 = (ORDER - 1) / 2;       // offset of the first node below m

#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int x = tx0 + wx * 8 + r;
        const float X = (float)min(x, N - 1) + G.x0c;
        const float dx = fmaf(G.a, X, bY);
        const float dy = fmaf(G.d, X, aY);
        const float fx = floorf(dx), fy = floorf(dy);
        float lx[ORDER], ly[ORDER];
        lagrange<ORDER>(dx - fx, lx);
        lagrange<ORDER>(dy - fy, ly);
        // tile coordinates of the first tap
        const int ix = (min(x, N - 1) - tx0) + H + (int)fx - O0;
        const int iy = (min(y, N - 1) - ty0) + H + (int)fy - O0;
        const float *t0 = tile + ix * pitch + iy;
        float acc = 0.0f;
#pragma unroll
        for (int i = 0; i < ORDER; ++i) {
            float rsum = ly[0] * t0[i * pitch];
#pragma unroll
            for (int j = 1; j < ORDER; ++j) rsum = fmaf(ly[j], t0[i * pitch + j], rsum);
            acc = (i == 0) ? lx[0] * rsum : fmaf(lx[i], rsum, acc);
        }
        acc *= sc;
        const bool ok = (x < N) && (y < N);
        if (ok) dst[(size_t)x * N + y] = acc;
        const float rs = warp_sum(ok ? acc : 0.0f);
        if (lane == 0) red[wx * 8 + r][wy] = rs;
    }
    __syncthreads();
    if (threadIdx.x < ROT_TX) {
        const int x = tx0 + threadIdx.x;
        if (x < N) {
            const float s = (red[threadIdx.x][0] + red[threadIdx.x][1]) +
                            (red[threadIdx.x][2] + red[threadIdx.x][3]);
            rho_part[((size_t)m * N + x) * tiles_y + (blockIdx.x % tiles_y)] = G.dp * s;
        }
    }
}

// ---------------------------------------------------------------- plain projection (get_profile)
// grid = (N, members), block = 128: rho[m][x] = dp * scale * sum_y psi(x,y); also the per-row
// p-moments sum_y Yc psi and sum_y Yc^2 psi (Yc = centred p index) for get_moments.
__global__ void __launch_bounds__(128)
k_project(GridConst G, const float *__restrict__ psi, const float *__restrict__ scale,
          float *__restrict__ rho, float *__restrict__ row_m1, float *__restrict__ row_m2)
{
    __shared__ double red[3][4];
    const int N = G.N, m = blockIdx.y, x = blockIdx.x;
    const float *row = psi + ((size_t)m * N + x) * N;
    const float yc = 0.5f * (float)(N - 1);
    double s0 = 0, s1 = 0, s2 = 0;
    for (int y = threadIdx.x; y < N; y += blockDim.x) {
        const double f = row[y], c = (float)y - yc;
        s0 += f; s1 += c * f; s2 += c * c * f;
    }
    s0 = warp_sum(s0); s1 = warp_sum(s1); s2 = warp_sum(s2);
    if ((threadIdx.x & 31) == 0) {
        red[0][threadIdx.x >> 5] = s0; red[1][threadIdx.x >> 5] = s1; red[2][threadIdx.x >> 5] = s2;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const double sc = G.renorm ? (double)scale[m] : 1.0;
        const size_t o = (size_t)m * N + x;
        rho[o] = (float)(G.dp * sc * (red[0][0] + red[0][1] + red[0][2] + red[0][3]));
        if (row_m1) row_m1[o] = (float)(sc * (red[1][0] + red[1][1] + red[1][2] + red[1][3]));
        if (row_m2) row_m2[o] = (float)(sc * (red[2][0] + red[2][1] + red[2][2] + red[2][3]));
    }
}

// ---------------------------------------------------------------- a3: wake by FFT (Eq. 5)
// One CTA per member, blockDim = min(1024, Nf/2).  Complex radix-2 FFT of length Nf in shared
// memory (two radix-2 stages per pass in registers): forward decimation-in-frequency (natural in,
// bit-reversed out), multiply by the
// Hermitian-extended impedance at the bit-reversed positions, inverse decimation-in-time
// (bit-reversed in, natural out) -- no permutation pass.  tw[j] = exp(-2 pi i j/Nf), j < Nf/2.
// Outputs: rho[m][x] (summed partials), V[m][x], qstat[m] = { sum rho, sum Xc rho, sum Xc^2 rho,
// P_raw } with Xc the centred q index and P_raw = (dq/Nf) sum_k Re Z_k |R_k|^2 (Eq. 16-17).
__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

__global__ void __launch_bounds__(1024)
k_wake_fft(int N, int Nf, int log2Nf, float dq, const float *__restrict__ rho_part, int nparts,
           const float2 *__restrict__ Z, const float2 *__restrict__ tw, float *__restrict__ rho_out,
           float *__restrict__ V, float *__restrict__ qstat)
{
    extern __shared__ float2 s[];          // Nf points, then Nf - 1 twiddles, one contiguous table per stage
    __shared__ float red[4][32];
    float2 *stw = s + Nf;
    const int m = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
    const float xc = 0.5f * (float)(N - 1);
    float s0 = 0, s1 = 0, s2 = 0, pw = 0;
    for (int x = tid; x < Nf; x += nt) {
        float r = 0.0f;
        if (x < N) {
            const float *pp = rho_part + ((size_t)m * N + x) * nparts;
#pragma unroll 8
            for (int k = 0; k < nparts; ++k) r += __ldg(pp + k);
            rho_out[(size_t)m * N + x] = r;
            const float c = (float)x - xc, t = c * r;
            s0 += r; s1 += t; s2 = fmaf(t, c, s2);
        }
        s[x] = make_float2(r, 0.0f);
    }
    if (Z != nullptr) {
        const float2 *Zm = Z + (size_t)m * (Nf / 2 + 1);
        // The twiddles are read 2 log2(Nf) times: stage them once, as one contiguous table per
        // butterfly span (entry half - 1 + pos = tw[pos * (Nf/2) / half]): reading the single
        // table with stride (Nf/2)/half put up to 32 lanes on one bank in most stages.
        for (int j = tid; j < Nf - 1; j += nt) {
            const int half = 1 << (31 - __clz(j + 1)), pos = j + 1 - half;
            stw[j] = __ldg(tw + pos * ((Nf >> 1) / half));
        }
        __syncthreads();
        // forward, decimation in frequency; two radix-2 stages (spans 2q and q) per pass in registers:
        // half as many passes over shared memory and half as many barriers
        int half = Nf >> 1;
        for (; half >= 2; half >>= 2) {
            const int q = half >> 1;
            const float2 *w2 = stw + (half - 1), *w1 = stw + (q - 1);
            for (int j = tid; j < (Nf >> 2); j += nt) {
                const int pos = j & (q - 1), i0 = ((j - pos) << 2) + pos, i1 = i0 + q, i2 = i1 + q, i3 = i2 + q;
                const float2 x0 = s[i0], x1 = s[i1], x2 = s[i2], x3 = s[i3];
                const float2 u0 = make_float2(x0.x + x2.x, x0.y + x2.y), u1 = make_float2(x1.x + x3.x, x1.y + x3.y);
                const float2 u2 = cmul(make_float2(x0.x - x2.x, x0.y - x2.y), w2[pos]);
                const float2 u3 = cmul(make_float2(x1.x - x3.x, x1.y - x3.y), w2[pos + q]);
                const float2 wq = w1[pos];
                s[i0] = make_float2(u0.x + u1.x, u0.y + u1.y);
                s[i1] = cmul(make_float2(u0.x - u1.x, u0.y - u1.y), wq);
                s[i2] = make_float2(u2.x + u3.x, u2.y + u3.y);
                s[i3] = cmul(make_float2(u2.x - u3.x, u2.y - u3.y), wq);
            }
            __syncthreads();
        }
        if (half == 1) {                                          // odd log2(Nf): one radix-2 stage left (w = 1)
            for (int j = tid; j < (Nf >> 1); j += nt) {
                const float2 u = s[2 * j], v = s[2 * j + 1];
                s[2 * j] = make_float2(u.x + v.x, u.y + v.y);
                s[2 * j + 1] = make_float2(u.x - v.x, u.y - v.y);
            }
            __syncthreads();
        }
        for (int i = tid; i < Nf; i += nt) {                      // x Z, power spectrum
            const int k = (int)(__brev((unsigned)i) >> (32 - log2Nf));
            float2 z;
            if (k <= (Nf >> 1)) {
                z = __ldg(Zm + k);
                if (k == 0 || k == (Nf >> 1)) z.y = 0.0f;
            } else {
                z = __ldg(Zm + (Nf - k));
                z.y = -z.y;
            }
            const float2 R = s[i];
            pw = fmaf(z.x, fmaf(R.x, R.x, R.y * R.y), pw);
            s[i] = cmul(R, z);
        }
        __syncthreads();
        // inverse, decimation in time, mirrored: the single radix-2 stage first if log2(Nf) is odd,
        // then spans q and 2q per pass
        int hq = 1;
        if (log2Nf & 1) {
            for (int j = tid; j < (Nf >> 1); j += nt) {
                const float2 u = s[2 * j], v = s[2 * j + 1];
                s[2 * j] = make_float2(u.x + v.x, u.y + v.y);
                s[2 * j + 1] = make_float2(u.x - v.x, u.y - v.y);
            }
            __syncthreads();
            hq = 2;
        }
        for (int q = hq; q <= (Nf >> 2); q <<= 2) {
            const float2 *w1 = stw + (q - 1), *w2 = stw + (2 * q - 1);
            for (int j = tid; j < (Nf >> 2); j += nt) {
                const int pos = j & (q - 1), i0 = ((j - pos) << 2) + pos, i1 = i0 + q, i2 = i1 + q, i3 = i2 + q;
                float2 wq = w1[pos], wa = w2[pos], wb = w2[pos + q];
                wq.y = -wq.y; wa.y = -wa.y; wb.y = -wb.y;
                const float2 x0 = s[i0], x2 = s[i2];
                const float2 v1 = cmul(s[i1], wq), v3 = cmul(s[i3], wq);
                const float2 y0 = make_float2(x0.x + v1.x, x0.y + v1.y), y1 = make_float2(x0.x - v1.x, x0.y - v1.y);
                const float2 y2 = make_float2(x2.x + v3.x, x2.y + v3.y), y3 = make_float2(x2.x - v3.x, x2.y - v3.y);
                const float2 t2 = cmul(y2, wa), t3 = cmul(y3, wb);
                s[i0] = make_float2(y0.x + t2.x, y0.y + t2.y);
                s[i2] = make_float2(y0.x - t2.x, y0.y - t2.y);
                s[i1] = make_float2(y1.x + t3.x, y1.y + t3.y);
                s[i3] = make_float2(y1.x - t3.x, y1.y - t3.y);
            }
            __syncthreads();
        }
        const float inv = 1.0f / (float)Nf;
        for (int x = tid; x < N; x += nt) V[(size_t)m * N + x] = s[x].x * inv;
    } else {
        for (int x = tid; x < N; x += nt) V[(size_t)m * N + x] = 0.0f;
    }
    // fp32 sums in a fixed order (fp64 adds and shuffles are ~50x slower on B200)
    s0 = warp_sum(s0); s1 = warp_sum(s1); s2 = warp_sum(s2); pw = warp_sum(pw);
    if ((tid & 31) == 0) {
        red[0][tid >> 5] = s0; red[1][tid >> 5] = s1; red[2][tid >> 5] = s2; red[3][tid >> 5] = pw;
    }
    __syncthreads();
    if (tid < 4) {
        float t = 0;
        for (int w = 0; w < (nt + 31) / 32; ++w) t += red[tid][w];
        if (tid == 3) t *= dq / (float)Nf;
        qstat[(size_t)m * 4 + tid] = t;
    }
}

// ---------------------------------------------------------------- a4 + a5 + a6: kick, FP, moments
struct KfpArgs {
    const float *psi_in;    // psi' (rotated, scaled)
    float *psi_out;         // psi''' (un-normalised)
    const float *V;         // [members][N]
    const float *qstat;     // [members][4] from k_wake_fft
    float *mom_part;        // [members][gridDim.x][5]: sum psi, sum Yc psi, sum Yc^2 psi, sum Xc psi, sum Xc^2 psi
    float *scale;           // [members] out: 1/C
    unsigned *blkctr;       // [members], zero between launches
    int *rowctr;            // [members] diagnostics row of this step
    float *const *diag;     // device cell holding the caller's diag pointer (may hold NULL)
    int members;
    int rows_per_cta;
};

// composite of kick (shift t along p, node m) and the Fokker-Planck update for one staged row.
// row: shared-memory row with KFP_PADL zeros before index 0 and KFP_PADR zeros after index N-1.
template <int ORDER>
__device__ __forceinline__ float kicked(const float *row, int N, int y, int m, const float (&l)[ORDER])
{
    // psi''(y) = sum_j l_j psi'(y + m + o_j); psi' = 0 outside [0, N)
    constexpr int O0 = (ORDER - 1) / 2;
    const int base = y + m - O0;
    float acc = 0.0f;
#pragma unroll
    for (int j = 0; j < ORDER; ++j) {
        const int i = base + j;
        const float v = (i >= -KFP_PADL && i < N + KFP_PADR) ? row[i] : 0.0f;
        acc = (j == 0) ? l[0] * v : fmaf(l[j], v, acc);
    }
    return acc;
}

// grid = (ceil(N / rows_per_cta), members), block = 256 (8 warps, one row per warp at a time).
// Shared memory: per warp two rows of (KFP_PADL + N + KFP_PADR) floats (psi' and psi'').
template <int ORDER>
__global__ void __launch_bounds__(KFP_THREADS)
k_kick_fp(GridConst G, KfpArgs A)
{
    extern __shared__ float smem[];
    __shared__ float red[5][KFP_WARPS];
    __shared__ bool is_last;
    const int N = G.N, m = blockIdx.y;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rowlen = KFP_PADL + N + KFP_PADR;
    float *r1 = smem + (size_t)warp * 2 * rowlen + KFP_PADL;     // psi'  (index 0 = y 0)
    float *r2 = r1 + rowlen;                                       // psi''
    const float *src = A.psi_in + (size_t)m * N * N;
    float *dst = A.psi_out + (size_t)m * N * N;
    const float yc = 0.5f * (float)(N - 1);
    // FP increment coefficients: incr = b*f0 + b*p*(-2 f-1 - 3 f0 + 6 f+1 - f+2)/(6 dp)
    //                                  + b*(f-1 - 2 f0 + f+1)/dp^2
    const float c1 = G.fp_b / (6.0f * G.dp);
    const float c2 = G.fp_b / (G.dp * G.dp);

    for (int i = lane; i < KFP_PADL; i += 32) { r1[-1 - i] = 0.0f; r2[-1 - i] = 0.0f; }
    for (int i = lane; i < KFP_PADR; i += 32) { r1[N + i] = 0.0f; r2[N + i] = 0.0f; }

    float s0 = 0.0f, s1 = 0.0f, s2 = 0.0f, q1 = 0.0f, q2 = 0.0f;
    const int x_begin = blockIdx.x * A.rows_per_cta;
    const int x_end = min(N, x_begin + A.rows_per_cta);
    for (int x = x_begin + warp; x < x_end; x += KFP_WARPS) {
        __syncwarp();
        const float4 *g4 = reinterpret_cast<const float4 *>(src + (size_t)x * N);
        for (int c = lane; c < N / 4; c += 32) *reinterpret_cast<float4 *>(r1 + 4 * c) = __ldg(g4 + c);
        // kick parameters of this row: y_r = y + sh, sh = (dphi/dp) * V_x  (Delta p = -dphi V)
        const float sh = G.kick_c * __ldg(A.V + (size_t)m * N + x);
        const float fm = floorf(sh);
        float l[ORDER];
        lagrange<ORDER>(sh - fm, l);
        const int mm = (int)fm;
        __syncwarp();
        for (int y = lane; y < N; y += 32) r2[y] = kicked<ORDER>(r1, N, y, mm, l);
        __syncwarp();
        float rs = 0.0f;
        for (int y = lane; y < N; y += 32) {
            const float fm1 = r2[y - 1], f0 = r2[y], fp1 = r2[y + 1], fp2 = r2[y + 2];
            const float p = fmaf((float)y, G.dp, G.p_min);
            const float d1 = fmaf(-2.0f, fm1, fmaf(-3.0f, f0, fmaf(6.0f, fp1, -fp2)));
            const float d2 = (fm1 + fp1) - 2.0f * f0;
            const float incr = fmaf(G.fp_b, f0, fmaf(c1 * p, d1, c2 * d2));
            const float out = f0 + incr;
            dst[(size_t)x * N + y] = out;
            const float yy = (float)y - yc;
            const float t = out * yy;
            rs += out; s1 += t; s2 = fmaf(t, yy, s2);
        }
        // q moments of the end-of-step psi from the row sum (every lane gets the same value)
        rs = warp_sum(rs);
        const float xx = (float)x - yc;
        const float tq = rs * xx;
        s0 += rs; q1 += tq; q2 = fmaf(tq, xx, q2);
    }
    s1 = warp_sum(s1); s2 = warp_sum(s2);
    if (lane == 0) { red[0][warp] = s0; red[1][warp] = s1; red[2][warp] = s2; red[3][warp] = q1; red[4][warp] = q2; }
    __syncthreads();
    if (threadIdx.x < 5) {
        float t = 0.0f;
#pragma unroll
        for (int w = 0; w < KFP_WARPS; ++w) t += red[threadIdx.x][w];
        A.mom_part[((size_t)m * gridDim.x + blockIdx.x) * 5 + threadIdx.x] = t;
    }
    // ---- last CTA of this member finalises the step (deterministic: fixed summation order)
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned done = atomicAdd(A.blkctr + m, 1u);
        is_last = (done == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    if (warp == 0) {
        double t0 = 0, t1 = 0, t2 = 0, t3 = 0, t4 = 0;
        const volatile float *mp = A.mom_part + (size_t)m * gridDim.x * 5;
        for (int i = lane; i < (int)gridDim.x; i += 32) {
            t0 += mp[5 * i]; t1 += mp[5 * i + 1]; t2 += mp[5 * i + 2]; t3 += mp[5 * i + 3]; t4 += mp[5 * i + 4];
        }
        t0 = warp_sum(t0); t1 = warp_sum(t1); t2 = warp_sum(t2); t3 = warp_sum(t3); t4 = warp_sum(t4);
        if (lane == 0) {
            const double C = (double)G.dq * (double)G.dp * t0;
            const double mp_c = t1 / t0;                       // <p> in centred cells
            const double vp = t2 / t0 - mp_c * mp_c;
            const float *qs = A.qstat + (size_t)m * 4;
            const double mq_c = t3 / t0, vq = t4 / t0 - mq_c * mq_c;
            A.scale[m] = (float)(1.0 / C);
            const int row = A.rowctr[m];
            A.rowctr[m] = row + 1;
            float *diag = *A.diag;
            if (diag != nullptr) {
                float *o = diag + ((size_t)row * A.members + m) * 6;
                const double xc = 0.5 * (double)(N - 1);
                const double cc = G.renorm ? C : 1.0;
                o[0] = (float)C;
                o[1] = (float)((double)G.q_min + (mq_c + xc) * (double)G.dq);
                o[2] = (float)((double)G.p_min + (mp_c + (double)yc) * (double)G.dp);
                o[3] = (float)(sqrt(fmax(vq, 0.0)) * (double)G.dq);
                o[4] = (float)(sqrt(fmax(vp, 0.0)) * (double)G.dp);
                o[5] = (float)((double)qs[3] / (cc * cc));
            }
            A.blkctr[m] = 0u;
        }
    }
}

// ---------------------------------------------------------------- helpers for set / get calls
__global__ void k_scale_copy(const float *__restrict__ psi, const float *__restrict__ scale,
                             float *__restrict__ out, size_t cells_per_member, int renorm)
{
    const int m = blockIdx.y;
    const float sc = renorm ? scale[m] : 1.0f;
    const size_t base = (size_t)m * cells_per_member;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < cells_per_member;
         i += (size_t)gridDim.x * blockDim.x)
        out[base + i] = psi[base + i] * sc;
}

__global__ void k_fill(float *p, float v, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

__global__ void k_set_ctl(float **diag_cell, float *diag, int *rowctr, unsigned *blkctr, int members)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) *diag_cell = diag;
    if (i < members) { rowctr[i] = 0; blkctr[i] = 0u; }
}

// { C, <q>, <p>, sigma_q, sigma_p, P } of the current psi from k_project's rows + k_wake_fft's P.
__global__ void __launch_bounds__(256)
k_moments_final(GridConst G, const float *__restrict__ rho, const float *__restrict__ row_m1,
                const float *__restrict__ row_m2, const float *__restrict__ qstat,
                float *__restrict__ out)
{
    __shared__ double red[5][8];
    const int N = G.N, m = blockIdx.x;
    const double xc = 0.5 * (double)(N - 1);
    double r0 = 0, q1 = 0, q2 = 0, p1 = 0, p2 = 0;
    for (int x = threadIdx.x; x < N; x += blockDim.x) {
        const size_t o = (size_t)m * N + x;
        const double r = rho[o], c = (double)x - xc;
        r0 += r; q1 += c * r; q2 += c * c * r; p1 += row_m1[o]; p2 += row_m2[o];
    }
    r0 = warp_sum(r0); q1 = warp_sum(q1); q2 = warp_sum(q2); p1 = warp_sum(p1); p2 = warp_sum(p2);
    if ((threadIdx.x & 31) == 0) {
        const int w = threadIdx.x >> 5;
        red[0][w] = r0; red[1][w] = q1; red[2][w] = q2; red[3][w] = p1; red[4][w] = p2;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t[5];
        for (int k = 0; k < 5; ++k) { t[k] = 0; for (int w = 0; w < 8; ++w) t[k] += red[k][w]; }
        const double S = t[0] / (double)G.dp;                 // sum of psi (scaled)
        const double mq = t[1] / t[0], vq = t[2] / t[0] - mq * mq;
        const double mp = t[3] / S, vp = t[4] / S - mp * mp;
        float *o = out + (size_t)m * 6;
        o[0] = (float)((double)G.dq * t[0]);
        o[1] = (float)((double)G.q_min + (mq + xc) * (double)G.dq);
        o[2] = (float)((double)G.p_min + (mp + xc) * (double)G.dp);
        o[3] = (float)(sqrt(fmax(vq, 0.0)) * (double)G.dq);
        o[4] = (float)(sqrt(fmax(vp, 0.0)) * (double)G.dp);
        o[5] = qstat[(size_t)m * 4 + 3];
    }
}

}  // namespace vfps
