// vfps_stream2.cuh -- second generation of the streaming (HBM / L2) kernels (sm_100a).
//
// ncu of the first generation at 2048^2 (profiles/r01_c4_grid_and_stream.md): k_rotate 27.5 us, bound by
// instruction issue (160 thread-instructions per cell, 79 % of the issue slots: tile staging with
// bounds checks, 16 shared loads and one 5-step warp reduction per cell); k_kick_fp 26 us with
// 12 % of the warp slots (132 KB of staged rows per CTA = one CTA of 8 warps per SM);
// k_wake_fft 44.5 us on ONE SM (24 serial FFT stages with global twiddle loads).  Here:
//   k_rotate2      a1 + a2: thread = column, 8 rows at a time from a register window of
//                  (8 + ORDER - 1) x ORDER taps fed by global loads that hit L1 (no staging, no
//                  bounds checks away from the grid edge; clamped loads at the edge); row sums by
//                  an 8-value transposed warp reduction
//   k_drift2       a1' first half of the Manhattan rotation (1-D shift along q) + a2
//   k_wake_direct  a3 by direct convolution (Eq. 4) on N/8 CTAs instead of one (the profile is
//                  completed by the last CTA of every row of rotation tiles)
//   k_kick_fp2     a4 + a5 + a6: four cells per thread in registers (12-value window, three
//                  128-bit loads), no shared memory, thousands of warps in flight
#pragma once
#include "vfps_cluster.cuh"

namespace vfps {

constexpr int R2_RT = 16;          // rows per rotation tile (two reduction groups of 8)
constexpr int R2_THREADS = 256;    // 8 warps = 256 columns per tile
constexpr int R2_WARPS = R2_THREADS / 32;
constexpr int K2_THREADS = 256;

// 8 values per lane -> sums over the 32 lanes.  On return v[0] of lane l holds the total of input
// value index ((l >> 4) & 1) * 4 + ((l >> 3) & 1) * 2 + ((l >> 2) & 1); 9 shuffles instead of 40.
__device__ __forceinline__ float warp_reduce8(float (&v)[8], int lane)
{
    const unsigned FULL = 0xffffffffu;
    {
        const bool up = (lane & 16) != 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float send = up ? v[i] : v[i + 4], keep = up ? v[i + 4] : v[i];
            v[i] = keep + __shfl_xor_sync(FULL, send, 16);
        }
    }
    {
        const bool up = (lane & 8) != 0;
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const float send = up ? v[i] : v[i + 2], keep = up ? v[i + 2] : v[i];
            v[i] = keep + __shfl_xor_sync(FULL, send, 8);
        }
    }
    {
        const bool up = (lane & 4) != 0;
        const float send = up ? v[0] : v[1], keep = up ? v[1] : v[0];
        v[0] = keep + __shfl_xor_sync(FULL, send, 4);
    }
    v[0] += __shfl_xor_sync(FULL, v[0], 2);
    v[0] += __shfl_xor_sync(FULL, v[0], 1);
    return v[0];
}

// read-only global load that the compiler keeps where it is written (all loads of a batch are
// issued before the arithmetic that consumes the first one)
__device__ __forceinline__ float ldg_nc(const float *p)
{
    float v;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}
// ---------------------------------------------------------------- a1 + a2: rotation + projection
// grid = (tiles_x * tiles_y, members), block = 256.  Tile = R2_RT rows x 256 columns; thread =
// column y, rows tx0 .. tx0 + R2_RT - 1 in groups of 8.  Taps come straight from global memory
// (a warp reads 128 contiguous bytes per tap; the four taps of a row and the next warp's overlap
// hit L1).  Fast path (warp-uniform): every tap of the group lies inside the grid and floor(dx),
// floor(dy) do not change along the group for any lane -> one register window for the 8 rows,
// (8 + ORDER - 1) * ORDER / 8 loads per cell.  Groups at the grid edge load clamped addresses and
// zero the outside taps; groups where a floor changes load every cell's own window with per-tap
// range checks (psi = 0 outside, A8).
// rho_part[m][x][tile_y] = dp * scale * sum over the tile's columns of psi'(x, .)
// NC: psi is read-only for the whole kernel (ld.global.nc); CLAMP: Eq. 14 (reading A9) -- the
// interpolated value is limited to the interval of the 2 x 2 nodes around the source point
template <int ORDER, bool NC = true, bool CLAMP = false>
struct GRot {
    static constexpr int O0 = (ORDER - 1) / 2;
    static __device__ __forceinline__ float ld(const float *p) { return NC ? ldg_nc(p) : *p; }
    float a, d, bY, aY, Xoff;
    const float *src;      // psi of this member
    int N, y;

    // one cell, its own floors, range-checked taps
    __device__ __forceinline__ float cell_checked(int x) const
    {
        const float X = (float)x + Xoff;
        int ix, iy;
        float tx, ty;
        floor_frac(fmaf(a, X, bY), ix, tx);
        floor_frac(fmaf(d, X, aY), iy, ty);
        float lx[ORDER], ly[ORDER];
        lagrange<ORDER>(tx, lx);
        lagrange<ORDER>(ty, ly);
        const int sx = x + ix - O0, sy = y + iy - O0;
        float acc = 0.0f, lo = 0.0f, hi = 0.0f;
#pragma unroll
        for (int i = 0; i < ORDER; ++i) {
            float rsum = 0.0f;
#pragma unroll
            for (int j = 0; j < ORDER; ++j) {
                const int xx = sx + i, yy = sy + j;
                const float v = (xx >= 0 && xx < N && yy >= 0 && yy < N) ? ld(src + (size_t)xx * N + yy) : 0.0f;
                rsum = fmaf(ly[j], v, rsum);
                if (CLAMP && (i == O0 || i == O0 + 1) && (j == O0 || j == O0 + 1)) {
                    if (i == O0 && j == O0) { lo = v; hi = v; }
                    else { lo = fminf(lo, v); hi = fmaxf(hi, v); }
                }
            }
            acc = fmaf(lx[i], rsum, acc);
        }
        if (CLAMP) acc = fminf(fmaxf(acc, lo), hi);
        return acc;
    }
    // rows x .. x+7 with floors (ix, iy) throughout and every tap inside the grid: all
    // (8 + ORDER - 1) x ORDER taps are requested before the first one is used (one exposed memory
    // latency per group instead of one per row), then row r interpolates rows r .. r+ORDER-1
    __device__ __forceinline__ void group8(const float *base, float X0, float fx, float fy, float (&out)[8]) const
    {
        float t[8 + ORDER - 1][ORDER];
        const float *p = base;
#pragma unroll
        for (int i = 0; i < 8 + ORDER - 1; ++i) {
#pragma unroll
            for (int j = 0; j < ORDER; ++j) t[i][j] = ld(p + j);      // one address per row, immediate offsets
            p += N;
        }
        interp8(t, X0, fx, fy, out);
    }
    // as group8 for a group whose taps may leave the grid (psi = 0 there, A8): rows and columns are
    // clamped into the grid for the load, and a value whose tap lies outside is replaced by zero
    __device__ __forceinline__ void group8_edge(int sx, int sy, float X0, float fx, float fy, float (&out)[8]) const
    {
        float t[8 + ORDER - 1][ORDER];
        int cy[ORDER];
        bool oky[ORDER];
#pragma unroll
        for (int j = 0; j < ORDER; ++j) {
            oky[j] = (sy + j >= 0) && (sy + j < N);
            cy[j] = min(max(sy + j, 0), N - 1);
        }
#pragma unroll
        for (int i = 0; i < 8 + ORDER - 1; ++i) {
            const bool okx = (sx + i >= 0) && (sx + i < N);
            const float *p = src + (size_t)min(max(sx + i, 0), N - 1) * N;
#pragma unroll
            for (int j = 0; j < ORDER; ++j) {
                const float v = ld(p + cy[j]);
                t[i][j] = (okx && oky[j]) ? v : 0.0f;
            }
        }
        interp8(t, X0, fx, fy, out);
    }
    // as group8 for a group at the top or bottom edge of the grid whose columns all lie inside:
    // rows outside the grid are read from a row of zeros (zrow, at least N floats) -- no per-tap
    // clamping or selection
    __device__ __forceinline__ void group8_rows(int sx, int sy, const float *zrow, float X0, float fx, float fy,
                                                float (&out)[8]) const
    {
        float t[8 + ORDER - 1][ORDER];
#pragma unroll
        for (int i = 0; i < 8 + ORDER - 1; ++i) {
            const int xx = sx + i;
            const float *p = ((xx >= 0 && xx < N) ? src + (size_t)xx * N : zrow) + sy;
#pragma unroll
            for (int j = 0; j < ORDER; ++j) t[i][j] = ld(p + j);
        }
        interp8(t, X0, fx, fy, out);
    }
    // rows r = 0..7 from the taps t[r .. r+ORDER-1][.]
    __device__ __forceinline__ void interp8(const float (&t)[8 + ORDER - 1][ORDER], float X0, float fx, float fy,
                                            float (&out)[8]) const
    {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const float X = X0 + (float)r;
            float lx[ORDER], ly[ORDER];
            lagrange<ORDER>(fmaf(a, X, bY) - fx, lx);
            lagrange<ORDER>(fmaf(d, X, aY) - fy, ly);
            float acc = 0.0f;
#pragma unroll
            for (int i = 0; i < ORDER; ++i) {
                float rsum = ly[0] * t[r + i][0];
#pragma unroll
                for (int j = 1; j < ORDER; ++j) rsum = fmaf(ly[j], t[r + i][j], rsum);
                acc = (i == 0) ? lx[0] * rsum : fmaf(lx[i], rsum, acc);
            }
            if (CLAMP) {
                const float a0 = t[r + O0][O0], a1 = t[r + O0][O0 + 1], b0 = t[r + O0 + 1][O0], b1 = t[r + O0 + 1][O0 + 1];
                acc = fminf(fmaxf(acc, fminf(fminf(a0, a1), fminf(b0, b1))), fmaxf(fmaxf(a0, a1), fmaxf(b0, b1)));
            }
            out[r] = acc;
        }
    }
};

template <int ORDER, bool CLAMP = false>
__global__ void __launch_bounds__(R2_THREADS)
k_rotate2(GridConst G, const float *__restrict__ psi_in, float *__restrict__ psi_out,
          const float *__restrict__ scale, float *__restrict__ rho_part, int tiles_y,
          float *__restrict__ rho, unsigned *__restrict__ tilectr)
{
    constexpr int O0 = (ORDER - 1) / 2;
    constexpr unsigned FULL = 0xffffffffu;
    __shared__ float red[R2_RT][R2_WARPS];
    const int N = G.N, m = blockIdx.y;
    const int tx0 = (blockIdx.x / tiles_y) * R2_RT, ty = blockIdx.x % tiles_y;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int y = ty * (32 * R2_WARPS) + warp * 32 + lane;
    const bool yok = (y < N);
    const float sc = G.renorm ? __ldg(scale + m) : 1.0f;
    float *dst = psi_out + (size_t)m * N * N;

    GRot<ORDER, true, CLAMP> rot;
    rot.src = psi_in + (size_t)m * N * N;
    rot.N = N; rot.y = min(y, N - 1);        // lanes beyond the grid compute a valid cell, never stored
    {
        const float Yc = (float)rot.y + G.y0c;
        rot.a = G.a; rot.d = G.d; rot.bY = G.b * Yc; rot.aY = G.a * Yc; rot.Xoff = G.x0c;
    }
    if (warp * 32 + ty * (32 * R2_WARPS) < N) {       // warps entirely beyond the grid have nothing to do
#pragma unroll 1
        for (int grp = 0; grp < R2_RT / 8; ++grp) {
            const int xg = tx0 + 8 * grp;             // rows xg .. xg+7 (clamped to the grid)
            float out[8];
            const int xl = min(xg + 7, N - 1), xf = min(xg, N - 1);
            const float X0 = (float)xf + rot.Xoff, XL = (float)xl + rot.Xoff;
            const float rx0 = __fadd_rd(fmaf(rot.a, X0, rot.bY), CL_MAGIC), ry0 = __fadd_rd(fmaf(rot.d, X0, rot.aY), CL_MAGIC);
            const float rxL = __fadd_rd(fmaf(rot.a, XL, rot.bY), CL_MAGIC), ryL = __fadd_rd(fmaf(rot.d, XL, rot.aY), CL_MAGIC);
            const int ix = __float_as_int(rx0) - CL_IMAGIC, iy = __float_as_int(ry0) - CL_IMAGIC;
            const int sx = xg + ix - O0, sy = rot.y + iy - O0;
            const bool uni = (rx0 == rxL) && (ry0 == ryL) && (xg + 7 < N);
            const bool inside = (sx >= 0) && (sx + 7 + ORDER - 1 < N) && (sy >= 0) && (sy + ORDER - 1 < N);
            if (__all_sync(FULL, uni && inside)) {
                rot.group8(rot.src + (size_t)sx * N + sy, X0, rx0 - CL_MAGIC, ry0 - CL_MAGIC, out);
            } else if (__all_sync(FULL, uni)) {
                rot.group8_edge(sx, sy, X0, rx0 - CL_MAGIC, ry0 - CL_MAGIC, out);
            } else {
#pragma unroll
                for (int r = 0; r < 8; ++r) out[r] = rot.cell_checked(min(xg + r, N - 1));
            }
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                out[r] *= sc;
                const bool ok = yok && (xg + r < N);
                if (ok) dst[(size_t)(xg + r) * N + y] = out[r];
                else out[r] = 0.0f;
            }
            const float tot = warp_reduce8(out, lane);
            if ((lane & 3) == 0) red[8 * grp + ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1)][warp] = tot;
        }
    } else {
        if (lane < R2_RT) red[lane][warp] = 0.0f;
    }
    __syncthreads();
    if (threadIdx.x < R2_RT) {
        const int x = tx0 + threadIdx.x;
        if (x < N) {
            float s = 0.0f;
#pragma unroll
            for (int w = 0; w < R2_WARPS; ++w) s += red[threadIdx.x][w];
            rho_part[((size_t)m * N + x) * tiles_y + ty] = G.dp * s;
            __threadfence();
        }
    }
    // ---- the last CTA of this row of tiles adds the tiles_y partial sums in a fixed order: the
    // profile is complete when the kernel ends (tilectr[m][tile row] returns to zero)
    __shared__ bool is_last;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned *ctr = tilectr + (size_t)m * gridDim.x / tiles_y + blockIdx.x / tiles_y;
        const unsigned done = atomicAdd(ctr, 1u);
        is_last = (done == (unsigned)tiles_y - 1);
        if (is_last) *ctr = 0u;
    }
    __syncthreads();
    if (is_last && threadIdx.x < R2_RT) {
        __threadfence();
        const int x = tx0 + threadIdx.x;
        if (x < N) {
            const volatile float *pp = rho_part + ((size_t)m * N + x) * tiles_y;
            float s = 0.0f;
            for (int k = 0; k < tiles_y; ++k) s += pp[k];
            rho[(size_t)m * N + x] = s;
        }
    }
}

// ---------------------------------------------------------------- a1' Manhattan rotation, first half
// Drift psi_A(q, p) = psi(q - dphi p, p) (reading A15): column y is shifted along q
// by s_y = mh_q * Y cells (Y = y + y0c), one 1-D Lagrange interpolation with per-column weights.
// Same tiling, stores, row sums and last-CTA profile as k_rotate2; thread = column, 8 rows per
// group from a window of 8 + ORDER - 1 loads (rows outside the grid read as zero, A8).  The
// second half (RF kick, a shift along p by mh_p * X cells) does not change the profile and is
// applied by k_kick_fp2<ORDER, true> together with the wake kick.
template <int ORDER, bool CLAMP = false>
__global__ void __launch_bounds__(R2_THREADS)
k_drift2(GridConst G, const float *__restrict__ psi_in, float *__restrict__ psi_out,
         const float *__restrict__ scale, float *__restrict__ rho_part, int tiles_y,
         float *__restrict__ rho, unsigned *__restrict__ tilectr)
{
    constexpr int O0 = (ORDER - 1) / 2;
    __shared__ float red[R2_RT][R2_WARPS];
    const int N = G.N, m = blockIdx.y;
    const int tx0 = (blockIdx.x / tiles_y) * R2_RT, ty = blockIdx.x % tiles_y;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int y = ty * (32 * R2_WARPS) + warp * 32 + lane, yl = min(y, N - 1);
    const float sc = G.renorm ? __ldg(scale + m) : 1.0f;
    const float *src = psi_in + (size_t)m * N * N + yl;
    float *dst = psi_out + (size_t)m * N * N;
    int mm;
    float t;
    floor_frac(G.mh_q * ((float)yl + G.y0c), mm, t);
    float l[ORDER];
    lagrange<ORDER>(t, l);
#pragma unroll
    for (int i = 0; i < ORDER; ++i) l[i] *= sc;
    if (warp * 32 + ty * (32 * R2_WARPS) < N) {
#pragma unroll 1
        for (int grp = 0; grp < R2_RT / 8; ++grp) {
            const int xg = tx0 + 8 * grp, sx = xg + mm - O0;       // first source row of the group
            float w[8 + ORDER - 1], out[8];
#pragma unroll
            for (int i = 0; i < 8 + ORDER - 1; ++i) {
                const int xx = sx + i;
                w[i] = (xx >= 0 && xx < N) ? __ldg(src + (size_t)xx * N) : 0.0f;
            }
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                float acc = l[0] * w[r];
#pragma unroll
                for (int i = 1; i < ORDER; ++i) acc = fmaf(l[i], w[r + i], acc);
                if (CLAMP)      // the weights carry the scale 1/C > 0, so do the bounds
                    acc = fminf(fmaxf(acc, sc * fminf(w[r + O0], w[r + O0 + 1])), sc * fmaxf(w[r + O0], w[r + O0 + 1]));
                const bool ok = (y < N) && (xg + r < N);
                if (ok) dst[(size_t)(xg + r) * N + y] = acc;
                out[r] = ok ? acc : 0.0f;
            }
            const float tot = warp_reduce8(out, lane);
            if ((lane & 3) == 0) red[8 * grp + ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1)][warp] = tot;
        }
    } else {
        if (lane < R2_RT) red[lane][warp] = 0.0f;
    }
    __syncthreads();
    if (threadIdx.x < R2_RT) {
        const int x = tx0 + threadIdx.x;
        if (x < N) {
            float s = 0.0f;
#pragma unroll
            for (int w = 0; w < R2_WARPS; ++w) s += red[threadIdx.x][w];
            rho_part[((size_t)m * N + x) * tiles_y + ty] = G.dp * s;
            __threadfence();
        }
    }
    __shared__ bool is_last;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned *ctr = tilectr + (size_t)m * gridDim.x / tiles_y + blockIdx.x / tiles_y;
        const unsigned done = atomicAdd(ctr, 1u);
        is_last = (done == (unsigned)tiles_y - 1);
        if (is_last) *ctr = 0u;
    }
    __syncthreads();
    if (is_last && threadIdx.x < R2_RT) {
        __threadfence();
        const int x = tx0 + threadIdx.x;
        if (x < N) {
            const volatile float *pp = rho_part + ((size_t)m * N + x) * tiles_y;
            float s = 0.0f;
            for (int k = 0; k < tiles_y; ++k) s += pp[k];
            rho[(size_t)m * N + x] = s;
        }
    }
}

// (k_wake_direct, the direct-convolution wake a3 of the stream / graph engines, is not a template and
// lives in vfps_kernels.cuh)

// (rf_stage, rf_value, rf_kick_fp_granule_any: the RF-kick stage of the Manhattan rotation, live in
// vfps_cluster.cuh beside kick_fp_granule)

// ---------------------------------------------------------------- a2 for Manhattan + clamp
// The RF kick is a shift along p and leaves the profile alone -- unless its interpolation is
// clamped (Eq. 14), which is not conservative.  Then the profile the wake needs is that of psi_B:
// one warp per row evaluates the RF stage of its row once more and sums it (nothing is stored).
// grid = (ceil(N / 8), members), block = 256.
template <int ORDER>
__global__ void __launch_bounds__(256)
k_rf_profile(GridConst G, const float *__restrict__ psi_A, float *__restrict__ rho)
{
    const int N = G.N, m = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int x = blockIdx.x * 8 + warp;
    if (x >= N) return;
    const float *row = psi_A + ((size_t)m * N + x) * N;
    int mm1;
    float t1;
    floor_frac(G.mh_p * ((float)x + G.x0c), mm1, t1);
    float l1[ORDER];
    lagrange<ORDER>(t1, l1);
    float s = 0.0f;
    for (int y = lane; y < N; y += 32) s += rf_value<ORDER, true>(row, N, y, mm1, l1);
    s = warp_sum(s);
    if (lane == 0) rho[(size_t)m * N + x] = G.dp * s;
}

// ---------------------------------------------------------------- a4 + a5 + a6: kick, FP, moments
struct Kfp2Args {
    const float *psi_in;    // rotated, scaled density (after a1)
    float *psi_out;         // end-of-step density, un-normalised
    const float *V;         // [members][N]
    const float *qstat;     // [members][4] from k_wake_fft (P_raw in slot 3), used if pw_part == nullptr
    const float *pw_part;   // [members][npw] from k_wake_direct, or nullptr
    int npw;
    const float *dpU;       // CLAMP: [members][N] dp (V + Vt) from k_wake_direct (see there)
    float *mom_part;        // [members][gridDim.x][5]: sum psi, sum Yc psi, sum Yc^2 psi, sum Xc psi, sum Xc^2 psi
    float *scale;           // [members] out: 1/C
    unsigned *blkctr;       // [members], zero between launches
    int *rowctr;            // [members] diagnostics row of this step
    float *const *diag;     // device cell holding the caller's diag pointer (may hold NULL)
    int members;
    int rows_per_cta;
};

// grid = (ceil(N / rows_per_cta), members), block = 256.  Thread = granule of four cells g..g+3 of
// one row: three 128-bit loads give the rotated density at g-4 .. g+7, kick and Fokker-Planck run
// in registers (kick_fp_granule of vfps_cluster.cuh), one 128-bit store.  The last CTA of each
// member finalises the diagnostics row and the renormalisation scalar (fixed summation order).
template <int ORDER, bool MANH = false, bool CLAMP = false>
__global__ void __launch_bounds__(K2_THREADS)
k_kick_fp2(GridConst G, Kfp2Args A)
{
    __shared__ float red[8][K2_THREADS / 32];
    __shared__ bool is_last;
    const int N = G.N, m = blockIdx.y, NQ = N >> 2, lgNQ = 31 - __clz(NQ);      // N is a power of two
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const float *src = A.psi_in + (size_t)m * N * N;
    float *dst = A.psi_out + (size_t)m * N * N;
    const float yc = 0.5f * (float)(N - 1);
    const float c1 = G.fp_b / (6.0f * G.dp), c2 = G.fp_b / (G.dp * G.dp);
    const int x_begin = blockIdx.x * A.rows_per_cta;
    const int nrows = min(N, x_begin + A.rows_per_cta) - x_begin;
    float acc[8] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f};   // s0 s1 s2 q1 q2 - - -

    if constexpr (MANH) {
        // Manhattan rotation: RF kick (shift s1 = mh_p X) then wake kick (shift kick_c V_x), two
        // successive 1-D interpolations along p in registers, then Fokker-Planck
        const int total = nrows * NQ;
        for (int idx = tid; idx < total; idx += K2_THREADS) {
            const int x = x_begin + (idx >> lgNQ), g = (idx & (NQ - 1)) << 2;
            const float *row = src + (size_t)x * N;
            const float4 z4 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            float4 v[5];
#pragma unroll
            for (int q = 0; q < 5; ++q) {
                const int c = g - 8 + 4 * q;
                v[q] = (c >= 0 && c < N) ? __ldg(reinterpret_cast<const float4 *>(row + c)) : z4;
            }
            int mm1, mm2;
            float t1, t2;
            floor_frac(G.mh_p * ((float)x + G.x0c), mm1, t1);
            floor_frac(G.kick_c * __ldg(A.V + (size_t)m * N + x), mm2, t2);
            float l1[ORDER], l2[ORDER], c1p[4], o[4];
            lagrange<ORDER>(t1, l1);
            lagrange<ORDER>(t2, l2);
#pragma unroll
            for (int c = 0; c < 4; ++c) c1p[c] = c1 * fmaf((float)(g + c), G.dp, G.p_min);
            if (mm1 >= -2 && mm1 <= 1 && mm2 >= -2 && mm2 <= 0) {
                float a[20], r[12];
#pragma unroll
                for (int q = 0; q < 5; ++q) { a[4 * q] = v[q].x; a[4 * q + 1] = v[q].y; a[4 * q + 2] = v[q].z; a[4 * q + 3] = v[q].w; }
                if (mm1 == 0) rf_stage<ORDER, 0, CLAMP>(a, l1, g, N, r);
                else if (mm1 == -1) rf_stage<ORDER, -1, CLAMP>(a, l1, g, N, r);
                else if (mm1 == 1) rf_stage<ORDER, 1, CLAMP>(a, l1, g, N, r);
                else rf_stage<ORDER, -2, CLAMP>(a, l1, g, N, r);
                if (mm2 == 0) kick_fp_granule<ORDER, 0, CLAMP>(r, l2, g, N, G.fp_b, c2, c1p, o);
                else if (mm2 == -1) kick_fp_granule<ORDER, -1, CLAMP>(r, l2, g, N, G.fp_b, c2, c1p, o);
                else kick_fp_granule<ORDER, -2, CLAMP>(r, l2, g, N, G.fp_b, c2, c1p, o);
            } else {
                rf_kick_fp_granule_any<ORDER, CLAMP>(row, l1, mm1, l2, mm2, g, N, G.fp_b, c2, c1p, o);
            }
            *reinterpret_cast<float4 *>(dst + (size_t)x * N + g) = make_float4(o[0], o[1], o[2], o[3]);
            float rs = 0.0f;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const float yy = (float)(g + c) - yc, tt = o[c] * yy;
                rs += o[c]; acc[1] += tt; acc[2] = fmaf(tt, yy, acc[2]);
            }
            const float xx = (float)x - yc, tq = rs * xx;
            acc[0] += rs; acc[3] += tq; acc[4] = fmaf(tq, xx, acc[4]);
            if (CLAMP && A.dpU != nullptr) acc[5] = fmaf(rs, __ldg(A.dpU + (size_t)m * N + x), acc[5]);
        }
    } else {
    // four granules per thread and pass: every load of the pass is issued before the first use
    const int total = nrows * NQ;
    for (int idx0 = tid; idx0 < total; idx0 += 4 * K2_THREADS) {
        float4 v0[4], v1[4], v2[4];
        float Vx[4];
        const float4 z4 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int idx = idx0 + u * K2_THREADS;
            v0[u] = v1[u] = v2[u] = z4; Vx[u] = 0.0f;
            if (idx < total) {
                const int x = x_begin + (idx >> lgNQ), g = (idx & (NQ - 1)) << 2;
                const float *row = src + (size_t)x * N;
                Vx[u] = __ldg(A.V + (size_t)m * N + x);
                if (g >= 4) v0[u] = __ldg(reinterpret_cast<const float4 *>(row + g - 4));
                v1[u] = __ldg(reinterpret_cast<const float4 *>(row + g));
                if (g + 4 < N) v2[u] = __ldg(reinterpret_cast<const float4 *>(row + g + 4));
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int idx = idx0 + u * K2_THREADS;
            if (idx < total) {
                const int x = x_begin + (idx >> lgNQ), g = (idx & (NQ - 1)) << 2;
                // kick of this row: y_r = y + sh, sh = (dphi/dp) V_x (Delta p = -dphi V)
                int mm;
                float t;
                floor_frac(G.kick_c * Vx[u], mm, t);
                float l[ORDER];
                lagrange<ORDER>(t, l);
                float c1p[4], o[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) c1p[c] = c1 * fmaf((float)(g + c), G.dp, G.p_min);
                if (mm >= -2 && mm <= 0) {
                    const float b[12] = {v0[u].x, v0[u].y, v0[u].z, v0[u].w, v1[u].x, v1[u].y, v1[u].z, v1[u].w,
                                         v2[u].x, v2[u].y, v2[u].z, v2[u].w};
                    if (mm == 0) kick_fp_granule<ORDER, 0, CLAMP>(b, l, g, N, G.fp_b, c2, c1p, o);
                    else if (mm == -1) kick_fp_granule<ORDER, -1, CLAMP>(b, l, g, N, G.fp_b, c2, c1p, o);
                    else kick_fp_granule<ORDER, -2, CLAMP>(b, l, g, N, G.fp_b, c2, c1p, o);
                } else {
                    kick_fp_granule_any<ORDER, CLAMP>(src + (size_t)x * N, l, mm, g, N, G.fp_b, c2, c1p, o);
                }
                *reinterpret_cast<float4 *>(dst + (size_t)x * N + g) = make_float4(o[0], o[1], o[2], o[3]);
                float rs = 0.0f;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float yy = (float)(g + c) - yc, tt = o[c] * yy;
                    rs += o[c]; acc[1] += tt; acc[2] = fmaf(tt, yy, acc[2]);
                }
                const float xx = (float)x - yc, tq = rs * xx;
                acc[0] += rs; acc[3] += tq; acc[4] = fmaf(tq, xx, acc[4]);
                if (CLAMP && A.dpU != nullptr) acc[5] = fmaf(rs, __ldg(A.dpU + (size_t)m * N + x), acc[5]);
            }
        }
    }
    }
    {
        const float tot = warp_reduce8(acc, lane);
        if ((lane & 3) == 0) red[((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1)][warp] = tot;
    }
    __syncthreads();
    if (tid < 6) {
        float tsum = 0.0f;
#pragma unroll
        for (int w = 0; w < K2_THREADS / 32; ++w) tsum += red[tid][w];
        A.mom_part[((size_t)m * gridDim.x + blockIdx.x) * 6 + tid] = tsum;
        __threadfence();
    }
    // ---- last CTA of this member finalises the step (deterministic: fixed summation order)
    __syncthreads();
    if (tid == 0) {
        const unsigned done = atomicAdd(A.blkctr + m, 1u);
        is_last = (done == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    if (warp == 0) {
        // (fp32 sums: fp64 adds and shuffles cost ~10 us of serial tail per step on B200)
        float f0 = 0, f1 = 0, f2 = 0, f3 = 0, f4 = 0, fp = 0;
        const float *mp = A.mom_part + (size_t)m * gridDim.x * 6;
#pragma unroll 4
        for (int i = lane; i < (int)gridDim.x; i += 32) {
            f0 += __ldcg(mp + 6 * i); f1 += __ldcg(mp + 6 * i + 1); f2 += __ldcg(mp + 6 * i + 2);
            f3 += __ldcg(mp + 6 * i + 3); f4 += __ldcg(mp + 6 * i + 4);
            if (CLAMP) fp += __ldcg(mp + 6 * i + 5);          // row sums times dp (V + Vt)
        }
        if (A.pw_part != nullptr)
            for (int i = lane; i < A.npw; i += 32) fp += __ldcg(A.pw_part + (size_t)m * A.npw + i);
        f0 = warp_sum(f0); f1 = warp_sum(f1); f2 = warp_sum(f2); f3 = warp_sum(f3); f4 = warp_sum(f4); fp = warp_sum(fp);
        if (lane == 0) {
            const double t0 = f0, t1 = f1, t2 = f2, t3 = f3, t4 = f4, tp = fp;
            const double C = (double)G.dq * (double)G.dp * t0;
            const double mp_c = t1 / t0, vp = t2 / t0 - mp_c * mp_c;
            const double mq_c = t3 / t0, vq = t4 / t0 - mq_c * mq_c;
            const double P_raw = (A.pw_part != nullptr) ? tp * (double)G.dq : (double)A.qstat[(size_t)m * 4 + 3];
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
                o[2] = (float)((double)G.p_min + (mp_c + xc) * (double)G.dp);
                o[3] = (float)(sqrt(fmax(vq, 0.0)) * (double)G.dq);
                o[4] = (float)(sqrt(fmax(vp, 0.0)) * (double)G.dp);
                o[5] = (float)(P_raw / (cc * cc));
            }
            A.blkctr[m] = 0u;
        }
    }
}

}  // namespace vfps
