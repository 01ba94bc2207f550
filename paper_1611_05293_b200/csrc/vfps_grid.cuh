// vfps_grid.cuh -- persistent cooperative-grid engine for grids that do not fit on chip (sm_100a).
//
// The streaming engines pay three kernel launches per split step; at 2048^2 each kernel has
// ~5-10 us of work and 3-5 us of ramp-up, tail and (for the reductions) a serial last-CTA epilogue
// (profiles/r01_c4_grid_and_stream.md).  Here ONE cooperative launch advances all n steps of a vfps_step
// call: every SM keeps CTAs resident, psi ping-pongs between two HBM buffers that stay in the
// 126 MB L2 (2 x 16 MB at 2048^2), and the two global dependencies of a step are grid barriers:
//   phase 1  a1 + a2: rotation tiles of GR_RT rows x 256 columns (register window, as k_rotate2),
//            per-tile row sums -> rho_part[tile_y][x]
//   -- grid barrier --
//   phase 2  every CTA sums the tile_y partial profiles (N * tiles_y coalesced L2 loads), then for
//            its KR rows: a3 direct-convolution wake (Eq. 4), a4 + a5 kick and Fokker-Planck in
//            registers (as k_kick_fp2), partial sums for a6 -> mom_part[cta]
//   -- grid barrier --
//   phase 3  every CTA reads the charge of the step from a 32.32 fixed-point accumulator that the
//            CTAs fed with integer atomics in phase 2 (exact, order-independent) -> C, 1/C;
//            CTA 0 sums the other partial sums in a fixed order and writes the diagnostics row.
// With VFPS_FLAG_ROT_MANHATTAN (template MANH) phase 1 is the drift (1-D shift along q) and phase 2
// applies the RF kick before the wake kick (vfps_stream2.cuh: k_drift2, rf_stage); with CLAMP as well the
// profile is that of the RF-kicked rows, formed by their owners behind a third grid barrier.
// Template CLAMP: clamped interpolation (Eq. 14, reading A9) in every interpolation of the step.
// One simulation per handle (members == 1); batches of on-chip grids use the cluster engine.
#pragma once
#include "vfps_stream2.cuh"

#include <cooperative_groups.h>

namespace vfps {

constexpr int GR_RT = 8;            // rows per rotation tile (one reduction group)
constexpr int GR_THREADS = 256;
constexpr int GR_WARPS = GR_THREADS / 32;
constexpr int GR_NPART = 8;         // partial sums per CTA per step

struct GridArgs {
    float *psi;          // [N][N] in/out, un-normalised
    float *psi_tmp;      // [N][N] rotated density
    float *scale;        // [1] in/out: 1/C of the last step
    const float *wfun;   // [2N] wake function, lag d at index d + N - 1; nullptr = no wake
    float *rho_part;     // [tiles_y][N]
    float *mom_part;     // [GR_NPART][gridDim.x]: sum psi, sum Yc psi, sum Yc^2 psi, sum Xc psi, sum Xc^2 psi, sum rho V
    float *diag;         // [nsteps][1][6] or nullptr
    int nsteps;
    int tiles_y;         // column tiles of 256
    int KR;              // rows per CTA in phase 2
    const float *zrow;          // N zeros: stands in for the rows outside the grid (A8)
    unsigned long long *qacc;   // [2] charge of the step in 32.32 fixed point (integer atomics: exact,
                                // order-independent), zero at launch; parity = step & 1
    long long *dbg;      // nullptr, or [CTA][64 steps][8] clock64 stamps (debug aid)
};

// profile (N), wake-function window (N + KR), V of the CTA's rows (KR); with clamped interpolation
// also the window of the transposed wake (N + KR) and dp (V + Vt) of the rows (KR)
__host__ __device__ inline size_t grid_smem_floats(int N, int KR, bool clamp = false)
{
    return (size_t)2 * N + 2 * KR + 8 + (clamp ? (size_t)N + 2 * KR : 0);
}

template <int ORDER, bool MANH = false, bool CLAMP = false>
__global__ void __launch_bounds__(GR_THREADS, 2)
k_grid_step(GridConst G, GridArgs A)
{
    namespace cg = cooperative_groups;
    constexpr int O0 = (ORDER - 1) / 2;
    constexpr unsigned FULL = 0xffffffffu;
    cg::grid_group grid = cg::this_grid();
    extern __shared__ float gsm[];
    __shared__ float red[8][GR_WARPS];
    __shared__ float redt[2][8][GR_WARPS];     // rotation tiles: two buffers, one barrier per tile
    __shared__ float s_sc;
    const int N = G.N, NQ = N >> 2, lgNQ = 31 - __clz(NQ);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    float *srho = gsm, *sw = gsm + N, *sV = gsm + 2 * N + A.KR;       // sw: N + KR - 1 lags
    float *sw2 = gsm + 2 * N + 2 * A.KR + 8, *sU = sw2 + N + A.KR;     // CLAMP only (grid_smem_floats)
    const int tiles_x = (N + GR_RT - 1) / GR_RT, ntiles = tiles_x * A.tiles_y;
    const int lg_ty = 31 - __clz(A.tiles_y);           // tiles_y is a power of two (N is; 256 columns per tile)
    const float yc = 0.5f * (float)(N - 1);
    const float c1 = G.fp_b / (6.0f * G.dp), c2 = G.fp_b / (G.dp * G.dp);
    float sc = G.renorm ? A.scale[0] : 1.0f;

    for (int step = 0; step < A.nsteps; ++step) {
        VFPS_STAMP(A.dbg, step, 0);
        // ================= phase 1: rotation psi -> psi_tmp (times 1/C), partial profiles
        // round k: CTA c takes tile k*grid + (c + k) mod grid.  (With the plain c + k*grid a CTA keeps
        // the same column tile in every round when grid is a multiple of tiles_y, so the CTAs that
        // own the edge columns -- clamped-load path -- are slower in every round and everybody
        // waits for them at the barrier.)
        for (int k = 0, tb = 0; tb < ntiles; ++k, tb += gridDim.x) {
            int rot_c = (int)blockIdx.x + k;
            while (rot_c >= (int)gridDim.x) rot_c -= (int)gridDim.x;
            const int t = tb + rot_c;
            if (t >= ntiles) continue;
            const int xg = (t >> lg_ty) * GR_RT, ty = t & (A.tiles_y - 1);
            const int y = ty * (32 * GR_WARPS) + warp * 32 + lane;
            float out[8];
#pragma unroll
            for (int r = 0; r < 8; ++r) out[r] = 0.0f;
            if (ty * (32 * GR_WARPS) + warp * 32 < N) {
                if constexpr (MANH) {
                    // Manhattan drift (L136): column y shifted along q by mh_q * Y cells
                    const int yl = min(y, N - 1);
                    int mm;
                    float t;
                    floor_frac(G.mh_q * ((float)yl + G.y0c), mm, t);
                    float l[ORDER], w[8 + ORDER - 1];
                    lagrange<ORDER>(t, l);
                    const int sx = xg + mm - O0;
                    const float *src = A.psi + yl;
#pragma unroll
                    for (int i = 0; i < 8 + ORDER - 1; ++i) {
                        const int xx = sx + i;
                        w[i] = (xx >= 0 && xx < N) ? src[(size_t)xx * N] : 0.0f;
                    }
#pragma unroll
                    for (int r = 0; r < 8; ++r) {
                        float a = l[0] * w[r];
#pragma unroll
                        for (int i = 1; i < ORDER; ++i) a = fmaf(l[i], w[r + i], a);
                        if (CLAMP) a = fminf(fmaxf(a, fminf(w[r + O0], w[r + O0 + 1])), fmaxf(w[r + O0], w[r + O0 + 1]));
                        out[r] = a;
                    }
                } else {
                GRot<ORDER, false, CLAMP> rot;
                rot.src = A.psi; rot.N = N; rot.y = min(y, N - 1);
                const float Yc = (float)rot.y + G.y0c;
                rot.a = G.a; rot.d = G.d; rot.bY = G.b * Yc; rot.aY = G.a * Yc; rot.Xoff = G.x0c;
                const int xl = min(xg + 7, N - 1);
                const float X0 = (float)xg + rot.Xoff, XL = (float)xl + rot.Xoff;
                const float rx0 = __fadd_rd(fmaf(rot.a, X0, rot.bY), CL_MAGIC), ry0 = __fadd_rd(fmaf(rot.d, X0, rot.aY), CL_MAGIC);
                const float rxL = __fadd_rd(fmaf(rot.a, XL, rot.bY), CL_MAGIC), ryL = __fadd_rd(fmaf(rot.d, XL, rot.aY), CL_MAGIC);
                const int ix = __float_as_int(rx0) - CL_IMAGIC, iy = __float_as_int(ry0) - CL_IMAGIC;
                const int sx = xg + ix - O0, sy = rot.y + iy - O0;
                const bool uni = (rx0 == rxL) && (ry0 == ryL) && (xg + 7 < N);
                const bool inside = (sx >= 0) && (sx + 7 + ORDER - 1 < N) && (sy >= 0) && (sy + ORDER - 1 < N);
                if (__all_sync(FULL, uni && inside)) {
                    rot.group8(A.psi + (size_t)sx * N + sy, X0, rx0 - CL_MAGIC, ry0 - CL_MAGIC, out);
                } else if (__all_sync(FULL, uni && (sy >= 0) && (sy + ORDER - 1 < N))) {
                    rot.group8_rows(sx, sy, A.zrow, X0, rx0 - CL_MAGIC, ry0 - CL_MAGIC, out);
                } else if (__all_sync(FULL, uni)) {
                    rot.group8_edge(sx, sy, X0, rx0 - CL_MAGIC, ry0 - CL_MAGIC, out);
                } else {
#pragma unroll
                    for (int r = 0; r < 8; ++r) out[r] = rot.cell_checked(min(xg + r, N - 1));
                }
                }
                float *orow = A.psi_tmp + (size_t)xg * N + y;
                if (__all_sync(FULL, y < N) && xg + 8 <= N) {           // whole 8 x 32 patch inside the grid
#pragma unroll
                    for (int r = 0; r < 8; ++r) {
                        out[r] *= sc;
                        *orow = out[r];
                        orow += N;
                    }
                } else {
#pragma unroll
                    for (int r = 0; r < 8; ++r) {
                        out[r] *= sc;
                        if (y < N && xg + r < N) orow[(size_t)r * N] = out[r];
                        else out[r] = 0.0f;
                    }
                }
            }
            // (buffer k & 1 was last read two tiles ago, i.e. before the barrier of the previous tile)
            const float tot = warp_reduce8(out, lane);
            if ((lane & 3) == 0) redt[k & 1][((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1)][warp] = tot;
            __syncthreads();
            if (!(MANH && CLAMP) && tid < GR_RT && xg + tid < N) {
                float s = 0.0f;
#pragma unroll
                for (int w = 0; w < GR_WARPS; ++w) s += redt[k & 1][tid][w];
                A.rho_part[(size_t)ty * N + xg + tid] = G.dp * s;
            }
        }
        VFPS_STAMP(A.dbg, step, 1);
        grid.sync();
        VFPS_STAMP(A.dbg, step, 2);
        const int r0 = blockIdx.x * A.KR, r1 = min(N, r0 + A.KR);
        if constexpr (MANH && CLAMP) {
            // The clamped RF kick does not conserve the row sums, and the wake acts on the profile AFTER
            // it (L136 order drift, RF kick, wake kick): row sums of the RF-kicked rows r0 .. r1-1 (as
            // k_rf_profile), then one more grid barrier before anybody reads the profile.
            for (int r = warp; r < r1 - r0; r += GR_WARPS) {
                const int x = r0 + r;
                const float *row = A.psi_tmp + (size_t)x * N;
                int mm1;
                float t1;
                floor_frac(G.mh_p * ((float)x + G.x0c), mm1, t1);
                float l1[ORDER];
                lagrange<ORDER>(t1, l1);
                float s = 0.0f;
                for (int y = lane; y < N; y += 32) s += rf_value<ORDER, true>(row, N, y, mm1, l1);
                s = warp_sum(s);
                if (lane == 0) A.rho_part[x] = G.dp * s;
            }
            grid.sync();
        }
        // ================= phase 2: profile, wake, kick + Fokker-Planck of the rows r0 .. r1-1
        float acc[8] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f};   // s0 s1 s2 q1 q2 pw - -
        if (r0 < N) {
            for (int x4 = tid; x4 < NQ; x4 += 2 * GR_THREADS) {   // two columns of float4 per pass: up to
                const int x4b = x4 + GR_THREADS;                   // 16 loads in flight per thread
                const bool two = (x4b < NQ);
                float4 r = make_float4(0.0f, 0.0f, 0.0f, 0.0f), q = r;
#pragma unroll 8
                for (int k = 0; k < ((MANH && CLAMP) ? 1 : A.tiles_y); ++k) {
                    const float4 *pk = reinterpret_cast<const float4 *>(A.rho_part + (size_t)k * N);
                    const float4 v = __ldcg(pk + x4);
                    const float4 u = two ? __ldcg(pk + x4b) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                    r.x += v.x; r.y += v.y; r.z += v.z; r.w += v.w;
                    q.x += u.x; q.y += u.y; q.z += u.z; q.w += u.w;
                }
                *reinterpret_cast<float4 *>(srho + 4 * x4) = r;
                if (two) *reinterpret_cast<float4 *>(srho + 4 * x4b) = q;
            }
            if (A.wfun != nullptr)
                for (int i = tid; i < N + A.KR - 1; i += GR_THREADS) sw[i] = (r0 + i < 2 * N - 1) ? __ldg(A.wfun + r0 + i) : 0.0f;
            if (CLAMP && A.wfun != nullptr) {
                // window of the transposed wake: sw2[i] = w at index N - r0 - KR + i, so that
                // w[x' - x] = sw2[x' + KR - 1 - (x - r0)]
                const int base2 = N - r0 - A.KR;
                for (int i = tid; i < N + A.KR - 1; i += GR_THREADS) {
                    const int k = base2 + i;
                    sw2[i] = (k >= 0 && k < 2 * N - 1) ? __ldg(A.wfun + k) : 0.0f;
                }
            }
            __syncthreads();
            VFPS_STAMP(A.dbg, step, 3);
            // a3: V_x = sum_x' w[x - x'] rho_x' (Eq. 4), one row per warp at a time
            for (int r = warp; r < r1 - r0; r += GR_WARPS) {
                float v0 = 0.0f, v1 = 0.0f;
                if (A.wfun != nullptr) {
                    const float *wx = sw + (r + N - 1);
                    int xp = lane;
                    for (; xp + 32 < N; xp += 64) {
                        v0 = fmaf(wx[-xp], srho[xp], v0);
                        v1 = fmaf(wx[-(xp + 32)], srho[xp + 32], v1);
                    }
                    if (xp < N) v0 = fmaf(wx[-xp], srho[xp], v0);
                }
                const float v = warp_sum(v0 + v1);
                if constexpr (CLAMP) {
                    // The clamped kick is not conservative: CSR power of the END-of-step profile rho' to first
                    // order in rho' - rho: sum rho' V' = sum rho V + sum (rho' - rho)(V + Vt), Vt the transposed
                    // wake.  Row term -rho_x Vt_x here; the kick adds its row sums times dp (V + Vt).
                    float u0 = 0.0f, u1 = 0.0f;
                    if (A.wfun != nullptr) {
                        const float *ux = sw2 + (A.KR - 1 - r);
                        int xp = lane;
                        for (; xp + 32 < N; xp += 64) {
                            u0 = fmaf(ux[xp], srho[xp], u0);
                            u1 = fmaf(ux[xp + 32], srho[xp + 32], u1);
                        }
                        if (xp < N) u0 = fmaf(ux[xp], srho[xp], u0);
                    }
                    const float vt = warp_sum(u0 + u1);
                    if (lane == 0) { sV[r] = v; sU[r] = G.dp * (v + vt); acc[5] = fmaf(-srho[r0 + r], vt, acc[5]); }
                } else {
                    if (lane == 0) { sV[r] = v; acc[5] = fmaf(srho[r0 + r], v, acc[5]); }
                }
            }
            __syncthreads();
            VFPS_STAMP(A.dbg, step, 4);
            if constexpr (MANH) {
                // Manhattan: RF kick, wake kick (two 1-D interpolations along p), Fokker-Planck
                const int total = (r1 - r0) * NQ;
                for (int idx = tid; idx < total; idx += GR_THREADS) {
                    const int rr = idx >> lgNQ, x = r0 + rr, g = (idx & (NQ - 1)) << 2;
                    const float *row = A.psi_tmp + (size_t)x * N;
                    const float4 z4 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                    float4 v[5];
#pragma unroll
                    for (int q = 0; q < 5; ++q) {
                        const int c = g - 8 + 4 * q;
                        v[q] = (c >= 0 && c < N) ? *reinterpret_cast<const float4 *>(row + c) : z4;
                    }
                    int mm1, mm2;
                    float t1, t2;
                    floor_frac(G.mh_p * ((float)x + G.x0c), mm1, t1);
                    floor_frac(G.kick_c * sV[rr], mm2, t2);
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
                    *reinterpret_cast<float4 *>(A.psi + (size_t)x * N + g) = make_float4(o[0], o[1], o[2], o[3]);
                    float rs = 0.0f;
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        const float yy = (float)(g + c) - yc, tt = o[c] * yy;
                        rs += o[c]; acc[1] += tt; acc[2] = fmaf(tt, yy, acc[2]);
                    }
                    const float xx = (float)x - yc, tq = rs * xx;
                    acc[0] += rs; acc[3] += tq; acc[4] = fmaf(tq, xx, acc[4]);
                    if (CLAMP) acc[5] = fmaf(rs, sU[rr], acc[5]);
                }
            } else {
            // a4 + a5: four cells per thread in registers; four granules per pass, loads first
            const int total = (r1 - r0) * NQ;
            for (int idx0 = tid; idx0 < total; idx0 += 4 * GR_THREADS) {
                float4 v0[4], v1[4], v2[4];
                const float4 z4 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int idx = idx0 + u * GR_THREADS;
                    v0[u] = v1[u] = v2[u] = z4;
                    if (idx < total) {
                        const int x = r0 + (idx >> lgNQ), g = (idx & (NQ - 1)) << 2;
                        const float4 *row = reinterpret_cast<const float4 *>(A.psi_tmp + (size_t)x * N + g);
                        if (g >= 4) v0[u] = row[-1];
                        v1[u] = row[0];
                        if (g + 4 < N) v2[u] = row[1];
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int idx = idx0 + u * GR_THREADS;
                    if (idx < total) {
                        const int rr = idx >> lgNQ, x = r0 + rr, g = (idx & (NQ - 1)) << 2;
                        int mm;
                        float t;
                        floor_frac(G.kick_c * sV[rr], mm, t);
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
                            kick_fp_granule_any<ORDER, CLAMP>(A.psi_tmp + (size_t)x * N, l, mm, g, N, G.fp_b, c2, c1p, o);
                        }
                        *reinterpret_cast<float4 *>(A.psi + (size_t)x * N + g) = make_float4(o[0], o[1], o[2], o[3]);
                        float rs = 0.0f;
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            const float yy = (float)(g + c) - yc, tt = o[c] * yy;
                            rs += o[c]; acc[1] += tt; acc[2] = fmaf(tt, yy, acc[2]);
                        }
                        const float xx = (float)x - yc, tq = rs * xx;
                        acc[0] += rs; acc[3] += tq; acc[4] = fmaf(tq, xx, acc[4]);
                        if (CLAMP) acc[5] = fmaf(rs, sU[rr], acc[5]);
                    }
                }
            }
            }
        }
        {
            const float tot = warp_reduce8(acc, lane);
            if ((lane & 3) == 0) red[((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1)][warp] = tot;
        }
        __syncthreads();
        if (tid < GR_NPART) {
            float s = 0.0f;
#pragma unroll
            for (int w = 0; w < GR_WARPS; ++w) s += red[tid][w];
            A.mom_part[(size_t)tid * gridDim.x + blockIdx.x] = s;
            // the charge also goes into one 64-bit fixed-point accumulator: after the barrier every CTA
            // needs just one load for 1/C (re-reading gridDim.x partials from every CTA at once cost
            // 3-4 k cycles per step); integer addition is associative, so the sum is deterministic
            if (tid == 0) atomicAdd(A.qacc + (step & 1), (unsigned long long)__float2ll_rn(s * 4294967296.0f));
        }
        VFPS_STAMP(A.dbg, step, 5);
        grid.sync();
        VFPS_STAMP(A.dbg, step, 6);
        // ================= phase 3: a6 -- every CTA forms C and 1/C in the same fixed order
        // Every CTA needs only the charge: one load of the fixed-point accumulator.  Warps 1-5 of
        // CTA 0 sum the other partials for the diagnostics row (fp32, fixed order).
        __shared__ float s_tot[6];
        if (tid == 0) {
            const long long q = (long long)__ldcg(A.qacc + (step & 1));
            const float f = (float)((double)q * (1.0 / 4294967296.0));
            s_tot[0] = f;
            s_sc = G.renorm ? 1.0f / ((G.dq * G.dp) * f) : 1.0f;
            if (blockIdx.x == 0) A.qacc[(step + 1) & 1] = 0ull;      // nobody touches it before the next barrier
        }
        if (blockIdx.x == 0 && warp >= 1 && warp < 6) {              // the other sums, for the diagnostics row
            const float *mp = A.mom_part + (size_t)warp * gridDim.x;
            float f = 0.0f;
#pragma unroll 8
            for (int i = lane; i < (int)gridDim.x; i += 32) f += __ldcg(mp + i);
            f = warp_sum(f);
            if (lane == 0) s_tot[warp] = f;
        }
        __syncthreads();
        if (blockIdx.x == 0 && tid == 0 && A.diag != nullptr) {
            // (fp32, as in the cluster engine: fp64 divisions and square roots would hold CTA 0 back)
            const float t0 = s_tot[0], i0 = 1.0f / t0;
            const float C = (G.dq * G.dp) * t0;
            const float mp_c = s_tot[1] * i0, vp = fmaf(-mp_c, mp_c, s_tot[2] * i0);
            const float mq_c = s_tot[3] * i0, vq = fmaf(-mq_c, mq_c, s_tot[4] * i0);
            const float cc = G.renorm ? C : 1.0f;
            float *o = A.diag + (size_t)step * 6;
            o[0] = C;
            o[1] = fmaf(mq_c + yc, G.dq, G.q_min);
            o[2] = fmaf(mp_c + yc, G.dp, G.p_min);
            o[3] = sqrtf(fmaxf(vq, 0.0f)) * G.dq;
            o[4] = sqrtf(fmaxf(vp, 0.0f)) * G.dp;
            o[5] = s_tot[5] * G.dq / (cc * cc);
        }
        sc = s_sc;
        VFPS_STAMP(A.dbg, step, 7);
    }
    if (blockIdx.x == 0 && tid == 0) A.scale[0] = sc;
}

}  // namespace vfps
