// vfps_grid2.cuh -- persistent cooperative engine for one large grid (2048^2), TMA-staged (sm_100a).
//
// The first grid engine (vfps_grid.cuh) gathers every rotation tap through L1 with per-thread
// address arithmetic and three edge paths, and kicks straight from global memory: 147
// thread-instructions per cell, 29 us per step at 2048^2.  This engine gives the large grid what the
// in-place cluster kernel (vfps_onchip.cuh) gives the on-chip ones:
//  * One CTA of 512 threads per SM owns a stripe of about N / gridDim rows for the whole launch (stripe
//    boundaries where floor(dy) changes from one row to the next: a stripe's rotation is one run).
//  * Rotation a1 + a2: the source region of a tile -- the stripe's rows plus H halo rows, 256
//    columns plus 8 each side -- comes in through TMA (cp.async.bulk.tensor.2d over a tensor map of
//    8-byte elements, so that one box holds the 272 floats of a tile row; completion on an
//    mbarrier).  psi is zero outside the grid (reading A8), and so is TMA's fill for the part of a
//    box that lies outside the tensor: no edge path exists.  A group of four warps rotates a tile
//    with the cluster kernel's walker: two columns per thread, ORDER x 6 register window,
//    per-launch weight tables (rows: L, L' in shared memory; columns: the fractional source
//    position at the stripe's centre row, rounded once from double, fetched a tile ahead), next
//    row's loads issued mid-row.  Two tile buffers per group where they fit (the tile after next is
//    in flight while a tile is rotated), else one.  The rotated cells stay in
//    shared memory (the stripe's rows: no psi_tmp round trip through L2), row sums (transposed warp
//    reduction) go to the profile.
//  -- grid barrier --
//  * Wake a3 for the stripe's rows (one warp per row, direct convolution, Eq. 4).
//  * Kick a4 + Fokker-Planck a5 + moments a6 from shared memory: a warp takes a (row, 256-column
//    block), a lane the 4-cell granules 4 lane + 128 k -- 128-bit loads with a lane stride of 16
//    bytes -- and writes psi with 128-bit stores.
//  ONE grid barrier per step: between a kick and the next rotation a CTA only needs the stripes above
//  and below (their halo rows), so it waits for those two CTAs' flags; the charge of a step (exact
//  32.32 fixed-point sum) and the partial sums for its diagnostics row are complete at the next
//  step's barrier, which is where 1/C is needed next.
// Template CLAMP: clamped interpolation (Eq. 14, reading A9); the CSR power is then that of the
// end-of-step profile to first order in its change (transposed wake, see k_wake_direct).
// Standard rotation only; one simulation per handle; N a multiple of 256.
#pragma once
#include "vfps_onchip.cuh"

#include <cooperative_groups.h>
#include <cuda.h>

namespace vfps {

constexpr int G2_THREADS = 512;
constexpr int G2_WARPS = G2_THREADS / 32;
constexpr int G2_GROUPS = 4;          // warp groups of four, one tile each at a time
constexpr int G2_SUBW = 272;          // floats per row of a tile: 256 columns + 8 each side (one TMA box of 136 8-byte elements)
constexpr int G2_PADC = 8;
constexpr int G2_NPART = 8;
constexpr int G2_MAX_H = 4;

struct Grid2Args {
    float *psi;            // [N][N] in/out, un-normalised (the tensor map of the kernel points at it)
    float *scale;          // [1] in/out: 1/C of the last step
    const float *wfun;     // [2N] wake function, lag d at index d + N - 1; nullptr = no wake
    float *rho;            // [N] profile of the step (dp * row sums, un-scaled)
    float *mom_part;       // [2][G2_NPART][gridDim.x], by step parity
    float *diag;           // [nsteps][1][6] or nullptr
    const float *coltab;   // [gridDim.x][N]: fractional source position along q of column y at the centre row of stripe c
    const int *colix;      // [gridDim.x][N]: floor(dx) of column y over the rows of stripe c, or OC_BAD
    const float *rowtab;   // [N][12]: as in the cluster kernel (a (X - Xc) relative to the stripe's centre row)
    unsigned long long *qacc;   // [3] charge of step t in slot t % 3, 32.32 fixed point, zero at launch
    unsigned int *bar;          // grid barrier counter, zero at launch
    unsigned int *flags;        // [gridDim.x][32] (one 128-byte line each): kicks finished by the CTA in this launch, zero at launch
    int nsteps;
    const int *row0;            // [gridDim.x + 1] first row of every stripe (stripe c: rows row0[c] .. row0[c + 1] - 1)
    int KRmax;                  // rows of the largest stripe
    int nbuf;                   // tile buffers per warp group: 2, or 1 where two do not fit beside the stripe's rows
    long long *dbg;
};

struct Grid2Layout {
    int box_rows, pitch, nct;
    size_t tile_floats, off_mbar, off_rowtab, off_rowpart, off_vtab, off_rho, off_sw, off_sw2, off_vpart, off_red, off_runend, off_rows, off_big,
        total_floats;
};

__host__ __device__ inline Grid2Layout grid2_layout(int N, int KRmax, int H, int nbuf, bool clamp)
{
    Grid2Layout L;
    L.box_rows = (KRmax + 2 * H + 1) & ~1;          // even: a tile of 272 floats x rows is then a multiple of 128 bytes (TMA)
    L.pitch = N + 2 * G2_PADC;
    L.nct = N / 256;
    L.tile_floats = (size_t)L.box_rows * G2_SUBW;
    size_t o = 0;
    L.off_mbar = o;     o += 32;                                // 2 x G2_GROUPS mbarriers
    L.off_rowtab = o;   o += (size_t)(KRmax + 2) * OC_ROWTAB;
    L.off_rowpart = o;  o += (size_t)KRmax * (N / 64);
    L.off_vtab = o;     o += (size_t)((KRmax * 8 + 3) & ~3);
    L.off_rho = o;      o += (size_t)N;
    const int KP = (KRmax + 3) & ~3;
    L.off_sw = o;       o += (size_t)(N + KP + 4);                // lags of the wake function the stripe's rows touch
    L.off_sw2 = o;      o += clamp ? (size_t)(N + KP + 4) : 0;    // ... and of the transposed wake
    L.off_vpart = o;    o += (size_t)8 * KP;                      // wake partial sums [4 quarters (+ 4 transposed)][KP rows]
    L.off_red = o;      o += (size_t)G2_WARPS * 8 + 8;
    L.off_runend = o;   o += (size_t)((KRmax + 3) & ~3);         // per row: end of its run of constant floor(dy)
    L.off_rows = o;     o += (size_t)KRmax * L.pitch;           // the stripe's rotated rows
    o = (o + 31) & ~(size_t)31;                                 // TMA destinations: 128-byte aligned
    L.off_big = o;      o += (size_t)nbuf * G2_GROUPS * L.tile_floats + G2_SUBW;   // + one row: the walker prefetches past the end
    L.total_floats = o;
    return L;
}

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, int c0, int c1, uint32_t mbar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
                 ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(mbar), "r"(c0), "r"(c1)
                 : "memory");
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}

// Grid barrier on one monotonic counter (zero at launch; the launch is cooperative, so every CTA is
// resident): arrival = one atomic, release = the counter reaching gen * gridDim.x.  About half the cost
// of cooperative_groups' grid.sync() here.
__device__ __forceinline__ void grid_barrier(unsigned int *ctr, unsigned int &gen)
{
    __syncthreads();
    ++gen;
    if (threadIdx.x == 0) {
        const unsigned int target = gen * gridDim.x;
        // release: the CTA's global stores before the __syncthreads above are ordered before the arrival;
        // acquire: the poll that sees the last arrival orders every CTA's stores before what follows the
        // __syncthreads below (no further fence needed: the readers use L1-bypassing loads)
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(ctr) : "memory");
        unsigned int seen;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(ctr) : "memory");
        } while ((int)(seen - target) < 0);
    }
    __syncthreads();
}

// d l_k / dt of the Lagrange weights (Eq. 13); multiplies a (X - Xc) ~ 1e-6 in the row-wise first-order correction
template <int ORDER>
__device__ __forceinline__ void lagrange_deriv(float t, float (&lp)[ORDER])
{
    if (ORDER == 2) {
        lp[0] = -1.0f; lp[1] = 1.0f;
    } else if (ORDER == 3) {
        lp[0] = t - 0.5f; lp[1] = -2.0f * t; lp[ORDER - 1] = t + 0.5f;
    } else {
        const float t2 = 3.0f * t * t;
        lp[0] = -(t2 - 6.0f * t + 2.0f) * (1.0f / 6.0f);
        lp[1] = (t2 - 4.0f * t - 1.0f) * 0.5f;
        lp[ORDER - 2] = -(t2 - 2.0f * t - 2.0f) * 0.5f;
        lp[ORDER - 1] = (t2 - 1.0f) * (1.0f / 6.0f);
    }
}

// one cell of a tile with its own floors (a floor changes inside the warp's columns or the chunk)
template <int ORDER, bool CLAMP>
__device__ __forceinline__ float rotate_cell_tile(const GridConst &G, uint32_t base00 /* tile address of source (row x, column y) */,
                                                  int x, int y)
{
    constexpr int O0 = (ORDER - 1) / 2;
    constexpr int P = G2_SUBW;
    const float X = (float)x + G.x0c, Y = (float)y + G.y0c;
    int ix, iy;
    float tx, ty;
    floor_frac(fmaf(G.a, X, G.b * Y), ix, tx);
    floor_frac(fmaf(G.d, X, G.a * Y), iy, ty);
    float lx[ORDER], ly[ORDER];
    lagrange<ORDER>(tx, lx);
    lagrange<ORDER>(ty, ly);
    const uint32_t base = base00 + (uint32_t)(((ix - O0) * P + (iy - O0)) * 4);
    float acc = 0.0f;
#pragma unroll
    for (int i = 0; i < ORDER; ++i) {
        float r = ly[0] * lds(base + (i * P) * 4);
#pragma unroll
        for (int j = 1; j < ORDER; ++j) r = fmaf(ly[j], lds(base + (i * P + j) * 4), r);
        acc = (i == 0) ? lx[0] * r : fmaf(lx[i], r, acc);
    }
    if (CLAMP) {
        const float a = lds(base + (O0 * P + O0) * 4), b = lds(base + (O0 * P + O0 + 1) * 4);
        const float c = lds(base + ((O0 + 1) * P + O0) * 4), d = lds(base + ((O0 + 1) * P + O0 + 1) * 4);
        acc = fminf(fmaxf(acc, fminf(fminf(a, b), fminf(c, d))), fmaxf(fmaxf(a, b), fmaxf(c, d)));
    }
    return acc;
}

template <int ORDER, bool CLAMP>
__global__ void __launch_bounds__(G2_THREADS, 1)
k_grid2_step(GridConst G, Grid2Args A, const __grid_constant__ CUtensorMap tmap)
{
    namespace cg = cooperative_groups;
    constexpr int O0 = (ORDER - 1) / 2;
    constexpr int CH = oc_chunk_rows(ORDER);
    constexpr int P4 = G2_SUBW * 4;
    constexpr unsigned FULL = 0xffffffffu;
    using Wk = Walker<ORDER, G2_SUBW, true, CLAMP>;

    const int N = G.N, H = G.H, KRmax = A.KRmax;
    const int nbuf = A.nbuf;
    const Grid2Layout LY = grid2_layout(N, KRmax, H, nbuf, CLAMP);
    const int nct = LY.nct, CWR = N / 64;                  // column tiles; row-sum partials per row
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int grp = warp >> 2, cw = warp & 3;
    const int c = (int)blockIdx.x;
    const int r0 = A.row0[c], rows = A.row0[c + 1] - r0;

    extern __shared__ __align__(128) float g2smem[];
    float *smem = g2smem;
    float *rowtab_s = smem + LY.off_rowtab + OC_ROWTAB;
    float *rowpart = smem + LY.off_rowpart;
    float *vtab = smem + LY.off_vtab;
    float *srho = smem + LY.off_rho, *sw = smem + LY.off_sw, *sw2 = smem + LY.off_sw2;
    float *red = smem + LY.off_red, *vpart = smem + LY.off_vpart;
    const int KP = (KRmax + 3) & ~3;
    const uint32_t sRho = smem_u32(srho), sSw = smem_u32(sw), sSw2 = smem_u32(sw2);
    float *big = smem + LY.off_big;
    float *rowsb = smem + LY.off_rows;               // [KRmax][PITCH]: the stripe's rotated rows, 8 zero floats each side
    const uint32_t sBig = smem_u32(big), sRows = smem_u32(rowsb), sRowtab = smem_u32(rowtab_s), sRowpart = smem_u32(rowpart), sVtab = smem_u32(vtab);
    const uint32_t sMbar = smem_u32(smem + LY.off_mbar);
    const uint32_t tile_bytes = (uint32_t)LY.tile_floats * 4u;
    const int PITCH = LY.pitch;

    // ---- one-time set-up
    for (int i = tid; i < (KRmax + 2) * OC_ROWTAB; i += G2_THREADS) {
        const int gi = (r0 - 1) * OC_ROWTAB + i;
        rowtab_s[i - OC_ROWTAB] = (gi >= 0 && gi < N * OC_ROWTAB) ? A.rowtab[gi] : 0.0f;
    }
    __syncthreads();
    // runs of consecutive rows with the same floor(dy) (the window slides through a run): end of the run of every row
    int *runend = reinterpret_cast<int *>(smem + LY.off_runend);
    if (tid < rows) {
        const int iy = __float_as_int(rowtab_s[tid * OC_ROWTAB + 10]);
        int ve = tid + 1;
        while (iy != OC_BAD && ve < rows && __float_as_int(rowtab_s[ve * OC_ROWTAB + 10]) == iy) ++ve;
        runend[tid] = ve;
    }
    if (A.wfun != nullptr) {
        // the lags this stripe's rows touch: sw[i] = w at index r0 + i (V_x = sum_x' sw[x - r0 + N - 1 - x'] rho_x');
        // CLAMP: sw2[i] = w at index N - r0 - KP + i (transposed wake: w[x' - x] = sw2[x' + KP - 1 - (x - r0)])
        for (int i = tid; i < N + KP + 4; i += G2_THREADS) sw[i] = (r0 + i < 2 * N - 1) ? __ldg(A.wfun + r0 + i) : 0.0f;
        if (CLAMP) {
            const int base2 = N - r0 - KP;
            for (int i = tid; i < N + KP + 4; i += G2_THREADS) {
                const int k = base2 + i;
                sw2[i] = (k >= 0 && k < 2 * N - 1) ? __ldg(A.wfun + k) : 0.0f;
            }
        }
    }
    for (int i = tid; i < KRmax * PITCH; i += G2_THREADS) rowsb[i] = 0.0f;       // the pads stay zero for ever
    if (tid == 0) {
        for (int i = 0; i < 2 * G2_GROUPS; ++i) mbar_init(sMbar + 8u * (uint32_t)i, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const float yc = 0.5f * (float)(N - 1);
    const float c1 = G.fp_b / (6.0f * G.dp), c2 = G.fp_b / (G.dp * G.dp);
    float sc = G.renorm ? A.scale[0] : 1.0f;
    // column data of the group's NEXT tile (cyclic: after the last tile of a step comes the first of the next):
    // two 64-bit loads, issued a whole tile ahead of their use (L2 latency off the tile-to-tile path)
    float2 tnx = make_float2(0.0f, 0.0f);
    int2 inx = make_int2(OC_BAD, OC_BAD);
#define G2_COL_FETCH(ct_)                                                                              \
    do {                                                                                                \
        const size_t o_ = (size_t)c * N + 256 * (ct_) + 64 * cw + 2 * lane;                             \
        tnx = __ldg(reinterpret_cast<const float2 *>(A.coltab + o_));                                   \
        inx = __ldg(reinterpret_cast<const int2 *>(A.colix + o_));                                      \
    } while (0)
    if (grp < nct) G2_COL_FETCH(grp);
    unsigned int bar_gen = 0u;
    unsigned use0 = 0u, use1 = 0u;             // how often this group has waited on its buffer 0 / 1
    const uint32_t mb0 = sMbar + 16u * (uint32_t)grp, mb1 = mb0 + 8u;
    const uint32_t buf0 = sBig + (uint32_t)(nbuf * grp) * tile_bytes, buf1 = buf0 + tile_bytes;     // buf1 only if nbuf == 2
    const bool rs_writer = ((lane & 7) == 0) && ((lane >> 3) < CH);
    const bool issuer = (cw == 0 && lane == 0);
    __shared__ float s_tot[6];
    __shared__ float s_sc;

    // The first tiles of a group's rotation.  psi was written with ordinary stores and TMA reads it
    // through the async proxy: proxy fence first.
#define G2_ISSUE_FIRST()                                                                                \
    do {                                                                                                \
        if (issuer) {                                                                                   \
            asm volatile("fence.proxy.async;" ::: "memory");                                            \
            for (int b_ = 0; b_ < nbuf; ++b_) {                                                         \
                const int ct_ = grp + G2_GROUPS * b_;                                                   \
                if (ct_ < nct) {                                                                        \
                    const uint32_t mb_ = b_ ? mb1 : mb0, dst_ = b_ ? buf1 : buf0;                       \
                    mbar_expect_tx(mb_, tile_bytes);                                                    \
                    tma_load_2d(dst_, &tmap, (256 * ct_ - G2_PADC) / 2, r0 - H, mb_);                   \
                }                                                                                       \
            }                                                                                           \
        }                                                                                               \
    } while (0)

    // diagnostics row of step T from the CTA partial sums (fp32, fixed order), by the last CTA
#define G2_DIAG(T)                                                                                      \
    do {                                                                                                \
        if (blockIdx.x == gridDim.x - 1 && A.diag != nullptr) {                                         \
            if (warp < 6) {                                                                             \
                const float *mp_ = A.mom_part + ((size_t)((T) & 1) * G2_NPART + warp) * gridDim.x;      \
                float f_ = 0.0f;                                                                        \
                for (int i_ = lane; i_ < (int)gridDim.x; i_ += 32) f_ += __ldcg(mp_ + i_);              \
                f_ = warp_sum(f_);                                                                      \
                if (lane == 0) s_tot[warp] = f_;                                                        \
            }                                                                                           \
            __syncthreads();                                                                            \
            if (tid == 0) {                                                                             \
                const float t0_ = s_tot[0], i0_ = 1.0f / t0_;                                           \
                const float C_ = (G.dq * G.dp) * t0_;                                                   \
                const float mp_c_ = s_tot[1] * i0_, vp_ = fmaf(-mp_c_, mp_c_, s_tot[2] * i0_);          \
                const float mq_c_ = s_tot[3] * i0_, vq_ = fmaf(-mq_c_, mq_c_, s_tot[4] * i0_);          \
                const float cc_ = G.renorm ? C_ : 1.0f;                                                 \
                float *o_ = A.diag + (size_t)(T) * 6;                                                   \
                o_[0] = C_;                                                                             \
                o_[1] = fmaf(mq_c_ + yc, G.dq, G.q_min);                                                \
                o_[2] = fmaf(mp_c_ + yc, G.dp, G.p_min);                                                \
                o_[3] = sqrtf(fmaxf(vq_, 0.0f)) * G.dq;                                                 \
                o_[4] = sqrtf(fmaxf(vp_, 0.0f)) * G.dp;                                                 \
                o_[5] = s_tot[5] * G.dq / (cc_ * cc_);                                                  \
            }                                                                                           \
            __syncthreads();                                                                            \
        }                                                                                               \
    } while (0)

    for (int step = 0; step < A.nsteps; ++step) {
        VFPS_STAMP(A.dbg, step, 0);
        // ================= phase 1: rotation psi -> the stripe's rows in shared memory, row sums.  Group grp: column tiles grp, grp + 4, ...
        if (step > 0) {
            // The halo rows of this step's tiles belong to the stripes above and below: those two CTAs must
            // have finished the kick of step - 1 (no grid barrier between a kick and the next rotation).  One
            // poller per flag, one 128-byte line per flag: hundreds of pollers on a few lines starve the writers.
            if (tid < 2) {                                  // the two flags in flight together: one L2 round trip, not two
                const int nb = c - 1 + 2 * tid;
                if (nb >= 0 && nb < (int)gridDim.x) {
                    unsigned int seen;
                    for (;;) {
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(A.flags + 32 * nb) : "memory");
                        if ((int)(seen - (unsigned int)step) >= 0) break;
                        __nanosleep(64);
                    }
                }
            }
            __syncthreads();
        }
        if (rows > 0) {
            G2_ISSUE_FIRST();
            int it = 0;
            for (int ct = grp; ct < nct; ct += G2_GROUPS, ++it) {
                const int b = (nbuf == 2) ? (it & 1) : 0;
                const uint32_t mb = b ? mb1 : mb0, tile = b ? buf1 : buf0;
                // this tile's columns: y0, y0 + 1; weights along q from the stripe's table
                const int y0 = 256 * ct + 64 * cw + 2 * lane;
                Wk wkr;
                int ixc;
                bool cols_ok;
                {
                    // weights along q at the stripe's centre row and their t-derivatives (Eq. 13) from the
                    // fractional positions the host rounded once from double
                    const int i0 = inx.x, i1 = inx.y;
                    const float t0 = tnx.x, t1 = tnx.y;
                    G2_COL_FETCH(ct + G2_GROUPS < nct ? ct + G2_GROUPS : grp);
                    ixc = i0;
                    cols_ok = __all_sync(FULL, i0 != OC_BAD && i0 == i1);
                    lagrange<ORDER>(t0, wkr.M0); lagrange_deriv<ORDER>(t0, wkr.M0p);
                    lagrange<ORDER>(t1, wkr.M1); lagrange_deriv<ORDER>(t1, wkr.M1p);
                    wkr.ey0 = G.a * ((float)y0 - yc);
                    wkr.ey1 = G.a * ((float)(y0 + 1) - yc);
                    wkr.a = G.a;
                    if (!cols_ok) ixc = 0;
                }
                mbar_wait(mb, (b ? use1 : use0) & 1u);
                if (b) ++use1; else ++use0;
                // local column of y0 inside the tile; the rotated cells go to the stripe's rows in shared memory
                const uint32_t box = tile;
                const int yl = G2_PADC + 64 * cw + 2 * lane;
                const uint32_t sout = sRows + (uint32_t)((G2_PADC + y0) * 4), RP4 = (uint32_t)PITCH * 4u;
                // runs of consecutive rows with the same floor(dy): the window slides through a run; a floor
                // changes at most once in a stripe (at the row through the rotation centre)
                int v = 0;
                while (v < rows) {
                    const int iy = __float_as_int(rowtab_s[v * OC_ROWTAB + 10]);
                    if (cols_ok && iy != OC_BAD) {
                        const int ve = runend[v];
                        const int par = (iy - O0) & 1;
                        // tile row of source row x is x - (r0 - H); tap row 0 of target v: v + ixc - O0
                        uint32_t src = box + (uint32_t)((v + H + ixc - O0) * P4 + (yl + iy - O0 - par) * 4);
                        OutSharedRt dst{sout + (uint32_t)v * RP4, RP4};
                        uint32_t tab = sRowtab + (uint32_t)(v * OC_ROWTAB * 4);
                        uint32_t rp = sRowpart + (uint32_t)(((v + (lane >> 3)) * CWR + 4 * ct + cw) * 4);
#define G2_RUN(PAR_)                                                                                   \
    do {                                                                                                \
        wkr.template start<PAR_>(src, tab);                                                             \
        for (int vv = v; vv < ve; vv += CH) {                                                           \
            const int left = ve - vv;                                                                   \
            if (left >= CH) wkr.template chunk<PAR_, 1>(src, dst, tab);                                 \
            else wkr.template chunk_n<PAR_, 1>(src, dst, tab, left);                                    \
            if (CH < 4) wkr.rs[3] = 0.0f;                                                               \
            const float tot = warp_reduce_transposed<4>(wkr.rs, lane);                                  \
            if (rs_writer && (lane >> 3) < left) sts(rp, tot);                                          \
            src += (uint32_t)(CH * P4); dst.a += (uint32_t)CH * RP4;                                    \
            tab += (uint32_t)(CH * OC_ROWTAB * 4); rp += (uint32_t)(CH * CWR * 4);                      \
        }                                                                                               \
    } while (0)
                        if (par) G2_RUN(1); else G2_RUN(0);
#undef G2_RUN
                        v = ve;
                    } else {
                        // one row, cell by cell: floor(dx) changes inside the warp's columns, or floor(dy) along the row
                        const uint32_t b00 = box + (uint32_t)(((v + H) * G2_SUBW + yl) * 4);
                        const float o0 = rotate_cell_tile<ORDER, CLAMP>(G, b00, r0 + v, y0);
                        const float o1 = rotate_cell_tile<ORDER, CLAMP>(G, b00 + 4u, r0 + v, y0 + 1);
                        sts2(sout + (uint32_t)v * RP4, o0, o1);
                        const float tot = warp_sum(o0 + o1);
                        if (lane == 0) rowpart[v * CWR + 4 * ct + cw] = tot;
                        ++v;
                    }
                }
                // the whole group has finished reading this buffer: refill it with the tile after next
                named_barrier(1 + grp, 128);
                const int ct2 = ct + nbuf * G2_GROUPS;
                if (issuer && ct2 < nct) {
                    mbar_expect_tx(mb, tile_bytes);
                    tma_load_2d(tile, &tmap, (256 * ct2 - G2_PADC) / 2, r0 - H, mb);
                }
            }
        }
        VFPS_STAMP(A.dbg, step, 1);
        __syncthreads();
        for (int r = warp; r < rows; r += G2_WARPS) {          // CWR <= 64 partials per row
            float s = (lane < CWR) ? rowpart[r * CWR + lane] : 0.0f;
            if (lane + 32 < CWR) s += rowpart[r * CWR + lane + 32];
            s = warp_sum(s);
            if (lane == 0) A.rho[r0 + r] = s * G.dp;
        }
        grid_barrier(A.bar, bar_gen);
        VFPS_STAMP(A.dbg, step, 2);
        // ================= phase 2: wake of the stripe's rows while its rotated rows stream into shared memory
        float acc[8] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f};   // s0 s1 s2 q1 q2 pw - -
        if (rows > 0) {
            for (int i = tid; i < N; i += G2_THREADS) srho[i] = __ldcg(A.rho + i);
            if (tid == 0 && step > 0) {
                // charge of the previous step: every CTA has added its share before it arrived at this step's barrier
                const long long q = (long long)__ldcg(A.qacc + (step - 1) % 3);
                const float f = (float)((double)q * (1.0 / 4294967296.0));
                s_sc = G.renorm ? 1.0f / ((G.dq * G.dp) * f) : 1.0f;
                if (blockIdx.x == 0) A.qacc[(step + 1) % 3] = 0ull;      // slot of step - 2: read by everybody before this barrier
            }
            __syncthreads();
            if (step > 0) sc = s_sc;
            VFPS_STAMP(A.dbg, step, 3);
            // a3: V_x = sum_x' w[x - x'] rho_x' (Eq. 4).  Warp (q, s) = (warp & 3, warp >> 2): the four rows
            // 4q .. 4q + 3 of the stripe against the quarter s of the profile, 128-bit loads of the wake
            // function as in the cluster kernel (index A + k - c, A = 3 mod 4); partial sums -> vpart
            {
                const int SL = N >> 2, xs = SL * (warp >> 2);
                for (int q = warp & 3; 4 * q < rows; q += 4) {
                    float vq[4] = {0.0f, 0.0f, 0.0f, 0.0f}, vt[4] = {0.0f, 0.0f, 0.0f, 0.0f};
                    if (A.wfun != nullptr) {
                        for (int xl = 4 * lane; xl < SL; xl += 128) {
                            const int xp = xs + xl;
                            const float4 r4 = lds4(sRho + (uint32_t)xp * 4u);
                            const float rc[4] = {r4.x, r4.y, r4.z, r4.w};
                            {
                                const int Aq = 4 * q - xp + N - 1;             // sw[i] = w at index r0 + i
                                const float4 wl = lds4(sSw + (uint32_t)(Aq - 3) * 4u), wh = lds4(sSw + (uint32_t)(Aq + 1) * 4u);
                                const float w7[8] = {wl.x, wl.y, wl.z, wl.w, wh.x, wh.y, wh.z, wh.w};
#pragma unroll
                                for (int k = 0; k < 4; ++k)
#pragma unroll
                                    for (int cc = 0; cc < 4; ++cc) vq[k] = fmaf(w7[3 + k - cc], rc[cc], vq[k]);
                            }
                            if (CLAMP) {
                                const int Bq = xp + KP - 1 - 4 * q;            // sw2[i] = w at index N - r0 - KP + i
                                const float4 ul = lds4(sSw2 + (uint32_t)(Bq - 3) * 4u), uh = lds4(sSw2 + (uint32_t)(Bq + 1) * 4u);
                                const float u7[8] = {ul.x, ul.y, ul.z, ul.w, uh.x, uh.y, uh.z, uh.w};
#pragma unroll
                                for (int k = 0; k < 4; ++k)
#pragma unroll
                                    for (int cc = 0; cc < 4; ++cc) vt[k] = fmaf(u7[3 + cc - k], rc[cc], vt[k]);
                            }
                        }
                    }
                    const float Vr = warp_reduce_transposed<4>(vq, lane);     // lanes 8k .. 8k + 7 hold row 4q + k
                    const float Vtr = CLAMP ? warp_reduce_transposed<4>(vt, lane) : 0.0f;
                    if ((lane & 7) == 0) {
                        vpart[(warp >> 2) * KP + 4 * q + (lane >> 3)] = Vr;
                        if (CLAMP) vpart[(4 + (warp >> 2)) * KP + 4 * q + (lane >> 3)] = Vtr;
                    }
                }
            }
            __syncthreads();
            if (tid < rows) {
                const int r = tid;
                const float Vr = (vpart[r] + vpart[KP + r]) + (vpart[2 * KP + r] + vpart[3 * KP + r]);
                const float V = Vr * sc, rho_x = srho[r0 + r] * sc;
                int mm;
                float t;
                floor_frac(G.kick_c * V, mm, t);
                float l[ORDER];
                lagrange<ORDER>(t, l);
                float pl[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
                for (int j = 0; j < ORDER; ++j) pl[j] = CLAMP ? l[j] : l[j] * sc;
                sts4(sVtab + (uint32_t)r * 32u, make_float4(pl[0], pl[1], pl[2], pl[3]));
                if (CLAMP) {
                    const float Vt = ((vpart[4 * KP + r] + vpart[5 * KP + r]) + (vpart[6 * KP + r] + vpart[7 * KP + r])) * sc;
                    sts4(sVtab + (uint32_t)r * 32u + 16u, make_float4(__int_as_float(mm), -rho_x * Vt, G.dp * (V + Vt), 0.0f));
                } else {
                    sts2(sVtab + (uint32_t)r * 32u + 16u, __int_as_float(mm), rho_x * V);
                }
            }
            __syncthreads();
            VFPS_STAMP(A.dbg, step, 4);
            // a4 + a5 + a6: a warp takes (row, 256-column block); a lane owns the granules 4 lane and 4 lane + 128 of the block
            // a warp keeps its column block: column sums serve the p-moments
            const int blk = warp % nct, rstride = G2_WARPS / nct;
            float cs[2][4] = {{0.0f, 0.0f, 0.0f, 0.0f}, {0.0f, 0.0f, 0.0f, 0.0f}};
            // ... and its Fokker-Planck coefficients (G-1, G0, G1, G2 of kick_fp4) stay in registers for the pass
            float4 gt[2][4];
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                float cm[4], c0[4], cp[4], c2p[4];
#pragma unroll
                for (int cc = 0; cc < 4; ++cc) {
                    const float c1p = c1 * fmaf((float)(256 * blk + 4 * lane + 128 * k + cc), G.dp, G.p_min);
                    cm[cc] = fmaf(-2.0f, c1p, c2);
                    c0[cc] = fmaf(-3.0f, c1p, fmaf(-2.0f, c2, G.fp_b));
                    cp[cc] = fmaf(6.0f, c1p, c2);
                    c2p[cc] = -c1p;
                }
                gt[k][0] = make_float4(cm[0], cm[1], cm[2], cm[3]);
                gt[k][1] = make_float4(c0[0], c0[1], c0[2], c0[3]);
                gt[k][2] = make_float4(cp[0], cp[1], cp[2], cp[3]);
                gt[k][3] = make_float4(c2p[0], c2p[1], c2p[2], c2p[3]);
            }
            for (int r = warp / nct; r < rows; r += rstride) {
                const float4 lw = lds4(sVtab + (uint32_t)r * 32u);
                float2 mv;
                float dpU = 0.0f;
                if (CLAMP) {
                    const float4 m4 = lds4(sVtab + (uint32_t)r * 32u + 16u);
                    mv = make_float2(m4.x, m4.y); dpU = m4.z;
                } else {
                    mv = lds2(sVtab + (uint32_t)r * 32u + 16u);
                }
                const int mm = __float_as_int(mv.x);
                const int g0 = 256 * blk + 4 * lane;
                const uint32_t own = sRows + (uint32_t)((r * PITCH + G2_PADC + g0) * 4);
                const float lws[4] = {lw.x, lw.y, lw.z, lw.w};
                float l[ORDER];
#pragma unroll
                for (int j = 0; j < ORDER; ++j) l[j] = lws[j];
                float o[2][4];
                if (mm >= -2 && mm <= 0) {
                    float b[2][12];
#pragma unroll
                    for (int k = 0; k < 2; ++k)
#pragma unroll
                        for (int i = 0; i < 3; ++i) {
                            const float4 v = lds4(own + (uint32_t)(512 * k + 16 * i - 16));
                            b[k][4 * i] = v.x; b[k][4 * i + 1] = v.y; b[k][4 * i + 2] = v.z; b[k][4 * i + 3] = v.w;
                        }
#pragma unroll
                    for (int k = 0; k < 2; ++k) {
                        const int g = g0 + 128 * k;
                        if (mm == 0) kick_fp4<ORDER, 0, CLAMP>(b[k], l, g, N, gt[k], o[k]);
                        else if (mm == -1) kick_fp4<ORDER, -1, CLAMP>(b[k], l, g, N, gt[k], o[k]);
                        else kick_fp4<ORDER, -2, CLAMP>(b[k], l, g, N, gt[k], o[k]);
                    }
                } else {
                    const float *rowp = rowsb + r * PITCH + G2_PADC;
#pragma unroll
                    for (int k = 0; k < 2; ++k) {
                        const int g = g0 + 128 * k;
                        float c1p[4];
#pragma unroll
                        for (int cc = 0; cc < 4; ++cc) c1p[cc] = c1 * fmaf((float)(g + cc), G.dp, G.p_min);
                        kick_fp_granule_any<ORDER, CLAMP>(rowp, l, mm, g, N, G.fp_b, c2, c1p, o[k]);
                    }
                }
                if (CLAMP) {
#pragma unroll
                    for (int k = 0; k < 2; ++k)
#pragma unroll
                        for (int cc = 0; cc < 4; ++cc) o[k][cc] *= sc;
                }
                float *orow = A.psi + (size_t)(r0 + r) * N + g0;
                float rs = 0.0f;
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    *reinterpret_cast<float4 *>(orow + 128 * k) = make_float4(o[k][0], o[k][1], o[k][2], o[k][3]);
#pragma unroll
                    for (int cc = 0; cc < 4; ++cc) { cs[k][cc] += o[k][cc]; rs += o[k][cc]; }
                }
                const float xx = (float)(r0 + r) - yc, tq = rs * xx;
                acc[3] += tq; acc[4] = fmaf(tq, xx, acc[4]);
                if (CLAMP) acc[5] = fmaf(rs, dpU, acc[5]);
                if (lane == 0 && blk == 0) acc[5] += mv.y;
            }
#pragma unroll
            for (int k = 0; k < 2; ++k)
#pragma unroll
                for (int cc = 0; cc < 4; ++cc) {
                    const float yy = (float)(256 * blk + 4 * lane + 128 * k + cc) - yc, tt = cs[k][cc] * yy;
                    acc[0] += cs[k][cc]; acc[1] += tt; acc[2] = fmaf(tt, yy, acc[2]);
                }
        }
        {
            const float tot = warp_reduce_transposed<8>(acc, lane);       // lanes 4 j .. 4 j + 3 hold sum j
            if ((lane & 3) == 0) red[warp * 8 + (lane >> 2)] = tot;
        }
        __syncthreads();
        if (tid < G2_NPART) {
            float s = 0.0f;
#pragma unroll
            for (int w = 0; w < G2_WARPS; ++w) s += red[w * 8 + tid];
            A.mom_part[((size_t)(step & 1) * G2_NPART + tid) * gridDim.x + blockIdx.x] = s;
            // charge: one 64-bit fixed-point accumulator (integer atomics: exact, order-independent)
            if (tid == 0) atomicAdd(A.qacc + step % 3, (unsigned long long)__float2ll_rn(s * 4294967296.0f));
        }
        // (psi of this step is read by the next rotations through TMA, i.e. the async proxy: the proxy fence sits on
        // the reader's side, in G2_ISSUE_FIRST, after the flags have been acquired)
        VFPS_STAMP(A.dbg, step, 5);
        __syncthreads();
        if (tid == 0)       // release: orders the CTA's psi stores (before the __syncthreads) before the flag
            asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(A.flags + 32 * c), "r"((unsigned int)(step + 1)) : "memory");
        // a6 of the previous step: the last CTA (the shortest stripe) writes its diagnostics row; the partial
        // sums of every CTA were complete at this step's barrier
        if (step > 0) G2_DIAG(step - 1);
        VFPS_STAMP(A.dbg, step, 7);
    }
    // ---- the last step's charge and diagnostics
    grid_barrier(A.bar, bar_gen);
    if (tid == 0) {
        const long long q = (long long)__ldcg(A.qacc + (A.nsteps - 1) % 3);
        const float f = (float)((double)q * (1.0 / 4294967296.0));
        if (blockIdx.x == 0) A.scale[0] = G.renorm ? 1.0f / ((G.dq * G.dp) * f) : 1.0f;
    }
    G2_DIAG(A.nsteps - 1);
#undef G2_DIAG
#undef G2_ISSUE_FIRST
#undef G2_COL_FETCH
}

}  // namespace vfps
