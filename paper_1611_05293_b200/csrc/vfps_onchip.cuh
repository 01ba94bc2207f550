// vfps_onchip.cuh -- persistent thread-block-cluster engine, second design (sm_100a).
//
// One cluster of S CTAs advances one simulation with psi resident in (distributed) shared memory;
// HBM is touched when a work item starts (load psi) and ends (store psi) and for the six
// diagnostics floats per step.  CTA `rank` owns the q-rows x in [rank*R, (rank+1)*R), R = N/S.
//
// What differs from the first design (one buffer pair, weights recomputed per cell):
//  * ONE buffer.  The rotation a1 works in place: a CTA's rows are cut into W "walker" segments
//    (W = 16 warps / (N/64) warps per row); segment w is stored as
//        [H apron rows][its rows][H apron rows] plus D free rows,
//    and a walker writes target row v into the slot D rows BEHIND it (above when it walks down,
//    below when it walks up), which every thread of the walker has finished reading because the
//    walker's warps meet at a named barrier every K rows and D = K + H.  The walk direction and
//    the position of the data inside the segment alternate from step to step (layout parity).
//    The apron rows are copies of the neighbouring segment's (or neighbouring CTA's) boundary
//    rows, written by the kick pass, so every walker sees one linear address range.
//    A 256^2 simulation therefore fits a cluster of TWO CTAs (all 148 SMs of B200 are usable by a
//    batch; a cluster of four strands 16 SMs).
//  * Per-launch geometry tables.  The source displacement of cell (x, y),
//        dx = a X + b Y,  dy = d X + a Y      (a = cos(dphi) - 1 ~ 1e-6, X, Y centred cell indices),
//    is the same in every step, and a X, a Y are tiny: with t0x(y) = b Y + a Xc - floor(dx),
//    the Lagrange weights along q are  l_i(t0x + a (X - Xc)) = M_i(y) + a (X - Xc) M'_i(y)  up to
//    (a R/2)^2 |l''|/2 <= 1.2e-7 (checked on the host; otherwise the weights are evaluated per
//    cell), and likewise along p with per-row tables L_j(x), L'_j(x).  M, M' live in registers
//    (a thread keeps its two columns for the whole launch), L, L' in shared memory; the host
//    builds them in double precision (vfps_api.cu: onchip_tables).  4 + 4 FMAs per cell replace
//    ~18 operations for floors, fractions and two cubic weight sets.
//  * A thread rotates TWO adjacent columns: the 4 x 6 register window slides down the rows with
//    three 64-bit shared loads per row (1.5 loads per cell instead of 4), one 64-bit store.
//  * Row sums (projection a2) are formed in the rotation pass in registers (transposed warp
//    reduction of 8 rows at a time); no second pass over psi'.
//  * The wake a3 is a Toeplitz product done by one warp per four rows with 128-bit loads of the
//    wake function (1.1 instructions per multiply-add); kick a4 + Fokker-Planck a5 own eight
//    consecutive cells per lane, with the Fokker-Planck stencil folded into four per-column
//    coefficients (5 operations per cell instead of 9) and column-sum moments.
//  * One DSMEM exchange fewer per step: the partial sums of step t travel with the profile of
//    step t+1 (double-buffered by step parity, one mbarrier per parity).
//
// One split step of a CTA (layout parity p = step & 1):
//   wait halo(t-1)                      neighbours' boundary rows (mbHalo), t > 0
//   1 rotation a1 + row sums a2         parity p -> parity p^1, walkers, K-row named barriers
//   -- __syncthreads --
//   2 send rho_raw(t) (own rows) and the CTA's partial sums of step t-1 to every CTA of the
//     cluster, itself included (st.async, counted on mbRho[p] of the receiver)
//   wait mbRho[p]                       all of rho(t) and all partial sums of t-1 are here
//   3 a6 of step t-1: C, 1/C, diagnostics row (rank 0)
//   4 wake a3: V for the own rows, kick weights -> vtab
//   -- __syncthreads --
//   5 kick a4 + Fokker-Planck a5 in place (parity p^1), apron copies (local stores / st.async
//     to the neighbour CTA, counted on its mbHalo), moments
//   -- __syncthreads --, warp 0 folds the CTA's partial sums of step t (sent in step t+1)
//
// Write-after-read safety of the exchanges needs no extra barrier:
//   rho/partials: buffer [p] is rewritten by rho(t+2); a CTA sends rho(t+2) after its rotation
//     (t+2), which needs its kick(t+1), which needs ALL of rho(t+1), which every CTA sends after it
//     has finished reading rho(t) (its wake phase of step t precedes its kick(t), rotation(t+1)).
//   halo: the aprons a neighbour writes during its kick(t) are those of layout parity p^1, dead
//     since this CTA's rotation(t-1) ... they are read by rotation(t+1) only; the neighbour's
//     kick(t) starts after it has rho(t) from this CTA, sent after this CTA's rotation(t).
//   mbarrier phases: thread 0 re-arms mbRho[p] for step t+2 right after its own wait; the bytes of
//     step t+2 cannot arrive before every warp of this CTA has passed its wait of step t (they
//     are sent after this CTA's rho(t+1), which follows a __syncthreads after that wait).
#pragma once
#include "vfps_cluster.cuh"

namespace vfps {

constexpr int OC_THREADS = 512;
constexpr int OC_WARPS = OC_THREADS / 32;
constexpr int OC_PADC = 8;            // zero floats left and right of every row (>= halo H)
constexpr int OC_MAX_S = 16;
constexpr int OC_NPART = 8;           // partial sums per CTA per step
constexpr int OC_ROWTAB = 12;         // floats per row of the row table
constexpr int OC_COLTAB = 8;          // floats per column of the column table
constexpr int OC_BAD = (int)0x80000000;
constexpr int OC_MAX_H = 7;

struct OnchipArgs {
    float *psi;            // [members][N][N] in/out, un-normalised
    float *scale;          // [members] in/out: 1/C of the last step
    const float *wfun;     // [members][2N] wake function, lag d at index d + N - 1; nullptr = no wake
    float *diag;           // [nsteps][members][6] or nullptr
    const float *coltab;   // [S][N][8]   TAB: M[4], M'[4] of column y for the rows of rank r; else {b Y - ix, a Y, ...}
    const int *colix;      // [S][N]      floor(dx) of column y over the rows of rank r, or OC_BAD
    const float *rowtab;   // [N][12]     TAB: L[4], L'[4], a (X - Xc), -, iy, -; else {-, ..., X (slot 8), d X - iy (slot 9), iy (slot 10)}
    int members;
    int nsteps;            // steps per work item of this launch (chunk)
    int S, R;
    int nchunks;           // work items per member in this launch; item = (chunk, member)
    int last_steps;        // steps of the last chunk (<= nsteps)
    unsigned long long *item_ctr;     // work queue head (never reset: item_base is the value at launch)
    unsigned long long item_base;
    unsigned int *member_done;        // [members] chunks finished over the life of the handle
    unsigned int done_base;           // value of member_done[m] when this launch starts
    long long *dbg;        // VFPS_PHASE_CLOCKS builds only: [CTA][64 steps][8] clock64 stamps
};

// ---- layout shared by host and device
struct OnchipLayout {
    int CW, W, RPW, H, KC, K, D, seg_rows, phys_rows, pitch, nch;
    size_t off_buf, off_rowtab, off_gtab, off_wf, off_rho, off_part, off_rowpart, off_vtab, off_rowaddr,
        off_chunk, off_wred, off_misc, total_floats;
};

__host__ __device__ inline OnchipLayout onchip_layout(int N, int S, int H, int order)
{
    OnchipLayout L;
    const int R = N / S;
    L.CW = N / 64;
    const int Wmax = OC_WARPS / L.CW;
    L.W = Wmax < R ? Wmax : R;                 // active walkers
    while (L.W > 1 && R / L.W < H) L.W /= 2;   // a walker's aprons come from its direct neighbours only
    L.RPW = R / L.W;
    L.H = H;
    L.KC = (order == 2) ? 4 : 2;               // chunks (of `order` rows) per named-barrier block
    L.K = L.KC * order;
    const int kb = L.K < L.RPW ? L.K : ((L.RPW + order - 1) / order) * order;
    L.D = kb + H;
    L.seg_rows = L.RPW + 2 * H + L.D;
    L.phys_rows = L.W * L.seg_rows;
    L.pitch = N + 2 * OC_PADC;
    L.nch = (L.RPW + order - 1) / order;
    size_t o = 0;
    L.off_buf = o;      o += (size_t)L.phys_rows * L.pitch;
    L.off_rowtab = o;   o += (size_t)R * OC_ROWTAB;
    L.off_gtab = o;     o += (size_t)N * 4;
    L.off_wf = o;       o += (size_t)2 * N;
    L.off_rho = o;      o += (size_t)2 * N;
    L.off_part = o;     o += (size_t)2 * OC_MAX_S * OC_NPART;
    L.off_rowpart = o;  o += (size_t)R * L.CW;
    L.off_vtab = o;     o += (size_t)R * 8;
    L.off_rowaddr = o;  o += (size_t)R * 4;
    L.off_chunk = o;    o += (size_t)((L.W * L.nch + 3) & ~3);
    L.off_wred = o;     o += (size_t)OC_WARPS * 8;
    L.off_misc = o;     o += 32;               // own partial sums (8), three mbarriers (6), spare
    L.total_floats = o;
    return L;
}

__device__ __forceinline__ float2 lds2(uint32_t a)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts2(uint32_t a, float x, float y)
{
    asm volatile("st.shared.v2.f32 [%0], {%1,%2};" ::"r"(a), "f"(x), "f"(y) : "memory");
}
__device__ __forceinline__ int ldsi(uint32_t a)
{
    int v;
    asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ int4 ldsi4(uint32_t a)
{
    int4 v;
    asm volatile("ld.shared.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ void named_barrier(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
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
        constexpr int LOG = (NV == 8) ? 3 : (NV == 4) ? 2 : 1;
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
            (void)LOG;
            return r;
        }
    }
}

// kick (shift by MM + t cells, Lagrange weights l already scaled by 1/C) and Fokker-Planck for the
// GW cells g..g+GW-1 of one row: b[i] = psi'(g - 4 + i), i = 0..GW+7.  k[i] = kicked value at
// position g - 1 + i (zero outside the grid, A8).  The Fokker-Planck update (Eq. 15 + 3-point
// second difference, explicit Euler) is  out = k0 + G[-1] k[-1] + G[0] k0 + G[1] k[1] + G[2] k[2]
// with the per-column coefficients gc[c] = (G-1, G0, G1, G2) of column g + c (all <= 1e-3, so the
// sum is exact to well below one ulp of k0).
template <int ORDER, int MM, int GW>
__device__ __forceinline__ void kick_fp_wide(const float (&b)[GW + 8], const float (&l)[ORDER], int g, int N,
                                             const float4 (&gc)[GW], float (&out)[GW])
{
    constexpr int O0 = (ORDER - 1) / 2;
    float k[GW + 3];
#pragma unroll
    for (int i = 0; i < GW + 3; ++i) {
        const int i0 = 3 + i + MM - O0;
        float acc = l[0] * b[i0];
#pragma unroll
        for (int j = 1; j < ORDER; ++j) acc = fmaf(l[j], b[i0 + j], acc);
        k[i] = acc;
    }
    if (g == 0) k[0] = 0.0f;
    if (g == N - GW) { k[GW + 1] = 0.0f; k[GW + 2] = 0.0f; }
#pragma unroll
    for (int c = 0; c < GW; ++c) {
        const float incr = fmaf(gc[c].w, k[c + 3], fmaf(gc[c].z, k[c + 2], fmaf(gc[c].y, k[c + 1], gc[c].x * k[c])));
        out[c] = k[c + 1] + incr;
    }
}
// any integer shift: reads the row in shared memory with bounds checks (rare: |shift| > 1 cell).
// Not inlined; weights by value, coefficients from the shared table, results through local memory,
// so that the fast path keeps its operands in registers.
template <int ORDER, int GW>
__device__ __noinline__ void kick_fp_wide_any(const float *row /* index 0 = y 0 */, float4 lw, int mm, int g, int N,
                                              const float4 *gtab, float *out)
{
    constexpr int O0 = (ORDER - 1) / 2;
    const float l[4] = {lw.x, lw.y, lw.z, lw.w};
    float k[GW + 3];
#pragma unroll 1
    for (int i = 0; i < GW + 3; ++i) {
        const int y = g - 1 + i;
        float acc = 0.0f;
        for (int j = 0; j < ORDER; ++j) {
            const int s = y + mm - O0 + j;
            const float v = (s >= 0 && s < N) ? row[s] : 0.0f;
            acc = fmaf(l[j], v, acc);
        }
        k[i] = (y >= 0 && y < N) ? acc : 0.0f;
    }
#pragma unroll 1
    for (int c = 0; c < GW; ++c) {
        const float4 gc = gtab[g + c];
        out[c] = k[c + 1] + fmaf(gc.w, k[c + 3], fmaf(gc.z, k[c + 2], fmaf(gc.y, k[c + 1], gc.x * k[c])));
    }
}

// ---------------------------------------------------------------- rotation of one walker
// A thread owns the columns y0 = 64 cw + 2 lane and y0 + 1.  The ORDER x (2 NP) register window
// holds ORDER source rows of the aligned column pairs that cover both cells' taps; it slides one
// row per target row.  PAR = (iy - O0) & 1 is the offset of cell y0's first tap inside the window,
// DIR the walk direction (+1: rows ascending).
template <int ORDER, int PITCH, bool TAB>
struct Walker {
    static constexpr int O0 = (ORDER - 1) / 2;
    static constexpr int NPMAX = (ORDER + 3) / 2;          // column pairs of the window (PAR = 1)
    float win[ORDER][2 * NPMAX];
    float M0[ORDER], M0p[ORDER], M1[ORDER], M1p[ORDER];    // TAB: weights along q of both columns and their t-derivatives
                                                           // !TAB: M0[0] = b Y0 - ix, M1[0] = b Y1 - ix
    float ey0, ey1;                                        // TAB: a (Y - Ymid); else a Y
    float a;                                               // cos(dphi) - 1 (only !TAB)
    float rs[8];                                           // row sums of the current barrier block

    template <int PAR>
    __device__ __forceinline__ void load_row(int slot, uint32_t addr)
    {
        constexpr int NP = (PAR + ORDER + 2) / 2;
#pragma unroll
        for (int k = 0; k < NP; ++k) {
            const float2 v = lds2(addr + 8 * k);
            win[slot][2 * k] = v.x; win[slot][2 * k + 1] = v.y;
        }
    }
    // weights of both cells for the target row whose table entry is at `tab`
    __device__ __forceinline__ void weights(uint32_t tab, float (&lx0)[ORDER], float (&lx1)[ORDER], float (&ly0)[ORDER],
                                            float (&ly1)[ORDER]) const
    {
        if (TAB) {
            float L[4], Lp[4];
            if (ORDER == 4) {
                const float4 v = lds4(tab), w = lds4(tab + 16);
                L[0] = v.x; L[1] = v.y; L[2] = v.z; L[3] = v.w; Lp[0] = w.x; Lp[1] = w.y; Lp[2] = w.z; Lp[3] = w.w;
            } else if (ORDER == 3) {
                const float4 v = lds4(tab); const float2 w = lds2(tab + 16);
                L[0] = v.x; L[1] = v.y; L[2] = v.z; Lp[0] = w.x; Lp[1] = w.y; Lp[2] = lds(tab + 24);
            } else {
                const float2 v = lds2(tab), w = lds2(tab + 16);
                L[0] = v.x; L[1] = v.y; Lp[0] = w.x; Lp[1] = w.y;
            }
            const float ex = lds(tab + 32);
#pragma unroll
            for (int j = 0; j < ORDER; ++j) {
                ly0[j] = fmaf(ey0, Lp[j], L[j]);
                ly1[j] = fmaf(ey1, Lp[j], L[j]);
                lx0[j] = fmaf(ex, M0p[j], M0[j]);
                lx1[j] = fmaf(ex, M1p[j], M1[j]);
            }
        } else {
            const float2 xv = lds2(tab + 32);                 // X, d X - iy
            lagrange<ORDER>(fmaf(a, xv.x, M0[0]), lx0);
            lagrange<ORDER>(fmaf(a, xv.x, M1[0]), lx1);
            lagrange<ORDER>(xv.y + ey0, ly0);
            lagrange<ORDER>(xv.y + ey1, ly1);
        }
    }
    // tensor product for both cells; slot0 = window slot of tap row i = 0
    template <int PAR, int SLOT0>
    __device__ __forceinline__ void eval(const float (&lx0)[ORDER], const float (&lx1)[ORDER], const float (&ly0)[ORDER],
                                         const float (&ly1)[ORDER], float &o0, float &o1) const
    {
        float a0 = 0.0f, a1 = 0.0f;
#pragma unroll
        for (int i = 0; i < ORDER; ++i) {
            const float(&wr)[2 * NPMAX] = win[(SLOT0 + i) % ORDER];
            float r0 = ly0[0] * wr[PAR], r1 = ly1[0] * wr[PAR + 1];
#pragma unroll
            for (int j = 1; j < ORDER; ++j) {
                r0 = fmaf(ly0[j], wr[PAR + j], r0);
                r1 = fmaf(ly1[j], wr[PAR + 1 + j], r1);
            }
            a0 = (i == 0) ? lx0[0] * r0 : fmaf(lx0[i], r0, a0);
            a1 = (i == 0) ? lx1[0] * r1 : fmaf(lx1[i], r1, a1);
        }
        o0 = a0; o1 = a1;
    }
    // one chunk of ORDER target rows, walking in direction DIR.  src = address of window column 0
    // of tap row i = 0 of the first target row; dst = address of its output pair; tab = its table
    // row; cont: the window already holds the ORDER - 1 rows shared with the previous chunk.
    // RS0 = index of the first row sum of this chunk in rs[].
    template <int PAR, int DIR, int RS0, int SUB = 0>
    __device__ __forceinline__ void chunk(uint32_t src, uint32_t dst, uint32_t tab, bool cont)
    {
        constexpr int P4 = PITCH * 4;
        if (SUB == 0 && !cont) {
            // tap rows i of the first target that later targets reuse: DIR > 0: i = 0..ORDER-2 (slots i),
            // DIR < 0: i = 1..ORDER-1 (slots i)
#pragma unroll
            for (int i = 0; i < ORDER - 1; ++i) {
                const int ii = (DIR > 0) ? i : i + 1;
                load_row<PAR>(ii, src + (uint32_t)(ii * P4));
            }
        }
        // target SUB: tap row i lives in slot (SUB + i) % ORDER (DIR > 0) or (i - SUB) mod ORDER (DIR < 0);
        // the entering tap row is i = ORDER-1 (DIR > 0) or i = 0 (DIR < 0)
        constexpr int SLOT0 = (DIR > 0) ? (SUB % ORDER) : ((ORDER - SUB % ORDER) % ORDER);
        constexpr int IN_I = (DIR > 0) ? ORDER - 1 : 0;
        load_row<PAR>((SLOT0 + IN_I) % ORDER, src + (uint32_t)((DIR * SUB + IN_I) * P4));
        float lx0[ORDER], lx1[ORDER], ly0[ORDER], ly1[ORDER];
        weights(tab + (uint32_t)(DIR * SUB * (OC_ROWTAB * 4)), lx0, lx1, ly0, ly1);
        float o0, o1;
        eval<PAR, SLOT0>(lx0, lx1, ly0, ly1, o0, o1);
        sts2(dst + (uint32_t)(DIR * SUB * P4), o0, o1);
        rs[RS0 + SUB] = o0 + o1;
        if constexpr (SUB + 1 < ORDER) chunk<PAR, DIR, RS0, SUB + 1>(src, dst, tab, cont);
    }
};

// one cell with its own floors and a full window (rows where a floor changes inside the thread's
// columns or along the chunk)
template <int ORDER, int PITCH>
__device__ __forceinline__ float rotate_cell_generic(const GridConst &G, uint32_t rowbase /* segment row 0, column 0 */,
                                                     int v, int x, int y)
{
    constexpr int O0 = (ORDER - 1) / 2;
    const float X = (float)x + G.x0c, Y = (float)y + G.y0c;
    int ix, iy;
    float tx, ty;
    floor_frac(fmaf(G.a, X, G.b * Y), ix, tx);
    floor_frac(fmaf(G.d, X, G.a * Y), iy, ty);
    float lx[ORDER], ly[ORDER];
    lagrange<ORDER>(tx, lx);
    lagrange<ORDER>(ty, ly);
    const uint32_t base = rowbase + (uint32_t)(((v + ix - O0) * PITCH + (y + iy - O0)) * 4);
    float acc = 0.0f;
#pragma unroll
    for (int i = 0; i < ORDER; ++i) {
        float r = ly[0] * lds(base + (i * PITCH) * 4);
#pragma unroll
        for (int j = 1; j < ORDER; ++j) r = fmaf(ly[j], lds(base + (i * PITCH + j) * 4), r);
        acc = (i == 0) ? lx[0] * r : fmaf(lx[i], r, acc);
    }
    return acc;
}

#define OC_STAMP(k) VFPS_STAMP(A.dbg, step, k)

// ---------------------------------------------------------------- the persistent kernel
// grid = S * (concurrent clusters), cluster = S CTAs, block = 512.  Clusters take work items
// (chunk j of member m, in the order j * members + m) from a queue in global memory; chunk j of a
// member starts after its chunk j-1 has been stored (member_done).
template <int ORDER, int N, bool TAB>
__global__ void __launch_bounds__(OC_THREADS, 1)
k_onchip_step(GridConst G, OnchipArgs A)
{
    static_assert(N >= 64 && N % 64 == 0, "N must be a multiple of 64");
    constexpr int PITCH = N + 2 * OC_PADC;
    constexpr int P4 = PITCH * 4;
    constexpr int O0 = (ORDER - 1) / 2;
    constexpr int CW = N / 64;
    constexpr int GW = (N >= 256) ? 8 : 4;                 // cells per lane in the kick pass
    constexpr int NG = (N / (32 * GW)) > 0 ? (N / (32 * GW)) : 1;   // granules per lane and row
    constexpr int KL = (32 * GW <= N) ? 32 : N / GW;       // active lanes in the kick pass
    constexpr int NW = N / 128 > 0 ? N / 128 : 1;          // float4 groups of rho per lane in the wake
    constexpr unsigned FULL = 0xffffffffu;

    cg::cluster_group cluster = cg::this_cluster();
    const int S = A.S, R = A.R, H = G.H;
    const OnchipLayout LY = onchip_layout(N, S, H, ORDER);
    const int W = LY.W, RPW = LY.RPW, D = LY.D, KC = LY.KC, nch = LY.nch, SEG = LY.seg_rows;
    const int rank = (int)cluster.block_rank();
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int x0 = rank * R;

    extern __shared__ __align__(16) float smem[];
    float *buf = smem + LY.off_buf;
    float *rowtab_s = smem + LY.off_rowtab;
    float *gtab = smem + LY.off_gtab;
    float *wf = smem + LY.off_wf;
    float *rhob = smem + LY.off_rho;
    float *partb = smem + LY.off_part;
    float *rowpart = smem + LY.off_rowpart;
    float *vtab = smem + LY.off_vtab;
    int *rowaddr = reinterpret_cast<int *>(smem + LY.off_rowaddr);
    int *chunkinfo = reinterpret_cast<int *>(smem + LY.off_chunk);
    float *wred = smem + LY.off_wred;
    float *misc = smem + LY.off_misc;                      // [0..7] own partial sums, [8..13] mbarriers, [16] item
    const uint32_t sBuf = smem_u32(buf), sRowtab = smem_u32(rowtab_s), sRho = smem_u32(rhob), sPart = smem_u32(partb);
    const uint32_t sVtab = smem_u32(vtab), sMisc = smem_u32(misc);
    const uint32_t mbRho0 = sMisc + 32, mbHalo = sMisc + 48;        // mbRho[p] = mbRho0 + 8 p
    const int nbrs = (rank > 0 ? 1 : 0) + (rank < S - 1 ? 1 : 0);
    const uint32_t bytesRho = (uint32_t)(N + S * OC_NPART) * 4u, bytesPart = (uint32_t)(S * OC_NPART) * 4u;
    const uint32_t bytesHalo = (uint32_t)(nbrs * H * N) * 4u;

    // ---- rotation role: walker wk, columns y0, y0 + 1
    const int wk = warp / CW, cw = warp % CW;
    const bool walker_on = wk < W;
    const int y0 = 64 * cw + 2 * lane;
    const int wb = wk * RPW;                               // first CTA-local row of the walker
    Walker<ORDER, PITCH, TAB> wkr;
    int ixc = 0;
    bool cols_ok = false;
    {
        const int c0 = A.colix[(size_t)rank * N + y0], c1 = A.colix[(size_t)rank * N + y0 + 1];
        ixc = c0;
        cols_ok = __all_sync(FULL, c0 != OC_BAD && c0 == c1);
        const float *ct0 = A.coltab + ((size_t)rank * N + y0) * OC_COLTAB, *ct1 = ct0 + OC_COLTAB;
#pragma unroll
        for (int i = 0; i < ORDER; ++i) {
            wkr.M0[i] = ct0[i]; wkr.M0p[i] = ct0[4 + i];
            wkr.M1[i] = ct1[i]; wkr.M1p[i] = ct1[4 + i];
        }
        // TAB: a (Y - Ymid) in slot 7 of the !TAB layout is unused; both layouts keep e_y in [7]... see host
        wkr.ey0 = TAB ? G.a * ((float)y0 - 0.5f * (float)(N - 1)) : ct0[1];
        wkr.ey1 = TAB ? G.a * ((float)(y0 + 1) - 0.5f * (float)(N - 1)) : ct1[1];
        wkr.a = G.a;
        if (!cols_ok) ixc = 0;
    }
    const uint32_t segA = sBuf + (uint32_t)(wk * SEG) * P4;     // physical row 0 of the walker's segment

    // ---- one-time set-up: zero the buffer (pads stay zero for ever), tables, barriers
    for (int i = tid; i < LY.phys_rows * PITCH; i += OC_THREADS) buf[i] = 0.0f;
    for (int i = tid; i < R * OC_ROWTAB; i += OC_THREADS) rowtab_s[i] = A.rowtab[(size_t)x0 * OC_ROWTAB + i];
    {
        const float c1 = G.fp_b / (6.0f * G.dp), c2 = G.fp_b / (G.dp * G.dp);
        for (int y = tid; y < N; y += OC_THREADS) {
            const float c1p = c1 * fmaf((float)y, G.dp, G.p_min);
            reinterpret_cast<float4 *>(gtab)[y] =
                make_float4(fmaf(-2.0f, c1p, c2), fmaf(-3.0f, c1p, fmaf(-2.0f, c2, G.fp_b)), fmaf(6.0f, c1p, c2), -c1p);
        }
    }
    // per row: parity-0 byte offsets (from sBuf, column 0) of its own slot and of the apron slots it
    // is copied to (0 = none); flags: 1 up copy is remote (rank-1), 2 down copy is remote (rank+1),
    // 4 up apron lies outside the grid (zero it), 8 down apron outside the grid
    for (int r = tid; r < R; r += OC_THREADS) {
        const int w = r / RPW, v = r - w * RPW;
        const int own = ((w * SEG + D + H + v) * PITCH + OC_PADC) * 4;
        int up = 0, dn = 0, fl = 0;
        if (v < H) {                                       // among the first H rows of its walker: bottom apron of the walker above
            if (w > 0) up = (((w - 1) * SEG + D + H + RPW + v) * PITCH + OC_PADC) * 4;
            else if (rank > 0) { up = (((W - 1) * SEG + D + H + RPW + v) * PITCH + OC_PADC) * 4; fl |= 1; }
            else { up = ((D + v) * PITCH + OC_PADC) * 4; fl |= 4; }        // grid edge: own top apron row -H + v := 0
        }
        if (v >= RPW - H) {                                // among the last H rows: top apron of the walker below
            const int k = v - (RPW - H);                   // apron row -H + k
            if (w < W - 1) dn = (((w + 1) * SEG + D + k) * PITCH + OC_PADC) * 4;
            else if (rank < S - 1) { dn = ((0 * SEG + D + k) * PITCH + OC_PADC) * 4; fl |= 2; }
            else { dn = (((W - 1) * SEG + D + H + RPW + k) * PITCH + OC_PADC) * 4; fl |= 8; }   // own bottom apron row RPW + k := 0
        }
        rowaddr[4 * r + 0] = own; rowaddr[4 * r + 1] = up; rowaddr[4 * r + 2] = dn; rowaddr[4 * r + 3] = fl;
    }
    __syncthreads();
    // per (walker, chunk): iy of its rows if they are all good and equal and the chunk is full, else OC_BAD
    for (int i = tid; i < W * nch; i += OC_THREADS) {
        const int w = i / nch, c = i - w * nch;
        int iy = OC_BAD;
        if ((c + 1) * ORDER <= RPW) {
            iy = __float_as_int(rowtab_s[(w * RPW + c * ORDER) * OC_ROWTAB + 10]);
            for (int k = 1; k < ORDER; ++k)
                if (__float_as_int(rowtab_s[(w * RPW + c * ORDER + k) * OC_ROWTAB + 10]) != iy) iy = OC_BAD;
        }
        chunkinfo[i] = iy;
    }
    if (tid == 0) {
        mbar_init(mbRho0, 1); mbar_init(mbRho0 + 8, 1); mbar_init(mbHalo, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    unsigned rho_use0 = 0u, rho_use1 = 0u;      // how often mbRho[p] has been waited on
    unsigned halo_use = 0u;
    __syncthreads();
    cluster.sync();

    const float yc = 0.5f * (float)(N - 1), xc = 0.5f * (float)(N - 1);
    const unsigned long long nitems = (unsigned long long)A.nchunks * (unsigned long long)A.members;

    for (;;) {
        // ---- next work item (one fetch per cluster, broadcast through rank 0's shared memory)
        if (tid == 0) {
            if (rank == 0) {
                const unsigned long long it = atomicAdd(A.item_ctr, 1ull) - A.item_base;
                const unsigned lo = (unsigned)it, hi = (unsigned)(it >> 32);
                for (int dd = 0; dd < S; ++dd) {
                    asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(mapa(sMisc + 64, dd)), "r"(lo) : "memory");
                    asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(mapa(sMisc + 68, dd)), "r"(hi) : "memory");
                }
            }
        }
        cluster.sync();
        const unsigned long long item =
            (unsigned long long)__float_as_uint(misc[16]) | ((unsigned long long)__float_as_uint(misc[17]) << 32);
        if (item >= nitems) break;
        const int chunk_j = (int)(item / (unsigned long long)A.members), m = (int)(item - (unsigned long long)chunk_j * A.members);
        const int nsteps = (chunk_j == A.nchunks - 1) ? A.last_steps : A.nsteps;
        const int step_base = chunk_j * A.nsteps;          // diagnostics row of the item's first step
        if (chunk_j > 0) {
            // the member's previous chunk must have been stored (by whichever cluster ran it)
            if (tid == 0) {
                const unsigned want = A.done_base + (unsigned)chunk_j;
                unsigned got;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(got) : "l"(A.member_done + m) : "memory");
                } while ((int)(got - want) < 0);
            }
            __syncthreads();
        }
        float *gpsi = A.psi + (size_t)m * N * N;
        const float *gw = A.wfun ? A.wfun + (size_t)m * 2 * N : nullptr;

        // ---- load psi into the parity-0 layout: every walker's rows and aprons (zero outside the grid)
        for (int i = tid; i < W * (RPW + 2 * H) * (N / 4); i += OC_THREADS) {
            const int c4 = i % (N / 4), rr = i / (N / 4);
            const int w = rr / (RPW + 2 * H), v = rr - w * (RPW + 2 * H) - H;     // segment-local row -H .. RPW+H-1
            const int x = x0 + w * RPW + v;
            float4 val = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            if (x >= 0 && x < N) val = __ldcg(reinterpret_cast<const float4 *>(gpsi + (size_t)x * N) + c4);
            *reinterpret_cast<float4 *>(buf + (size_t)(w * SEG + D + H + v) * PITCH + OC_PADC + 4 * c4) = val;
        }
        for (int i = tid; i < 2 * N; i += OC_THREADS) wf[i] = (gw && i < 2 * N - 1) ? gw[i] : 0.0f;
        float sc = G.renorm ? A.scale[m] : 1.0f;
        if (tid == 0) {
            mbar_expect_tx(mbRho0, nsteps >= 1 ? bytesRho : bytesPart);
            mbar_expect_tx(mbRho0 + 8, nsteps >= 2 ? bytesRho : bytesPart);      // unused if nsteps == 0
            if (nbrs > 0 && nsteps >= 1) mbar_expect_tx(mbHalo, bytesHalo);
        }
        // nobody may store into this CTA before it has finished initialising
        cluster.sync();

        for (int step = 0; step <= nsteps; ++step) {
            const bool last = (step == nsteps);
            const int p = step & 1;                        // layout parity at the start of the step
            if (step > 0 && nbrs > 0) {
                // ---- the neighbours' boundary rows of psi_t have arrived
                mbar_wait(mbHalo, halo_use & 1u);
                ++halo_use;
                if (tid == 0 && !last) mbar_expect_tx(mbHalo, bytesHalo);
            }
            OC_STAMP(0);
            // ================= 1. rotation a1 + row sums a2, parity p -> p ^ 1
            if (!last && walker_on) {
                // physical row of segment-local row 0: parity 0 -> D + H, parity 1 -> H
                const int row0 = p ? H : D + H;
                const uint32_t rbase = segA + (uint32_t)(row0 * P4);                 // row 0, buffer column -PADC
                const int dsh = p ? D : -D;                                            // output slot shift (rows)
                int prev_iy = OC_BAD;
#pragma unroll
                for (int k = 0; k < 8; ++k) wkr.rs[k] = 0.0f;
                int blk_row0 = p ? (RPW - 1) : 0;          // first row (walk order) of the current barrier block
                for (int ci = 0; ci < nch; ++ci) {
                    const int c = p ? nch - 1 - ci : ci;
                    const int iy = chunkinfo[wk * nch + c];
                    const int kk = ci % KC;                // chunk index inside the barrier block
                    const int vlo = c * ORDER, nrow = min(ORDER, RPW - vlo);
                    if (cols_ok && iy != OC_BAD) {
                        const bool cont = (prev_iy == iy);
                        const int par = (iy - O0) & 1;
                        const int v0 = p ? vlo + ORDER - 1 : vlo;                      // first target row in walk order
                        // window column 0 = grid column y0 + iy - O0 - par
                        const uint32_t src = rbase + (uint32_t)((v0 + ixc - O0) * P4 + (OC_PADC + y0 + iy - O0 - par) * 4);
                        const uint32_t dst = rbase + (uint32_t)((v0 + dsh) * P4 + (OC_PADC + y0) * 4);
                        const uint32_t tab = sRowtab + (uint32_t)((wb + v0) * OC_ROWTAB * 4);
#define OC_CHUNK(PAR_, DIR_)                                                                       \
    do {                                                                                            \
        if constexpr (ORDER == 2) {                                                                 \
            if (kk == 0) wkr.template chunk<PAR_, DIR_, 0>(src, dst, tab, cont);                    \
            else if (kk == 1) wkr.template chunk<PAR_, DIR_, 2>(src, dst, tab, cont);               \
            else if (kk == 2) wkr.template chunk<PAR_, DIR_, 4>(src, dst, tab, cont);               \
            else wkr.template chunk<PAR_, DIR_, 6>(src, dst, tab, cont);                            \
        } else {                                                                                    \
            if (kk == 0) wkr.template chunk<PAR_, DIR_, 0>(src, dst, tab, cont);                    \
            else wkr.template chunk<PAR_, DIR_, 4>(src, dst, tab, cont);                            \
        }                                                                                           \
    } while (0)
                        if (p == 0) { if (par) OC_CHUNK(1, 1); else OC_CHUNK(0, 1); }
                        else        { if (par) OC_CHUNK(1, -1); else OC_CHUNK(0, -1); }
#undef OC_CHUNK
                        prev_iy = iy;
                    } else {
                        const uint32_t gbase = rbase + (uint32_t)(OC_PADC * 4);
                        for (int s = 0; s < nrow; ++s) {
                            const int v = p ? vlo + nrow - 1 - s : vlo + s;
                            const float o0 = rotate_cell_generic<ORDER, PITCH>(G, gbase, v, x0 + wb + v, y0);
                            const float o1 = rotate_cell_generic<ORDER, PITCH>(G, gbase, v, x0 + wb + v, y0 + 1);
                            sts2(rbase + (uint32_t)((v + dsh) * P4 + (OC_PADC + y0) * 4), o0, o1);
                            const int ri = kk * ((ORDER == 3) ? 4 : ORDER) + s;
                            // rs[] is indexed statically: add through a select chain
#pragma unroll
                            for (int k = 0; k < 8; ++k) if (k == ri) wkr.rs[k] = o0 + o1;
                        }
                        prev_iy = OC_BAD;
                    }
                    if (kk == KC - 1 || ci == nch - 1) {
                        // row sums of this block: rs[kk' * stride + s] belongs to the row s of chunk kk'
                        const float tot = warp_reduce_transposed<8>(wkr.rs, lane);
                        const int idx = lane >> 2;                                     // value index 0..7
                        constexpr int ST = (ORDER == 3) ? 4 : ORDER;                   // rs slots per chunk
                        const int kq = idx / ST, s = idx - kq * ST;
                        const int cq = (ci - kk) + kq;                                 // chunk (walk order) of that value
                        if ((lane & 3) == 0 && s < ORDER && cq <= ci) {
                            const int cc = p ? nch - 1 - cq : cq;
                            const int nr = min(ORDER, RPW - cc * ORDER);
                            // fast chunks run in walk order; generic rows too (s-th row in walk order)
                            const int v = p ? cc * ORDER + nr - 1 - s : cc * ORDER + s;
                            if (s < nr) rowpart[(wb + v) * CW + cw] = tot;
                        }
#pragma unroll
                        for (int k = 0; k < 8; ++k) wkr.rs[k] = 0.0f;
                        if (ci != nch - 1) {
                            if (CW > 1) named_barrier(1 + wk, CW * 32); else __syncwarp();
                        }
                        (void)blk_row0;
                    }
                }
            }
            OC_STAMP(1);
            __syncthreads();
            OC_STAMP(2);
            // ================= 2. send rho_raw(t) and the partial sums of t-1 to every CTA (self included)
            {
                const uint32_t rb = sRho + (uint32_t)(p * N) * 4u, pb = sPart + (uint32_t)(p * OC_MAX_S * OC_NPART) * 4u;
                const uint32_t mb = mbRho0 + 8u * (uint32_t)p;
                if (!last) {
                    const int nq = R >> 2;
                    for (int i = tid; i < S * nq; i += OC_THREADS) {
                        const int dd = i / nq, q = i - dd * nq;
                        float pv[4];
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            float s = 0.0f;
#pragma unroll
                            for (int c = 0; c < CW; ++c) s += rowpart[(4 * q + k) * CW + c];
                            pv[k] = s * G.dp;
                        }
                        st_async4(mapa(rb + (uint32_t)(x0 + 4 * q) * 4u, dd), make_float4(pv[0], pv[1], pv[2], pv[3]), mapa(mb, dd));
                    }
                }
                if (tid >= OC_THREADS - 2 * S) {
                    const int i = tid - (OC_THREADS - 2 * S), dd = i >> 1, hh = i & 1;
                    st_async4(mapa(pb + (uint32_t)(rank * OC_NPART + 4 * hh) * 4u, dd), lds4(sMisc + 16 * hh), mapa(mb, dd));
                }
                OC_STAMP(3);
                mbar_wait(mb, (p ? rho_use1 : rho_use0) & 1u);
                if (p) ++rho_use1; else ++rho_use0;
                if (tid == 0 && step + 2 <= nsteps) mbar_expect_tx(mb, (step + 2 < nsteps) ? bytesRho : bytesPart);
                OC_STAMP(4);
                // ================= 3. a6 of step t-1: charge, scale, diagnostics
                if (step > 0) {
                    // lane = (g4, j): partial j summed over the CTAs g4, g4 + 4, ..., then over the four
                    // lane groups -- the same order in every warp of every CTA
                    float tj = 0.0f;
                    for (int dd = lane >> 3; dd < S; dd += 4) tj += lds(pb + (uint32_t)(dd * OC_NPART + (lane & 7)) * 4u);
                    tj += __shfl_xor_sync(FULL, tj, 8);
                    tj += __shfl_xor_sync(FULL, tj, 16);
                    const float t0 = __shfl_sync(FULL, tj, 0);
                    const float C = (G.dq * G.dp) * t0;
                    sc = G.renorm ? 1.0f / C : 1.0f;
                    if (rank == 0 && warp == OC_WARPS - 1 && A.diag != nullptr) {
                        float t[OC_NPART];
#pragma unroll
                        for (int j = 0; j < OC_NPART; ++j) t[j] = __shfl_sync(FULL, tj, j);
                        if (lane == 0) {
                            const float i0 = 1.0f / t[0];
                            const float mp_c = t[1] * i0, vp = fmaf(-mp_c, mp_c, t[2] * i0);
                            const float mq_c = t[3] * i0, vq = fmaf(-mq_c, mq_c, t[4] * i0);
                            const float cc = G.renorm ? C : 1.0f;
                            float *o = A.diag + ((size_t)(step_base + step - 1) * A.members + m) * 6;
                            o[0] = C;
                            o[1] = fmaf(mq_c + xc, G.dq, G.q_min);
                            o[2] = fmaf(mp_c + yc, G.dp, G.p_min);
                            o[3] = sqrtf(fmaxf(vq, 0.0f)) * G.dq;
                            o[4] = sqrtf(fmaxf(vp, 0.0f)) * G.dp;
                            o[5] = t[5] * G.dq / (cc * cc);
                        }
                    }
                }
                if (last) break;
                // ================= 4. wake a3: one warp per four rows, V_x = sum_x' w[x - x'] rho_x'
                // lane covers x' = 4 lane + 128 j + c; for the rows x + k (x % 4 == 0) it needs
                // w[A + k - c], A = x - 4 lane - 128 j + N - 1 = 3 mod 4: two aligned 128-bit loads
                {
                    float4 rr[NW];
#pragma unroll
                    for (int j = 0; j < NW; ++j)
                        rr[j] = (4 * lane + 128 * j < N) ? lds4(rb + (uint32_t)(4 * lane + 128 * j) * 4u) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                    const uint32_t sWf = smem_u32(wf);
                    for (int q = warp; q < (R >> 2); q += OC_WARPS) {
                        const int x = x0 + 4 * q;
                        float vq[4] = {0.0f, 0.0f, 0.0f, 0.0f};
                        if (gw != nullptr) {
#pragma unroll
                            for (int j = 0; j < NW; ++j) {
                                if (4 * lane + 128 * j < N) {
                                    const int Aq = x - 4 * lane - 128 * j + N - 1;
                                    const float4 wl = lds4(sWf + (uint32_t)(Aq - 3) * 4u);   // w[A-3 .. A]
                                    const float4 wh = (Aq + 1 < 2 * N) ? lds4(sWf + (uint32_t)(Aq + 1) * 4u)
                                                                       : make_float4(0.0f, 0.0f, 0.0f, 0.0f);   // w[A+1 .. A+4]
                                    const float w7[8] = {wl.x, wl.y, wl.z, wl.w, wh.x, wh.y, wh.z, wh.w};   // w7[i] = w[A - 3 + i]
                                    const float rc[4] = {rr[j].x, rr[j].y, rr[j].z, rr[j].w};
#pragma unroll
                                    for (int k = 0; k < 4; ++k)
#pragma unroll
                                        for (int c = 0; c < 4; ++c) vq[k] = fmaf(w7[3 + k - c], rc[c], vq[k]);
                                }
                            }
                        }
                        const float Vr = warp_reduce_transposed<4>(vq, lane);     // lanes 8k .. 8k+7 hold row x + k
                        if ((lane & 7) == 0) {
                            const int k = lane >> 3, r = 4 * q + k;
                            const float V = Vr * sc;
                            const float rho_x = lds(rb + (uint32_t)(x + k) * 4u) * sc;
                            int mm;
                            float t;
                            floor_frac(G.kick_c * V, mm, t);
                            float l[ORDER];
                            lagrange<ORDER>(t, l);
                            float pl[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
                            for (int j = 0; j < ORDER; ++j) pl[j] = l[j] * sc;
                            sts4(sVtab + (uint32_t)r * 32u, make_float4(pl[0], pl[1], pl[2], pl[3]));
                            sts2(sVtab + (uint32_t)r * 32u + 16u, __int_as_float(mm), rho_x * V);
                        }
                    }
                }
            }
            OC_STAMP(5);
            __syncthreads();
            // ================= 5. kick a4 + Fokker-Planck a5 in place (parity p ^ 1), aprons, moments
            {
                const int pshift = (p ^ 1) ? D * P4 : 0;       // parity 1 lies D rows above the parity-0 slot
                float cs[NG][GW];
#pragma unroll
                for (int k = 0; k < NG; ++k)
#pragma unroll
                    for (int c = 0; c < GW; ++c) cs[k][c] = 0.0f;
                float q1 = 0.0f, q2 = 0.0f, pw = 0.0f;
                // Fokker-Planck coefficients of the lane's columns: registers for the whole pass when a lane
                // owns one granule per row, re-read per granule otherwise (N = 512: 64 registers too many)
                float4 gc[GW];
                if (NG == 1 && lane < KL) {
#pragma unroll
                    for (int c = 0; c < GW; ++c) gc[c] = reinterpret_cast<const float4 *>(gtab)[GW * lane + c];
                }
                const uint32_t mbUp = (rank > 0) ? mapa(mbHalo, rank - 1) : 0u, mbDn = (rank < S - 1) ? mapa(mbHalo, rank + 1) : 0u;
                for (int r = warp; r < R; r += OC_WARPS) {
                    const float4 lw = lds4(sVtab + (uint32_t)r * 32u);
                    const float2 mv = lds2(sVtab + (uint32_t)r * 32u + 16u);
                    const int mm = __float_as_int(mv.x);
                    const int4 ra = ldsi4(smem_u32(rowaddr) + (uint32_t)r * 16u);
                    const float lws[4] = {lw.x, lw.y, lw.z, lw.w};
                    float l[ORDER];
#pragma unroll
                    for (int j = 0; j < ORDER; ++j) l[j] = lws[j];
                    const uint32_t own = sBuf + (uint32_t)(ra.x - pshift);
                    float o[NG][GW];
                    if (lane < KL) {
                        if (mm >= -2 && mm <= 0) {
                            float b[NG][GW + 8];
#pragma unroll
                            for (int k = 0; k < NG; ++k) {
                                const int g = GW * lane + 32 * GW * k;
#pragma unroll
                                for (int i = 0; i < (GW + 8) / 4; ++i) {
                                    const float4 v = lds4(own + (uint32_t)((g - 4 + 4 * i) * 4));
                                    b[k][4 * i] = v.x; b[k][4 * i + 1] = v.y; b[k][4 * i + 2] = v.z; b[k][4 * i + 3] = v.w;
                                }
                            }
#pragma unroll
                            for (int k = 0; k < NG; ++k) {
                                const int g = GW * lane + 32 * GW * k;
                                if (NG > 1) {
#pragma unroll
                                    for (int c = 0; c < GW; ++c) gc[c] = reinterpret_cast<const float4 *>(gtab)[g + c];
                                }
                                if (mm == 0) kick_fp_wide<ORDER, 0, GW>(b[k], l, g, N, gc, o[k]);
                                else if (mm == -1) kick_fp_wide<ORDER, -1, GW>(b[k], l, g, N, gc, o[k]);
                                else kick_fp_wide<ORDER, -2, GW>(b[k], l, g, N, gc, o[k]);
                            }
                        } else {
                            const float *rowp = buf + ((ra.x - pshift) >> 2);
#pragma unroll
                            for (int k = 0; k < NG; ++k) {
                                float tmp[GW];
                                kick_fp_wide_any<ORDER, GW>(rowp, lw, mm, GW * lane + 32 * GW * k, N,
                                                            reinterpret_cast<const float4 *>(gtab), tmp);
#pragma unroll
                                for (int c = 0; c < GW; ++c) o[k][c] = tmp[c];
                            }
                        }
                    }
                    __syncwarp();                              // every lane has read the row before anyone overwrites it
                    if (lane < KL) {
                        const bool up = ra.y != 0, dn = ra.z != 0;
                        const uint32_t aup = up ? ((ra.w & 1) ? mapa(sBuf + (uint32_t)(ra.y - pshift), rank - 1) : sBuf + (uint32_t)(ra.y - pshift)) : 0u;
                        const uint32_t adn = dn ? ((ra.w & 2) ? mapa(sBuf + (uint32_t)(ra.z - pshift), rank + 1) : sBuf + (uint32_t)(ra.z - pshift)) : 0u;
                        float q0 = 0.0f;
#pragma unroll
                        for (int k = 0; k < NG; ++k) {
                            const int g = GW * lane + 32 * GW * k;
#pragma unroll
                            for (int h4 = 0; h4 < GW / 4; ++h4) {
                                const float4 ov = make_float4(o[k][4 * h4], o[k][4 * h4 + 1], o[k][4 * h4 + 2], o[k][4 * h4 + 3]);
                                const float4 z4 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                                const uint32_t off = (uint32_t)((g + 4 * h4) * 4);
                                sts4(own + off, ov);
                                if (up) { if (ra.w & 1) st_async4(aup + off, ov, mbUp); else sts4(aup + off, (ra.w & 4) ? z4 : ov); }
                                if (dn) { if (ra.w & 2) st_async4(adn + off, ov, mbDn); else sts4(adn + off, (ra.w & 8) ? z4 : ov); }
                            }
#pragma unroll
                            for (int c = 0; c < GW; ++c) { cs[k][c] += o[k][c]; q0 += o[k][c]; }
                        }
                        const float X = (float)(x0 + r) - xc, tq = q0 * X;
                        q1 += tq; q2 = fmaf(tq, X, q2);
                        if (lane == 0) pw += mv.y;
                    }
                }
                OC_STAMP(6);
                // ---- per-warp sums -> wred; s0, s1, s2 from the column sums
                float v8[8] = {0.0f, 0.0f, 0.0f, q1, q2, pw, 0.0f, 0.0f};
                if (lane < KL) {
#pragma unroll
                    for (int k = 0; k < NG; ++k)
#pragma unroll
                        for (int c = 0; c < GW; ++c) {
                            const float yy = (float)(GW * lane + 32 * GW * k + c) - yc;
                            const float tt = cs[k][c] * yy;
                            v8[0] += cs[k][c]; v8[1] += tt; v8[2] = fmaf(tt, yy, v8[2]);
                        }
                }
                const float tot = warp_reduce_transposed<8>(v8, lane);       // lanes 4 j .. 4 j + 3 hold sum j
                if ((lane & 3) == 0) wred[warp * 8 + (lane >> 2)] = tot;
            }
            __syncthreads();
            if (warp == 0) {
                // lane = (g4, j): partial j of the warps g4, g4 + 4, ...; then across the four lane groups
                const int j = lane & 7, g4 = lane >> 3;
                float v = 0.0f;
#pragma unroll
                for (int w = 0; w < OC_WARPS / 4; ++w) v += wred[(g4 + 4 * w) * 8 + j];
                v += __shfl_xor_sync(FULL, v, 8);
                v += __shfl_xor_sync(FULL, v, 16);
                if (lane < OC_NPART) misc[lane] = v;          // sent with rho of the next step (after a __syncthreads)
            }
            OC_STAMP(7);
        }
        // ---- store own rows (layout parity nsteps & 1) and the scale
        __syncthreads();
        {
            const int row0 = (nsteps & 1) ? H : D + H;
            for (int i = tid; i < R * (N / 4); i += OC_THREADS) {
                const int r = i / (N / 4), c4 = i - r * (N / 4);
                const int w = r / RPW, v = r - w * RPW;
                __stcg(reinterpret_cast<float4 *>(gpsi + (size_t)(x0 + r) * N) + c4,
                       *reinterpret_cast<const float4 *>(buf + (size_t)(w * SEG + row0 + v) * PITCH + OC_PADC + 4 * c4));
            }
        }
        if (rank == 0 && tid == 0) A.scale[m] = sc;
        __threadfence();
        cluster.sync();       // every CTA has stored its rows: publish the chunk, then take the next item
        if (rank == 0 && tid == 0) {
            __threadfence();
            atomicAdd(A.member_done + m, 1u);
        }
    }
}

}  // namespace vfps
