// vfps_onchip.cuh -- persistent thread-block-cluster engine, in-place design (sm_100a).
//
// One cluster of S CTAs advances one simulation with psi resident in (distributed) shared memory;
// HBM is touched when a work item starts (load psi) and ends (store psi) and for the six
// diagnostics floats per step.  CTA `rank` owns the q-rows x in [rank*R, (rank+1)*R), R = N/S.
//
// What differs from the first design (vfps_cluster.cuh: one buffer pair, weights recomputed per cell):
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
//  * A thread rotates TWO adjacent columns: the ORDER x 6 register window slides along the rows
//    with three 64-bit shared loads per row (1.5 loads per cell instead of 4), one 64-bit store.
//    The loads of the NEXT target row (its entering window row, its table row) are issued in the
//    middle of the current row's arithmetic -- the window row that leaves is consumed first -- so
//    the shared-memory latency hides behind ~45 FMAs instead of stalling every row.
//  * Row sums (projection a2) are formed in the rotation pass in registers (transposed warp
//    reduction of one chunk of rows at a time); no second pass over psi'.
//  * The wake a3 is a Toeplitz product done by one warp per four rows with 128-bit loads of the
//    wake function (1.1 instructions per multiply-add); kick a4 + Fokker-Planck a5: a lane owns
//    the 4-cell granules 4 lane + 128 k of a row (128-bit loads with a lane stride of 16 bytes:
//    free of bank conflicts), with the Fokker-Planck stencil folded into four per-column
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

// rows a walker rotates between two checks of its floors (a multiple of the window period ORDER)
__host__ __device__ constexpr int oc_chunk_rows(int order) { return order == 3 ? 3 : 4; }

struct OnchipArgs {
    float *psi;            // [members][N][N] in/out, un-normalised
    float *scale;          // [members] in/out: 1/C of the last step
    const float *wfun;     // [members][2N] wake function, lag d at index d + N - 1; nullptr = no wake
    float *diag;           // [nsteps][members][6] or nullptr
    const float *coltab;   // [S][N][8]   TAB: M[4], M'[4] of column y for the rows of rank r; else {b Y - ix, a Y, ...}
    const int *colix;      // [S][N]      floor(dx) of column y over the rows of rank r, or OC_BAD
    const float *rowtab;   // [N][12]     per-row weights along p, see onchip_tables (vfps_api.cu)
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

// ---- layout shared by host and device.  The psi buffer comes last, after at least one row's
// worth of tables and before one spare row: the rotation prefetches one window row past either
// end of a walker's range (the value is never used, the address must be inside the allocation).
struct OnchipLayout {
    int CW, W, RPW, H, KC, K, D, seg_rows, phys_rows, pitch, nch;
    size_t off_buf, off_rowtab, off_gtab, off_wf, off_rho, off_part, off_rowpart, off_vtab, off_rowaddr,
        off_chunk, off_wred, off_misc, total_floats;
};

__host__ __device__ inline OnchipLayout onchip_layout(int N, int S, int H, int order)
{
    OnchipLayout L;
    const int R = N / S, CH = oc_chunk_rows(order);
    L.CW = N / 64;
    const int Wmax = OC_WARPS / L.CW;
    L.W = Wmax < R ? Wmax : R;                 // active walkers
    while (L.W > 1 && R / L.W < H) L.W /= 2;   // a walker's aprons come from its direct neighbours only
    L.RPW = R / L.W;
    L.H = H;
    L.KC = 2;                                  // chunks per named-barrier block
    L.K = L.KC * CH;
    const int kb = L.K < L.RPW ? L.K : ((L.RPW + CH - 1) / CH) * CH;
    L.D = kb + H;
    L.seg_rows = L.RPW + 2 * H + L.D;
    L.phys_rows = L.W * L.seg_rows;
    L.pitch = N + 2 * OC_PADC;
    L.nch = (L.RPW + CH - 1) / CH;
    size_t o = 0;
    L.off_misc = o;     o += 32;               // own partial sums (8), three mbarriers (6), work item (2)
    L.off_gtab = o;     o += (size_t)N * 4;    // [4 coefficients][N columns]
    L.off_wf = o;       o += (size_t)2 * N;
    L.off_rho = o;      o += (size_t)2 * N;
    L.off_part = o;     o += (size_t)2 * OC_MAX_S * OC_NPART;
    L.off_rowpart = o;  o += (size_t)((R * L.CW + 3) & ~3);
    L.off_vtab = o;     o += (size_t)R * 8;
    L.off_rowaddr = o;  o += (size_t)R * 4;
    L.off_chunk = o;    o += (size_t)((3 * L.W * L.nch + 3) & ~3);   // per (walker, chunk): iy, run length walking down, walking up
    L.off_wred = o;     o += (size_t)OC_WARPS * 8;
    L.off_rowtab = o;   o += (size_t)(R + 2) * OC_ROWTAB;      // one spare entry before and after (prefetch)
    L.off_buf = o;      o += (size_t)(L.phys_rows + 1) * L.pitch;
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

// kick (shift by MM + t cells, Lagrange weights l already scaled by 1/C -- un-scaled with CLAMP,
// where the caller scales the results) and Fokker-Planck for the
// four cells g..g+3 of one row: b[i] = psi'(g - 4 + i), i = 0..11.  k[i] = kicked value at
// position g - 1 + i (zero outside the grid, A8).  The Fokker-Planck update (Eq. 15 + 3-point
// second difference, explicit Euler) is  out = k0 + G[-1] k[-1] + G[0] k0 + G[1] k[1] + G[2] k[2]
// with the per-column coefficients (G-1, G0, G1, G2): gt[j] holds coefficient j of the columns
// g..g+3 (all <= 1e-3, so the sum is exact to well below one ulp of k0).
template <int ORDER, int MM, bool CLAMP = false>
__device__ __forceinline__ void kick_fp4(const float (&b)[12], const float (&l)[ORDER], int g, int N,
                                         const float4 (&gt)[4], float (&out)[4])
{
    constexpr int O0 = (ORDER - 1) / 2;
    float k[7];
#pragma unroll
    for (int i = 0; i < 7; ++i) {
        const int i0 = 3 + i + MM - O0;
        float acc = l[0] * b[i0];
#pragma unroll
        for (int j = 1; j < ORDER; ++j) acc = fmaf(l[j], b[i0 + j], acc);
        // Eq. 14 (reading A9): limit to the interval of the two nodes that bracket the source point
        if (CLAMP) acc = fminf(fmaxf(acc, fminf(b[i0 + O0], b[i0 + O0 + 1])), fmaxf(b[i0 + O0], b[i0 + O0 + 1]));
        k[i] = acc;
    }
    if (g == 0) k[0] = 0.0f;
    if (g == N - 4) { k[5] = 0.0f; k[6] = 0.0f; }
    const float gm[4] = {gt[0].x, gt[0].y, gt[0].z, gt[0].w}, g0[4] = {gt[1].x, gt[1].y, gt[1].z, gt[1].w};
    const float g1[4] = {gt[2].x, gt[2].y, gt[2].z, gt[2].w}, g2[4] = {gt[3].x, gt[3].y, gt[3].z, gt[3].w};
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float incr = fmaf(g2[c], k[c + 3], fmaf(g1[c], k[c + 2], fmaf(g0[c], k[c + 1], gm[c] * k[c])));
        out[c] = k[c + 1] + incr;
    }
}
// any integer shift: reads the row in shared memory with bounds checks (rare: |shift| > 1 cell).
// Not inlined; weights by value, coefficients from the shared table [4][N], results through local
// memory, so that the fast path keeps its operands in registers.
template <int ORDER, bool CLAMP = false>
__device__ __noinline__ void kick_fp4_any(const float *row /* index 0 = y 0 */, float4 lw, int mm, int g, int N,
                                          const float *gtab, float *out)
{
    constexpr int O0 = (ORDER - 1) / 2;
    const float l[4] = {lw.x, lw.y, lw.z, lw.w};
    float k[7];
#pragma unroll 1
    for (int i = 0; i < 7; ++i) {
        const int y = g - 1 + i;
        float acc = 0.0f, lo = 0.0f, hi = 0.0f;
        for (int j = 0; j < ORDER; ++j) {
            const int s = y + mm - O0 + j;
            const float v = (s >= 0 && s < N) ? row[s] : 0.0f;
            acc = fmaf(l[j], v, acc);
            if (CLAMP && j == O0) lo = v;
            if (CLAMP && j == O0 + 1) hi = v;
        }
        if (CLAMP) acc = fminf(fmaxf(acc, fminf(lo, hi)), fmaxf(lo, hi));
        k[i] = (y >= 0 && y < N) ? acc : 0.0f;
    }
#pragma unroll 1
    for (int c = 0; c < 4; ++c) {
        const int y = g + c;
        out[c] = k[c + 1] + fmaf(gtab[3 * N + y], k[c + 3], fmaf(gtab[2 * N + y], k[c + 2],
                                                                  fmaf(gtab[N + y], k[c + 1], gtab[y] * k[c])));
    }
}

// ---------------------------------------------------------------- rotation of one walker
// A thread owns the columns y0 = 64 cw + 2 lane and y0 + 1.  The ORDER x (2 NP) register window
// holds ORDER source rows of the aligned column pairs that cover both cells' taps; it slides one
// row per target row.  PAR = (iy - O0) & 1 is the offset of cell y0's first tap inside the window,
// DIR the walk direction (+1: rows ascending).  At the start of a target row the window and the
// table row `tb` of that target are complete; its step loads those of the next target.
template <int ORDER, int PITCH, bool TAB, bool CLAMP>
struct Walker {
    static constexpr int O0 = (ORDER - 1) / 2;
    static constexpr int NPMAX = (ORDER + 3) / 2;          // column pairs of the window (PAR = 1)
    static constexpr int CH = oc_chunk_rows(ORDER);
    static constexpr int NTB = TAB ? 2 * ORDER + 1 : 2;
    static constexpr int P4 = PITCH * 4;
    float win[ORDER][2 * NPMAX];
    float M0[ORDER], M0p[ORDER], M1[ORDER], M1p[ORDER];    // TAB: weights along q of both columns and their t-derivatives
                                                           // !TAB: M0[0] = b Y0 - ix, M1[0] = b Y1 - ix
    float ey0, ey1;                                        // TAB: a (Y - Ymid); else a Y
    float a;                                               // cos(dphi) - 1 (only !TAB)
    float tb[NTB];                                         // TAB: L[ORDER], L'[ORDER], a (X - Xc); else X, d X - iy
    float rs[4];                                           // row sums of the current chunk

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
    // the table row at `tab` (layouts: onchip_tables in vfps_api.cu)
    __device__ __forceinline__ void load_tab(uint32_t tab)
    {
        if (TAB) {
            if (ORDER == 4) {
                // L0 L1 L2 L3 | L'1 L'2 L'3 L'0: a 128-bit load fills four consecutive registers and the
                // register file has four banks (register number mod 4, measured: csrc/peaks); L'_j
                // rotated by one keeps L_j and L'_j, two operands of one FMA, out of the same bank
                const float4 v = lds4(tab), w = lds4(tab + 16);
                tb[0] = v.x; tb[1] = v.y; tb[2] = v.z; tb[3] = v.w; tb[5] = w.x; tb[6] = w.y; tb[7] = w.z; tb[4] = w.w;
                tb[2 * ORDER] = lds(tab + 32);
            } else if (ORDER == 3) {
                const float4 v = lds4(tab), w = lds4(tab + 16);            // L0 L1 L2 ex | L'0 L'1 L'2 -
                tb[0] = v.x; tb[1] = v.y; tb[2] = v.z; tb[2 * ORDER] = v.w; tb[3] = w.x; tb[4] = w.y; tb[5] = w.z;
            } else {
                const float4 v = lds4(tab);                                 // L0 L1 L'0 L'1
                tb[0] = v.x; tb[1] = v.y; tb[2] = v.z; tb[3] = v.w;
                tb[2 * ORDER] = lds(tab + 16);
            }
        } else {
            const float2 xv = lds2(tab + 32);                               // X, d X - iy
            tb[0] = xv.x; tb[1] = xv.y;
        }
    }
    // weights of both cells from the table row in tb
    __device__ __forceinline__ void weights(float (&lx0)[ORDER], float (&lx1)[ORDER], float (&ly0)[ORDER],
                                            float (&ly1)[ORDER]) const
    {
        if (TAB) {
            const float ex = tb[2 * ORDER];
#pragma unroll
            for (int j = 0; j < ORDER; ++j) {
                ly0[j] = fmaf(ey0, tb[ORDER + j], tb[j]);
                ly1[j] = fmaf(ey1, tb[ORDER + j], tb[j]);
                lx0[j] = fmaf(ex, M0p[j], M0[j]);
                lx1[j] = fmaf(ex, M1p[j], M1[j]);
            }
        } else {
            lagrange<ORDER>(fmaf(a, tb[0], M0[0]), lx0);
            lagrange<ORDER>(fmaf(a, tb[0], M1[0]), lx1);
            lagrange<ORDER>(tb[1] + ey0, ly0);
            lagrange<ORDER>(tb[1] + ey1, ly1);
        }
    }
    // inner products of one window row with the weights along p of both cells
    template <int PAR>
    __device__ __forceinline__ void inner(int slot, const float (&ly0)[ORDER], const float (&ly1)[ORDER], float &r0,
                                          float &r1) const
    {
        const float(&wr)[2 * NPMAX] = win[slot];
        r0 = ly0[0] * wr[PAR]; r1 = ly1[0] * wr[PAR + 1];
#pragma unroll
        for (int j = 1; j < ORDER; ++j) {
            r0 = fmaf(ly0[j], wr[PAR + j], r0);
            r1 = fmaf(ly1[j], wr[PAR + 1 + j], r1);
        }
    }
    // start of a run of chunks: the whole window and the table row of the first target.
    // src = address of window column 0 of tap row i = 0 of that target, tab = its table row.
    template <int PAR>
    __device__ __forceinline__ void start(uint32_t src, uint32_t tab)
    {
#pragma unroll
        for (int i = 0; i < ORDER; ++i) load_row<PAR>(i, src + (uint32_t)(i * P4));
        load_tab(tab);
    }
    // target row SUB of a chunk.  Tap row i lives in slot (SUB + i) % ORDER (DIR > 0) or
    // (i - SUB) mod ORDER (DIR < 0).  The tap row that leaves the window (i = 0 walking down,
    // i = ORDER - 1 walking up) is consumed first; its slot then receives the entering row of the
    // next target, and tb the next table row, while the rest of this target is computed.
    template <int PAR, int DIR, int SUB, class OUT>
    __device__ __forceinline__ void row_step(uint32_t src, const OUT &dst, uint32_t tab)
    {
        constexpr int SLOT0 = (DIR > 0) ? (SUB % ORDER) : ((ORDER - SUB % ORDER) % ORDER);
        constexpr int IL = (DIR > 0) ? 0 : ORDER - 1;
        float lx0[ORDER], lx1[ORDER], ly0[ORDER], ly1[ORDER];
        weights(lx0, lx1, ly0, ly1);
        load_tab(tab + (uint32_t)(DIR * (SUB + 1) * (OC_ROWTAB * 4)));
        // Eq. 14 (reading A9): interval of the 2 x 2 nodes around each source point -- tap rows O0, O0 + 1
        // (taken before the window slides), columns O0, O0 + 1 of each cell's stencil
        float lo0 = 0.0f, hi0 = 0.0f, lo1 = 0.0f, hi1 = 0.0f;
        if (CLAMP) {
            const float(&wa)[2 * NPMAX] = win[(SLOT0 + O0) % ORDER];
            const float(&wb)[2 * NPMAX] = win[(SLOT0 + O0 + 1) % ORDER];
            float cmn[3], cmx[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) { cmn[k] = fminf(wa[PAR + O0 + k], wb[PAR + O0 + k]); cmx[k] = fmaxf(wa[PAR + O0 + k], wb[PAR + O0 + k]); }
            lo0 = fminf(cmn[0], cmn[1]); hi0 = fmaxf(cmx[0], cmx[1]);
            lo1 = fminf(cmn[1], cmn[2]); hi1 = fmaxf(cmx[1], cmx[2]);
        }
        float r0[ORDER], r1[ORDER];
        inner<PAR>((SLOT0 + IL) % ORDER, ly0, ly1, r0[IL], r1[IL]);
        load_row<PAR>((SLOT0 + IL) % ORDER, src + (uint32_t)((DIR > 0 ? SUB + ORDER : -(SUB + 1)) * P4));
#pragma unroll
        for (int i = 0; i < ORDER; ++i)
            if (i != IL) inner<PAR>((SLOT0 + i) % ORDER, ly0, ly1, r0[i], r1[i]);
        float a0 = lx0[0] * r0[0], a1 = lx1[0] * r1[0];
#pragma unroll
        for (int i = 1; i < ORDER; ++i) { a0 = fmaf(lx0[i], r0[i], a0); a1 = fmaf(lx1[i], r1[i], a1); }
        if (CLAMP) { a0 = fminf(fmaxf(a0, lo0), hi0); a1 = fminf(fmaxf(a1, lo1), hi1); }
        dst.template put<DIR * SUB>(a0, a1);
        rs[SUB] = a0 + a1;
    }
    template <int PAR, int DIR, class OUT, int SUB = 0>
    __device__ __forceinline__ void chunk(uint32_t src, const OUT &dst, uint32_t tab)
    {
        row_step<PAR, DIR, SUB>(src, dst, tab);
        if constexpr (SUB + 1 < CH) chunk<PAR, DIR, OUT, SUB + 1>(src, dst, tab);
    }
    // a ragged last chunk: only the first nrows (< CH) target rows exist (warp-uniform)
    template <int PAR, int DIR, class OUT, int SUB = 0>
    __device__ __forceinline__ void chunk_n(uint32_t src, const OUT &dst, uint32_t tab, int nrows)
    {
        if (SUB < nrows) row_step<PAR, DIR, SUB>(src, dst, tab); else rs[SUB] = 0.0f;
        if constexpr (SUB + 1 < CH) chunk_n<PAR, DIR, OUT, SUB + 1>(src, dst, tab, nrows);
    }
};

// where a walker puts the two rotated cells of target row R (relative to the chunk's first target)
template <int P4>
struct OutShared {                     // shared memory, row pitch P4 bytes
    uint32_t a;
    template <int R>
    __device__ __forceinline__ void put(float x, float y) const { sts2(a + (uint32_t)(R * P4), x, y); }
};
struct OutSharedRt {                   // shared memory, row pitch p4 bytes known at run time
    uint32_t a, p4;
    template <int R>
    __device__ __forceinline__ void put(float x, float y) const { sts2(a + (uint32_t)R * p4, x, y); }
};
struct OutGlobal {                     // global memory, row pitch n floats
    float *p;
    int n;
    template <int R>
    __device__ __forceinline__ void put(float x, float y) const
    {
        *reinterpret_cast<float2 *>(p + (ptrdiff_t)R * n) = make_float2(x, y);
    }
};

// one cell with its own floors and a full window (rows where a floor changes inside the thread's
// columns or along the chunk)
template <int ORDER, int PITCH, bool CLAMP>
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
    if (CLAMP) {
        const float a = lds(base + (O0 * PITCH + O0) * 4), b = lds(base + (O0 * PITCH + O0 + 1) * 4);
        const float c = lds(base + ((O0 + 1) * PITCH + O0) * 4), d = lds(base + ((O0 + 1) * PITCH + O0 + 1) * 4);
        acc = fminf(fmaxf(acc, fminf(fminf(a, b), fminf(c, d))), fmaxf(fmaxf(a, b), fmaxf(c, d)));
    }
    return acc;
}

#define OC_STAMP(k) VFPS_STAMP(A.dbg, step, k)

// ---------------------------------------------------------------- the persistent kernel
// grid = S * (concurrent clusters), cluster = S CTAs, block = 512.  Clusters take work items
// (chunk j of member m, in the order j * members + m) from a queue in global memory; chunk j of a
// member starts after its chunk j-1 has been stored (member_done).
template <int ORDER, int N, bool TAB, bool CLAMP = false>
__global__ void __launch_bounds__(OC_THREADS, 1)
k_onchip_step(GridConst G, OnchipArgs A)
{
    static_assert(N >= 64 && N % 64 == 0, "N must be a multiple of 64");
    constexpr int PITCH = N + 2 * OC_PADC;
    constexpr int P4 = PITCH * 4;
    constexpr int O0 = (ORDER - 1) / 2;
    constexpr int CW = N / 64;
    constexpr int CH = oc_chunk_rows(ORDER);
    // kick pass: a warp takes a block of up to 256 columns of a row; a lane owns the 4-cell granules 4 lane + 128 k
    // of the block.  N = 512: two warps per row, each keeps its half for the whole pass, so the Fokker-Planck
    // coefficients of a lane's columns (2 x 4 float4) stay in registers for every N.
    constexpr int NBLK = (N > 256) ? N / 256 : 1;          // column blocks (= warps) per row
    constexpr int NG = (N >= 256) ? 2 : 1;                 // granules per lane and block
    constexpr int KL = (N >= 128) ? 32 : N / 4;            // active lanes in the kick pass
    constexpr int NW = N / 128 > 0 ? N / 128 : 1;          // float4 groups of rho per lane in the wake
    constexpr unsigned FULL = 0xffffffffu;
    using Wk = Walker<ORDER, PITCH, TAB, CLAMP>;

    cg::cluster_group cluster = cg::this_cluster();
    const int S = A.S, R = A.R, H = G.H;
    const OnchipLayout LY = onchip_layout(N, S, H, ORDER);
    const int W = LY.W, RPW = LY.RPW, D = LY.D, KC = LY.KC, nch = LY.nch, SEG = LY.seg_rows;
    const int rank = (int)cluster.block_rank();
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int x0 = rank * R;

    extern __shared__ __align__(16) float smem[];
    float *buf = smem + LY.off_buf;
    float *rowtab_s = smem + LY.off_rowtab + OC_ROWTAB;    // entry 0 = first own row (one spare entry before)
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
    const uint32_t sVtab = smem_u32(vtab), sMisc = smem_u32(misc), sRowaddr = smem_u32(rowaddr), sGtab = smem_u32(gtab);
    const uint32_t sRowpart = smem_u32(rowpart);
    const uint32_t mbRho0 = sMisc + 32, mbHalo = sMisc + 48;        // mbRho[p] = mbRho0 + 8 p
    const int nbrs = (rank > 0 ? 1 : 0) + (rank < S - 1 ? 1 : 0);
    const uint32_t bytesRho = (uint32_t)(N + S * OC_NPART) * 4u, bytesPart = (uint32_t)(S * OC_NPART) * 4u;
    const uint32_t bytesHalo = (uint32_t)(nbrs * H * N) * 4u;

    // ---- rotation role: walker wk, columns y0, y0 + 1
    const int wk = warp / CW, cw = warp % CW;
    const bool walker_on = wk < W;
    const int y0 = 64 * cw + 2 * lane;
    const int wb = wk * RPW;                               // first CTA-local row of the walker
    Wk wkr;
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
        wkr.ey0 = TAB ? G.a * ((float)y0 - 0.5f * (float)(N - 1)) : ct0[1];
        wkr.ey1 = TAB ? G.a * ((float)(y0 + 1) - 0.5f * (float)(N - 1)) : ct1[1];
        wkr.a = G.a;
        if (!cols_ok) ixc = 0;
    }
    const uint32_t segA = sBuf + (uint32_t)(wk * SEG) * P4;     // physical row 0 of the walker's segment
    // lanes 8 k (k < CH) publish the row sum of the chunk's k-th target row
    const bool rs_writer = ((lane & 7) == 0) && ((lane >> 3) < CH);

    // ---- one-time set-up: zero the buffer (pads stay zero for ever), tables, barriers
    for (int i = tid; i < (LY.phys_rows + 1) * PITCH; i += OC_THREADS) buf[i] = 0.0f;
    for (int i = tid; i < (R + 2) * OC_ROWTAB; i += OC_THREADS) {
        const int gi = (x0 - 1) * OC_ROWTAB + i;           // entries x0 - 1 .. x0 + R (the outer two are only ever prefetched)
        rowtab_s[i - OC_ROWTAB] = (gi >= 0 && gi < N * OC_ROWTAB) ? A.rowtab[gi] : 0.0f;
    }
    {
        // Fokker-Planck coefficients by column, transposed: gtab[j][y], j = 0..3 <-> G-1, G0, G1, G2
        const float c1 = G.fp_b / (6.0f * G.dp), c2 = G.fp_b / (G.dp * G.dp);
        for (int y = tid; y < N; y += OC_THREADS) {
            const float c1p = c1 * fmaf((float)y, G.dp, G.p_min);
            gtab[y] = fmaf(-2.0f, c1p, c2);
            gtab[N + y] = fmaf(-3.0f, c1p, fmaf(-2.0f, c2, G.fp_b));
            gtab[2 * N + y] = fmaf(6.0f, c1p, c2);
            gtab[3 * N + y] = -c1p;
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
        if ((c + 1) * CH <= RPW) {
            iy = __float_as_int(rowtab_s[(w * RPW + c * CH) * OC_ROWTAB + 10]);
            for (int k = 1; k < CH; ++k)
                if (__float_as_int(rowtab_s[(w * RPW + c * CH + k) * OC_ROWTAB + 10]) != iy) iy = OC_BAD;
        }
        chunkinfo[i] = iy;
    }
    __syncthreads();
    // ... and how many chunks with the same floors follow it in either walk direction (the window slides through the
    // whole run): found once here, not by a chain of dependent loads in front of every step's rotation
    for (int i = tid; i < W * nch; i += OC_THREADS) {
        const int w = i / nch, c = i - w * nch, iy = chunkinfo[i];
        int nd = 1, nu = 1;
        if (iy != OC_BAD) {
            while (c + nd < nch && chunkinfo[w * nch + c + nd] == iy) ++nd;
            while (c - nu >= 0 && chunkinfo[w * nch + c - nu] == iy) ++nu;
        }
        chunkinfo[W * nch + 2 * i] = nd;
        chunkinfo[W * nch + 2 * i + 1] = nu;
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
                const int dir = p ? -1 : 1;
                int kk = 0;                                // chunks since the last named barrier
                int ci = 0;                                // chunk index in walk order
                while (ci < nch) {
                    const int c = p ? nch - 1 - ci : ci;
                    const int iy = chunkinfo[wk * nch + c];
                    int nrun = 1;                          // chunks handled in this round
                    if (cols_ok && iy != OC_BAD) {
                        // ---- a run of chunks with the same floors: the window slides through all of them
                        nrun = chunkinfo[W * nch + 2 * (wk * nch + c) + p];
                        const int par = (iy - O0) & 1;
                        const int v0 = p ? c * CH + CH - 1 : c * CH;                   // first target row in walk order
                        // window column 0 = grid column y0 + iy - O0 - par
                        uint32_t src = rbase + (uint32_t)((v0 + ixc - O0) * P4 + (OC_PADC + y0 + iy - O0 - par) * 4);
                        uint32_t dst = rbase + (uint32_t)((v0 + dsh) * P4 + (OC_PADC + y0) * 4);
                        uint32_t tab = sRowtab + (uint32_t)((wb + v0) * OC_ROWTAB * 4);
                        // lane 8 k publishes the sum of the k-th target row of every chunk
                        uint32_t rp = sRowpart + (uint32_t)(((wb + v0 + dir * (lane >> 3)) * CW + cw) * 4);
#define OC_RUN(PAR_, DIR_)                                                                                   \
    do {                                                                                                      \
        wkr.template start<PAR_>(src, tab);                                                                   \
        for (int q = 0; q < nrun; ++q) {                                                                      \
            wkr.template chunk<PAR_, DIR_>(src, OutShared<P4>{dst}, tab);                                     \
            if (CH < 4) wkr.rs[3] = 0.0f;                                                                     \
            const float tot = warp_reduce_transposed<4>(wkr.rs, lane);                                        \
            if (rs_writer) sts(rp, tot);                                                                      \
            src += (uint32_t)(DIR_ * CH * P4); dst += (uint32_t)(DIR_ * CH * P4);                             \
            tab += (uint32_t)(DIR_ * CH * OC_ROWTAB * 4); rp += (uint32_t)(DIR_ * CH * CW * 4);               \
            if (++kk == KC) {                                                                                 \
                kk = 0;                                                                                       \
                if (ci + q + 1 < nch) { if (CW > 1) named_barrier(1 + wk, CW * 32); else __syncwarp(); }      \
            }                                                                                                 \
        }                                                                                                     \
    } while (0)
                        if (p == 0) { if (par) OC_RUN(1, 1); else OC_RUN(0, 1); }
                        else        { if (par) OC_RUN(1, -1); else OC_RUN(0, -1); }
#undef OC_RUN
                    } else {
                        // ---- cell by cell: a floor changes inside the chunk or the thread's columns, or a ragged last chunk
                        const uint32_t gbase = rbase + (uint32_t)(OC_PADC * 4);
                        const int vlo = c * CH, nrow = min(CH, RPW - vlo);
                        float rs4[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
                        for (int s = 0; s < CH; ++s) {
                            if (s < nrow) {
                                const int v = p ? vlo + nrow - 1 - s : vlo + s;
                                const float o0 = rotate_cell_generic<ORDER, PITCH, CLAMP>(G, gbase, v, x0 + wb + v, y0);
                                const float o1 = rotate_cell_generic<ORDER, PITCH, CLAMP>(G, gbase, v, x0 + wb + v, y0 + 1);
                                sts2(rbase + (uint32_t)((v + dsh) * P4 + (OC_PADC + y0) * 4), o0, o1);
                                rs4[s] = o0 + o1;
                            }
                        }
                        const float tot = warp_reduce_transposed<4>(rs4, lane);
                        const int s = lane >> 3;
                        if (rs_writer && s < nrow) {
                            const int v = p ? vlo + nrow - 1 - s : vlo + s;
                            rowpart[(wb + v) * CW + cw] = tot;
                        }
                        if (++kk == KC) {
                            kk = 0;
                            if (ci + 1 < nch) { if (CW > 1) named_barrier(1 + wk, CW * 32); else __syncwarp(); }
                        }
                    }
                    ci += nrun;
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
                    // thread t < R: the sum of row t's CW partials (one vector load, lane stride CW floats: no bank
                    // conflicts); the four lanes of a row quad gather its four sums and share the destinations
                    float pv = 0.0f;
                    if (tid < R) {
                        float pc[CW];
                        const uint32_t a = sRowpart + (uint32_t)(tid * CW) * 4u;
                        if (CW >= 4) {
#pragma unroll
                            for (int c = 0; c < CW; c += 4) {
                                const float4 v = lds4(a + 4u * (uint32_t)c);
                                pc[c] = v.x; pc[(c + 1) % CW] = v.y; pc[(c + 2) % CW] = v.z; pc[(c + 3) % CW] = v.w;
                            }
                        } else if (CW == 2) {
                            const float2 v = lds2(a);
                            pc[0] = v.x; pc[CW - 1] = v.y;
                        } else {
                            pc[0] = lds(a);
                        }
                        float sum = 0.0f;
#pragma unroll
                        for (int c = 0; c < CW; ++c) sum += pc[c];
                        pv = sum * G.dp;
                    }
                    const int l4 = lane & ~3;
                    const float4 quad = make_float4(__shfl_sync(FULL, pv, l4), __shfl_sync(FULL, pv, l4 + 1),
                                                    __shfl_sync(FULL, pv, l4 + 2), __shfl_sync(FULL, pv, l4 + 3));
                    if (tid < R) {
                        const uint32_t dsta = rb + (uint32_t)(x0 + (tid & ~3)) * 4u;
                        for (int dd = lane & 3; dd < S; dd += 4) st_async4(mapa(dsta, dd), quad, mapa(mb, dd));
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
                        float vt[4] = {0.0f, 0.0f, 0.0f, 0.0f};        // CLAMP: transposed wake, sum_x' w[x' - x] rho_x'
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
                                    if (CLAMP) {
                                        // w[(x' + c) - (x + k)] at index B + c - k, B = 4 lane + 128 j - x + N - 1 = 3 mod 4
                                        const int Bq = 4 * lane + 128 * j - x + N - 1;
                                        const float4 ul = lds4(sWf + (uint32_t)(Bq - 3) * 4u);
                                        const float4 uh = (Bq + 1 < 2 * N) ? lds4(sWf + (uint32_t)(Bq + 1) * 4u)
                                                                           : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                                        const float u7[8] = {ul.x, ul.y, ul.z, ul.w, uh.x, uh.y, uh.z, uh.w};
#pragma unroll
                                        for (int k = 0; k < 4; ++k)
#pragma unroll
                                            for (int c = 0; c < 4; ++c) vt[k] = fmaf(u7[3 + c - k], rc[c], vt[k]);
                                    }
                                }
                            }
                        }
                        const float Vr = warp_reduce_transposed<4>(vq, lane);     // lanes 8k .. 8k+7 hold row x + k
                        const float Vtr = CLAMP ? warp_reduce_transposed<4>(vt, lane) : 0.0f;
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
                            for (int j = 0; j < ORDER; ++j) pl[j] = CLAMP ? l[j] : l[j] * sc;   // CLAMP: the kick scales its results
                            sts4(sVtab + (uint32_t)r * 32u, make_float4(pl[0], pl[1], pl[2], pl[3]));
                            if (CLAMP) {
                                // The clamped kick is not conservative: the profile after it, rho', differs from rho.
                                // CSR power of the END-of-step density to first order in rho' - rho (the neglected
                                // term is quadratic, < 1e-6 relative):  sum rho' V' = sum rho V + sum (rho' - rho) U,
                                // U = V + Vt.  Row term: rho_x V_x - rho_x U_x = -rho_x Vt_x; the kick adds dp U_x
                                // times its row sums.
                                const float Vt = Vtr * sc;
                                sts4(sVtab + (uint32_t)r * 32u + 16u, make_float4(__int_as_float(mm), -rho_x * Vt, G.dp * (V + Vt), 0.0f));
                            } else {
                                sts2(sVtab + (uint32_t)r * 32u + 16u, __int_as_float(mm), rho_x * V);
                            }
                        }
                    }
                }
            }
            OC_STAMP(5);
            __syncthreads();
            // ================= 5. kick a4 + Fokker-Planck a5 in place (parity p ^ 1), aprons, moments
            {
                const int pshift = (p ^ 1) ? D * P4 : 0;       // parity 1 lies D rows above the parity-0 slot
                float cs[NG][4];
#pragma unroll
                for (int k = 0; k < NG; ++k)
#pragma unroll
                    for (int c = 0; c < 4; ++c) cs[k][c] = 0.0f;
                float q1 = 0.0f, q2 = 0.0f, pw = 0.0f;
                const int blk = warp % NBLK;                  // this warp's column block
                // Fokker-Planck coefficients of the lane's columns: registers for the whole pass
                float4 gt[NG][4];
                if (lane < KL) {
#pragma unroll
                    for (int k = 0; k < NG; ++k)
#pragma unroll
                        for (int j = 0; j < 4; ++j) gt[k][j] = lds4(sGtab + (uint32_t)((j * N + 256 * blk + 4 * lane + 128 * k) * 4));
                }
                const uint32_t mbUp = (rank > 0) ? mapa(mbHalo, rank - 1) : 0u, mbDn = (rank < S - 1) ? mapa(mbHalo, rank + 1) : 0u;
                const uint32_t lane_off = (uint32_t)(1024 * blk + 16 * lane);
                float Xf = (float)(x0 + warp / NBLK) - xc;
                for (int r = warp / NBLK; r < R; r += OC_WARPS / NBLK, Xf += (float)(OC_WARPS / NBLK)) {
                    const float4 lw = lds4(sVtab + (uint32_t)r * 32u);
                    float2 mv;
                    float dpU = 0.0f;                          // CLAMP: dp (V + Vt) of the row
                    if (CLAMP) {
                        const float4 m4 = lds4(sVtab + (uint32_t)r * 32u + 16u);
                        mv = make_float2(m4.x, m4.y); dpU = m4.z;
                    } else {
                        mv = lds2(sVtab + (uint32_t)r * 32u + 16u);
                    }
                    const int mm = __float_as_int(mv.x);
                    const int4 ra = ldsi4(sRowaddr + (uint32_t)r * 16u);
                    const uint32_t own = sBuf + (uint32_t)(ra.x - pshift) + lane_off;     // cell 4 lane of the row
                    float o[NG][4];
                    if (lane < KL) {
                        if (mm >= -2 && mm <= 0) {
                            const float lws[4] = {lw.x, lw.y, lw.z, lw.w};
                            float l[ORDER];
#pragma unroll
                            for (int j = 0; j < ORDER; ++j) l[j] = lws[j];
                            float b[NG][12];
#pragma unroll
                            for (int k = 0; k < NG; ++k)
#pragma unroll
                                for (int i = 0; i < 3; ++i) {
                                    const float4 v = lds4(own + (uint32_t)(512 * k + 16 * i - 16));
                                    b[k][4 * i] = v.x; b[k][4 * i + 1] = v.y; b[k][4 * i + 2] = v.z; b[k][4 * i + 3] = v.w;
                                }
#pragma unroll
                            for (int k = 0; k < NG; ++k) {
                                const int g = 256 * blk + 4 * lane + 128 * k;
                                if (mm == 0) kick_fp4<ORDER, 0, CLAMP>(b[k], l, g, N, gt[k], o[k]);
                                else if (mm == -1) kick_fp4<ORDER, -1, CLAMP>(b[k], l, g, N, gt[k], o[k]);
                                else kick_fp4<ORDER, -2, CLAMP>(b[k], l, g, N, gt[k], o[k]);
                            }
                        } else {
                            const float *rowp = buf + ((ra.x - pshift) >> 2);
#pragma unroll
                            for (int k = 0; k < NG; ++k) {
                                float tmp[4];
                                kick_fp4_any<ORDER, CLAMP>(rowp, lw, mm, 256 * blk + 4 * lane + 128 * k, N, gtab, tmp);
#pragma unroll
                                for (int c = 0; c < 4; ++c) o[k][c] = tmp[c];
                            }
                        }
                        if (CLAMP) {
#pragma unroll
                            for (int k = 0; k < NG; ++k)
#pragma unroll
                                for (int c = 0; c < 4; ++c) o[k][c] *= sc;
                        }
                    }
                    // every lane has read the row before anyone overwrites it (N = 512: both warps of the row)
                    if (NBLK > 1) named_barrier(8 + warp / NBLK, 32 * NBLK); else __syncwarp();
                    if (lane < KL) {
#pragma unroll
                        for (int k = 0; k < NG; ++k) sts4(own + (uint32_t)(512 * k), make_float4(o[k][0], o[k][1], o[k][2], o[k][3]));
                        if ((ra.y | ra.z) != 0) {
                            // boundary row of a walker: copy into the neighbour's apron (local, or in the next CTA)
                            if (ra.y != 0) {
                                uint32_t aup = sBuf + (uint32_t)(ra.y - pshift) + lane_off;
                                if (ra.w & 1) {
                                    aup = mapa(aup, rank - 1);
#pragma unroll
                                    for (int k = 0; k < NG; ++k) st_async4(aup + (uint32_t)(512 * k), make_float4(o[k][0], o[k][1], o[k][2], o[k][3]), mbUp);
                                } else {
                                    const float z = (ra.w & 4) ? 0.0f : 1.0f;
#pragma unroll
                                    for (int k = 0; k < NG; ++k) sts4(aup + (uint32_t)(512 * k), make_float4(z * o[k][0], z * o[k][1], z * o[k][2], z * o[k][3]));
                                }
                            }
                            if (ra.z != 0) {
                                uint32_t adn = sBuf + (uint32_t)(ra.z - pshift) + lane_off;
                                if (ra.w & 2) {
                                    adn = mapa(adn, rank + 1);
#pragma unroll
                                    for (int k = 0; k < NG; ++k) st_async4(adn + (uint32_t)(512 * k), make_float4(o[k][0], o[k][1], o[k][2], o[k][3]), mbDn);
                                } else {
                                    const float z = (ra.w & 8) ? 0.0f : 1.0f;
#pragma unroll
                                    for (int k = 0; k < NG; ++k) sts4(adn + (uint32_t)(512 * k), make_float4(z * o[k][0], z * o[k][1], z * o[k][2], z * o[k][3]));
                                }
                            }
                        }
                        float q0 = 0.0f;
#pragma unroll
                        for (int k = 0; k < NG; ++k)
#pragma unroll
                            for (int c = 0; c < 4; ++c) { cs[k][c] += o[k][c]; q0 += o[k][c]; }
                        const float tq = q0 * Xf;
                        q1 += tq; q2 = fmaf(tq, Xf, q2);
                        if (CLAMP) pw = fmaf(q0, dpU, pw);
                        if (lane == 0 && blk == 0) pw += mv.y;
                    }
                }
                OC_STAMP(6);
                // ---- per-warp sums -> wred; s0, s1, s2 from the column sums
                float v8[8] = {0.0f, 0.0f, 0.0f, q1, q2, pw, 0.0f, 0.0f};
                if (lane < KL) {
#pragma unroll
                    for (int k = 0; k < NG; ++k)
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            const float yy = (float)(256 * blk + 4 * lane + 128 * k + c) - yc;
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
