// vfps_cluster.cuh -- persistent thread-block-cluster engine (sm_100a).
//
// One cluster of S CTAs advances one simulation by all n steps of a vfps_step call with psi
// resident in (distributed) shared memory; HBM is touched at entry (load psi), at exit (store psi)
// and for the six diagnostics floats per step.  CTA `rank` owns the q-rows
// x in [rank*R, (rank+1)*R), R = N/S, of two buffers:
//   bufA  psi_t (un-normalised), own rows plus H halo rows on each side (neighbours push them)
//   bufB  psi'  (rotated, un-scaled), own rows
// Rows are stored with CL_PAD zero floats on both sides, so every out-of-grid tap along p reads 0.
//
// One split step:
//   1 rotation a1: bufA -> bufB.  A thread keeps column y and walks down the rows with a sliding
//     ORDER x ORDER register window (ORDER new shared-memory loads per cell instead of ORDER^2).
//   2 projection a2: one warp per row sums bufB -> rho_x (times dp and the renormalisation scalar)
//     and stores it into the rho array of EVERY CTA of the cluster (DSMEM all-gather).
//   -- cluster barrier 1 --
//   3 wake a3: V_x = sum_x' w[x-x'] rho_x' for the own rows (direct convolution, Eq. 4, with
//     the wake function w = Re IDFT(Z) computed once at create); the same warp then
//   4 kick a4 + Fokker-Planck a5 on its row in registers, bufB -> bufA, pushing the first/last H
//     rows into the neighbours' halo; partial sums for a6.
//   5 the partial sums of every CTA are broadcast to every CTA.
//   -- cluster barrier 2 --
//   6 a6: every CTA forms C and the scalar 1/C; rank 0 writes the diagnostics row.
#pragma once
#include "vfps_common.cuh"

#include <cooperative_groups.h>

namespace vfps {

namespace cg = cooperative_groups;

constexpr int CL_THREADS = 512;
constexpr int CL_WARPS = CL_THREADS / 32;
constexpr int CL_PAD = 4;           // zero floats left and right of every staged row (>= halo H)
constexpr int CL_MAX_S = 16;        // largest cluster (non-portable size)
constexpr int CL_NPART = 8;         // partial sums per CTA per step

struct ClusterArgs {
    float *psi;          // [members][N][N] in/out, un-normalised
    float *scale;        // [members] in/out: 1/C of the last step
    const float *wfun;   // [members][2N] wake function, lag d at index d + N - 1; nullptr = no wake
    float *diag;         // [nsteps][members][6] or nullptr
    int members;
    int nsteps;
    int S;               // CTAs per cluster
    int R;               // rows per CTA = N / S
    long long *dbg;      // nullptr, or [CTA][64 steps][8] clock64 stamps of the packed kernel's phases (debug aid)
};

__host__ __device__ inline size_t cluster_smem_floats(int N, int S, int H)
{
    const int R = N / S, pitch = N + 2 * CL_PAD;
    return (size_t)(R + 2 * H) * pitch      // bufA
           + (size_t)R * pitch              // bufB
           + 2 * (size_t)N                  // wake function
           + 2 * (size_t)N                  // rho (all rows), two parities
           + 2 * CL_MAX_S * CL_NPART        // partial sums of all CTAs, two parities
           + CL_WARPS * 8 + 16;             // block reduction scratch, five mbarriers
}

// floor for |v| < 2^22 on the FMA pipe: v + 1.5*2^23 rounded toward -inf has floor(v) in its low
// mantissa bits.  (FRND/F2I run at a quarter of the FFMA rate.)
constexpr float CL_MAGIC = 12582912.0f;
constexpr int CL_IMAGIC = 0x4B400000;

__device__ __forceinline__ void floor_frac(float v, int &i, float &t)
{
    const float r = __fadd_rd(v, CL_MAGIC);
    i = __float_as_int(r) - CL_IMAGIC;
    t = v - (r - CL_MAGIC);
}

// ---- shared-memory / DSMEM / mbarrier primitives (32-bit shared-window addresses)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ float lds(uint32_t a)      // constant offsets fold into [R + imm]
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ float4 lds4(uint32_t a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts(uint32_t a, float v)
{
    asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory");
}
__device__ __forceinline__ void sts4(uint32_t a, float4 v)
{
    asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
// address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa(uint32_t a, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}
// asynchronous remote stores that count their bytes on an mbarrier of the destination CTA: the
// receiver's wait on that mbarrier is the only synchronisation (no cluster barrier, no fence)
__device__ __forceinline__ void st_async(uint32_t ra, float v, uint32_t rmbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f32 [%0], %1, [%2];" ::"r"(ra), "f"(v),
                 "r"(rmbar)
                 : "memory");
}
__device__ __forceinline__ void st_async4(uint32_t ra, float4 v, uint32_t rmbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1,%2,%3,%4}, [%5];" ::"r"(ra),
                 "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "r"(rmbar)
                 : "memory");
}
__device__ __forceinline__ void mbar_init(uint32_t mbar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t mbar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "DONE:\n\t"
        "}" ::"r"(mbar), "r"(parity)
        : "memory");
}

// kick (shift by mm + t cells, Lagrange weights l already scaled) and Fokker-Planck for the four
// cells g..g+3 of one row held in registers: b[i] = psi'(g - 4 + i), i = 0..11.
// MM = integer part of the shift (compile time).  Returns the four new values and adds to the
// moment sums.  k[i] = kicked value at position g - 1 + i, zero outside the grid (ghosts, A8).
// CLAMP: Eq. 14 (reading A9) -- the kicked value is limited to the interval of its two bracketing
// nodes (taps O0 and O0 + 1 of its stencil); only valid with un-scaled weights.
template <int ORDER, int MM, bool CLAMP = false>
__device__ __forceinline__ void kick_fp_granule(const float (&b)[12], const float (&l)[ORDER], int g, int N,
                                                float fp_b, float c2, const float (&c1p)[4],
                                                float (&out)[4])
{
    constexpr int O0 = (ORDER - 1) / 2;
    float k[7];
#pragma unroll
    for (int i = 0; i < 7; ++i) {
        // position g - 1 + i, first tap at g - 1 + i + MM - O0  ->  b index 3 + i + MM - O0
        const int i0 = 3 + i + MM - O0;
        float acc = l[0] * b[i0];
#pragma unroll
        for (int j = 1; j < ORDER; ++j) acc = fmaf(l[j], b[i0 + j], acc);
        if (CLAMP) acc = fminf(fmaxf(acc, fminf(b[i0 + O0], b[i0 + O0 + 1])), fmaxf(b[i0 + O0], b[i0 + O0 + 1]));
        k[i] = acc;
    }
    if (g == 0) k[0] = 0.0f;
    if (g == N - 4) { k[5] = 0.0f; k[6] = 0.0f; }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float fm1 = k[c], f0 = k[c + 1], fp1 = k[c + 2], fp2 = k[c + 3];
        const float d1 = fmaf(-2.0f, fm1, fmaf(-3.0f, f0, fmaf(6.0f, fp1, -fp2)));
        const float d2 = (fm1 + fp1) - 2.0f * f0;
        const float incr = fmaf(fp_b, f0, fmaf(c1p[c], d1, c2 * d2));
        out[c] = f0 + incr;
    }
}

// generic (any integer shift) version reading the staged row with bounds checks
template <int ORDER, bool CLAMP = false>
__device__ __forceinline__ void kick_fp_granule_any(const float *row /* index 0 = y 0 */, const float (&l)[ORDER],
                                                    int mm, int g, int N, float fp_b, float c2,
                                                    const float (&c1p)[4], float (&out)[4])
{
    constexpr int O0 = (ORDER - 1) / 2;
    float k[7];
#pragma unroll
    for (int i = 0; i < 7; ++i) {
        const int y = g - 1 + i;
        float acc = 0.0f, lo = 0.0f, hi = 0.0f;
#pragma unroll
        for (int j = 0; j < ORDER; ++j) {
            const int s = y + mm - O0 + j;
            const float v = (s >= 0 && s < N) ? row[s] : 0.0f;
            acc = fmaf(l[j], v, acc);
            if (j == O0) { lo = v; hi = v; }
            if (j == O0 + 1) { lo = fminf(lo, v); hi = fmaxf(hi, v); }
        }
        if (CLAMP) acc = fminf(fmaxf(acc, lo), hi);
        k[i] = (y >= 0 && y < N) ? acc : 0.0f;
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float fm1 = k[c], f0 = k[c + 1], fp1 = k[c + 2], fp2 = k[c + 3];
        const float d1 = fmaf(-2.0f, fm1, fmaf(-3.0f, f0, fmaf(6.0f, fp1, -fp2)));
        const float d2 = (fm1 + fp1) - 2.0f * f0;
        const float incr = fmaf(fp_b, f0, fmaf(c1p[c], d1, c2 * d2));
        out[c] = f0 + incr;
    }
}

// Manhattan rotation, second half (RF kick): psi_B(x, y) = psi_A(x, y + s1),
// s1 = mh_p * X cells, for the 12 columns g-4 .. g+7 that the wake kick of the granule g..g+3
// reads.  a[i] = psi_A(x, g - 8 + i), i = 0..19; MM1 = floor(s1) (compile time), l1 = weights of
// its fraction; columns outside the grid are zero before and after (A8).
template <int ORDER, int MM1, bool CLAMP = false>
__device__ __forceinline__ void rf_stage(const float (&a)[20], const float (&l1)[ORDER], int g, int N, float (&r)[12])
{
    constexpr int O0 = (ORDER - 1) / 2;
#pragma unroll
    for (int i = 0; i < 12; ++i) {
        const int i0 = i + 4 + MM1 - O0;
        float acc = l1[0] * a[i0];
#pragma unroll
        for (int j = 1; j < ORDER; ++j) acc = fmaf(l1[j], a[i0 + j], acc);
        if (CLAMP) acc = fminf(fmaxf(acc, fminf(a[i0 + O0], a[i0 + O0 + 1])), fmaxf(a[i0 + O0], a[i0 + O0 + 1]));
        r[i] = acc;
    }
    // columns g-4 .. g-1 lie outside the grid only for the first granule, g+4 .. g+7 only for the last
    if (g == 0) { r[0] = 0.0f; r[1] = 0.0f; r[2] = 0.0f; r[3] = 0.0f; }
    if (g == N - 4) { r[8] = 0.0f; r[9] = 0.0f; r[10] = 0.0f; r[11] = 0.0f; }
}
// any integer parts: psi_B at column s of the row (bounds-checked loads), and the whole granule
template <int ORDER, bool CLAMP = false>
__device__ __forceinline__ float rf_value(const float *row, int N, int s, int mm1, const float (&l1)[ORDER])
{
    constexpr int O0 = (ORDER - 1) / 2;
    if (s < 0 || s >= N) return 0.0f;
    float acc = 0.0f, lo = 0.0f, hi = 0.0f;
#pragma unroll
    for (int j = 0; j < ORDER; ++j) {
        const int c = s + mm1 - O0 + j;
        const float v = (c >= 0 && c < N) ? row[c] : 0.0f;
        acc = fmaf(l1[j], v, acc);
        if (j == O0) { lo = v; hi = v; }
        if (j == O0 + 1) { lo = fminf(lo, v); hi = fmaxf(hi, v); }
    }
    if (CLAMP) acc = fminf(fmaxf(acc, lo), hi);
    return acc;
}
template <int ORDER, bool CLAMP = false>
__device__ __noinline__ void rf_kick_fp_granule_any(const float *row, const float (&l1)[ORDER], int mm1,
                                                    const float (&l2)[ORDER], int mm2, int g, int N, float fp_b,
                                                    float c2, const float (&c1p)[4], float (&out)[4])
{
    constexpr int O0 = (ORDER - 1) / 2;
    float k[7];
#pragma unroll 1
    for (int i = 0; i < 7; ++i) {
        const int y = g - 1 + i;
        float acc = 0.0f, lo = 0.0f, hi = 0.0f;
        for (int j = 0; j < ORDER; ++j) {
            const float v = rf_value<ORDER, CLAMP>(row, N, y + mm2 - O0 + j, mm1, l1);
            acc = fmaf(l2[j], v, acc);
            if (j == O0) { lo = v; hi = v; }
            if (j == O0 + 1) { lo = fminf(lo, v); hi = fmaxf(hi, v); }
        }
        if (CLAMP) acc = fminf(fmaxf(acc, lo), hi);
        k[i] = (y >= 0 && y < N) ? acc : 0.0f;
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float fm1 = k[c], f0 = k[c + 1], fp1 = k[c + 2], fp2 = k[c + 3];
        const float d1 = fmaf(-2.0f, fm1, fmaf(-3.0f, f0, fmaf(6.0f, fp1, -fp2)));
        const float d2 = (fm1 + fp1) - 2.0f * f0;
        const float incr = fmaf(fp_b, f0, fmaf(c1p[c], d1, c2 * d2));
        out[c] = f0 + incr;
    }
}

// ---------------------------------------------------------------- rotation of a range of rows
// Thread = column y; rows r0..r1-1 (local indices) of bufA -> bufB.  aA / aB: shared addresses of
// bufA[row 0][CL_PAD + y - O0] and bufB[row 0][CL_PAD + y].  Rows are taken in chunks of ORDER:
// when floor(dx), floor(dy) are the same at both ends of a chunk (dx, dy are monotonic in x) the
// ORDER x ORDER register window slides down one row per cell (ORDER loads); otherwise every row
// loads its full window.
template <int ORDER, int PITCH>
struct Rotator {
    static constexpr int O0 = (ORDER - 1) / 2;
    static constexpr unsigned FULL = 0xffffffffu;
    float win[ORDER][ORDER];
    float a, d, bY, aY, Xoff;     // dx = a*X + bY, dy = d*X + aY, X = x + Xoff
    uint32_t aA, aB;
    int H;

    template <int SUB, bool FULLWIN>
    __device__ __forceinline__ void load(uint32_t base)
    {
        if (FULLWIN) {
#pragma unroll
            for (int i = 0; i < ORDER; ++i)
#pragma unroll
                for (int j = 0; j < ORDER; ++j) win[(SUB + i) % ORDER][j] = lds(base + (i * PITCH + j) * 4);
        } else {
#pragma unroll
            for (int j = 0; j < ORDER; ++j)
                win[(SUB + ORDER - 1) % ORDER][j] = lds(base + ((ORDER - 1) * PITCH + j) * 4);
        }
    }
    template <int SUB>
    __device__ __forceinline__ float eval(float tx, float ty) const
    {
        float lx[ORDER], ly[ORDER];
        lagrange<ORDER>(tx, lx);
        lagrange<ORDER>(ty, ly);
        float acc = 0.0f;
#pragma unroll
        for (int i = 0; i < ORDER; ++i) {
            const float(&wr)[ORDER] = win[(SUB + i) % ORDER];
            float rsum = ly[0] * wr[0];
#pragma unroll
            for (int j = 1; j < ORDER; ++j) rsum = fmaf(ly[j], wr[j], rsum);
            acc = (i == 0) ? lx[0] * rsum : fmaf(lx[i], rsum, acc);
        }
        return acc;
    }
    // one row with its own floors and a full window load
    __device__ __forceinline__ void row_generic(int r, int x0)
    {
        const float X = (float)(x0 + r) + Xoff;
        int ix, iy;
        float tx, ty;
        floor_frac(fmaf(a, X, bY), ix, tx);
        floor_frac(fmaf(d, X, aY), iy, ty);
        const uint32_t base = aA + (uint32_t)(((r + H + ix - O0) * PITCH + iy) * 4);
        load<0, true>(base);
        sts(aB + (uint32_t)(r * PITCH * 4), eval<0>(tx, ty));
    }
    // rows r .. r+n-1 of one chunk whose floors are (fx, fy) throughout; GUARD: n < ORDER possible
    template <int SUB, bool GUARD>
    __device__ __forceinline__ void chunk_rows(uint32_t base, uint32_t ob, float X0, float fx, float fy, bool cont, int n)
    {
        if (!GUARD || SUB < n) {
            if (SUB == 0) {
                if (cont) load<0, false>(base); else load<0, true>(base);
            } else {
                load<SUB, false>(base + SUB * PITCH * 4);
            }
            const float X = X0 + (float)SUB;
            const float tx = fmaf(a, X, bY) - fx, ty = fmaf(d, X, aY) - fy;
            sts(ob + SUB * PITCH * 4, eval<SUB>(tx, ty));
            if constexpr (SUB + 1 < ORDER) chunk_rows<SUB + 1, GUARD>(base, ob, X0, fx, fy, cont, n);
        }
    }
    __device__ __forceinline__ void run(int r0, int r1, int x0)
    {
        if (r0 >= r1) return;
        {   // dx, dy are monotonic in x: equal floors at the first and last row = equal floors throughout
            const float X0 = (float)(x0 + r0) + Xoff, XL = (float)(x0 + r1 - 1) + Xoff;
            const float rx0 = __fadd_rd(fmaf(a, X0, bY), CL_MAGIC), ry0 = __fadd_rd(fmaf(d, X0, aY), CL_MAGIC);
            const float rxL = __fadd_rd(fmaf(a, XL, bY), CL_MAGIC), ryL = __fadd_rd(fmaf(d, XL, aY), CL_MAGIC);
            if (__all_sync(FULL, (rx0 == rxL) && (ry0 == ryL))) {
                const int ix = __float_as_int(rx0) - CL_IMAGIC, iy = __float_as_int(ry0) - CL_IMAGIC;
                const float fx = rx0 - CL_MAGIC, fy = ry0 - CL_MAGIC;
                uint32_t base = aA + (uint32_t)(((r0 + H + ix - O0) * PITCH + iy) * 4);
                uint32_t ob = aB + (uint32_t)(r0 * PITCH * 4);
                float X = X0;
                int r = r0;
                bool cont = false;
                for (; r + ORDER <= r1; r += ORDER) {
                    chunk_rows<0, false>(base, ob, X, fx, fy, cont, ORDER);
                    cont = true;
                    base += ORDER * PITCH * 4; ob += ORDER * PITCH * 4; X += (float)ORDER;
                }
                if (r < r1) chunk_rows<0, true>(base, ob, X, fx, fy, cont, r1 - r);
                return;
            }
        }
        // a floor changes inside this range of rows: decide chunk by chunk
        bool have = false;
        int wix = 0, wiy = 0;
        for (int r = r0; r < r1; r += ORDER) {
            const int n = min(ORDER, r1 - r);
            const float X0 = (float)(x0 + r) + Xoff, XL = X0 + (float)(n - 1);
            const float rx0 = __fadd_rd(fmaf(a, X0, bY), CL_MAGIC), ry0 = __fadd_rd(fmaf(d, X0, aY), CL_MAGIC);
            const float rxL = __fadd_rd(fmaf(a, XL, bY), CL_MAGIC), ryL = __fadd_rd(fmaf(d, XL, aY), CL_MAGIC);
            const int ix = __float_as_int(rx0) - CL_IMAGIC, iy = __float_as_int(ry0) - CL_IMAGIC;
            if (__all_sync(FULL, (rx0 == rxL) && (ry0 == ryL))) {
                const bool cont = have && __all_sync(FULL, ix == wix && iy == wiy);
                const uint32_t base = aA + (uint32_t)(((r + H + ix - O0) * PITCH + iy) * 4);
                chunk_rows<0, true>(base, aB + (uint32_t)(r * PITCH * 4), X0, rx0 - CL_MAGIC, ry0 - CL_MAGIC, cont, n);
                have = (n == ORDER); wix = ix; wiy = iy;
            } else {
                for (int s = 0; s < n; ++s) row_generic(r + s, x0);
                have = false;
            }
        }
    }
};

// ---------------------------------------------------------------- the persistent kernel
// grid = S * (concurrent clusters), cluster = S CTAs, block = CL_THREADS.  Cluster c advances the
// members c, c + nclusters, ... one after the other, each by A.nsteps steps.
//
// Synchronisation between the CTAs of a cluster is pure data flow: every remote store is an
// st.async that counts its bytes on an mbarrier of the receiving CTA, and a consumer waits for the
// expected byte count of the current phase (one phase per step and barrier):
//   MB_RHO[t & 1]  N floats      un-normalised rho_x of step t from every CTA (all-gather), buffer t & 1
//   MB_HALO  nbrs * H * N floats  the neighbours' boundary rows of psi_t
//   MB_PART[t & 1]  S * CL_NPART floats  the partial sums of step t from every CTA
// The charge of step t-1 (-> 1/C) is formed from part(t-1) AFTER rho(t) has been sent, inside the latency of
// the all-gather; rho travels un-normalised and V and rho are scaled where they are used.
// Write-after-read safety needs no extra barrier: rho is double-buffered with a barrier per parity, and a
// CTA can send rho(t+2) only after it has rho(t+1) from every CTA, which each CTA sends after its kick of
// step t, i.e. after it has consumed rho(t); halo(t+1) and part(t+1) are sent after rho(t+1) has arrived
// from every CTA, which each CTA sends after it has consumed halo(t); part(t) (buffer and barrier t & 1) is
// consumed before the wait for rho(t+1), and part(t+2) is sent after rho(t+2) has arrived from every CTA.
template <int ORDER, int N, bool MANH = false>
__global__ void __launch_bounds__(CL_THREADS, 1)
k_cluster_step(GridConst G, ClusterArgs A)
{
    static_assert(N >= 32 && N % 32 == 0, "N must be a multiple of 32");
    constexpr int PITCH = N + 2 * CL_PAD;
    constexpr int O0 = (ORDER - 1) / 2;
    constexpr int CW = N / 32;                       // warps across one row in the rotation
    constexpr int RG = (CL_WARPS / CW) > 0 ? (CL_WARPS / CW) : 1;   // row groups
    constexpr int NG = (N + 127) / 128;              // float4 granules per lane in kick/FP
    constexpr unsigned FULL = 0xffffffffu;

    cg::cluster_group cluster = cg::this_cluster();
    const int S = A.S, R = A.R, H = G.H;
    const int rank = (int)cluster.block_rank();
    const int nclusters = (int)gridDim.x / S, cid = (int)blockIdx.x / S;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int x0 = rank * R;

    extern __shared__ __align__(16) float smem[];
    float *bufA = smem;                                   // (R + 2H) rows
    float *bufB = bufA + (size_t)(R + 2 * H) * PITCH;     // R rows
    float *wf = bufB + (size_t)R * PITCH;                 // 2N
    float *rho2 = wf + 2 * N;                             // 2 x N (step parity)
    float *part = rho2 + 2 * N;                           // 2 * CL_MAX_S * CL_NPART
    float *wred = part + 2 * CL_MAX_S * CL_NPART;         // CL_WARPS * 8
    float *scal = wred + CL_WARPS * 8;                    // [2..11] = five mbarriers
    const uint32_t sA = smem_u32(bufA), sB = smem_u32(bufB), sRho2 = smem_u32(rho2), sPart = smem_u32(part);
    const uint32_t mbRho0 = smem_u32(scal + 2), mbHalo = mbRho0 + 16, mbPart0 = mbRho0 + 24;    // mbRho[p] = mbRho0 + 8 p, mbPart[p] = mbPart0 + 8 p
    const int nbrs = (rank > 0 ? 1 : 0) + (rank < S - 1 ? 1 : 0);
    const uint32_t bytesRho = ((R & 3) == 0 ? (uint32_t)(N - R) : (uint32_t)N) * 4u, bytesHalo = (uint32_t)(nbrs * H * N) * 4u, bytesPart = (uint32_t)(S - 1) * CL_NPART * 4u;

    // ---- rotation: thread = column y of row group rg
    const int cw = warp % CW, rg = warp / CW;
    const int RPG = (R + RG - 1) / RG;
    const int rbeg = min(R, rg * RPG), rend = (rg < RG) ? min(R, rbeg + RPG) : rbeg;
    const int y = cw * 32 + lane;
    Rotator<ORDER, PITCH> rot;
    {
        const float Yc = (float)y + G.y0c;
        rot.a = G.a; rot.d = G.d; rot.bY = G.b * Yc; rot.aY = G.a * Yc; rot.Xoff = G.x0c; rot.H = H;
        rot.aA = sA + (uint32_t)((CL_PAD + y - O0) * 4);
        rot.aB = sB + (uint32_t)((CL_PAD + y) * 4);
        asm volatile("" : "+r"(rot.aA), "+r"(rot.aB));      // opaque: do not re-derive per use
    }

    // ---- Manhattan drift: shift of this thread's column and its weights (un-scaled)
    int mmq = 0;
    float lq[ORDER];
    {
        float tq;
        floor_frac(G.mh_q * ((float)y + G.y0c), mmq, tq);
        lagrange<ORDER>(tq, lq);
    }

    // ---- kick / Fokker-Planck: lane = granules g = 4*lane + 128*k of one row per warp
    const float c1 = G.fp_b / (6.0f * G.dp), c2 = G.fp_b / (G.dp * G.dp);
    const float yc = 0.5f * (float)(N - 1), xc = 0.5f * (float)(N - 1);
    float c1p[NG][4];
#pragma unroll
    for (int k = 0; k < NG; ++k)
#pragma unroll
        for (int c = 0; c < 4; ++c) c1p[k][c] = c1 * fmaf((float)(4 * lane + 128 * k + c), G.dp, G.p_min);

    if (tid == 0) {
        mbar_init(mbRho0, 1); mbar_init(mbRho0 + 8, 1); mbar_init(mbHalo, 1); mbar_init(mbPart0, 1); mbar_init(mbPart0 + 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    unsigned phase = 0;      // parity of the current phase of the halo barrier
    unsigned rho_use0 = 0u, rho_use1 = 0u;      // how often mbRho[p] has been waited on
    unsigned part_use0 = 0u, part_use1 = 0u;    // ... and mbPart[p]

    for (int m = cid; m < A.members; m += nclusters) {
        float *gpsi = A.psi + (size_t)m * N * N;
        const float *gw = A.wfun ? A.wfun + (size_t)m * 2 * N : nullptr;
        // ---- load: own rows + halo rows of bufA straight from HBM, zero pads, zero bufB pads
        for (int i = tid; i < (R + 2 * H) * PITCH; i += CL_THREADS) {
            const int r = i / PITCH, c = i - r * PITCH - CL_PAD;
            const int x = x0 - H + r;
            float v = 0.0f;
            if (x >= 0 && x < N && c >= 0 && c < N) v = gpsi[(size_t)x * N + c];
            bufA[i] = v;
        }
        for (int i = tid; i < R * PITCH; i += CL_THREADS) bufB[i] = 0.0f;
        for (int i = tid; i < 2 * N; i += CL_THREADS) wf[i] = (gw && i < 2 * N - 1) ? gw[i] : 0.0f;
        float sc = G.renorm ? A.scale[m] : 1.0f;
        // a barrier that expects no bytes (S = 1; the halo of an edge-less cluster) is neither armed nor
        // waited on: arming it would complete its phase at once, and a warp that has not yet reached
        // its wait would see the parity flip twice and hang
        if (tid == 0) {
            if (bytesRho) mbar_expect_tx(mbRho0, bytesRho);
            if (bytesRho && A.nsteps > 1) mbar_expect_tx(mbRho0 + 8, bytesRho);
            if (bytesHalo) mbar_expect_tx(mbHalo, bytesHalo);
            if (bytesPart) mbar_expect_tx(mbPart0, bytesPart);
            if (bytesPart && A.nsteps > 1) mbar_expect_tx(mbPart0 + 8, bytesPart);
        }
        // nobody may store into this CTA before it has finished initialising
        cluster.sync();

        for (int step = 0; step <= A.nsteps; ++step) {
            const bool last = (step == A.nsteps);
            if (step > 0) {
                // ---- the neighbours' boundary rows of psi_t have arrived
                if (bytesHalo) mbar_wait(mbHalo, phase ^ 1u);
                if (tid == 0 && !last && bytesHalo) mbar_expect_tx(mbHalo, bytesHalo);
            }
            VFPS_STAMP(A.dbg, step, 0);
            // ================= 1. rotation: bufA -> bufB
            if (!last) {
                if constexpr (MANH) {
                    // Manhattan drift (L136): column y shifted along q by mh_q * Y cells -- one 1-D
                    // interpolation with per-column weights; the taps of row r are the rows
                    // r + mmq - O0 .. r + mmq - O0 + ORDER - 1 of bufA (|shift| <= the halo, as for
                    // the standard rotation)
                    uint32_t src = sA + (uint32_t)(((rbeg + H + mmq - O0) * PITCH + CL_PAD + y) * 4);
                    uint32_t dstb = sB + (uint32_t)((rbeg * PITCH + CL_PAD + y) * 4);
                    for (int r = rbeg; r < rend; ++r) {
                        float acc = lq[0] * lds(src);
#pragma unroll
                        for (int i = 1; i < ORDER; ++i) acc = fmaf(lq[i], lds(src + i * PITCH * 4), acc);
                        sts(dstb, acc);
                        src += PITCH * 4; dstb += PITCH * 4;
                    }
                } else {
                    rot.run(rbeg, rend, x0);
                }
            }
            VFPS_STAMP(A.dbg, step, 1);
            __syncthreads();
            VFPS_STAMP(A.dbg, step, 2);
            const int p = step & 1;
            float *rho = rho2 + p * N;
            const uint32_t sRho = sRho2 + (uint32_t)(p * N) * 4u, mbRho = mbRho0 + 8u * (uint32_t)p;
            VFPS_STAMP(A.dbg, step, 3);
            if (!last) {
                // ================= 2. projection: rho_x = dp * sum_y bufB(x, y) (un-normalised), all-gathered into buffer p
                for (int r = warp; r < R; r += CL_WARPS) {
                    const uint32_t row = sB + (uint32_t)((r * PITCH + CL_PAD) * 4);
                    float s = 0.0f;
#pragma unroll
                    for (int k = 0; k < NG; ++k) {
                        const int g = 4 * lane + 128 * k;
                        if (g < N) {
                            const float4 v = lds4(row + g * 4);
                            s += (v.x + v.y) + (v.z + v.w);
                        }
                    }
                    s = warp_sum(s) * G.dp;
                    if ((R & 3) != 0) {
                        if (lane < S) st_async(mapa(sRho + (uint32_t)(x0 + r) * 4u, lane), s, mapa(mbRho, lane));
                    } else if (lane == 0) {
                        rho[x0 + r] = s;          // own slot of the local rho array doubles as staging
                    }
                }
                if ((R & 3) == 0) {
                    // one 16-byte message per four rows and destination (few large DSMEM transactions)
                    __syncthreads();
                    const int nq = R >> 2;
                    for (int i = tid; i < (S - 1) * nq; i += CL_THREADS) {
                        const int dd0 = i / nq, q = i - dd0 * nq, dd = dd0 + (dd0 >= rank ? 1 : 0);
                        const uint32_t a = sRho + (uint32_t)(x0 + 4 * q) * 4u;
                        st_async4(mapa(a, dd), lds4(a), mapa(mbRho, dd));
                    }
                }
            }
            if (step > 0) {
                // ================= 6. a6 of step t-1: charge, scale, diagnostics -- inside the latency of the all-gather
                const int pq = (step - 1) & 1;             // part(t) travels on barrier t & 1; part(t + 2) re-uses it
                if (bytesPart) mbar_wait(mbPart0 + 8u * (uint32_t)pq, (pq ? part_use1 : part_use0) & 1u);
                if (pq) ++part_use1; else ++part_use0;
                if (tid == 0 && step + 1 < A.nsteps && bytesPart) mbar_expect_tx(mbPart0 + 8u * (uint32_t)pq, bytesPart);
                // lane = (g4, j): partial j summed over the CTAs g4, g4 + 4, ..., then over the four
                // lane groups -- the same order in every warp of every CTA
                const float *pp = part + ((step - 1) & 1) * (CL_MAX_S * CL_NPART);
                float tj = 0.0f;
                for (int dd = lane >> 3; dd < S; dd += 4) tj += pp[dd * CL_NPART + (lane & 7)];
                tj += __shfl_xor_sync(FULL, tj, 8);
                tj += __shfl_xor_sync(FULL, tj, 16);
                const float t0 = __shfl_sync(FULL, tj, 0);
                const float C = (G.dq * G.dp) * t0;
                sc = G.renorm ? 1.0f / C : 1.0f;
                if (rank == 0 && warp == CL_WARPS - 1 && A.diag != nullptr) {
                    float t[CL_NPART];
#pragma unroll
                    for (int j = 0; j < CL_NPART; ++j) t[j] = __shfl_sync(FULL, tj, j);
                    if (lane == 0) {
                        const float i0 = 1.0f / t[0];
                        const float mp_c = t[1] * i0, vp = fmaf(-mp_c, mp_c, t[2] * i0);
                        const float mq_c = t[3] * i0, vq = fmaf(-mq_c, mq_c, t[4] * i0);
                        const float cc = G.renorm ? C : 1.0f;
                        float *o = A.diag + ((size_t)(step - 1) * A.members + m) * 6;
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
            VFPS_STAMP(A.dbg, step, 4);
            if (bytesRho) mbar_wait(mbRho, (p ? rho_use1 : rho_use0) & 1u);
            if (p) ++rho_use1; else ++rho_use0;
            VFPS_STAMP(A.dbg, step, 5);
            if (tid == 0 && step + 2 < A.nsteps && bytesRho) mbar_expect_tx(mbRho, bytesRho);
            // ================= 3.+4. wake (own rows), kick + Fokker-Planck: bufB -> bufA
            // per-warp sums: s0 sum psi, s1/s2 p moments (per lane), q1/q2 q moments, pw = sum rho V
            float s0 = 0.0f, s1 = 0.0f, s2 = 0.0f, q1 = 0.0f, q2 = 0.0f, pw = 0.0f;
            for (int r = warp; r < R; r += CL_WARPS) {
                const int x = x0 + r;
                float V = 0.0f;
                if (gw != nullptr) {
                    // V_x = sum_x' w[x - x'] rho_x'; w[d] at wf[d + N - 1]
#pragma unroll
                    for (int k = 0; k < CW; ++k) {
                        const int xp = lane + 32 * k;
                        V = fmaf(wf[x - xp + N - 1], rho[xp], V);
                    }
                    V = warp_sum(V) * sc;
                }
                pw = fmaf(rho[x] * sc, V, pw);
                int mm;
                float t;
                floor_frac(G.kick_c * V, mm, t);
                float l[ORDER];
                lagrange<ORDER>(t, l);
#pragma unroll
                for (int j = 0; j < ORDER; ++j) l[j] *= sc;
                int mm1 = 0;
                float l1[ORDER];
                if constexpr (MANH) {
                    float t1;
                    floor_frac(G.mh_p * ((float)x + G.x0c), mm1, t1);
                    lagrange<ORDER>(t1, l1);
                }
                const uint32_t row = sB + (uint32_t)((r * PITCH + CL_PAD) * 4);
                const uint32_t orow = sA + (uint32_t)(((r + H) * PITCH + CL_PAD) * 4);
                // halo pushes: the first H rows go to rank-1's lower halo, the last H to rank+1's upper
                const bool up = (r < H) && (rank > 0), dn = (r >= R - H) && (rank < S - 1);
                uint32_t aup = 0, mup = 0, adn = 0, mdn = 0;
                if (up) { aup = mapa(sA + (uint32_t)(((R + H + r) * PITCH + CL_PAD) * 4), rank - 1); mup = mapa(mbHalo, rank - 1); }
                if (dn) { adn = mapa(sA + (uint32_t)(((r - (R - H)) * PITCH + CL_PAD) * 4), rank + 1); mdn = mapa(mbHalo, rank + 1); }
                float rs = 0.0f;
#pragma unroll
                for (int k = 0; k < NG; ++k) {
                    const int g = 4 * lane + 128 * k;
                    if (g < N) {
                        float o[4];
                        if constexpr (MANH) {
                            // RF kick (shift mh_p * X cells, weights l1) then wake kick, both along p
                            if (mm >= -2 && mm <= 0 && mm1 >= -2 && mm1 <= 1) {
                                const float4 z4 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                                const float4 v0 = (g >= 4) ? lds4(row + (g - 8) * 4) : z4;
                                const float4 v1 = lds4(row + (g - 4) * 4), v2 = lds4(row + g * 4), v3 = lds4(row + (g + 4) * 4);
                                const float4 v4 = (g <= N - 8) ? lds4(row + (g + 8) * 4) : z4;
                                const float a[20] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w, v2.x, v2.y,
                                                     v2.z, v2.w, v3.x, v3.y, v3.z, v3.w, v4.x, v4.y, v4.z, v4.w};
                                float rr[12];
                                if (mm1 == 0) rf_stage<ORDER, 0>(a, l1, g, N, rr);
                                else if (mm1 == -1) rf_stage<ORDER, -1>(a, l1, g, N, rr);
                                else if (mm1 == 1) rf_stage<ORDER, 1>(a, l1, g, N, rr);
                                else rf_stage<ORDER, -2>(a, l1, g, N, rr);
                                if (mm == 0) kick_fp_granule<ORDER, 0>(rr, l, g, N, G.fp_b, c2, c1p[k], o);
                                else if (mm == -1) kick_fp_granule<ORDER, -1>(rr, l, g, N, G.fp_b, c2, c1p[k], o);
                                else kick_fp_granule<ORDER, -2>(rr, l, g, N, G.fp_b, c2, c1p[k], o);
                            } else {
                                rf_kick_fp_granule_any<ORDER>(bufB + r * PITCH + CL_PAD, l1, mm1, l, mm, g, N, G.fp_b, c2, c1p[k], o);
                            }
                        } else
                        if (mm >= -2 && mm <= 0) {
                            float b[12];
                            const float4 v0 = lds4(row + (g - 4) * 4), v1 = lds4(row + g * 4), v2 = lds4(row + (g + 4) * 4);
                            b[0] = v0.x; b[1] = v0.y; b[2] = v0.z; b[3] = v0.w;
                            b[4] = v1.x; b[5] = v1.y; b[6] = v1.z; b[7] = v1.w;
                            b[8] = v2.x; b[9] = v2.y; b[10] = v2.z; b[11] = v2.w;
                            if (mm == 0) kick_fp_granule<ORDER, 0>(b, l, g, N, G.fp_b, c2, c1p[k], o);
                            else if (mm == -1) kick_fp_granule<ORDER, -1>(b, l, g, N, G.fp_b, c2, c1p[k], o);
                            else kick_fp_granule<ORDER, -2>(b, l, g, N, G.fp_b, c2, c1p[k], o);
                        } else {
                            kick_fp_granule_any<ORDER>(bufB + r * PITCH + CL_PAD, l, mm, g, N, G.fp_b, c2, c1p[k], o);
                        }
                        const float4 ov = make_float4(o[0], o[1], o[2], o[3]);
                        sts4(orow + g * 4, ov);
                        if (up) st_async4(aup + g * 4, ov, mup);
                        if (dn) st_async4(adn + g * 4, ov, mdn);
                        float q0 = 0.0f;
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            const float yy = (float)(g + c) - yc;
                            const float tt = o[c] * yy;
                            q0 += o[c]; s1 += tt; s2 = fmaf(tt, yy, s2);
                        }
                        rs += q0;
                    }
                }
                // q moments of the END-of-step psi from the lane's share of the row sum (reduced over the lanes
                // once, at the end of the pass, together with the other sums)
                const float X = (float)x - xc, tq = rs * X;
                s0 += rs; q1 += tq; q2 = fmaf(tq, X, q2);
            }
            VFPS_STAMP(A.dbg, step, 6);
            // ================= 5. partial sums of this CTA -> every CTA
            {
                // one transposed reduction of all six sums (pw is the same in every lane: lane 0's counts)
                float v8[8] = {s0, s1, s2, q1, q2, lane == 0 ? pw : 0.0f, 0.0f, 0.0f};
                const float tot = warp_reduce_transposed<8>(v8, lane);       // lanes 4 j .. 4 j + 3 hold sum j
                if ((lane & 3) == 0) wred[warp * 8 + (lane >> 2)] = tot;
            }
            __syncthreads();
            if (warp == 0) {
                // lane = (g4, j): partial j of the warps g4, g4 + 4, ...; then across the four lane groups
                const int j = lane & 7, g4 = lane >> 3;
                float v = 0.0f;
#pragma unroll
                for (int w = 0; w < CL_WARPS / 4; ++w) v += wred[(g4 + 4 * w) * 8 + j];
                v += __shfl_xor_sync(FULL, v, 8);
                v += __shfl_xor_sync(FULL, v, 16);
                // lanes 0..7 now hold the CTA's partials: stage them, then two 16-byte messages per CTA
                const uint32_t slot = sPart + (uint32_t)(((step & 1) * CL_MAX_S + rank) * CL_NPART) * 4u;
                if (lane < CL_NPART) sts(slot + lane * 4, v);
                __syncwarp();
                for (int i = lane; i < 2 * (S - 1); i += 32) {
                    const int dd0 = i >> 1, hh = i & 1, dd = dd0 + (dd0 >= rank ? 1 : 0);
                    st_async4(mapa(slot + hh * 16, dd), lds4(slot + hh * 16), mapa(mbPart0 + 8u * (uint32_t)(step & 1), dd));
                }
            }
            VFPS_STAMP(A.dbg, step, 7);
            phase ^= 1u;
        }
        // ---- store own rows and the scale (all remote stores into this CTA have been waited for)
        __syncthreads();
        for (int i = tid; i < R * (N / 4); i += CL_THREADS) {
            const int r = i / (N / 4), c = (i - r * (N / 4)) * 4;
            *reinterpret_cast<float4 *>(gpsi + (size_t)(x0 + r) * N + c) =
                *reinterpret_cast<const float4 *>(bufA + (r + H) * PITCH + CL_PAD + c);
        }
        if (rank == 0 && tid == 0) A.scale[m] = sc;
        cluster.sync();       // every CTA is done with this member before anyone re-initialises
    }
}

}  // namespace vfps
