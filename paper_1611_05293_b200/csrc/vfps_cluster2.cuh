// vfps_cluster2.cuh -- persistent thread-block-cluster engine, packed-fp32 version (sm_100a).
//
// Same step, same cluster protocol (st.async + mbarrier data flow) and same HBM behaviour as
// vfps_cluster.cuh; what changes is how a CTA computes.  The v1 kernel is bound by instruction
// issue (profiles/r01_c1_cluster.md: 113-126 thread-instructions per cell per step, 59 % of the
// issue slots used, no memory level above 35 %).  sm_100a has two-wide packed fp32 arithmetic
// (fma.rn.f32x2 / FFMA2: one issue slot, two lanes of the FMA pipe for two cycles), so this
// kernel lets every thread advance TWO cells at once -- the same column y of the rows r and
// r + R/2 of the CTA's R rows -- and keeps both shared-memory buffers "pair-interleaved":
//   element (pair-row p, column y) is a float2 { row p, row p + R/2 }.
// One 64-bit shared load then fetches one rotation tap of both cells, one 128-bit load two columns
// of both rows for the kick / Fokker-Planck pass, and every arithmetic instruction of a1, a4, a5
// is a packed one.  (The two rows are R/2 apart, so floor(dx), floor(dy) of their back-rotated
// source points agree except where a floor changes inside the CTA's rows; those rows take a scalar
// path.)  Issue slots per cell drop to ~45; the FMA pipe (~65 lane-cycles per cell) becomes the
// bound.
//
// bufA  psi_t, local rows lr = 0 .. R+2H-1 (H halo rows above and below the R own rows):
//       pair-row p = 0 .. R/2+2H-1 holds { lr = p, lr = p + R/2 }.  Local rows R/2 .. R/2+2H-1
//       therefore live in two slots (.x of p = lr and .y of p = lr - R/2); both are written.
// bufB  psi' (rotated), own rows only: pair-row w holds { own row w, own row w + R/2 }.
#pragma once
#include "vfps_cluster.cuh"

namespace vfps {

// Column order inside a pair-row.  A pair-row is cut into 16-byte chunks of two columns
// { (A,B)(y), (A,B)(y+1) }, y even, counted from column -CL_PAD; the even chunks lie in one region
// and the odd chunks in a second one, NH2 chunks further on.  A thread of the kick pass owns four
// columns = one even and one odd chunk, so a warp's 128-bit accesses are contiguous in each region
// (no bank conflict; with the plain column order they are 32 bytes apart = two-way conflicts, which
// made the kick pass shared-memory bound).  NH2 = 4 mod 8 keeps the 64-bit accesses of the
// rotation (thread = column) on disjoint banks for even column offsets.
__host__ __device__ constexpr int cluster2_nh2(int N)
{
    int n = (N + 2 * CL_PAD) / 4;
    while ((n & 7) != 4) ++n;
    return n;
}
// byte offset of column y (-CL_PAD <= y < N + CL_PAD) inside a pair-row
template <int NH2>
__device__ __forceinline__ uint32_t col_off(int y)
{
    const int yy = y + CL_PAD, cp = yy >> 1;
    return (uint32_t)((((cp >> 1) + (cp & 1) * NH2) << 4) + ((yy & 1) << 3));
}

__host__ __device__ inline size_t cluster2_smem_floats(int N, int S, int H)
{
    const int R = N / S, Rh = R / 2, pitch = 4 * cluster2_nh2(N);   // float2 slots per pair-row
    return (size_t)(Rh + 2 * H) * pitch * 2     // bufA
           + (size_t)Rh * pitch * 2             // bufB
           + 2 * (size_t)N                      // wake function
           + (size_t)N                          // rho (all rows)
           + 2 * CL_MAX_S * CL_NPART            // partial sums of all CTAs, two parities
           + CL_WARPS * 8 + 8                   // block reduction scratch, mbarriers
           + 8 * (size_t)R;                     // kick weights and integer shift of every own row
}

// ---- packed fp32 (two independent lanes .x / .y per instruction)
__device__ __forceinline__ float2 f2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }

__device__ __forceinline__ float2 lds2(uint32_t a)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts2(uint32_t a, float2 v)
{
    asm volatile("st.shared.v2.f32 [%0], {%1,%2};" ::"r"(a), "f"(v.x), "f"(v.y) : "memory");
}

// Lagrange weights (Eq. 13) of both lanes; written without operand negation (packed instructions
// have no negate modifier).  Nodes o_k = k - floor((ORDER-1)/2), t in [0,1).
template <int ORDER>
__device__ __forceinline__ void lagrange2(float2 t, float2 (&l)[ORDER]);

template <>
__device__ __forceinline__ void lagrange2<2>(float2 t, float2 (&l)[2])
{
    l[0] = fma2(t, f2(-1.0f), f2(1.0f));
    l[1] = t;
}
template <>
__device__ __forceinline__ void lagrange2<3>(float2 t, float2 (&l)[3])
{
    const float2 h = mul2(t, f2(0.5f));
    l[0] = mul2(h, add2(t, f2(-1.0f)));
    l[1] = fma2(mul2(t, f2(-1.0f)), t, f2(1.0f));
    l[2] = fma2(h, t, h);
}
template <>
__device__ __forceinline__ void lagrange2<4>(float2 t, float2 (&l)[4])
{
    // A = t(t-1)/6, B = (t+1)(t-2)/2 = t(t-1)/2 - 1:  l0 = A (2-t), l1 = B (t-1), l2 = -B t, l3 = A (t+1)
    const float2 tm1 = add2(t, f2(-1.0f));
    const float2 u = mul2(t, tm1);
    const float2 A = mul2(u, f2(1.0f / 6.0f));
    const float2 B = fma2(u, f2(0.5f), f2(-1.0f));
    const float2 nB = fma2(u, f2(-0.5f), f2(1.0f));
    l[0] = mul2(A, fma2(t, f2(-1.0f), f2(2.0f)));
    l[1] = mul2(B, tm1);
    l[2] = mul2(nB, t);
    l[3] = fma2(A, t, A);
}

// ---------------------------------------------------------------- packed kick + Fokker-Planck
// Four columns g..g+3 of a row pair: b[i] = psi'(., g - 4 + i) of both rows, i = 0..11.
// W[j], j < NW: kick weights of both rows on the common nodes MM - O0 + j (a row whose integer
// shift is MM + 1 carries a leading zero weight, one whose shift is MM a trailing one, when
// NW = ORDER + 1).  k[i] = kicked value at column g - 1 + i, zero outside the grid (A8).
template <int ORDER, int MM, int NW>
__device__ __forceinline__ void kick_fp_granule2(const float2 (&b)[12], const float2 (&W)[ORDER + 1], int g, int N,
                                                 float2 fp_b, float2 c2, const float2 (&c1p)[4], float2 (&out)[4])
{
    constexpr int O0 = (ORDER - 1) / 2;
    float2 k[7];
#pragma unroll
    for (int i = 0; i < 7; ++i) {
        const int i0 = 3 + i + MM - O0;
        float2 acc = mul2(W[0], b[i0]);
#pragma unroll
        for (int j = 1; j < NW; ++j) acc = fma2(W[j], b[i0 + j], acc);
        k[i] = acc;
    }
    if (g == 0) k[0] = f2(0.0f);
    if (g == N - 4) { k[5] = f2(0.0f); k[6] = f2(0.0f); }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float2 fm1 = k[c], f0 = k[c + 1], fp1 = k[c + 2], fp2 = k[c + 3];
        // d1 = -2 f-1 - 3 f0 + 6 f+1 - f+2 (Eq. 15 x 6 dp), d2 = f-1 - 2 f0 + f+1
        const float2 d1 = fma2(f2(6.0f), fp1, fma2(f2(-3.0f), f0, fma2(f2(-2.0f), fm1, mul2(f2(-1.0f), fp2))));
        const float2 d2 = fma2(f2(-2.0f), f0, add2(fm1, fp1));
        const float2 incr = fma2(fp_b, f0, fma2(c1p[c], d1, mul2(c2, d2)));
        out[c] = add2(f0, incr);
    }
}

// any integer shift, one row of the pair (h = 0 / 1), scalar, bounds-checked taps.
// row: shared address of the pair-row.
template <int ORDER, int NH2>
__device__ __forceinline__ void kick_fp_granule_any2(uint32_t row, int h, const float (&l)[ORDER], int mm, int g,
                                                     int N, float fp_b, float c2, const float2 (&c1p)[4],
                                                     float (&out)[4])
{
    constexpr int O0 = (ORDER - 1) / 2;
    float k[7];
#pragma unroll
    for (int i = 0; i < 7; ++i) {
        const int y = g - 1 + i;
        float acc = 0.0f;
#pragma unroll
        for (int j = 0; j < ORDER; ++j) {
            const int s = y + mm - O0 + j;
            const float v = (s >= 0 && s < N) ? lds(row + col_off<NH2>(s) + h * 4) : 0.0f;
            acc = fmaf(l[j], v, acc);
        }
        k[i] = (y >= 0 && y < N) ? acc : 0.0f;
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float fm1 = k[c], f0 = k[c + 1], fp1 = k[c + 2], fp2 = k[c + 3];
        const float d1 = fmaf(-2.0f, fm1, fmaf(-3.0f, f0, fmaf(6.0f, fp1, -fp2)));
        const float d2 = (fm1 + fp1) - 2.0f * f0;
        const float incr = fmaf(fp_b, f0, fmaf(c1p[c].x, d1, c2 * d2));
        out[c] = f0 + incr;
    }
}

// Everything the kick pass of one pair-row needs besides the weights (addresses are shared-window).
struct KickRow2 {
    uint32_t row, orow;          // bufB pair-row, bufA pair-row (start of the row)
    uint32_t adupA, adupB;       // second slots of rows stored twice
    uint32_t aup, mup, adn, mdn; // halo slots in the neighbours and their mbarriers
    bool dupA, dupB, up, dn;
};

// all NG granules of one pair-row with compile-time shift MM and NW common nodes:
// bufB -> bufA (+ second slots, + halo pushes); adds the new values to colsum (per column, both
// rows packed) -- every moment of a6 is formed from colsum and the row sums rs afterwards.
template <int ORDER, int N, int MM, int NW>
__device__ __forceinline__ void kick_fp_row2(const KickRow2 &K, const float2 (&W)[ORDER + 1], int lane, float2 fp_b,
                                             float2 c2, const float2 (&c1p)[N / 128][4], float2 (&colsum)[N / 128][4],
                                             float2 &rs)
{
    constexpr int NG = N / 128, NH2 = cluster2_nh2(N);
#pragma unroll
    for (int k = 0; k < NG; ++k) {
        const int g = 4 * lane + 128 * k;
        float2 b[12], o[4];
        // columns g - 4 + 2q, q = 0..5: chunk 2 (lane + 32 k) + q -> even chunks in region 0, odd in 1
        const uint32_t c0 = (uint32_t)((lane + 32 * k) * 16);
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            const float4 v = lds4(K.row + c0 + (uint32_t)(((q >> 1) + (q & 1) * NH2) * 16));
            b[2 * q] = make_float2(v.x, v.y);
            b[2 * q + 1] = make_float2(v.z, v.w);
        }
        kick_fp_granule2<ORDER, MM, NW>(b, W, g, N, fp_b, c2, c1p[k], o);
        // columns g, g+1 = chunk 2 (lane + 32 k) + 2, columns g+2, g+3 = the odd chunk after it
        const uint32_t e0 = c0 + 16, e1 = c0 + 16 + NH2 * 16;
        sts4(K.orow + e0, make_float4(o[0].x, o[0].y, o[1].x, o[1].y));
        sts4(K.orow + e1, make_float4(o[2].x, o[2].y, o[3].x, o[3].y));
        if (K.dupA) {
            sts(K.adupA + e0, o[0].x); sts(K.adupA + e0 + 8, o[1].x); sts(K.adupA + e1, o[2].x); sts(K.adupA + e1 + 8, o[3].x);
        }
        if (K.dupB) {
            sts(K.adupB + e0, o[0].y); sts(K.adupB + e0 + 8, o[1].y); sts(K.adupB + e1, o[2].y); sts(K.adupB + e1 + 8, o[3].y);
        }
        if (K.up) {
            st_async(K.aup + e0, o[0].x, K.mup); st_async(K.aup + e0 + 8, o[1].x, K.mup);
            st_async(K.aup + e1, o[2].x, K.mup); st_async(K.aup + e1 + 8, o[3].x, K.mup);
        }
        if (K.dn) {
            st_async(K.adn + e0, o[0].y, K.mdn); st_async(K.adn + e0 + 8, o[1].y, K.mdn);
            st_async(K.adn + e1, o[2].y, K.mdn); st_async(K.adn + e1 + 8, o[3].y, K.mdn);
        }
        rs = add2(rs, add2(add2(o[0], o[1]), add2(o[2], o[3])));
#pragma unroll
        for (int c = 0; c < 4; ++c) colsum[k][c] = add2(colsum[k][c], o[c]);
    }
}

// ---------------------------------------------------------------- packed rotation of pair-rows
// Thread = column y; pair-rows w0..w1-1 of bufA -> bufB, i.e. the cells (x0 + w, y) and
// (x0 + w + Rh, y).  aA: shared address of bufA's pair-row 0; aB: of this thread's column in
// bufB's pair-row 0; toff[j]: byte offset of tap column y + iy - O0 + j inside a pair-row.
template <int ORDER, int NH2>
struct Rotator2 {
    static constexpr int O0 = (ORDER - 1) / 2;
    static constexpr int PB = NH2 * 32;           // bytes per pair-row
    static constexpr unsigned FULL = 0xffffffffu;
    float2 win[ORDER][ORDER];
    float a, d, bY, aY, Xoff;     // dx = a*X + bY, dy = d*X + aY, X = x + Xoff
    uint32_t aA, aB;
    uint32_t toff[ORDER];
    int H, Rh, y;

    __device__ __forceinline__ void set_taps(int iy)
    {
#pragma unroll
        for (int j = 0; j < ORDER; ++j) toff[j] = col_off<NH2>(y + iy - O0 + j);
    }

    template <int SUB, bool FULLWIN>
    __device__ __forceinline__ void load(uint32_t base)
    {
        if (FULLWIN) {
#pragma unroll
            for (int i = 0; i < ORDER; ++i)
#pragma unroll
                for (int j = 0; j < ORDER; ++j) win[(SUB + i) % ORDER][j] = lds2(base + i * PB + toff[j]);
        } else {
#pragma unroll
            for (int j = 0; j < ORDER; ++j) win[(SUB + ORDER - 1) % ORDER][j] = lds2(base + (ORDER - 1) * PB + toff[j]);
        }
    }
    template <int SUB>
    __device__ __forceinline__ float2 eval(float2 tx, float2 ty) const
    {
        float2 lx[ORDER], ly[ORDER];
        lagrange2<ORDER>(tx, lx);
        lagrange2<ORDER>(ty, ly);
        float2 acc = f2(0.0f);
#pragma unroll
        for (int i = 0; i < ORDER; ++i) {
            const float2(&wr)[ORDER] = win[(SUB + i) % ORDER];
            float2 rsum = mul2(ly[0], wr[0]);
#pragma unroll
            for (int j = 1; j < ORDER; ++j) rsum = fma2(ly[j], wr[j], rsum);
            acc = (i == 0) ? mul2(lx[0], rsum) : fma2(lx[i], rsum, acc);
        }
        return acc;
    }
    // one cell of pair-row w (h = 0: row w, h = 1: row w + Rh), scalar, its own floors
    __device__ __forceinline__ void cell_generic(int w, int h, int x0)
    {
        const float X = (float)(x0 + w + h * Rh) + Xoff;
        int ix, iy;
        float tx, ty;
        floor_frac(fmaf(a, X, bY), ix, tx);
        floor_frac(fmaf(d, X, aY), iy, ty);
        const uint32_t base = aA + (uint32_t)((w + H + ix - O0) * PB + h * 4);
        uint32_t to[ORDER];
#pragma unroll
        for (int j = 0; j < ORDER; ++j) to[j] = col_off<NH2>(y + iy - O0 + j);
        float lx[ORDER], ly[ORDER];
        lagrange<ORDER>(tx, lx);
        lagrange<ORDER>(ty, ly);
        float acc = 0.0f;
#pragma unroll
        for (int i = 0; i < ORDER; ++i) {
            float rsum = ly[0] * lds(base + i * PB + to[0]);
#pragma unroll
            for (int j = 1; j < ORDER; ++j) rsum = fmaf(ly[j], lds(base + i * PB + to[j]), rsum);
            acc = (i == 0) ? lx[0] * rsum : fmaf(lx[i], rsum, acc);
        }
        sts(aB + (uint32_t)(w * PB + h * 4), acc);
    }
    // pair-rows of one chunk whose floors are (fx, fy) for both rows throughout; GUARD: n < ORDER possible
    template <int SUB, bool GUARD>
    __device__ __forceinline__ void chunk_rows(uint32_t base, uint32_t ob, float2 X0, float fx, float fy, bool cont, int n)
    {
        if (!GUARD || SUB < n) {
            if (SUB == 0) {
                if (cont) load<0, false>(base); else load<0, true>(base);
            } else {
                load<SUB, false>(base + SUB * PB);
            }
            const float2 X = add2(X0, f2((float)SUB));
            const float2 tx = add2(fma2(f2(a), X, f2(bY)), f2(-fx));
            const float2 ty = add2(fma2(f2(d), X, f2(aY)), f2(-fy));
            sts2(ob + SUB * PB, eval<SUB>(tx, ty));
            if constexpr (SUB + 1 < ORDER) chunk_rows<SUB + 1, GUARD>(base, ob, X0, fx, fy, cont, n);
        }
    }
    __device__ __forceinline__ void run(int w0, int w1, int x0)
    {
        if (w0 >= w1) return;
        {   // dx, dy are monotonic in x: equal floors at the first row of the lower half and the last
            // row of the upper half = equal floors for every cell this thread touches
            const float X0 = (float)(x0 + w0) + Xoff, XL = (float)(x0 + w1 - 1 + Rh) + Xoff;
            const float rx0 = __fadd_rd(fmaf(a, X0, bY), CL_MAGIC), ry0 = __fadd_rd(fmaf(d, X0, aY), CL_MAGIC);
            const float rxL = __fadd_rd(fmaf(a, XL, bY), CL_MAGIC), ryL = __fadd_rd(fmaf(d, XL, aY), CL_MAGIC);
            if (__all_sync(FULL, (rx0 == rxL) && (ry0 == ryL))) {
                const int ix = __float_as_int(rx0) - CL_IMAGIC, iy = __float_as_int(ry0) - CL_IMAGIC;
                const float fx = rx0 - CL_MAGIC, fy = ry0 - CL_MAGIC;
                set_taps(iy);
                uint32_t base = aA + (uint32_t)((w0 + H + ix - O0) * PB);
                uint32_t ob = aB + (uint32_t)(w0 * PB);
                float2 X = make_float2(X0, X0 + (float)Rh);
                int w = w0;
                bool cont = false;
                for (; w + ORDER <= w1; w += ORDER) {
                    chunk_rows<0, false>(base, ob, X, fx, fy, cont, ORDER);
                    cont = true;
                    base += ORDER * PB; ob += ORDER * PB; X = add2(X, f2((float)ORDER));
                }
                if (w < w1) chunk_rows<0, true>(base, ob, X, fx, fy, cont, w1 - w);
                return;
            }
        }
        // a floor changes somewhere in this thread's cells: decide pair-row by pair-row
        for (int w = w0; w < w1; ++w) {
            const float XA = (float)(x0 + w) + Xoff, XB = XA + (float)Rh;
            const float rxA = __fadd_rd(fmaf(a, XA, bY), CL_MAGIC), ryA = __fadd_rd(fmaf(d, XA, aY), CL_MAGIC);
            const float rxB = __fadd_rd(fmaf(a, XB, bY), CL_MAGIC), ryB = __fadd_rd(fmaf(d, XB, aY), CL_MAGIC);
            if (__all_sync(FULL, (rxA == rxB) && (ryA == ryB))) {
                // (lanes may still differ from one another: every lane has its own base address)
                const int ix = __float_as_int(rxA) - CL_IMAGIC, iy = __float_as_int(ryA) - CL_IMAGIC;
                set_taps(iy);
                const uint32_t base = aA + (uint32_t)((w + H + ix - O0) * PB);
                chunk_rows<0, true>(base, aB + (uint32_t)(w * PB), make_float2(XA, XB), rxA - CL_MAGIC, ryA - CL_MAGIC, false, 1);
            } else {
                cell_generic(w, 0, x0);
                cell_generic(w, 1, x0);
            }
        }
    }
};

// ---------------------------------------------------------------- the persistent kernel (packed)
// grid = S * (concurrent clusters), cluster = S CTAs, block = NT.  Protocol between the CTAs:
// exactly that of k_cluster_step (MB_RHO / MB_HALO / MB_PART, one phase per step).
template <int ORDER, int N, int NT>
__global__ void __launch_bounds__(NT, (NT <= 256) ? 2 : 1)
k_cluster2_step(GridConst G, ClusterArgs A)
{
    static_assert(N >= 128 && N % 128 == 0, "N must be a multiple of 128");
    constexpr int NH2 = cluster2_nh2(N);             // 16-byte chunks per region of a pair-row
    constexpr int PITCH = 4 * NH2;                   // float2 slots per pair-row (two regions)
    constexpr int PB = PITCH * 8;                    // bytes per pair-row
    constexpr int NWARPS = NT / 32;
    constexpr int CW = N / 32;                       // warps across one row in the rotation
    static_assert(NWARPS >= CW && NWARPS % CW == 0, "block must cover a row");
    constexpr int RG = NWARPS / CW;                  // row groups
    constexpr int NG = N / 128;                      // float4 granules per lane in kick/FP
    constexpr unsigned FULL = 0xffffffffu;

    cg::cluster_group cluster = cg::this_cluster();
    const int S = A.S, R = A.R, Rh = R >> 1, H = G.H;
    const int PA = Rh + 2 * H;                       // pair-rows of bufA
    const int rank = (int)cluster.block_rank();
    const int nclusters = (int)gridDim.x / S, cid = (int)blockIdx.x / S;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int x0 = rank * R;

    extern __shared__ __align__(16) float smem[];
    float *bufA = smem;                                   // PA pair-rows
    float *bufB = bufA + (size_t)PA * PITCH * 2;          // Rh pair-rows
    float *wf = bufB + (size_t)Rh * PITCH * 2;            // 2N
    float *rho = wf + 2 * N;                              // N
    float *part = rho + N;                                // 2 * CL_MAX_S * CL_NPART
    float *wred = part + 2 * CL_MAX_S * CL_NPART;         // CL_WARPS * 8
    float *scal = wred + CL_WARPS * 8;                    // [2..7] = three mbarriers
    float *rowinfo = scal + 8;                            // R x { l_0..l_3 (times 1/C), mm, -, -, - }
    const uint32_t sA = smem_u32(bufA), sB = smem_u32(bufB), sRho = smem_u32(rho), sPart = smem_u32(part);
    const uint32_t sInfo = smem_u32(rowinfo);
    const uint32_t mbRho = smem_u32(scal + 2), mbHalo = mbRho + 8, mbPart = mbRho + 16;
    const int nbrs = (rank > 0 ? 1 : 0) + (rank < S - 1 ? 1 : 0);
    const uint32_t bytesRho = (uint32_t)(N - R) * 4u, bytesHalo = (uint32_t)(nbrs * H * N) * 4u,
                   bytesPart = (uint32_t)(S - 1) * CL_NPART * 4u;

    // ---- rotation: thread = column y of row group rg
    const int cw = warp % CW, rg = warp / CW;
    const int PPG = (Rh + RG - 1) / RG;
    const int wbeg = min(Rh, rg * PPG), wend = min(Rh, wbeg + PPG);
    Rotator2<ORDER, NH2> rot;
    {
        constexpr int O0 = (ORDER - 1) / 2;
        const int y = cw * 32 + lane;
        const float Yc = (float)y + G.y0c;
        rot.a = G.a; rot.d = G.d; rot.bY = G.b * Yc; rot.aY = G.a * Yc; rot.Xoff = G.x0c; rot.H = H; rot.Rh = Rh;
        rot.y = y;
        rot.aA = sA;
        rot.aB = sB + col_off<NH2>(y);
        asm volatile("" : "+r"(rot.aA), "+r"(rot.aB));      // opaque: do not re-derive per use
    }

    // ---- kick / Fokker-Planck: lane = granules g = 4*lane + 128*k of one pair-row per warp
    const float c1 = G.fp_b / (6.0f * G.dp), c2 = G.fp_b / (G.dp * G.dp);
    const float yc = 0.5f * (float)(N - 1), xc = 0.5f * (float)(N - 1);
    float2 c1p[NG][4];
#pragma unroll
    for (int k = 0; k < NG; ++k)
#pragma unroll
        for (int c = 0; c < 4; ++c) c1p[k][c] = f2(c1 * fmaf((float)(4 * lane + 128 * k + c), G.dp, G.p_min));

    if (tid == 0) {
        mbar_init(mbRho, 1); mbar_init(mbHalo, 1); mbar_init(mbPart, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    unsigned phase = 0;      // parity of the current phase of all three barriers

    for (int m = cid; m < A.members; m += nclusters) {
        float *gpsi = A.psi + (size_t)m * N * N;
        const float *gw = A.wfun ? A.wfun + (size_t)m * 2 * N : nullptr;
        // ---- load: own rows + halo rows straight from HBM into one or two slots of bufA
        // (every pad column, and the unused chunks between the regions, stay zero for good)
        for (int i = tid; i < (PA + Rh) * PITCH * 2; i += NT) bufA[i] = 0.0f;       // bufA and bufB
        __syncthreads();
        for (int i = tid; i < (R + 2 * H) * N; i += NT) {
            const int lr = i / N, c = i - lr * N;
            const int x = x0 - H + lr;
            if (x >= 0 && x < N) {
                const float v = gpsi[(size_t)x * N + c];
                const uint32_t o = col_off<NH2>(c);
                if (lr < PA) sts(sA + (uint32_t)(lr * PB) + o, v);
                if (lr >= Rh) sts(sA + (uint32_t)((lr - Rh) * PB) + o + 4, v);
            }
        }
        for (int i = tid; i < 2 * N; i += NT) wf[i] = (gw && i < 2 * N - 1) ? gw[i] : 0.0f;
        float sc = G.renorm ? A.scale[m] : 1.0f;
        if (tid == 0) { mbar_expect_tx(mbRho, bytesRho); mbar_expect_tx(mbHalo, bytesHalo); mbar_expect_tx(mbPart, bytesPart); }
        // nobody may store into this CTA before it has finished initialising
        cluster.sync();

        for (int step = 0; step <= A.nsteps; ++step) {
            const bool last = (step == A.nsteps);
            if (step > 0) {
                // ---- the neighbours' boundary rows of psi_t have arrived
                mbar_wait(mbHalo, phase ^ 1u);
                if (tid == 0 && !last) mbar_expect_tx(mbHalo, bytesHalo);
            }
            if (A.dbg != nullptr && tid == 0 && step < 64) A.dbg[((size_t)blockIdx.x * 64 + step) * 8 + 0] = clock64();
            // ================= 1. rotation: bufA -> bufB
            if (!last) rot.run(wbeg, wend, x0);
            if (A.dbg != nullptr && tid == 0 && step < 64) A.dbg[((size_t)blockIdx.x * 64 + step) * 8 + 1] = clock64();
            __syncthreads();
            if (A.dbg != nullptr && tid == 0 && step < 64) A.dbg[((size_t)blockIdx.x * 64 + step) * 8 + 2] = clock64();
            if (step > 0) {
                // ================= 6. a6 of step t-1: charge, scale, diagnostics
                mbar_wait(mbPart, phase ^ 1u);
                if (tid == 0 && !last) mbar_expect_tx(mbPart, bytesPart);
                const float *pp = part + ((step - 1) & 1) * (CL_MAX_S * CL_NPART);
                float tj = 0.0f;
                for (int dd = lane >> 3; dd < S; dd += 4) tj += pp[dd * CL_NPART + (lane & 7)];
                tj += __shfl_xor_sync(FULL, tj, 8);
                tj += __shfl_xor_sync(FULL, tj, 16);
                const float t0 = __shfl_sync(FULL, tj, 0);
                const float C = (G.dq * G.dp) * t0;
                sc = G.renorm ? 1.0f / C : 1.0f;
                if (rank == 0 && warp == NWARPS - 1 && A.diag != nullptr) {
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
            if (A.dbg != nullptr && tid == 0 && step < 64) A.dbg[((size_t)blockIdx.x * 64 + step) * 8 + 3] = clock64();
            // ================= 2. projection: rho_x = dp * sc * sum_y bufB(x, y), all-gathered
            for (int w = warp; w < Rh; w += NWARPS) {
                // every 16-byte chunk of the pair-row (pads and gaps are zero), in storage order
                const uint32_t row = sB + (uint32_t)(w * PB);
                float2 s = f2(0.0f);
#pragma unroll
                for (int k = 0; k < (2 * NH2 + 31) / 32; ++k) {
                    const int ch = lane + 32 * k;
                    if (ch < 2 * NH2) {
                        const float4 v = lds4(row + (uint32_t)(ch * 16));
                        s = add2(s, add2(make_float2(v.x, v.y), make_float2(v.z, v.w)));
                    }
                }
                const float sa = warp_sum(s.x) * (G.dp * sc), sb = warp_sum(s.y) * (G.dp * sc);
                if (lane == 0) { rho[x0 + w] = sa; rho[x0 + w + Rh] = sb; }   // own slots double as staging
            }
            {
                // one 16-byte message per four rows and destination (few large DSMEM transactions)
                __syncthreads();
                const int nq = R >> 2;
                for (int i = tid; i < (S - 1) * nq; i += NT) {
                    const int dd0 = i / nq, q = i - dd0 * nq, dd = dd0 + (dd0 >= rank ? 1 : 0);
                    const uint32_t a = sRho + (uint32_t)(x0 + 4 * q) * 4u;
                    st_async4(mapa(a, dd), lds4(a), mapa(mbRho, dd));
                }
            }
            if (A.dbg != nullptr && tid == 0 && step < 64) A.dbg[((size_t)blockIdx.x * 64 + step) * 8 + 4] = clock64();
            mbar_wait(mbRho, phase);
            if (A.dbg != nullptr && tid == 0 && step < 64) A.dbg[((size_t)blockIdx.x * 64 + step) * 8 + 5] = clock64();
            if (tid == 0 && step + 1 < A.nsteps) mbar_expect_tx(mbRho, bytesRho);
            // ================= 3. wake a3 of the own rows, then the kick weights of every row, once:
            // TPR threads share one row (x' interleaved), V_x = sum_x' w[x - x'] rho_x' (Eq. 4;
            // w[d] at wf[d + N - 1]); the group's first lane turns V_x into the integer shift mm and
            // the Lagrange weights (times 1/C) and leaves them in rowinfo[row].
            float pw = 0.0f;                                   // sum rho V (group leaders only)
            {
                const int TPR = min(32, max(1, NT / R)), sub = tid & (TPR - 1);
                for (int r = tid / TPR; r < R; r += NT / TPR) {
                    const int x = x0 + r;
                    float V = 0.0f;
                    if (gw != nullptr) {
                        float v0 = 0.0f, v1 = 0.0f, v2 = 0.0f, v3 = 0.0f;
                        const float *wx = wf + (x + N - 1);
                        for (int xp = sub; xp < N; xp += 4 * TPR) {
                            v0 = fmaf(wx[-xp], rho[xp], v0);
                            v1 = fmaf(wx[-(xp + TPR)], rho[xp + TPR], v1);
                            v2 = fmaf(wx[-(xp + 2 * TPR)], rho[xp + 2 * TPR], v2);
                            v3 = fmaf(wx[-(xp + 3 * TPR)], rho[xp + 3 * TPR], v3);
                        }
                        V = (v0 + v1) + (v2 + v3);
                        for (int o = TPR >> 1; o > 0; o >>= 1) V += __shfl_xor_sync(FULL, V, o);
                    }
                    if (sub == 0) {
                        pw = fmaf(rho[x], V, pw);
                        int mm;
                        float t;
                        floor_frac(G.kick_c * V, mm, t);
                        float l[ORDER];
                        lagrange<ORDER>(t, l);
                        float4 lw = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                        lw.x = l[0] * sc; lw.y = l[1] * sc;
                        if (ORDER > 2) lw.z = l[ORDER > 2 ? 2 : 0] * sc;
                        if (ORDER > 3) lw.w = l[ORDER > 3 ? 3 : 0] * sc;
                        *reinterpret_cast<float4 *>(rowinfo + 8 * r) = lw;
                        *reinterpret_cast<int *>(rowinfo + 8 * r + 4) = mm;
                    }
                }
            }
            __syncthreads();
            if (A.dbg != nullptr && tid == 0 && step < 64) A.dbg[((size_t)blockIdx.x * 64 + step) * 8 + 6] = clock64();
            // ================= 4. kick + Fokker-Planck: bufB -> bufA
            // per lane: column sums of the new psi (both rows packed), q-moment sums of its part of
            // every row
            float2 q1v = f2(0.0f), q2v = f2(0.0f);
            float2 colsum[NG][4];
#pragma unroll
            for (int k = 0; k < NG; ++k)
#pragma unroll
                for (int c = 0; c < 4; ++c) colsum[k][c] = f2(0.0f);
            const float2 fb2 = f2(G.fp_b), cc2 = f2(c2);
            for (int w = warp; w < Rh; w += NWARPS) {
                const int xA = x0 + w, xB = xA + Rh;
                float lA[ORDER], lB[ORDER];
                int mmA, mmB;
                {
                    const float4 a4 = lds4(sInfo + (uint32_t)(w * 32)), b4 = lds4(sInfo + (uint32_t)((w + Rh) * 32));
                    mmA = __float_as_int(lds(sInfo + (uint32_t)(w * 32 + 16)));
                    mmB = __float_as_int(lds(sInfo + (uint32_t)((w + Rh) * 32 + 16)));
                    const float la[4] = {a4.x, a4.y, a4.z, a4.w}, lb[4] = {b4.x, b4.y, b4.z, b4.w};
#pragma unroll
                    for (int j = 0; j < ORDER; ++j) { lA[j] = la[j]; lB[j] = lb[j]; }
                }
                const int mlo = min(mmA, mmB), dm = max(mmA, mmB) - mlo;
                // common-node weights of both rows (see kick_fp_granule2)
                float2 W[ORDER + 1];
                {
                    const bool sa = (mmA != mlo), sb = (mmB != mlo);   // row shifted one node up
#pragma unroll
                    for (int j = 0; j <= ORDER; ++j) {
                        const float a0 = (j < ORDER) ? lA[j < ORDER ? j : 0] : 0.0f, a1 = (j > 0) ? lA[j > 0 ? j - 1 : 0] : 0.0f;
                        const float b0 = (j < ORDER) ? lB[j < ORDER ? j : 0] : 0.0f, b1 = (j > 0) ? lB[j > 0 ? j - 1 : 0] : 0.0f;
                        W[j] = make_float2(sa ? a1 : a0, sb ? b1 : b0);
                    }
                }
                const int mode = (dm == 0 && mlo >= -2 && mlo <= 0) ? (mlo + 2)            // 0,1,2: same shift
                                 : (dm == 1 && mlo >= -2 && mlo <= -1) ? (mlo + 5)         // 3,4: shifts differ by one
                                                                       : 5;                // generic
                KickRow2 K;
                K.row = sB + (uint32_t)(w * PB);
                K.orow = sA + (uint32_t)((w + H) * PB);
                // second slots of the rows stored twice, and halo pushes (first H rows -> rank-1's
                // lower halo, last H rows -> rank+1's upper halo)
                K.dupA = (w + H >= Rh); K.dupB = (w < H);
                K.adupA = sA + (uint32_t)((w + H - Rh) * PB + 4);
                K.adupB = sA + (uint32_t)((w + H + Rh) * PB);
                K.up = (w < H) && (rank > 0); K.dn = (w >= Rh - H) && (rank < S - 1);
                K.aup = K.mup = K.adn = K.mdn = 0;
                if (K.up) { K.aup = mapa(sA + (uint32_t)((Rh + H + w) * PB + 4), rank - 1); K.mup = mapa(mbHalo, rank - 1); }
                if (K.dn) { K.adn = mapa(sA + (uint32_t)((w - Rh + H) * PB), rank + 1); K.mdn = mapa(mbHalo, rank + 1); }
                float2 rs = f2(0.0f);
                switch (mode) {
                    case 0: kick_fp_row2<ORDER, N, -2, ORDER>(K, W, lane, fb2, cc2, c1p, colsum, rs); break;
                    case 1: kick_fp_row2<ORDER, N, -1, ORDER>(K, W, lane, fb2, cc2, c1p, colsum, rs); break;
                    case 2: kick_fp_row2<ORDER, N, 0, ORDER>(K, W, lane, fb2, cc2, c1p, colsum, rs); break;
                    case 3: kick_fp_row2<ORDER, N, -2, ORDER + 1>(K, W, lane, fb2, cc2, c1p, colsum, rs); break;
                    case 4: kick_fp_row2<ORDER, N, -1, ORDER + 1>(K, W, lane, fb2, cc2, c1p, colsum, rs); break;
                    default: {
#pragma unroll
                        for (int k = 0; k < NG; ++k) {
                            const int g = 4 * lane + 128 * k;
                            float oa[4], ob[4];
                            kick_fp_granule_any2<ORDER, NH2>(K.row, 0, lA, mmA, g, N, G.fp_b, c2, c1p[k], oa);
                            kick_fp_granule_any2<ORDER, NH2>(K.row, 1, lB, mmB, g, N, G.fp_b, c2, c1p[k], ob);
#pragma unroll
                            for (int c = 0; c < 4; ++c) {
                                const uint32_t e = col_off<NH2>(g + c);
                                const float2 oc = make_float2(oa[c], ob[c]);
                                sts2(K.orow + e, oc);
                                if (K.dupA) sts(K.adupA + e, oa[c]);
                                if (K.dupB) sts(K.adupB + e, ob[c]);
                                if (K.up) st_async(K.aup + e, oa[c], K.mup);
                                if (K.dn) st_async(K.adn + e, ob[c], K.mdn);
                                rs = add2(rs, oc);
                                colsum[k][c] = add2(colsum[k][c], oc);
                            }
                        }
                    }
                }
                // q moments of the END-of-step psi: this lane's part of the two row sums
                const float2 X2 = make_float2((float)xA - xc, (float)xB - xc);
                const float2 tq = mul2(rs, X2);
                q1v = add2(q1v, tq);
                q2v = fma2(tq, X2, q2v);
            }
            // charge and p moments from the per-lane column sums
            float s0 = 0.0f, s1 = 0.0f, s2 = 0.0f;
#pragma unroll
            for (int k = 0; k < NG; ++k)
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float yy = (float)(4 * lane + 128 * k + c) - yc;
                    const float cs = colsum[k][c].x + colsum[k][c].y;
                    const float tt = cs * yy;
                    s0 += cs; s1 += tt; s2 = fmaf(tt, yy, s2);
                }
            float q1 = q1v.x + q1v.y, q2 = q2v.x + q2v.y;
            s0 = warp_sum(s0); q1 = warp_sum(q1); q2 = warp_sum(q2); pw = warp_sum(pw);
            if (A.dbg != nullptr && tid == 0 && step < 64) A.dbg[((size_t)blockIdx.x * 64 + step) * 8 + 7] = clock64();
            // ================= 5. partial sums of this CTA -> every CTA
            s1 = warp_sum(s1); s2 = warp_sum(s2);
            if (lane == 0) {
                *reinterpret_cast<float4 *>(wred + warp * 8) = make_float4(s0, s1, s2, q1);
                *reinterpret_cast<float4 *>(wred + warp * 8 + 4) = make_float4(q2, pw, 0.0f, 0.0f);
            }
            __syncthreads();
            if (warp == 0) {
                const int j = lane & 7, g4 = lane >> 3;
                float v = 0.0f;
#pragma unroll
                for (int w = 0; w < NWARPS / 4; ++w) v += wred[(g4 + 4 * w) * 8 + j];
                v += __shfl_xor_sync(FULL, v, 8);
                v += __shfl_xor_sync(FULL, v, 16);
                const uint32_t slot = sPart + (uint32_t)(((step & 1) * CL_MAX_S + rank) * CL_NPART) * 4u;
                if (lane < CL_NPART) sts(slot + lane * 4, v);
                __syncwarp();
                for (int i = lane; i < 2 * (S - 1); i += 32) {
                    const int dd0 = i >> 1, hh = i & 1, dd = dd0 + (dd0 >= rank ? 1 : 0);
                    st_async4(mapa(slot + hh * 16, dd), lds4(slot + hh * 16), mapa(mbPart, dd));
                }
            }
            phase ^= 1u;
        }
        // ---- store own rows and the scale (all remote stores into this CTA have been waited for)
        __syncthreads();
        for (int i = tid; i < R * (N / 4); i += NT) {
            const int r = i / (N / 4), c = (i - r * (N / 4)) * 4;
            const uint32_t src = (r < Rh) ? sA + (uint32_t)((r + H) * PB) : sA + (uint32_t)((r + H - Rh) * PB + 4);
            *reinterpret_cast<float4 *>(gpsi + (size_t)(x0 + r) * N + c) =
                make_float4(lds(src + col_off<NH2>(c)), lds(src + col_off<NH2>(c + 1)), lds(src + col_off<NH2>(c + 2)),
                            lds(src + col_off<NH2>(c + 3)));
        }
        if (rank == 0 && tid == 0) A.scale[m] = sc;
        cluster.sync();       // every CTA is done with this member before anyone re-initialises
    }
}

}  // namespace vfps
