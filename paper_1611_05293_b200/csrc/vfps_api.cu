// vfps_api.cu -- the C ABI of include/vfps.h over the sm_100a kernels.  Host logic only:
// argument checks, device-memory ownership, launch configuration, engine selection.
#include "../../include/vfps.h"
#include "vfps_kernels.cuh"
#include "vfps_cluster.cuh"
#include "vfps_onchip.cuh"
#include "vfps_stream2.cuh"
#include "vfps_grid.cuh"
#include "vfps_grid2.cuh"
#include "vfps_launch.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <algorithm>
#include <utility>
#include <vector>

using namespace vfps;

namespace {

thread_local std::string g_create_error;

struct Ctl {
    float *diag;
};

}  // namespace

struct vfps_sim {
    vfps_params P{};
    GridConst G{};
    int N = 0, Nf = 0, log2Nf = 0, members = 1;
    bool has_wake = false;
    cudaStream_t stream = nullptr;
    int engine_opt = VFPS_ENGINE_AUTO, wake_opt = VFPS_WAKE_AUTO;

    float *psi = nullptr, *psi_tmp = nullptr;   // [members][N][N]; psi holds the current state
    float2 *Z = nullptr;                         // [members][Nf/2+1]
    float2 *tw = nullptr;                        // [Nf/2]
    float *rho_part = nullptr;                   // [members][N][tiles_y2]
    float *rho = nullptr, *V = nullptr;          // [members][N]
    float *qstat = nullptr;                      // [members][4]
    float *mom_part = nullptr;                   // [members][kfp2_blocks][6]
    float *scale = nullptr;                      // [members]
    unsigned *blkctr = nullptr;                  // [members]
    int *rowctr = nullptr;                       // [members]
    float **diag_cell = nullptr;                 // device cell with the caller's diag pointer
    // scratch for the stateless get_* calls
    float *g_rho = nullptr, *g_V = nullptr, *g_m1 = nullptr, *g_m2 = nullptr, *g_qstat = nullptr;
    float *g_out = nullptr;                      // [members][max(N,6)] staging for *_host variants

    float *wfun = nullptr;                       // [members][2N] wake function w = Re IDFT(Z)
    // cluster engine (0 = not available for this grid)
    int cl_S = 0, cl_S_opt = 0, cl_max_clusters = 0;
    int cl_ver = 0, cl_ver_opt = 0;              // kernel in use (1 k_cluster_step, 3 k_onchip_step), request
    size_t cl_smem = 0;
    std::string cl_why;                          // why the cluster engine is unavailable
    // second cluster design (vfps_onchip.cuh, cl_ver == 3): geometry tables and the work queue
    bool oc_tab = false;                         // per-launch weight tables are accurate enough
    int oc_tab_S = 0;                            // cluster size the tables on the device were built for
    float *oc_coltab = nullptr, *oc_rowtab = nullptr;
    int *oc_colix = nullptr;
    unsigned long long *oc_item_ctr = nullptr;
    unsigned int *oc_member_done = nullptr;
    unsigned long long oc_item_base = 0;
    unsigned int oc_done_base = 0;

    // streaming kernels (vfps_stream2.cuh)
    int tiles_x2 = 0, tiles_y2 = 0, kfp2_rows = 0, kfp2_blocks = 0, wd_blocks = 0;
    float *pw_part = nullptr;                    // [members][wd_blocks]
    float *dpU = nullptr;                        // [members][N], clamped interpolation only (k_wake_direct)
    // persistent cooperative-grid engine (vfps_grid.cuh); gr_blocks = 0: not available
    int gr_blocks = 0, gr_KR = 0;
    size_t gr_smem = 0;
    float *gr_mom = nullptr;                     // [gr_blocks][GR_NPART]
    unsigned long long *gr_qacc = nullptr;       // [2] fixed-point charge accumulators
    float *gr_zrow = nullptr;                    // [N] zeros
    std::string gr_why;
    // TMA-staged grid engine (vfps_grid2.cuh, grid kernel 2); g2_blocks = 0: not available
    int gr_ver_opt = 0;                          // 0 auto (2 where available), 1 k_grid_step, 2 k_grid2_step
    int g2_blocks = 0, g2_KRmax = 0, g2_nbuf = 0;
    int *g2_row0 = nullptr;
    size_t g2_smem = 0;
    float *g2_coltab = nullptr, *g2_rowtab = nullptr, *g2_rho = nullptr, *g2_mom = nullptr;
    int *g2_colix = nullptr;
    unsigned long long *g2_qacc = nullptr;
    CUtensorMap g2_tmap;
    std::string g2_why;
    unsigned *tilectr = nullptr;                 // [members][tiles_x2], zero between launches
    size_t fft_smem = 0;
    int fft_threads = 0;

    // CUDA-graph engine: GRAPH_STEPS split steps captured once, replayed
    cudaGraphExec_t graph_exec = nullptr;
    long long graph_launches = 0;                // kernel nodes of the captured graph
    // per-kernel device timing (VFPS_OPT_TIMING): event pairs around launches, resolved lazily
    bool timing = false;
    std::vector<cudaEvent_t> ev_pool;
    std::vector<int> ev_kind;                    // kernel id of pair i (events 2i, 2i+1)
    double k_ms[VFPS_NUM_KERNELS] = {};
    long long k_cnt[VFPS_NUM_KERNELS] = {};
    float *diag_scratch = nullptr;               // vfps_step_host staging (grow-only)
    size_t diag_scratch_n = 0;

    bool psi_set = false;
    long long steps = 0, launches = 0;
    std::string err;
    std::vector<void *> owned;

    size_t cells() const { return (size_t)N * N; }
};

namespace {

int fail(vfps_sim *h, int code, const std::string &msg)
{
    if (h) h->err = msg; else g_create_error = msg;
    return code;
}

#define CU(call)                                                                              \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(h, e_ == cudaErrorMemoryAllocation ? VFPS_ERR_NOMEM : VFPS_ERR_CUDA,  \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                  \
    } while (0)

template <typename T>
cudaError_t dalloc(vfps_sim *h, T **p, size_t n)
{
    void *q = nullptr;
    cudaError_t e = cudaMalloc(&q, n * sizeof(T) > 0 ? n * sizeof(T) : 1);
    if (e == cudaSuccess) { *p = (T *)q; h->owned.push_back(q); }
    return e;
}

bool is_pow2(long long v) { return v > 0 && (v & (v - 1)) == 0; }

int validate(const vfps_params *p, std::string &why)
{
    if (!p) { why = "params is NULL"; return VFPS_ERR_ARG; }
    if (p->N < 8) { why = "N must be >= 8"; return VFPS_ERR_ARG; }
    if (!(p->q_max > p->q_min) || !(p->p_max > p->p_min)) { why = "empty q or p range"; return VFPS_ERR_ARG; }
    if (p->steps_per_period < 1) { why = "steps_per_period must be >= 1"; return VFPS_ERR_ARG; }
    if (!(p->beta >= 0.0)) { why = "beta must be >= 0"; return VFPS_ERR_ARG; }
    if (p->interp_order < 2 || p->interp_order > 4) { why = "interp_order must be 2, 3 or 4"; return VFPS_ERR_ARG; }
    if (p->pad < 2 || !is_pow2(p->pad)) { why = "pad must be a power of two >= 2"; return VFPS_ERR_ARG; }
    if (!is_pow2((long long)p->N * p->pad)) { why = "N*pad must be a power of two"; return VFPS_ERR_ARG; }
    if (p->members < 1) { why = "members must be >= 1"; return VFPS_ERR_ARG; }
    if (p->members > 65535) { why = "at most 65535 members per handle (batched launches use gridDim.y = members)"; return VFPS_ERR_UNSUPPORTED; }
    if (p->flags & ~(VFPS_FLAG_RENORMALISE | VFPS_FLAG_CLAMP | VFPS_FLAG_ROT_MANHATTAN)) { why = "unknown flag"; return VFPS_ERR_ARG; }
    if (p->N % 4 != 0) { why = "N must be a multiple of 4 (float4 rows)"; return VFPS_ERR_UNSUPPORTED; }
    if ((long long)p->N * p->pad > 8192) { why = "N*pad > 8192: wake FFT does not fit one CTA's shared memory"; return VFPS_ERR_UNSUPPORTED; }
    return VFPS_OK;
}

void grid_constants(vfps_sim *h)
{
    const vfps_params &P = h->P;
    const double PI = 3.14159265358979323846;
    const double dq = (P.q_max - P.q_min) / (P.N - 1), dp = (P.p_max - P.p_min) / (P.N - 1);
    const double dphi = 2.0 * PI / P.steps_per_period;
    const double sh = std::sin(0.5 * dphi);
    const double a = -2.0 * sh * sh, s = std::sin(dphi);        // a = cos(dphi) - 1, no cancellation
    const double b = -s * dp / dq, d = s * dq / dp;
    const double x0c = P.q_min / dq, y0c = P.p_min / dp;
    GridConst &G = h->G;
    G.N = P.N; G.order = P.interp_order;
    G.a = (float)a; G.b = (float)b; G.d = (float)d;
    G.x0c = (float)x0c; G.y0c = (float)y0c;
    G.dq = (float)dq; G.dp = (float)dp;
    G.kick_c = (float)(dphi / dp);
    G.mh_q = (float)(-dphi * dp / dq);
    G.mh_p = (float)(dphi * dq / dp);
    G.fp_b = (float)(P.beta / P.steps_per_period);
    G.p_min = (float)P.p_min; G.q_min = (float)P.q_min;
    G.renorm = (P.flags & VFPS_FLAG_RENORMALISE) ? 1 : 0;
    // largest source displacement in cells over the grid, then stencil reach
    const double Xm = std::fmax(std::fabs(x0c), std::fabs(P.N - 1 + x0c));
    const double Ym = std::fmax(std::fabs(y0c), std::fabs(P.N - 1 + y0c));
    const double dmax = std::fmax(std::fabs(a) * Xm + std::fabs(b) * Ym, std::fabs(d) * Xm + std::fabs(a) * Ym);
    G.H = (int)std::floor(dmax * 1.0001 + 1e-6) + 2;
}

constexpr int GRAPH_STEPS = 50;          // split steps per captured graph (150 kernel nodes)
constexpr size_t EV_PAIRS_MAX = 3 * 256;  // timed launches per vfps_step call

// bracket the next launch of kernel `kind` with an event pair (timing mode, stream engine only)
struct Bracket {
    vfps_sim *h; cudaEvent_t e1 = nullptr;
    Bracket(vfps_sim *h_, int kind, bool on) : h(h_)
    {
        if (!on || h->ev_kind.size() >= EV_PAIRS_MAX) return;
        const size_t i = h->ev_kind.size();
        while (h->ev_pool.size() < 2 * (i + 1)) {
            cudaEvent_t e;
            if (cudaEventCreate(&e) != cudaSuccess) return;
            h->ev_pool.push_back(e);
        }
        h->ev_kind.push_back(kind);
        cudaEventRecord(h->ev_pool[2 * i], h->stream);
        e1 = h->ev_pool[2 * i + 1];
    }
    ~Bracket() { if (e1) cudaEventRecord(e1, h->stream); }
};

// fold finished event pairs into the per-kernel totals (synchronises the stream)
void resolve_timing(vfps_sim *h)
{
    if (h->ev_kind.empty()) return;
    cudaStreamSynchronize(h->stream);
    for (size_t i = 0; i < h->ev_kind.size(); ++i) {
        float ms = 0.0f;
        if (cudaEventElapsedTime(&ms, h->ev_pool[2 * i], h->ev_pool[2 * i + 1]) == cudaSuccess) {
            h->k_ms[h->ev_kind[i]] += ms;
            h->k_cnt[h->ev_kind[i]] += 1;
        }
    }
    h->ev_kind.clear();
}


// ---------------------------------------------------------------- wake function w = Re IDFT(Z)
// One thread per (member, lag d = -(N-1)..N-1); double precision, angle reduced in integers.
// w[d] = (1/Nf) [ Re Z_0 + 2 sum_{k=1}^{Nf/2-1} Re(Z_k e^{2 pi i k d/Nf}) + Re Z_{Nf/2} (-1)^d ]
// (Hermitian spectrum, L149); stored at index d + N - 1 of a row of 2N floats.
__global__ void k_wake_function(int N, int Nf, int members, const float2 *__restrict__ Z, float *__restrict__ w)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= members * 2 * N) return;
    const int m = i / (2 * N), j = i - m * 2 * N;
    if (j >= 2 * N - 1) { w[i] = 0.0f; return; }
    const int d = j - (N - 1);
    const float2 *Zm = Z + (size_t)m * (Nf / 2 + 1);
    double acc = (double)Zm[0].x;
    for (int k = 1; k < Nf / 2; ++k) {
        long long kd = ((long long)k * d) % Nf;
        double sn, cs;
        sincospi(2.0 * (double)kd / (double)Nf, &sn, &cs);
        acc += 2.0 * ((double)Zm[k].x * cs - (double)Zm[k].y * sn);
    }
    acc += (double)Zm[Nf / 2].x * ((d & 1) ? -1.0 : 1.0);
    w[i] = (float)(acc / (double)Nf);
}

#ifdef VFPS_PHASE_CLOCKS
// Instrumented builds only: VFPS_PHASE_DUMP=<file> in the environment writes the per-phase clock
// stamps (first 64 steps of every CTA) of each persistent-kernel launch; synchronises the stream.
struct PhaseDump {
    vfps_sim *h; long long *dbg = nullptr; size_t n = 0; const char *path = nullptr;
    PhaseDump(vfps_sim *h_, size_t nctas) : h(h_)
    {
        path = std::getenv("VFPS_PHASE_DUMP");
        n = nctas * 64 * 8;
        if (path && cudaMalloc((void **)&dbg, n * sizeof(long long)) != cudaSuccess) { dbg = nullptr; path = nullptr; }
        if (dbg) cudaMemsetAsync(dbg, 0, n * sizeof(long long), h->stream);
    }
    ~PhaseDump()
    {
        if (!dbg) return;
        std::vector<long long> t(n);
        cudaMemcpyAsync(t.data(), dbg, n * sizeof(long long), cudaMemcpyDeviceToHost, h->stream);
        cudaStreamSynchronize(h->stream);
        cudaFree(dbg);
        if (FILE *f = std::fopen(path, "w")) {
            for (size_t i = 0; i < n; i += 8) {
                std::fprintf(f, "%zu %zu", i / (64 * 8), (i / 8) % 64);
                for (int k = 0; k < 8; ++k) std::fprintf(f, " %lld", t[i + k]);
                std::fprintf(f, "\n");
            }
            std::fclose(f);
        }
    }
};
#else
struct PhaseDump {
    long long *dbg = nullptr;
    PhaseDump(vfps_sim *, size_t) {}
};
#endif

// Launch (or occupancy query) of a persistent cluster kernel: grid = S x nclusters CTAs of `threads`
// threads, cluster dimension S, h->cl_smem bytes of dynamic shared memory; args = {&GridConst, &Args}.
cudaError_t cluster_launch_ptr(vfps_sim *h, const void *kern, int threads, int S, int nclusters, void **args,
                               bool query, int *max_clusters)
{
    if (!kern) return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->cl_smem);
    if (e != cudaSuccess) return e;
    if (S > 8) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(S * nclusters));
    cfg.blockDim = dim3((unsigned)threads);
    cfg.dynamicSmemBytes = h->cl_smem;
    cfg.stream = h->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)S;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (query) return cudaOccupancyMaxActiveClusters(max_clusters, kern, &cfg);
    return cudaLaunchKernelExC(&cfg, kern, args);
}

cudaError_t cluster_launch(vfps_sim *h, const ClusterArgs &A, int nclusters, bool query, int *mc)
{
    const bool manh = (h->P.flags & VFPS_FLAG_ROT_MANHATTAN) != 0;
    const void *kern = h->P.interp_order == 2 ? cluster_kernel_o2(h->N, manh)
                     : h->P.interp_order == 3 ? cluster_kernel_o3(h->N, manh) : cluster_kernel_o4(h->N, manh);
    void *args[2] = {(void *)&h->G, (void *)&A};
    return cluster_launch_ptr(h, kern, CL_THREADS, A.S, nclusters, args, query, mc);
}

// ---------------------------------------------------------------- second cluster design: host side
// Lagrange weights l_k(t) and their derivatives (Eq. 13, nodes k - floor((order-1)/2)), double.
void lagrange_d(int order, double t, double *l, double *lp)
{
    if (order == 2) {
        l[0] = 1.0 - t; l[1] = t; lp[0] = -1.0; lp[1] = 1.0;
    } else if (order == 3) {
        l[0] = 0.5 * t * (t - 1.0); l[1] = 1.0 - t * t; l[2] = 0.5 * t * (t + 1.0);
        lp[0] = t - 0.5; lp[1] = -2.0 * t; lp[2] = t + 0.5;
    } else {
        l[0] = -t * (t - 1.0) * (t - 2.0) / 6.0;
        l[1] = (t + 1.0) * (t - 1.0) * (t - 2.0) / 2.0;
        l[2] = -(t + 1.0) * t * (t - 2.0) / 2.0;
        l[3] = (t + 1.0) * t * (t - 1.0) / 6.0;
        lp[0] = -(3.0 * t * t - 6.0 * t + 2.0) / 6.0;
        lp[1] = (3.0 * t * t - 4.0 * t - 1.0) / 2.0;
        lp[2] = -(3.0 * t * t - 2.0 * t - 2.0) / 2.0;
        lp[3] = (3.0 * t * t - 1.0) / 6.0;
    }
}

// Geometry of the rotation in double precision (the same formulas as grid_constants)
struct RotGeomD {
    double a, b, d, x0c, y0c;
};
RotGeomD rot_geom_d(const vfps_params &P)
{
    const double PI = 3.14159265358979323846;
    const double dq = (P.q_max - P.q_min) / (P.N - 1), dp = (P.p_max - P.p_min) / (P.N - 1);
    const double dphi = 2.0 * PI / P.steps_per_period;
    const double sh = std::sin(0.5 * dphi), s = std::sin(dphi);
    RotGeomD g;
    g.a = -2.0 * sh * sh; g.b = -s * dp / dq; g.d = s * dq / dp;
    g.x0c = P.q_min / dq; g.y0c = P.p_min / dp;
    return g;
}

// First-order weight tables are used when the neglected term (a * half-span)^2 |l''| / 2 stays
// at the level of one fp32 ulp of a weight (|l''| <= 2 for the cubic basis).
bool onchip_tab_ok(const vfps_sim *h, int S)
{
    const RotGeomD g = rot_geom_d(h->P);
    const double span = 0.5 * (double)((h->N / S > h->N / 2 ? h->N / S : h->N) );
    (void)span;
    const double ex = std::fabs(g.a) * 0.5 * (double)(h->N / S), ey = std::fabs(g.a) * 0.5 * (double)h->N;
    const double e = ex > ey ? ex : ey;
    return e * e <= 1.2e-7;
}

// Column table (per rank and column), row table (per row), built in double and rounded once:
//   dx(x, y) = a X + b Y,  dy(x, y) = d X + a Y,  X = x + x0c, Y = y + y0c
//   column y of rank r is "good" if floor(dx) is the same for all rows of the rank (ix),
//   row x is "good" if floor(dy) is the same for all columns (iy)
//   TAB:  M_i(y) = l_i(t0x), M'_i = l_i'(t0x), t0x = a Xc(r) + b Y - ix, Xc = centre row of the rank
//         L_j(x) = l_j(t0y), L'_j = l_j'(t0y), t0y = d X + a Ymid - iy;  e_x(x) = a (X - Xc)
//         packed per order so that the kernel fetches a row with two or three vector loads
//         (the kernel forms e_y(y) = a (y - (N-1)/2) itself)
//   else: column {b Y - ix, a Y}, row {X, d X - iy}: the kernel evaluates the weights per cell
int onchip_tables(vfps_sim *h, int S)
{
    const int N = h->N, R = N / S, order = h->P.interp_order;
    const RotGeomD g = rot_geom_d(h->P);
    const bool tab = onchip_tab_ok(h, S);
    std::vector<float> col((size_t)S * N * OC_COLTAB, 0.0f), row((size_t)N * OC_ROWTAB, 0.0f);
    std::vector<int> cix((size_t)S * N, OC_BAD);
    const double Ymid = 0.5 * (double)(N - 1) + g.y0c;
    for (int r = 0; r < S; ++r) {
        const double Xlo = (double)(r * R) + g.x0c, Xhi = (double)(r * R + R - 1) + g.x0c, Xc = 0.5 * (Xlo + Xhi);
        for (int y = 0; y < N; ++y) {
            const double Y = (double)y + g.y0c;
            const double f0 = std::floor(g.a * Xlo + g.b * Y), f1 = std::floor(g.a * Xhi + g.b * Y);
            float *c = &col[((size_t)r * N + y) * OC_COLTAB];
            if (f0 != f1) continue;                                   // dx is monotonic in x
            cix[(size_t)r * N + y] = (int)f0;
            if (tab) {
                double l[4] = {0, 0, 0, 0}, lp[4] = {0, 0, 0, 0};
                lagrange_d(order, g.a * Xc + g.b * Y - f0, l, lp);
                for (int i = 0; i < 4; ++i) { c[i] = (float)l[i]; c[4 + i] = (float)lp[i]; }
            } else {
                c[0] = (float)(g.b * Y - f0);
                c[1] = (float)(g.a * Y);
            }
        }
    }
    for (int x = 0; x < N; ++x) {
        const double X = (double)x + g.x0c;
        const double Ylo = g.y0c, Yhi = (double)(N - 1) + g.y0c;
        const double f0 = std::floor(g.d * X + g.a * Ylo), f1 = std::floor(g.d * X + g.a * Yhi);
        float *t = &row[(size_t)x * OC_ROWTAB];
        int iy = OC_BAD;
        if (f0 == f1) {
            iy = (int)f0;
            const int r = x / R;
            const double Xc = 0.5 * ((double)(r * R) + (double)(r * R + R - 1)) + g.x0c;
            if (tab) {
                // order 4: L[0..3] L'[1,2,3,0] ex;  order 3: L[0..2] ex L'[0..2];  order 2: L[0..1] L'[0..1] ex
                double l[4] = {0, 0, 0, 0}, lp[4] = {0, 0, 0, 0};
                lagrange_d(order, g.d * X + g.a * Ymid - f0, l, lp);
                const int olp = (order == 2) ? 2 : 4, oex = (order == 4) ? 8 : (order == 3) ? 3 : 4;
                // order 4: L' rotated by one (L'1 L'2 L'3 L'0), see Walker::load_tab
                for (int j = 0; j < order; ++j) { t[j] = (float)l[j]; t[olp + (order == 4 ? (j + 3) % 4 : j)] = (float)lp[j]; }
                t[oex] = (float)(g.a * (X - Xc));
            } else {
                t[8] = (float)X;
                t[9] = (float)(g.d * X - f0);
            }
        }
        std::memcpy(&t[10], &iy, sizeof(int));
    }
    if (!h->oc_coltab) {
        CU(dalloc(h, &h->oc_coltab, (size_t)OC_MAX_S * N * OC_COLTAB));
        CU(dalloc(h, &h->oc_colix, (size_t)OC_MAX_S * N));
        CU(dalloc(h, &h->oc_rowtab, (size_t)N * OC_ROWTAB));
        CU(dalloc(h, &h->oc_item_ctr, (size_t)1));
        CU(dalloc(h, &h->oc_member_done, (size_t)h->members));
        CU(cudaMemsetAsync(h->oc_item_ctr, 0, sizeof(unsigned long long), h->stream));
        CU(cudaMemsetAsync(h->oc_member_done, 0, (size_t)h->members * sizeof(unsigned int), h->stream));
    }
    // pageable host memory: the copies are staged before the calls return
    CU(cudaMemcpyAsync(h->oc_coltab, col.data(), col.size() * sizeof(float), cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(h->oc_colix, cix.data(), cix.size() * sizeof(int), cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(h->oc_rowtab, row.data(), row.size() * sizeof(float), cudaMemcpyHostToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    h->oc_tab = tab;
    h->oc_tab_S = S;
    return VFPS_OK;
}

cudaError_t onchip_launch(vfps_sim *h, const OnchipArgs &A, int nclusters, bool query, int *mc)
{
    const bool clamp = (h->P.flags & VFPS_FLAG_CLAMP) != 0;
    const void *kern = h->P.interp_order == 2 ? onchip_kernel_o2(h->N, h->oc_tab, clamp)
                     : h->P.interp_order == 3 ? onchip_kernel_o3(h->N, h->oc_tab, clamp)
                                              : onchip_kernel_o4(h->N, h->oc_tab, clamp);
    void *args[2] = {(void *)&h->G, (void *)&A};
    return cluster_launch_ptr(h, kern, OC_THREADS, A.S, nclusters, args, query, mc);
}

// feasibility of the second cluster design for cluster size S; fills cl_smem / cl_max_clusters
bool onchip_try(vfps_sim *h, int S, int smem_max)
{
    const int N = h->N, H = h->G.H;
    if (!(N == 64 || N == 128 || N == 256 || N == 512)) return false;
    if (h->P.flags & VFPS_FLAG_ROT_MANHATTAN) return false;
    if (H > OC_MAX_H || N % S) return false;
    const int R = N / S;
    if (R < 4 || (R & 3) || R < H) return false;
    const OnchipLayout L = onchip_layout(N, S, H, h->P.interp_order);
    if (L.RPW < H) return false;
    const size_t bytes = L.total_floats * sizeof(float);
    if (bytes > (size_t)smem_max) return false;
    const size_t keep = h->cl_smem;
    const bool keep_tab = h->oc_tab;
    h->cl_smem = bytes;
    h->oc_tab = onchip_tab_ok(h, S);
    OnchipArgs A{};
    A.S = S; A.R = R;
    int mc = 0;
    cudaError_t e = onchip_launch(h, A, 1, true, &mc);
    if (e != cudaSuccess || mc < 1) { cudaGetLastError(); h->cl_smem = keep; h->oc_tab = keep_tab; return false; }
    h->cl_max_clusters = mc;
    return true;
}

// split the n steps of a call into chunks so that (chunks x members) work items fill the
// resident clusters evenly (a 256-member batch on 74 clusters: 2 chunks -> 512 items, 98.8 %)
void onchip_chunks(const vfps_sim *h, int n, int nclusters, int *nchunks, int *chunk)
{
    *nchunks = 1; *chunk = n;
    if (h->members <= nclusters) return;
    double best = 0.0;
    for (int c = 1; c <= 8 && n / c >= 32; ++c) {
        const long long items = (long long)c * h->members;
        const long long rounds = (items + nclusters - 1) / nclusters;
        const double eff = (double)items / (double)(rounds * nclusters);
        if (eff > best + 1e-9) { best = eff; *nchunks = c; }
        if (eff >= 0.97) break;
    }
    *chunk = (n + *nchunks - 1) / *nchunks;
    *nchunks = (n + *chunk - 1) / *chunk;
}

int launch_onchip_steps(vfps_sim *h, int n, float *diag)
{
    if (h->oc_tab_S != h->cl_S) {
        int rc = onchip_tables(h, h->cl_S);
        if (rc != VFPS_OK) return rc;
    }
    OnchipArgs A{};
    A.psi = h->psi; A.scale = h->scale; A.wfun = h->has_wake ? h->wfun : nullptr; A.diag = diag;
    A.coltab = h->oc_coltab; A.colix = h->oc_colix; A.rowtab = h->oc_rowtab;
    A.members = h->members; A.S = h->cl_S; A.R = h->N / h->cl_S;
    const int nclusters = h->members < h->cl_max_clusters ? h->members : h->cl_max_clusters;
    int nchunks = 1, chunk = n;
    onchip_chunks(h, n, nclusters, &nchunks, &chunk);
    A.nsteps = chunk; A.nchunks = nchunks; A.last_steps = n - (nchunks - 1) * chunk;
    A.item_ctr = h->oc_item_ctr; A.item_base = h->oc_item_base;
    A.member_done = h->oc_member_done; A.done_base = h->oc_done_base;
    cudaError_t e;
    {
        PhaseDump pd(h, (size_t)A.S * nclusters);
        A.dbg = pd.dbg;
        Bracket br(h, VFPS_KERNEL_CLUSTER, h->timing);
        e = onchip_launch(h, A, nclusters, false, nullptr);
    }
    if (e != cudaSuccess) return fail(h, VFPS_ERR_CUDA, std::string("cluster launch: ") + cudaGetErrorString(e));
    // every cluster fetches until it draws an item past the end: nclusters extra fetches per launch
    h->oc_item_base += (unsigned long long)nchunks * (unsigned long long)h->members + (unsigned long long)nclusters;
    h->oc_done_base += (unsigned int)nchunks;
    h->launches += 1;
    return VFPS_OK;
}

// Pick the cluster kernel and size.  Kernel: the request (cl_ver_opt) or, on AUTO, the scalar
// kernel (1).  Size: the request (cl_S_opt) if
// feasible; otherwise the largest feasible size for a single simulation (shortest step), the
// smallest for a batch (most work per barrier).
void cluster_configure(vfps_sim *h)
{
    h->cl_S = 0; h->cl_max_clusters = 0; h->cl_ver = 0; h->cl_why.clear();
    const int N = h->N, H = h->G.H;
    int dev = 0, smem_max = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    const int cand_single[5] = {16, 8, 4, 2, 1}, cand_batch[5] = {1, 2, 4, 8, 16};
    const int *cand = (h->members == 1) ? cand_single : cand_batch;
    // in-place design (k_onchip_step, kernel id 3): standard rotation, free or clamped interpolation
    auto try_inplace = [&]() -> bool {
        for (int c = 0; c < 5; ++c) {
            const int S = cand[c];
            if (h->cl_S_opt && S != h->cl_S_opt) continue;
            if (!onchip_try(h, S, smem_max)) continue;
            h->cl_S = S; h->cl_ver = 3;
            return true;
        }
        return false;
    };
    // first design (k_cluster_step, kernel id 1): free interpolation; also the Manhattan rotation
    auto try_first = [&]() -> bool {
        if (h->P.flags & VFPS_FLAG_CLAMP) { h->cl_why = "k_cluster_step implements free (un-clamped) interpolation only"; return false; }
        if (!(N == 32 || N == 64 || N == 128 || N == 256 || N == 512)) { h->cl_why = "cluster engine supports N = 32, 64, 128, 256, 512"; return false; }
        if (H > CL_PAD) { h->cl_why = "rotation halo exceeds the cluster engine's row padding"; return false; }
        for (int c = 0; c < 5; ++c) {
            const int S = cand[c];
            if (h->cl_S_opt && S != h->cl_S_opt) continue;
            if (N / S < (H > 1 ? H : 1) || N % S) continue;
            const int R = N / S;
            const size_t bytes = cluster_smem_floats(N, S, H) * sizeof(float);
            if (bytes > (size_t)smem_max) continue;
            h->cl_smem = bytes;
            h->cl_ver = 1;
            ClusterArgs A{};
            A.S = S; A.R = R;
            int mc = 0;
            cudaError_t e = cluster_launch(h, A, 1, true, &mc);
            if (e != cudaSuccess || mc < 1) { cudaGetLastError(); continue; }
            h->cl_S = S; h->cl_max_clusters = mc;
            return true;
        }
        h->cl_why = "no feasible cluster size (shared memory or cluster scheduling)";
        return false;
    };
    if (h->cl_ver_opt == 3) {
        if (!try_inplace()) h->cl_why = "in-place cluster kernel not feasible for this grid / flags / cluster size";
        return;
    }
    if (h->cl_ver_opt == 1) { try_first(); return; }
    // AUTO.  A batch: the in-place kernel (a 256^2 member on two CTAs: every SM busy).  One simulation of up to
    // 256^2 on 16 CTAs is a chain of short phases, where the first design's lighter per-step set-up wins
    // (measured: C0 1.79 against 2.99 us per step, C1 3.56 against 3.79; 512^2: 9.40 against 9.20).
    const bool first_preferred = (h->members == 1 && N <= 256);
    if (first_preferred) { if (try_first()) return; h->cl_ver = 0; if (try_inplace()) { h->cl_why.clear(); return; } return; }
    if (try_inplace()) return;
    if (try_first()) return;
    h->cl_ver = 0;
    h->cl_why = "no feasible cluster size (shared memory or cluster scheduling)";
}

int launch_cluster_steps(vfps_sim *h, int n, float *diag)
{
    if (h->cl_ver == 3) return launch_onchip_steps(h, n, diag);
    ClusterArgs A{};
    A.psi = h->psi; A.scale = h->scale; A.wfun = h->has_wake ? h->wfun : nullptr; A.diag = diag;
    A.members = h->members; A.nsteps = n; A.S = h->cl_S; A.R = h->N / h->cl_S;
    const int nclusters = h->members < h->cl_max_clusters ? h->members : h->cl_max_clusters;
    cudaError_t e;
    {
        PhaseDump pd(h, (size_t)A.S * nclusters);
        A.dbg = pd.dbg;
        Bracket br(h, VFPS_KERNEL_CLUSTER, h->timing);
        e = cluster_launch(h, A, nclusters, false, nullptr);
    }
    if (e != cudaSuccess) return fail(h, VFPS_ERR_CUDA, std::string("cluster launch: ") + cudaGetErrorString(e));
    h->launches += 1;
    return VFPS_OK;
}

const void *grid_kernel(const vfps_sim *h)
{
    const bool manh = (h->P.flags & VFPS_FLAG_ROT_MANHATTAN) != 0, clamp = (h->P.flags & VFPS_FLAG_CLAMP) != 0;
    switch (h->P.interp_order) {
        case 2: return grid_kernel_o2(manh, clamp);
        case 3: return grid_kernel_o3(manh, clamp);
        default: return grid_kernel_o4(manh, clamp);
    }
}

// The cooperative-grid engine needs every CTA resident at once: grid = SMs x (CTAs per SM, at most
// two), rows of the kick phase dealt out evenly.
void grid_configure(vfps_sim *h)
{
    h->gr_blocks = 0; h->gr_why.clear();
    if (h->members != 1) { h->gr_why = "grid engine advances one simulation per handle"; return; }
    int dev = 0, coop = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (!coop) { h->gr_why = "device does not support cooperative launches"; return; }
    const int N = h->N;
    int blocks = 2 * sms;
    for (int pass = 0; pass < 2; ++pass) {
        const int KR = (N + blocks - 1) / blocks;
        const size_t smem = grid_smem_floats(N, KR, (h->P.flags & VFPS_FLAG_CLAMP) != 0) * sizeof(float);
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, grid_kernel(h), GR_THREADS, smem);
        if (e != cudaSuccess || per_sm < 1) { cudaGetLastError(); h->gr_why = "grid kernel does not fit an SM"; return; }
        const int fit = sms * (per_sm < 2 ? per_sm : 2);
        if (fit >= blocks) { h->gr_blocks = blocks; h->gr_KR = KR; h->gr_smem = smem; return; }
        blocks = fit;
    }
    h->gr_why = "grid kernel occupancy query did not converge";
}

// ---------------------------------------------------------------- TMA-staged grid engine: host side
const void *grid2_kernel(const vfps_sim *h)
{
    const bool clamp = (h->P.flags & VFPS_FLAG_CLAMP) != 0;
    switch (h->P.interp_order) {
        case 2: return grid2_kernel_o2(false);      // linear interpolation: the clamp is the identity
        case 3: return grid2_kernel_o3(clamp);
        default: return grid2_kernel_o4(clamp);
    }
}

// Weight tables of k_grid2_step for `nb` row stripes (as onchip_tables, one stripe per CTA) and the
// tensor map of psi with a box of 144 columns x (KRmax + 2H) rows.  Leaves g2_blocks = 0 with the
// reason in g2_why when the engine does not apply.
int grid2_configure(vfps_sim *h)
{
    h->g2_blocks = 0; h->g2_why.clear();
    const int N = h->N, H = h->G.H, order = h->P.interp_order;
    if (h->members != 1) { h->g2_why = "one simulation per handle"; return VFPS_OK; }
    if (h->P.flags & VFPS_FLAG_ROT_MANHATTAN) { h->g2_why = "standard rotation only"; return VFPS_OK; }
    if (N % 256 != 0) { h->g2_why = "N must be a multiple of 256"; return VFPS_OK; }
    if (H > G2_MAX_H) { h->g2_why = "rotation halo exceeds 4 rows"; return VFPS_OK; }
    int dev = 0, coop = 0, sms = 0, smem_max = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (!coop) { h->g2_why = "device does not support cooperative launches"; return VFPS_OK; }
    const int nb = sms < N ? sms : N;
    const RotGeomD g = rot_geom_d(h->P);
    // Row stripes.  floor(dy) is constant along a row and changes between two rows at most a few times over the grid
    // (once, through the rotation centre, for the usual boxes); a stripe that contains such a change splits its rotation
    // into two runs and is the last to arrive at every barrier.  So the stripes are dealt out per segment of constant
    // floor(dy), CTAs in proportion to the rows, as evenly as possible inside a segment -- unless that makes the
    // tallest stripe taller than the even split of all rows does.
    std::vector<int> row0(nb + 1, 0);
    int KRmax = (N + nb - 1) / nb;
    {
        auto row_floor = [&](int x) {
            const double X = (double)x + g.x0c;
            const double f0 = std::floor(g.d * X + g.a * g.y0c), f1 = std::floor(g.d * X + g.a * ((double)(N - 1) + g.y0c));
            return f0 == f1 ? (int)f0 : OC_BAD;
        };
        std::vector<int> seg(1, 0);                          // first rows of the segments
        for (int x = 1, last = row_floor(0); x < N; ++x) {
            const int f = row_floor(x);
            if (f == OC_BAD) continue;                       // a row that changes along itself stays with its predecessor
            if (last != OC_BAD && f != last) seg.push_back(x);
            last = f;
        }
        seg.push_back(N);
        const int ns = (int)seg.size() - 1;
        std::vector<int> cnt(ns, 0);
        bool ok = ns >= 2 && ns <= nb;
        if (ok) {
            int used = 0;
            std::vector<std::pair<double, int>> frac;
            for (int i = 0; i < ns; ++i) {
                const double share = (double)nb * (seg[i + 1] - seg[i]) / N;
                cnt[i] = (int)share < 1 ? 1 : (int)share;
                used += cnt[i];
                frac.push_back({share - std::floor(share), i});
            }
            std::sort(frac.begin(), frac.end(), [](const std::pair<double, int> &a, const std::pair<double, int> &b) { return a.first > b.first; });
            for (int k = 0; used < nb && k < ns; ++k, ++used) ++cnt[frac[k].second];
            ok = used == nb;
            for (int i = 0; ok && i < ns; ++i) ok = (seg[i + 1] - seg[i] + cnt[i] - 1) / cnt[i] <= KRmax && cnt[i] <= seg[i + 1] - seg[i];
        }
        if (ok) {
            int c = 0;
            for (int i = 0; i < ns; ++i) {
                const int len = seg[i + 1] - seg[i], lo = len / cnt[i], extra = len % cnt[i];
                for (int k = 0; k < cnt[i]; ++k, ++c) row0[c + 1] = row0[c] + lo + (k < extra ? 1 : 0);
            }
        } else {
            const int lo = N / nb, extra = N % nb;
            for (int c = 0; c < nb; ++c) row0[c + 1] = row0[c] + lo + (c < extra ? 1 : 0);
        }
    }
    const bool clamp = (h->P.flags & VFPS_FLAG_CLAMP) != 0 && order > 2;
    // two tile buffers per warp group where they fit beside the stripe's rows, else one
    int nbuf = 2;
    Grid2Layout L = grid2_layout(N, KRmax, H, nbuf, clamp);
    if (L.total_floats * sizeof(float) + 256 > (size_t)smem_max) { nbuf = 1; L = grid2_layout(N, KRmax, H, nbuf, clamp); }
    const size_t bytes = L.total_floats * sizeof(float);
    if (bytes + 256 > (size_t)smem_max) { h->g2_why = "tiles and row buffer do not fit shared memory"; return VFPS_OK; }
    if (L.box_rows > 256) { h->g2_why = "TMA box too tall"; return VFPS_OK; }
    {   // first-order weight tables must be exact to fp32 rounding over a stripe and over the columns
        const double ex = std::fabs(g.a) * 0.5 * (double)KRmax, ey = std::fabs(g.a) * 0.5 * (double)N;
        const double e = ex > ey ? ex : ey;
        if (e * e > 1.2e-7) { h->g2_why = "rotation angle too large for first-order weight tables"; return VFPS_OK; }
    }
    const void *kern = grid2_kernel(h);
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess) {
        cudaGetLastError(); h->g2_why = "shared-memory opt-in refused"; return VFPS_OK;
    }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, G2_THREADS, bytes) != cudaSuccess || per_sm < 1) {
        cudaGetLastError(); h->g2_why = "kernel does not fit an SM"; return VFPS_OK;
    }
    // ---- tensor map of psi: dim 0 = p (contiguous), dim 1 = q; out-of-range parts of a box read as zero (A8)
    typedef CUresult (*EncodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError(); h->g2_why = "cuTensorMapEncodeTiled not available"; return VFPS_OK;
    }
    // (8-byte elements = pairs of floats: a box dimension is limited to 256 elements, a tile row has 272 floats)
    const cuuint64_t gdim[2] = {(cuuint64_t)N / 2, (cuuint64_t)N};
    const cuuint64_t gstr[1] = {(cuuint64_t)N * sizeof(float)};
    const cuuint32_t box[2] = {(cuuint32_t)G2_SUBW / 2, (cuuint32_t)L.box_rows};
    const cuuint32_t estr[2] = {1, 1};
    if (((EncodeTiled)fn)(&h->g2_tmap, CU_TENSOR_MAP_DATA_TYPE_UINT64, 2, (void *)h->psi, gdim, gstr, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) {
        h->g2_why = "cuTensorMapEncodeTiled failed"; return VFPS_OK;
    }
    // ---- tables, in double, rounded once
    std::vector<float> col((size_t)nb * N, 0.0f), row((size_t)N * OC_ROWTAB, 0.0f);
    std::vector<int> cix((size_t)nb * N, OC_BAD);
    const double Ymid = 0.5 * (double)(N - 1) + g.y0c;
    for (int c = 0; c < nb; ++c) {
        const int r0 = row0[c], nr = row0[c + 1] - r0;
        const double Xlo = (double)r0 + g.x0c, Xhi = (double)(r0 + nr - 1) + g.x0c, Xc = 0.5 * (Xlo + Xhi);
        for (int y = 0; y < N; ++y) {
            const double Y = (double)y + g.y0c;
            const double f0 = std::floor(g.a * Xlo + g.b * Y), f1 = std::floor(g.a * Xhi + g.b * Y);
            if (f0 != f1) continue;
            cix[(size_t)c * N + y] = (int)f0;
            col[(size_t)c * N + y] = (float)(g.a * Xc + g.b * Y - f0);     // the kernel forms M, M' from it (Eq. 13)
        }
        for (int x = r0; x < r0 + nr; ++x) {
            const double X = (double)x + g.x0c;
            const double f0 = std::floor(g.d * X + g.a * g.y0c), f1 = std::floor(g.d * X + g.a * ((double)(N - 1) + g.y0c));
            float *t = &row[(size_t)x * OC_ROWTAB];
            int iy = OC_BAD;
            if (f0 == f1) {
                iy = (int)f0;
                double l[4] = {0, 0, 0, 0}, lp[4] = {0, 0, 0, 0};
                lagrange_d(order, g.d * X + g.a * Ymid - f0, l, lp);
                const int olp = (order == 2) ? 2 : 4, oex = (order == 4) ? 8 : (order == 3) ? 3 : 4;
                for (int j = 0; j < order; ++j) { t[j] = (float)l[j]; t[olp + (order == 4 ? (j + 3) % 4 : j)] = (float)lp[j]; }
                t[oex] = (float)(g.a * (X - Xc));
            }
            std::memcpy(&t[10], &iy, sizeof(int));
        }
    }
    if (!h->g2_coltab) {
        CU(dalloc(h, &h->g2_coltab, col.size()));
        CU(dalloc(h, &h->g2_colix, cix.size()));
        CU(dalloc(h, &h->g2_rowtab, row.size()));
        CU(dalloc(h, &h->g2_row0, row0.size()));
        CU(dalloc(h, &h->g2_rho, (size_t)N));
        CU(dalloc(h, &h->g2_mom, (size_t)2 * nb * G2_NPART));
        CU(dalloc(h, &h->g2_qacc, (size_t)16 + (size_t)16 * nb));   // three charge accumulators, barrier counter, one 128-byte flag line per CTA
    }
    CU(cudaMemcpyAsync(h->g2_coltab, col.data(), col.size() * sizeof(float), cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(h->g2_colix, cix.data(), cix.size() * sizeof(int), cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(h->g2_rowtab, row.data(), row.size() * sizeof(float), cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(h->g2_row0, row0.data(), row0.size() * sizeof(int), cudaMemcpyHostToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    h->g2_nbuf = nbuf;
    h->g2_blocks = nb; h->g2_KRmax = KRmax; h->g2_smem = bytes;
    return VFPS_OK;
}

int launch_grid2_steps(vfps_sim *h, int n, float *diag)
{
    Grid2Args A{};
    A.psi = h->psi; A.scale = h->scale; A.wfun = h->has_wake ? h->wfun : nullptr;
    A.rho = h->g2_rho; A.mom_part = h->g2_mom; A.diag = diag; A.nsteps = n;
    A.coltab = h->g2_coltab; A.colix = h->g2_colix; A.rowtab = h->g2_rowtab; A.qacc = h->g2_qacc;
    A.row0 = h->g2_row0; A.KRmax = h->g2_KRmax; A.nbuf = h->g2_nbuf;
    A.bar = reinterpret_cast<unsigned int *>(h->g2_qacc + 3);
    A.flags = reinterpret_cast<unsigned int *>(h->g2_qacc + 16);
    if (cudaMemsetAsync(h->g2_qacc, 0, (16 + (size_t)16 * h->g2_blocks) * sizeof(unsigned long long), h->stream) != cudaSuccess)
        return fail(h, VFPS_ERR_CUDA, "cudaMemsetAsync failed");
    const void *kern = grid2_kernel(h);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->g2_smem);
    if (e == cudaSuccess) {
        PhaseDump pd(h, (size_t)h->g2_blocks);
        A.dbg = pd.dbg;
        void *args[3] = {(void *)&h->G, (void *)&A, (void *)&h->g2_tmap};
        Bracket br(h, VFPS_KERNEL_GRID2, h->timing);
        e = cudaLaunchCooperativeKernel(kern, dim3((unsigned)h->g2_blocks), dim3(G2_THREADS), args, h->g2_smem, h->stream);
    }
    if (e != cudaSuccess) return fail(h, VFPS_ERR_CUDA, std::string("cooperative launch (grid2): ") + cudaGetErrorString(e));
    h->launches += 1;
    return VFPS_OK;
}

// which kernel the GRID engine runs: the request, else the TMA-staged one where it applies
int grid_kernel_in_use(const vfps_sim *h)
{
    if (h->gr_ver_opt == 1) return h->gr_blocks > 0 ? 1 : 0;
    if (h->gr_ver_opt == 2) return h->g2_blocks > 0 ? 2 : 0;
    if (h->g2_blocks > 0) return 2;
    return h->gr_blocks > 0 ? 1 : 0;
}

int launch_grid_steps(vfps_sim *h, int n, float *diag)
{
    GridArgs A{};
    A.psi = h->psi; A.psi_tmp = h->psi_tmp; A.scale = h->scale; A.wfun = h->has_wake ? h->wfun : nullptr;
    A.rho_part = h->rho_part; A.mom_part = h->gr_mom; A.diag = diag; A.nsteps = n;
    A.tiles_y = h->tiles_y2; A.KR = h->gr_KR; A.qacc = h->gr_qacc; A.zrow = h->gr_zrow;
    if (cudaMemsetAsync(h->gr_qacc, 0, 2 * sizeof(unsigned long long), h->stream) != cudaSuccess)
        return fail(h, VFPS_ERR_CUDA, "cudaMemsetAsync failed");
    void *args[2] = {(void *)&h->G, (void *)&A};
    const void *kern = grid_kernel(h);
    cudaError_t e;
    {
        PhaseDump pd(h, (size_t)h->gr_blocks);
        A.dbg = pd.dbg;
        Bracket br(h, VFPS_KERNEL_GRID, h->timing);
        e = cudaLaunchCooperativeKernel(kern, dim3((unsigned)h->gr_blocks), dim3(GR_THREADS), args, h->gr_smem, h->stream);
    }
    if (e != cudaSuccess) return fail(h, VFPS_ERR_CUDA, std::string("cooperative launch: ") + cudaGetErrorString(e));
    h->launches += 1;
    return VFPS_OK;
}

// k_wake_fft needs the opt-in for more than 48 KB of dynamic shared memory (Nf >= 4096).  The
// attribute belongs to the function, not to a handle: it is only ever raised (per device).
cudaError_t wake_fft_attr(const vfps_sim *h)
{
    static size_t granted[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) dev = 0;
    if (h->fft_smem <= granted[dev]) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(k_wake_fft, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->fft_smem);
    if (e == cudaSuccess) granted[dev] = h->fft_smem;
    return e;
}

// how the STREAM / GRAPH engines evaluate the wake
bool wake_is_direct(const vfps_sim *h) { return h->wake_opt != VFPS_WAKE_FFT; }

template <int ORDER, bool CLAMP>
int launch_step_stream2(vfps_sim *h, bool timed)
{
    const int N = h->N;
    const bool direct = wake_is_direct(h);
    const bool manh = (h->P.flags & VFPS_FLAG_ROT_MANHATTAN) != 0;
    {
        Bracket br(h, VFPS_KERNEL_ROTATE2, timed);
        if (manh)
            k_drift2<ORDER, CLAMP><<<dim3(h->tiles_x2 * h->tiles_y2, h->members), R2_THREADS, 0, h->stream>>>(
                h->G, h->psi, h->psi_tmp, h->scale, h->rho_part, h->tiles_y2, h->rho, h->tilectr);
        else
            k_rotate2<ORDER, CLAMP><<<dim3(h->tiles_x2 * h->tiles_y2, h->members), R2_THREADS, 0, h->stream>>>(
                h->G, h->psi, h->psi_tmp, h->scale, h->rho_part, h->tiles_y2, h->rho, h->tilectr);
    }
    // Manhattan + clamp: the clamped RF kick changes the profile (k_rf_profile); rho then replaces
    // the drift's partial sums as the wake's input
    const bool rfp = manh && CLAMP && h->has_wake;
    if (rfp) {
        k_rf_profile<ORDER><<<dim3((N + 7) / 8, h->members), 256, 0, h->stream>>>(h->G, h->psi_tmp, h->rho);
        h->launches += 1;
    }
    if (!direct) {
        Bracket br(h, VFPS_KERNEL_WAKE, timed);
        wake_fft_attr(h);
        k_wake_fft<<<h->members, h->fft_threads, h->fft_smem, h->stream>>>(
            N, h->Nf, h->log2Nf, h->G.dq, rfp ? h->rho : h->rho_part, rfp ? 1 : h->tiles_y2,
            h->has_wake ? h->Z : nullptr, h->tw, h->rho, h->V, h->qstat);
        h->launches += 1;
    } else if (h->has_wake) {      // without an impedance V stays 0 (set at create) and P = 0
        Bracket br(h, VFPS_KERNEL_WAKE_DIRECT, timed);
        const size_t wd_smem = (size_t)((CLAMP ? 3 : 2) * N + 2 * WD_ROWS) * sizeof(float);
        if (wd_smem > 48 * 1024) {       // N = 4096 with the transposed wake: opt-in, only ever raised
            static size_t granted = 0;
            if (wd_smem > granted &&
                cudaFuncSetAttribute(k_wake_direct, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)wd_smem) == cudaSuccess)
                granted = wd_smem;
        }
        k_wake_direct<<<dim3(h->wd_blocks, h->members), WD_THREADS, wd_smem, h->stream>>>(
            N, h->rho, h->wfun, h->V, h->pw_part, CLAMP ? h->dpU : nullptr, h->G.dp);
        h->launches += 1;
    }
    Kfp2Args A;
    A.psi_in = h->psi_tmp; A.psi_out = h->psi; A.V = h->V; A.qstat = h->qstat;
    A.pw_part = direct ? h->pw_part : nullptr; A.npw = h->wd_blocks;
    A.dpU = (CLAMP && direct && h->has_wake) ? h->dpU : nullptr;
    A.mom_part = h->mom_part; A.scale = h->scale; A.blkctr = h->blkctr; A.rowctr = h->rowctr;
    A.diag = h->diag_cell; A.members = h->members; A.rows_per_cta = h->kfp2_rows;
    {
        Bracket br(h, VFPS_KERNEL_KICK_FP2, timed);
        if (manh) k_kick_fp2<ORDER, true, CLAMP><<<dim3(h->kfp2_blocks, h->members), K2_THREADS, 0, h->stream>>>(h->G, A);
        else k_kick_fp2<ORDER, false, CLAMP><<<dim3(h->kfp2_blocks, h->members), K2_THREADS, 0, h->stream>>>(h->G, A);
    }
    h->launches += 2;
    return VFPS_OK;
}

int launch_step(vfps_sim *h, bool timed)
{
    const bool clamp = (h->P.flags & VFPS_FLAG_CLAMP) != 0;
    switch (h->P.interp_order) {
        case 2: return clamp ? launch_step_stream2<2, true>(h, timed) : launch_step_stream2<2, false>(h, timed);
        case 3: return clamp ? launch_step_stream2<3, true>(h, timed) : launch_step_stream2<3, false>(h, timed);
        default: return clamp ? launch_step_stream2<4, true>(h, timed) : launch_step_stream2<4, false>(h, timed);
    }
}

// the engine the next vfps_step uses
int resolved_engine(const vfps_sim *h)
{
    if (h->engine_opt == VFPS_ENGINE_STREAM) return VFPS_ENGINE_STREAM;
    if (h->engine_opt == VFPS_ENGINE_GRAPH) return VFPS_ENGINE_GRAPH;
    if (h->engine_opt == VFPS_ENGINE_GRID) return VFPS_ENGINE_GRID;
    if (h->engine_opt == VFPS_ENGINE_CLUSTER) return VFPS_ENGINE_CLUSTER;
    // AUTO: on-chip grids -> cluster; one large simulation -> cooperative grid; else graph replay.
    // One 512^2 simulation: the TMA-staged grid kernel on 148 SMs beats the cluster of 16 (8.3 against 8.85 us per step)
    if (h->members == 1 && h->N >= 512 && h->g2_blocks > 0 && h->gr_ver_opt != 1) return VFPS_ENGINE_GRID;
    if (h->cl_S > 0) return VFPS_ENGINE_CLUSTER;
    return (h->gr_blocks > 0 || h->g2_blocks > 0) ? VFPS_ENGINE_GRID : VFPS_ENGINE_GRAPH;
}

// the captured graph depends on the kernel generation and the wake mode
void drop_graph(vfps_sim *h)
{
    if (!h->graph_exec) return;
    cudaStreamSynchronize(h->stream);
    cudaGraphExecDestroy(h->graph_exec);
    h->graph_exec = nullptr;
}

// capture GRAPH_STEPS split steps once; every step is the same three launches (the diag row and
// the caller's diag pointer live in device memory), so the instantiated graph is reusable
int ensure_graph(vfps_sim *h)
{
    if (h->graph_exec) return VFPS_OK;
    cudaStream_t cap = nullptr;
    CU(cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    cudaStream_t user = h->stream;
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
        h->stream = cap;
        const long long l0 = h->launches;
        for (int i = 0; i < GRAPH_STEPS; ++i) launch_step(h, false);
        h->graph_launches = h->launches - l0;
        h->launches = l0;
        h->stream = user;
        e = cudaStreamEndCapture(cap, &g);
    }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&h->graph_exec, g, 0);
    if (g) cudaGraphDestroy(g);
    cudaStreamDestroy(cap);
    if (e != cudaSuccess) {
        h->graph_exec = nullptr;
        return fail(h, VFPS_ERR_CUDA, std::string("CUDA graph capture: ") + cudaGetErrorString(e));
    }
    return VFPS_OK;
}

int create_impl(const vfps_params *p, const vfps_complex *Z, bool z_on_host, void *cuda_stream,
                vfps_handle *out)
{
    vfps_sim *h = nullptr;
    if (!out) return fail(nullptr, VFPS_ERR_ARG, "out is NULL");
    *out = nullptr;
    std::string why;
    int rc = validate(p, why);
    if (rc != VFPS_OK) return fail(nullptr, rc, why);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return fail(nullptr, VFPS_ERR_CUDA, "no CUDA device: this library has no CPU fallback");
    h = new (std::nothrow) vfps_sim();
    if (!h) return fail(nullptr, VFPS_ERR_NOMEM, "host allocation failed");
    h->P = *p;
    h->N = p->N; h->Nf = p->N * p->pad; h->members = p->members;
    h->log2Nf = 0; while ((1 << h->log2Nf) < h->Nf) ++h->log2Nf;
    h->stream = (cudaStream_t)cuda_stream;
    h->has_wake = (Z != nullptr);
    grid_constants(h);

    auto bail = [&](int code, const std::string &msg) {
        g_create_error = msg;
        vfps_destroy(h);
        return code;
    };
    if (h->G.H > ROT_MAX_H)
        return bail(VFPS_ERR_UNSUPPORTED, "rotation displacement per step exceeds the supported halo (too few steps_per_period for this grid)");

    const int N = h->N, M = h->members;
    h->tiles_x2 = (N + R2_RT - 1) / R2_RT;
    h->tiles_y2 = (N + 32 * R2_WARPS - 1) / (32 * R2_WARPS);
    h->kfp2_rows = 4096 / N > 0 ? (4096 / N < N ? 4096 / N : N) : 1;
    h->kfp2_blocks = (N + h->kfp2_rows - 1) / h->kfp2_rows;
    h->wd_blocks = (N + WD_ROWS - 1) / WD_ROWS;
    h->fft_threads = h->Nf / 2 < 1024 ? (h->Nf / 2 < 32 ? 32 : h->Nf / 2) : 1024;
    h->fft_smem = (size_t)h->Nf * sizeof(float2);                    // Nf/2 packed points + per-stage twiddle tables

#define CUB(call)                                                                             \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return bail(e_ == cudaErrorMemoryAllocation ? VFPS_ERR_NOMEM : VFPS_ERR_CUDA,     \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                  \
    } while (0)

    CUB(dalloc(h, &h->psi, (size_t)M * N * N));
    CUB(dalloc(h, &h->psi_tmp, (size_t)M * N * N));
    CUB(dalloc(h, &h->tw, (size_t)h->Nf / 2));
    CUB(dalloc(h, &h->rho_part, (size_t)M * N * h->tiles_y2));
    CUB(dalloc(h, &h->pw_part, (size_t)M * h->wd_blocks));
    CUB(dalloc(h, &h->tilectr, (size_t)M * h->tiles_x2));
    CUB(cudaMemsetAsync(h->tilectr, 0, (size_t)M * h->tiles_x2 * sizeof(unsigned), h->stream));
    CUB(cudaMemsetAsync(h->pw_part, 0, (size_t)M * h->wd_blocks * sizeof(float), h->stream));
    CUB(dalloc(h, &h->rho, (size_t)M * N));
    CUB(dalloc(h, &h->V, (size_t)M * N));
    CUB(dalloc(h, &h->qstat, (size_t)M * 4));
    CUB(dalloc(h, &h->mom_part, (size_t)M * h->kfp2_blocks * 6));
    if (p->flags & VFPS_FLAG_CLAMP) CUB(dalloc(h, &h->dpU, (size_t)M * N));
    CUB(dalloc(h, &h->scale, (size_t)M));
    CUB(dalloc(h, &h->blkctr, (size_t)M));
    CUB(dalloc(h, &h->rowctr, (size_t)M));
    CUB(dalloc(h, &h->diag_cell, (size_t)1));
    CUB(dalloc(h, &h->g_rho, (size_t)M * N));
    CUB(dalloc(h, &h->g_V, (size_t)M * N));
    CUB(dalloc(h, &h->g_m1, (size_t)M * N));
    CUB(dalloc(h, &h->g_m2, (size_t)M * N));
    CUB(dalloc(h, &h->g_qstat, (size_t)M * 4));
    CUB(dalloc(h, &h->g_out, (size_t)M * (N > 6 ? N : 6)));
    CUB(cudaMemsetAsync(h->psi, 0, (size_t)M * N * N * sizeof(float), h->stream));
    CUB(cudaMemsetAsync(h->V, 0, (size_t)M * N * sizeof(float), h->stream));

    if (h->has_wake) {
        const size_t nz = (size_t)M * (h->Nf / 2 + 1);
        CUB(dalloc(h, &h->Z, nz));
        CUB(cudaMemcpyAsync(h->Z, Z, nz * sizeof(float2),
                            z_on_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, h->stream));
    }
    {   // twiddles exp(-2 pi i j / Nf), evaluated in double, rounded once
        std::vector<float2> tw(h->Nf / 2);
        const double PI = 3.14159265358979323846;
        for (int j = 0; j < h->Nf / 2; ++j) {
            const double ang = -2.0 * PI * (double)j / (double)h->Nf;
            tw[j] = make_float2((float)std::cos(ang), (float)std::sin(ang));
        }
        CUB(cudaMemcpyAsync(h->tw, tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice, h->stream));
        CUB(cudaStreamSynchronize(h->stream));
    }
    k_fill<<<(M + 255) / 256, 256, 0, h->stream>>>(h->scale, 1.0f, M);
    k_set_ctl<<<(M + 255) / 256, 256, 0, h->stream>>>(h->diag_cell, nullptr, h->rowctr, h->blkctr, M);
    h->launches += 2;
    if (h->has_wake) {
        CUB(dalloc(h, &h->wfun, (size_t)M * 2 * N));
        const int nw = M * 2 * N;
        k_wake_function<<<(nw + 127) / 128, 128, 0, h->stream>>>(N, h->Nf, M, h->Z, h->wfun);
        h->launches += 1;
    }
    cluster_configure(h);
    grid_configure(h);
    {
        const int rc2 = grid2_configure(h);
        if (rc2 != VFPS_OK) return bail(rc2, h->err);
    }
    if (h->gr_blocks > 0) CUB(dalloc(h, &h->gr_mom, (size_t)h->gr_blocks * GR_NPART));
    if (h->gr_blocks > 0) CUB(dalloc(h, &h->gr_qacc, (size_t)2));
    if (h->gr_blocks > 0) {
        CUB(dalloc(h, &h->gr_zrow, (size_t)N));
        CUB(cudaMemsetAsync(h->gr_zrow, 0, (size_t)N * sizeof(float), h->stream));
    }
    CUB(cudaGetLastError());
#undef CUB
    *out = h;
    return VFPS_OK;
}

// rho / V / moments of the CURRENT psi into the g_* scratch (stateless: touches no step state)
int current_profile(vfps_sim *h, bool want_wake)
{
    const int N = h->N, M = h->members;
    k_project<<<dim3(N, M), 128, 0, h->stream>>>(h->G, h->psi, h->scale, h->g_rho, h->g_m1, h->g_m2);
    h->launches += 1;
    if (want_wake) {
        CU(wake_fft_attr(h));
        k_wake_fft<<<M, h->fft_threads, h->fft_smem, h->stream>>>(N, h->Nf, h->log2Nf, h->G.dq, h->g_rho, 1,
                                                                  h->has_wake ? h->Z : nullptr, h->tw,
                                                                  h->g_rho, h->g_V, h->g_qstat);
        h->launches += 1;
    }
    CU(cudaGetLastError());
    return VFPS_OK;
}

int to_host(vfps_sim *h, float *dst_host, const float *src_dev, size_t n)
{
    CU(cudaMemcpyAsync(dst_host, src_dev, n * sizeof(float), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return VFPS_OK;
}

}  // namespace

extern "C" {

int vfps_create(const vfps_params *p, const vfps_complex *Z, void *cuda_stream, vfps_handle *out)
{
    return create_impl(p, Z, false, cuda_stream, out);
}

int vfps_create_host(const vfps_params *p, const vfps_complex *Z_host, void *cuda_stream, vfps_handle *out)
{
    return create_impl(p, Z_host, true, cuda_stream, out);
}

int vfps_destroy(vfps_handle h)
{
    if (!h) return VFPS_OK;
    cudaStreamSynchronize(h->stream);
    if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
    for (cudaEvent_t e : h->ev_pool) cudaEventDestroy(e);
    if (h->diag_scratch) cudaFree(h->diag_scratch);
    for (void *p : h->owned) cudaFree(p);
    delete h;
    return VFPS_OK;
}

int vfps_set_option(vfps_handle h, int option, int value)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (option == VFPS_OPT_ENGINE) {
        if (value == VFPS_ENGINE_AUTO || value == VFPS_ENGINE_STREAM || value == VFPS_ENGINE_GRAPH) {
            h->engine_opt = value;
            return VFPS_OK;
        }
        if (value == VFPS_ENGINE_CLUSTER) {
            if (h->cl_S == 0) return fail(h, VFPS_ERR_UNSUPPORTED, "cluster engine unavailable: " + h->cl_why);
            h->engine_opt = value;
            return VFPS_OK;
        }
        if (value == VFPS_ENGINE_GRID) {
            if (grid_kernel_in_use(h) == 0)
                return fail(h, VFPS_ERR_UNSUPPORTED, "grid engine unavailable: " + (h->gr_blocks == 0 ? h->gr_why : h->g2_why));
            h->engine_opt = value;
            return VFPS_OK;
        }
        return fail(h, VFPS_ERR_ARG, "unknown engine");
    }
    if (option == VFPS_OPT_CLUSTER_SIZE) {
        if (!(value == 0 || value == 1 || value == 2 || value == 4 || value == 8 || value == 16))
            return fail(h, VFPS_ERR_ARG, "cluster size must be 0 (auto), 1, 2, 4, 8 or 16");
        const int old = h->cl_S_opt;
        h->cl_S_opt = value;
        cluster_configure(h);
        if (h->cl_S == 0) {
            const std::string why = h->cl_why;
            h->cl_S_opt = old;
            cluster_configure(h);
            return fail(h, VFPS_ERR_UNSUPPORTED, "cluster size not feasible for this grid: " + why);
        }
        return VFPS_OK;
    }
    if (option == VFPS_OPT_CLUSTER_KERNEL) {
        if (!(value == 0 || value == 1 || value == 3))
            return fail(h, VFPS_ERR_ARG, "cluster kernel must be 0 (auto), 1 (k_cluster_step) or 3 (k_onchip_step)");
        const int old = h->cl_ver_opt;
        h->cl_ver_opt = value;
        cluster_configure(h);
        if (h->cl_S == 0) {
            const std::string why = h->cl_why;
            h->cl_ver_opt = old;
            cluster_configure(h);
            return fail(h, VFPS_ERR_UNSUPPORTED, "cluster kernel not available for this grid: " + why);
        }
        return VFPS_OK;
    }
    if (option == VFPS_OPT_GRID_KERNEL) {
        if (!(value == 0 || value == 1 || value == 2))
            return fail(h, VFPS_ERR_ARG, "grid kernel must be 0 (auto), 1 (k_grid_step) or 2 (k_grid2_step)");
        if (value == 1 && h->gr_blocks == 0) return fail(h, VFPS_ERR_UNSUPPORTED, "k_grid_step unavailable: " + h->gr_why);
        if (value == 2 && h->g2_blocks == 0) return fail(h, VFPS_ERR_UNSUPPORTED, "k_grid2_step unavailable: " + h->g2_why);
        h->gr_ver_opt = value;
        return VFPS_OK;
    }
    if (option == VFPS_OPT_TIMING) {
        if (value != 0 && value != 1) return fail(h, VFPS_ERR_ARG, "timing must be 0 or 1");
        if (!value) resolve_timing(h);
        h->timing = (value == 1);
        return VFPS_OK;
    }
    if (option == VFPS_OPT_WAKE) {
        if (!(value == VFPS_WAKE_AUTO || value == VFPS_WAKE_FFT || value == VFPS_WAKE_DIRECT))
            return fail(h, VFPS_ERR_ARG, "unknown wake mode");
        if (value == VFPS_WAKE_FFT && (h->P.flags & VFPS_FLAG_CLAMP) && h->has_wake)
            return fail(h, VFPS_ERR_UNSUPPORTED, "clamped interpolation needs the direct-convolution wake (its transposed "
                                                   "wake gives the CSR power of the end-of-step profile)");
        if (value != h->wake_opt) drop_graph(h);
        h->wake_opt = value;
        return VFPS_OK;
    }
    return fail(h, VFPS_ERR_ARG, "unknown option");
}

int vfps_get_option(vfps_handle h, int option, int *value)
{
    if (!h || !value) return fail(h, VFPS_ERR_ARG, "NULL argument");
    if (option == VFPS_OPT_ENGINE) { *value = h->engine_opt; return VFPS_OK; }
    if (option == VFPS_OPT_WAKE) { *value = h->wake_opt; return VFPS_OK; }
    if (option == VFPS_OPT_TIMING) { *value = h->timing ? 1 : 0; return VFPS_OK; }
    if (option == VFPS_OPT_CLUSTER_SIZE) { *value = h->cl_S; return VFPS_OK; }
    if (option == VFPS_OPT_CLUSTER_KERNEL) { *value = h->cl_ver; return VFPS_OK; }
    if (option == VFPS_OPT_GRID_KERNEL) { *value = grid_kernel_in_use(h); return VFPS_OK; }
    return fail(h, VFPS_ERR_ARG, "unknown option");
}

const char *vfps_engine_name(vfps_handle h)
{
    if (!h) return "";
    switch (resolved_engine(h)) {
        case VFPS_ENGINE_STREAM: return "stream";
        case VFPS_ENGINE_GRAPH: return "graph";
        case VFPS_ENGINE_GRID: return "grid";
        default: return "cluster";
    }
}
const char *vfps_wake_name(vfps_handle h)
{
    if (!h) return "";
    if (resolved_engine(h) == VFPS_ENGINE_CLUSTER || resolved_engine(h) == VFPS_ENGINE_GRID) return "direct";
    return wake_is_direct(h) ? "direct" : "fft";
}

static int set_psi_impl(vfps_handle h, const float *psi, cudaMemcpyKind kind)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (!psi) return fail(h, VFPS_ERR_ARG, "psi is NULL");
    const size_t n = (size_t)h->members * h->cells();
    CU(cudaMemcpyAsync(h->psi, psi, n * sizeof(float), kind, h->stream));
    k_fill<<<(h->members + 255) / 256, 256, 0, h->stream>>>(h->scale, 1.0f, h->members);
    h->launches += 1;
    CU(cudaGetLastError());
    if (kind == cudaMemcpyHostToDevice) CU(cudaStreamSynchronize(h->stream));
    h->psi_set = true;
    h->steps = 0;
    return VFPS_OK;
}

static int set_impedance_impl(vfps_handle h, const vfps_complex *Z, cudaMemcpyKind kind)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (!Z) return fail(h, VFPS_ERR_ARG, "Z is NULL");
    if (!h->has_wake) return fail(h, VFPS_ERR_STATE, "the simulation was created without an impedance");
    const size_t nz = (size_t)h->members * (h->Nf / 2 + 1);
    CU(cudaMemcpyAsync(h->Z, Z, nz * sizeof(float2), kind, h->stream));
    const int nw = h->members * 2 * h->N;
    k_wake_function<<<(nw + 127) / 128, 128, 0, h->stream>>>(h->N, h->Nf, h->members, h->Z, h->wfun);
    h->launches += 1;
    CU(cudaGetLastError());
    if (kind == cudaMemcpyHostToDevice) CU(cudaStreamSynchronize(h->stream));
    return VFPS_OK;
}

int vfps_set_impedance(vfps_handle h, const vfps_complex *Z) { return set_impedance_impl(h, Z, cudaMemcpyDeviceToDevice); }
int vfps_set_impedance_host(vfps_handle h, const vfps_complex *Z) { return set_impedance_impl(h, Z, cudaMemcpyHostToDevice); }

int vfps_set_psi(vfps_handle h, const float *psi) { return set_psi_impl(h, psi, cudaMemcpyDeviceToDevice); }
int vfps_set_psi_host(vfps_handle h, const float *psi) { return set_psi_impl(h, psi, cudaMemcpyHostToDevice); }

int vfps_step(vfps_handle h, int n, float *diag)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (n < 0) return fail(h, VFPS_ERR_ARG, "n must be >= 0");
    if (!h->psi_set) return fail(h, VFPS_ERR_STATE, "vfps_step before vfps_set_psi");
    if (n == 0) return VFPS_OK;
    if (resolved_engine(h) == VFPS_ENGINE_GRID) {
        if (h->timing) resolve_timing(h);
        int rc = (grid_kernel_in_use(h) == 2) ? launch_grid2_steps(h, n, diag) : launch_grid_steps(h, n, diag);
        if (rc != VFPS_OK) return rc;
        h->steps += n;
        return VFPS_OK;
    }
    if (resolved_engine(h) == VFPS_ENGINE_CLUSTER) {
        if (h->timing) resolve_timing(h);
        int rc = launch_cluster_steps(h, n, diag);
        if (rc != VFPS_OK) return rc;
        h->steps += n;
        return VFPS_OK;
    }
    k_set_ctl<<<(h->members + 255) / 256, 256, 0, h->stream>>>(h->diag_cell, diag, h->rowctr, h->blkctr, h->members);
    h->launches += 1;
    int done = 0;
    if (resolved_engine(h) == VFPS_ENGINE_GRAPH && n >= GRAPH_STEPS) {
        int rc = ensure_graph(h);
        if (rc != VFPS_OK) return rc;
        for (; done + GRAPH_STEPS <= n; done += GRAPH_STEPS) {
            CU(cudaGraphLaunch(h->graph_exec, h->stream));
            h->launches += h->graph_launches;
        }
    }
    // stream engine, and the remainder of a graph run
    const bool timed = h->timing && resolved_engine(h) == VFPS_ENGINE_STREAM;
    if (timed) resolve_timing(h);
    for (; done < n; ++done) {
        int rc = launch_step(h, timed);
        if (rc != VFPS_OK) return rc;
    }
    CU(cudaGetLastError());
    h->steps += n;
    return VFPS_OK;
}

int vfps_step_host(vfps_handle h, int n, float *diag_host)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (n < 0) return fail(h, VFPS_ERR_ARG, "n must be >= 0");
    float *d = nullptr;
    const size_t cnt = (size_t)n * h->members * 6;
    if (diag_host && cnt) {
        if (cnt > h->diag_scratch_n) {
            CU(cudaStreamSynchronize(h->stream));
            if (h->diag_scratch) cudaFree(h->diag_scratch);
            h->diag_scratch = nullptr; h->diag_scratch_n = 0;
            CU(cudaMalloc((void **)&h->diag_scratch, cnt * sizeof(float)));
            h->diag_scratch_n = cnt;
        }
        d = h->diag_scratch;
    }
    int rc = vfps_step(h, n, d);
    if (rc == VFPS_OK) {
        cudaError_t e = d ? cudaMemcpyAsync(diag_host, d, cnt * sizeof(float), cudaMemcpyDeviceToHost, h->stream)
                          : cudaSuccess;
        if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
        if (e != cudaSuccess) rc = fail(h, VFPS_ERR_CUDA, cudaGetErrorString(e));
    }
    return rc;
}

int vfps_get_psi(vfps_handle h, float *psi_out)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (!psi_out) return fail(h, VFPS_ERR_ARG, "psi_out is NULL");
    const size_t cells = h->cells();
    int bx = (int)((cells + 1023) / 1024); if (bx > 1184) bx = 1184;
    k_scale_copy<<<dim3(bx, h->members), 256, 0, h->stream>>>(h->psi, h->scale, psi_out, cells, h->G.renorm);
    h->launches += 1;
    CU(cudaGetLastError());
    return VFPS_OK;
}

int vfps_get_psi_host(vfps_handle h, float *psi_out_host)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (!psi_out_host) return fail(h, VFPS_ERR_ARG, "psi_out is NULL");
    int rc = vfps_get_psi(h, h->psi_tmp);          // psi_tmp is dead between steps
    if (rc != VFPS_OK) return rc;
    return to_host(h, psi_out_host, h->psi_tmp, (size_t)h->members * h->cells());
}

int vfps_get_profile(vfps_handle h, float *rho_out)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (!rho_out) return fail(h, VFPS_ERR_ARG, "rho_out is NULL");
    int rc = current_profile(h, false);
    if (rc != VFPS_OK) return rc;
    CU(cudaMemcpyAsync(rho_out, h->g_rho, (size_t)h->members * h->N * sizeof(float), cudaMemcpyDeviceToDevice, h->stream));
    return VFPS_OK;
}

int vfps_get_profile_host(vfps_handle h, float *rho_out_host)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (!rho_out_host) return fail(h, VFPS_ERR_ARG, "rho_out is NULL");
    int rc = current_profile(h, false);
    if (rc != VFPS_OK) return rc;
    return to_host(h, rho_out_host, h->g_rho, (size_t)h->members * h->N);
}

int vfps_get_wake(vfps_handle h, float *V_out)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (!V_out) return fail(h, VFPS_ERR_ARG, "V_out is NULL");
    int rc = current_profile(h, true);
    if (rc != VFPS_OK) return rc;
    CU(cudaMemcpyAsync(V_out, h->g_V, (size_t)h->members * h->N * sizeof(float), cudaMemcpyDeviceToDevice, h->stream));
    return VFPS_OK;
}

int vfps_get_wake_host(vfps_handle h, float *V_out_host)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (!V_out_host) return fail(h, VFPS_ERR_ARG, "V_out is NULL");
    int rc = current_profile(h, true);
    if (rc != VFPS_OK) return rc;
    return to_host(h, V_out_host, h->g_V, (size_t)h->members * h->N);
}

static int moments_impl(vfps_handle h)
{
    int rc = current_profile(h, true);
    if (rc != VFPS_OK) return rc;
    k_moments_final<<<h->members, 256, 0, h->stream>>>(h->G, h->g_rho, h->g_m1, h->g_m2, h->g_qstat, h->g_out);
    h->launches += 1;
    CU(cudaGetLastError());
    return VFPS_OK;
}

int vfps_get_moments(vfps_handle h, float *out)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (!out) return fail(h, VFPS_ERR_ARG, "out is NULL");
    int rc = moments_impl(h);
    if (rc != VFPS_OK) return rc;
    CU(cudaMemcpyAsync(out, h->g_out, (size_t)h->members * 6 * sizeof(float), cudaMemcpyDeviceToDevice, h->stream));
    return VFPS_OK;
}

int vfps_get_moments_host(vfps_handle h, float *out_host)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    if (!out_host) return fail(h, VFPS_ERR_ARG, "out is NULL");
    int rc = moments_impl(h);
    if (rc != VFPS_OK) return rc;
    return to_host(h, out_host, h->g_out, (size_t)h->members * 6);
}

int vfps_step_count(vfps_handle h, long long *count)
{
    if (!h || !count) return fail(h, VFPS_ERR_ARG, "NULL argument");
    *count = h->steps;
    return VFPS_OK;
}

int vfps_launch_count(vfps_handle h, long long *count)
{
    if (!h || !count) return fail(h, VFPS_ERR_ARG, "NULL argument");
    *count = h->launches;
    return VFPS_OK;
}

int vfps_kernel_time(vfps_handle h, int kernel, double *ms_total, long long *launches)
{
    if (!h || !ms_total || !launches) return fail(h, VFPS_ERR_ARG, "NULL argument");
    if (kernel < 0 || kernel >= VFPS_NUM_KERNELS) return fail(h, VFPS_ERR_ARG, "unknown kernel id");
    resolve_timing(h);
    *ms_total = h->k_ms[kernel];
    *launches = h->k_cnt[kernel];
    return VFPS_OK;
}

int vfps_reset_kernel_times(vfps_handle h)
{
    if (!h) return fail(nullptr, VFPS_ERR_ARG, "handle is NULL");
    resolve_timing(h);
    for (int k = 0; k < VFPS_NUM_KERNELS; ++k) { h->k_ms[k] = 0.0; h->k_cnt[k] = 0; }
    return VFPS_OK;
}

const char *vfps_kernel_name(int kernel)
{
    switch (kernel) {
        case VFPS_KERNEL_WAKE: return "k_wake_fft";
        case VFPS_KERNEL_CLUSTER: return "k_cluster_step";
        case VFPS_KERNEL_ROTATE2: return "k_rotate2";
        case VFPS_KERNEL_WAKE_DIRECT: return "k_wake_direct";
        case VFPS_KERNEL_KICK_FP2: return "k_kick_fp2";
        case VFPS_KERNEL_GRID: return "k_grid_step";
        case VFPS_KERNEL_GRID2: return "k_grid2_step";
        default: return nullptr;
    }
}

const char *vfps_last_error(vfps_handle h) { return h ? h->err.c_str() : g_create_error.c_str(); }

const char *vfps_version(void) { return "vfps 0.1 (sm_100a)"; }

}  // extern "C"
