// vfps_noalloc.cu -- vfps_wake_noalloc (include/vfps.h): the wake a3 of a caller-held profile with NO
// device allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
// serving loops, harnesses that forbid it).
//
// The library's wake path keeps the wake function w = Re IDFT(Z) (Eq. 4-5) in a buffer that
// vfps_create allocates.  This variant keeps it in a file-scope device array of fixed size instead:
//     g_na_wfun[2 * VFPS_NOALLOC_MAX_N] floats = 32 KB, held by every GPU that loads the library
//     until the process exits.
// In host code the NAME of that array is a host-side stand-in, not a device address: a kernel given
// it would fault (or, where the GPU can reach host memory, use the wrong memory).  Its device address
// comes from cudaGetSymbolAddress, once per device, with that device current; the kernels get that
// pointer.
// Every call shares the array: it holds the wake function of the LAST call until the next call
// overwrites it.  Nothing in it accumulates -- k_na_wake_function writes all 2N entries a call reads
// before k_na_wake reads them (same stream) -- so nothing needs clearing; but two calls that overlap
// on the GPU (different streams, or graphs replayed concurrently) race on it.
// Self-contained: shares no kernel with vfps_api.cu and changes no existing path.
#include "../../include/vfps.h"
#include "vfps_common.cuh"

#include <cstdio>
#include <mutex>

namespace {

constexpr int NA_MAX_N = VFPS_NOALLOC_MAX_N;
constexpr int NA_MAX_DEVICES = 64;
constexpr int NA_ROWS = 8;          // rows per CTA of k_na_wake (one per warp)
constexpr int NA_THREADS = 256;

// the scratch: wake function, lag d at index d + N - 1, entry 2N - 1 zero
static __device__ __align__(256) float g_na_wfun[2 * NA_MAX_N];

float *g_na_ptr[NA_MAX_DEVICES];    // device address of g_na_wfun per device, nullptr = not looked up yet
std::mutex g_na_mutex;
thread_local char g_na_error[256] = "";

int na_fail(int code, const char *msg, const char *detail = "")
{
    std::snprintf(g_na_error, sizeof(g_na_error), "vfps_wake_noalloc: %s%s", msg, detail);
    return code;
}

bool na_pow2(long long v) { return v > 0 && (v & (v - 1)) == 0; }

// w[d] = (1/Nf) [ Re Z_0 + 2 sum_{k=1}^{Nf/2-1} Re(Z_k e^{2 pi i k d / Nf}) + Re Z_{Nf/2} (-1)^d ],
// d = -(N-1) .. N-1: the inverse DFT of the Hermitian spectrum (L149) at the lags a grid of N points
// can see.  One thread per lag, double precision, the angle reduced in integers.
__global__ void k_na_wake_function(int N, int Nf, const float2 *__restrict__ Z, float *__restrict__ w)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= 2 * N) return;
    if (j == 2 * N - 1) { w[j] = 0.0f; return; }
    const int d = j - (N - 1);
    double acc = (double)Z[0].x;
    for (int k = 1; k < Nf / 2; ++k) {
        const long long kd = ((long long)k * d) % Nf;
        double sn, cs;
        sincospi(2.0 * (double)kd / (double)Nf, &sn, &cs);
        acc += 2.0 * ((double)Z[k].x * cs - (double)Z[k].y * sn);
    }
    acc += (double)Z[Nf / 2].x * ((d & 1) ? -1.0 : 1.0);
    w[j] = (float)(acc / (double)Nf);
}

// V_x = sum_x' w[x - x'] rho_x' (Eq. 4).  grid = ceil(N / NA_ROWS), block = 256, dynamic shared
// memory (2N + NA_ROWS) floats: the profile and the N + NA_ROWS - 1 lags this CTA's rows touch are
// staged with coalesced loads; warp k forms row r0 + k.
__global__ void __launch_bounds__(NA_THREADS)
k_na_wake(int N, const float *__restrict__ rho, const float *__restrict__ w, float *__restrict__ V)
{
    extern __shared__ float na_smem[];
    float *srho = na_smem, *sw = na_smem + N;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int r0 = blockIdx.x * NA_ROWS;
    for (int i = tid; i < N; i += NA_THREADS) srho[i] = rho[i];
    for (int i = tid; i < N + NA_ROWS - 1; i += NA_THREADS) sw[i] = (r0 + i < 2 * N - 1) ? w[r0 + i] : 0.0f;
    __syncthreads();
    const int x = r0 + warp;
    if (x >= N) return;
    // w[x - x'] sits at index x - x' + N - 1 of the array, i.e. at sw[warp + N - 1 - x']
    const float *wx = sw + (warp + N - 1);
    float v0 = 0.0f, v1 = 0.0f;
    int xp = lane;
    for (; xp + 32 < N; xp += 64) {
        v0 = fmaf(wx[-xp], srho[xp], v0);
        v1 = fmaf(wx[-(xp + 32)], srho[xp + 32], v1);
    }
    if (xp < N) v0 = fmaf(wx[-xp], srho[xp], v0);
    const float v = vfps::warp_sum(v0 + v1);
    if (lane == 0) V[x] = v;
}

// device address of the scratch on the current device (looked up once per device)
int na_scratch(float **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail(VFPS_ERR_CUDA, "cudaGetDevice: ", cudaGetErrorString(e));
    if (dev < 0 || dev >= NA_MAX_DEVICES) return na_fail(VFPS_ERR_UNSUPPORTED, "device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (g_na_ptr[dev] == nullptr) {
        float *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_na_wfun);
        if (e != cudaSuccess || p == nullptr) {
            cudaGetLastError();
            return na_fail(VFPS_ERR_CUDA, "cudaGetSymbolAddress(g_na_wfun): ", cudaGetErrorString(e));
        }
        g_na_ptr[dev] = p;
    }
    *out = g_na_ptr[dev];
    return VFPS_OK;
}

}  // namespace

extern "C" int vfps_wake_noalloc(int N, int pad, const vfps_complex *Z, const float *rho, float *V_out, void *cuda_stream)
{
    g_na_error[0] = '\0';
    if (!Z || !rho || !V_out) return na_fail(VFPS_ERR_ARG, "Z, rho and V_out must not be NULL");
    if (N < 8) return na_fail(VFPS_ERR_ARG, "N must be >= 8");
    if (pad < 2 || !na_pow2(pad) || !na_pow2((long long)N * pad)) return na_fail(VFPS_ERR_ARG, "pad and N*pad must be powers of two, pad >= 2");
    if (N > NA_MAX_N) return na_fail(VFPS_ERR_UNSUPPORTED, "N exceeds VFPS_NOALLOC_MAX_N = 4096 (the size of the built-in scratch array)");
    if ((long long)N * pad > 8192) return na_fail(VFPS_ERR_UNSUPPORTED, "N*pad > 8192 (the limit of the library's wake)");
    float *w = nullptr;
    const int rc = na_scratch(&w);
    if (rc != VFPS_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int Nf = N * pad;
    k_na_wake_function<<<(2 * N + 127) / 128, 128, 0, st>>>(N, Nf, reinterpret_cast<const float2 *>(Z), w);
    k_na_wake<<<(N + NA_ROWS - 1) / NA_ROWS, NA_THREADS, (size_t)(2 * N + NA_ROWS) * sizeof(float), st>>>(N, rho, w, V_out);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(VFPS_ERR_CUDA, "kernel launch: ", cudaGetErrorString(e));
    return VFPS_OK;
}

extern "C" const char *vfps_noalloc_last_error(void) { return g_na_error; }
