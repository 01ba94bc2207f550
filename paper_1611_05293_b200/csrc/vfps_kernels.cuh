// vfps_kernels.cuh -- the non-template kernels of the library (sm_100a), included by vfps_api.cu
// only: the stateless get_* calls (k_project, k_moments_final, k_scale_copy), the literal Eq. 5
// wake (k_wake_fft: zero-padded shared-memory FFT, x Z, inverse FFT), and small set-up helpers.
// psi is stored UN-normalised together with a per-member scalar `scale` = 1/C of the previous
// step; the rotation applies it (it is linear), so renormalisation costs no extra pass.
#pragma once
#include "vfps_common.cuh"

namespace vfps {

constexpr int WD_ROWS = 8;         // rows per CTA of k_wake_direct (one per warp)
constexpr int WD_THREADS = 256;

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
// One CTA per member, blockDim = min(1024, Nf/4).  The zero-padded profile is real and the impedance
// Hermitian, so only wave numbers k >= 0 are needed (L149: "a factor of two"): the Nf real samples are
// packed as M = Nf/2 complex points z[n] = rho[2n] + i rho[2n+1], ONE complex FFT of length M runs in
// shared memory (two radix-2 stages per pass in registers; forward decimation in frequency, natural
// in, bit-reversed out), the spectrum R_k, k = 0..M, of the real sequence is split off pairwise
//     R_k = (A + conj B)/2 - (i/2) w_k (A - conj B),   A = Z_k, B = Z_{M-k},  w_k = exp(-2 pi i k/Nf),
// multiplied by the impedance, Y_k = Z_k^imp R_k, and packed again for the inverse transform of the
// real result,  E_k = (Y_k + conj Y_{M-k}) + i conj(w_k) (Y_k - conj Y_{M-k}),  which an inverse
// decimation-in-time FFT of length M (bit-reversed in, natural out: no permutation pass) turns into
// V[2n] + i V[2n+1].  tw[j] = exp(-2 pi i j/Nf), j < Nf/2.
// Outputs: rho[m][x] (summed partials), V[m][x], qstat[m] = { sum rho, sum Xc rho, sum Xc^2 rho,
// P_raw } with Xc the centred q index and P_raw = (dq/Nf) sum_k Re Z_k |R_k|^2 over all Nf wave
// numbers (Eq. 16-17; k and Nf - k contribute equally).
__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

__global__ void __launch_bounds__(1024)
k_wake_fft(int N, int Nf, int log2Nf, float dq, const float *rho_part, int nparts,
           const float2 *__restrict__ Z, const float2 *__restrict__ tw, float *rho_out /* may be rho_part (nparts = 1) */,
           float *__restrict__ V, float *__restrict__ qstat)
{
    extern __shared__ float2 s[];          // M points, then M - 1 twiddles, one contiguous table per stage
    __shared__ float red[4][32];
    const int M = Nf >> 1, logM = log2Nf - 1;
    float2 *stw = s + M;
    const int m = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
    const float xc = 0.5f * (float)(N - 1);
    float s0 = 0, s1 = 0, s2 = 0, pw = 0;
    for (int n = tid; n < M; n += nt) {
        float r[2] = {0.0f, 0.0f};
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int x = 2 * n + h;
            if (x < N) {
                const float *pp = rho_part + ((size_t)m * N + x) * nparts;
                float acc = 0.0f;
#pragma unroll 8
                for (int k = 0; k < nparts; ++k) acc += pp[k];
                rho_out[(size_t)m * N + x] = acc;
                const float c = (float)x - xc, t = c * acc;
                s0 += acc; s1 += t; s2 = fmaf(t, c, s2);
                r[h] = acc;
            }
        }
        s[n] = make_float2(r[0], r[1]);
    }
    if (Z != nullptr) {
        const float2 *Zm = Z + (size_t)m * (Nf / 2 + 1);
        // The twiddles are read 2 log2(M) times: stage them once, as one contiguous table per
        // butterfly span (entry half - 1 + pos = exp(-2 pi i pos / (2 half)) = tw[pos * (Nf/2) / half]):
        // reading the single table with a stride put up to 32 lanes on one bank in most stages.
        for (int j = tid; j < M - 1; j += nt) {
            const int half = 1 << (31 - __clz(j + 1)), pos = j + 1 - half;
            stw[j] = __ldg(tw + pos * ((Nf >> 1) / half));
        }
        __syncthreads();
        // forward, decimation in frequency; two radix-2 stages (spans 2q and q) per pass in registers
        int half = M >> 1;
        for (; half >= 2; half >>= 2) {
            const int q = half >> 1;
            const float2 *w2 = stw + (half - 1), *w1 = stw + (q - 1);
            for (int j = tid; j < (M >> 2); j += nt) {
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
        if (half == 1) {                                          // odd log2(M): one radix-2 stage left (w = 1)
            for (int j = tid; j < (M >> 1); j += nt) {
                const float2 u = s[2 * j], v = s[2 * j + 1];
                s[2 * j] = make_float2(u.x + v.x, u.y + v.y);
                s[2 * j + 1] = make_float2(u.x - v.x, u.y - v.y);
            }
            __syncthreads();
        }
        // split off the spectrum of the real sequence, x Z, power spectrum, pack for the inverse transform;
        // thread k handles the pair (k, M - k); Z_k of the packed sequence sits at the bit-reversed position
        for (int k = tid; k <= (M >> 1); k += nt) {
            const int ia = (int)(__brev((unsigned)k) >> (32 - logM));
            if (k == 0) {
                const float2 A = s[ia];
                const float R0 = A.x + A.y, RM = A.x - A.y;                 // k = 0 and the Nyquist wave number M: real
                const float z0 = __ldg(Zm).x, zM = __ldg(Zm + M).x;           // their imaginary parts are ignored
                pw = fmaf(z0, R0 * R0, fmaf(zM, RM * RM, pw));
                const float Y0 = z0 * R0, YM = zM * RM;
                s[ia] = make_float2(Y0 + YM, Y0 - YM);                        // E_0 = (Y_0 + Y_M) + i (Y_0 - Y_M)
                continue;
            }
            const int ib = (int)(__brev((unsigned)(M - k)) >> (32 - logM));
            const float2 A = s[ia], B = s[ib], w = __ldg(tw + k);
            // R_k = (A + conj B)/2 - (i/2) w (A - conj B);  R_{M-k} = (B + conj A)/2 + (i/2) conj(w) (B - conj A)
            const float2 sm = make_float2(0.5f * (A.x + B.x), 0.5f * (A.y - B.y));      // (A + conj B)/2
            const float2 df = make_float2(0.5f * (A.x - B.x), 0.5f * (A.y + B.y));      // (A - conj B)/2
            const float2 t = cmul(w, df);                                                // w (A - conj B)/2
            const float2 Rk = make_float2(sm.x + t.y, sm.y - t.x);                       // sm - i t
            // R_{M-k} = conj(sm) + (i/2) conj(w) (B - conj A), and B - conj A = -conj(A - conj B):  = conj(sm) - i conj(t)
            const float2 Rm = make_float2(sm.x - t.y, -sm.y - t.x);
            const float2 zk = __ldg(Zm + k), zm = __ldg(Zm + (M - k));
            pw = fmaf(2.0f * zk.x, fmaf(Rk.x, Rk.x, Rk.y * Rk.y), pw);     // every 0 < k < M stands for k and Nf - k
            const float2 Yk = cmul(Rk, zk);
            if (2 * k == M) {
                // E = (Y + conj Y) + i conj(w) (Y - conj Y), conj(w) = i:  2 Re Y - 2 i ... = (2 Re Y, -2 Im Y)
                s[ia] = make_float2(2.0f * Yk.x, -2.0f * Yk.y);
                continue;
            }
            pw = fmaf(2.0f * zm.x, fmaf(Rm.x, Rm.x, Rm.y * Rm.y), pw);
            const float2 Ym = cmul(Rm, zm);
            // E_k = (Y_k + conj Y_m) + i conj(w) (Y_k - conj Y_m);  E_{M-k} = (Y_m + conj Y_k) - i w (Y_m - conj Y_k)
            const float2 sp = make_float2(Yk.x + Ym.x, Yk.y - Ym.y), dm = make_float2(Yk.x - Ym.x, Yk.y + Ym.y);
            const float2 u = cmul(make_float2(w.x, -w.y), dm);                           // conj(w) (Y_k - conj Y_m)
            s[ia] = make_float2(sp.x - u.y, sp.y + u.x);                                 // sp + i u
            // Y_m - conj Y_k = -conj(dm):  -i w (-conj dm) = i w conj(dm) = i conj(conj(w) dm) = i conj(u)
            s[ib] = make_float2(sp.x + u.y, -sp.y + u.x);                                // conj(sp) + i conj(u)
        }
        __syncthreads();
        // inverse, decimation in time, mirrored: the single radix-2 stage first if log2(M) is odd,
        // then spans q and 2q per pass
        int hq = 1;
        if (logM & 1) {
            for (int j = tid; j < (M >> 1); j += nt) {
                const float2 u = s[2 * j], v = s[2 * j + 1];
                s[2 * j] = make_float2(u.x + v.x, u.y + v.y);
                s[2 * j + 1] = make_float2(u.x - v.x, u.y - v.y);
            }
            __syncthreads();
            hq = 2;
        }
        for (int q = hq; q <= (M >> 2); q <<= 2) {
            const float2 *w1 = stw + (q - 1), *w2 = stw + (2 * q - 1);
            for (int j = tid; j < (M >> 2); j += nt) {
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
        for (int n = tid; 2 * n < N; n += nt) {
            const float2 v = s[n];
            V[(size_t)m * N + 2 * n] = v.x * inv;
            if (2 * n + 1 < N) V[(size_t)m * N + 2 * n + 1] = v.y * inv;
        }
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

// ---------------------------------------------------------------- a3: direct wake
// grid = (ceil(N / WD_ROWS), members), block = 256 (one row per warp), dynamic shared memory
// (2N + WD_ROWS) floats: the profile (complete after k_rotate2) and the N + WD_ROWS - 1 lags of the
// wake function this CTA's rows touch are staged with coalesced loads, then warp w evaluates
// V_x = sum_x' w[x - x'] rho_x' (Eq. 4; w = Re IDFT(Z) from create, lag d at index d + N - 1)
// for x = r0 + w.  pw_part[m][cta] = sum over the CTA's rows of rho_x V_x.
// dpU != nullptr (clamped interpolation; N + WD_ROWS more floats of shared memory): the clamped
// kick is not conservative, so the CSR power of the END-of-step profile rho' is formed to first
// order in rho' - rho:  sum rho' V' = sum rho V + sum (rho' - rho)(V + Vt),  Vt_x = sum_x' w[x' - x]
// rho_x' (transposed wake).  Then pw_part = sum -rho_x Vt_x and dpU[m][x] = dp (V_x + Vt_x), which
// the kick kernel multiplies with its row sums.
__global__ void __launch_bounds__(WD_THREADS)
k_wake_direct(int N, const float *__restrict__ rho, const float *__restrict__ wfun, float *__restrict__ V,
              float *__restrict__ pw_part, float *__restrict__ dpU, float dp)
{
    extern __shared__ float wd_smem[];
    __shared__ float wpw[WD_THREADS / 32];
    float *srho = wd_smem, *sw = wd_smem + N, *sw2 = wd_smem + 2 * N + WD_ROWS;
    const int m = blockIdx.y, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int r0 = blockIdx.x * WD_ROWS;
    const float *gr = rho + (size_t)m * N, *gw = wfun + (size_t)m * 2 * N;
    for (int i = tid; i < N; i += WD_THREADS) srho[i] = __ldg(gr + i);
    for (int i = tid; i < N + WD_ROWS - 1; i += WD_THREADS) sw[i] = (r0 + i < 2 * N - 1) ? __ldg(gw + r0 + i) : 0.0f;
    const int base2 = N - r0 - WD_ROWS;                // sw2[i] = w at index base2 + i
    if (dpU != nullptr)
        for (int i = tid; i < N + WD_ROWS - 1; i += WD_THREADS) {
            const int k = base2 + i;
            sw2[i] = (k >= 0 && k < 2 * N - 1) ? __ldg(gw + k) : 0.0f;
        }
    __syncthreads();
    const int x = r0 + warp;
    float v0 = 0.0f, v1 = 0.0f, u0 = 0.0f, u1 = 0.0f;
    if (x < N) {
        const float *wx = sw + (warp + N - 1);
        int xp = lane;
        for (; xp + 32 < N; xp += 64) {
            v0 = fmaf(wx[-xp], srho[xp], v0);
            v1 = fmaf(wx[-(xp + 32)], srho[xp + 32], v1);
        }
        if (xp < N) v0 = fmaf(wx[-xp], srho[xp], v0);
        if (dpU != nullptr) {
            const float *ux = sw2 + (WD_ROWS - 1 - warp);      // w[x' - x] at ux[x']
            xp = lane;
            for (; xp + 32 < N; xp += 64) {
                u0 = fmaf(ux[xp], srho[xp], u0);
                u1 = fmaf(ux[xp + 32], srho[xp + 32], u1);
            }
            if (xp < N) u0 = fmaf(ux[xp], srho[xp], u0);
        }
    }
    const float v = warp_sum(v0 + v1);
    const float vt = (dpU != nullptr) ? warp_sum(u0 + u1) : 0.0f;
    if (lane == 0) {
        float pw = 0.0f;
        if (x < N) {
            V[(size_t)m * N + x] = v;
            if (dpU != nullptr) { dpU[(size_t)m * N + x] = dp * (v + vt); pw = -srho[x] * vt; }
            else pw = srho[x] * v;
        }
        wpw[warp] = pw;
    }
    __syncthreads();
    if (tid == 0) {
        float t = 0.0f;
#pragma unroll
        for (int i = 0; i < WD_THREADS / 32; ++i) t += wpw[i];
        pw_part[(size_t)m * gridDim.x + blockIdx.x] = t;
    }
}

}  // namespace vfps
