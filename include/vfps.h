/*
 * vfps.h -- C ABI of the B200-native Vlasov-Fokker-Planck phase-space step.
 *
 * One call of vfps_step(h, n, diag) advances the discretised longitudinal phase-space density
 * psi(q,p) by n full Warnock-Ellison split steps (arXiv:1611.05293; citations are PAPER.md lines):
 *
 *   a1 rotation     semi-Lagrangian rotation by dphi = 2*pi/steps_per_period about (q,p) = (0,0),
 *                   interp_order x interp_order Lagrange interpolation at the back-rotated source
 *                   point ("standard rotation", L136; Eq. 10-13; flow of Eq. 1)
 *   a2 projection   bunch profile rho_x = dp * sum_y psi(x,y)                              (L56)
 *   a3 wake         V = Re IDFT_Nf[ Z .* DFT_Nf(rho zero-padded to Nf = pad*N) ], first N samples
 *                   (Eq. 5; Hermitian spectrum, only k = 0..Nf/2 stored, L149)
 *   a4 kick         psi(x, p) <- psi(x, p - Dp_x), Dp_x = -dphi * V_x, 1-D Lagrange interpolation
 *                   along p                                                              (L40, L149)
 *   a5 Fokker-Planck psi <- psi + b*(psi + p*D1 psi + D2 psi), b = beta/steps_per_period,
 *                   D1 = Eq. 15 (L144), D2 = three-point second difference (L138-147), along p
 *   a6 diagnostics  C = dq*dp*sum psi (pre-renormalisation charge); psi <- psi/C (flag);
 *                   <q>, <p>, sigma_q (bunch length), sigma_p (energy spread), CSR power
 *                   P = (dq/Nf) sum_k Re Z_k |rho~_k|^2                      (Eq. 16-17)
 *
 * Grid and layout: N points per axis; x = q index, y = p index; q_x = q_min + x*dq with
 * dq = (q_max - q_min)/(N-1) (both ends are nodes), same for p; psi = 0 outside the grid.
 * psi arrays are [members][N][N] fp32, index (m, x, y), p (y) contiguous (flat z = N*x + y, L124).
 * Batched mode: `members` independent simulations advance together, member m uses row m of Z.
 *
 * Conventions of every call:
 *   - returns VFPS_OK (0) or a negative vfps_status; vfps_last_error(h) gives text.  No exception
 *     crosses the ABI.  Unsupported combinations return VFPS_ERR_UNSUPPORTED -- there is no CPU
 *     fallback and no silent change of method.
 *   - the handle is opaque and owned by the library; every array argument is caller-owned and is
 *     not retained after the call returns (inputs are copied into library-owned device memory).
 *   - array pointers are DEVICE pointers, used asynchronously on the handle's stream, unless the
 *     function name ends in `_host` (then: host pointers, and the call returns after the copy
 *     has completed).
 *   - nothing in vfps_step synchronises with the host.
 */
#ifndef VFPS_H
#define VFPS_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vfps_sim *vfps_handle;

typedef enum vfps_status {
    VFPS_OK = 0,
    VFPS_ERR_ARG = -1,         /* NULL / out-of-range argument */
    VFPS_ERR_STATE = -2,       /* call not valid in the handle's state (e.g. step before set_psi) */
    VFPS_ERR_CUDA = -3,        /* a CUDA runtime call failed; text in vfps_last_error */
    VFPS_ERR_NOMEM = -4,       /* device or host allocation failed */
    VFPS_ERR_UNSUPPORTED = -5  /* valid request this build does not implement */
} vfps_status;

/* interleaved complex fp32, layout-compatible with CUDA float2 / C99 float _Complex */
typedef struct vfps_complex { float re, im; } vfps_complex;

enum {
    VFPS_FLAG_RENORMALISE = 1,   /* psi <- psi / C after every step (BASELINE north_star (6)) */
    VFPS_FLAG_CLAMP = 2,         /* clamped interpolation (Eq. 14, read as: limit every
                                    interpolated value to the interval of its bracketing nodes);
                                    every engine (with ROT_MANHATTAN: STREAM / GRAPH / GRID); the
                                    wake must be evaluated by direct convolution                 */
    VFPS_FLAG_ROT_MANHATTAN = 4  /* a1 is the symplectic "Manhattan" rotation (L136): drift along q then
                                    RF kick along p, two 1-D interpolations; every engine (CLUSTER:
                                    k_cluster_step, GRID: k_grid_step)                              */
};

typedef struct vfps_params {
    int N;                 /* grid points per axis, >= 8; N*pad must be a power of two          */
    double q_min, q_max;   /* position axis, units of sigma_z0                                    */
    double p_min, p_max;   /* energy axis, units of sigma_delta0                                  */
    int steps_per_period;  /* time steps per synchrotron period; dphi = 2*pi/steps_per_period     */
    double beta;           /* 1/(f_s tau_d): damping per synchrotron period (Eq. 1)          */
    int interp_order;      /* Lagrange points per axis: 2 linear, 3 quadratic, 4 cubic (Eq. 10)  */
    int pad;               /* zero-padding factor of the wake FFT, power of two >= 2             */
    int members;           /* independent simulations advanced per call, 1 .. 65535              */
    int flags;             /* VFPS_FLAG_*                                                        */
} vfps_params;

/* Run-time options (vfps_set_option).  All engines and wake modes compute the same step. */
enum {
    VFPS_OPT_ENGINE = 1,   /* how n steps are issued                                             */
    VFPS_OPT_WAKE = 2,     /* how a3 is evaluated                                                */
    VFPS_OPT_TIMING = 3,   /* 0/1: bracket kernel launches with CUDA events (measurement aid; while
                              on, vfps_step may synchronise the stream to read finished events)  */
    VFPS_OPT_CLUSTER_SIZE = 4, /* CTAs per cluster of the CLUSTER engine: 0 = auto, 1, 2, 4, 8, 16;
                              vfps_get_option returns the size in use (0 = engine unavailable)  */
    VFPS_OPT_GRID_KERNEL = 6,    /* kernel of the GRID engine: 0 = auto, 1 = k_grid_step (taps gathered
                              through L1; also the Manhattan rotation), 2 = k_grid2_step (tiles staged
                              by TMA, row stripes kicked from shared memory; N a multiple of 256);
                              get returns the one in use (0 = engine unavailable)                */
    VFPS_OPT_CLUSTER_KERNEL = 5  /* kernel of the CLUSTER engine: 0 = auto, 1 = first design
                              (k_cluster_step: two buffers, weights per cell; also the Manhattan
                              rotation), 3 = in-place design (k_onchip_step: one buffer, per-launch
                              weight tables; a 256^2 grid fits two CTAs); get returns the one in use */
};
/* kernel ids of vfps_kernel_time / vfps_kernel_name */
enum {
    VFPS_KERNEL_WAKE = 0,     /* k_wake_fft: a2 finish + a3 by FFT (Eq. 5) + q-moments + CSR power */
    VFPS_KERNEL_CLUSTER = 1,  /* a1..a6 for all n steps of one vfps_step call (cluster engine)   */
    VFPS_KERNEL_ROTATE2 = 2,  /* k_rotate2 / k_drift2: a1 + a2, streaming (register window)      */
    VFPS_KERNEL_WAKE_DIRECT = 3, /* k_wake_direct: a3 by direct convolution (Eq. 4) on N/8 CTAs   */
    VFPS_KERNEL_KICK_FP2 = 4, /* k_kick_fp2: a4 + a5 + a6 (four cells per thread)                */
    VFPS_KERNEL_GRID = 5,     /* a1..a6 for all n steps of one vfps_step call (grid engine)      */
    VFPS_KERNEL_GRID2 = 6,    /* the same, TMA-staged kernel of the grid engine                  */
    VFPS_NUM_KERNELS = 7
};
enum {
    VFPS_ENGINE_AUTO = 0,     /* one simulation with N >= 512: GRID where its TMA kernel is
                                 feasible; else CLUSTER if the grid fits on chip, else GRID (one
                                 simulation) or GRAPH (a batch)                                  */
    VFPS_ENGINE_STREAM = 1,   /* one launch per kernel per step on the stream                    */
    VFPS_ENGINE_GRAPH = 2,    /* the same kernels replayed from a CUDA graph of many steps       */
    VFPS_ENGINE_CLUSTER = 3,  /* persistent thread-block-cluster kernel, psi resident in
                                 distributed shared memory for all n steps                       */
    VFPS_ENGINE_GRID = 4      /* persistent cooperative kernel on every SM, psi in L2 / HBM, grid
                                 barriers where the step has global dependencies (members = 1)   */
};
enum {
    VFPS_WAKE_AUTO = 0,       /* DIRECT                                                          */
    VFPS_WAKE_FFT = 1,        /* zero-padded length-Nf FFT, x Z, inverse FFT, every step (Eq. 5) */
    VFPS_WAKE_DIRECT = 2      /* w = Re IDFT(Z) once at create; V = w * rho by direct convolution
                                 (Eq. 4) -- identical result, no serial FFT chain per step  */
};

/* Create a simulation.  Z: device pointer to [members][pad*N/2 + 1] impedance samples Z_k at
 * wavenumber index k = 0..Nf/2 in the normalisation V = Re IDFT(Z .* DFT(rho)) (the caller folds
 * every physical constant, e.g. 4*pi*S_csr, into Z), or NULL for no collective force (kick = exact
 * identity, CSR power = 0).  Im Z_0 and Im Z_{Nf/2} are ignored (Hermitian spectrum).
 * cuda_stream: a cudaStream_t (NULL = the legacy default stream); all work of this handle is
 * issued there.  psi is zero until vfps_set_psi. */
int vfps_create(const vfps_params *p, const vfps_complex *Z, void *cuda_stream, vfps_handle *out);
int vfps_create_host(const vfps_params *p, const vfps_complex *Z_host, void *cuda_stream,
                     vfps_handle *out);

/* Free everything the handle owns.  NULL is accepted. */
int vfps_destroy(vfps_handle h);

/* Engine / wake-mode selection; may be called any time between steps. */
int vfps_set_option(vfps_handle h, int option, int value);
int vfps_get_option(vfps_handle h, int option, int *value);

/* Replace the impedance of a simulation that was created with one (same layout as in vfps_create);
 * psi and the step counter are kept.  This is the paper's adiabatic current scan (L239, L290-298,
 * App. A): the final distribution of one bunch current is the starting distribution of the next.
 * VFPS_ERR_STATE if the handle was created with Z = NULL. */
int vfps_set_impedance(vfps_handle h, const vfps_complex *Z);
int vfps_set_impedance_host(vfps_handle h, const vfps_complex *Z_host);

/* Copy psi [members][N][N] into the simulation; no renormalisation; step counter := 0. */
int vfps_set_psi(vfps_handle h, const float *psi);
int vfps_set_psi_host(vfps_handle h, const float *psi_host);

/* Advance n >= 0 steps a1..a6.  diag: NULL or [n][members][6] floats; row (i, m) =
 * { C (charge before renormalisation), <q>, <p>, sigma_q, sigma_p, P_csr } after step i.
 * All moments are those of the end-of-step psi (the STREAM / GRAPH engines take <q>, sigma_q from the
 * post-rotation profile).  P_csr (Eq. 16-17, normalised as the energy loss per radian) is formed from
 * the profile the wake acts on in the same step, scaled by 1/C^2: kick and Fokker-Planck act along p
 * only and leave the profile unchanged up to the charge that crosses the p edges of the box during the
 * step (< 1e-6 relative for densities that fit their box).  With VFPS_FLAG_CLAMP, where the kick is not
 * conservative, it is the CSR power of the END-of-step profile rho' to first order in rho' - rho
 * (transposed wake; the neglected term is quadratic in the change of the profile).
 * Asynchronous on the handle's stream.  vfps_step_host copies diag to host memory and returns
 * when the n steps have completed. */
int vfps_step(vfps_handle h, int n, float *diag);
int vfps_step_host(vfps_handle h, int n, float *diag_host);

/* Current density psi_t (renormalised if the flag is set), [members][N][N]. */
int vfps_get_psi(vfps_handle h, float *psi_out);
int vfps_get_psi_host(vfps_handle h, float *psi_out_host);

/* Bunch profile rho_x = dp * sum_y psi_t(x,y) of the current psi, [members][N]. */
int vfps_get_profile(vfps_handle h, float *rho_out);
int vfps_get_profile_host(vfps_handle h, float *rho_out_host);

/* Wake potential V_x of the current profile (recomputed, stateless), [members][N]; zeros if the
 * simulation was created with Z = NULL. */
int vfps_get_wake(vfps_handle h, float *V_out);
int vfps_get_wake_host(vfps_handle h, float *V_out_host);

/* { C = dq*dp*sum psi_t, <q>, <p>, sigma_q, sigma_p, P_csr } of the current psi, [members][6]. */
int vfps_get_moments(vfps_handle h, float *out);
int vfps_get_moments_host(vfps_handle h, float *out_host);

/* Steps taken since the last vfps_set_psi. */
int vfps_step_count(vfps_handle h, long long *count);

/* Kernel launches (graph nodes included) issued by this handle so far. */
int vfps_launch_count(vfps_handle h, long long *count);

/* Device time spent in one kernel of the hot path, accumulated while VFPS_OPT_TIMING is 1:
 * total milliseconds between the CUDA events bracketing each launch, and the number of launches
 * bracketed (STREAM engine: the first 256 steps of every vfps_step call; CLUSTER engine: every
 * call; the GRAPH engine replays a captured graph and brackets nothing).  Synchronises the stream.
 * vfps_kernel_name(k) is NULL for k outside 0..VFPS_NUM_KERNELS-1. */
int vfps_kernel_time(vfps_handle h, int kernel, double *ms_total, long long *launches);
int vfps_reset_kernel_times(vfps_handle h);
const char *vfps_kernel_name(int kernel);

/* Name of the engine / wake mode the next vfps_step will use ("stream", "graph", "cluster", "grid";
 * "fft", "direct"); static strings. */
const char *vfps_engine_name(vfps_handle h);
const char *vfps_wake_name(vfps_handle h);

/* ---- a3 without a handle and without any allocation ------------------------------------------
 * Wake potential of a caller-held profile (Eq. 4-5):
 *     V_x = sum_x' w[x - x'] rho_x',  w = Re IDFT(Z) of the Hermitian spectrum Z_k, k = 0..N*pad/2
 * -- what vfps_get_wake returns for the profile of its handle (identical up to rounding: direct
 * convolution here, FFT there).  For callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it): the call makes no cudaMalloc / cudaFree
 * and uses no allocating library routine.  Its scratch, the wake function w (2N floats), lives in a
 * built-in device array of 2 * VFPS_NOALLOC_MAX_N floats (32 KB) that every GPU that loads the
 * library holds until the process exits.
 *   N, pad   grid points and zero-padding factor: pad >= 2 and N*pad powers of two, N >= 8;
 *            N > VFPS_NOALLOC_MAX_N or N*pad > 8192 -> VFPS_ERR_UNSUPPORTED
 *   Z        DEVICE, N*pad/2 + 1 values (as vfps_create's, one member), read only
 *   rho      DEVICE, N floats, read only;  V_out  DEVICE, N floats, written (must not alias rho)
 *   cuda_stream  a cudaStream_t (NULL = the legacy default stream); two kernels are launched on it,
 *            the call does not synchronise.  The first call on each device looks up the address
 *            of the scratch array (cudaGetSymbolAddress): make it outside a graph capture.
 * All calls on a device share the scratch array, which keeps the last call's wake function until
 * the next call overwrites it (nothing in it accumulates, so nothing needs clearing): calls that
 * overlap on the GPU -- different streams, concurrently replayed graphs -- race on it; serialise them.
 * Returns VFPS_OK or a negative vfps_status; vfps_noalloc_last_error() gives the text (per thread,
 * valid until the thread's next vfps_wake_noalloc call). */
#define VFPS_NOALLOC_MAX_N 4096
int vfps_wake_noalloc(int N, int pad, const vfps_complex *Z, const float *rho, float *V_out, void *cuda_stream);
const char *vfps_noalloc_last_error(void);

/* Text of the last error on this handle (or of the last failed vfps_create when h is NULL).
 * Valid until the next call on the same handle. */
const char *vfps_last_error(vfps_handle h);

const char *vfps_version(void);

#ifdef __cplusplus
}
#endif
#endif /* VFPS_H */
