/*
 * vfps_oracle.c -- TEST INFRASTRUCTURE.  Plain, slow, double-precision CPU restatement of one
 * Warnock-Ellison split step of the Vlasov-Fokker-Planck equation as described in
 * arXiv:1611.05293, written from the paper's text only.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this.  It shares no code, header, table or constant generator with the CUDA path
 * (paper_1611_05293_b200/csrc) and neither includes the other.
 *
 * Every function follows the cited passage step by step, in the paper's order and notation,
 * with no blocking, fusion or reordering.  The only parallelism is an OpenMP "parallel for" over
 * independent output elements (it does not change any arithmetic or summation order).
 *
 * Notation: N grid points per axis; x = q index, y = p index; flat index
 * z = N*x + y (p contiguous); q_x = q_min + x*dq, dq = (q_max-q_min)/(N-1) (reading A2 in
 * both ends are nodes); dphi = 2*pi/steps_per_period (reading A1); b = beta/spp.
 *
 * Pins (tests/test_oracle_pins.py, all independent of this file's formulas): polynomial
 * exactness of the interpolation, closed-form moment laws of rotation / kick / Fokker-Planck,
 * Parseval identity wake <-> CSR power, free-space radiated-power closed form, quarter-period
 * displacement of a blob, stationarity of the Gaussian, and for the Manhattan rotation the exact
 * linear symplectic map of means and covariances (P14), no-overshoot of the clamped interpolation (P15).  The full nonlinear CSR run has no closed
 * form: "parity unpinned" beyond those pins.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define VFPO_MAX_ORDER 4

int vfpo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void vfpo_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---- Lagrange interpolation, PAPER.md L91-108 (Eq. 10-13) ---------------------------------
 * N_i-point stencil around m = floor(m_r): nodes m - floor((N_i-1)/2) ... m + ceil((N_i-1)/2)
 * (Eq. 11), i.e. node offsets o_k = k - floor((N_i-1)/2); weights are the Lagrange basis
 * polynomials l_nu(t) = prod_{k != nu} (t - o_k)/(o_nu - o_k) at t = {m} = m_r - m (Eq. 13). */
static int node_offset(int order, int k) { return k - (order - 1) / 2; }

void vfpo_lagrange_weights(int order, double t, double *l)
{
    for (int nu = 0; nu < order; ++nu) {
        double w = 1.0;
        for (int k = 0; k < order; ++k) {
            if (k == nu) continue;
            w *= (t - (double)node_offset(order, k)) /
                 ((double)node_offset(order, nu) - (double)node_offset(order, k));
        }
        l[nu] = w;
    }
}

/* psi = 0 outside the grid for every tap of every step (reading A8). */
static double at(const double *psi, int N, int x, int y)
{
    if (x < 0 || x >= N || y < 0 || y >= N) return 0.0;
    return psi[(size_t)N * x + y];
}

/* Eq. 14 as read in DESIGN.md A9: the printed formula always returns
 * max(a, b); the intended "clamped or saturated" interpolation limits the interpolated value to
 * the interval spanned by the nodes that bracket the evaluation point. */
static double clamp_to(double v, double lo, double hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* 1-D interpolation along p of column x at real grid coordinate y_r (Eq. 10). */
static double interp_p(const double *psi, int N, int order, int x, double y_r, int clamp)
{
    double l[VFPO_MAX_ORDER];
    double m = floor(y_r);
    vfpo_lagrange_weights(order, y_r - m, l);
    double acc = 0.0;
    for (int j = 0; j < order; ++j)
        acc += l[j] * at(psi, N, x, (int)m + node_offset(order, j));
    if (clamp) {
        double a = at(psi, N, x, (int)m), b = at(psi, N, x, (int)m + 1);
        acc = clamp_to(acc, fmin(a, b), fmax(a, b));
    }
    return acc;
}

/* ---- O1 rotation ("standard rotation"; flow of Eq. 1: dq/dtheta = +p,
 * dp/dtheta = -q).  Target (x,y) takes the value interpolated (N_i x N_i taps) at the
 * back-rotated source point q_s = c q - s p, p_s = s q + c p with exact cos/sin (reading A3). */
void vfpo_rotate(int N, double q_min, double q_max, double p_min, double p_max, double dphi,
                 int order, const double *psi, double *out, int clamp)
{
    const double dq = (q_max - q_min) / (N - 1), dp = (p_max - p_min) / (N - 1);
    const double c = cos(dphi), s = sin(dphi);
#pragma omp parallel for schedule(static)
    for (int x = 0; x < N; ++x) {
        for (int y = 0; y < N; ++y) {
            double q = q_min + x * dq, p = p_min + y * dp;
            double q_s = c * q - s * p, p_s = s * q + c * p;
            double x_r = (q_s - q_min) / dq, y_r = (p_s - p_min) / dp;   /* Eq. 9 */
            double mx = floor(x_r), my = floor(y_r);
            double lx[VFPO_MAX_ORDER], ly[VFPO_MAX_ORDER];
            vfpo_lagrange_weights(order, x_r - mx, lx);
            vfpo_lagrange_weights(order, y_r - my, ly);
            double acc = 0.0;
            for (int i = 0; i < order; ++i)
                for (int j = 0; j < order; ++j)
                    acc += lx[i] * ly[j] *
                           at(psi, N, (int)mx + node_offset(order, i), (int)my + node_offset(order, j));
            if (clamp) {          /* the 2 x 2 nodes around the source point */
                double a = at(psi, N, (int)mx, (int)my), b = at(psi, N, (int)mx, (int)my + 1);
                double c2 = at(psi, N, (int)mx + 1, (int)my), d2 = at(psi, N, (int)mx + 1, (int)my + 1);
                acc = clamp_to(acc, fmin(fmin(a, b), fmin(c2, d2)), fmax(fmax(a, b), fmax(c2, d2)));
            }
            out[(size_t)N * x + y] = acc;
        }
    }
}

/* 1-D interpolation along q of column y at real grid coordinate x_r (Eq. 10). */
static double interp_q(const double *psi, int N, int order, double x_r, int y, int clamp)
{
    double l[VFPO_MAX_ORDER];
    double m = floor(x_r);
    vfpo_lagrange_weights(order, x_r - m, l);
    double acc = 0.0;
    for (int i = 0; i < order; ++i)
        acc += l[i] * at(psi, N, (int)m + node_offset(order, i), y);
    if (clamp) {
        double a = at(psi, N, (int)m, y), b = at(psi, N, (int)m + 1, y);
        acc = clamp_to(acc, fmin(a, b), fmax(a, b));
    }
    return acc;
}

/* ---- O1' "Manhattan rotation" (the symplectic map "splits the rotation into a
 * energy-dependent drift followed by a location dependent RF kick.  Each requires a
 * one-dimensional interpolation").  With the flow of Eq. 1 (dq/dtheta = +p, dp/dtheta = -q) and
 * the first-order symplectic (Euler) map of the paper's ref. [23] (reading A15):
 *   drift    q' = q + dphi p      psi_A(q, p) = psi(q - dphi p, p)       interpolation along q
 *   RF kick  p' = p - dphi q'     psi_B(q, p) = psi_A(q, p + dphi q)     interpolation along p */
void vfpo_drift(int N, double q_min, double q_max, double p_min, double p_max, double dphi, int order,
                const double *psi, double *out, int clamp)
{
    const double dq = (q_max - q_min) / (N - 1), dp = (p_max - p_min) / (N - 1);
#pragma omp parallel for schedule(static)
    for (int x = 0; x < N; ++x)
        for (int y = 0; y < N; ++y) {
            double p = p_min + y * dp;
            out[(size_t)N * x + y] = interp_q(psi, N, order, (double)x - dphi * p / dq, y, clamp);
        }
}

void vfpo_rf_kick(int N, double q_min, double q_max, double p_min, double p_max, double dphi, int order,
                  const double *psi, double *out, int clamp)
{
    const double dq = (q_max - q_min) / (N - 1), dp = (p_max - p_min) / (N - 1);
#pragma omp parallel for schedule(static)
    for (int x = 0; x < N; ++x) {
        double q = q_min + x * dq;
        for (int y = 0; y < N; ++y)
            out[(size_t)N * x + y] = interp_p(psi, N, order, x, (double)y + dphi * q / dp, clamp);
    }
}

/* ---- O2 projection: bunch profile rho_x = dp * sum_y psi(x,y). */
void vfpo_project(int N, double dp, const double *psi, double *rho)
{
#pragma omp parallel for schedule(static)
    for (int x = 0; x < N; ++x) {
        double acc = 0.0;
        for (int y = 0; y < N; ++y) acc += psi[(size_t)N * x + y];
        rho[x] = dp * acc;
    }
}

/* ---- wake function from the impedance.  Z holds k = 0..N_f/2 as (re,im) pairs; the spectrum is
 * Hermitian, so the real inverse DFT of Z sampled at lag d is
 *   w[d] = (1/N_f) [ Re Z_0 + 2 sum_{k=1}^{N_f/2-1} Re(Z_k e^{2 pi i k d/N_f}) + Re Z_{N_f/2} (-1)^d ].
 * Stored for d = -(N-1)..(N-1) at index d + N - 1. */
void vfpo_wake_function(int N, int Nf, const double *Z, double *w)
{
    const double PI = 3.14159265358979323846;
#pragma omp parallel for schedule(static)
    for (int d = -(N - 1); d <= N - 1; ++d) {
        double acc = Z[0];
        for (int k = 1; k < Nf / 2; ++k) {
            /* reduce k*d mod N_f in integers so the angle stays small and exact */
            long long kd = ((long long)k * d) % Nf;
            double ang = 2.0 * PI * (double)kd / (double)Nf;
            acc += 2.0 * (Z[2 * k] * cos(ang) - Z[2 * k + 1] * sin(ang));
        }
        acc += Z[2 * (Nf / 2)] * ((d % 2) ? -1.0 : 1.0);
        w[d + N - 1] = acc / (double)Nf;
    }
}

/* ---- O3 wake potential by direct convolution, Eq. 4:
 * V_x = sum_{x'} w[x - x'] rho_{x'}.  Equal to Re IDFT(Z .* DFT(zero-padded rho)) of Eq. 5
 * (L52-54) because |x - x'| < N <= N_f/2 never wraps. */
void vfpo_wake(int N, const double *w, const double *rho, double *V)
{
#pragma omp parallel for schedule(static)
    for (int x = 0; x < N; ++x) {
        double acc = 0.0;
        for (int xp = 0; xp < N; ++xp) acc += w[(x - xp) + N - 1] * rho[xp];
        V[x] = acc;
    }
}

/* ---- O4 kick: every particle of column x changes its energy by
 * Delta p_x = -dphi * V_x (readings A1, A6), so psi''(x,p) = psi'(x, p - Delta p_x):
 * y_r = y - Delta p_x / dp, 1-D interpolation along p. */
void vfpo_kick(int N, double dp, double dphi, int order, const double *V, const double *psi,
               double *out, int clamp)
{
#pragma omp parallel for schedule(static)
    for (int x = 0; x < N; ++x) {
        double delta_p = -dphi * V[x];
        for (int y = 0; y < N; ++y)
            out[(size_t)N * x + y] = interp_p(psi, N, order, x, (double)y - delta_p / dp, clamp);
    }
}

/* ---- O5 Fokker-Planck (right-hand side of Eq. 1; discretisation L138-147):
 * beta d/dp (p psi + dpsi/dp) = beta (psi + p psi_p + psi_pp), explicit Euler with b = beta/spp,
 * psi_p from Eq. 15 (derivative of the cubic P_4 at x_0), psi_pp the three-point formula
 * (= second derivative of P_4 at x_0), zero ghosts (readings A7, A8). */
void vfpo_fokker_planck(int N, double p_min, double p_max, double b, const double *psi, double *out)
{
    const double dp = (p_max - p_min) / (N - 1);
#pragma omp parallel for schedule(static)
    for (int x = 0; x < N; ++x) {
        for (int y = 0; y < N; ++y) {
            double fm1 = at(psi, N, x, y - 1), f0 = at(psi, N, x, y);
            double fp1 = at(psi, N, x, y + 1), fp2 = at(psi, N, x, y + 2);
            double p = p_min + y * dp;
            double d1 = (-2.0 * fm1 - 3.0 * f0 + 6.0 * fp1 - fp2) / (6.0 * dp);   /* Eq. 15 */
            double d2 = (fm1 - 2.0 * f0 + fp1) / (dp * dp);
            out[(size_t)N * x + y] = f0 + b * (f0 + p * d1 + d2);
        }
    }
}

/* ---- O6 diagnostics.  out = { M0, <q>, <p>, sigma_q, sigma_p } with M0 = dq dp sum psi,
 * <q> = dq dp sum q_x psi / M0, sigma_q^2 = dq dp sum q_x^2 psi / M0 - <q>^2 (bunch length,
 * energy spread: PAPER.md L153, L176). */
void vfpo_moments(int N, double q_min, double q_max, double p_min, double p_max, const double *psi,
                  double *out)
{
    const double dq = (q_max - q_min) / (N - 1), dp = (p_max - p_min) / (N - 1);
    double s0 = 0, sq = 0, sqq = 0, sp = 0, spp = 0;
    for (int x = 0; x < N; ++x) {
        double q = q_min + x * dq;
        for (int y = 0; y < N; ++y) {
            double p = p_min + y * dp, f = psi[(size_t)N * x + y];
            s0 += f; sq += q * f; sqq += q * q * f; sp += p * f; spp += p * p * f;
        }
    }
    double M0 = dq * dp * s0;
    double mq = sq / s0, mp = sp / s0;
    out[0] = M0;
    out[1] = mq;
    out[2] = mp;
    out[3] = sqrt(sqq / s0 - mq * mq);
    out[4] = sqrt(spp / s0 - mp * mp);
}

/* CSR power, Eq. 16-17: P(k) ~ Re Z_k |rho~_k|^2, P = integral over k.
 * Normalised (reading A10) as P = (dq/N_f) sum_{k=0}^{N_f-1} Re Z_k |R_k|^2 with
 * R = DFT_{N_f}(zero-padded rho), folded onto k = 0..N_f/2 by Hermitian symmetry. */
double vfpo_csr_power(int N, int Nf, double dq, const double *Z, const double *rho)
{
    const double PI = 3.14159265358979323846;
    double total = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : total)
    for (int k = 0; k <= Nf / 2; ++k) {
        double re = 0.0, im = 0.0;
        for (int x = 0; x < N; ++x) {
            long long kx = ((long long)k * x) % Nf;
            double ang = -2.0 * PI * (double)kx / (double)Nf;
            re += rho[x] * cos(ang);
            im += rho[x] * sin(ang);
        }
        double fold = (k == 0 || k == Nf / 2) ? 1.0 : 2.0;
        total += fold * Z[2 * k] * (re * re + im * im);
    }
    return total * dq / (double)Nf;
}

/* ---- one full split step (BASELINE order a1..a6, reading A14), state held by the caller ---- */
typedef struct {
    int N;
    double q_min, q_max, p_min, p_max;
    int steps_per_period;
    double beta;       /* per synchrotron period */
    int interp_order;  /* 2, 3, 4 */
    int pad;           /* N_f = pad * N */
    int renormalise;   /* 1: psi_{t+1} = psi''' / C */
    int manhattan;     /* 1: a1 is the Manhattan rotation (drift, RF kick) instead of the standard one */
    int clamp;         /* 1: every interpolation is clamped (Eq. 14, reading A9) */
} vfpo_params;

/* psi: in/out [N][N] double.  Z: (N_f/2+1) (re,im) pairs or NULL (no wake).  w: wake function
 * from vfpo_wake_function (ignored if Z NULL).  diag (nullable): {C, <q>, <p>, sigma_q, sigma_p,
 * P_csr} of this step; rho_out/V_out (nullable): post-rotation profile and its wake. */
void vfpo_step(const vfpo_params *P, const double *Z, const double *w, double *psi, double *diag,
               double *rho_out, double *V_out)
{
    const int N = P->N;
    const size_t cells = (size_t)N * N;
    const double PI = 3.14159265358979323846;
    const double dq = (P->q_max - P->q_min) / (N - 1), dp = (P->p_max - P->p_min) / (N - 1);
    const double dphi = 2.0 * PI / P->steps_per_period;
    const double b = P->beta / P->steps_per_period;
    double *t1 = (double *)malloc(cells * sizeof(double));
    double *t2 = (double *)malloc(cells * sizeof(double));
    double *rho = (double *)malloc(N * sizeof(double));
    double *V = (double *)calloc(N, sizeof(double));

    if (P->manhattan) {                                                                      /* a1 */
        vfpo_drift(N, P->q_min, P->q_max, P->p_min, P->p_max, dphi, P->interp_order, psi, t2, P->clamp);
        vfpo_rf_kick(N, P->q_min, P->q_max, P->p_min, P->p_max, dphi, P->interp_order, t2, t1, P->clamp);
    } else {
        vfpo_rotate(N, P->q_min, P->q_max, P->p_min, P->p_max, dphi, P->interp_order, psi, t1, P->clamp);
    }
    vfpo_project(N, dp, t1, rho);                                                            /* a2 */
    if (Z) vfpo_wake(N, w, rho, V);                                                          /* a3 */
    vfpo_kick(N, dp, dphi, P->interp_order, V, t1, t2, P->clamp);                                      /* a4 */
    vfpo_fokker_planck(N, P->p_min, P->p_max, b, t2, t1);                                    /* a5 */
    double C = 0.0;                                                                          /* a6 */
    for (size_t z = 0; z < cells; ++z) C += t1[z];
    C *= dq * dp;
    if (P->renormalise)
        for (size_t z = 0; z < cells; ++z) psi[z] = t1[z] / C;
    else
        memcpy(psi, t1, cells * sizeof(double));
    if (rho_out) memcpy(rho_out, rho, N * sizeof(double));
    if (V_out) memcpy(V_out, V, N * sizeof(double));
    if (diag) {
        double m[5];
        vfpo_moments(N, P->q_min, P->q_max, P->p_min, P->p_max, psi, m);
        diag[0] = C;
        diag[1] = m[1]; diag[2] = m[2]; diag[3] = m[3]; diag[4] = m[4];
        if (Z) {
            vfpo_project(N, dp, psi, rho);
            diag[5] = vfpo_csr_power(N, P->pad * N, dq, Z, rho);
        } else {
            diag[5] = 0.0;
        }
    }
    free(t1); free(t2); free(rho); free(V);
}

/* n steps; diag (nullable) [n][6]; diag_every: compute diagnostics only every k-th step
 * (rows of skipped steps are left untouched), 1 = every step. */
void vfpo_run(const vfpo_params *P, const double *Z, double *psi, int n, double *diag,
              int diag_every)
{
    double *w = NULL;
    if (Z) {
        w = (double *)malloc((2 * (size_t)P->N - 1) * sizeof(double));
        vfpo_wake_function(P->N, P->pad * P->N, Z, w);
    }
    for (int i = 0; i < n; ++i) {
        double *d = NULL;
        if (diag && diag_every > 0 && ((i + 1) % diag_every == 0 || i == n - 1)) d = diag + 6 * (size_t)i;
        vfpo_step(P, Z, w, psi, d, NULL, NULL);
    }
    free(w);
}
