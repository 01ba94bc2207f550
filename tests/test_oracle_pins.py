"""Pins for the CPU oracle: every check here is fixed by the paper or by mathematics, and none
re-types the oracle's own formulas (PAPER.md citations beside each pin; pin numbers follow
DESIGN.md section 5 / SURVEY.md section 8(c))."""
import math

import numpy as np
import pytest

from workloads import get_workload, make_impedance, make_psi0
from workloads.psi0 import grid_axis

TWO_PI = 2.0 * math.pi


def gauss(N, L, sq=1.0, sp=1.0, q0=0.0, p0=0.0):
    return make_psi0(N, -L, L, -L, L, sq, sp, 0.0, 0, q0, p0).astype(np.float64)


# ---------------------------------------------------------------- P11 interpolation (Eq. 10-13)
@pytest.mark.parametrize("order", [2, 3, 4])
def test_p11_weights_reproduce_monomials(orc, order):
    """sum_k l_k(t) o_k^j = t^j for j < order, nodes o_k = k - floor((order-1)/2) (Eq. 11, 13)."""
    nodes = np.arange(order) - (order - 1) // 2
    for t in (0.0, 0.125, 0.5, 0.73, 0.999):
        l = orc.lagrange_weights(order, t)
        for j in range(order):
            assert abs(np.dot(l, nodes.astype(float) ** j) - t ** j) < 1e-14
    # cardinal property: at t = 0 only the node m itself contributes
    l0 = orc.lagrange_weights(order, 0.0)
    assert l0[(order - 1) // 2] == 1.0 and np.count_nonzero(l0) == 1


def test_p11_cubic_weights_match_eq13_by_hand(orc):
    """Eq. 13 written out by hand for N=4, t = 1/2: (-1/16, 9/16, 9/16, -1/16)."""
    np.testing.assert_allclose(orc.lagrange_weights(4, 0.5), [-1 / 16, 9 / 16, 9 / 16, -1 / 16],
                               atol=1e-16)
    np.testing.assert_allclose(orc.lagrange_weights(3, 0.5), [-1 / 8, 3 / 4, 3 / 8], atol=1e-16)


@pytest.mark.parametrize("order", [2, 3, 4])
def test_p11_rotation_exact_on_polynomials(orc, order):
    """A tensor polynomial of degree < order per axis is interpolated exactly, so the rotated
    grid function equals the polynomial at the back-rotated point of the flow of Eq. 1 (L25):
    q(-dphi) = q cos + ... with dq/dtheta = +p, dp/dtheta = -q.  The polynomial is not
    symmetric in (q, p), so a transposed operand or a wrong rotation sense fails."""
    N, L = 12, 2.0
    q = grid_axis(N, -L, 1.5 * L)[:, None]          # non-symmetric box: q_min != -q_max
    p = grid_axis(N, -0.5 * L, L)[None, :]
    cq = [1.0, 0.7, -0.4, 0.3][:order]
    cp = [2.0, -1.1, 0.25, 0.6][:order]
    f = lambda qq, pp: (sum(c * qq ** i for i, c in enumerate(cq)) *
                        sum(c * pp ** i for i, c in enumerate(cp)))
    psi = f(q, p) + 0.0 * q * p
    dphi = 0.11
    out = orc.rotate(psi, -L, 1.5 * L, -0.5 * L, L, dphi, order)
    # independent statement of the characteristic: solve the ODE backwards with a fine RK4
    def back(q1, p1, n=2000):
        h = -dphi / n
        for _ in range(n):
            k1 = (p1, -q1)
            k2 = (p1 + h / 2 * k1[1], -(q1 + h / 2 * k1[0]))
            k3 = (p1 + h / 2 * k2[1], -(q1 + h / 2 * k2[0]))
            k4 = (p1 + h * k3[1], -(q1 + h * k3[0]))
            q1, p1 = (q1 + h / 6 * (k1[0] + 2 * k2[0] + 2 * k3[0] + k4[0]),
                      p1 + h / 6 * (k1[1] + 2 * k2[1] + 2 * k3[1] + k4[1]))
        return q1, p1
    qs, ps = back(q + 0 * p, p + 0 * q)
    expect = f(qs, ps)
    inner = slice(3, N - 3)       # stencils of these targets lie fully inside the grid
    np.testing.assert_allclose(out[inner, inner], expect[inner, inner], rtol=0, atol=2e-11)


# ---------------------------------------------------------------- P12 rotation sense (Eq. 1)
def test_p12_blob_moves_clockwise(orc):
    """dq/dtheta = +p, dp/dtheta = -q (L25): a blob at (q,p) = (+2,0) is at (0,-2) a quarter
    period later."""
    N, L, spp = 128, 6.0, 400
    psi = gauss(N, L, 0.5, 0.5, q0=2.0, p0=0.0)
    for _ in range(spp // 4):
        psi = orc.rotate(psi, -L, L, -L, L, TWO_PI / spp, 4)
    m = orc.moments(psi, -L, L, -L, L)
    assert abs(m[1] - 0.0) < 2e-4 and abs(m[2] + 2.0) < 2e-4


# ---------------------------------------------------------------- P6 / 2 f_s (L208)
def test_p6_mismatched_gaussian_breathes_at_2fs(orc):
    """Rotation only: sigma_q^2(n) = sigma_q0^2 cos^2(n dphi) + sigma_p0^2 sin^2(n dphi)."""
    N, L, spp = 256, 6.0, 400
    s_q, s_p = 1.2, 0.8
    psi = gauss(N, L, s_q, s_p)
    dphi = TWO_PI / spp
    for n in range(1, spp // 2 + 1):
        psi = orc.rotate(psi, -L, L, -L, L, dphi, 4)
        if n % 25 == 0:
            m = orc.moments(psi, -L, L, -L, L)
            want_q = math.sqrt(s_q ** 2 * math.cos(n * dphi) ** 2 + s_p ** 2 * math.sin(n * dphi) ** 2)
            want_p = math.sqrt(s_p ** 2 * math.cos(n * dphi) ** 2 + s_q ** 2 * math.sin(n * dphi) ** 2)
            assert abs(m[3] - want_q) < 1e-4 and abs(m[4] - want_p) < 1e-4
    # half a period later the bunch length is back: oscillation at 2 f_s
    assert abs(m[3] - s_q) < 1e-4


# ---------------------------------------------------------------- P4 full period
def test_p4_full_period_returns_psi(orc):
    N, L, spp = 128, 6.0, 500
    psi0 = gauss(N, L, 1.3, 0.7, q0=0.4, p0=-0.3)
    psi = psi0
    for _ in range(spp):
        psi = orc.rotate(psi, -L, L, -L, L, TWO_PI / spp, 4)
    assert np.max(np.abs(psi - psi0)) < 5e-3 * psi0.max()   # discretisation error only


# ---------------------------------------------------------------- P1 stationarity (L196)
def test_p1_gaussian_is_stationary_with_cubic(orc):
    """sigma = 1 Gaussian, no wake, rotation + Fokker-Planck: 'stays constant with time'."""
    wl = get_workload("C0").with_(interp_order=4)
    o = orc.Oracle.from_workload(wl)
    psi0 = o.psi.copy()
    d = o.step(wl.steps_per_period)
    assert np.all(np.abs(d[:, 3] - 1.0) < 2e-4) and np.all(np.abs(d[:, 4] - 1.0) < 2e-4)
    assert np.max(np.abs(o.psi - psi0)) < 1e-2 * psi0.max()
    assert np.all(np.abs(d[:, 0] - 1.0) < 1e-6)           # P3: cubic rotation, tiny charge drift


def test_p1_bilinear_diffusion_matches_prediction(orc):
    """C0 uses linear interpolation: one 1-D linear shift by a fraction t of a cell adds
    t(1-t) cell^2 of variance (variance of the two-point weight distribution).  With
    |shift| = sin(dphi)|p|/dq cells, averaging over the Gaussian gives
    d(sigma^2)/dn = sin(dphi) * dq * sqrt(2/pi) * sigma - sin(dphi)^2 * sigma^2 per step."""
    wl = get_workload("C0")
    o = orc.Oracle.from_workload(wl)
    n = wl.steps_per_period
    d = o.step(n)
    s = math.sin(TWO_PI / n)
    sig = 1.0
    for _ in range(n):
        sig = math.sqrt(sig ** 2 + s * wl.dq * math.sqrt(2 / math.pi) * sig - s * s * sig ** 2)
    assert abs(d[-1, 3] - sig) < 0.02 * sig and abs(d[-1, 4] - sig) < 0.02 * sig
    assert d[-1, 3] > 1.3                                   # violently diffusive, not a bug (H6)
    assert abs(d[-1, 0] - 1.0) < 1e-4                       # per-step charge stays ~1 (renormalised)


# ---------------------------------------------------------------- P5 Fokker-Planck closed form
def test_p5_fokker_planck_variance_law(orc):
    """FP only: (sigma_p^2 - 1)_n = (1 - 2b)^n (sigma_p0^2 - 1) exactly for this stencil pair
    (summation by parts), sigma_q untouched, charge conserved (P2)."""
    N, L, b, n = 160, 10.0, 1e-3, 300      # box wide enough that edge flux < 1e-13
    psi = gauss(N, L, 0.9, 1.25)
    m0 = orc.moments(psi, -L, L, -L, L)
    for _ in range(n):
        psi = orc.fokker_planck(psi, -L, L, b)
    m = orc.moments(psi, -L, L, -L, L)
    want = 1.0 + (1.0 - 2.0 * b) ** n * (m0[4] ** 2 - 1.0)
    assert abs(m[4] ** 2 - want) < 1e-9
    assert abs(m[3] - m0[3]) < 1e-12
    assert abs(m[0] - m0[0]) < 1e-9
    assert abs(m[2]) < 1e-12


def test_p5_relaxation_rate_with_rotation(orc):
    """With rotation the damping is shared between q and p: sigma^2 - 1 decays as
    exp(-beta*theta) (theta in periods), i.e. any distribution relaxes to sigma = 1 (L170)."""
    N, L, spp, beta = 128, 8.0, 200, 0.05
    o = orc.Oracle(N, -L, L, -L, L, spp, beta, 4)
    o.set_psi(gauss(N, L, 1.4, 1.4))
    d = o.step(4 * spp, diag_every=spp)
    s2 = d[spp - 1::spp, 3] ** 2 - 1.0
    rate = -np.log(s2[1:] / s2[:-1])          # per period
    np.testing.assert_allclose(rate, beta, rtol=0.02)


def test_eq15_derivative_stencil(orc):
    """Eq. 15 (L144) is the derivative of the cubic through x0-1..x0+2: exact for p^3, and for
    p^4 off by exactly -2 dp^3 (interpolation error f''''/4! * prod(x0 - x_k), k != 0); the
    mirrored stencil would give +2 dp^3, a transposed one would act along q."""
    N, L, b = 16, 2.0, 0.01
    p = grid_axis(N, -L, L)
    dp = p[1] - p[0]
    q = grid_axis(N, -L, L)
    for deg, err in ((3, 0.0), (4, -2.0 * dp ** 3)):
        f = np.tile(p ** deg, (N, 1)) * (1.0 + 0.1 * q[:, None])
        out = orc.fokker_planck(f, -L, L, b)
        d1 = deg * p ** (deg - 1) + err
        d2_exact_stencil = (np.roll(p, 1) ** deg - 2 * p ** deg + np.roll(p, -1) ** deg) / dp ** 2
        want = (p ** deg + b * (p ** deg + p * d1 + d2_exact_stencil)) * (1.0 + 0.1 * q[:, None])
        np.testing.assert_allclose(out[:, 2:-3], want[:, 2:-3], rtol=1e-12)


# ---------------------------------------------------------------- P7 kick moments
@pytest.mark.parametrize("order", [2, 3, 4])
def test_p7_kick_shifts_mean_exactly(orc, order):
    """Column x is displaced in energy by Delta p_x = -dphi V_x: the mean moves by exactly that,
    the variance is unchanged for order >= 3 and grows by t(1-t) dp^2 for order 2."""
    N, L = 64, 8.0
    dp = 2 * L / (N - 1)
    psi = gauss(N, L, 1.0, 1.0)
    dphi = 0.01
    shifts_cells = np.linspace(-1.7, 2.3, N)               # includes |shift| > 1 cell
    V = -shifts_cells * dp / dphi                           # so that Delta p_x = shifts * dp
    out = orc.kick(psi, dp, dphi, order, V)
    p = grid_axis(N, -L, L)
    for x in (5, N // 2, N - 7):
        col0, col1 = psi[x], out[x]
        mean0, mean1 = np.dot(p, col0) / col0.sum(), np.dot(p, col1) / col1.sum()
        var0 = np.dot(p * p, col0) / col0.sum() - mean0 ** 2
        var1 = np.dot(p * p, col1) / col1.sum() - mean1 ** 2
        assert abs(col1.sum() - col0.sum()) < 1e-12         # P2: charge per column
        assert abs((mean1 - mean0) - shifts_cells[x] * dp) < 1e-10
        t = shifts_cells[x] - math.floor(shifts_cells[x])
        extra = t * (1 - t) * dp * dp if order == 2 else 0.0
        assert abs(var1 - var0 - extra) < 1e-10
    out0 = orc.kick(psi, dp, dphi, order, np.zeros(N))
    assert np.array_equal(out0, psi)                         # zero wake: identity, bit for bit


def test_kick_sign_energy_loss(orc):
    """Re Z > 0 must take energy out of the bunch (reading A6): with a purely resistive
    impedance V = R rho > 0 and every column moves to lower p."""
    N, L = 64, 6.0
    dq = dp = 2 * L / (N - 1)
    psi = gauss(N, L)
    Z = np.full(N + 1, 3.0 + 0j)
    w = orc.wake_function(N, 2 * N, Z)
    rho = orc.project(psi, dp)
    V = orc.wake(w, rho)
    np.testing.assert_allclose(V, 3.0 * rho, atol=1e-13)     # resistive: w = R delta_{d,0}
    out = orc.kick(psi, dp, 0.05, 4, V)
    assert orc.moments(out, -L, L, -L, L)[2] < -1e-3


# ---------------------------------------------------------------- O2 projection (L56)
def test_projection_is_the_marginal_over_p(orc):
    """rho_x = dp * sum_y psi(x, y) ("bunch profile"), pinned without the oracle on
    the other side: (i) a separable psi = f(x) g(y) with asymmetric, different f and g has the
    profile dp * f(x) * sum(g) -- a sum over x instead of y, or dq in place of dp, fails;
    (ii) the marginal of a bivariate Gaussian with sigma_q != sigma_p on a box with dq != dp is
    the 1-D Gaussian exp(-q^2 / 2 sigma_q^2) / (sqrt(2 pi) sigma_q) (the trapezoid sum of a
    Gaussian over +-8 sigma is exact to rounding)."""
    N = 24
    x = np.arange(N, dtype=np.float64)
    f = 1.0 + 0.3 * x + 0.01 * x ** 2                      # not symmetric, not equal to g
    g = np.exp(-0.2 * x) * (2.0 + np.sin(0.7 * x))
    psi = f[:, None] * g[None, :]
    dp, dq = 0.37, 0.91
    rho = orc.project(psi, dp)
    np.testing.assert_allclose(rho, dp * f * g.sum(), rtol=1e-14)
    wrong_axis = dp * g * f.sum()                          # what a transposed sum would give
    assert np.max(np.abs(rho - wrong_axis)) > 0.1 * np.max(np.abs(rho))
    assert np.max(np.abs(rho - dq * f * g.sum())) > 0.1 * np.max(np.abs(rho))
    # (ii) closed-form marginal, non-square box and spacings
    N, sq, sp = 96, 0.8, 1.3
    q = grid_axis(N, -7.0, 6.0)
    p = grid_axis(N, -10.4, 10.4)
    psi = (np.exp(-0.5 * (q[:, None] / sq) ** 2 - 0.5 * (p[None, :] / sp) ** 2) / (TWO_PI * sq * sp))
    rho = orc.project(psi, p[1] - p[0])
    np.testing.assert_allclose(rho, np.exp(-0.5 * (q / sq) ** 2) / (math.sqrt(TWO_PI) * sq), rtol=0, atol=1e-13)


# ---------------------------------------------------------------- wake: Eq. 4 == Eq. 5
def test_wake_matches_library_fft_convolution(orc):
    """Direct convolution with w (Eq. 4) equals Re IDFT(Z . DFT(zero-padded rho)) (Eq. 5,
    L54) evaluated with numpy's real FFT -- a library routine independent of the oracle."""
    wl = get_workload("C1")
    Z = wl.impedance()[0].astype(np.complex128)
    N, Nf = wl.N, wl.Nf
    rng = np.random.default_rng(3)
    rho = np.exp(-0.5 * grid_axis(N, -6, 6) ** 2) * (1 + 0.1 * rng.standard_normal(N))
    V = orc.wake(orc.wake_function(N, Nf, Z), rho)
    V_fft = np.fft.irfft(Z * np.fft.rfft(rho, Nf), Nf)[:N]
    np.testing.assert_allclose(V, V_fft, rtol=0, atol=1e-11 * np.abs(V_fft).max())


def test_wake_delay_impedance_shifts_profile(orc):
    """Z_k = exp(-2 pi i k d0/N_f) is a pure delay: V_x = rho_{x-d0}.  Pins the sign of the
    exponent in Eq. 5 (e^{+ikq}) and the orientation of w[x - x']."""
    N, Nf, d0 = 32, 64, 5
    k = np.arange(Nf // 2 + 1)
    Z = np.exp(-2j * np.pi * k * d0 / Nf)
    Z[-1] = Z[-1].real
    rho = np.zeros(N); rho[7] = 1.0; rho[11] = -2.0
    V = orc.wake(orc.wake_function(N, Nf, Z), rho)
    want = np.zeros(N); want[7 + d0] = 1.0; want[11 + d0] = -2.0
    np.testing.assert_allclose(V, want, atol=1e-13)


# ---------------------------------------------------------------- P8 Parseval
def test_p8_parseval_power_equals_work_done_by_wake(orc):
    """sum_x rho_x V_x dq (space, direct convolution) == P_csr (frequency, Eq. 16-17): the
    radiated power equals the energy-loss rate per radian, -(1/dphi) sum rho_x Delta p_x dq."""
    wl = get_workload("C1")
    Z = wl.impedance()[0].astype(np.complex128)
    psi = wl.psi0()[0].astype(np.float64)
    rho = orc.project(psi, wl.dp)
    V = orc.wake(orc.wake_function(wl.N, wl.Nf, Z), rho)
    P_space = wl.dq * np.dot(rho, V)
    P_freq = orc.csr_power(rho, wl.Nf, wl.dq, Z)
    assert P_freq > 0
    assert abs(P_space - P_freq) < 1e-12 * P_freq


# ---------------------------------------------------------------- P9 free-space closed form
@pytest.mark.parametrize("pad,rtol", [(2, 3e-4), (4, 5e-5), (8, 1e-5), (16, 1e-5)])
def test_p9_free_space_power_closed_form(orc, pad, rtol):
    """Free-space impedance (Eq. 6), unit Gaussian bunch: with Z_k = 4 pi S Zhat(kappa_k),
    P = 2 S int Re Zhat e^{-kappa^2} dkappa = 3^{1/6} Gamma(2/3)^2 S (= 2.20208 S) for pad -> inf;
    the k-sum is a trapezoid rule for a kappa^{1/3} endpoint singularity whose Euler-Maclaurin
    correction is zeta(-1/3) dkappa^{4/3}."""
    import mpmath
    from scipy.special import gamma
    N, L, S = 256, 6.0, 0.5
    dq = 2 * L / (N - 1)
    Z = make_impedance(N, pad, dq, S, None, dtype=np.complex128)
    q = grid_axis(N, -L, L)
    rho = np.exp(-0.5 * q * q) / math.sqrt(TWO_PI)
    P = orc.csr_power(rho, pad * N, dq, Z)
    dkap = TWO_PI / (pad * N * dq)
    zeta = float(mpmath.zeta(mpmath.mpf(-1) / 3))
    want = 3 ** (1 / 6) * gamma(2 / 3) ** 2 * S * (1 + zeta * dkap ** (4 / 3) / (0.5 * gamma(2 / 3)))
    assert abs(P - want) < rtol * want


# ---------------------------------------------------------------- P2/P3 charge per sub-step
def test_p2_charge_conservation_per_substep(orc):
    wl = get_workload("C1")
    psi = wl.psi0()[0].astype(np.float64)
    Z = wl.impedance()[0].astype(np.complex128)
    dphi = TWO_PI / wl.steps_per_period
    cell = wl.dq * wl.dp
    c0 = psi.sum() * cell
    rot = orc.rotate(psi, -6, 6, -6, 6, dphi, 4)
    assert abs(rot.sum() * cell - c0) < 1e-6                 # rotation: corners leak the noise floor
    V = orc.wake(orc.wake_function(wl.N, wl.Nf, Z), orc.project(rot, wl.dp))
    kicked = orc.kick(rot, wl.dp, dphi, 4, V)
    assert abs(kicked.sum() - rot.sum()) * cell < 1e-9       # kick: only edge flux of the noise
    fp = orc.fokker_planck(kicked, -6, 6, wl.beta / wl.steps_per_period)
    assert abs(fp.sum() - kicked.sum()) * cell < 1e-9


def test_full_step_composition_and_renormalisation(orc):
    """vfpo_step = a1..a6 in BASELINE order; C is the pre-renormalisation charge and the
    stored psi integrates to 1."""
    wl = get_workload("C1")
    o = orc.Oracle.from_workload(wl)
    psi = o.psi.copy()
    Z = wl.impedance()[0].astype(np.complex128)
    dphi = TWO_PI / wl.steps_per_period
    d = o.step(1)
    rot = orc.rotate(psi, -6, 6, -6, 6, dphi, 4)
    V = orc.wake(orc.wake_function(wl.N, wl.Nf, Z), orc.project(rot, wl.dp))
    fp = orc.fokker_planck(orc.kick(rot, wl.dp, dphi, 4, V), -6, 6, wl.beta / wl.steps_per_period)
    C = fp.sum() * wl.dq * wl.dp
    assert abs(d[0, 0] - C) < 1e-13          # numpy sums pairwise, the oracle serially
    np.testing.assert_allclose(o.psi, fp / C, rtol=1e-13)
    assert abs(o.psi.sum() * wl.dq * wl.dp - 1.0) < 1e-14
    np.testing.assert_allclose(o.moments6(), np.r_[1.0, d[0, 1:]], rtol=1e-12, atol=1e-14)


# ---------------------------------------------------------------- P13 (soft) Table I / II scale
def test_p13_converged_bunch_length_close_to_one(orc):
    """Table I (L155-164): the converged sigma_z deviates ~1e-4 from the analytic value 1; run
    parameters are not stated, so this is an order-of-magnitude check (< 1e-3, Table II < 1 %)."""
    N, L, spp, beta = 128, 6.0, 250, 0.2
    o = orc.Oracle(N, -L, L, -L, L, spp, beta, 4)
    o.set_psi(gauss(N, L, 1.3, 1.3))
    d = o.step(40 * spp, diag_every=spp)
    assert abs(d[-1, 3] - 1.0) < 1e-3 and abs(d[-1, 4] - 1.0) < 1e-3


# ---------------------------------------------------------------- P14 Manhattan rotation (L136)
def _cov(psi, L):
    """<q>, <p> and the covariance matrix of psi on the box [-L, L]^2, formed here in numpy."""
    N = psi.shape[0]
    q = np.linspace(-L, L, N)
    w = psi / psi.sum()
    mq, mp = (w.sum(1) * q).sum(), (w.sum(0) * q).sum()
    dq, dp = q - mq, q - mp
    return np.array([mq, mp]), np.array([[(w.sum(1) * dq * dq).sum(), (w * np.outer(dq, dp)).sum()],
                                         [(w * np.outer(dq, dp)).sum(), (w.sum(0) * dp * dp).sum()]])


def test_p14_manhattan_moments_follow_the_symplectic_map(orc):
    """Drift q' = q + dphi p, RF kick p' = p - dphi q' (Eq. 1 signs, L25; symplectic split, L136).
    A 1-D Lagrange shift of order >= 3 moves the mean of every line by exactly the shift and keeps
    its variance, so means and covariances of psi follow the linear map M = [[1, dphi],
    [-dphi, 1 - dphi^2]] exactly: m_n = M^n m_0, S_n = M^n S_0 (M^n)^T; det M = 1 (area
    preserved: the emittance det S is invariant)."""
    N, L, spp, n = 128, 6.0, 400, 100
    dphi = TWO_PI / spp
    psi = gauss(N, L, 0.8, 0.6, 0.5, -0.3)          # 7 sigma inside the box: no edge loss
    m0, S0 = _cov(psi, L)
    M = np.array([[1.0, dphi], [-dphi, 1.0 - dphi * dphi]])
    assert abs(np.linalg.det(M) - 1.0) < 1e-15
    o = orc.Oracle(N, -L, L, -L, L, spp, 0.0, 4, 2, None, renormalise=False, manhattan=True)
    o.set_psi(psi)
    o.step(n, diag=False)
    Mn = np.linalg.matrix_power(M, n)
    m, S = _cov(o.psi, L)
    np.testing.assert_allclose(m, Mn @ m0, atol=2e-9)
    np.testing.assert_allclose(S, Mn @ S0 @ Mn.T, atol=2e-8)
    assert abs(np.linalg.det(S) - np.linalg.det(S0)) < 1e-7
    # and it IS a rotation to O(dphi): a quarter period takes (q, p) to (p, -q)
    assert abs(m[0] - m0[1]) < 0.01 and abs(m[1] + m0[0]) < 0.01


@pytest.mark.parametrize("order", [2, 3, 4])
def test_p14_manhattan_substeps_conserve_charge_and_shift_lines(orc, order):
    """Each half is a family of 1-D shifts: charge is conserved to rounding (interior support) and
    the line at p_y (resp. q_x) moves by exactly dphi p_y (resp. -dphi q_x)."""
    N, L = 64, 6.0
    dphi = TWO_PI / 150
    q = np.linspace(-L, L, N)
    psi = gauss(N, L, 0.6, 0.7, 0.4, 0.2)           # > 8 sigma inside the box: no edge loss
    a = orc.drift(psi, -L, L, -L, L, dphi, order)
    b = orc.rf_kick(a, -L, L, -L, L, dphi, order)
    assert abs(a.sum() / psi.sum() - 1.0) < 1e-12 and abs(b.sum() / psi.sum() - 1.0) < 1e-12
    y = 40                                                        # the line p = q[y]
    mean_q = lambda f: (f[:, y] * q).sum() / f[:, y].sum()
    assert abs(mean_q(a) - mean_q(psi) - dphi * q[y]) < 1e-10
    x = 22                                                        # the line q = q[x]
    mean_p = lambda f: (f[x, :] * q).sum() / f[x, :].sum()
    assert abs(mean_p(b) - mean_p(a) + dphi * q[x]) < 1e-10


def test_p14_manhattan_keeps_the_gaussian(orc):
    """L196 / Fig. 5: with Manhattan rotation a sigma = 1 Gaussian stays put (sigma_p within 1 %
    over a period, Table II), here 256^2 at 1000 steps per period without damping."""
    N, L, spp = 256, 6.0, 1000
    o = orc.Oracle(N, -L, L, -L, L, spp, 0.0, 4, 2, None, renormalise=False, manhattan=True)
    o.set_psi(gauss(N, L))
    d = o.step(spp, diag_every=100)
    rows = d[~np.isnan(d[:, 0])]
    assert np.all(np.abs(rows[:, 3] - 1.0) < 0.01) and np.all(np.abs(rows[:, 4] - 1.0) < 0.01)
    assert abs(rows[-1, 0] - 1.0) < 1e-7          # only the 6-sigma tails leave through the box edge


# ---------------------------------------------------------------- P15 clamped interpolation (Eq. 14)
@pytest.mark.parametrize("order", [3, 4])
def test_p15_clamped_interpolation_has_no_overshoot(orc, order):
    """L110-116: "Interpolation using these polynomials sometimes overshoots the values of the
    neighboring grid cells ... To avoid overshooting, one has to use clamped ... interpolation"
    (Eq. 14, read as clamp to the interval of the bracketing nodes, A9).  On a step
    the unclamped quadratic / cubic shift over- and undershoots; the clamped one stays inside
    [min, max] of the data, creates no new extremum, and equals the unclamped one wherever that
    already lies between its two bracketing nodes."""
    N, L = 32, 6.0
    dp = 2 * L / (N - 1)
    psi = np.zeros((N, N))
    psi[:, 10:20] = 1.0                                           # a box along p in every column
    V = np.full(N, -0.37 * dp / (TWO_PI / 100))                   # shift of +0.37 cell... (sign per A6)
    free = orc.kick(psi, dp, TWO_PI / 100, order, V)
    clamped = orc.kick(psi, dp, TWO_PI / 100, order, V, clamp=True)
    assert free.max() > 1.0 + 1e-3 and free.min() < -1e-3         # the artifact the paper describes
    assert clamped.max() <= 1.0 and clamped.min() >= 0.0
    row_f, row_c = free[5], clamped[5]
    inside = (row_f >= 0.0) & (row_f <= 1.0)
    # away from the two edges the interpolant is exact (constant data) and untouched
    np.testing.assert_allclose(row_c[:8], 0.0, atol=0)
    np.testing.assert_allclose(row_c[13:17], 1.0, atol=1e-15)
    assert np.count_nonzero(~inside) >= 2
    # linear interpolation never leaves the bracket: clamping is the identity
    lin = orc.kick(psi, dp, TWO_PI / 100, 2, V)
    np.testing.assert_array_equal(lin, orc.kick(psi, dp, TWO_PI / 100, 2, V, clamp=True))


def test_p15_clamp_is_identity_on_smooth_data_and_bounds_the_rotation(orc):
    """On a smooth Gaussian the cubic interpolant lies between its bracketing nodes almost
    everywhere, so clamped and free rotation agree to the interpolation error; on a 2-D box the
    clamped rotation stays within [0, 1] while the free one does not."""
    N, L = 64, 6.0
    g = gauss(N, L)
    dphi = TWO_PI / 500
    a = orc.rotate(g, -L, L, -L, L, dphi, 4)
    b = orc.rotate(g, -L, L, -L, L, dphi, 4, clamp=True)
    assert np.max(np.abs(a - b)) < 2e-4 * g.max()
    box = np.zeros((N, N))
    box[20:40, 24:44] = 1.0
    a = orc.rotate(box, -L, L, -L, L, 25 * dphi, 4)
    b = orc.rotate(box, -L, L, -L, L, 25 * dphi, 4, clamp=True)
    assert a.max() > 1.01 and a.min() < -0.01
    assert b.max() <= 1.0 and b.min() >= 0.0
    # Manhattan halves: same statement line by line
    for f in (orc.drift, orc.rf_kick):
        c = f(box, -L, L, -L, L, 25 * dphi, 4, clamp=True)
        assert c.max() <= 1.0 and c.min() >= 0.0


# ---------------------------------------------------------------- the whole step, written out from the paper
def _lagrange_bf(order, t):
    """Eq. 13 (L107) literally: l_k(t) = prod_{m != k} (t - o_m) / (o_k - o_m), nodes o_k = k - floor((order-1)/2)."""
    o = [k - (order - 1) // 2 for k in range(order)]
    w = []
    for k in range(order):
        v = 1.0
        for m in range(order):
            if m != k:
                v *= (t - o[m]) / (o[k] - o[m])
        w.append(v)
    return o, w


def _step_bruteforce(psi, box, spp, beta, order, pad, Z, manhattan=False, clamp=False):
    """One Warnock-Ellison split step (L29-40) with explicit Python loops over cells and taps, straight from the
    paper's formulas and the readings A1-A14 of DESIGN.md -- no call into oracle/: rotation about the origin by
    the angle 2 pi / spp (Eq. 1: q_s = c q - s p, p_s = s q + c p, tensor-product Lagrange interpolation, psi = 0
    outside the grid), profile, wake through numpy's FFT (Eq. 5), kick by -dphi V, Fokker-Planck (Eq. 15 and the
    three-point second difference), charge, renormalisation, moments and CSR power (Eq. 16-17) of the end-of-step
    density.  manhattan: the rotation is the drift psi_A(q, p) = psi(q - dphi p, p) followed by the RF kick
    psi_B(q, p) = psi_A(q, p + dphi q), two 1-D interpolations (L136, reading A15).  clamp: every interpolated value
    is limited to the interval of the nodes that bracket its source point (Eq. 14, reading A9)."""
    N = psi.shape[0]
    qmin, qmax, pmin, pmax = box
    dq, dp = (qmax - qmin) / (N - 1), (pmax - pmin) / (N - 1)
    dphi = TWO_PI / spp
    c, s = math.cos(dphi), math.sin(dphi)

    def at(a, x, y):
        return a[x, y] if 0 <= x < N and 0 <= y < N else 0.0

    def interp1(a, x, ysrc, along_q):
        """1-D Lagrange interpolation of row / column through (x, .) at the fractional index ysrc"""
        m = math.floor(ysrc)
        o, w = _lagrange_bf(order, ysrc - m)
        get = (lambda k: at(a, m + k, x)) if along_q else (lambda k: at(a, x, m + k))
        v = sum(w[j] * get(o[j]) for j in range(order))
        if clamp:
            v = min(max(v, min(get(0), get(1))), max(get(0), get(1)))
        return v

    rot = np.zeros((N, N))
    if manhattan:
        dr = np.zeros((N, N))
        for x in range(N):
            for y in range(N):
                dr[x, y] = interp1(psi, y, x - dphi * (pmin + y * dp) / dq, True)
        for x in range(N):
            for y in range(N):
                rot[x, y] = interp1(dr, x, y + dphi * (qmin + x * dq) / dp, False)
    else:
        for x in range(N):
            for y in range(N):
                q, p = qmin + x * dq, pmin + y * dp
                xs, ys = (c * q - s * p - qmin) / dq, (s * q + c * p - pmin) / dp
                mx, my = math.floor(xs), math.floor(ys)
                ox, wx = _lagrange_bf(order, xs - mx)
                oy, wy = _lagrange_bf(order, ys - my)
                v = sum(wx[i] * wy[j] * at(psi, mx + ox[i], my + oy[j]) for i in range(order) for j in range(order))
                if clamp:
                    nb = [at(psi, mx + i, my + j) for i in (0, 1) for j in (0, 1)]
                    v = min(max(v, min(nb)), max(nb))
                rot[x, y] = v
    rho = dp * rot.sum(axis=1)
    Nf = pad * N
    V = np.fft.irfft(Z * np.fft.rfft(rho, Nf), Nf)[:N] if Z is not None else np.zeros(N)
    kick = np.zeros((N, N))
    for x in range(N):
        for y in range(N):
            kick[x, y] = interp1(rot, x, y + dphi * V[x] / dp, False)      # delta p = -dphi V: source = y + dphi V / dp
    b = beta / spp
    fp = np.zeros((N, N))
    for x in range(N):
        for y in range(N):
            f = [at(kick, x, y + k) for k in (-1, 0, 1, 2)]
            d1 = (-2 * f[0] - 3 * f[1] + 6 * f[2] - f[3]) / (6 * dp)
            d2 = (f[0] - 2 * f[1] + f[2]) / dp ** 2
            fp[x, y] = f[1] + b * (f[1] + (pmin + y * dp) * d1 + d2)
    C = fp.sum() * dq * dp
    out = fp / C
    qa, pa = qmin + dq * np.arange(N), pmin + dp * np.arange(N)
    tot = out.sum()
    mq, mp = (out.sum(axis=1) * qa).sum() / tot, (out.sum(axis=0) * pa).sum() / tot
    sq = math.sqrt((out.sum(axis=1) * qa ** 2).sum() / tot - mq ** 2)
    sp = math.sqrt((out.sum(axis=0) * pa ** 2).sum() / tot - mp ** 2)
    P = 0.0
    if Z is not None:
        R = np.fft.rfft(dp * out.sum(axis=1), Nf)
        wgt = np.full(Nf // 2 + 1, 2.0)
        wgt[0] = wgt[-1] = 1.0
        P = dq / Nf * float((wgt * Z.real * np.abs(R) ** 2).sum())
    return out, np.array([C, mq, mp, sq, sp, P])


@pytest.mark.parametrize("manhattan,clamp", [(False, False), (True, False), (False, True), (True, True)])
@pytest.mark.parametrize("order", [2, 3, 4])
def test_whole_step_against_loops_written_from_the_paper(orc, order, manhattan, clamp):
    """Pins the composition of vfpo_step -- sub-step order a1..a6 (A14), kick sign (A6), which density the
    diagnostics refer to (A10), renormalisation -- and every sub-step once more, against an implementation that
    shares nothing with oracle/: 16 x 16 cells, asymmetric box, off-centre bunch, a step large enough that the
    stencil floors change across the grid, an impedance strong enough that the kick moves rows by more than a cell;
    three consecutive steps; standard and Manhattan rotation (A15), free and clamped interpolation (A9)."""
    N, spp, beta, pad = 16, 40, 0.3, 2
    box = (-4.0, 5.0, -4.5, 3.5)
    rng = np.random.default_rng(7)
    psi = make_psi0(N, *box, 1.1, 0.8, 0.0, 0, q0=0.4, p0=-0.3).astype(np.float64)
    psi += 1e-3 * psi.max() * rng.random((N, N))
    dq, dp = 9.0 / (N - 1), 8.0 / (N - 1)
    psi /= psi.sum() * dq * dp
    k = np.arange(pad * N // 2 + 1)
    Z = (18.0 + 8.0j * np.sin(0.37 * k)) * np.exp(-0.02 * k)
    Z[0] = 0.0
    Z[-1] = Z[-1].real
    o = orc.Oracle(N, *box, spp, beta, order, pad, Z.astype(np.complex128), manhattan=manhattan, clamp=clamp)
    o.set_psi(psi)
    ref = psi.copy()
    moved = 0.0
    for step in range(3):
        d = o.step(1)
        ref, dref = _step_bruteforce(ref, box, spp, beta, order, pad, Z, manhattan, clamp)
        np.testing.assert_allclose(o.psi, ref, rtol=0, atol=1e-12 * ref.max(), err_msg=f"order {order}, step {step}")
        np.testing.assert_allclose(d[0], dref, rtol=1e-10, atol=1e-12)
        moved = max(moved, np.abs(o.wake()).max() * TWO_PI / spp / dp)
    assert moved > 1.0            # the kick did move some row by more than a cell
