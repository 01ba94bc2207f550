"""Input generators (workloads/): impedance pins P10 and the psi0 recipe (reading A12)."""
import numpy as np
import pytest

from workloads import (CONFIGS, get_workload, kappa_grid, make_impedance, make_psi0,
                       uniform_noise, zhat_free_space, zhat_parallel_plates)


def test_p10_shielded_converges_to_free_space():
    """'For high frequencies both impedances converge' (Fig. 1)."""
    kap = np.array([30.0, 100.0, 300.0])
    ratio = zhat_parallel_plates(kap, 1.0) / zhat_free_space(kap)
    assert np.max(np.abs(ratio - 1.0)) < 1e-8


def test_p10_shielding_suppresses_low_frequencies():
    """'For f -> 0 both impedances approach Z = 0' (L65): below the shielding cutoff the real
    (radiating) part vanishes exponentially."""
    z = zhat_parallel_plates(np.array([0.3]), 1.0)[0]
    assert abs(z.real) < 1e-10 and z.imag < 0
    assert make_impedance(256, 2, 12 / 255, 0.5, 1.0)[0] == 0


def test_p10_against_mpmath():
    """Eq. 7-8 evaluated term by term with 40-digit Airy functions (mpmath), p < 3000."""
    import mpmath as mp
    mp.mp.dps = 40
    Pi = mp.mpf(1)
    for kappa in (0.26077673, 1.3, 5.2):
        k = mp.mpf(kappa)
        tot = mp.mpc(0)
        for p in range(3000):
            u = mp.pi ** 2 * (2 * p + 1) ** 2 * mp.mpf(2) ** (mp.mpf(-8) / 3) * (Pi / k) ** (mp.mpf(4) / 3)
            if u < 200:
                ai, aip = mp.airyai(u), mp.airyai(u, derivative=1)
                bi, bip = mp.airybi(u), mp.airybi(u, derivative=1)
                tot += aip * (aip - 1j * bip) + u * ai * (ai - 1j * bi)
            else:      # two-term asymptote of -(Ai'Bi' + u Ai Bi), good to 1e-10 relative here
                tot += -1j * (3 / (16 * mp.pi * u ** mp.mpf(2.5)))
        want = complex(2 * mp.pi ** 2 * mp.mpf(2) ** (mp.mpf(1) / 3) * k ** (-mp.mpf(1) / 3) * tot)
        got = zhat_parallel_plates(np.array([kappa]), 1.0)[0]
        assert abs(got - want) < 2e-8 * abs(want)


def test_p10_golden_samples_c1():
    """tests/golden/impedance_c1.txt: Z_k = 4 pi S Zhat_pp(kappa_k), Pi=1, S=0.5, N_f=512,
    dq=12/255, from a 40-digit mpmath evaluation (pin P10)."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "impedance_c1.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    Z = make_impedance(256, 2, 12 / 255, 0.5, 1.0, dtype=np.complex128)
    assert abs(kappa_grid(256, 2, 12 / 255)[1] - 0.26077673) < 1e-8
    for k, re, im in rows:
        want = complex(float(re), float(im))
        assert abs(Z[int(k)] - want) < 2e-8 * max(abs(want), 1e-3)


def test_impedance_array_contract():
    wl = get_workload("C3")
    Z = wl.impedance([0, 255])
    assert Z.shape == (2, wl.Nf // 2 + 1) and Z.dtype == np.complex64
    assert np.all(Z[:, 0] == 0) and np.all(Z[:, -1].imag == 0)
    np.testing.assert_allclose(Z[1] / wl.S_csr[255], Z[0] / wl.S_csr[0], rtol=1e-6)
    assert get_workload("C0").impedance() is None


def test_psi0_recipe():
    wl = get_workload("C1")
    psi = wl.psi0()[0]
    assert psi.dtype == np.float32 and psi.shape == (256, 256)
    assert abs(psi.astype(np.float64).sum() * wl.dq * wl.dp - 1.0) < 1e-6
    assert psi.min() >= 0                                   # noise is absolute, non-negative
    corner = psi[:8, :8].astype(np.float64)                 # Gaussian ~1e-16 there: noise only
    assert 0.2e-6 < corner.mean() < 0.8e-6
    assert np.array_equal(psi, wl.psi0()[0])                # reproducible
    assert not np.array_equal(get_workload("C3").psi0([0])[0], get_workload("C3").psi0([1])[0])


def test_uniform_noise_statistics():
    u = uniform_noise(1 << 16, 7)
    assert u.min() >= 0 and u.max() < 1
    assert abs(u.mean() - 0.5) < 5e-3 and abs(u.var() - 1 / 12) < 2e-3
    assert abs(np.corrcoef(u[:-1], u[1:])[0, 1]) < 0.02


def test_config_table():
    assert [CONFIGS[c].N for c in ("C0", "C1", "C2", "C3", "C4")] == [64, 256, 512, 256, 2048]
    assert CONFIGS["C3"].members == 256 and abs(CONFIGS["C3"].S_csr[-1] - 1.0) < 1e-12
    assert CONFIGS["C1"].total_steps == 80000 and CONFIGS["C4"].Nf == 4096
