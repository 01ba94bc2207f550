"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded fp32 inputs.  Tolerances are BASELINE.json's north_star:
  max|psi_gpu - psi_ref| <= 1e-5 * max psi after 1 step, <= 1e-3 * max psi after 1000 steps;
  moments and CSR power within 1e-4 relative (means, which are ~0: 1e-4 absolute in units of
  sigma)."""
import numpy as np
import pytest

from workloads import get_workload, make_impedance, make_psi0
from workloads.configs import Workload

pytestmark = pytest.mark.gpu

TOL_1 = 1e-5
TOL_1000 = 1e-3
TOL_MOM = 1e-4


def assert_psi(sim_psi, ref_psi, tol, what=""):
    ref = np.asarray(ref_psi, dtype=np.float64)
    err = np.max(np.abs(sim_psi.astype(np.float64) - ref)) / ref.max()
    assert err <= tol, f"{what}: max|dpsi|/max psi = {err:.3e} > {tol:.1e}"
    return err


def test_maximum_grid_4096(vfps, orc):
    """The largest grid the library accepts (N * pad = 8192 is the limit of the wake FFT's shared
    memory): 4096^2, asymmetric box, cubic interpolation, parallel-plates wake.  AUTO (the grid engine)
    for 1 and 4 more steps, then the stream engine with the FFT wake at its maximum
    length for 2 more, every cell against the oracle."""
    N, spp = 4096, 16000
    box = (-5.0, 7.0, -6.5, 5.5)
    Z = make_impedance(N, 2, 12.0 / (N - 1), 0.4, 0.8)[None, :]
    psi0 = make_psi0(N, *box, 1.1, 0.9, 0.0, 5, q0=0.4, p0=-0.3)[None]
    sim = vfps.Simulation(N, *box, spp, 2e-3, 4, 2, 1, Z=Z)
    sim.set_psi_host(psi0)
    o = orc.Oracle(N, *box, spp, 2e-3, 4, 2, Z[0])
    o.set_psi(psi0[0])
    # a stripe of 4096 / 148 = 28 rows of 4096 cells does not fit the shared memory of an SM: the TMA-staged
    # kernel is refused and AUTO takes the first grid kernel (psi through L2)
    assert sim.engine_name == "grid" and sim.grid_kernel == 1
    with pytest.raises(vfps.VfpsError) as e:
        sim.set_grid_kernel(2)
    assert e.value.code == -5
    d = sim.step_host(1)
    dr = o.step(1)
    assert_psi(sim.get_psi_host()[0], o.psi, TOL_1, "4096^2, 1 step")
    assert_diag(d[0, 0], dr[0])
    d = sim.step_host(4)
    dr = o.step(4)
    assert_psi(sim.get_psi_host()[0], o.psi, 2e-5, "4096^2, 5 steps")
    assert_diag(d[3, 0], dr[3])
    sim.set_engine(vfps.ENGINE_STREAM)
    sim.set_wake_mode(vfps.WAKE_FFT)
    d = sim.step_host(2)
    dr = o.step(2)
    assert sim.wake_name == "fft"
    assert_psi(sim.get_psi_host()[0], o.psi, 3e-5, "4096^2, 7 steps, FFT wake of length 8192")
    assert_diag(d[1, 0], dr[1])
    sim.close()
    with pytest.raises(vfps.VfpsError) as e:
        vfps.Simulation(8192, *box, spp, 2e-3, 4, 2, 1)
    assert e.value.code == -5


@pytest.mark.parametrize("engine", ["stream", "cluster", "cluster3", "grid", "grid2"])
@pytest.mark.parametrize("order", [3, 4])
def test_single_cell_density_and_zero_steps(vfps, orc, engine, order):
    """Degenerate inputs: all of the charge in ONE cell (after a step the density is the 4 x 4 / 3 x 3
    stencil of Lagrange weights around the image of that cell, positive and negative lobes included, then
    the kick of a one-row profile) and a vfps_step of zero steps (no change, nothing written)."""
    N, spp = 256, 4000
    Z = make_impedance(N, 2, 12.0 / (N - 1), 0.05, 0.8)[None, :]
    psi0 = np.zeros((1, N, N), dtype=np.float32)
    psi0[0, 171, 90] = 1.0 / (12.0 / (N - 1)) ** 2
    sim = vfps.Simulation(N, -6, 6, -6, 6, spp, 1e-3, order, 2, 1, Z=Z)
    if engine in ("cluster", "cluster3"):
        sim.set_cluster_kernel(1 if engine == "cluster" else 3)
    if engine in ("grid", "grid2"):
        sim.set_grid_kernel(1 if engine == "grid" else 2)
    sim.set_engine(_engine_id(vfps, engine))
    sim.set_psi_host(psi0)
    d0 = sim.step_host(0)
    assert d0.shape[0] == 0
    np.testing.assert_array_equal(sim.get_psi_host(), psi0)
    o = orc.Oracle(N, -6, 6, -6, 6, spp, 1e-3, order, 2, Z[0])
    o.set_psi(psi0[0])
    d = sim.step_host(1)
    dr = o.step(1)
    psi = sim.get_psi_host()[0]
    assert_psi(psi, o.psi, TOL_1, f"single cell, {engine}, order {order}, 1 step")
    assert (psi != 0).sum() <= 6 * (order + 3) and psi.min() < 0          # the stencil and nothing else
    d = sim.step_host(20)
    dr = o.step(20)
    assert_psi(sim.get_psi_host()[0], o.psi, 5e-5, f"single cell, {engine}, order {order}, 21 steps")
    # sigma of a few-cell density is a difference of nearly equal sums: absolute tolerance in cells
    assert abs(d[19, 0, 0] - dr[19][0]) < 1e-4 and abs(d[19, 0, 1] - dr[19][1]) < 1e-3 * 12.0 / (N - 1)
    sim.close()


def edge_flux_tol(C):
    """P_csr of a step is formed from the profile the wake acts on, renormalised by the step's
    charge: P = dq sum rho_x V_x / C^2 (include/vfps.h).  Kick and Fokker-Planck move charge along p
    only, so the end-of-step profile differs from that one exactly by the charge that crosses the
    p-edges of the box during the step (C: the step's pre-renormalisation charge of a density that
    entered it normalised).  P is quadratic in the profile: depending on where the lost charge sat,
    the end-of-step value lies between P and P / C^2 -- bound 1.5 (1 / C^2 - 1), i.e. 3 |1 - C| for
    small losses."""
    C = float(C)
    return TOL_MOM + 1.5 * abs(1.0 / (C * C) - 1.0)


def assert_diag(got, want, has_wake=True, tol_q=TOL_MOM, tol_p=None):
    """tol_q: tolerance of the numbers that may be taken from the post-rotation profile (P_csr; in
    the stream engine also <q>, sigma_q); equal to TOL_MOM unless the bunch overflows the box
    (edge flux).  tol_p overrides it for P_csr alone (edge_flux_tol)."""
    tol_p = tol_q if tol_p is None else tol_p
    got = np.array(got, dtype=np.float64)
    want = np.array(want, dtype=np.float64)
    # a negative variance (quadratic/cubic overshoot on a grid too coarse for the bunch) has no
    # sigma: the oracle reports NaN, the library 0 -- both mean "undefined"
    for k in (3, 4):
        if np.isnan(want[k]):
            assert got[k] == 0.0, ("undefined sigma", k, got[k])
            got[k] = want[k] = 1.0
    assert abs(got[0] - want[0]) <= TOL_MOM * abs(want[0]), ("C", got[0], want[0])
    assert abs(got[1] - want[1]) <= tol_q * want[3], ("<q>", got[1], want[1])
    assert abs(got[2] - want[2]) <= TOL_MOM * want[4], ("<p>", got[2], want[2])
    assert abs(got[3] - want[3]) <= tol_q * want[3], ("sigma_q", got[3], want[3])
    assert abs(got[4] - want[4]) <= TOL_MOM * want[4], ("sigma_p", got[4], want[4])
    if has_wake:
        assert abs(got[5] - want[5]) <= tol_p * abs(want[5]), ("P_csr", got[5], want[5])
    else:
        assert got[5] == 0.0


def run_pair(vfps, orc, wl, nsteps, members=None, engine=None, wake=None, diag_every=1, cluster_kernel=None):
    idx = list(range(wl.members) if members is None else members)
    sim = vfps.Simulation.from_workload(wl, idx)
    if cluster_kernel is not None:
        sim.set_cluster_kernel(cluster_kernel)
    if engine is not None:
        sim.set_engine(engine)
    if wake is not None:
        sim.set_wake_mode(wake)
    d_gpu = sim.step_host(nsteps)
    psi_gpu = sim.get_psi_host()
    refs, d_ref = [], []
    for m in idx:
        o = orc.Oracle.from_workload(wl, m)
        d_ref.append(o.step(nsteps, diag_every=diag_every))
        refs.append(o)
    return sim, psi_gpu, d_gpu, refs, d_ref


# ---------------------------------------------------------------- the BASELINE configs
def test_c0_one_step_and_1000_steps(vfps, orc):
    wl = get_workload("C0")
    sim, psi, d, refs, dr = run_pair(vfps, orc, wl, 1)
    assert_psi(psi[0], refs[0].psi, TOL_1, "C0 1 step")
    assert_diag(d[0, 0], dr[0][0], has_wake=False)
    sim.close()
    sim, psi, d, refs, dr = run_pair(vfps, orc, wl, 1000)
    assert_psi(psi[0], refs[0].psi, TOL_1000, "C0 1000 steps")
    for i in (0, 499, 999):
        assert_diag(d[i, 0], dr[0][i], has_wake=False)
    # charge conservation and the stationarity statement for C0 (bilinear: predicted diffusion)
    assert np.all(np.abs(d[:, 0, 0] - 1.0) < 1e-4)
    sim.close()


def test_c1_one_step(vfps, orc):
    wl = get_workload("C1")
    sim, psi, d, refs, dr = run_pair(vfps, orc, wl, 1)
    err = assert_psi(psi[0], refs[0].psi, TOL_1, "C1 1 step")
    assert_diag(d[0, 0], dr[0][0])
    print(f"C1 1 step err {err:.2e}")
    sim.close()


def test_c1_1000_steps(vfps, orc):
    wl = get_workload("C1")
    sim, psi, d, refs, dr = run_pair(vfps, orc, wl, 1000, diag_every=100)
    err = assert_psi(psi[0], refs[0].psi, TOL_1000, "C1 1000 steps")
    for i in (99, 499, 999):
        assert_diag(d[i, 0], dr[0][i])
    print(f"C1 1000 steps err {err:.2e}")
    sim.close()


def test_c2_one_step_and_1000_steps(vfps, orc):
    wl = get_workload("C2")
    for S in (0.2, 1.0):
        w = wl.with_(S_csr=(S,))
        sim, psi, d, refs, dr = run_pair(vfps, orc, w, 1)
        assert_psi(psi[0], refs[0].psi, TOL_1, f"C2 S={S} 1 step")
        assert_diag(d[0, 0], dr[0][0])
        sim.close()
    sim, psi, d, refs, dr = run_pair(vfps, orc, wl.with_(S_csr=(0.6,)), 1000, diag_every=100)
    assert_psi(psi[0], refs[0].psi, TOL_1000, "C2 1000 steps")
    for i in (99, 499, 999):
        assert_diag(d[i, 0], dr[0][i])
    sim.close()


def test_c3_batched_members(vfps, orc):
    """Batched scan: a slice of C3's members in one handle, each with its own Z and noise."""
    wl = get_workload("C3")
    idx = [0, 37, 128, 255]
    sim, psi, d, refs, dr = run_pair(vfps, orc, wl, 50, members=idx, diag_every=10)
    for i, m in enumerate(idx):
        assert_psi(psi[i], refs[i].psi, 1e-4, f"C3 member {m} 50 steps")
        assert_diag(d[49, i], dr[i][49])
    assert not np.allclose(d[49, 0, 5], d[49, 3, 5])        # members really differ
    sim.close()


def test_c4_one_step_and_1000_steps(vfps, orc):
    wl = get_workload("C4")
    sim, psi, d, refs, dr = run_pair(vfps, orc, wl, 1)
    assert sim.engine_name == "grid" and sim.grid_kernel == 2         # what AUTO picks, what bench.py times
    assert_psi(psi[0], refs[0].psi, TOL_1, "C4 1 step")
    assert_diag(d[0, 0], dr[0][0])
    sim.close()
    sim, psi, d, refs, dr = run_pair(vfps, orc, wl, 1000, diag_every=100)
    assert_psi(psi[0], refs[0].psi, TOL_1000, "C4 1000 steps")
    for i in (99, 499, 999):
        assert_diag(d[i, 0], dr[0][i])
    sim.close()


# ---------------------------------------------------------------- the paper's Table III
@pytest.mark.parametrize("order", [4, 3])
def test_t3_table3_one_step_and_1000_steps(vfps, orc, order):
    """PAPER.md L202-229, Table III: 256^2, 4000 steps per T_s, free-space CSR, xi = 0.516 (read as
    S_csr, reading A16), damping time 200 T_s; cubic as in the table and quadratic as in the text's
    second run.  Cluster engine (what AUTO picks), north_star's two bars."""
    wl = get_workload("T3").with_(interp_order=order)
    sim, psi, d, refs, dr = run_pair(vfps, orc, wl, 1)
    assert sim.engine_name == "cluster"
    assert_psi(psi[0], refs[0].psi, TOL_1, f"T3 order {order} 1 step")
    assert_diag(d[0, 0], dr[0][0])
    sim.close()
    sim, psi, d, refs, dr = run_pair(vfps, orc, wl, 1000, diag_every=100)
    assert_psi(psi[0], refs[0].psi, TOL_1000, f"T3 order {order} 1000 steps")
    for i in (99, 499, 999):
        assert_diag(d[i, 0], dr[0][i])
    sim.close()


def test_t3_quadratic_interpolation_ripples(vfps):
    """The qualitative statement of L212-229 / Fig. 6-7: with quadratic interpolation the run
    develops non-physical structures "with a period length of two grid cells" in the bunch profile,
    with cubic interpolation it does not.  Measure of the two-cell content of a profile: its
    Nyquist component |sum_x (-1)^x rho_x| relative to its charge.  Over three synchrotron periods
    (the ripples of Fig. 7 appear around T = 1 T_s) the largest two-cell content seen with
    quadratic interpolation must exceed that seen with cubic interpolation by two orders of
    magnitude, and the cubic run must stay calm (sigma_delta within a few per cent of 1: L208-210)."""
    wl = get_workload("T3")
    sign = np.where(np.arange(wl.N) % 2 == 0, 1.0, -1.0)
    content = {}
    for order in (4, 3):
        sim = vfps.Simulation.from_workload(wl.with_(interp_order=order))
        worst = 0.0
        for _ in range(int(3 * wl.steps_per_period / 250)):
            d = sim.step_host(250)
            rho = sim.get_profile_host()[0].astype(np.float64)
            worst = max(worst, abs(np.dot(sign, rho)) / rho.sum())
        content[order] = worst
        if order == 4:
            # "a relatively calm state with just little oscillation" (L208); the level itself depends on
            # the xi <-> S_csr reading (A16) and on the Gaussian start, so only calmness is asserted
            assert 0.85 < d[-1, 0, 4] < 1.15, ("energy spread of the cubic run", d[-1, 0, 4])
        assert np.all(np.isfinite(d))
        sim.close()
    print("two-cell content of the profile: cubic %.2e quadratic %.2e" % (content[4], content[3]))
    assert content[3] > 100.0 * content[4], content


# ---------------------------------------------------------------- full-size runs in bench.py's configuration
# (engine AUTO, one vfps_step call per synchrotron period with the diagnostics of every step).
# Above threshold the end state is chaotic (parity unpinned beyond 1000
# steps), so the whole-length runs are checked through what holds at any size: the renormalised
# charge, finite and bounded moments, P_csr = energy loss > 0 for the resistive CSR impedance,
# no overshoot beyond the interpolation's; and the full C3 batch against the oracle on sampled
# members.
def _invariants(d, has_wake=True, sig_lo=0.7, sig_hi=2.0):
    d = np.asarray(d, dtype=np.float64)
    assert np.all(np.isfinite(d)), "non-finite diagnostics"
    assert np.all(np.abs(d[..., 0] - 1.0) < 2e-4), ("charge", d[..., 0].min(), d[..., 0].max())
    assert np.all((d[..., 3] > sig_lo) & (d[..., 3] < sig_hi)), ("sigma_q", d[..., 3].min(), d[..., 3].max())
    assert np.all((d[..., 4] > sig_lo) & (d[..., 4] < sig_hi)), ("sigma_p", d[..., 4].min(), d[..., 4].max())
    # (the CSR energy loss shifts the centroid by a fraction of sigma -- the synchronous-phase shift)
    assert np.all(np.abs(d[..., 1]) < 1.5) and np.all(np.abs(d[..., 2]) < 1.5), \
        ("centroid", np.abs(d[..., 1]).max(), np.abs(d[..., 2]).max())
    if has_wake:
        assert np.all(d[..., 5] > 0.0), "CSR power must be an energy loss"


@pytest.mark.parametrize("name,periods", [("C1", 20), ("C2", 5), ("C4", 2)])
def test_full_size_runs_invariants(vfps, name, periods):
    wl = get_workload(name)
    sim = vfps.Simulation.from_workload(wl)
    psi0 = sim.get_psi_host()[0].astype(np.float64)
    for _ in range(periods):
        d = sim.step_host(wl.steps_per_period)
        _invariants(d)
    psi = sim.get_psi_host()[0].astype(np.float64)
    dq = (wl.q_max - wl.q_min) / (wl.N - 1)
    dp = (wl.p_max - wl.p_min) / (wl.N - 1)
    assert abs(psi.sum() * dq * dp - 1.0) < 1e-5                    # get_psi returns the renormalised density
    # cubic interpolation of the micro-structures above threshold undershoots zero a little (the
    # artifact the paper discusses, L212-229): observed -6e-3 max psi at C1 after 20 periods
    assert psi.min() > -2e-2 * psi.max()
    assert 0.5 * psi0.max() < psi.max() < 2.0 * psi0.max()
    assert sim.step_count() == periods * wl.steps_per_period
    sim.close()


def test_full_c3_batch_all_members(vfps, orc):
    """All 256 members in one handle (the launch configuration bench.py times for C3): sampled
    members element by element against the oracle after 1 step and after 1000 steps (north_star's
    two bars), every member through the invariants over one synchrotron period; P_csr grows
    monotonically with S_csr across members."""
    wl = get_workload("C3")
    sim = vfps.Simulation.from_workload(wl)
    sample = (0, 101, 255)
    orcs = [orc.Oracle.from_workload(wl, m) for m in sample]
    d = sim.step_host(1)
    psi = sim.get_psi_host()
    for o, m in zip(orcs, sample):
        dr = o.step(1)
        assert_psi(psi[m], o.psi, TOL_1, f"full C3 batch, member {m}, 1 step")
        assert_diag(d[0, m], dr[0])
    d = sim.step_host(999)
    psi = sim.get_psi_host()
    for o, m in zip(orcs, sample):
        dr = o.step(999, diag_every=100)
        assert_psi(psi[m], o.psi, TOL_1000, f"full C3 batch, member {m}, 1000 steps")
        for i in (99, 499, 998):
            assert_diag(d[i, m], dr[i])
    d = sim.step_host(wl.steps_per_period - 1000)
    _invariants(d)
    assert np.all(np.diff(d[-1, :, 5]) > 0.0)
    sim.close()


# ---------------------------------------------------------------- small / ragged / degenerate
@pytest.mark.parametrize("order", [2, 3, 4])
@pytest.mark.parametrize("N", [8, 32, 128])
def test_orders_and_small_grids(vfps, orc, order, N):
    """Asymmetric box, off-centre mismatched bunch, free-space wake: several tiles and partial
    tiles (N < tile), all three interpolation orders."""
    wl = Workload(f"t{N}", N, -5.0, 7.0, -6.5, 5.5, 300, 2e-3, order, pad=4, S_csr=(0.4,), seeds=(9,),
                  noise=1e-5, sigma_q=1.2, sigma_p=0.8)
    Z = make_impedance(N, 4, wl.dq, 0.4, None)[None, :]
    psi0 = make_psi0(N, -5.0, 7.0, -6.5, 5.5, 1.2, 0.8, 1e-5, 9, q0=0.5, p0=-0.4)[None]
    sim = vfps.Simulation(N, -5.0, 7.0, -6.5, 5.5, 300, 2e-3, order, 4, 1, Z=Z)
    sim.set_psi_host(psi0)
    o = orc.Oracle(N, -5.0, 7.0, -6.5, 5.5, 300, 2e-3, order, 4, Z[0])
    o.set_psi(psi0[0])
    # N = 8: the bunch overflows the 8-point box (2e-3 of the charge leaves per step), so the
    # edge flux of kick and Fokker-Planck shows in the profile-derived diagnostics
    tol_q = 1e-3 if N == 8 else TOL_MOM
    d = sim.step_host(1)
    dr = o.step(1)
    assert_psi(sim.get_psi_host()[0], o.psi, TOL_1, f"N={N} order={order} 1 step")
    assert_diag(d[0, 0], dr[0], tol_q=tol_q)
    d = sim.step_host(99)
    dr = o.step(99)
    assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, f"N={N} order={order} 100 steps")
    assert_diag(d[98, 0], dr[98], tol_q=tol_q)
    assert sim.step_count() == 100
    sim.close()


def test_large_kick_shift_beyond_one_cell(vfps, orc):
    """A strong resistive impedance gives |kick shift| > 1 cell: integer part of the shift and
    zero boundary are exercised."""
    N = 64
    Z = np.full((1, N + 1), 60.0 + 0j, dtype=np.complex64)
    psi0 = make_psi0(N, -6, 6, -6, 6, 1.0, 1.0, 0, 0)[None]
    sim = vfps.Simulation(N, -6, 6, -6, 6, 100, 1e-3, 4, 2, 1, Z=Z)
    sim.set_psi_host(psi0)
    o = orc.Oracle(N, -6, 6, -6, 6, 100, 1e-3, 4, 2, Z[0])
    o.set_psi(psi0[0])
    V = sim.get_wake_host()[0]
    assert np.max(np.abs(V)) * (2 * np.pi / 100) / (12 / 63) > 1.5       # shift in cells
    sim.step_host(3, diag=False)
    o.step(3, diag=False)
    assert_psi(sim.get_psi_host()[0], o.psi, 3e-5, "large kick")
    sim.close()


def test_no_wake_kick_is_identity_and_no_renormalise(vfps, orc):
    wl = get_workload("C0").with_(interp_order=4)
    psi0 = wl.psi0()
    sim = vfps.Simulation(wl.N, -6, 6, -6, 6, wl.steps_per_period, wl.beta, 4, 2, 1, flags=0)
    sim.set_psi_host(psi0)
    o = orc.Oracle(wl.N, -6, 6, -6, 6, wl.steps_per_period, wl.beta, 4, 2, None, renormalise=False)
    o.set_psi(psi0[0])
    d = sim.step_host(20)
    dr = o.step(20)
    assert_psi(sim.get_psi_host()[0], o.psi, 2e-5, "no renormalise")
    assert_diag(d[19, 0], dr[19], has_wake=False)
    assert np.all(sim.get_wake_host() == 0)
    sim.close()


def test_get_calls_match_oracle_and_are_stateless(vfps, orc):
    wl = get_workload("C1")
    sim = vfps.Simulation.from_workload(wl)
    o = orc.Oracle.from_workload(wl)
    sim.step_host(5, diag=False)
    o.step(5, diag=False)
    for _ in range(2):                                       # second round: nothing was disturbed
        rho, V, mom = sim.get_profile_host()[0], sim.get_wake_host()[0], sim.get_moments_host()[0]
        np.testing.assert_allclose(rho, o.profile(), rtol=0, atol=2e-6 * o.profile().max())
        np.testing.assert_allclose(V, o.wake(), rtol=0, atol=1e-5 * np.abs(o.wake()).max())
        assert_diag(mom, o.moments6())
    d = sim.step_host(5)
    dr = o.step(5)
    assert_psi(sim.get_psi_host()[0], o.psi, 2e-5, "after get calls")
    assert_diag(d[4, 0], dr[4])
    sim.close()


def test_device_pointer_calls_and_diag_on_device(vfps, orc):
    import torch
    wl = get_workload("C1")
    sim = vfps.Simulation.from_workload(wl)
    psi_dev = torch.from_numpy(wl.psi0()).cuda()
    sim.set_psi(psi_dev)
    diag = torch.zeros(7, 1, 6, device="cuda")
    sim.step(7, diag)
    sim.step(0)
    out = sim.get_psi()
    torch.cuda.synchronize()
    o = orc.Oracle.from_workload(wl)
    dr = o.step(7)
    assert_psi(out.cpu().numpy()[0], o.psi, 2e-5, "device path")
    for i in range(7):
        assert_diag(diag[i, 0].cpu().numpy(), dr[i])
    rho = sim.get_profile(); V = sim.get_wake(); mom = sim.get_moments()
    torch.cuda.synchronize()
    assert rho.shape == (1, 256) and V.shape == (1, 256) and mom.shape == (1, 6)
    assert sim.launch_count() > 0
    sim.close()


def test_error_paths_on_gpu(vfps):
    sim = vfps.Simulation(64, -6, 6, -6, 6, 500, 1e-3, 2)
    with pytest.raises(vfps.VfpsError) as e:
        sim.step_host(1)
    assert e.value.code == -2                               # step before set_psi
    with pytest.raises(vfps.VfpsError):
        sim.set_option(99, 0)
    sim.close()
    with pytest.raises(vfps.VfpsError) as e:
        vfps.Simulation(64, -6, 6, -6, 6, 2, 1e-3, 4)      # 2 steps per period: halo too large
    assert e.value.code == -5


# ---------------------------------------------------------------- engines
def _engine_id(vfps, name):
    return {"stream": vfps.ENGINE_STREAM, "graph": vfps.ENGINE_GRAPH, "cluster": vfps.ENGINE_CLUSTER,
            "cluster3": vfps.ENGINE_CLUSTER, "grid": vfps.ENGINE_GRID, "grid2": vfps.ENGINE_GRID}[name]


@pytest.mark.parametrize("engine", ["stream", "graph", "cluster", "cluster3", "grid", "grid2"])
def test_c1_every_engine_100_steps(vfps, orc, engine):
    """The same 100 steps of C1 through each engine (graph: two replays of 50 captured steps;
    cluster: what AUTO picks for one 256^2 simulation, the first design k_cluster_step; cluster3:
    the in-place kernel k_onchip_step; grid / grid2: the two persistent cooperative kernels)."""
    wl = get_workload("C1")
    idx = [0]
    sim = vfps.Simulation.from_workload(wl, idx)
    if engine == "cluster3":
        sim.set_cluster_kernel(3)
    if engine.startswith("grid"):
        sim.set_grid_kernel(2 if engine == "grid2" else 1)
    sim.set_engine(_engine_id(vfps, engine))
    assert sim.engine_name == engine.rstrip("23")
    if engine.startswith("cluster"):
        assert sim.cluster_kernel == (3 if engine == "cluster3" else 1)
    if engine.startswith("grid"):
        assert sim.grid_kernel == (2 if engine == "grid2" else 1)
    d = sim.step_host(100)
    psi = sim.get_psi_host()
    o = orc.Oracle.from_workload(wl, 0)
    dr = o.step(100)
    assert_psi(psi[0], o.psi, 1e-4, f"C1 100 steps, {engine}")
    for i in (0, 1, 49, 50, 99):
        assert_diag(d[i, 0], dr[i])
    sim.close()


@pytest.mark.parametrize("wake", ["fft", "direct"])
@pytest.mark.parametrize("order,N", [(4, 256), (3, 128), (2, 64), (4, 32)])
def test_stream_wake_modes(vfps, orc, wake, order, N):
    """The streaming kernels with both wake evaluations (Eq. 5 FFT, Eq. 4 direct convolution) on
    the stream and the graph engine: asymmetric box, off-centre bunch, free-space wake, 300 steps
    per period (edge tiles, floors changing inside a tile; N = 32 and 64 are narrower than one
    256-column tile)."""
    pad = 2
    Z = make_impedance(N, pad, 12.0 / (N - 1), 0.4, None)[None, :]
    psi0 = make_psi0(N, -5.0, 7.0, -6.5, 5.5, 1.2, 0.8, 1e-5, 9, q0=0.5, p0=-0.4)[None]
    sim = vfps.Simulation(N, -5.0, 7.0, -6.5, 5.5, 300, 2e-3, order, pad, 1, Z=Z)
    sim.set_wake_mode({"fft": vfps.WAKE_FFT, "direct": vfps.WAKE_DIRECT}[wake])
    sim.set_engine(vfps.ENGINE_STREAM)
    assert sim.wake_name == wake
    sim.set_psi_host(psi0)
    o = orc.Oracle(N, -5.0, 7.0, -6.5, 5.5, 300, 2e-3, order, pad, Z[0])
    o.set_psi(psi0[0])
    d = sim.step_host(1)
    dr = o.step(1)
    assert_psi(sim.get_psi_host()[0], o.psi, TOL_1, f"stream {wake} N={N} order={order} 1 step")
    assert_diag(d[0, 0], dr[0])
    sim.set_engine(vfps.ENGINE_GRAPH)
    d = sim.step_host(59)
    dr = o.step(59)
    assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, f"graph {wake} N={N} order={order} 60 steps")
    for i in (0, 30, 58):
        assert_diag(d[i, 0], dr[i])
    sim.close()


@pytest.mark.parametrize("wake", ["direct", "fft"])
@pytest.mark.parametrize("order,N", [(4, 256), (3, 128), (2, 64), (4, 32)])
def test_manhattan_rotation(vfps, orc, order, N, wake):
    """VFPS_FLAG_ROT_MANHATTAN (drift along q, RF kick along p) against the oracle's
    Manhattan step: asymmetric box, off-centre bunch, free-space wake, 300 steps per period (the
    drift and the RF kick move the outer lines by more than one cell: integer parts -2..1), stream
    engine for 1 step, graph engine for 59 more, grid engine for 20 more, then the cluster engine
    (first design) at several cluster sizes."""
    Z = make_impedance(N, 2, 12.0 / (N - 1), 0.4, None)[None, :]
    psi0 = make_psi0(N, -5.0, 7.0, -6.5, 5.5, 1.2, 0.8, 1e-5, 9, q0=0.5, p0=-0.4)[None]
    flags = vfps.FLAG_RENORMALISE | vfps.FLAG_ROT_MANHATTAN
    sim = vfps.Simulation(N, -5.0, 7.0, -6.5, 5.5, 300, 2e-3, order, 2, 1, Z=Z, flags=flags)
    sim.set_wake_mode({"fft": vfps.WAKE_FFT, "direct": vfps.WAKE_DIRECT}[wake])
    sim.set_engine(vfps.ENGINE_STREAM)
    sim.set_psi_host(psi0)
    o = orc.Oracle(N, -5.0, 7.0, -6.5, 5.5, 300, 2e-3, order, 2, Z[0], manhattan=True)
    o.set_psi(psi0[0])
    d = sim.step_host(1)
    dr = o.step(1)
    assert_psi(sim.get_psi_host()[0], o.psi, TOL_1, f"manhattan N={N} order={order} 1 step")
    assert_diag(d[0, 0], dr[0])
    sim.set_engine(vfps.ENGINE_GRAPH)
    d = sim.step_host(59)
    dr = o.step(59)
    assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, f"manhattan N={N} order={order} 60 steps")
    for i in (0, 30, 58):
        assert_diag(d[i, 0], dr[i])
    sim.set_engine(vfps.ENGINE_GRID)
    d = sim.step_host(20)
    dr = o.step(20)
    assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, f"manhattan N={N} order={order} 80 steps, grid engine")
    for i in (0, 19):
        assert_diag(d[i, 0], dr[i])
    try:
        sim.set_engine(vfps.ENGINE_CLUSTER)          # first design; needs halo <= 4 rows (not N = 256 here)
    except vfps.VfpsError as err:
        assert err.code == -5 and N == 256
        sim.close()
        return
    assert sim.engine_name == "cluster" and sim.cluster_kernel == 1
    for S in (16, 4, 1):
        try:
            sim.set_cluster_size(S)
        except vfps.VfpsError:
            continue
        d = sim.step_host(20)
        dr = o.step(20)
        assert_psi(sim.get_psi_host()[0], o.psi, 2e-4, f"manhattan N={N} order={order}, cluster engine S={S}")
        for i in (0, 19):
            assert_diag(d[i, 0], dr[i])
    with pytest.raises(vfps.VfpsError) as e:
        sim.set_cluster_kernel(3)                    # the in-place kernel has the standard rotation only
    assert e.value.code == -5
    sim.close()


def test_manhattan_c1_and_large_kick(vfps, orc):
    """C1 physics with the Manhattan rotation (100 steps), and a resistive impedance strong enough
    for wake shifts of several cells (generic two-stage path)."""
    wl = get_workload("C1")
    flags = vfps.FLAG_RENORMALISE | vfps.FLAG_ROT_MANHATTAN
    sim = vfps.Simulation(wl.N, wl.q_min, wl.q_max, wl.p_min, wl.p_max, wl.steps_per_period, wl.beta,
                          wl.interp_order, wl.pad, 1, Z=wl.impedance([0]), flags=flags)
    sim.set_psi_host(wl.psi0([0]))
    o = orc.Oracle.from_workload(wl, 0, manhattan=True)
    d = sim.step_host(100)
    dr = o.step(100)
    assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, "manhattan C1 100 steps")
    for i in (0, 49, 99):
        assert_diag(d[i, 0], dr[i])
    sim.close()
    N = 64
    Z = np.full((1, N + 1), 60.0 + 0j, dtype=np.complex64)
    psi0 = make_psi0(N, -6, 6, -6, 6, 1.0, 1.0, 0, 0)[None]
    sim = vfps.Simulation(N, -6, 6, -6, 6, 100, 1e-3, 4, 2, 1, Z=Z, flags=flags)
    sim.set_psi_host(psi0)
    o = orc.Oracle(N, -6, 6, -6, 6, 100, 1e-3, 4, 2, Z[0], manhattan=True)
    o.set_psi(psi0[0])
    d = sim.step_host(3)
    dr = o.step(3)
    # three steps of three successive fp32 interpolations with shifts of up to 8 cells on a 64^2 grid
    assert_psi(sim.get_psi_host()[0], o.psi, 6e-5, "manhattan large kick")
    assert_diag(d[2, 0], dr[2], tol_p=edge_flux_tol(dr[2][0]))
    sim.close()


@pytest.mark.parametrize("manhattan", [False, True])
@pytest.mark.parametrize("order,N", [(4, 256), (3, 128), (4, 32)])
def test_clamped_interpolation(vfps, orc, order, N, manhattan):
    """VFPS_FLAG_CLAMP (Eq. 14, reading A9) against the oracle's clamped step, standard
    and Manhattan rotation.  The input is a bunch with a sharp-edged hole, where the free cubic /
    quadratic interpolant overshoots and the clamp is active in thousands of cells; stream engine
    for 1 step, graph for 29 more, grid engine for 10 more.  The clamped and the free run must
    differ (the flag does something) and the clamped density never leaves [0, max psi_0]."""
    Z = make_impedance(N, 2, 12.0 / (N - 1), 0.4, None)[None, :]
    psi0 = make_psi0(N, -5.0, 7.0, -6.5, 5.5, 1.2, 0.8, 0.0, 9, q0=0.5, p0=-0.4)
    a, b = N // 2 - N // 8, N // 2 + N // 8
    psi0[a:b, a:b] = 0.0                                           # sharp edges inside the bunch
    psi0 = (psi0 / (psi0.astype(np.float64).sum() * (12.0 / (N - 1)) ** 2)).astype(np.float32)[None]
    flags = vfps.FLAG_RENORMALISE | vfps.FLAG_CLAMP | (vfps.FLAG_ROT_MANHATTAN if manhattan else 0)
    sim = vfps.Simulation(N, -5.0, 7.0, -6.5, 5.5, 300, 2e-3, order, 2, 1, Z=Z, flags=flags)
    if manhattan or N < 64:
        # the in-place cluster kernel has the standard rotation on N >= 64; the first design no clamp
        with pytest.raises(vfps.VfpsError) as e:
            sim.set_engine(vfps.ENGINE_CLUSTER)
        assert e.value.code == -5
    sim.set_engine(vfps.ENGINE_STREAM)
    sim.set_psi_host(psi0)
    o = orc.Oracle(N, -5.0, 7.0, -6.5, 5.5, 300, 2e-3, order, 2, Z[0], manhattan=manhattan, clamp=True)
    o.set_psi(psi0[0])
    free = orc.Oracle(N, -5.0, 7.0, -6.5, 5.5, 300, 2e-3, order, 2, Z[0], manhattan=manhattan)
    free.set_psi(psi0[0])
    d = sim.step_host(1)
    dr = o.step(1)
    free.step(1)
    # a clamp decision (is P below min / above max of its nodes?) taken in fp32 against fp64 can
    # differ only where P is within rounding of the bound, and then both results are within
    # rounding of each other: the usual tolerance holds
    assert_psi(sim.get_psi_host()[0], o.psi, TOL_1, f"clamp N={N} order={order} manhattan={manhattan} 1 step")
    # the clamped kick is not conservative: P_csr is that of the end-of-step profile (to first order
    # in its change, include/vfps.h), so the 1e-4 bar holds on this sharp-edged input too
    assert_diag(d[0, 0], dr[0])
    assert np.max(np.abs(o.psi - free.psi)) > 1e-3 * o.psi.max()
    sim.set_engine(vfps.ENGINE_GRAPH)
    d = sim.step_host(29)
    dr = o.step(29)
    assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, f"clamp N={N} order={order} manhattan={manhattan} 30 steps")
    assert_diag(d[28, 0], dr[28])
    # (Manhattan: the clamped RF kick changes the profile, so the wake needs the profile after it --
    # an extra pass in the stream / graph engines, a third grid barrier in k_grid_step)
    sim.set_engine(vfps.ENGINE_GRID)
    assert sim.engine_name == "grid" and (sim.grid_kernel == 1 if manhattan else sim.grid_kernel in (1, 2))
    d = sim.step_host(10)
    dr = o.step(10)
    psi = sim.get_psi_host()[0]
    assert_psi(psi, o.psi, 1e-4, f"clamp N={N} order={order} manhattan={manhattan} 40 steps, {sim.engine_name} engine")
    assert_diag(d[9, 0], dr[9])
    # the Fokker-Planck update is the only place left that can produce a (tiny) negative value
    assert psi.min() > -1e-4 * psi.max() and psi.max() < 1.02 * psi0.max()
    if not manhattan and N >= 64:
        # cluster engine (in-place kernel): clamped rotation and kick on chip; its P_csr is that of the
        # end-of-step density to first order in the profile change of the clamped kick: 1e-4 holds
        ran = 0
        for S in (16, 4, 2):
            try:
                sim.set_cluster_size(S)
            except vfps.VfpsError as err:
                assert err.code == -5
                continue
            sim.set_engine(vfps.ENGINE_CLUSTER)
            assert sim.engine_name == "cluster" and sim.cluster_kernel == 3
            d = sim.step_host(10)
            dr = o.step(10)
            assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, f"clamp N={N} order={order}, cluster engine S={S}")
            for i in (0, 9):
                assert_diag(d[i, 0], dr[i])
            ran += 1
        assert ran >= 2
    sim.close()


@pytest.mark.parametrize("order,S", [(4, 16), (4, 2), (3, 8)])
def test_clamped_interpolation_cluster_c1(vfps, orc, order, S):
    """VFPS_FLAG_CLAMP on the cluster engine in the regime of the BASELINE configs (256^2, 4000 steps
    per period: per-launch weight tables): C1 physics on a bunch with a sharp-edged hole, 1 step and
    100 steps against the oracle's clamped step, every diagnostic (P_csr included) at 1e-4."""
    wl = get_workload("C1").with_(interp_order=order)
    N = wl.N
    psi0 = wl.psi0([0])[0].copy()
    a, b = N // 2 - N // 8, N // 2 + N // 8
    psi0[a:b, a:b] = 0.0
    psi0 = (psi0 / (psi0.astype(np.float64).sum() * wl.dq * wl.dp)).astype(np.float32)[None]
    Z = wl.impedance([0])
    sim = vfps.Simulation(N, wl.q_min, wl.q_max, wl.p_min, wl.p_max, wl.steps_per_period, wl.beta, order, wl.pad, 1,
                          Z=Z, flags=vfps.FLAG_RENORMALISE | vfps.FLAG_CLAMP)
    sim.set_cluster_size(S)
    sim.set_engine(vfps.ENGINE_CLUSTER)
    assert sim.cluster_kernel == 3 and sim.cluster_size == S
    sim.set_psi_host(psi0)
    o = orc.Oracle(N, wl.q_min, wl.q_max, wl.p_min, wl.p_max, wl.steps_per_period, wl.beta, order, wl.pad, Z[0], clamp=True)
    o.set_psi(psi0[0])
    free = orc.Oracle(N, wl.q_min, wl.q_max, wl.p_min, wl.p_max, wl.steps_per_period, wl.beta, order, wl.pad, Z[0])
    free.set_psi(psi0[0])
    d = sim.step_host(1)
    dr = o.step(1)
    assert_psi(sim.get_psi_host()[0], o.psi, TOL_1, f"clamp C1 order={order} S={S} 1 step")
    assert_diag(d[0, 0], dr[0])
    d = sim.step_host(99)
    dr = o.step(99)
    free.step(100)
    psi = sim.get_psi_host()[0]
    assert_psi(psi, o.psi, 1e-4, f"clamp C1 order={order} S={S} 100 steps")
    for i in (0, 49, 98):
        assert_diag(d[i, 0], dr[i])
    assert np.max(np.abs(o.psi - free.psi)) > 1e-3 * o.psi.max()       # the flag does something
    assert psi.min() > -1e-4 * psi.max() and psi.max() < 1.02 * psi0.max()
    sim.close()


def test_adiabatic_scan_set_impedance(vfps, orc):
    """The paper's adiabatic current scan (L239, L290-298): the final distribution of one current
    seeds the next.  vfps_set_impedance swaps Z (and the wake function) of a running simulation:
    three currents S_csr = 0.6 -> 0.5 -> 0.4 of the C1 physics, 150 steps each, on every engine in
    turn, against the oracle chained the same way."""
    wl = get_workload("C1")
    dq = (wl.q_max - wl.q_min) / (wl.N - 1)
    sim = vfps.Simulation.from_workload(wl.with_(S_csr=(0.6,)))
    o = orc.Oracle.from_workload(wl.with_(S_csr=(0.6,)))
    engines = [vfps.ENGINE_CLUSTER, vfps.ENGINE_GRID, vfps.ENGINE_GRAPH]
    P = []
    for S, eng in zip((0.6, 0.5, 0.4), engines):
        Z = make_impedance(wl.N, wl.pad, dq, S, 1.0)
        if S != 0.6:
            sim.set_impedance_host(Z[None, :])
            psi_prev = o.psi.copy()
            o = orc.Oracle(wl.N, wl.q_min, wl.q_max, wl.p_min, wl.p_max, wl.steps_per_period, wl.beta,
                           wl.interp_order, wl.pad, Z)
            o.set_psi(psi_prev)
        sim.set_engine(eng)
        d = sim.step_host(150)
        dr = o.step(150)
        assert_psi(sim.get_psi_host()[0], o.psi, 2e-4, f"adiabatic scan, S = {S}")
        assert_diag(d[149, 0], dr[149])
        P.append(d[149, 0, 5])
    assert P[0] > P[1] > P[2] > 0                    # the radiated power follows the current down
    assert sim.step_count() == 450
    sim.close()
    nowake = vfps.Simulation(64, -6, 6, -6, 6, 500, 1e-3, 2)
    with pytest.raises(vfps.VfpsError) as e:
        nowake.set_impedance_host(np.zeros((1, 65), dtype=np.complex64))
    assert e.value.code == -2
    nowake.close()


@pytest.mark.parametrize("order,N", [(4, 512), (4, 256), (3, 128), (2, 64), (4, 8)])
def test_grid_engine(vfps, orc, order, N):
    """Persistent cooperative-grid engine: asymmetric box, off-centre bunch, free-space wake, 300
    steps per period (slow rotation paths at the edges and where a floor changes), 1 step and 60
    steps with the diagnostics of every step; then hand-over to the stream engine and back."""
    Z = make_impedance(N, 2, 12.0 / (N - 1), 0.4, None)[None, :]
    psi0 = make_psi0(N, -5.0, 7.0, -6.5, 5.5, 1.2, 0.8, 1e-5, 9, q0=0.5, p0=-0.4)[None]
    sim = vfps.Simulation(N, -5.0, 7.0, -6.5, 5.5, 300, 2e-3, order, 2, 1, Z=Z)
    sim.set_engine(vfps.ENGINE_GRID)
    assert sim.engine_name == "grid" and sim.wake_name == "direct"
    sim.set_psi_host(psi0)
    o = orc.Oracle(N, -5.0, 7.0, -6.5, 5.5, 300, 2e-3, order, 2, Z[0])
    o.set_psi(psi0[0])
    tol_q = 2e-3 if N == 8 else TOL_MOM          # N = 8: the bunch overflows the box (edge flux)
    d = sim.step_host(1)
    dr = o.step(1)
    assert_psi(sim.get_psi_host()[0], o.psi, TOL_1, f"grid N={N} order={order} 1 step")
    assert_diag(d[0, 0], dr[0], tol_q=tol_q)
    d = sim.step_host(59)
    dr = o.step(59)
    assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, f"grid N={N} order={order} 60 steps")
    for i in (0, 30, 58):
        assert_diag(d[i, 0], dr[i], tol_q=tol_q)
    sim.set_engine(vfps.ENGINE_STREAM)
    sim.step_host(2)
    sim.set_engine(vfps.ENGINE_GRID)
    d = sim.step_host(2)
    dr = o.step(4)
    assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, f"grid -> stream -> grid N={N}")
    assert_diag(d[1, 0], dr[3], tol_q=tol_q)
    assert sim.step_count() == 64
    sim.close()


@pytest.mark.parametrize("order,clamp", [(2, False), (3, False), (4, False), (3, True), (4, True)])
@pytest.mark.parametrize("N,spp", [(256, 4000), (512, 4000), (1024, 8000)])
def test_grid2_engine(vfps, orc, N, spp, order, clamp):
    """TMA-staged kernel of the grid engine (k_grid2_step): asymmetric box (the grid edges cut through
    tiles on all four sides: TMA's zero fill is reading A8), off-centre mismatched bunch, free-space
    wake; stripes of 1-2 (N = 256), 3-4 (512) and 6-7 (1024) rows per CTA, so ragged chunks and
    stripes shorter than the halo all occur (the clamp is the identity for linear interpolation, so
    order 2 runs without the flag only).  1 step and 60 steps with every diagnostics row, then
    hand-over to the first grid kernel and back."""
    Z = make_impedance(N, 2, 12.0 / (N - 1), 0.4, None)[None, :]
    psi0 = make_psi0(N, -5.0, 7.0, -6.5, 5.5, 1.2, 0.8, 1e-5, 9, q0=0.5, p0=-0.4)
    if clamp:
        a, b = N // 2 - N // 8, N // 2 + N // 8
        psi0[a:b, a:b] = 0.0
        psi0 = (psi0 / (psi0.astype(np.float64).sum() * (12.0 / (N - 1)) ** 2)).astype(np.float32)
    psi0 = psi0[None]
    flags = vfps.FLAG_RENORMALISE | (vfps.FLAG_CLAMP if clamp else 0)
    sim = vfps.Simulation(N, -5.0, 7.0, -6.5, 5.5, spp, 2e-3, order, 2, 1, Z=Z, flags=flags)
    sim.set_grid_kernel(2)
    sim.set_engine(vfps.ENGINE_GRID)
    assert sim.engine_name == "grid" and sim.grid_kernel == 2 and sim.wake_name == "direct"
    sim.set_psi_host(psi0)
    o = orc.Oracle(N, -5.0, 7.0, -6.5, 5.5, spp, 2e-3, order, 2, Z[0], clamp=clamp)
    o.set_psi(psi0[0])
    d = sim.step_host(1)
    dr = o.step(1)
    assert_psi(sim.get_psi_host()[0], o.psi, TOL_1, f"grid2 N={N} order={order} 1 step")
    assert_diag(d[0, 0], dr[0])
    d = sim.step_host(59)
    dr = o.step(59)
    assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, f"grid2 N={N} order={order} 60 steps")
    for i in (0, 30, 58):
        assert_diag(d[i, 0], dr[i])
    sim.set_grid_kernel(1)
    assert sim.grid_kernel == 1
    sim.step_host(2)
    sim.set_grid_kernel(2)
    d = sim.step_host(2)
    dr = o.step(4)
    assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, f"grid2 -> grid -> grid2 N={N}")
    assert_diag(d[1, 0], dr[3])
    assert sim.step_count() == 64
    sim.close()


def test_grid2_engine_refusals(vfps):
    """k_grid2_step needs N % 256 == 0, the standard rotation and a rotation angle small enough for
    first-order weight tables; the request is refused otherwise (AUTO then keeps k_grid_step)."""
    sim = vfps.Simulation(128, -6, 6, -6, 6, 4000, 1e-3, 4)
    with pytest.raises(vfps.VfpsError) as e:
        sim.set_grid_kernel(2)
    assert e.value.code == -5
    sim.set_engine(vfps.ENGINE_GRID)
    assert sim.grid_kernel == 1
    sim.close()
    sim = vfps.Simulation(256, -6, 6, -6, 6, 300, 1e-3, 4)            # 1.2 degrees per step
    with pytest.raises(vfps.VfpsError) as e:
        sim.set_grid_kernel(2)
    assert e.value.code == -5
    sim.close()
    sim = vfps.Simulation(256, -6, 6, -6, 6, 4000, 1e-3, 4, flags=vfps.FLAG_RENORMALISE | vfps.FLAG_ROT_MANHATTAN)
    with pytest.raises(vfps.VfpsError) as e:
        sim.set_grid_kernel(2)
    assert e.value.code == -5
    sim.close()


def test_grid_engine_rejects_batches(vfps):
    wl = get_workload("C3")
    sim = vfps.Simulation.from_workload(wl, [0, 1])
    with pytest.raises(vfps.VfpsError) as e:
        sim.set_engine(vfps.ENGINE_GRID)
    assert e.value.code == -5
    sim.close()


def _cluster_cases():
    """(N, kernel, steps_per_period, S) for test_cluster_engine_sizes.  300 steps per period moves
    the corner cells by up to N/60 cells per step (floors change inside a CTA's rows and columns:
    the per-cell paths run, and the in-place kernel evaluates its weights per cell); 4000 steps per
    period is the regime of the BASELINE configs (per-launch weight tables).  The first design
    (kernel 1) has 4 halo rows, so its steps per period grow with N; the in-place kernel (3) takes
    halos up to 7 rows.  Combinations the library refuses (listed in _CLUSTER_INFEASIBLE with the
    reason) are checked to be refused with VFPS_ERR_UNSUPPORTED."""
    cases = []
    for N, spps in ((64, (300, 4000)), (128, (300, 4000)), (256, (300, 4000)), (512, (1200, 4000))):
        for spp in spps:
            for S in (1, 2, 4, 8, 16):
                cases.append((N, 3, spp, S))
    for N, spp in ((32, 300), (64, 300), (128, 300), (256, 1200), (512, 2400)):
        for S in (1, 2, 4, 8, 16):
            cases.append((N, 1, spp, S))
    return cases


@pytest.mark.parametrize("order", [2, 3, 4])
@pytest.mark.parametrize("N,kernel,spp,S", _cluster_cases())
def test_cluster_engine_sizes(vfps, orc, N, order, S, kernel, spp):
    """Persistent cluster engine, both kernels, every grid size / interpolation order / cluster
    size: asymmetric box, off-centre mismatched bunch, free-space wake (as
    test_orders_and_small_grids), 1 step and 60 steps, diagnostics of every step; the wake of the
    0.4-strength free-space impedance shifts rows by different integer parts."""
    Z = make_impedance(N, 2, 12.0 / (N - 1), 0.4, None)[None, :]
    psi0 = make_psi0(N, -5.0, 7.0, -6.5, 5.5, 1.2, 0.8, 1e-5, 9, q0=0.5, p0=-0.4)[None]
    sim = vfps.Simulation(N, -5.0, 7.0, -6.5, 5.5, spp, 2e-3, order, 2, 1, Z=Z)
    try:
        sim.set_cluster_kernel(kernel)
        sim.set_cluster_size(S)
    except vfps.VfpsError as e:
        assert e.code == -5
        sim.close()
        reason = _cluster_infeasible(N, kernel, spp, S, order)
        assert reason, f"kernel {kernel} refused N={N} S={S} spp={spp}: {e}"
        return
    assert not _cluster_infeasible(N, kernel, spp, S, order)
    sim.set_engine(vfps.ENGINE_CLUSTER)
    assert sim.engine_name == "cluster" and sim.cluster_size == S and sim.wake_name == "direct"
    assert sim.cluster_kernel == kernel
    sim.set_psi_host(psi0)
    o = orc.Oracle(N, -5.0, 7.0, -6.5, 5.5, spp, 2e-3, order, 2, Z[0])
    o.set_psi(psi0[0])
    d = sim.step_host(1)
    dr = o.step(1)
    assert_psi(sim.get_psi_host()[0], o.psi, TOL_1, f"cluster N={N} order={order} S={S} 1 step")
    assert_diag(d[0, 0], dr[0])
    d = sim.step_host(59)
    dr = o.step(59)
    assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, f"cluster N={N} order={order} S={S} 60 steps")
    for i in (0, 30, 58):
        assert_diag(d[i, 0], dr[i])
    assert sim.step_count() == 60
    sim.close()


def _cluster_infeasible(N, kernel, spp, S, order):
    """Why the library is expected to refuse this combination ('' = it must run)."""
    rows = N // S
    smem_floats = 227 * 1024 // 4
    halo = {300: {32: 2, 64: 3, 128: 4, 256: 6}, 1200: {256: 3, 512: 4}, 2400: {512: 3},
            4000: {64: 2, 128: 2, 256: 2, 512: 2}}[spp][N]
    if kernel == 1:
        if rows < halo:
            return "fewer rows per CTA than halo rows"
        if (2 * rows + 8) * (N + 8) > smem_floats:
            return "two row buffers do not fit 227 KB of shared memory"
        return ""
    if rows < 4 or rows < halo:
        return "fewer rows per CTA than halo rows"
    if rows * (N + 16) > smem_floats:
        return "the rows of a CTA do not fit 227 KB of shared memory"
    if (N, spp, S) == (256, 300, 2) or ((N, spp, S) == (512, 1200, 8) and order != 3):
        return "rows + aprons + free rows of the in-place walkers (halo 6 / 4) exceed 227 KB"
    return ""


@pytest.mark.parametrize("kernel", [1, 3])
def test_cluster_engine_c2_512(vfps, orc, kernel):
    wl = get_workload("C2").with_(S_csr=(0.6,))
    sim, psi, d, refs, dr = run_pair(vfps, orc, wl, 40, engine=vfps.ENGINE_CLUSTER, diag_every=1, cluster_kernel=kernel)
    assert sim.engine_name == "cluster" and sim.cluster_size == 16 and sim.cluster_kernel == kernel
    assert_psi(psi[0], refs[0].psi, 5e-5, "C2 cluster 40 steps")
    for i in (0, 20, 39):
        assert_diag(d[i, 0], dr[0][i])
    sim.close()


@pytest.mark.parametrize("kernel,S", [(1, 4), (1, 8), (1, 16), (3, 2), (3, 4), (3, 8), (3, 16)])
def test_cluster_engine_batched(vfps, orc, S, kernel):
    """More members than one cluster: every cluster walks through its members one after another."""
    wl = get_workload("C3")
    idx = [0, 37, 128, 255, 3, 64]
    sim = vfps.Simulation.from_workload(wl, idx)
    sim.set_cluster_kernel(kernel)
    sim.set_cluster_size(S)
    sim.set_engine(vfps.ENGINE_CLUSTER)
    d = sim.step_host(30)
    psi = sim.get_psi_host()
    for i, m in enumerate(idx):
        o = orc.Oracle.from_workload(wl, m)
        dr = o.step(30)
        assert_psi(psi[i], o.psi, 5e-5, f"C3 member {m} cluster S={S}")
        assert_diag(d[29, i], dr[29])
        assert_diag(d[0, i], dr[0])
    sim.close()


def test_cluster_engine_batch_of_single_cta_clusters_long_run(vfps):
    """64 members of 128^2 on clusters of ONE CTA (what AUTO picks for this batch) for 100 000
    steps: every exchange of the cluster protocol degenerates to a CTA talking to itself.  A lost
    or doubled mbarrier phase hangs or corrupts the run; the renormalised charge of every step of
    the last period and the end state must be sane for every member."""
    wl = get_workload("C3").with_(N=128, members=64, S_csr=tuple(0.05 + 0.01 * m for m in range(64)),
                                  seeds=tuple(range(64)), steps_per_period=2000)
    for kernel in (3, 1):
        sim = vfps.Simulation.from_workload(wl)
        sim.set_cluster_kernel(kernel)
        sim.set_cluster_size(1)
        sim.set_engine(vfps.ENGINE_CLUSTER)
        assert sim.cluster_size == 1
        for _ in range(49):
            sim.step_host(2000, diag=False)
        d = sim.step_host(2000)
        _invariants(d)
        assert sim.step_count() == 100000
        sim.close()


@pytest.mark.parametrize("N,kernel", [(64, 1), (128, 1), (64, 3), (128, 3)])
def test_cluster_engine_large_kick_and_switching(vfps, orc, N, kernel):
    """|kick shift| > 1 cell (generic-shift path of the cluster engine, both kernels), then
    continue the same simulation on the stream engine: state hand-over between engines is exact."""
    Z = np.full((1, N + 1), 60.0 + 0j, dtype=np.complex64)
    psi0 = make_psi0(N, -6, 6, -6, 6, 1.0, 1.0, 0, 0)[None]
    spp = 100 * N // 64          # the same rotation displacement in cells on both grids
    sim = vfps.Simulation(N, -6, 6, -6, 6, spp, 1e-3, 4, 2, 1, Z=Z)
    sim.set_cluster_kernel(kernel)
    sim.set_engine(vfps.ENGINE_CLUSTER)
    assert sim.cluster_kernel == kernel
    sim.set_psi_host(psi0)
    o = orc.Oracle(N, -6, 6, -6, 6, spp, 1e-3, 4, 2, Z[0])
    o.set_psi(psi0[0])
    d = sim.step_host(3)
    dr = o.step(3)
    # this kick pushes 1.7 % of the charge over the p edge per step: P_csr (taken from the
    # post-rotation profile, include/vfps.h) differs from the end-of-step value by that flux
    assert_psi(sim.get_psi_host()[0], o.psi, 3e-5, "cluster large kick")
    assert_diag(d[2, 0], dr[2], tol_p=edge_flux_tol(dr[2][0]))
    sim.set_engine(vfps.ENGINE_STREAM)
    d = sim.step_host(3)
    dr = o.step(3)
    assert_psi(sim.get_psi_host()[0], o.psi, 5e-5, "cluster -> stream")
    assert_diag(d[2, 0], dr[2], tol_p=edge_flux_tol(dr[2][0]))      # by now a third of the charge leaves per step
    sim.set_engine(vfps.ENGINE_CLUSTER)
    d = sim.step_host(2)
    dr = o.step(2)
    assert_psi(sim.get_psi_host()[0], o.psi, 8e-5, "stream -> cluster")
    assert_diag(d[1, 0], dr[1], tol_p=edge_flux_tol(dr[1][0]))
    sim.close()


@pytest.mark.parametrize("kernel", [1, 3])
def test_cluster_engine_no_wake_no_renormalise(vfps, orc, kernel):
    wl = get_workload("C0")
    psi0 = wl.psi0()
    sim = vfps.Simulation(wl.N, -6, 6, -6, 6, wl.steps_per_period, wl.beta, 2, 2, 1, flags=0)
    sim.set_cluster_kernel(kernel)
    sim.set_engine(vfps.ENGINE_CLUSTER)
    sim.set_psi_host(psi0)
    o = orc.Oracle(wl.N, -6, 6, -6, 6, wl.steps_per_period, wl.beta, 2, 2, None, renormalise=False)
    o.set_psi(psi0[0])
    d = sim.step_host(500)
    dr = o.step(500)
    assert_psi(sim.get_psi_host()[0], o.psi, 5e-4, "cluster C0 no renormalise")
    assert_diag(d[499, 0], dr[499], has_wake=False)
    sim.close()


# ---------------------------------------------------------------- seeded random configurations
def _random_case(seed):
    """A seeded draw of grid size, box, step, damping, current, interpolation order, flags and bunch: the boxes are
    asymmetric and of unequal aspect, the steps range from a few hundred to several thousand per period, the bunch
    sits off centre -- the combinations no hand-written case happens to pick."""
    rng = np.random.default_rng(1000 + seed)
    N = int(rng.choice([64, 128, 256, 512]))
    order = int(rng.choice([4, 3, 4, 2]))
    qmin, qmax = -float(rng.uniform(4.5, 7.0)), float(rng.uniform(4.5, 7.0))
    pmin, pmax = -float(rng.uniform(4.5, 7.0)), float(rng.uniform(4.5, 7.0))
    spp = int(np.exp(rng.uniform(np.log(12.0 * N), np.log(16000.0))))      # |displacement| stays within the 4-row halo
    beta = float(np.exp(rng.uniform(np.log(1e-4), np.log(2e-2))))
    S = float(rng.uniform(0.05, 0.8))
    plates = None if rng.random() < 0.3 else float(rng.uniform(0.3, 2.0))
    clamp = bool(rng.random() < 0.3)
    manhattan = bool(rng.random() < 0.25)
    bunch = dict(sigma_q=float(rng.uniform(0.7, 1.3)), sigma_p=float(rng.uniform(0.7, 1.3)), noise=1e-6, seed=seed,
                 q0=float(rng.uniform(-0.5, 0.5)), p0=float(rng.uniform(-0.5, 0.5)))
    return dict(N=N, order=order, box=(qmin, qmax, pmin, pmax), spp=spp, beta=beta, S=S, plates=plates, clamp=clamp,
                manhattan=manhattan, bunch=bunch)


@pytest.mark.parametrize("seed", range(24))
def test_random_configurations(vfps, orc, seed):
    """24 seeded random configurations, each on the engine AUTO picks and then on every other engine that accepts
    it: 1 step at 1e-5, 25 steps at 1e-4, all six diagnostics at 1e-4 (P_csr with the edge-flux allowance)."""
    cs = _random_case(seed)
    N, order, box = cs["N"], cs["order"], cs["box"]
    dq = (box[1] - box[0]) / (N - 1)
    Z = make_impedance(N, 2, dq, cs["S"], cs["plates"])[None, :]
    b = cs["bunch"]
    psi0 = make_psi0(N, *box, b["sigma_q"], b["sigma_p"], b["noise"], b["seed"], q0=b["q0"], p0=b["p0"])[None]
    flags = vfps.FLAG_RENORMALISE | (vfps.FLAG_CLAMP if cs["clamp"] else 0) | (vfps.FLAG_ROT_MANHATTAN if cs["manhattan"] else 0)
    sim = vfps.Simulation(N, *box, cs["spp"], cs["beta"], order, 2, 1, Z=Z, flags=flags)
    o = orc.Oracle(N, *box, cs["spp"], cs["beta"], order, 2, Z[0], manhattan=cs["manhattan"], clamp=cs["clamp"])
    sim.set_psi_host(psi0)
    o.set_psi(psi0[0])
    what = f"seed {seed}: {cs}"
    d = sim.step_host(1)
    dr = o.step(1)
    assert_psi(sim.get_psi_host()[0], o.psi, TOL_1, what + f" 1 step, {sim.engine_name}")
    assert_diag(d[0, 0], dr[0], tol_p=edge_flux_tol(dr[0][0]))
    d = sim.step_host(24)
    dr = o.step(24)
    assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, what + f" 25 steps, {sim.engine_name}")
    assert_diag(d[23, 0], dr[23], tol_p=edge_flux_tol(dr[23][0]))
    auto = sim.engine_name
    ran = [auto]
    for name, eng in (("stream", vfps.ENGINE_STREAM), ("graph", vfps.ENGINE_GRAPH), ("cluster", vfps.ENGINE_CLUSTER),
                      ("grid", vfps.ENGINE_GRID)):
        if name == auto:
            continue
        try:
            sim.set_engine(eng)
        except vfps.VfpsError as e:
            assert e.code == -5                           # refused with a reason, never a wrong answer
            continue
        sim.set_psi_host(psi0)
        o.set_psi(psi0[0])
        d = sim.step_host(25)
        dr = o.step(25)
        assert_psi(sim.get_psi_host()[0], o.psi, 1e-4, what + f" 25 steps, {name}")
        assert_diag(d[24, 0], dr[24], tol_p=edge_flux_tol(dr[24][0]))
        ran.append(name)
    assert len(ran) >= 3, ran
    sim.close()
