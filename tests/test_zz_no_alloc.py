"""vfps_wake_noalloc (include/vfps.h): the wake of a caller-held profile with its scratch -- the wake function --
in an array built into the library instead of in memory from cudaMalloc.  Checked against the existing path
(vfps_get_wake of a handle, which allocates at create) on consecutive calls that share the built-in array, at
the tolerance the parity tests use for V (1e-5 of max |V|, tests/test_gpu_parity.py), and against the oracle.

Collected last on purpose (the suite runs with pytest -x): a failure here hides nothing after it.  Needs
nothing from the tests before it: passes alone in a fresh process as well."""
import numpy as np
import pytest

from workloads import make_impedance, make_psi0

pytestmark = pytest.mark.gpu

TOL_V = 1e-5


def _case(vfps, N, pad, S_csr, plates, bunch):
    """Profile and wake of a Gaussian bunch through the EXISTING path: a handle, vfps_get_profile, vfps_get_wake."""
    import torch
    box = (-6.0, 6.0, -6.0, 6.0)
    Z = make_impedance(N, pad, 12.0 / (N - 1), S_csr, plates)
    psi0 = make_psi0(N, *box, *bunch)[None]
    sim = vfps.Simulation(N, *box, 4000, 1e-3, 4, pad, 1, Z=Z[None, :])
    sim.set_psi_host(psi0)
    rho = sim.get_profile()[0].clone()
    V_ref = sim.get_wake()[0].clone()
    torch.cuda.synchronize()
    sim.close()
    return torch.from_numpy(Z).cuda(), rho, V_ref, Z


def _assert_close(V, V_ref, what):
    a, b = V.cpu().numpy().astype(np.float64), np.asarray(V_ref.cpu().numpy() if hasattr(V_ref, "cpu") else V_ref, dtype=np.float64)
    err = np.max(np.abs(a - b)) / np.max(np.abs(b))
    assert err <= TOL_V, f"{what}: max|dV| / max|V| = {err:.3e} > {TOL_V:.0e}"


def test_wake_noalloc_matches_get_wake_on_consecutive_calls(vfps, orc):
    import torch
    # A: C1-like (256, parallel plates); B: a larger grid, longer padding, free space, off-centre narrow bunch
    ZA, rhoA, VA_ref, ZA_host = _case(vfps, 256, 2, 0.5, 0.8, (1.0, 1.0, 1e-6, 3))
    ZB, rhoB, VB_ref, _ = _case(vfps, 1024, 4, 0.3, None, (0.6, 1.2, 0.0, 0, 1.1, -0.4))
    assert float(VA_ref.abs().max()) > 0 and float(VB_ref.abs().max()) > 0
    VA1, VB, VA2 = torch.full_like(rhoA, 7.0), torch.full_like(rhoB, 7.0), torch.full_like(rhoA, 7.0)
    vfps.wake_noalloc(256, 2, ZA, rhoA, VA1)                   # first call on this device: looks up the scratch address
    torch.cuda.synchronize()
    vfps.wake_noalloc(1024, 4, ZB, rhoB, VB)                   # overwrites the shared scratch with another wake function
    vfps.wake_noalloc(256, 2, ZA, rhoA, VA2)                   # ... and back: nothing of call B may survive
    torch.cuda.synchronize()
    _assert_close(VA1, VA_ref, "call 1 (N = 256)")
    _assert_close(VB, VB_ref, "call 2 (N = 1024, same scratch)")
    _assert_close(VA2, VA_ref, "call 3 (N = 256 again)")
    assert torch.equal(VA1, VA2)                               # same inputs, same bits: no state leaks between calls
    # ... and against the oracle's plain definition (Eq. 4-5) on the same profile
    V_orc = orc.wake(orc.wake_function(256, 512, ZA_host.astype(np.complex128)), rhoA.cpu().numpy().astype(np.float64))
    _assert_close(VA1, V_orc, "call 1 against the oracle")
    # on a side stream as well (the caller's stream is honoured)
    st = torch.cuda.Stream()
    VA3 = torch.zeros_like(rhoA)
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        vfps.wake_noalloc(256, 2, ZA, rhoA, VA3, stream=st)
    st.synchronize()
    assert torch.equal(VA1, VA3)


def test_wake_noalloc_rejects_what_does_not_fit(vfps):
    import torch
    N = vfps.NOALLOC_MAX_N
    Z = torch.zeros(2 * N * 2 // 2 + 1, dtype=torch.complex64, device="cuda")
    rho = torch.zeros(2 * N, device="cuda")
    V = torch.zeros(2 * N, device="cuda")
    with pytest.raises(vfps.VfpsError) as e:
        vfps.wake_noalloc(2 * N, 2, Z, rho, V)                 # beyond the built-in array
    assert e.value.code == -5 and "VFPS_NOALLOC_MAX_N" in str(e.value)
    with pytest.raises(vfps.VfpsError) as e:
        vfps.wake_noalloc(256, 2, None, rho[:256].contiguous(), V[:256].contiguous())
    assert e.value.code == -1
    with pytest.raises(vfps.VfpsError) as e:
        vfps.wake_noalloc(256, 3, Z[:385].contiguous(), rho[:256].contiguous(), V[:256].contiguous())
    assert e.value.code == -1
    # the maximum itself is served: N = 4096, pad = 2, a delay-free resistive impedance Z_k = R: w = R delta, V = R rho
    Zr = torch.full((N * 2 // 2 + 1,), 2.5 + 0j, dtype=torch.complex64, device="cuda")
    rho = torch.rand(N, device="cuda")
    V = torch.zeros(N, device="cuda")
    vfps.wake_noalloc(N, 2, Zr, rho, V)
    torch.cuda.synchronize()
    np.testing.assert_allclose(V.cpu().numpy(), 2.5 * rho.cpu().numpy(), rtol=0, atol=TOL_V * 2.5)


def test_wake_noalloc_runs_under_stream_capture(vfps):
    """The caller the entry point exists for: under a stream capture in global mode every allocating CUDA call
    (cudaMalloc, cudaFree, ...) fails with cudaErrorStreamCaptureUnsupported and invalidates the capture.  The call is
    captured into a CUDA graph (after one call outside the capture, which looks up the scratch address) and the graph
    is replayed twice, the second time on new contents of the input buffer."""
    import torch
    ZA, rhoA, VA_ref, _ = _case(vfps, 256, 2, 0.5, 0.8, (1.0, 1.0, 1e-6, 3))
    rho_buf, V_buf = rhoA.clone(), torch.zeros_like(rhoA)
    vfps.wake_noalloc(256, 2, ZA, rho_buf, V_buf)              # set-up call, not captured
    torch.cuda.synchronize()
    V_buf.zero_()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, capture_error_mode="global"):
        vfps.wake_noalloc(256, 2, ZA, rho_buf, V_buf)
    g.replay()
    torch.cuda.synchronize()
    _assert_close(V_buf, VA_ref, "graph replay 1")
    rho_buf.mul_(-0.5)                                         # the wake is linear in the profile
    g.replay()
    torch.cuda.synchronize()
    _assert_close(V_buf, -0.5 * VA_ref, "graph replay 2 (new input in the same buffer)")
