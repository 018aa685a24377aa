"""sc_ivr_fourier_static: the Fourier sum of Eq. 11 for callers that cannot allocate device memory.

Some users of this library have no way to get a workspace: a plug-in inside a program whose own memory pool took all of
HBM at start-up (cudaMalloc fails for everybody else afterwards), a step of a latency-bound loop (cudaMalloc / cudaFree
synchronise the device), a process with a fixed and already spent device-memory budget.  For them the library keeps the
scratch of this one stage in a static 16 MiB device array (include/sc_ivr.h, SC_IVR_STATIC_SCRATCH_BYTES), which every call
shares and which keeps the previous call's contents.  So the test makes calls IN A ROW, of different shapes, through the
C ABI, and compares each with the existing workspace path (sc_ivr_fourier) on the same inputs, within the tolerance
test_fourier_parity uses against the oracle: a scratch address that is wrong, or padding that is not cleared between
calls, shows up here.

This file is collected last on purpose (pytest -x stops at the first failure: a failure here hides nothing), and it makes
no assumption about what ran before it: it passes alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

from paper_1312_4698_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = 1e-11  # of max |A|, as in test_gpu_parity.py::test_fourier_parity


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    torch.cuda.set_device(0)
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_1312_4698_b200 import binding
    binding.lib()
    return binding


def _case(torch, B, seed, nsteps, n, k, emax):
    """Seeded z series and grid on the device, and the existing path's answer (sc_ivr_fourier with a caller's workspace)."""
    rng = np.random.default_rng(seed)
    w = inputs.make_config(1, ntraj=2, nsteps=nsteps, k=k)
    E = inputs.energy_grid(k, 0.0, emax)
    z = (rng.standard_normal((nsteps + 1, n)) + 1j * rng.standard_normal((nsteps + 1, n))) * 0.3
    z_dev = torch.from_numpy(z).cuda()
    E_dev = torch.from_numpy(np.ascontiguousarray(E)).cuda()
    ref = B.ScIvr.from_workload(w).fourier(z_dev, E)
    torch.cuda.synchronize()
    return w, z_dev, E_dev, ref


def _close(torch, A, ref):
    return float((A - ref).abs().max()) <= TOL * float(ref.abs().max())


def test_static_scratch_entry_matches_the_workspace_path_on_calls_in_a_row(torch_cuda, B, oracle):
    torch = torch_cuda
    # call 1: ragged against every tile (128 trajectories, 64 energies, 16 time samples)
    w1, z1, E1, ref1 = _case(torch, B, 5, nsteps=333, n=150, k=70, emax=20000.0)
    # call 2: a smaller problem of another shape; its padding lies where call 1 left z values and twiddles
    w2, z2, E2, ref2 = _case(torch, B, 6, nsteps=100, n=37, k=200, emax=9000.0)
    A1 = torch.full((150, 70), float("nan"), dtype=torch.complex128, device="cuda")
    A2 = torch.full((37, 200), float("nan"), dtype=torch.complex128, device="cuda")
    A3 = torch.full((150, 70), float("nan"), dtype=torch.complex128, device="cuda")
    assert 0 < B.fourier_static_scratch_bytes(150, 333, 70) <= B.STATIC_SCRATCH_BYTES

    B.fourier_static(z1, E1, w1.dt, A1)  # first call on this device: also looks up the array's address
    B.fourier_static(z2, E2, w2.dt, A2)  # back to back on the same stream, no synchronisation in between
    free_before = torch.cuda.mem_get_info()[0]
    B.fourier_static(z1, E1, w1.dt, A3)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]

    assert _close(torch, A1, ref1)
    assert _close(torch, A2, ref2)
    assert torch.equal(A1, A3)               # same inputs, same bits: nothing of call 2 leaked into call 3
    assert free_after >= free_before         # a warmed-up call takes no device memory
    # and the existing path is itself right: the definition, one cexp per term (oracle), on call 2's inputs
    Ao = oracle.fourier(z2.cpu().numpy().T.copy(), w2.dt, inputs.energy_grid(200, 0.0, 9000.0), mode=0)
    assert np.max(np.abs(A2.cpu().numpy() - Ao)) <= TOL * np.max(np.abs(Ao))


def test_static_scratch_entry_rejects_what_does_not_fit(torch_cuda, B):
    torch = torch_cuda
    nsteps, n, k = 4000, 150, 4000   # 16 * 4016 * (256 + 4032) bytes = 275 MB: far beyond the 16 MiB array
    need = B.fourier_static_scratch_bytes(n, nsteps, k)
    assert need > B.STATIC_SCRATCH_BYTES
    z = torch.zeros((nsteps + 1, n), dtype=torch.complex128, device="cuda")
    E = torch.zeros(k, dtype=torch.float64, device="cuda")
    A = torch.full((n, k), 7.0, dtype=torch.complex128, device="cuda")
    with pytest.raises(B.ScIvrError) as e:
        B.fourier_static(z, E, 10.0, A)
    assert e.value.status == B.EINVAL
    assert str(need) in str(e.value) and str(B.STATIC_SCRATCH_BYTES) in str(e.value)
    torch.cuda.synchronize()
    assert bool((A == 7.0).all())    # rejected before anything was launched
    # the largest documented shape still goes through: 128 trajectories x 1001 samples x 896 energies
    assert B.fourier_static_scratch_bytes(128, 1000, 896) <= B.STATIC_SCRATCH_BYTES
    assert B.fourier_static_scratch_bytes(0, 10, 10) == 0 and B.fourier_static_scratch_bytes(10, -1, 10) == 0
