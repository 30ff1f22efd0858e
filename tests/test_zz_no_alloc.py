"""gpe_norm_theta_noalloc (include/gpe.h): the norm / cavity-overlap reduction through the entry point that
allocates nothing (scratch in a fixed static __device__ array inside libgpe.so), against the existing path
(a plan's gpe_observables), on two calls in a row that share that array.  Collected last on purpose (the file
name): the suite runs with pytest -x.  Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu


def _setup(nx, ny, batch, dtype, seed):
    import torch
    import paper_2404_14401_b200 as G
    L = 8.0 * np.pi
    p = W._base(nx, ny, L, batch)
    p["cavity_on"], p["cavity_k"], p["eta_mode"] = 1, 4.0, 0
    p["eta_or_u"], p["delta"], p["kappa"] = np.full(batch, 1.0), np.full(batch, -1.0), np.full(batch, 0.5)
    rng = np.random.default_rng(seed)
    base = W.noisy_gaussian(nx, ny, L, L, 1.5, seed)
    psi0 = np.stack([base * (1.0 + 0.3 * b) * (1.0 + 0.2 * rng.standard_normal((nx, ny))) for b in range(batch)])
    cd = np.complex64 if dtype == "c64" else np.complex128
    psi = torch.from_numpy(np.ascontiguousarray(psi0.astype(cd))).cuda()
    plan = G.Plan(nx, ny, L, L, dtype, batch)
    plan.set_potential(p)
    return G, torch, plan, psi, L


@pytest.mark.parametrize("dtype", ["c64", "c128"])
def test_no_alloc_entry_point_matches_observables_twice(dtype):
    tol = 1e-5 if dtype == "c64" else 1e-10
    # two calls in a row on different inputs and shapes (the second smaller: stale partial sums and counters of the
    # first call are still in the shared array), each against the existing path
    for call, (nx, ny, batch, seed) in enumerate(((512, 256, 5, 3), (128, 384, 2, 4))):
        G, torch, plan, psi, L = _setup(nx, ny, batch, dtype, seed)
        out = torch.full((batch, 2), -7.0, dtype=torch.float64, device="cuda")
        dt = G.GPE_C64 if dtype == "c64" else G.GPE_C128
        before = torch.cuda.memory_allocated()
        G.gpe_norm_theta_noalloc(psi.data_ptr(), nx, ny, L, L, dt, batch, 4.0, out.data_ptr(),
                                 torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == before
        got = out.cpu().numpy()
        ref = plan.observables(psi)[0]
        for b in range(batch):
            assert abs(got[b, 0] - ref[b]["norm"]) <= tol * abs(ref[b]["norm"]), (call, b, got[b, 0], ref[b]["norm"])
            assert abs(got[b, 1] - ref[b]["theta"]) <= tol * max(abs(ref[b]["theta"]), 1e-2 * ref[b]["norm"]), (call, b)
        assert len({round(float(v), 12) for v in got[:, 0]}) == batch      # the members really differ
        plan.close()


def test_no_alloc_entry_point_limits():
    import torch
    import paper_2404_14401_b200 as G
    psi = torch.zeros((2, 64, 64), dtype=torch.complex64, device="cuda")
    out = torch.zeros((65, 2), dtype=torch.float64, device="cuda")
    for nx, ny, batch, status in ((64, 64, 65, 2), (4097, 64, 1, 2), (64, 8192, 1, 2), (0, 64, 1, 1), (64, 64, 0, 1)):
        with pytest.raises(G.GpeError) as e:
            G.gpe_norm_theta_noalloc(psi.data_ptr(), nx, ny, 1.0, 1.0, G.GPE_C64, batch, 1.0, out.data_ptr())
        assert e.value.status == status, (nx, ny, batch)
    with pytest.raises(G.GpeError) as e:
        G.gpe_norm_theta_noalloc(0, 64, 64, 1.0, 1.0, G.GPE_C64, 1, 1.0, out.data_ptr())
    assert e.value.status == 1
    with pytest.raises(G.GpeError) as e:
        G.gpe_norm_theta_noalloc(psi.data_ptr(), 64, 64, 1.0, 1.0, G.GPE_C64, 65, 1.0, out.data_ptr())
    assert "64" in str(e.value) and "4096" in str(e.value)
