"""Grid sizes that are not powers of two: the mixed-radix passes of
csrc/gpe_mixed.cuh against the oracle (whose transform for these lengths is the plain DFT definition,
pinned in tests/test_oracle_fft.py).  Same tolerances as tests/test_gpu_parity.py."""
import numpy as np
import pytest

import workloads as W
from oracle import gpe_oracle
from oracle.gpe_oracle import Oracle
from tests.test_gpu_branches import _records_ok
from tests.test_gpu_parity import PER_STEP, _general_workload, _gpu_plan, _oracle_input, _rel, _to_dev, _torch

pytestmark = pytest.mark.gpu

# radices met: 96 = 8.4.3, 160 = 8.5.4, 240 = 8.5.3.2, 90 = 5.3.3.2, 250 = 5.5.5.2, 1000 = 8.5.5.5, 1536 = 8.8.8.3, 162 = 3^4.2
SIZES = [(96, 96), (160, 240), (240, 64), (128, 90), (250, 96), (162, 100), (1000, 64), (64, 1536)]


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("nx,ny", SIZES)
def test_fft2_forward_mixed_radix(nx, ny, dtype):
    """The transform alone: shifted impulse (sign, axis order), noise against the oracle, Parseval."""
    import paper_2404_14401_b200 as G
    torch = _torch()
    cd = np.complex64 if dtype == "c64" else np.complex128
    eps = 6e-8 if dtype == "c64" else 1.2e-16
    plan = G.Plan(nx, ny, 1.0, 1.0, dtype, 1)
    rng = np.random.default_rng(nx * 7 + ny)
    i0, j0 = 3, ny // 2 + 5
    imp = np.zeros((nx, ny), dtype=cd); imp[i0, j0] = 2.0 - 1.0j
    noise = (rng.standard_normal((nx, ny)) + 1j * rng.standard_normal((nx, ny))).astype(cd)
    for name, a in (("shifted impulse", imp), ("noise", noise)):
        src = torch.from_numpy(a.copy()).cuda()
        dst = torch.empty_like(src)
        G.gpe_fft2_forward(plan.plan, src.data_ptr(), dst.data_ptr())
        got = dst.cpu().numpy().astype(np.complex128)
        if name == "noise":
            want = gpe_oracle.fft2(a.astype(np.complex128))
            lhs, rhs = np.sum(np.abs(got) ** 2), nx * ny * np.sum(np.abs(a.astype(np.complex128)) ** 2)
            assert abs(lhs - rhs) <= 200 * eps * rhs
        else:
            ph = ((np.arange(nx) * i0) % nx)[:, None] / nx + ((np.arange(ny) * j0) % ny)[None, :] / ny
            want = (2.0 - 1.0j) * np.exp(-2j * np.pi * ph)
        e = _rel(got, want)
        assert e <= 40 * eps, f"{name}: {e:.3e}"
    plan.close()


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("mode", ["real", "imag"])
@pytest.mark.parametrize("nx,ny,batch", [(96, 96, 1), (160, 240, 2), (240, 64, 1), (128, 90, 1), (250, 96, 1)])
def test_per_step_parity_mixed_radix(nx, ny, batch, mode, dtype):
    """Everything switched on (2-D array, lattice ramp, cavity, g), one step and then eleven more with a record
    per step, a batch; observables at the end."""
    p = _general_workload(nx, ny, batch=batch)
    plan = _gpu_plan(p, dtype, use_separable=False)
    psi, ref = _to_dev(p["psi0"], dtype), _oracle_input(p["psi0"], dtype)
    o = Oracle(p)
    plan.evolve(psi, 1e-3, 1, mode)
    o.evolve(ref, 1e-3, 1, mode == "imag")
    e1 = _rel(psi.cpu().numpy(), ref)
    assert e1 <= PER_STEP[dtype], f"1 step: {e1:.3e}"
    rg = plan.evolve(psi, 1e-3, 11, mode, record_every=1).cpu().numpy()
    ro = o.evolve(ref, 1e-3, 11, mode == "imag", record_every=1)
    e = _rel(psi.cpu().numpy(), ref)
    assert e <= 12 * PER_STEP[dtype], f"12 steps: {e:.3e}"
    tol = 1e-5 if dtype == "c64" else 1e-10
    _records_ok(rg, ro, tol)
    og, oo = plan.observables(psi)[0], o.observables(ref)[0]
    for b in range(batch):
        for k in ("norm", "e_kin", "e_pot", "e_int", "theta"):
            assert abs(og[b][k] - oo[b][k]) <= tol * max(abs(oo[b][k]), 1e-2), (b, k)
    assert plan.step == 12
    plan.close()


def test_mixed_radix_large_and_unsupported():
    """One step at 500 x 960 in complex64 (960 = 8.8.5.3, 500 = 5.5.5.4) against the oracle;
    ordering = 1 is refused for these sizes; odd sizes and prime factors above 5 are GPE_EUNSUPPORTED."""
    import paper_2404_14401_b200 as G
    p = _general_workload(500, 960)
    plan = _gpu_plan(p, "c64")          # the trap as vx + vy on the GPU, as a 2-D array in the oracle
    psi, ref = _to_dev(p["psi0"], "c64"), _oracle_input(p["psi0"], "c64")
    plan.evolve(psi, 1e-3, 1, "real")
    Oracle(p).evolve(ref, 1e-3, 1, False)
    e = _rel(psi.cpu().numpy(), ref)
    assert e <= PER_STEP["c64"], f"{e:.3e}"
    plan.set_potential({**p, "ordering": 1})
    with pytest.raises(G.GpeError) as ex:
        plan.evolve(psi, 1e-3, 1, "real")
    assert ex.value.status == 2
    plan.close()
    for bad in ((75, 64), (98, 64), (64, 2050), (62, 64)):
        with pytest.raises(G.GpeError) as ex:
            G.gpe_plan_create(bad[0], bad[1], 1.0, 1.0, G.GPE_C64, 1)
        assert ex.value.status == 2
