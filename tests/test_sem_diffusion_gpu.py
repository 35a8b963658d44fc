"""GPU parity of crf_sem_diffusion against oracle/sem_oracle.py, through the C ABI: the fields are
what crf_rhs_pointwise produces on seeded states (Y, Wbar, lambda, rho D_k, T) on seeded affine elements.  Every
output is a difference operator applied to the fields (a small difference of large terms wherever a field is nearly
constant over an element), so the tolerance is 1e-12 of the GROSS sum of the products that cancel
(sem_oracle.sem_diffusion_scale: the same contractions with magnitudes), the analogue of S_k for omega_k."""
import numpy as np
import pytest
import torch

from oracle import sem_oracle
from paper_2409_06404_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    assert torch.cuda.is_available()
    from paper_2409_06404_b200 import binding as b
    b.lib()
    return b


def _case(binding, name, nel, seed=0):
    desc = wl.make_mechanism(name)
    gm = binding.Mechanism(desc)
    n = 512 * nel
    st = wl.make_state(name, n=n, total=n)
    rng = np.random.default_rng(100 + seed)
    h3 = rng.uniform(0.2e-3, 1.5e-3, (nel, 3))
    d = parity.to_dev(st)
    rhs = gm.rhs_pointwise(d["T"], d["p"], d["Y"], want_cpk=False)
    dY, dT = gm.sem_diffusion(torch.from_numpy(h3).cuda(), d["T"], rhs["Wbar"], d["Y"], rhs["lam"], rhs["rhoD"])
    torch.cuda.synchronize()
    args = (desc["W"], h3, st["T"], rhs["Wbar"].cpu().numpy(), st["Y"], rhs["lam"].cpu().numpy(), rhs["rhoD"].cpu().numpy())
    ref = sem_oracle.sem_diffusion(*args)
    ref["scale"] = sem_oracle.sem_diffusion_scale(*args)
    return desc, dY.cpu().numpy(), dT.cpu().numpy(), ref, nel


def _err(got, ref, scale):
    return float(np.max(np.abs(got - ref) / (1e-12 * scale + 1e-300)))


@pytest.mark.parametrize("name, nel", [("C1", 1), ("C2", 7), ("C3", 5), ("C4", 3), ("C5", 2)])
def test_sem_diffusion_parity(binding, name, nel):
    desc, dY, dT, ref, nel = _case(binding, name, nel)
    eY, eT = _err(dY, ref["dY"], ref["scale"]["dY"]), _err(dT, ref["dT"], ref["scale"]["dT"])
    print(name, nel, f"dY {eY:.3g} dT {eT:.3g} of the tolerance")
    assert eY <= 1.0 and eT <= 1.0, (eY, eT)
    # the identities of the weak form hold on the GPU result too: every residual sums to zero over its element
    # (partition of unity) and the species fluxes cancel (correction velocity, sum_k Y_k = 1)
    sc = ref["scale"]["dY"]
    assert np.all(np.abs(dY.reshape(-1, nel, 512).sum(axis=2)) <= 1e-12 * sc.reshape(-1, nel, 512).sum(axis=2))
    assert np.all(np.abs(dY.sum(axis=0)) <= 1e-12 * sc.sum(axis=0))


def test_sem_diffusion_arguments(binding):
    desc = wl.make_mechanism("C1")
    gm = binding.Mechanism(desc)
    L = binding.lib()
    z = torch.ones(512 * 9 + 8, dtype=torch.float64, device="cuda")
    p = z.data_ptr()
    assert L.crf_sem_diffusion(gm._h, p, p, p, p, p, p, 0, p, p) == 0          # nel = 0 is a no-op
    assert L.crf_sem_diffusion(gm._h, p, p, p, p, p, p, -1, p, p) == -1
    assert L.crf_sem_diffusion(gm._h, p, p, p, p, p, p, 1, p + 8, p) == -1     # misaligned
    assert L.crf_sem_diffusion(gm._h, None, p, p, p, p, p, 1, p, p) == -1
