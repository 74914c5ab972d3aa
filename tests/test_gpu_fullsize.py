"""-m gpu parity at BASELINE.json's full size, in the launch configuration bench.py times (SURVEY.md 8(d) protocol 5):
48^3 x 96 periodic, smooth links with plaquette ~0.6 generated on the device and DOWNLOADED for the oracle (parity
always compares the same arrays), kappa = 0.137, csw = 1.9; the oracle computes D psi and D^+ psi one site at a time
(clover term on the fly) on 4096 seeded random sites plus the 16 lattice corners."""
import numpy as np
import pytest
import torch

import oracle
from paper_2503_16994_b200 import binding as B
from paper_2503_16994_b200 import synth

from gpu_util import round_f32

pytestmark = pytest.mark.gpu

L = (48, 48, 48, 96)
KAPPA, CSW = 0.137, 1.9
TOL = {B.F64: 1e-12, B.F32: 2e-6}


def sample_sites():
    rng = np.random.Generator(np.random.PCG64(synth.seed_for(5, 7)))
    V = synth.vol(L)
    sites = list(rng.integers(0, V, size=4096))
    for c in range(16):
        x = [(L[mu] - 1) if (c >> mu) & 1 else 0 for mu in range(4)]
        sites.append(synth.site_index(L, x))
    return np.array(sorted(set(int(s) for s in sites)), dtype=np.int64)


@pytest.fixture(scope="module")
def fields():
    free, _ = torch.cuda.mem_get_info()
    if free < 60 * (1 << 30):
        pytest.skip("needs ~60 GB of device memory")
    dev = torch.device("cuda", torch.cuda.current_device())
    Uc = synth.smooth_gauge_torch(L, synth.seed_for(5, 0), dev)
    psic = synth.gaussian_spinor_torch(L, synth.seed_for(5, 1), dev)
    g = B.geom_create(L)
    d = {"g": g, "Uc": Uc, "psic": psic, "U_host": Uc.cpu().numpy(), "psi_host": psic.cpu().numpy()}
    yield d
    B.geom_destroy(g)


@pytest.mark.parametrize("prec,recon", [(B.F64, B.RECON_18), (B.F64, B.RECON_12), (B.F32, B.RECON_18)])
def test_dw_48x48x48x96_sampled(fields, prec, recon):
    g = fields["g"]
    assert "dw_pipe_kernel" in B.dw_plan(g, prec, recon, True)      # the kernel bench.py times
    V = synth.vol(L)
    U64 = B.alloc_field(g, B.FIELD_GAUGE, B.F64, recon)
    B.gauge_import(g, fields["Uc"], U64, B.F64, recon)
    A = B.alloc_field(g, B.FIELD_CLOVER, prec)
    B.clover_build(g, KAPPA, CSW, U64, A, None, recon, prec)
    if prec == B.F32:
        U = B.alloc_field(g, B.FIELD_GAUGE, prec, recon)
        B.field_to_f32(g, B.FIELD_GAUGE, recon, U64, U)
        del U64
    else:
        U = U64
    src = B.alloc_field(g, B.FIELD_SPINOR, prec)
    dst = B.alloc_field(g, B.FIELD_SPINOR, prec)
    B.spinor_import(g, fields["psic"], src, prec)
    sites = sample_sites()
    canon = torch.empty((V, 4, 3), dtype=torch.complex128, device="cuda")
    for dagger, fn in ((False, B.dw_apply), (True, B.dwdag_apply)):
        dst.fill_(0x7F)
        fn(g, KAPPA, U, A, src, dst, prec, recon)
        B.spinor_export(g, dst, canon, prec)
        torch.cuda.synchronize()
        got = canon[torch.from_numpy(sites).cuda()].cpu().numpy()
        ref = oracle.dw_at_sites(L, fields["U_host"], fields["psi_host"], sites, KAPPA, CSW, dagger=dagger)
        err = np.linalg.norm((got - ref).reshape(len(sites), -1), axis=1) / np.linalg.norm(ref.reshape(len(sites), -1), axis=1)
        # fp32: the GPU consumes inputs rounded once to fp32 (R14) while this full-size oracle call uses the fp64 arrays;
        # the input rounding itself is within the same 2e-6 budget (relative 6e-8 per datum)
        assert err.max() <= TOL[prec], (dagger, err.max())
    del canon, src, dst, A, U
    torch.cuda.empty_cache()
