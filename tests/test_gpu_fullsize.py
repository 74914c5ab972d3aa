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


def rounded_inputs(fields):
    if "rounded" not in fields:
        fields["rounded"] = (round_f32(fields["U_host"]), round_f32(fields["psi_host"]))
    return fields["rounded"]


@pytest.mark.parametrize("prec,recon", [(B.F64, B.RECON_18), (B.F64, B.RECON_12), (B.F32, B.RECON_18), (B.F32, B.RECON_12)])
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
        # fp32 (R14): the oracle consumes the same inputs rounded once to fp32 and promoted back.  (Its clover term is
        # then formed on the fly from the rounded links, the library's in fp64 from the fp64 links and rounded: a
        # 6e-8 relative difference in A, inside the budget.)
        Uo, po = (fields["U_host"], fields["psi_host"]) if prec == B.F64 else rounded_inputs(fields)
        ref = oracle.dw_at_sites(L, Uo, po, sites, KAPPA, CSW, dagger=dagger)
        err = np.linalg.norm((got - ref).reshape(len(sites), -1), axis=1) / np.linalg.norm(ref.reshape(len(sites), -1), axis=1)
        assert err.max() <= TOL[prec], (dagger, err.max())
    fields.pop("rounded", None)
    del canon, src, dst, A, U
    torch.cuda.empty_cache()


def test_slab_decomposition_48x48x48x96_sampled(fields):
    """NEXT-3 at full size: the lattice as two 48^3 x 48 time slabs (what two ranks would hold), clover term of each
    slab from lqcd_clover_build_slab with the one-slice gauge halo, pack -> face copies -> pipeline kernel -> face
    kernel; sampled sites (plus 256 on each of the four face slices) against the oracle on the whole lattice."""
    from paper_2503_16994_b200 import slab

    P, V = 2, synth.vol(L)
    ns, T = L[0] * L[1] * L[2], L[3] // P
    Uc, psic = fields["Uc"], fields["psic"]
    rng = np.random.Generator(np.random.PCG64(synth.seed_for(5, 8)))
    face = np.concatenate([t * ns + rng.integers(0, ns, size=256) for t in (0, T - 1, T, L[3] - 1)])
    sites = np.array(sorted(set(int(s) for s in np.concatenate([sample_sites(), face]))), dtype=np.int64)
    ranks = []
    for r in range(P):
        g = slab.slab_geom_create(L, P, None)
        assert "dw_pipe_kernel" in B.dw_plan(g, B.F64, B.RECON_18, True)
        lo, hi = r * T * ns, (r + 1) * T * ns
        U = B.alloc_field(g, B.FIELD_GAUGE)
        B.gauge_import(g, Uc[lo:hi], U)
        below = Uc[((lo - ns) % V):((lo - ns) % V) + ns].contiguous()
        above = Uc[(hi % V):(hi % V) + ns].contiguous()
        A = B.alloc_field(g, B.FIELD_CLOVER)
        B.clover_build_slab(g, KAPPA, CSW, U, below, above, A)
        src, dst = B.alloc_field(g, B.FIELD_SPINOR), B.alloc_field(g, B.FIELD_SPINOR)
        B.spinor_import(g, psic[lo:hi], src)
        faces = [B.alloc_field(g, B.FIELD_FACE) for _ in range(4)]   # send_lo, send_hi, recv_lo, recv_hi
        ranks.append(dict(g=g, U=U, A=A, src=src, dst=dst, f=faces, lo=lo, hi=hi))
    canon = torch.empty((V, 4, 3), dtype=torch.complex128, device="cuda")
    for dagger, fn in ((False, B.dw_apply), (True, B.dwdag_apply)):
        for R in ranks:
            B.dw_slab_pack(R["g"], KAPPA, R["U"], R["src"], R["f"][0], R["f"][1], dagger)
        for r, R in enumerate(ranks):
            ranks[(r - 1) % P]["f"][3].copy_(R["f"][0])
            ranks[(r + 1) % P]["f"][2].copy_(R["f"][1])
        for R in ranks:
            R["dst"].fill_(0x7F)
            fn(R["g"], KAPPA, R["U"], R["A"], R["src"], R["dst"])
            B.dw_slab_faces(R["g"], KAPPA, R["U"], R["f"][2], R["f"][3], R["dst"], dagger)
            B.spinor_export(R["g"], R["dst"], canon[R["lo"]:R["hi"]])
        torch.cuda.synchronize()
        got = canon[torch.from_numpy(sites).cuda()].cpu().numpy()
        ref = oracle.dw_at_sites(L, fields["U_host"], fields["psi_host"], sites, KAPPA, CSW, dagger=dagger)
        err = np.linalg.norm((got - ref).reshape(len(sites), -1), axis=1) / np.linalg.norm(ref.reshape(len(sites), -1), axis=1)
        assert err.max() <= 1e-12, (dagger, err.max())
    for R in ranks:
        B.geom_destroy(R["g"])
    del ranks, canon
    torch.cuda.empty_cache()
