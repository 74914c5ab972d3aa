"""-m gpu parity of the twisted-mass term: D = A + 2 i kappa mu gamma5 - kappa H,
D^+ = gamma5 D(-mu) gamma5, in every stencil-kernel variant, both precisions, with and without the clover term, in
the multi-right-hand-side call, the host-buffer call and the CG solve, against the CPU oracle (pin P13).
Tolerances are north_star's (1e-12 fp64, 2e-6 fp32 per-site relative)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2503_16994_b200 import binding as B
from paper_2503_16994_b200 import synth

from gpu_util import Lattice, interior, round_f32, site_rel_err

pytestmark = pytest.mark.gpu

TOL = {B.F64: 1e-12, B.F32: 2e-6}
MODES = ["pipe", "stream", "split", "direct"]
MU = 0.37   # large enough that a dropped or sign-flipped term is far outside the tolerance

CASES = [
    ((8, 8, 8, 8), B.BC_PERIODIC, (0.3, -0.2, 0.1, np.pi), None),
    ((8, 4, 4, 12), B.BC_OPEN, (0.5, 0.5, 0.5, 0.0), None),
    ((12, 6, 10, 8), B.BC_PERIODIC, None, None),          # no 4^4 tiles: the one-thread-per-site kernels
    ((4, 4, 4, 8), B.BC_SF_ORBI, (0.5, 0.5, 0.5, 0.0), synth.SF_PHIT),
]


@pytest.fixture
def mode(request):
    B.set_option("dw_mode", request.param)
    yield request.param
    B.set_option("dw_mode", "pipe")


def inputs(L, bc, seed):
    U = synth.smooth_gauge(L, seed)
    if bc in (B.BC_SF_ORBI, B.BC_SF_AFWB):
        U = synth.apply_sf_boundary(L, U)
    return U, synth.gaussian_spinor(L, seed + 1)


def dw_tm(lat, kappa, mu, psi, prec, recon, dagger, clover=True):
    src = lat.spinor(psi, prec)
    dst = lat.alloc(B.FIELD_SPINOR, prec)
    dst.fill_(0x7F)
    fn = B.dwdag_apply if dagger else B.dw_apply
    fn(lat.g, kappa, lat.U[(prec, recon)], lat.A.get(prec) if clover else None, src, dst, prec, recon, mu=mu)
    return lat.spinor_to_host(dst, prec)


@pytest.mark.parametrize("mode", MODES, indirect=True)
@pytest.mark.parametrize("L,bc,theta,phiT", CASES)
@pytest.mark.parametrize("prec,recon", [(B.F64, B.RECON_18), (B.F32, B.RECON_12)])
def test_dw_twisted_parity(mode, L, bc, theta, phiT, prec, recon):
    kappa, csw = 0.137, 1.9
    U, psi = inputs(L, bc, 91)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=phiT)
    Uo, psio, Ao = (round_f32(U), round_f32(psi), round_f32(A)) if prec == B.F32 else (U, psi, A)
    lat = Lattice(L, bc, theta, synth.SF_PHI0, phiT)
    lat.set_gauge(U, recons=(recon,), precs=(prec,))
    lat.build_clover(kappa, csw, recon=recon, precs=(prec,))
    mask = interior(L, bc)
    for dagger in (False, True):
        for clover in (True, False):
            ref = oracle.dw(L, Uo, psio, kappa, Ao if clover else None, bc=bc, theta=theta, dagger=dagger, mu=MU)
            got = dw_tm(lat, kappa, MU, psi, prec, recon, dagger, clover)
            assert site_rel_err(got, ref, mask) <= TOL[prec]
            assert np.all(got[~mask] == 0)
    # the term is really there: mu = 0 differs from mu = MU by 2 kappa mu |psi| per site
    ref0 = oracle.dw(L, Uo, psio, kappa, Ao, bc=bc, theta=theta)
    got = dw_tm(lat, kappa, MU, psi, prec, recon, False)
    d = np.linalg.norm((got - ref0).reshape(lat.V, -1)[mask], axis=1)
    n = np.linalg.norm(psio.reshape(lat.V, -1)[mask], axis=1)
    assert np.allclose(d, 2 * kappa * MU * n, rtol=1e-4)
    lat.close()


@pytest.mark.parametrize("prec", [B.F64, B.F32])
def test_dw_multi_twisted(prec):
    L, kappa, csw, nrhs = (8, 8, 4, 8), 0.135, 1.7, 3
    U = synth.smooth_gauge(L, 93)
    A = oracle.clover_blocks(L, U, kappa, csw)
    Uo, Ao = (round_f32(U), round_f32(A)) if prec == B.F32 else (U, A)
    lat = Lattice(L)
    lat.set_gauge(U, precs=(prec,))
    lat.build_clover(kappa, csw, precs=(prec,))
    fb = B.field_bytes(lat.g, B.FIELD_SPINOR, prec)
    src = torch.empty(nrhs * fb, dtype=torch.uint8, device="cuda")
    dst = torch.empty_like(src)
    psis = [synth.gaussian_spinor(L, 94 + i) for i in range(nrhs)]
    for i, psi in enumerate(psis):
        src[i * fb:(i + 1) * fb].copy_(lat.spinor(psi, prec))
    for dagger in (False, True):
        dst.fill_(0x7F)
        B.dw_apply_multi(lat.g, kappa, lat.U[(prec, 18)], lat.A[prec], src, dst, nrhs, prec, dagger=dagger, mu=MU)
        for i, psi in enumerate(psis):
            po = round_f32(psi) if prec == B.F32 else psi
            ref = oracle.dw(L, Uo, po, kappa, Ao, dagger=dagger, mu=MU)
            assert site_rel_err(lat.spinor_to_host(dst[i * fb:(i + 1) * fb], prec), ref) <= TOL[prec]
    lat.close()


def test_dw_apply_host_twisted():
    L = (4, 4, 4, 8)
    U = synth.smooth_gauge(L, 95)
    psi = synth.gaussian_spinor(L, 96)
    A = oracle.clover_blocks(L, U, 0.135, 1.7)
    out = np.empty_like(psi)
    for dagger in (False, True):
        B.dw_apply_host(L, 0.135, 1.7, U, psi, out, dagger=dagger, mu=MU)
        assert site_rel_err(out, oracle.dw(L, U, psi, 0.135, A, dagger=dagger, mu=MU)) <= 1e-12


@pytest.mark.parametrize("mixed", [False, True])
def test_cg_twisted(mixed):
    """D(mu)^+ D(mu) x = D(mu)^+ b: the twisted mass lifts the spectrum (D^+D >= (2 kappa mu)^2 for csw = 0), so the
    solve converges in fewer iterations than at mu = 0; solution and iteration count against the oracle's CG."""
    L, kappa, csw, mu = (8, 8, 4, 8), 0.13, 1.0, 0.25
    U, b = inputs(L, B.BC_PERIODIC, 97)
    A = oracle.clover_blocks(L, U, kappa, csw)
    lat = Lattice(L)
    lat.set_gauge(U, precs=(B.F64, B.F32))
    lat.build_clover(kappa, csw, precs=(B.F64, B.F32))
    src = lat.spinor(b)
    x = lat.alloc(B.FIELD_SPINOR)
    ws = lat.alloc(B.FIELD_WORKSPACE)
    kw = dict(U32=lat.U[(B.F32, 18)], clover32=lat.A[B.F32], mixed=True) if mixed else {}
    info = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], src, x, ws, tol=1e-10, maxiter=4000, mu=mu, **kw)
    assert info["status"] == B.OK and info["rel_resid_true"] <= 2e-10
    xo, it_o, _, _ = oracle.cg(L, U, b, kappa, A, tol=1e-10, mu=mu)
    got = lat.spinor_to_host(x)
    assert np.linalg.norm(got - xo) / np.linalg.norm(xo) <= 1e-8
    if not mixed:
        assert abs(info["iters"] - it_o) <= 2
    # D(mu) x = b to the accuracy the normal-equation residual implies
    r = oracle.dw(L, U, got, kappa, A, mu=mu) - b
    assert np.linalg.norm(r) / np.linalg.norm(b) <= 1e-8
    Ai = lat.alloc(B.FIELD_CLOVER)
    B.clover_build(lat.g, kappa, csw, lat.U[(B.F64, 18)], lat.A[B.F64], Ai)
    with pytest.raises(B.LqcdError):   # even-odd + twisted mass: refused, not silently ignored
        B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], src, x, ws, clover_inv64=Ai, eo=True, mu=mu)
    lat.close()
