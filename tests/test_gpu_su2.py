"""-m gpu parity of the SU(2) fundamental representation through the C-ABI
against the N-colour oracle (oracle.sun_*, nc = 2; pinned in tests/test_oracle_su2_pins.py): layout round trip of the
Cayley-Dickson links, clover blocks, D and D^+ in both precisions, periodic (with theta) and open lattices, several tile
shapes, and the CG solve.  Tolerances are north_star's (1e-12 fp64, 2e-6 fp32 per-site relative)."""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2503_16994_b200 import binding as B
from paper_2503_16994_b200 import synth

from gpu_util import f32_storage_err, interior, round_f32, site_rel_err, to_dev

pytestmark = pytest.mark.gpu

TOL = {B.F64: 1e-12, B.F32: 2e-6}
CASES = [
    ((4, 4, 4, 4), B.BC_PERIODIC, (0, 0, 0, math.pi)),
    ((2, 2, 2, 2), B.BC_PERIODIC, (0.3, -0.2, 0.1, math.pi)),
    ((8, 8, 4, 8), B.BC_PERIODIC, (0.5, 0.5, 0.5, 0.0)),       # several 4^4 tiles
    ((12, 6, 10, 8), B.BC_PERIODIC, None),                      # 4x2x2x8-ish tiles
    ((4, 4, 4, 8), B.BC_OPEN, (0.5, 0.5, 0.5, 0.0)),
    ((8, 4, 6, 12), B.BC_OPEN, None),
]


class Su2Lattice:
    def __init__(self, L, bc, theta, Uz, kappa, csw, precs):
        self.L, self.V = L, synth.vol(L)
        self.g = B.geom_create(L, bc, theta)
        self.U, self.A = {}, {}
        Uc = to_dev(synth.su2_matrices(Uz))
        for prec in set(precs) | {B.F64}:
            self.U[prec] = B.su2_alloc_field(self.g, B.FIELD_GAUGE, prec)
            B.su2_gauge_import(self.g, Uc, self.U[prec], prec)
        for prec in precs:
            self.A[prec] = B.su2_alloc_field(self.g, B.FIELD_CLOVER, prec)
            B.su2_clover_build(self.g, kappa, csw, self.U[B.F64], self.A[prec], prec)
        torch.cuda.synchronize()

    def spinor(self, psi, prec=B.F64):
        buf = B.su2_alloc_field(self.g, B.FIELD_SPINOR, prec)
        B.su2_spinor_import(self.g, to_dev(psi), buf, prec)
        return buf

    def to_host(self, buf, prec=B.F64):
        out = torch.empty((self.V, 4, 2), dtype=torch.complex128, device="cuda")
        B.su2_spinor_export(self.g, buf, out, prec)
        torch.cuda.synchronize()
        return out.cpu().numpy()

    def close(self):
        B.geom_destroy(self.g)


@pytest.mark.parametrize("L,bc,theta", CASES)
def test_su2_layout_and_clover(L, bc, theta):
    kappa, csw = 0.1355, 1.8
    Uz = synth.haar_su2_cd(L, 201) if L == (4, 4, 4, 4) else synth.smooth_su2_cd(L, 201)
    U = synth.su2_matrices(Uz)
    lat = Su2Lattice(L, bc, theta, Uz, kappa, csw, (B.F64, B.F32))
    back = torch.empty((lat.V, 4, 2, 2), dtype=torch.complex128, device="cuda")
    B.su2_gauge_export(lat.g, lat.U[B.F64], back)
    torch.cuda.synchronize()
    assert np.array_equal(back.cpu().numpy(), U)                      # (z1, z2) kept bit-exactly, second row rebuilt
    psi = synth.gaussian_spinor_nc(L, 202, 2)
    assert np.array_equal(lat.to_host(lat.spinor(psi)), psi)
    assert np.array_equal(lat.to_host(lat.spinor(psi, B.F32), B.F32), round_f32(psi))
    ref = oracle.sun_clover_blocks(2, L, U, kappa, csw, bc=bc)
    got = torch.empty((lat.V, 2, 4, 4), dtype=torch.complex128, device="cuda")
    B.su2_clover_export(lat.g, lat.A[B.F64], got)
    torch.cuda.synchronize()
    assert np.max(np.abs(got.cpu().numpy() - ref)) <= 2e-14
    B.su2_clover_export(lat.g, lat.A[B.F32], got, B.F32)
    torch.cuda.synchronize()
    assert f32_storage_err(got.cpu().numpy(), ref) <= 0             # fp64 build, rounded once (R14)
    lat.close()


@pytest.mark.parametrize("L,bc,theta", CASES)
@pytest.mark.parametrize("prec", [B.F64, B.F32])
def test_su2_dw_parity(L, bc, theta, prec):
    kappa, csw = 0.137, 1.9
    Uz = synth.haar_su2_cd(L, 211) if L == (4, 4, 4, 4) else synth.smooth_su2_cd(L, 211)
    U = synth.su2_matrices(Uz)
    psi = synth.gaussian_spinor_nc(L, 212, 2)
    A = oracle.sun_clover_blocks(2, L, U, kappa, csw, bc=bc)
    Uo, psio, Ao = (round_f32(U), round_f32(psi), round_f32(A)) if prec == B.F32 else (U, psi, A)
    lat = Su2Lattice(L, bc, theta, Uz, kappa, csw, (prec,))
    src = lat.spinor(psi, prec)
    mask = interior(L, bc)
    for clover in (True, False):
        for dagger in (False, True):
            dst = B.su2_alloc_field(lat.g, B.FIELD_SPINOR, prec)
            dst.fill_(0x7F)
            B.su2_dw_apply(lat.g, kappa, lat.U[prec], lat.A[prec] if clover else None, src, dst, dagger, prec)
            got = lat.to_host(dst, prec)
            ref = oracle.sun_dw(2, L, Uo, psio, kappa, Ao if clover else None, bc=bc, theta=theta, dagger=dagger)
            assert site_rel_err(got, ref, mask) <= TOL[prec], (clover, dagger)
            assert np.all(got[~mask] == 0)
    assert np.array_equal(lat.to_host(src, prec), psi if prec == B.F64 else round_f32(psi))   # input untouched
    lat.close()


@pytest.mark.parametrize("L,bc,theta", [CASES[0], CASES[2], CASES[4]])
def test_su2_cg_matches_oracle(L, bc, theta):
    kappa, csw, tol = 0.125, 1.0, 1e-10
    Uz = synth.smooth_su2_cd(L, 221)
    U = synth.su2_matrices(Uz)
    A = oracle.sun_clover_blocks(2, L, U, kappa, csw, bc=bc)
    lat = Su2Lattice(L, bc, theta, Uz, kappa, csw, (B.F64,))
    y = (0, 0, 0, 0) if bc == B.BC_PERIODIC else (1, 2, 3, L[3] // 2)
    b = np.zeros((lat.V, 4, 2), dtype=np.complex128)
    b[synth.site_index(L, y), 2, 1] = 1.0
    if bc == B.BC_OPEN:
        b[synth.site_index(L, (0, 1, 0, 0)), 0, 0] = 3.0      # on a frozen slice: ignored (D7)
    xo, it_o, rn_o, rt_o = oracle.sun_cg(2, L, U, b, kappa, A, bc=bc, theta=theta, tol=tol)
    assert it_o > 0
    x = B.su2_alloc_field(lat.g, B.FIELD_SPINOR)
    ws = B.su2_alloc_field(lat.g, B.FIELD_WORKSPACE)
    for check_every in (1, 16):
        info = B.su2_cg_solve(lat.g, kappa, lat.U[B.F64], lat.A[B.F64], lat.spinor(b), x, ws, tol=tol, check_every=check_every)
        got = lat.to_host(x)
        assert info["status"] == B.OK and abs(info["iters"] - it_o) <= 2
        assert np.linalg.norm(got - xo) / np.linalg.norm(xo) <= 1e-8
        # P9: residuals of the GPU solution through the ORACLE operator
        bm = b.copy()
        bm[~interior(L, bc)] = 0
        r = bm - oracle.sun_dw(2, L, U, got, kappa, A, bc=bc, theta=theta)
        rn = np.linalg.norm(oracle.sun_dw(2, L, U, r, kappa, A, bc=bc, theta=theta, dagger=True)) / np.linalg.norm(
            oracle.sun_dw(2, L, U, bm, kappa, A, bc=bc, theta=theta, dagger=True))
        assert rn <= 2 * tol
        assert abs(info["rel_resid_true"] - np.linalg.norm(r) / np.linalg.norm(bm)) <= 0.5 * info["rel_resid_true"] + 1e-13
        assert np.all(got[~interior(L, bc)] == 0)
    with pytest.raises(B.LqcdError) as e:
        B.su2_cg_solve(lat.g, kappa, lat.U[B.F64], lat.A[B.F64], lat.spinor(b), x, ws, tol=tol, maxiter=3)
    assert e.value.status == B.ENOTCONV
    lat.close()


def test_su2_refuses_what_it_does_not_support():
    L = (4, 4, 4, 8)
    g = B.geom_create(L, B.BC_SF_ORBI, None, synth.SF_PHI0, synth.SF_PHIT)
    buf = B.su2_alloc_field(g, B.FIELD_SPINOR)
    U = B.su2_alloc_field(g, B.FIELD_GAUGE)
    out = B.su2_alloc_field(g, B.FIELD_SPINOR)
    with pytest.raises(B.LqcdError) as e:
        B.su2_dw_apply(g, 0.125, U, None, buf, out)
    assert e.value.status == B.EINVAL
    B.geom_destroy(g)
    g = B.geom_create(L)
    with pytest.raises(B.LqcdError):
        B.su2_dw_apply(g, 0.0, U, None, buf, out)          # kappa must be positive
    with pytest.raises(B.LqcdError):
        B.su2_dw_apply(g, 0.125, U, None, buf, buf)        # aliasing
    B.geom_destroy(g)
