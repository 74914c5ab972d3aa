"""-m gpu parity: layout, clover builder, Dw / Dw^+ and the even-odd operator against the CPU oracle,
element by element on the same seeded inputs, through the C-ABI (tolerances
are north_star's: 1e-12 per-site relative for fp64, 2e-6 for fp32)."""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2503_16994_b200 import binding as B
from paper_2503_16994_b200 import synth

from gpu_util import Lattice, coords, f32_storage_err, interior, round_f32, site_rel_err, to_dev

pytestmark = pytest.mark.gpu

TOL = {B.F64: 1e-12, B.F32: 2e-6}
PI = math.pi

# (L, bc, theta, phiT): small lattices that still span several tiles and odd tile counts
CASES = [
    ((4, 4, 4, 4), B.BC_PERIODIC, (0, 0, 0, PI), None),
    ((2, 2, 2, 2), B.BC_PERIODIC, (0.3, -0.2, 0.1, PI), None),
    ((12, 6, 10, 8), B.BC_PERIODIC, (0.5, 0.5, 0.5, 0.0), None),
    ((4, 4, 4, 8), B.BC_OPEN, None, None),
    ((8, 4, 6, 12), B.BC_OPEN, (0.5, 0.5, 0.5, 0.0), None),
    ((4, 4, 4, 8), B.BC_SF_ORBI, (0.5, 0.5, 0.5, 0.0), synth.SF_PHIT),
    ((6, 8, 4, 6), B.BC_SF_AFWB, (0.5, 0.5, 0.5, 0.0), synth.SF_PHIT),
]


def make_inputs(L, bc, seed, haar=False):
    U = synth.haar_gauge(L, seed) if haar else synth.smooth_gauge(L, seed)
    if bc in (B.BC_SF_ORBI, B.BC_SF_AFWB):
        U = synth.apply_sf_boundary(L, U)
    psi = synth.gaussian_spinor(L, seed + 1)
    return U, psi


def test_config1_4to4_haar_fp64():
    """configs[0]: 4^4, Haar links, antiperiodic time (theta_4 = pi), kappa=0.125, csw=1.0, fp64."""
    L = (4, 4, 4, 4)
    theta = (0, 0, 0, PI)
    U = synth.haar_gauge(L, synth.seed_for(1, 0))
    psi = synth.gaussian_spinor(L, synth.seed_for(1, 1))
    A = oracle.clover_blocks(L, U, 0.125, 1.0)
    lat = Lattice(L, B.BC_PERIODIC, theta)
    lat.set_gauge(U)
    lat.build_clover(0.125, 1.0)
    for dagger in (False, True):
        ref = oracle.dw(L, U, psi, 0.125, A, theta=theta, dagger=dagger)
        got = lat.dw(0.125, psi, dagger=dagger)
        assert site_rel_err(got, ref) <= 1e-12
    lat.close()


def test_layout_roundtrip():
    L = (12, 6, 10, 8)
    U = synth.smooth_gauge(L, 11)
    psi = synth.gaussian_spinor(L, 12)
    lat = Lattice(L)
    dU = to_dev(U)
    for prec in (B.F64, B.F32):
        for recon in (B.RECON_18, B.RECON_12):
            buf = lat.alloc(B.FIELD_GAUGE, prec, recon)
            B.gauge_import(lat.g, dU, buf, prec, recon)
            back = torch.empty_like(dU)
            B.gauge_export(lat.g, buf, back, prec, recon)
            torch.cuda.synchronize()
            got = back.cpu().numpy()
            if prec == B.F64 and recon == B.RECON_18:
                assert np.array_equal(got, U)  # bit-exact
            elif prec == B.F64:
                assert np.array_equal(got[:, :, :2], U[:, :, :2])
                assert np.max(np.abs(got - U)) < 1e-14  # row 3 = conj(row1 x row2), R16
            else:
                assert np.max(np.abs(got - U)) < 3e-7
        got = lat.spinor_to_host(lat.spinor(psi, prec), prec)
        if prec == B.F64:
            assert np.array_equal(got, psi)
        else:
            assert np.array_equal(got, round_f32(psi))
    assert torch.equal(dU.cpu(), torch.from_numpy(U))  # input untouched
    lat.close()


@pytest.mark.parametrize("L,bc,theta,phiT", CASES)
def test_clover_build(L, bc, theta, phiT):
    U, _ = make_inputs(L, bc, 21, haar=(L == (4, 4, 4, 4)))
    kappa, csw = 0.1355, 1.8
    ref = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=phiT)
    lat = Lattice(L, bc, theta, synth.SF_PHI0, phiT)
    lat.set_gauge(U, recons=(B.RECON_18, B.RECON_12))
    for recon in (B.RECON_18, B.RECON_12):
        lat.build_clover(kappa, csw, recon=recon, inverse=True)
        got = lat.clover_to_host(lat.A[B.F64])
        assert np.max(np.abs(got - ref)) <= 2e-14
        gi = lat.clover_to_host(lat.Ainv[B.F64])
        ri = oracle.clover_inverse(L, ref)
        assert np.max(np.abs(gi - ri)) <= 1e-12
    # fp32 storage = fp64 build rounded once (R14)
    lat.build_clover(kappa, csw, precs=(B.F32,))
    got32 = lat.clover_to_host(lat.A[B.F32], B.F32)
    assert f32_storage_err(got32, ref) <= 0
    lat.close()


def test_clover_ct_term():
    """R10: c~_t != 1 adds 2 kappa (ct-1) on the slices next to the frozen ones."""
    L, bc = (4, 4, 4, 8), B.BC_OPEN
    U, _ = make_inputs(L, bc, 23)
    ref = oracle.clover_blocks(L, U, 0.13, 1.5, bc=bc, ct=1.2)
    lat = Lattice(L, bc)
    lat.set_gauge(U)
    lat.build_clover(0.13, 1.5, ct=1.2)
    assert np.max(np.abs(lat.clover_to_host(lat.A[B.F64]) - ref)) <= 2e-14
    lat.close()


@pytest.mark.parametrize("L,bc,theta,phiT", CASES)
@pytest.mark.parametrize("prec", [B.F64, B.F32])
@pytest.mark.parametrize("recon", [B.RECON_18, B.RECON_12])
def test_dw_parity(L, bc, theta, phiT, prec, recon):
    kappa, csw = 0.1365, 1.9
    U, psi = make_inputs(L, bc, 31)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=phiT)
    if prec == B.F32:
        Uo, psio, Ao = round_f32(U), round_f32(psi), round_f32(A)
    else:
        Uo, psio, Ao = U, psi, A
    lat = Lattice(L, bc, theta, synth.SF_PHI0, phiT)
    lat.set_gauge(U, recons=(recon,), precs=(prec,))
    lat.build_clover(kappa, csw, recon=recon, precs=(prec,))
    mask = interior(L, bc)
    for dagger in (False, True):
        ref = oracle.dw(L, Uo, psio, kappa, Ao, bc=bc, theta=theta, dagger=dagger)
        got = lat.dw(kappa, psi, prec, recon, dagger)
        assert site_rel_err(got, ref, mask) <= TOL[prec]
        assert np.all(got[~mask] == 0)  # frozen slices: exactly zero (D7)
    # clover == NULL is the plain Wilson operator (csw term absent until Csw! is called)
    ref = oracle.dw(L, Uo, psio, kappa, None, bc=bc, theta=theta)
    got = lat.dw(kappa, psi, prec, recon, clover=False)
    assert site_rel_err(got, ref, mask) <= TOL[prec]
    lat.close()


def test_dw_inputs_unchanged_and_aliasing():
    L = (4, 4, 4, 8)
    U, psi = make_inputs(L, B.BC_PERIODIC, 41)
    lat = Lattice(L)
    lat.set_gauge(U)
    lat.build_clover(0.13, 1.7)
    src = lat.spinor(psi)
    dst = lat.alloc(B.FIELD_SPINOR)
    keep = [t.clone() for t in (lat.U[(B.F64, 18)], lat.A[B.F64], src)]
    B.dw_apply(lat.g, 0.13, lat.U[(B.F64, 18)], lat.A[B.F64], src, dst)
    B.dwdag_apply(lat.g, 0.13, lat.U[(B.F64, 18)], lat.A[B.F64], src, dst)
    torch.cuda.synchronize()
    for a, b in zip(keep, (lat.U[(B.F64, 18)], lat.A[B.F64], src)):
        assert torch.equal(a, b)
    with pytest.raises(B.LqcdError) as e:
        B.dw_apply(lat.g, 0.13, lat.U[(B.F64, 18)], lat.A[B.F64], src, src)
    assert e.value.status == B.EINVAL
    lat.close()


def test_geom_errors():
    with pytest.raises(B.LqcdError) as e:
        B.geom_create((4, 4, 3, 4))
    assert e.value.status == B.EINVAL
    with pytest.raises(B.LqcdError):
        B.geom_create((4, 4, 4, 2), B.BC_OPEN)
    with pytest.raises(B.LqcdError):
        B.geom_create((4, 4, 4, 4), 7)


@pytest.mark.parametrize("bc,phiT", [(B.BC_OPEN, None), (B.BC_SF_ORBI, synth.SF_PHIT)])
def test_P7_frozen_slices_do_not_leak(bc, phiT):
    """NaN stored on the frozen slices of the input (and, open BC, in the wrap-around time links)
    must not reach the output: the kernel masks, it does not multiply by zero."""
    L = (4, 4, 4, 8)
    U, psi = make_inputs(L, bc, 51)
    mask = interior(L, bc)
    A = oracle.clover_blocks(L, U, 0.13, 1.6, bc=bc, phiT=phiT)
    ref = oracle.dw(L, U, psi, 0.13, A, bc=bc)
    psi_bad = psi.copy()
    psi_bad[~mask] = np.nan
    U_bad = U.copy()
    if bc == B.BC_OPEN:
        last = coords(L)[:, 3] == L[3] - 1
        U_bad[last, 3] = np.nan
    lat = Lattice(L, bc, None, synth.SF_PHI0, phiT)
    lat.set_gauge(U_bad)
    lat.build_clover(0.13, 1.6)
    got = lat.dw(0.13, psi_bad)
    assert np.all(np.isfinite(got))
    assert site_rel_err(got, ref, mask) <= 1e-12
    assert np.all(got[~mask] == 0)
    lat.close()


@pytest.mark.parametrize("L,bc,theta,phiT", CASES[2:])
@pytest.mark.parametrize("prec", [B.F64, B.F32])
def test_dw_eo_parity(L, bc, theta, phiT, prec):
    kappa, csw = 0.1355, 1.8
    U, psi = make_inputs(L, bc, 61)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=phiT)
    Ai = oracle.clover_inverse(L, A)
    if prec == B.F32:
        Uo, psio, Ao, Aio = round_f32(U), round_f32(psi), round_f32(A), round_f32(Ai)
    else:
        Uo, psio, Ao, Aio = U, psi, A, Ai
    even = (coords(L).sum(axis=1) % 2 == 0) & interior(L, bc)
    lat = Lattice(L, bc, theta, synth.SF_PHI0, phiT)
    lat.set_gauge(U, precs=(prec,))
    lat.build_clover(kappa, csw, precs=(prec,), inverse=True)
    src = lat.spinor(psi, prec)
    tmp = lat.alloc(B.FIELD_SPINOR, prec)
    for dagger in (False, True):
        ref = oracle.dhat(L, Uo, psio, kappa, Ao, Aio, bc=bc, theta=theta, dagger=dagger)
        dst = lat.alloc(B.FIELD_SPINOR, prec)
        dst.zero_()
        B.dw_eo_apply(lat.g, kappa, lat.U[(prec, 18)], lat.A[prec], lat.Ainv[prec], src, dst, tmp, dagger, prec)
        got = lat.spinor_to_host(dst, prec)
        assert site_rel_err(got, ref, even) <= TOL[prec] * 2
    lat.close()


def test_dw_apply_host_end_to_end():
    L = (4, 4, 4, 8)
    U, psi = make_inputs(L, B.BC_PERIODIC, 71)
    A = oracle.clover_blocks(L, U, 0.135, 1.7)
    ref = oracle.dw(L, U, psi, 0.135, A)
    out = np.empty_like(psi)
    B.dw_apply_host(L, 0.135, 1.7, U, psi, out)
    assert site_rel_err(out, ref) <= 1e-12
    out32 = np.empty_like(psi)
    B.dw_apply_host(L, 0.135, 1.7, U, psi, out32, prec=B.F32, recon=B.RECON_12)
    ref32 = oracle.dw(L, round_f32(U), round_f32(psi), 0.135, round_f32(A))
    assert site_rel_err(out32, ref32) <= 2e-6


def test_blas_reductions():
    L = (8, 4, 6, 12)
    a = synth.gaussian_spinor(L, 81)
    b = synth.gaussian_spinor(L, 82)
    lat = Lattice(L)
    ws = lat.alloc(B.FIELD_WORKSPACE)
    for prec in (B.F64, B.F32):
        da, db = lat.spinor(a, prec), lat.spinor(b, prec)
        ao, bo = (a, b) if prec == B.F64 else (round_f32(a), round_f32(b))
        n2 = B.spinor_norm2(lat.g, da, ws, prec=prec)
        assert abs(n2 - np.vdot(ao, ao).real) <= 1e-12 * n2
        d = B.spinor_dot(lat.g, da, db, ws, prec=prec)
        assert abs(d - np.vdot(ao, bo)) <= 1e-12 * n2
        # run-to-run bit reproducibility (fixed-order reduction)
        assert B.spinor_norm2(lat.g, da, ws, prec=prec) == n2
    lat.close()


@pytest.mark.parametrize("L,bc,theta,phiT", [c for c in CASES if c[0] != (2, 2, 2, 2)])
@pytest.mark.parametrize("slab", [0, 1, 3])
def test_dw_apply_host_time_slabs(L, bc, theta, phiT, slab):
    """The host path stages the gauge field in time slabs and builds the clover term slab by slab as the neighbours
    arrive (slab = 3 leaves a ragged last slab; 1 = slice by slice; 0 = automatic, one slab on these small lattices):
    same result as the oracle for every boundary condition; the cached context is reused by the second call and
    rebuilt when the lattice or the slab size changes."""
    kappa, csw, ct = 0.1355, 1.8, (1.0 if bc == B.BC_PERIODIC else 1.15)
    U, psi = make_inputs(L, bc, 171)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=phiT, ct=ct)
    mask = interior(L, bc)
    B.set_option("host_slab", str(slab))
    try:
        for rep, (prec, recon) in enumerate(((B.F64, B.RECON_18), (B.F64, B.RECON_18), (B.F32, B.RECON_12))):
            for dagger in (False, True):
                out = np.full_like(psi, np.nan)
                B.dw_apply_host(L, kappa, csw, U, psi, out, bc=bc, theta=theta, phi0=synth.SF_PHI0, phiT=phiT,
                                dagger=dagger, prec=prec, recon=recon, ct=ct)
                if prec == B.F64:
                    ref = oracle.dw(L, U, psi, kappa, A, bc=bc, theta=theta, dagger=dagger)
                else:
                    ref = oracle.dw(L, round_f32(U), round_f32(psi), kappa, round_f32(A), bc=bc, theta=theta, dagger=dagger)
                assert site_rel_err(out, ref, mask) <= TOL[prec]
                assert np.all(out[~mask] == 0)
    finally:
        B.set_option("host_slab", "0")
        B.host_cache_release()
