"""-m gpu parity: CG! / propagator! through the C-ABI against the oracle's step-by-step CG (SURVEY.md 8(c)
"Algorithm CG", R11, P8-P10).  "Agree to the requested residual" is checked as P9: the ORACLE operator's
normal-equation residual of the GPU solution is <= 2 tol, and on these oracle-sized lattices the solutions
agree to 1e-8 relative (forward error <= cond * residual)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2503_16994_b200 import binding as B
from paper_2503_16994_b200 import synth

from gpu_util import Lattice, interior, round_f32, site_rel_err

pytestmark = pytest.mark.gpu

TOL = 1e-10


def oracle_normal_resid(L, U, A, b, x, kappa, bc, theta):
    r = b - oracle.dw(L, U, x, kappa, A, bc=bc, theta=theta)
    q = oracle.dw(L, U, r, kappa, A, bc=bc, theta=theta, dagger=True)
    bp = oracle.dw(L, U, b, kappa, A, bc=bc, theta=theta, dagger=True)
    return np.linalg.norm(q) / np.linalg.norm(bp), np.linalg.norm(r) / np.linalg.norm(b)


def setup(L, bc, theta, phiT, kappa, csw, seed, mixed=False):
    U = synth.smooth_gauge(L, seed)
    if bc in (B.BC_SF_ORBI, B.BC_SF_AFWB):
        U = synth.apply_sf_boundary(L, U)
    lat = Lattice(L, bc, theta, synth.SF_PHI0, phiT)
    precs = (B.F64, B.F32) if mixed else (B.F64,)
    lat.set_gauge(U, precs=precs)
    lat.build_clover(kappa, csw, precs=precs, inverse=True)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=phiT)
    return U, A, lat


def solve(lat, kappa, b_canon, eo=False, mixed=False, tol=TOL, **kw):
    b = lat.spinor(b_canon)
    x = lat.alloc(B.FIELD_SPINOR)
    ws = lat.alloc(B.FIELD_WORKSPACE)
    f32 = dict(U32=lat.U.get((B.F32, 18)), clover32=lat.A.get(B.F32), clover_inv32=lat.Ainv.get(B.F32)) if mixed else {}
    info = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], b, x, ws, tol=tol, maxiter=10000,
                      clover_inv64=lat.Ainv[B.F64], eo=eo, mixed=mixed, **f32, **kw)
    return lat.spinor_to_host(x), info


CG_CASES = [
    ((4, 4, 4, 4), B.BC_PERIODIC, (0, 0, 0, np.pi), None, 0.125, 1.0),
    ((4, 4, 4, 8), B.BC_OPEN, None, None, 0.1365, 1.9),
    ((4, 4, 4, 8), B.BC_SF_ORBI, (0.5, 0.5, 0.5, 0.0), synth.SF_PHIT, 0.1355, 1.8),
]


@pytest.mark.parametrize("L,bc,theta,phiT,kappa,csw", CG_CASES)
@pytest.mark.parametrize("mode", ["plain", "eo", "mixed", "eo_mixed"])
def test_cg_matches_oracle(L, bc, theta, phiT, kappa, csw, mode):
    U, A, lat = setup(L, bc, theta, phiT, kappa, csw, 101, mixed="mixed" in mode)
    y = (0, 0, 0, 0) if bc == B.BC_PERIODIC else (0, 0, 0, L[3] // 2)  # R12
    b = synth.point_source(L, y, 1, 2)
    xo, it_o, rn_o, rt_o = oracle.cg(L, U, b, kappa, A, bc=bc, theta=theta, tol=TOL)
    assert it_o > 0
    x, info = solve(lat, kappa, b, eo="eo" in mode, mixed="mixed" in mode)
    assert info["status"] == B.OK and info["iters"] > 0
    rn, rt = oracle_normal_resid(L, U, A, b, x, kappa, bc, theta)
    if "eo" in mode:
        # the preconditioned system's residual was driven to tol; the full system's true residual follows (P10)
        assert rt <= 50 * TOL
    else:
        assert rn <= 2 * TOL  # P9
        assert abs(info["rel_resid_normal"] - rn) <= 0.5 * rn + 1e-13
    assert abs(info["rel_resid_true"] - rt) <= 0.5 * rt + 1e-13
    assert np.linalg.norm(x - xo) / np.linalg.norm(xo) <= 1e-8
    assert np.all(x[~interior(L, bc)] == 0)  # P7: the solution vanishes on frozen slices
    if mode == "plain":
        assert abs(info["iters"] - it_o) <= 2  # same algorithm, same arithmetic up to rounding order
    lat.close()


def test_cg_gaussian_source_and_iteration_count():
    L, bc, kappa, csw = (8, 4, 6, 12), B.BC_PERIODIC, 0.13, 1.7
    U, A, lat = setup(L, bc, None, None, kappa, csw, 111)
    b = synth.gaussian_spinor(L, 112)
    xo, it_o, _, _ = oracle.cg(L, U, b, kappa, A, tol=TOL)
    for check_every in (1, 7, 16):
        x, info = solve(lat, kappa, b, check_every=check_every)
        assert abs(info["iters"] - it_o) <= 2
        assert site_rel_err(x, xo) <= 1e-7
    lat.close()


def test_cg_maxiter_and_zero_rhs():
    L, kappa = (4, 4, 4, 4), 0.125
    U, A, lat = setup(L, B.BC_PERIODIC, None, None, kappa, 1.0, 121)
    b = synth.gaussian_spinor(L, 122)
    bd = lat.spinor(b)
    x = lat.alloc(B.FIELD_SPINOR)
    ws = lat.alloc(B.FIELD_WORKSPACE)
    with pytest.raises(B.LqcdError) as e:
        B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], bd, x, ws, tol=1e-10, maxiter=3)
    assert e.value.status == B.ENOTCONV
    info = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], bd, x, ws, tol=1e-10, maxiter=3,
                      raise_on_notconv=False)
    assert info["iters"] == 3
    bd.zero_()
    info = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], bd, x, ws, tol=1e-10, maxiter=100)
    assert info["iters"] == 0
    assert torch.count_nonzero(x).item() == 0
    lat.close()


def test_propagator_12_columns():
    """propagator! point-source method: 12 columns at the origin, each against the oracle's CG."""
    L, kappa, csw = (4, 4, 4, 4), 0.125, 1.0
    theta = (0, 0, 0, np.pi)
    U, A, lat = setup(L, B.BC_PERIODIC, theta, None, kappa, csw, 131)
    nbytes = B.field_bytes(lat.g, B.FIELD_SPINOR)
    cols = torch.empty(12 * nbytes, dtype=torch.uint8, device="cuda")
    ws = lat.alloc(B.FIELD_WORKSPACE)
    infos = B.propagator(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], (0, 0, 0, 0), cols, ws, tol=TOL)
    for c in (0, 5, 11):
        b = synth.point_source(L, (0, 0, 0, 0), c // 3, c % 3)
        xo, it_o, _, _ = oracle.cg(L, U, b, kappa, A, theta=theta, tol=TOL)
        x = lat.spinor_to_host(cols[c * nbytes:(c + 1) * nbytes])
        assert np.linalg.norm(x - xo) / np.linalg.norm(xo) <= 1e-8
        assert abs(infos[c]["iters"] - it_o) <= 2
    lat.close()


@pytest.mark.parametrize("L,bc", [((8, 4, 8, 12), B.BC_PERIODIC), ((6, 4, 10, 8), B.BC_OPEN)])
@pytest.mark.parametrize("prec", [B.F64, B.F32])
def test_correlator_ps_matches_oracle(L, bc, prec):
    """NEXT-2: C(x4) of a set of columns against the oracle's plain loops (fp64 accumulation on both sides; the
    fp32 case feeds the oracle the same rounded columns), on 4^4 tiles and on a lattice without them."""
    V = synth.vol(L)
    lat = Lattice(L, bc)
    ncol = 5
    fb = B.field_bytes(lat.g, B.FIELD_SPINOR, prec)
    cols_dev = torch.empty(ncol * fb, dtype=torch.uint8, device="cuda")
    cols = []
    for c in range(ncol):
        psi = synth.gaussian_spinor(L, 300 + c)
        cols.append(round_f32(psi) if prec == B.F32 else psi)
        cols_dev[c * fb:(c + 1) * fb].copy_(lat.spinor(psi, prec))
    ws = lat.alloc(B.FIELD_WORKSPACE)
    got = np.array(B.correlator_ps(lat.g, cols_dev, ncol, ws, L[3], prec))
    ref = oracle.correlator_ps(L, np.array(cols))
    assert np.max(np.abs(got - ref) / ref) <= 1e-13
    lat.close()


def test_propagator_to_correlator_and_noise_source():
    """The paper's use of the solver: 12 point-source columns -> pseudoscalar correlator, and the
    noise-source method of propagator! (a Gaussian source on one time slice, drawn by the seeded generator and
    passed in), both against the oracle end to end."""
    L, kappa, csw = (4, 4, 4, 8), 0.125, 1.0
    theta = (0, 0, 0, np.pi)
    U, A, lat = setup(L, B.BC_PERIODIC, theta, None, kappa, csw, 141)
    V = synth.vol(L)
    nbytes = B.field_bytes(lat.g, B.FIELD_SPINOR)
    cols = torch.empty(12 * nbytes, dtype=torch.uint8, device="cuda")
    ws = lat.alloc(B.FIELD_WORKSPACE)
    B.propagator(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], (0, 0, 0, 0), cols, ws, tol=1e-12)
    got = np.array(B.correlator_ps(lat.g, cols, 12, ws, L[3]))
    ref_cols = []
    for c in range(12):
        b = synth.point_source(L, (0, 0, 0, 0), c // 3, c % 3)
        ref_cols.append(oracle.cg(L, U, b, kappa, A, theta=theta, tol=1e-12)[0])
    ref = oracle.correlator_ps(L, np.array(ref_cols))
    assert np.max(np.abs(got - ref) / ref) <= 1e-8
    assert np.all(got > 0) and got[0] == got.max()
    # noise source on time slice 2
    V3 = L[0] * L[1] * L[2]
    eta = np.zeros((V, 4, 3), dtype=np.complex128)
    eta[2 * V3:3 * V3] = synth.gaussian_spinor(L, 142)[2 * V3:3 * V3]
    x = lat.alloc(B.FIELD_SPINOR)
    info = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], lat.spinor(eta), x, ws, tol=1e-12)
    xo, it_o, _, _ = oracle.cg(L, U, eta, kappa, A, theta=theta, tol=1e-12)
    assert abs(info["iters"] - it_o) <= 2
    assert np.linalg.norm(lat.spinor_to_host(x) - xo) / np.linalg.norm(xo) <= 1e-8
    c_gpu = np.array(B.correlator_ps(lat.g, x, 1, ws, L[3]))
    c_ref = oracle.correlator_ps(L, xo[None])
    assert np.max(np.abs(c_gpu - c_ref) / c_ref) <= 1e-8
    lat.close()
