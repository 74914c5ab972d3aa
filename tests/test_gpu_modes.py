"""-m gpu parity of every stencil-kernel variant ("dw_mode": pipe, stream, split, direct) against the CPU oracle
on lattices cut into several 4^4 tiles in every direction -- the shape the warp-specialised pipeline kernel
(dw_pipe_kernel: TMA ring + LDGSTS halo gathers) needs -- for all boundary conditions, both precisions, both link
formats, D and D^+, with and without the clover term, and through a CG solve (the fused epilogues).
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
KERNEL = {"pipe": "dw_pipe_kernel", "stream": "dw_kernel<", "split": "dw_kernel_h<", "direct": "dw_kernel<"}

# several 4^4 tiles per direction, unequal tile counts, odd tile counts (3 along one axis)
CASES = [
    ((8, 8, 8, 8), B.BC_PERIODIC, (0.3, -0.2, 0.1, np.pi), None),
    ((8, 4, 12, 8), B.BC_OPEN, (0.5, 0.5, 0.5, 0.0), None),
    ((4, 8, 8, 12), B.BC_SF_ORBI, (0.5, 0.5, 0.5, 0.0), synth.SF_PHIT),
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


@pytest.mark.parametrize("mode", MODES, indirect=True)
@pytest.mark.parametrize("L,bc,theta,phiT", CASES)
@pytest.mark.parametrize("prec,recon", [(B.F64, B.RECON_18), (B.F64, B.RECON_12), (B.F32, B.RECON_18), (B.F32, B.RECON_12)])
def test_dw_parity_every_kernel(mode, L, bc, theta, phiT, prec, recon):
    kappa, csw = 0.137, 1.9
    U, psi = inputs(L, bc, 61)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=phiT)
    Uo, psio, Ao = (round_f32(U), round_f32(psi), round_f32(A)) if prec == B.F32 else (U, psi, A)
    lat = Lattice(L, bc, theta, synth.SF_PHI0, phiT)
    assert B.geom_info(lat.g)[0] == [4, 4, 4, 4]
    assert KERNEL[mode] in B.dw_plan(lat.g, prec, recon, True)
    lat.set_gauge(U, recons=(recon,), precs=(prec,))
    lat.build_clover(kappa, csw, recon=recon, precs=(prec,))
    mask = interior(L, bc)
    for dagger in (False, True):
        ref = oracle.dw(L, Uo, psio, kappa, Ao, bc=bc, theta=theta, dagger=dagger)
        got = lat.dw(kappa, psi, prec, recon, dagger)
        assert site_rel_err(got, ref, mask) <= TOL[prec]
        assert np.all(got[~mask] == 0)
    ref = oracle.dw(L, Uo, psio, kappa, None, bc=bc, theta=theta)
    got = lat.dw(kappa, psi, prec, recon, clover=False)
    assert site_rel_err(got, ref, mask) <= TOL[prec]
    lat.close()


@pytest.mark.parametrize("mode", MODES, indirect=True)
def test_cg_every_kernel(mode):
    """The fused epilogues (|Dp|^2 in the D kernel; r -= alpha D^+t and |r|^2 in the D^+ kernel) of each variant:
    a full CG solve must reach the requested residual and agree with the oracle's solution."""
    L, kappa, csw = (8, 8, 4, 8), 0.125, 1.0
    U, b = inputs(L, B.BC_PERIODIC, 71)
    A = oracle.clover_blocks(L, U, kappa, csw)
    lat = Lattice(L)
    lat.set_gauge(U)
    lat.build_clover(kappa, csw)
    src = lat.spinor(b)
    x = lat.alloc(B.FIELD_SPINOR)
    ws = lat.alloc(B.FIELD_WORKSPACE)
    info = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], src, x, ws, tol=1e-10, maxiter=4000)
    assert info["status"] == B.OK and info["rel_resid_normal"] <= 1e-10
    xo, it_o, _, _ = oracle.cg(L, U, b, kappa, A, tol=1e-10)
    got = lat.spinor_to_host(x)
    assert np.linalg.norm(got - xo) / np.linalg.norm(xo) <= 1e-8
    assert abs(info["iters"] - it_o) <= 2
    lat.close()


def test_plan_and_option_errors():
    lat = Lattice((8, 8, 8, 8))
    assert "dw_pipe_kernel<double,18,1>" in B.dw_plan(lat.g)
    assert "ring_slots=3" in B.dw_plan(lat.g)                       # fp64: 3 x 36 KB stages + 2 x 33 KB halos + 48 KB tile
    assert "dw_pipe_half_kernel<float,12,1>" in B.dw_plan(lat.g, B.F32, B.RECON_12, True, parity=1)   # even-odd pass
    with pytest.raises(B.LqcdError):
        B.set_option("dw_mode", "bogus")
    with pytest.raises(B.LqcdError):
        B.set_option("nonsense", "1")
    lat.close()
    small = Lattice((12, 6, 10, 8))    # extents not divisible by 4: no 4^4 tiles, the pipeline does not apply
    assert "dw_pipe_kernel" not in B.dw_plan(small.g)
    small.close()


@pytest.mark.parametrize("mode", ["pipe", "stream"], indirect=True)
@pytest.mark.parametrize("prec", [B.F64, B.F32])
@pytest.mark.parametrize("nrhs,grid", [(3, 0), (8, 0), (8, 5)])
def test_dw_apply_multi(mode, prec, nrhs, grid):
    """several right-hand sides in one pass share the links and clover blocks; the result
    is the oracle's for every column and bit-identical to separate lqcd_dw_apply calls.  The pipeline kernel shares a
    tile's columns out over up to four work units (3 columns: three units of one; 8: four units of two); with a grid
    of 5 CTAs every CTA walks many units."""
    L, bc, theta, kappa, csw = (8, 4, 8, 12), B.BC_OPEN, (0.5, 0.5, 0.5, 0.0), 0.137, 1.9
    B.set_option("pipe_grid", str(grid))
    U = synth.smooth_gauge(L, 81)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc)
    psis = [synth.gaussian_spinor(L, 82 + n) for n in range(nrhs)]
    Uo, Ao = (round_f32(U), round_f32(A)) if prec == B.F32 else (U, A)
    lat = Lattice(L, bc, theta)
    lat.set_gauge(U, precs=(prec,))
    lat.build_clover(kappa, csw, precs=(prec,))
    fb = B.field_bytes(lat.g, B.FIELD_SPINOR, prec)
    src = torch.empty(nrhs * fb, dtype=torch.uint8, device="cuda")
    dst = torch.full((nrhs * fb,), 0x7F, dtype=torch.uint8, device="cuda")
    for n in range(nrhs):
        src[n * fb:(n + 1) * fb].copy_(lat.spinor(psis[n], prec))
    mask = interior(L, bc)
    for dagger in (False, True):
        B.dw_apply_multi(lat.g, kappa, lat.U[(prec, 18)], lat.A[prec], src, dst, nrhs, prec, dagger=dagger)
        for n in range(nrhs):
            got = lat.spinor_to_host(dst[n * fb:(n + 1) * fb], prec)
            po = round_f32(psis[n]) if prec == B.F32 else psis[n]
            ref = oracle.dw(L, Uo, po, kappa, Ao, bc=bc, theta=theta, dagger=dagger)
            assert site_rel_err(got, ref, mask) <= TOL[prec]
            single = lat.alloc(B.FIELD_SPINOR, prec)
            fn = B.dwdag_apply if dagger else B.dw_apply
            fn(lat.g, kappa, lat.U[(prec, 18)], lat.A[prec], src[n * fb:(n + 1) * fb], single, prec)
            torch.cuda.synchronize()
            assert torch.equal(single, dst[n * fb:(n + 1) * fb])
    B.set_option("pipe_grid", "0")
    with pytest.raises(B.LqcdError):   # overlapping arrays
        B.dw_apply_multi(lat.g, kappa, lat.U[(prec, 18)], lat.A[prec], src, src[fb:], 2, prec)
    lat.close()


@pytest.mark.parametrize("nrhs", [1, 7, 64])
def test_dw_apply_multi_column_counts(nrhs):
    """The limits of lqcd_dw_apply_multi: one column, a prime number of columns (no split into work units possible), the
    maximum of 64 (four work units of 16) -- each column bit-identical to a single application -- and 0 / 65 rejected."""
    L, kappa, csw = (8, 8, 4, 8), 0.137, 1.9
    dev = torch.device("cuda", torch.cuda.current_device())
    lat = Lattice(L)
    lat.set_gauge(synth.smooth_gauge_torch(L, 91, dev))
    lat.build_clover(kappa, csw)
    fb = B.field_bytes(lat.g, B.FIELD_SPINOR)
    src = torch.empty(nrhs * fb, dtype=torch.uint8, device="cuda")
    dst = torch.full((nrhs * fb,), 0x7F, dtype=torch.uint8, device="cuda")
    for n in range(nrhs):
        src[n * fb:(n + 1) * fb].copy_(lat.spinor(synth.gaussian_spinor_torch(L, 92 + n, dev)))
    B.dw_apply_multi(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], src, dst, nrhs)
    single = lat.alloc(B.FIELD_SPINOR)
    for n in range(nrhs):
        B.dw_apply(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], src[n * fb:(n + 1) * fb], single)
        torch.cuda.synchronize()
        assert torch.equal(single, dst[n * fb:(n + 1) * fb]), n
    for bad in (0, 65):
        with pytest.raises(B.LqcdError):
            B.dw_apply_multi(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], src, dst, bad)
    lat.close()


def test_kappa_must_be_positive():
    """kappa <= 0 (or not finite) is refused by every operator / solver entry point instead of producing NaN on the
    pipeline kernel (which folds the diagonal term in as -(1/kappa) A psi) and A psi on the others."""
    L = (4, 4, 4, 4)
    U, psi = inputs(L, B.BC_PERIODIC, 91)
    lat = Lattice(L)
    lat.set_gauge(U)
    lat.build_clover(0.125, 1.0)
    src, dst = lat.spinor(psi), lat.alloc(B.FIELD_SPINOR)
    ws = lat.alloc(B.FIELD_WORKSPACE)
    for kappa in (0.0, -0.1, float("inf"), float("nan")):
        with pytest.raises(B.LqcdError) as e:
            B.dw_apply(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], src, dst)
        assert e.value.status == B.EINVAL
        with pytest.raises(B.LqcdError) as e:
            B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], src, dst, ws)
        assert e.value.status == B.EINVAL
    lat.close()


@pytest.mark.parametrize("mode", ["split", "stream"], indirect=True)
def test_cg_partial_buffer_split_grid(mode):
    """16x16x16x6: tiles of 64 sites per parity and 192 tiles, so that dw_mode = split launches 2 * ntiles = 384 CTAs,
    each writing one partial sum of the fused CG epilogues -- more than ntiles and more than the BLAS-1 grids; the
    workspace's partial-sum buffer has to hold them (the solution is compared with the oracle's CG)."""
    L, kappa, csw = (16, 16, 16, 6), 0.13, 1.5
    U, _ = inputs(L, B.BC_PERIODIC, 95)
    A = oracle.clover_blocks(L, U, kappa, csw)
    lat = Lattice(L)
    lat.set_gauge(U)
    lat.build_clover(kappa, csw)
    b = synth.point_source(L, (3, 2, 1, 4), 2, 1)
    xo, it_o, _, _ = oracle.cg(L, U, b, kappa, A, tol=1e-10)
    x, ws = lat.alloc(B.FIELD_SPINOR), lat.alloc(B.FIELD_WORKSPACE)
    info = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], lat.spinor(b), x, ws, tol=1e-10)
    assert abs(info["iters"] - it_o) <= 2
    xg = lat.spinor_to_host(x)
    assert np.linalg.norm(xg - xo) / np.linalg.norm(xo) <= 1e-8
    lat.close()


@pytest.mark.parametrize("eo", [False, True])
def test_cg_source_on_frozen_slice_is_ignored(eo):
    """D7: the solve lives on the interior.  Components of b on frozen slices are ignored by both solver branches: a
    source with support on the frozen slice as well gives the solution and the residuals of its interior part."""
    L, bc, kappa, csw = (4, 4, 4, 8), B.BC_OPEN, 0.13, 1.5
    U, _ = inputs(L, bc, 97)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc)
    lat = Lattice(L, bc)
    lat.set_gauge(U)
    lat.build_clover(kappa, csw, inverse=True)
    b_in = synth.point_source(L, (1, 2, 3, 4), 0, 1)
    b = b_in + 5.0 * synth.point_source(L, (0, 1, 0, 0), 3, 2) + 2.0 * synth.point_source(L, (2, 1, 0, L[3] - 1), 1, 0)
    xo, _, _, rt_o = oracle.cg(L, U, b_in, kappa, A, bc=bc, tol=1e-10)
    x, ws = lat.alloc(B.FIELD_SPINOR), lat.alloc(B.FIELD_WORKSPACE)
    info = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], lat.spinor(b), x, ws, tol=1e-10,
                      clover_inv64=lat.Ainv[B.F64], eo=eo)
    xg = lat.spinor_to_host(x)
    assert np.linalg.norm(xg - xo) / np.linalg.norm(xo) <= 1e-8
    assert info["rel_resid_true"] <= 50e-10
    # a source living on frozen slices only: x = 0, converged at once
    bz = synth.point_source(L, (0, 1, 0, 0), 3, 2)
    info = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], lat.spinor(bz), x, ws, tol=1e-10,
                      clover_inv64=lat.Ainv[B.F64], eo=eo)
    assert info["iters"] == 0 and torch.count_nonzero(x).item() == 0
    lat.close()


@pytest.mark.parametrize("grid", [1, 2, 5])
@pytest.mark.parametrize("prec,recon", [(B.F64, B.RECON_18), (B.F32, B.RECON_12)])
def test_pipeline_rings_many_wraps(grid, prec, recon):
    """compute-sanitizer is closed on this GPU pool, so the hand-rolled mbarrier rings of dw_pipe_kernel (stage ring,
    halo ring, spinor buffer, tile queue) are stressed instead: with 1, 2 or 5 CTAs for 128 tiles each CTA walks up to
    128 tiles -- 1024 ring stages, every slot and both phase parities hundreds of times, the tile counter drawn 127
    times -- and the result must still be the oracle's, for D and D^+ and through the fused CG epilogues."""
    L, bc, theta, kappa, csw = (16, 8, 8, 16), B.BC_OPEN, (0.5, 0.5, 0.5, 0.0), 0.137, 1.9
    U, psi = inputs(L, bc, 71)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc)
    Uo, psio, Ao = (round_f32(U), round_f32(psi), round_f32(A)) if prec == B.F32 else (U, psi, A)
    lat = Lattice(L, bc, theta)
    lat.set_gauge(U, recons=(recon,), precs=(prec,))
    lat.build_clover(kappa, csw, recon=recon, precs=(prec,))
    assert B.geom_info(lat.g)[1] == [4, 2, 2, 4]
    B.set_option("pipe_grid", str(grid))
    try:
        assert "grid=%d " % grid in B.dw_plan(lat.g, prec, recon, True)
        mask = interior(L, bc)
        for dagger in (False, True):
            ref = oracle.dw(L, Uo, psio, kappa, Ao, bc=bc, theta=theta, dagger=dagger)
            for rep in range(2):   # twice: the self-resetting tile counter must be back at zero
                got = lat.dw(kappa, psi, prec, recon, dagger)
                assert site_rel_err(got, ref, mask) <= TOL[prec]
                assert np.all(got[~mask] == 0)
        if prec == B.F64:
            b = synth.point_source(L, (3, 2, 1, 8), 1, 1)
            xo, it_o, _, _ = oracle.cg(L, U, b, kappa, A, bc=bc, theta=theta, tol=1e-9, maxiter=400)
            x, ws = lat.alloc(B.FIELD_SPINOR), lat.alloc(B.FIELD_WORKSPACE)
            info = B.cg_solve(lat.g, kappa, lat.U[(B.F64, recon)], lat.A[B.F64], lat.spinor(b), x, ws, tol=1e-9,
                              maxiter=400, recon=recon, raise_on_notconv=False)
            assert abs(info["iters"] - abs(it_o)) <= 2
    finally:
        B.set_option("pipe_grid", "0")
    lat.close()


@pytest.mark.parametrize("mode", MODES, indirect=True)
@pytest.mark.parametrize("prec", [B.F64, B.F32])
def test_no_write_outside_the_output(mode, prec):
    """Out-of-bounds evidence without a sanitizer: every field lives inside one allocation between poisoned guard
    bands; after D, D^+ and a CG solve in each kernel variant the guards and all the INPUT fields are bit-unchanged."""
    L, kappa, csw = (8, 8, 4, 8), 0.13, 1.5
    U, psi = inputs(L, B.BC_PERIODIC, 75)
    lat = Lattice(L)
    lat.set_gauge(U, precs=(prec,))
    lat.build_clover(kappa, csw, precs=(prec,))
    G = 1 << 16   # guard bytes on both sides
    nb = B.field_bytes(lat.g, B.FIELD_SPINOR, prec)
    def guarded(n):
        buf = torch.full((n + 2 * G,), 0xA5, dtype=torch.uint8, device="cuda")
        return buf, buf[G:G + n]
    src_all, src = guarded(nb)
    dst_all, dst = guarded(nb)
    src.copy_(lat.spinor(psi, prec))
    Ucopy, Acopy, src_copy = lat.U[(prec, 18)].clone(), lat.A[prec].clone(), src_all.clone()
    for fn in (B.dw_apply, B.dwdag_apply):
        fn(lat.g, kappa, lat.U[(prec, 18)], lat.A[prec], src, dst, prec, 18)
    if prec == B.F64:
        ws_n = B.field_bytes(lat.g, B.FIELD_WORKSPACE)
        ws_all, ws = guarded(ws_n)
        B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], src, dst, ws, tol=1e-8, maxiter=50, raise_on_notconv=False)
        torch.cuda.synchronize()
        assert torch.all(ws_all[:G] == 0xA5) and torch.all(ws_all[G + ws_n:] == 0xA5)
    torch.cuda.synchronize()
    assert torch.all(dst_all[:G] == 0xA5) and torch.all(dst_all[G + nb:] == 0xA5)
    assert torch.equal(src_all, src_copy)
    assert torch.equal(lat.U[(prec, 18)], Ucopy) and torch.equal(lat.A[prec], Acopy)
    lat.close()


@pytest.mark.parametrize("mode", ["pipe", "stream"], indirect=True)
@pytest.mark.parametrize("L,bc,theta,phiT", CASES)
@pytest.mark.parametrize("prec,recon", [(B.F64, B.RECON_18), (B.F64, B.RECON_12), (B.F32, B.RECON_18), (B.F32, B.RECON_12)])
def test_dhat_parity_multi_tile(mode, L, bc, theta, phiT, prec, recon):
    """Even-odd operator D^ = A_ee - kappa^2 H_eo A_oo^-1 H_oe (D8) and its dagger on lattices of several 4^4 tiles per
    direction, every boundary condition: the half-lattice pipeline kernel (dw_pipe_half_kernel: forward / backward hops
    on two warp groups, halves swapped through shared memory, one chirality of the block multiply per group) and the
    one-thread-per-site kernel against oracle.dhat; also with one and three CTAs (every ring slot and phase)."""
    kappa, csw = 0.1355, 1.8
    U, psi = inputs(L, bc, 81)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=phiT)
    Ai = oracle.clover_inverse(L, A)
    Uo, psio, Ao, Aio = (round_f32(U), round_f32(psi), round_f32(A), round_f32(Ai)) if prec == B.F32 else (U, psi, A, Ai)
    x = np.arange(synth.vol(L))
    par = np.zeros_like(x)
    for mu in range(4):
        par += x % L[mu]
        x = x // L[mu]
    even = (par % 2 == 0) & interior(L, bc)
    lat = Lattice(L, bc, theta, synth.SF_PHI0, phiT)
    lat.set_gauge(U, recons=(recon,), precs=(prec,))
    lat.build_clover(kappa, csw, recon=recon, precs=(prec,), inverse=True)
    plan = B.dw_plan(lat.g, prec, recon, True, parity=0)
    assert ("dw_pipe_half_kernel" in plan) == (mode == "pipe"), plan
    src = lat.spinor(psi, prec)
    tmp = lat.alloc(B.FIELD_SPINOR, prec)
    try:
        for grid in ((0, 1, 3) if mode == "pipe" else (0,)):
            B.set_option("pipe_grid", str(grid))
            for dagger in (False, True):
                ref = oracle.dhat(L, Uo, psio, kappa, Ao, Aio, bc=bc, theta=theta, dagger=dagger)
                dst = lat.alloc(B.FIELD_SPINOR, prec)
                dst.zero_()
                B.dw_eo_apply(lat.g, kappa, lat.U[(prec, recon)], lat.A[prec], lat.Ainv[prec], src, dst, tmp, dagger, prec, recon)
                got = lat.spinor_to_host(dst, prec)
                assert site_rel_err(got, ref, even) <= TOL[prec] * 2, (grid, dagger)
                frozen_even = (par % 2 == 0) & ~interior(L, bc)
                assert np.all(got[frozen_even] == 0)
    finally:
        B.set_option("pipe_grid", "0")
    lat.close()


@pytest.mark.parametrize("mode", ["pipe", "stream"], indirect=True)
@pytest.mark.parametrize("mixed", [False, True])
def test_cg_eo_multi_tile(mode, mixed):
    """The even-odd solver (fused epilogues of the half-lattice kernels; fp32 inner solver when mixed) on a lattice of
    32 tiles with open boundaries against the oracle's CG."""
    L, bc, kappa, csw = (8, 8, 8, 16), B.BC_OPEN, 0.13, 1.7
    U, _ = inputs(L, bc, 85)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc)
    precs = (B.F64, B.F32) if mixed else (B.F64,)
    lat = Lattice(L, bc)
    lat.set_gauge(U, precs=precs)
    lat.build_clover(kappa, csw, precs=precs, inverse=True)
    b = synth.point_source(L, (1, 2, 3, 8), 2, 0)
    xo, it_o, _, rt_o = oracle.cg(L, U, b, kappa, A, bc=bc, tol=1e-10)
    x, ws = lat.alloc(B.FIELD_SPINOR), lat.alloc(B.FIELD_WORKSPACE)
    kw = dict(U32=lat.U[(B.F32, 18)], clover32=lat.A[B.F32], clover_inv32=lat.Ainv[B.F32]) if mixed else {}
    info = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], lat.spinor(b), x, ws, tol=1e-10, maxiter=5000,
                      clover_inv64=lat.Ainv[B.F64], eo=True, mixed=mixed, **kw)
    assert info["status"] == B.OK
    got = lat.spinor_to_host(x)
    rt = np.linalg.norm(b - oracle.dw(L, U, got, kappa, A, bc=bc))
    assert rt <= 50e-10 and abs(info["rel_resid_true"] - rt) <= 0.5 * rt + 1e-13
    assert np.linalg.norm(got - xo) / np.linalg.norm(xo) <= 200 * (rt + rt_o)
    assert np.all(got[~interior(L, bc)] == 0)
    lat.close()


def test_concurrent_launches_on_one_geometry():
    """The pipeline kernel's tile counters come from a pool owned by the geometry (one pair per launch in flight): D on
    two CUDA streams at the same time, on the same geometry and gauge field, must give what two launches one after the
    other give (bit for bit: the arithmetic per tile does not depend on which CTA draws it)."""
    L, kappa, csw = (16, 16, 16, 16), 0.137, 1.9
    dev = torch.device("cuda", torch.cuda.current_device())
    lat = Lattice(L)
    lat.set_gauge(synth.smooth_gauge_torch(L, 401, dev))
    lat.build_clover(kappa, csw)
    srcs = [lat.spinor(synth.gaussian_spinor_torch(L, 402 + i, dev)) for i in range(2)]
    ref = []
    for s in srcs:
        d = lat.alloc(B.FIELD_SPINOR)
        B.dw_apply(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], s, d)
        ref.append(d)
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for rep in range(20):
        outs = [lat.alloc(B.FIELD_SPINOR) for _ in range(2)]
        for o in outs:
            o.fill_(0x7F)
        torch.cuda.synchronize()
        for i in range(2):
            for _ in range(3):   # three launches per stream, interleaved with the other stream's
                B.dw_apply(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], srcs[i], outs[i], stream=streams[i].cuda_stream)
        torch.cuda.synchronize()
        for i in range(2):
            assert torch.equal(outs[i], ref[i]), rep
    lat.close()


@pytest.mark.parametrize("prec", [B.F64, B.F32])
def test_full_grid_launches_repeat_bit_for_bit(prec):
    """Race evidence without a sanitizer, at a size where all 148 CTAs run and draw their tiles from the counter in a
    different order every launch (32^4 = 4096 tiles): D, D^+, both passes of D^ and the staged clover builder, 25
    launches each into a poisoned output, must reproduce the first launch bit for bit.  (The half-lattice kernel's
    buffer-release race of round 2 showed up exactly like this: a few tiles per launch, different ones every run.)"""
    L, kappa, csw = (32, 32, 32, 32), 0.137, 1.9
    dev = torch.device("cuda", torch.cuda.current_device())
    lat = Lattice(L)
    lat.set_gauge(synth.smooth_gauge_torch(L, 501, dev), precs=(prec,))
    lat.build_clover(kappa, csw, precs=(prec,), inverse=True)
    assert B.geom_info(lat.g)[0] == [4, 4, 4, 4]
    U, A, Ai = lat.U[(prec, 18)], lat.A[prec], lat.Ainv[prec]
    src = lat.spinor(synth.gaussian_spinor_torch(L, 502, dev), prec)
    tmp = lat.alloc(B.FIELD_SPINOR, prec)
    A2, Ai2 = lat.alloc(B.FIELD_CLOVER, prec), lat.alloc(B.FIELD_CLOVER, prec)

    def clover(out):
        A2.fill_(0x7F)
        B.clover_build(lat.g, kappa, csw, lat.U[(B.F64, 18)], A2, Ai2 if prec == B.F64 else None, 18, prec)
        return A2

    def stencil(fn):
        def run(out):
            fn(out)
            return out
        return run

    ops = {
        "D": stencil(lambda out: B.dw_apply(lat.g, kappa, U, A, src, out, prec, 18)),
        "D^+": stencil(lambda out: B.dwdag_apply(lat.g, kappa, U, A, src, out, prec, 18)),
        "D^": stencil(lambda out: B.dw_eo_apply(lat.g, kappa, U, A, Ai, src, out, tmp, False, prec, 18)),
        "Csw": clover,
    }
    for name, op in ops.items():
        first = None
        for rep in range(25):
            out = lat.alloc(B.FIELD_SPINOR, prec)
            out.fill_(0x7F)
            res = op(out)
            torch.cuda.synchronize()
            if first is None:
                first = res.clone()
            else:
                assert torch.equal(res, first), (name, rep)
    if prec == B.F64:   # (fp32 blocks with an inverse come from the one-thread-per-site kernel: equal up to one rounding)
        assert torch.equal(A2, A) and torch.equal(Ai2, Ai)
    lat.close()


def test_concurrent_solves_on_one_geometry():
    """Two lqcd_cg_solve calls on ONE geometry from two host threads on two CUDA streams, ten times: iteration counts
    and solutions must be those of the serial solves, bit for bit.  (Each solve replays its iterations as a CUDA graph
    whose stencil launches keep their tile-scheduler counters; they come from the solve's own workspace, not from the
    geometry's pool, so that two solves can never share one.)"""
    import threading
    L, kappa, csw = (16, 16, 16, 16), 0.13, 1.5
    dev = torch.device("cuda", torch.cuda.current_device())
    lat = Lattice(L)
    lat.set_gauge(synth.smooth_gauge_torch(L, 701, dev))
    lat.build_clover(kappa, csw)
    srcs = [lat.spinor(synth.gaussian_spinor_torch(L, 702 + i, dev)) for i in range(2)]
    ws = [lat.alloc(B.FIELD_WORKSPACE) for _ in range(2)]
    ref = []
    for i in range(2):
        x = lat.alloc(B.FIELD_SPINOR)
        info = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], srcs[i], x, ws[i], tol=1e-8, maxiter=2000)
        ref.append((x.clone(), info["iters"]))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for rep in range(10):
        outs = [lat.alloc(B.FIELD_SPINOR) for _ in range(2)]
        infos, errs = [None, None], []

        def work(i):
            try:
                infos[i] = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], srcs[i], outs[i], ws[i], tol=1e-8,
                                      maxiter=2000, stream=streams[i])
            except Exception as e:   # surfaces in the main thread below
                errs.append(e)

        torch.cuda.synchronize()
        threads = [threading.Thread(target=work, args=(i,)) for i in range(2)]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        torch.cuda.synchronize()
        assert not errs, errs
        for i in range(2):
            assert infos[i]["iters"] == ref[i][1] and torch.equal(outs[i], ref[i][0]), (rep, i)
    lat.close()
