"""-m gpu parity of the lock-step solver lqcd_cg_solve_multi / lqcd_propagator_batched (SURVEY.md 8(f) NEXT-1 carried
into CG!) against the oracle's step-by-step CG column by column, and against lqcd_cg_solve: per
column the arithmetic is the same, so iteration counts are equal and the solutions agree to rounding."""
import numpy as np
import pytest
import torch

import oracle
from paper_2503_16994_b200 import binding as B
from paper_2503_16994_b200 import synth

from gpu_util import Lattice, interior

pytestmark = pytest.mark.gpu

TOL = 1e-10


def make(L, bc, theta, kappa, csw, seed):
    U = synth.smooth_gauge(L, seed)
    lat = Lattice(L, bc, theta)
    lat.set_gauge(U)
    lat.build_clover(kappa, csw)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc)
    return U, A, lat


def field_array(lat, fields):
    fb = B.field_bytes(lat.g, B.FIELD_SPINOR)
    dev = torch.empty(len(fields) * fb, dtype=torch.uint8, device="cuda")
    for n, psi in enumerate(fields):
        dev[n * fb:(n + 1) * fb].copy_(lat.spinor(psi))
    return dev, fb


@pytest.mark.parametrize("L,bc,theta,kappa,csw", [
    ((8, 4, 4, 8), B.BC_PERIODIC, (0, 0, 0, np.pi), 0.125, 1.0),
    ((4, 8, 4, 12), B.BC_OPEN, (0.5, 0.5, 0.5, 0.0), 0.1365, 1.9),
])
def test_cg_solve_multi_matches_oracle_and_single_solves(L, bc, theta, kappa, csw):
    """Five columns that converge after different numbers of iterations (point sources, a Gaussian source, a source that
    is zero: that column is finished before it starts), one of them with support on a frozen slice for open boundaries."""
    U, A, lat = make(L, bc, theta, kappa, csw, 611)
    assert B.geom_info(lat.g)[0] == [4, 4, 4, 4] and "dw_pipe_kernel" in B.dw_plan(lat.g)
    V = synth.vol(L)
    y = (1, 2, 3, L[3] // 2)
    srcs = [synth.point_source(L, y, 0, 0), synth.point_source(L, y, 3, 2), synth.gaussian_spinor(L, 612),
            np.zeros((V, 4, 3), dtype=np.complex128), 0.01 * synth.gaussian_spinor(L, 613)]
    nrhs = len(srcs)
    b, fb = field_array(lat, srcs)
    x = torch.full((nrhs * fb,), 0x7F, dtype=torch.uint8, device="cuda")
    ws = torch.empty(B.cg_multi_workspace_bytes(lat.g, nrhs), dtype=torch.uint8, device="cuda")
    infos = B.cg_solve_multi(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], b, x, nrhs, ws, tol=TOL, maxiter=5000)
    ws1 = lat.alloc(B.FIELD_WORKSPACE)
    mask = interior(L, bc)
    iters = []
    for n in range(nrhs):
        got = lat.spinor_to_host(x[n * fb:(n + 1) * fb])
        src = srcs[n] * mask[:, None, None]     # D7: components on frozen slices are ignored
        if not np.any(src):
            assert infos[n]["iters"] == 0 and not np.any(got)
            iters.append(0)
            continue
        xo, it_o, _, _ = oracle.cg(L, U, src, kappa, A, bc=bc, theta=theta, tol=TOL, maxiter=5000)
        assert abs(infos[n]["iters"] - abs(it_o)) <= 2, (n, infos[n], it_o)
        assert np.linalg.norm(got - xo) / np.linalg.norm(xo) <= 1e-8
        assert infos[n]["rel_resid_normal"] <= 2 * TOL
        assert np.all(got[~mask] == 0)
        # the single-column solver: same arithmetic per column
        x1 = lat.alloc(B.FIELD_SPINOR)
        i1 = B.cg_solve(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], b[n * fb:(n + 1) * fb], x1, ws1, tol=TOL, maxiter=5000)
        assert i1["iters"] == infos[n]["iters"]
        g1 = lat.spinor_to_host(x1)
        assert np.linalg.norm(got - g1) <= 1e-12 * np.linalg.norm(g1)
        assert abs(i1["rel_resid_true"] - infos[n]["rel_resid_true"]) <= 1e-3 * i1["rel_resid_true"] + 1e-16
        iters.append(infos[n]["iters"])
    assert len(set(iters)) >= 3   # the columns really did stop at different iterations
    lat.close()


def test_propagator_batched_equals_propagator():
    """The 12 point-source columns: batched against the column-by-column lqcd_propagator (iteration counts equal,
    solutions to rounding) and three columns against the oracle's CG."""
    L, kappa, csw, theta = (4, 4, 8, 8), 0.13, 1.5, (0, 0, 0, np.pi)
    U, A, lat = make(L, B.BC_PERIODIC, theta, kappa, csw, 621)
    fb = B.field_bytes(lat.g, B.FIELD_SPINOR)
    y = (1, 0, 5, 3)
    cols = torch.empty(12 * fb, dtype=torch.uint8, device="cuda")
    cols_b = torch.full((12 * fb,), 0x7F, dtype=torch.uint8, device="cuda")
    srcs = torch.empty(12 * fb, dtype=torch.uint8, device="cuda")
    infos = B.propagator(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], y, cols, lat.alloc(B.FIELD_WORKSPACE), tol=TOL)
    ws = torch.empty(B.cg_multi_workspace_bytes(lat.g, 12), dtype=torch.uint8, device="cuda")
    infos_b = B.propagator_batched(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], y, cols_b, srcs, ws, tol=TOL)
    for c in range(12):
        assert infos_b[c]["iters"] == infos[c]["iters"]
        a, b = lat.spinor_to_host(cols[c * fb:(c + 1) * fb]), lat.spinor_to_host(cols_b[c * fb:(c + 1) * fb])
        assert np.linalg.norm(a - b) <= 1e-12 * np.linalg.norm(a)
    for c in (0, 7, 11):
        xo, it_o, _, _ = oracle.cg(L, U, synth.point_source(L, y, c // 3, c % 3), kappa, A, theta=theta, tol=TOL)
        got = lat.spinor_to_host(cols_b[c * fb:(c + 1) * fb])
        assert np.linalg.norm(got - xo) / np.linalg.norm(xo) <= 1e-8 and abs(infos_b[c]["iters"] - abs(it_o)) <= 2
    lat.close()


def test_cg_solve_multi_falls_back_and_rejects():
    """A lattice without 4^4 tiles (no pipeline kernel), and the even-odd mode: solved column by column, same results;
    bad column counts and overlapping arrays are rejected."""
    L, kappa, csw = (6, 4, 4, 8), 0.125, 1.0
    U, A, lat = make(L, B.BC_PERIODIC, None, kappa, csw, 631)
    assert B.geom_info(lat.g)[0] != [4, 4, 4, 4]
    srcs = [synth.point_source(L, (0, 0, 0, 0), 1, 1), synth.gaussian_spinor(L, 632)]
    b, fb = field_array(lat, srcs)
    x = torch.empty(2 * fb, dtype=torch.uint8, device="cuda")
    ws = torch.empty(B.cg_multi_workspace_bytes(lat.g, 2), dtype=torch.uint8, device="cuda")
    infos = B.cg_solve_multi(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], b, x, 2, ws, tol=TOL)
    for n in range(2):
        xo, it_o, _, _ = oracle.cg(L, U, srcs[n], kappa, A, tol=TOL)
        got = lat.spinor_to_host(x[n * fb:(n + 1) * fb])
        assert np.linalg.norm(got - xo) / np.linalg.norm(xo) <= 1e-8 and abs(infos[n]["iters"] - abs(it_o)) <= 2
    for bad in (0, 65):
        with pytest.raises(B.LqcdError):
            B.cg_solve_multi(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], b, x, bad, ws, tol=TOL)
    with pytest.raises(B.LqcdError):
        B.cg_solve_multi(lat.g, kappa, lat.U[(B.F64, 18)], lat.A[B.F64], b, b[fb:], 2, ws, tol=TOL)
    assert B.cg_multi_workspace_bytes(lat.g, 0) == 0 and B.cg_multi_workspace_bytes(lat.g, 65) == 0
    lat.close()
