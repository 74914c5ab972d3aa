"""-m gpu: lqcd_correlator_ps_static, the entry point that allocates nothing (its scratch is a static array in device
memory; include/lqcd.h), against the existing path lqcd_correlator_ps with a caller-owned workspace, and against the
oracle, within the tolerance the correlator tests use (1e-13 relative; the two GPU paths run the same kernels, so
they are also bit-identical).  Two calls in a row with different inputs: the array keeps the first call's contents and
the second call must not see them.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2503_16994_b200 import binding as B
from paper_2503_16994_b200 import synth

from gpu_util import Lattice, round_f32

pytestmark = pytest.mark.gpu

TOL = 1e-13


def columns(lat, L, prec, ncol, seed):
    fb = B.field_bytes(lat.g, B.FIELD_SPINOR, prec)
    dev = torch.empty(ncol * fb, dtype=torch.uint8, device="cuda")
    host = []
    for c in range(ncol):
        psi = synth.gaussian_spinor(L, seed + c)
        host.append(round_f32(psi) if prec == B.F32 else psi)
        dev[c * fb:(c + 1) * fb].copy_(lat.spinor(psi, prec))
    return dev, np.array(host)


@pytest.mark.parametrize("L,bc", [((8, 4, 8, 12), B.BC_PERIODIC), ((6, 4, 10, 8), B.BC_OPEN)])
@pytest.mark.parametrize("prec", [B.F64, B.F32])
def test_static_scratch_matches_workspace_path_two_calls(L, bc, prec):
    lat = Lattice(L, bc)
    ws = lat.alloc(B.FIELD_WORKSPACE)
    # second call: fewer columns and a scaled field, so anything left over from the first call would show
    for ncol, seed, scale in ((5, 700, 1.0), (2, 760, 2.0)):
        dev, host = columns(lat, L, prec, ncol, seed)
        if scale != 1.0:
            typed = dev.view(torch.float64 if prec == B.F64 else torch.float32)
            typed.mul_(scale)
            host = host * scale
        torch.cuda.synchronize()
        ref_gpu = np.array(B.correlator_ps(lat.g, dev, ncol, ws, L[3], prec))
        got = np.array(B.correlator_ps_static(lat.g, dev, ncol, L[3], prec))
        ref = oracle.correlator_ps(L, host)
        assert np.max(np.abs(got - ref_gpu) / ref_gpu) <= TOL
        assert np.array_equal(got, ref_gpu)
        assert np.max(np.abs(got - ref) / ref) <= TOL
    lat.close()


def test_static_scratch_call_allocates_nothing():
    """Device memory in use does not move across calls: free memory before a call equals free memory after it.  (The
    array is part of the library's device image and comes into being when that image is loaded -- with CUDA's lazy
    module loading at the first call -- so the comparison starts after one call.)"""
    L = (8, 8, 8, 8)
    lat = Lattice(L)
    dev, _ = columns(lat, L, B.F64, 3, 800)
    first = B.correlator_ps_static(lat.g, dev, 3, L[3])
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        assert B.correlator_ps_static(lat.g, dev, 3, L[3]) == first
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        assert free1 == free0
    lat.close()


def test_static_scratch_rejects_lattices_beyond_its_size():
    """64^3 x 128 needs 131072 tiles x 4 + 128 doubles > LQCD_CORRELATOR_STATIC_MAX_DOUBLES: a clear error before any
    kernel is launched (the column pointer is never followed); 48^3 x 96 is inside the limit."""
    assert 41472 * 4 + 96 <= B.CORRELATOR_STATIC_MAX_DOUBLES < 131072 * 4 + 128
    big = Lattice((64, 64, 64, 128))
    dummy = torch.zeros(256, dtype=torch.uint8, device="cuda")
    n0 = B.launch_count()
    with pytest.raises(B.LqcdError, match="static scratch holds"):
        B.correlator_ps_static(big.g, dummy, 1, 128)
    assert B.launch_count() == n0
    with pytest.raises(B.LqcdError):
        B.correlator_ps_static(big.g, dummy, 0, 128)
    big.close()
