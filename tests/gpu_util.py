"""Helpers shared by the -m gpu parity tests: device allocations and layout marshalling through the C-ABI.

Nothing here computes any part of the method: the CUDA side is reached only through
paper_2503_16994_b200.binding, the expected values only through oracle/.
"""
import numpy as np
import torch

from paper_2503_16994_b200 import binding as B


def to_dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class Lattice:
    """Geometry handle + imported gauge field (+ clover term) on the device."""

    def __init__(self, L, bc=B.BC_PERIODIC, theta=None, phi0=None, phiT=None):
        self.L = tuple(int(v) for v in L)
        self.V = int(np.prod(self.L))
        self.bc = bc
        self.g = B.geom_create(self.L, bc, theta, phi0, phiT)
        self.U = {}
        self.A = {}
        self.Ainv = {}

    def close(self):
        B.geom_destroy(self.g)

    def alloc(self, kind, prec=B.F64, recon=B.RECON_18):
        return B.alloc_field(self.g, kind, prec, recon)

    def set_gauge(self, U_canon, recons=(B.RECON_18,), precs=(B.F64,)):
        """U_canon: numpy [V,4,3,3] complex128 or a cuda complex128 tensor."""
        dU = U_canon if torch.is_tensor(U_canon) else to_dev(U_canon)
        for recon in recons:
            for prec in set(precs) | {B.F64}:
                buf = self.alloc(B.FIELD_GAUGE, prec, recon)
                B.gauge_import(self.g, dU, buf, prec, recon)
                self.U[(prec, recon)] = buf
        torch.cuda.synchronize()

    def build_clover(self, kappa, csw, recon=B.RECON_18, precs=(B.F64,), inverse=False, ct=1.0):
        for prec in precs:
            A = self.alloc(B.FIELD_CLOVER, prec)
            Ai = self.alloc(B.FIELD_CLOVER, prec) if inverse else None
            B.clover_build(self.g, kappa, csw, self.U[(B.F64, recon)], A, Ai, recon, prec, ct)
            self.A[prec] = A
            self.Ainv[prec] = Ai
        torch.cuda.synchronize()

    def spinor(self, psi_canon, prec=B.F64):
        d = psi_canon if torch.is_tensor(psi_canon) else to_dev(psi_canon)
        buf = self.alloc(B.FIELD_SPINOR, prec)
        B.spinor_import(self.g, d, buf, prec)
        return buf

    def spinor_to_host(self, buf, prec=B.F64):
        out = torch.empty((self.V, 4, 3), dtype=torch.complex128, device="cuda")
        B.spinor_export(self.g, buf, out, prec)
        torch.cuda.synchronize()
        return out.cpu().numpy()

    def clover_to_host(self, buf, prec=B.F64):
        out = torch.empty((self.V, 2, 6, 6), dtype=torch.complex128, device="cuda")
        B.clover_export(self.g, buf, out, prec)
        torch.cuda.synchronize()
        return out.cpu().numpy()

    def dw(self, kappa, psi_canon, prec=B.F64, recon=B.RECON_18, dagger=False, clover=True):
        """import -> lqcd_dw_apply / lqcd_dwdag_apply -> export"""
        src = self.spinor(psi_canon, prec)
        dst = self.alloc(B.FIELD_SPINOR, prec)
        dst.fill_(0x7F)  # poison: every output element must be written
        A = self.A.get(prec) if clover else None
        fn = B.dwdag_apply if dagger else B.dw_apply
        fn(self.g, kappa, self.U[(prec, recon)], A, src, dst, prec, recon)
        return self.spinor_to_host(dst, prec)


def coords(L):
    """[V,4] integer coordinates in canonical site order."""
    L = [int(v) for v in L]
    n = np.arange(int(np.prod(L)))
    x = np.empty((len(n), 4), dtype=np.int64)
    for mu in range(4):
        x[:, mu] = n % L[mu]
        n = n // L[mu]
    return x


def interior(L, bc):
    t = coords(L)[:, 3]
    if bc == B.BC_OPEN:
        return (t >= 1) & (t <= L[3] - 2)
    if bc in (B.BC_SF_ORBI, B.BC_SF_AFWB):
        return t >= 1
    return np.ones(len(t), dtype=bool)


def site_rel_err(got, ref, mask=None):
    """R15: max over (non-frozen) sites of |g(x) - o(x)|_2 / |o(x)|_2."""
    g = got.reshape(got.shape[0], -1)
    o = ref.reshape(ref.shape[0], -1)
    if mask is not None:
        g, o = g[mask], o[mask]
    num = np.linalg.norm(g - o, axis=1)
    den = np.linalg.norm(o, axis=1)
    return float(np.max(num / den))


def round_f32(a):
    """R14: the fp32 path's inputs, rounded once, promoted back to fp64 for the oracle."""
    return a.astype(np.complex64).astype(np.complex128)


def f32_storage_err(got32, ref64, build_tol=2e-14):
    """fp32 storage of a field built in fp64 (R14: built in fp64, rounded once).  The library's fp64 value agrees with
    the oracle's to build_tol, so the stored fp32 number is the rounding of a value within build_tol of ref64: its
    distance from ref64 is at most half an fp32 spacing at |ref64| plus build_tol.  Returns the worst excess over
    that bound (<= 0 means every element is a correct rounding); the same rule is used by every test of an fp32 clover
    term (whole lattice and slabs)."""
    worst = -np.inf
    for part in (np.real, np.imag):
        g, r = part(got32).astype(np.float64), part(ref64).astype(np.float64)
        half = 0.5 * np.spacing(np.abs(r).astype(np.float32)).astype(np.float64)
        worst = max(worst, float(np.max(np.abs(g - r) - half - build_tol)))
    return worst
