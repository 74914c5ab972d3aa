"""CPU oracle (test infrastructure, not the product): ctypes view of oracle/lqcd_oracle.cpp.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It imports nothing from paper_2503_16994_b200 and shares no code with the CUDA path.
All arrays are numpy complex128 / float64 in the canonical layouts of SURVEY.md 8(b):
gauge [V,4,3,3], spinor [V,4,3], clover blocks [V,2,6,6], site n = x1 + L1*(x2 + L2*(x3 + L3*x4)).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lqcd_oracle.cpp")
_LIB = os.path.join(_HERE, "liblqcd_oracle.so")

BC_PERIODIC, BC_OPEN, BC_SF_ORBI, BC_SF_AFWB = 0, 1, 2, 3


_SRC_SUN = os.path.join(_HERE, "lqcd_oracle_sun.cpp")
_LIB_SUN = os.path.join(_HERE, "liblqcd_oracle_sun.so")


def build(force=False):
    """Compile the oracles with g++ -O2 -fopenmp (no fast-math: fp64 results must be plain IEEE): the SU(3) oracle
    and, separately, the N-colour oracle of the SU(2) fundamental representation."""
    for src, lib_ in ((_SRC, _LIB), (_SRC_SUN, _LIB_SUN)):
        if not force and os.path.exists(lib_) and os.path.getmtime(lib_) >= os.path.getmtime(src):
            continue
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", lib_, src])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.oracle_plaquette.restype = ctypes.c_double
        _lib.oracle_cg.restype = ctypes.c_int
        _lib.oracle_cg_eo.restype = ctypes.c_int
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _c(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _L(L):
    return (ctypes.c_int * 4)(*[int(v) for v in L])


def _d(v, n):
    if v is None:
        v = [0.0] * n
    return (ctypes.c_double * n)(*[float(t) for t in v])


class _twisted:
    """Sets the oracle's twisted mass for the duration of one call (NEXT-4; 0 = plain Wilson-clover)."""

    def __init__(self, mu):
        self.mu = float(mu)

    def __enter__(self):
        lib().oracle_set_twisted_mass(ctypes.c_double(self.mu))

    def __exit__(self, *exc):
        lib().oracle_set_twisted_mass(ctypes.c_double(0.0))


def vol(L):
    return int(L[0]) * int(L[1]) * int(L[2]) * int(L[3])


def num_threads():
    return int(lib().oracle_num_threads())


def set_num_threads(n):
    lib().oracle_set_num_threads(ctypes.c_int(int(n)))


def gamma(mu):
    """gamma_mu for mu = 0..3 (directions 1..4), gamma5 for mu = 4, as 4x4 complex (D2)."""
    out = np.zeros((4, 4), dtype=np.complex128)
    lib().oracle_gamma(ctypes.c_int(mu), _p(out))
    return out


def sigma(mu, nu):
    out = np.zeros((4, 4), dtype=np.complex128)
    lib().oracle_sigma(ctypes.c_int(mu), ctypes.c_int(nu), _p(out))
    return out


def plaquette(L, U):
    U = _c(U, (vol(L), 4, 3, 3))
    return float(lib().oracle_plaquette(_L(L), _p(U)))


def fhat_site(L, U, x, mu, nu, bc=BC_PERIODIC, phiT=None):
    U = _c(U, (vol(L), 4, 3, 3))
    out = np.zeros((3, 3), dtype=np.complex128)
    lib().oracle_fhat_site(_L(L), ctypes.c_int(bc), _d(phiT, 3), _p(U), _L(x), ctypes.c_int(mu),
                           ctypes.c_int(nu), _p(out))
    return out


def clover_dense(L, U, kappa, csw, bc=BC_PERIODIC, phiT=None, ct=1.0):
    U = _c(U, (vol(L), 4, 3, 3))
    out = np.zeros((vol(L), 12, 12), dtype=np.complex128)
    lib().oracle_clover_dense(_L(L), ctypes.c_int(bc), _d(phiT, 3), ctypes.c_double(kappa),
                              ctypes.c_double(csw), ctypes.c_double(ct), _p(U), _p(out))
    return out


def clover_blocks(L, U, kappa, csw, bc=BC_PERIODIC, phiT=None, ct=1.0):
    U = _c(U, (vol(L), 4, 3, 3))
    out = np.zeros((vol(L), 2, 6, 6), dtype=np.complex128)
    lib().oracle_clover_blocks(_L(L), ctypes.c_int(bc), _d(phiT, 3), ctypes.c_double(kappa),
                               ctypes.c_double(csw), ctypes.c_double(ct), _p(U), _p(out))
    return out


def clover_inverse(L, Ablk):
    Ablk = _c(Ablk, (vol(L), 2, 6, 6))
    out = np.zeros_like(Ablk)
    lib().oracle_clover_inverse(_L(L), _p(Ablk), _p(out))
    return out


def dw(L, U, psi, kappa, Ablk=None, bc=BC_PERIODIC, theta=None, dagger=False, mu=0.0):
    """D psi (or D^+ psi); mu = twisted mass: D = A + 2 i kappa mu gamma5 - kappa H."""
    U = _c(U, (vol(L), 4, 3, 3))
    psi = _c(psi, (vol(L), 4, 3))
    out = np.zeros_like(psi)
    ap = None
    if Ablk is not None:
        Ablk = _c(Ablk, (vol(L), 2, 6, 6))
        ap = _p(Ablk)
    with _twisted(mu):
        lib().oracle_dw(_L(L), ctypes.c_int(bc), _d(theta, 4), ctypes.c_double(kappa), _p(U), ap, _p(psi),
                        _p(out), ctypes.c_int(1 if dagger else 0))
    return out


def hop(L, U, psi, bc=BC_PERIODIC, theta=None):
    U = _c(U, (vol(L), 4, 3, 3))
    psi = _c(psi, (vol(L), 4, 3))
    out = np.zeros_like(psi)
    lib().oracle_hop(_L(L), ctypes.c_int(bc), _d(theta, 4), _p(U), _p(psi), _p(out))
    return out


def dw_at_sites(L, U, psi, sites, kappa, csw, bc=BC_PERIODIC, theta=None, phiT=None, ct=1.0, dagger=False):
    U = _c(U, (vol(L), 4, 3, 3))
    psi = _c(psi, (vol(L), 4, 3))
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.zeros((len(sites), 4, 3), dtype=np.complex128)
    lib().oracle_dw_at_sites(_L(L), ctypes.c_int(bc), _d(theta, 4), _d(phiT, 3), ctypes.c_double(kappa),
                             ctypes.c_double(csw), ctypes.c_double(ct), _p(U), _p(psi),
                             ctypes.c_int(1 if dagger else 0), ctypes.c_long(len(sites)), _p(sites), _p(out))
    return out


def dhat(L, U, psi, kappa, Ablk, Ainv, bc=BC_PERIODIC, theta=None, dagger=False):
    U = _c(U, (vol(L), 4, 3, 3))
    psi = _c(psi, (vol(L), 4, 3))
    Ablk = _c(Ablk, (vol(L), 2, 6, 6))
    Ainv = _c(Ainv, (vol(L), 2, 6, 6))
    out = np.zeros_like(psi)
    lib().oracle_dhat(_L(L), ctypes.c_int(bc), _d(theta, 4), ctypes.c_double(kappa), _p(U), _p(Ablk),
                      _p(Ainv), _p(psi), _p(out), ctypes.c_int(1 if dagger else 0))
    return out


def cg(L, U, b, kappa, Ablk=None, bc=BC_PERIODIC, theta=None, tol=1e-10, maxiter=10000, mu=0.0):
    """Returns (x, iters, rel_resid_normal, rel_resid_true); iters < 0 means maxiter was hit."""
    U = _c(U, (vol(L), 4, 3, 3))
    b = _c(b, (vol(L), 4, 3))
    x = np.zeros_like(b)
    ap = None
    if Ablk is not None:
        Ablk = _c(Ablk, (vol(L), 2, 6, 6))
        ap = _p(Ablk)
    rn, rt = ctypes.c_double(0), ctypes.c_double(0)
    with _twisted(mu):
        it = lib().oracle_cg(_L(L), ctypes.c_int(bc), _d(theta, 4), ctypes.c_double(kappa), _p(U), ap, _p(b),
                             _p(x), ctypes.c_double(tol), ctypes.c_int(maxiter), ctypes.byref(rn),
                             ctypes.byref(rt))
    return x, int(it), rn.value, rt.value


def cg_eo(L, U, b, kappa, Ablk, Ainv, bc=BC_PERIODIC, theta=None, tol=1e-10, maxiter=10000):
    U = _c(U, (vol(L), 4, 3, 3))
    b = _c(b, (vol(L), 4, 3))
    Ablk = _c(Ablk, (vol(L), 2, 6, 6))
    Ainv = _c(Ainv, (vol(L), 2, 6, 6))
    x = np.zeros_like(b)
    rn, rt = ctypes.c_double(0), ctypes.c_double(0)
    it = lib().oracle_cg_eo(_L(L), ctypes.c_int(bc), _d(theta, 4), ctypes.c_double(kappa), _p(U), _p(Ablk),
                            _p(Ainv), _p(b), _p(x), ctypes.c_double(tol), ctypes.c_int(maxiter),
                            ctypes.byref(rn), ctypes.byref(rt))
    return x, int(it), rn.value, rt.value


def correlator_ps(L, cols):
    """C(x4) = sum_{xvec} sum_{columns, spin, colour} |S|^2 for columns [ncol, V, 4, 3] (NEXT-2)."""
    cols = np.ascontiguousarray(cols, dtype=np.complex128)
    assert cols.ndim == 4 and cols.shape[1:] == (vol(L), 4, 3), cols.shape
    C = np.zeros(int(L[3]), dtype=np.float64)
    lib().oracle_correlator_ps(_L(L), _p(cols), ctypes.c_int(cols.shape[0]), _p(C))
    return C


# ---- SU(2) fundamental representation: the N-colour oracle of lqcd_oracle_sun.cpp -------------------
# gauge [V,4,N,N], spinor [V,4,N], blocks [V,2,2N,2N]; nc = 2 is the representation under test, nc = 3 exists to pin
# the generic loops against the SU(3) oracle above.
_lib_sun = None


def lib_sun():
    global _lib_sun
    if _lib_sun is None:
        build()
        _lib_sun = ctypes.CDLL(_LIB_SUN)
    return _lib_sun


def su2_from_cayley_dickson(z):
    """[..., 2] Cayley-Dickson pairs (z1, z2) -> [..., 2, 2] matrices [[z1, z2], [-conj z2, conj z1]]."""
    z = np.ascontiguousarray(z, dtype=np.complex128)
    out = np.zeros(z.shape[:-1] + (2, 2), dtype=np.complex128)
    lib_sun().oracle_su2_from_cayley_dickson(ctypes.c_long(z.size // 2), _p(z), _p(out))
    return out


def sun_dw(nc, L, U, psi, kappa, Ablk=None, bc=BC_PERIODIC, theta=None, dagger=False):
    U = _c(U, (vol(L), 4, nc, nc))
    psi = _c(psi, (vol(L), 4, nc))
    out = np.zeros_like(psi)
    ap = None
    if Ablk is not None:
        Ablk = _c(Ablk, (vol(L), 2, 2 * nc, 2 * nc))
        ap = _p(Ablk)
    rc = lib_sun().oracle_sun_dw(ctypes.c_int(nc), _L(L), ctypes.c_int(bc), _d(theta, 4), ctypes.c_double(kappa), _p(U), ap,
                                 _p(psi), _p(out), ctypes.c_int(1 if dagger else 0))
    assert rc == 0
    return out


def sun_hop(nc, L, U, psi, bc=BC_PERIODIC, theta=None):
    U = _c(U, (vol(L), 4, nc, nc))
    psi = _c(psi, (vol(L), 4, nc))
    out = np.zeros_like(psi)
    assert lib_sun().oracle_sun_hop(ctypes.c_int(nc), _L(L), ctypes.c_int(bc), _d(theta, 4), _p(U), _p(psi), _p(out)) == 0
    return out


def sun_fhat_site(nc, L, U, x, mu, nu):
    U = _c(U, (vol(L), 4, nc, nc))
    out = np.zeros((nc, nc), dtype=np.complex128)
    assert lib_sun().oracle_sun_fhat_site(ctypes.c_int(nc), _L(L), _p(U), _L(x), ctypes.c_int(mu), ctypes.c_int(nu), _p(out)) == 0
    return out


def sun_clover_blocks(nc, L, U, kappa, csw, bc=BC_PERIODIC):
    U = _c(U, (vol(L), 4, nc, nc))
    out = np.zeros((vol(L), 2, 2 * nc, 2 * nc), dtype=np.complex128)
    assert lib_sun().oracle_sun_clover_blocks(ctypes.c_int(nc), _L(L), ctypes.c_int(bc), ctypes.c_double(kappa),
                                              ctypes.c_double(csw), _p(U), _p(out)) == 0
    return out


def sun_cg(nc, L, U, b, kappa, Ablk=None, bc=BC_PERIODIC, theta=None, tol=1e-10, maxiter=10000):
    """Returns (x, iters, rel_resid_normal, rel_resid_true); iters < 0 means maxiter was hit."""
    U = _c(U, (vol(L), 4, nc, nc))
    b = _c(b, (vol(L), 4, nc))
    x = np.zeros_like(b)
    ap = None
    if Ablk is not None:
        Ablk = _c(Ablk, (vol(L), 2, 2 * nc, 2 * nc))
        ap = _p(Ablk)
    rn, rt = ctypes.c_double(0), ctypes.c_double(0)
    f = lib_sun().oracle_sun_cg
    f.restype = ctypes.c_int
    it = f(ctypes.c_int(nc), _L(L), ctypes.c_int(bc), _d(theta, 4), ctypes.c_double(kappa), _p(U), ap, _p(b), _p(x),
           ctypes.c_double(tol), ctypes.c_int(maxiter), ctypes.byref(rn), ctypes.byref(rt))
    return x, int(it), rn.value, rt.value
