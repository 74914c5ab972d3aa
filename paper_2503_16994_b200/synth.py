"""Seeded synthetic inputs (the one module the oracle-side tests and the CUDA-side tests both use).

Holds NONE of the method's arithmetic (no Dirac operator, clover term or solver): only random SU(3)
gauge fields, Gaussian spinors and point sources in the canonical interchange layout of
include/lqcd.h (site n = x1 + L1*(x2 + L2*(x3 + L3*x4)), gauge [V,4,3,3], spinor [V,4,3]).

The paper's workloads are quenched SU(3) configurations from its own HMC or openQCD-format files
(PAPER.md:78-90,153); none exist here.  These generators stand in for them (DESIGN.md "Input recipe",
SURVEY.md 8(d)): same shapes (4-D, SU(3) links, 4x3 spinors), plaquette ~0.6 for the smooth fields.
"""
import math

import numpy as np

EPS_PLAQ06 = 0.4322  # <plaq> = 0.600 for independent links U = exp(i eps H)  (pin P11)

# SU(3) Schroedinger-functional background at eta = nu = 0 (ref. [10] of the paper)
SF_PHI0 = (-math.pi / 3.0, 0.0, math.pi / 3.0)
SF_PHIT = (-math.pi, math.pi / 3.0, 2.0 * math.pi / 3.0)


def vol(L):
    return int(L[0]) * int(L[1]) * int(L[2]) * int(L[3])


def seed_for(config, j):
    """seed = 1000*c + j  (c = config number 1..5; j = 0 gauge, 1 spinor)."""
    return 1000 * int(config) + int(j)


def haar_gauge(L, seed):
    """G-Haar: Z = X + iY Gaussian 3x3; QR; fix the phases of R's diagonal; divide by det^(1/3)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = vol(L) * 4
    z = rng.standard_normal((n, 3, 3)) + 1j * rng.standard_normal((n, 3, 3))
    q, r = np.linalg.qr(z)
    d = np.diagonal(r, axis1=1, axis2=2)
    q = q * (d / np.abs(d))[:, None, :]
    det = np.linalg.det(q)
    q = q * (det ** (-1.0 / 3.0))[:, None, None]  # principal root
    return np.ascontiguousarray(q.reshape(vol(L), 4, 3, 3))


def gell_mann():
    lam = np.zeros((8, 3, 3), dtype=np.complex128)
    lam[0][0, 1] = lam[0][1, 0] = 1
    lam[1][0, 1] = -1j
    lam[1][1, 0] = 1j
    lam[2][0, 0] = 1
    lam[2][1, 1] = -1
    lam[3][0, 2] = lam[3][2, 0] = 1
    lam[4][0, 2] = -1j
    lam[4][2, 0] = 1j
    lam[5][1, 2] = lam[5][2, 1] = 1
    lam[6][1, 2] = -1j
    lam[6][2, 1] = 1j
    lam[7][0, 0] = lam[7][1, 1] = 1 / math.sqrt(3)
    lam[7][2, 2] = -2 / math.sqrt(3)
    return lam


def smooth_gauge(L, seed, eps=EPS_PLAQ06, chunk=1 << 18):
    """G-smooth: h_a ~ N(0,1), H = sum_a h_a lambda_a/2, U = exp(i eps H) by Hermitian eigendecomposition."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = vol(L) * 4
    lam = gell_mann() / 2.0
    out = np.empty((n, 3, 3), dtype=np.complex128)
    for s in range(0, n, chunk):
        m = min(chunk, n - s)
        h = rng.standard_normal((m, 8))
        H = np.einsum("na,aij->nij", h, lam)
        w, v = np.linalg.eigh(H)
        out[s:s + m] = np.einsum("nij,nj,nkj->nik", v, np.exp(1j * eps * w), v.conj())
    return np.ascontiguousarray(out.reshape(vol(L), 4, 3, 3))


def smooth_gauge_torch(L, seed, device, eps=EPS_PLAQ06, chunk=1 << 22):
    """Same definition as smooth_gauge, drawn and exponentiated on `device` with torch (for the
    48^3x96 / 64^3x128 benches, where 10^8 host eigendecompositions are too slow).  A different
    random stream than smooth_gauge: parity checks always download THIS array, never re-generate."""
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    n = vol(L) * 4
    lam = torch.from_numpy(gell_mann() / 2.0).to(device)
    out = torch.empty((n, 3, 3), dtype=torch.complex128, device=device)
    for s in range(0, n, chunk):
        m = min(chunk, n - s)
        h = torch.randn((m, 8), generator=g, device=device, dtype=torch.float64)
        H = torch.einsum("na,aij->nij", h.to(torch.complex128), lam)
        out[s:s + m] = torch.linalg.matrix_exp(1j * eps * H)
    return out.reshape(vol(L), 4, 3, 3)


def gaussian_spinor(L, seed):
    """G-spinor: re, im ~ N(0,1) per component."""
    rng = np.random.Generator(np.random.PCG64(seed))
    v = vol(L)
    z = rng.standard_normal((v, 4, 3, 2))
    return np.ascontiguousarray(z[..., 0] + 1j * z[..., 1])


def gaussian_spinor_torch(L, seed, device):
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    z = torch.randn((vol(L), 4, 3, 2), generator=g, device=device, dtype=torch.float64)
    return torch.view_as_complex(z)


def site_index(L, x):
    return int(x[0]) + L[0] * (int(x[1]) + L[1] * (int(x[2]) + L[2] * int(x[3])))


def point_source(L, y, spin, colour):
    b = np.zeros((vol(L), 4, 3), dtype=np.complex128)
    b[site_index(L, y), spin, colour] = 1.0
    return b


def sf_boundary_links(L, phi, mu):
    """W_k = exp(i diag(phi)/L_k), the abelian SF boundary link in spatial direction mu."""
    return np.diag(np.exp(1j * np.asarray(phi, dtype=np.float64) / L[mu]))


def apply_sf_boundary(L, U, phi0=SF_PHI0):
    """Overwrite the spatial links on slice x4 = 0 with W (R8: the x4 = 0 boundary lives in the array)."""
    U = U.copy()
    n0 = L[0] * L[1] * L[2]
    for mu in range(3):
        U[:n0, mu] = sf_boundary_links(L, phi0, mu)
    return U


def random_su3_field(L, seed):
    """One Haar SU(3) matrix per site (gauge transformations for covariance tests)."""
    return haar_gauge(L, seed)[:, 0].copy()


# ---- SU(2): links as Cayley-Dickson pairs (z1, z2), |z1|^2 + |z2|^2 = 1 -------------------------
def haar_su2_cd(L, seed):
    """Haar SU(2): a uniformly random point on S^3, as the pair (z1, z2) = (a0 + i a3, a2 + i a1); [V,4,2]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    a = rng.standard_normal((vol(L) * 4, 4))
    a /= np.linalg.norm(a, axis=1)[:, None]
    z = np.stack([a[:, 0] + 1j * a[:, 3], a[:, 2] + 1j * a[:, 1]], axis=1)
    return np.ascontiguousarray(z.reshape(vol(L), 4, 2))


def smooth_su2_cd(L, seed, eps=0.55):
    """U = exp(i eps H), H = sum_a h_a sigma_a / 2, h_a ~ N(0,1), in closed form:
    exp(i (eps |h| / 2) n.sigma) = cos(w) + i sin(w) n.sigma, w = eps |h| / 2  =>  z1 = cos w + i n3 sin w,
    z2 = (n2 + i n1) sin w.  eps = 0.55 gives a plaquette of about 0.6 (checked in the tests); [V,4,2]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    h = rng.standard_normal((vol(L) * 4, 3))
    nh = np.linalg.norm(h, axis=1)
    w = 0.5 * eps * nh
    n = h / nh[:, None]
    z = np.stack([np.cos(w) + 1j * n[:, 2] * np.sin(w), (n[:, 1] + 1j * n[:, 0]) * np.sin(w)], axis=1)
    return np.ascontiguousarray(z.reshape(vol(L), 4, 2))


def su2_matrices(z):
    """[..., 2] Cayley-Dickson pairs -> [..., 2, 2] matrices [[z1, z2], [-conj z2, conj z1]] (the canonical gauge layout)."""
    z = np.asarray(z)
    out = np.empty(z.shape[:-1] + (2, 2), dtype=np.complex128)
    out[..., 0, 0] = z[..., 0]
    out[..., 0, 1] = z[..., 1]
    out[..., 1, 0] = -np.conj(z[..., 1])
    out[..., 1, 1] = np.conj(z[..., 0])
    return out


def gaussian_spinor_nc(L, seed, nc):
    """Gaussian spinor with nc colours, [V,4,nc]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    z = rng.standard_normal((vol(L), 4, nc, 2))
    return np.ascontiguousarray(z[..., 0] + 1j * z[..., 1])
