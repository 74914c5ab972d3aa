"""Pins for the CPU oracle: the oracle is checked against what the theory fixes,
never against itself.  Everything the oracle is compared with here is typed out independently in
numpy: gamma matrices from the Pauli matrices, plane waves, np.roll-based plaquette leaves, a dense
matrix built from the element formula, closed forms.  No GPU.
"""
import itertools
import math

import numpy as np
import pytest

import oracle
from paper_2503_16994_b200 import synth

PAULI = [np.array([[0, 1], [1, 0]], dtype=complex),
         np.array([[0, -1j], [1j, 0]], dtype=complex),
         np.array([[1, 0], [0, -1]], dtype=complex)]
Z2 = np.zeros((2, 2), dtype=complex)
I2 = np.eye(2, dtype=complex)
# D2, typed independently of the oracle
GAMMA = [np.block([[Z2, -1j * s], [1j * s, Z2]]) for s in PAULI] + [np.block([[Z2, I2], [I2, Z2]])]
GAMMA5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(complex)


def lat(arr, L, tail):
    """[V, ...] -> [x4, x3, x2, x1, ...]"""
    return arr.reshape((L[3], L[2], L[1], L[0]) + tuple(tail))


def sh(a, mu, d):
    """field at x + d*mu_hat (periodic)"""
    return np.roll(a, -d, axis=3 - mu)


def mm(a, b):
    return a @ b


def dg(a):
    return np.conj(np.swapaxes(a, -1, -2))


def fhat_numpy(L, U, mu, nu):
    """D4 with whole-lattice shifts (periodic): independent of the oracle's per-site index code."""
    u = lat(U, L, (4, 3, 3))
    Um, Un = u[..., mu, :, :], u[..., nu, :, :]
    l1 = mm(mm(Um, sh(Un, mu, 1)), mm(dg(sh(Um, nu, 1)), dg(Un)))
    l2 = mm(mm(Un, dg(sh(sh(Um, mu, -1), nu, 1))), mm(dg(sh(Un, mu, -1)), sh(Um, mu, -1)))
    l3 = mm(mm(dg(sh(Um, mu, -1)), dg(sh(sh(Un, mu, -1), nu, -1))),
            mm(sh(sh(Um, mu, -1), nu, -1), sh(Un, nu, -1)))
    l4 = mm(mm(dg(sh(Un, nu, -1)), sh(Um, nu, -1)), mm(sh(sh(Un, mu, 1), nu, -1), dg(Um)))
    Q = l1 + l2 + l3 + l4
    return ((Q - dg(Q)) / 8.0).reshape(-1, 3, 3)


def clover_numpy(L, U, kappa, csw):
    """D5 as dense [V,12,12] from fhat_numpy and sigma = (i/2)[gamma,gamma]."""
    V = synth.vol(L)
    A = np.tile(np.eye(12, dtype=complex), (V, 1, 1))
    for mu in range(4):
        for nu in range(4):
            if mu == nu:
                continue
            sig = 0.5j * (GAMMA[mu] @ GAMMA[nu] - GAMMA[nu] @ GAMMA[mu])
            F = fhat_numpy(L, U, mu, nu)
            A += kappa * csw * 0.5j * np.einsum("st,nab->nsatb", sig, F).reshape(V, 12, 12)
    return A


def dense_dirac(L, U, kappa, theta, A12=None):
    """Element formula of D6 on a periodic lattice: a [12V, 12V] matrix, index 12*n + 3*s + a."""
    V = synth.vol(L)
    M = np.zeros((12 * V, 12 * V), dtype=complex)
    th = [np.exp(1j * theta[mu] / L[mu]) for mu in range(4)]
    for n in range(V):
        x = [n % L[0], (n // L[0]) % L[1], (n // (L[0] * L[1])) % L[2], n // (L[0] * L[1] * L[2])]
        M[12 * n:12 * n + 12, 12 * n:12 * n + 12] += np.eye(12) if A12 is None else A12[n]
        for mu in range(4):
            xp = list(x)
            xp[mu] = (x[mu] + 1) % L[mu]
            xm = list(x)
            xm[mu] = (x[mu] - 1) % L[mu]
            npl, nmi = synth.site_index(L, xp), synth.site_index(L, xm)
            M[12 * n:12 * n + 12, 12 * npl:12 * npl + 12] += -kappa * th[mu] * np.kron(np.eye(4) - GAMMA[mu], U[n, mu])
            M[12 * n:12 * n + 12, 12 * nmi:12 * nmi + 12] += -kappa * np.conj(th[mu]) * np.kron(
                np.eye(4) + GAMMA[mu], U[nmi, mu].conj().T)
    return M


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def inner(a, b):
    return np.vdot(a, b)


# ------------------------------------------------------------------------------------------------
def test_gamma_algebra_D2():
    g = [oracle.gamma(mu) for mu in range(4)]
    g5 = oracle.gamma(4)
    for mu in range(4):
        assert np.array_equal(g[mu], GAMMA[mu])
        assert np.allclose(g[mu], g[mu].conj().T)
        for nu in range(4):
            assert np.allclose(g[mu] @ g[nu] + g[nu] @ g[mu], 2 * (mu == nu) * np.eye(4))
    assert np.allclose(g5, g[0] @ g[1] @ g[2] @ g[3])
    assert np.allclose(g5, GAMMA5)
    # sigma_ij = -eps_ijk diag(sigma_k, sigma_k);  sigma_k4 = diag(sigma_k, -sigma_k)
    eps = {(0, 1): (2, 1), (1, 2): (0, 1), (2, 0): (1, 1)}
    for (i, j), (k, sgn) in eps.items():
        want = -sgn * np.block([[PAULI[k], Z2], [Z2, PAULI[k]]])
        assert np.allclose(oracle.sigma(i, j), want)
        assert np.allclose(oracle.sigma(j, i), -want)
    for k in range(3):
        assert np.allclose(oracle.sigma(k, 3), np.block([[PAULI[k], Z2], [Z2, -PAULI[k]]]))


def test_generators():
    L = (4, 4, 4, 4)
    U = synth.haar_gauge(L, 11)
    W = U.reshape(-1, 3, 3)
    assert np.allclose(W @ dg(W), np.eye(3), atol=1e-13)
    assert np.allclose(np.linalg.det(W), 1.0, atol=1e-13)
    assert abs(oracle.plaquette(L, U)) < 0.05  # Haar: <plaq> = 0
    S = synth.smooth_gauge(L, 12).reshape(-1, 3, 3)
    assert np.allclose(S @ dg(S), np.eye(3), atol=1e-13)
    assert np.allclose(np.linalg.det(S), 1.0, atol=1e-13)
    one = np.tile(np.eye(3, dtype=complex), (synth.vol(L), 4, 1, 1))
    assert abs(oracle.plaquette(L, one) - 1.0) < 1e-15


def test_P11_generator_plaquette():
    # independent links U = exp(i eps H): <plaq> = c(eps)^4 with c = <Re Tr U>/3 ; eps = 0.4322 -> 0.600
    L = (8, 8, 8, 8)
    U = synth.smooth_gauge(L, 5000)
    c = np.mean(np.trace(U.reshape(-1, 3, 3), axis1=1, axis2=2).real) / 3.0
    plaq = oracle.plaquette(L, U)
    assert abs(plaq - c ** 4) < 3e-3
    assert abs(plaq - 0.600) < 5e-3


@pytest.mark.parametrize("theta", [(0.0, 0.0, 0.0, 0.0), (0.5, 0.5, 0.5, math.pi), (0.3, -0.7, 1.1, 0.2)])
def test_P1_free_field(theta):
    L = (4, 6, 4, 8)
    V = synth.vol(L)
    kappa = 0.124
    U = np.tile(np.eye(3, dtype=complex), (V, 4, 1, 1))
    rng = np.random.default_rng(3)
    # clover vanishes identically on U = 1 even with csw != 0
    A = oracle.clover_blocks(L, U, kappa, 1.7)
    assert np.abs(A - np.eye(6)).max() == 0.0
    n = np.arange(V)
    xs = [n % L[0], (n // L[0]) % L[1], (n // (L[0] * L[1])) % L[2], n // (L[0] * L[1] * L[2])]
    for mom in [(0, 0, 0, 0), (1, 0, 0, 0), (0, 2, 0, 0), (0, 0, 1, 0), (0, 0, 0, 3), (1, 5, 2, 7), (3, 1, 3, 2)]:
        p = [2 * math.pi * mom[mu] / L[mu] for mu in range(4)]
        pt = [p[mu] + theta[mu] / L[mu] for mu in range(4)]
        u = rng.standard_normal(12) + 1j * rng.standard_normal(12)
        phase = np.exp(1j * sum(p[mu] * xs[mu] for mu in range(4)))
        psi = (phase[:, None] * u[None, :]).reshape(V, 4, 3)
        scal = 1 - 2 * kappa * sum(math.cos(t) for t in pt)
        gs = sum(math.sin(pt[mu]) * GAMMA[mu] for mu in range(4))
        Dm = np.kron(scal * np.eye(4) + 2j * kappa * gs, np.eye(3))
        want = (phase[:, None] * (Dm @ u)[None, :]).reshape(V, 4, 3)
        got = oracle.dw(L, U, psi, kappa, Ablk=A, theta=theta)
        npsi = np.linalg.norm(psi)  # errors relative to |psi|: (1 - 2k sum cos) nearly cancels at p = 0
        assert np.linalg.norm(got - want) / npsi < 1e-14
        # D^dagger on a plane wave: hermitian conjugate of the momentum-space matrix
        wantd = (phase[:, None] * (Dm.conj().T @ u)[None, :]).reshape(V, 4, 3)
        gotd = oracle.dw(L, U, psi, kappa, Ablk=A, theta=theta, dagger=True)
        assert np.linalg.norm(gotd - wantd) / npsi < 1e-14
        # D^+ D = (1 - 2k sum cos)^2 + 4 k^2 sum sin^2
        dd = scal ** 2 + 4 * kappa ** 2 * sum(math.sin(t) ** 2 for t in pt)
        assert np.linalg.norm(oracle.dw(L, U, got, kappa, theta=theta, dagger=True) - dd * psi) / npsi < 1e-14


def test_P1_free_field_cg():
    # D^-1 = [(1 - 2k sum cos) - 2k i sum gamma sin] / (D^+D scalar) on a plane wave
    L = (4, 4, 4, 4)
    V = synth.vol(L)
    kappa = 0.11
    theta = (0.5, 0.5, 0.5, math.pi)
    U = np.tile(np.eye(3, dtype=complex), (V, 4, 1, 1))
    n = np.arange(V)
    xs = [n % L[0], (n // L[0]) % L[1], (n // (L[0] * L[1])) % L[2], n // (L[0] * L[1] * L[2])]
    mom = (1, 0, 2, 3)
    p = [2 * math.pi * mom[mu] / L[mu] for mu in range(4)]
    pt = [p[mu] + theta[mu] / L[mu] for mu in range(4)]
    u = np.arange(1, 13) * (1 - 0.5j)
    phase = np.exp(1j * sum(p[mu] * xs[mu] for mu in range(4)))
    b = (phase[:, None] * u[None, :]).reshape(V, 4, 3)
    scal = 1 - 2 * kappa * sum(math.cos(t) for t in pt)
    gs = sum(math.sin(pt[mu]) * GAMMA[mu] for mu in range(4))
    dd = scal ** 2 + 4 * kappa ** 2 * sum(math.sin(t) ** 2 for t in pt)
    Dinv = np.kron((scal * np.eye(4) - 2j * kappa * gs) / dd, np.eye(3))
    want = (phase[:, None] * (Dinv @ u)[None, :]).reshape(V, 4, 3)
    x, it, rn, rt = oracle.cg(L, U, b, kappa, theta=theta, tol=1e-14)
    assert it >= 0
    assert rel(x, want) < 1e-13


BCS = [(oracle.BC_PERIODIC, None), (oracle.BC_OPEN, None), (oracle.BC_SF_ORBI, synth.SF_PHIT)]


def interior_mask(L, bc):
    x4 = np.arange(synth.vol(L)) // (L[0] * L[1] * L[2])
    if bc == oracle.BC_OPEN:
        return (x4 != 0) & (x4 != L[3] - 1)
    if bc in (oracle.BC_SF_ORBI, oracle.BC_SF_AFWB):
        return x4 != 0
    return np.ones(synth.vol(L), dtype=bool)


@pytest.mark.parametrize("bc,phiT", BCS)
def test_P2_gamma5_hermiticity(bc, phiT):
    L = (4, 4, 4, 6)
    kappa, csw = 0.13, 1.3
    theta = (0.5, -0.2, 0.1, 0.9)
    U = synth.haar_gauge(L, 21)
    if bc == oracle.BC_SF_ORBI:
        U = synth.apply_sf_boundary(L, U)
    A12 = oracle.clover_dense(L, U, kappa, csw, bc=bc, phiT=phiT)
    # A hermitian, commutes with gamma5 (chirally block diagonal) -- exactly zero off-blocks
    assert np.abs(A12 - np.conj(np.swapaxes(A12, 1, 2))).max() < 1e-15
    assert np.abs(A12[:, :6, 6:]).max() == 0.0 and np.abs(A12[:, 6:, :6]).max() == 0.0
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=phiT)
    assert np.array_equal(A[:, 0], A12[:, :6, :6]) and np.array_equal(A[:, 1], A12[:, 6:, 6:])
    # trace of each block is 6 (sigma traceless)
    assert np.abs(np.trace(A, axis1=2, axis2=3) - 6.0).max() < 1e-13
    psi = synth.gaussian_spinor(L, 22)
    chi = synth.gaussian_spinor(L, 23)
    lhs = inner(chi, oracle.dw(L, U, psi, kappa, Ablk=A, bc=bc, theta=theta))
    rhs = inner(oracle.dw(L, U, chi, kappa, Ablk=A, bc=bc, theta=theta, dagger=True), psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-14
    # D^+ equals gamma5 D gamma5 computed outside the oracle
    g5 = np.array([1, 1, -1, -1.0])[None, :, None]
    viaD = g5 * oracle.dw(L, U, g5 * chi, kappa, Ablk=A, bc=bc, theta=theta)
    assert rel(oracle.dw(L, U, chi, kappa, Ablk=A, bc=bc, theta=theta, dagger=True), viaD) < 1e-15


@pytest.mark.parametrize("bc,phiT", BCS)
def test_P3_gauge_covariance(bc, phiT):
    L = (4, 4, 4, 6)
    V = synth.vol(L)
    kappa, csw = 0.13, 1.9
    theta = (0.5, 0.5, 0.5, 0.3)
    U = synth.smooth_gauge(L, 31, eps=0.9)
    if bc == oracle.BC_SF_ORBI:
        U = synth.apply_sf_boundary(L, U)
    g = synth.random_su3_field(L, 32)
    if bc != oracle.BC_PERIODIC:
        # gauge transformations fixed to 1 on the boundary slices (R8)
        g = lat(g, L, (3, 3)).copy()
        g[0] = np.eye(3)
        if bc == oracle.BC_OPEN:
            g[-1] = np.eye(3)
        g = g.reshape(V, 3, 3)
    gl = lat(g, L, (3, 3))
    Ul = lat(U, L, (4, 3, 3))
    Up = np.empty_like(Ul)
    for mu in range(4):
        gsh = sh(gl, mu, 1)
        if bc == oracle.BC_SF_ORBI and mu == 3:
            gsh = gsh.copy()
            gsh[-1] = np.eye(3)  # g(x4 = T) = 1 on the unstored boundary slice
        Up[..., mu, :, :] = gl @ Ul[..., mu, :, :] @ dg(gsh)
    Up = Up.reshape(V, 4, 3, 3)
    psi = synth.gaussian_spinor(L, 33)
    psip = np.einsum("nab,nsb->nsa", g, psi)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=phiT)
    Ap = oracle.clover_blocks(L, Up, kappa, csw, bc=bc, phiT=phiT)
    lhs = oracle.dw(L, Up, psip, kappa, Ablk=Ap, bc=bc, theta=theta)
    rhs = np.einsum("nab,nsb->nsa", g, oracle.dw(L, U, psi, kappa, Ablk=A, bc=bc, theta=theta))
    assert rel(lhs, rhs) < 1e-14
    # F' = g F g^+ at a few sites
    for x in [(1, 2, 3, 2), (0, 0, 0, 1), (3, 3, 3, L[3] - 2)]:
        n = synth.site_index(L, x)
        F = oracle.fhat_site(L, U, x, 1, 3, bc=bc, phiT=phiT)
        Fp = oracle.fhat_site(L, Up, x, 1, 3, bc=bc, phiT=phiT)
        assert np.abs(Fp - g[n] @ F @ g[n].conj().T).max() < 1e-14


def test_fhat_vs_numpy_rolls():
    L = (4, 6, 4, 4)
    U = synth.haar_gauge(L, 41)
    for mu, nu in itertools.permutations(range(4), 2):
        F = fhat_numpy(L, U, mu, nu)
        for x in [(0, 0, 0, 0), (3, 5, 3, 3), (1, 2, 3, 0), (2, 0, 1, 3)]:
            got = oracle.fhat_site(L, U, x, mu, nu)
            assert np.abs(got - F[synth.site_index(L, x)]).max() < 1e-14
    A = oracle.clover_dense(L, U, 0.12, 1.5)
    assert np.abs(A - clover_numpy(L, U, 0.12, 1.5)).max() < 1e-13


@pytest.mark.parametrize("csw", [0.0, 1.0])
def test_P4_dense_matrix_2to4(csw):
    L = (2, 2, 2, 2)
    kappa = 0.125
    theta = (0.0, 0.0, 0.0, math.pi)
    U = synth.haar_gauge(L, 51)
    A12 = clover_numpy(L, U, kappa, csw)
    M = dense_dirac(L, U, kappa, theta, A12)
    A = oracle.clover_blocks(L, U, kappa, csw)
    psi = synth.gaussian_spinor(L, 52)
    got = oracle.dw(L, U, psi, kappa, Ablk=A, theta=theta)
    assert rel(got.reshape(-1), M @ psi.reshape(-1)) < 1e-14
    gotd = oracle.dw(L, U, psi, kappa, Ablk=A, theta=theta, dagger=True)
    assert rel(gotd.reshape(-1), M.conj().T @ psi.reshape(-1)) < 1e-14
    G5 = np.kron(np.eye(16), np.kron(GAMMA5, np.eye(3)))
    assert np.abs(G5 @ M @ G5 - M.conj().T).max() < 1e-14
    # P8: CG = dense inverse
    b = synth.gaussian_spinor(L, 53)
    want = np.linalg.solve(M, b.reshape(-1))
    x, it, rn, rt = oracle.cg(L, U, b, kappa, Ablk=A, theta=theta, tol=1e-13, maxiter=2000)
    assert it > 0
    cond = np.linalg.cond(M)
    assert rel(x.reshape(-1), want) < 10 * cond * 1e-13
    assert rt < 1e-11 and rn < 1e-12


def test_P4_dense_matrix_L2_mixed():
    # L = 2 in some directions only (x + mu and x - mu coincide there: both hops are applied, R13)
    L = (2, 4, 2, 4)
    kappa = 0.12
    theta = (0.4, 0.0, -0.3, 1.0)
    U = synth.haar_gauge(L, 54)
    M = dense_dirac(L, U, kappa, theta, clover_numpy(L, U, kappa, 1.2))
    A = oracle.clover_blocks(L, U, kappa, 1.2)
    psi = synth.gaussian_spinor(L, 55)
    assert rel(oracle.dw(L, U, psi, kappa, Ablk=A, theta=theta).reshape(-1), M @ psi.reshape(-1)) < 1e-14


@pytest.mark.parametrize("plane", [(0, 1), (0, 2), (1, 2), (0, 3), (1, 3), (2, 3)])
def test_P5_constant_flux(plane):
    """U_mu(x) = exp(-i phi x_nu t), U_nu(x) = exp(+i phi L_nu x_mu t) on x_nu = L_nu - 1 (else 1),
    t = diag(1,1,-2), phi = 2 pi m/(L_mu L_nu): every mu-nu plaquette is exp(i phi t), so
    F^_{mu nu} = i sin(phi t), all other planes 0, and
    A = 1 + kappa csw (i/2)(sigma_{mu nu} F_{mu nu} + sigma_{nu mu} F_{nu mu}) = 1 - kappa csw sigma_{mu nu} (x) sin(phi t)."""
    mu, nu = plane
    L = (4, 6, 4, 8)
    V = synth.vol(L)
    m = 1
    phi = 2 * math.pi * m / (L[mu] * L[nu])
    t = np.array([1.0, 1.0, -2.0])
    n = np.arange(V)
    xs = [n % L[0], (n // L[0]) % L[1], (n // (L[0] * L[1])) % L[2], n // (L[0] * L[1] * L[2])]
    U = np.tile(np.eye(3, dtype=complex), (V, 4, 1, 1))
    for a in range(3):
        U[:, mu, a, a] = np.exp(-1j * phi * xs[nu] * t[a])
        U[:, nu, a, a] = np.where(xs[nu] == L[nu] - 1, np.exp(1j * phi * L[nu] * xs[mu] * t[a]), 1.0)
    kappa, csw = 0.137, 1.9
    Fwant = np.diag(1j * np.sin(phi * t))
    for x in [(0, 0, 0, 0), (3, 5, 3, 7), (1, 2, 0, 4)]:
        assert np.abs(oracle.fhat_site(L, U, x, mu, nu) - Fwant).max() < 1e-15
        assert np.abs(oracle.fhat_site(L, U, x, nu, mu) + Fwant).max() < 1e-15
        for (a, b) in itertools.combinations(range(4), 2):
            if (a, b) != (mu, nu):
                assert np.abs(oracle.fhat_site(L, U, x, a, b)).max() < 1e-15
    sig = 0.5j * (GAMMA[mu] @ GAMMA[nu] - GAMMA[nu] @ GAMMA[mu])
    want = np.eye(12) - kappa * csw * np.kron(sig, np.diag(np.sin(phi * t)))
    A12 = oracle.clover_dense(L, U, kappa, csw)
    assert np.abs(A12 - want[None]).max() < 1e-15
    # closed form in the chiral blocks (D5): sigma_12 = -diag(s3,s3) => A+- = 1 + k csw s3 (x) sin(phi t);
    # sigma_k4 = diag(s_k,-s_k) => A+ = 1 - k csw s_k (x) sin, A- = 1 + k csw s_k (x) sin
    A = oracle.clover_blocks(L, U, kappa, csw)
    s = np.diag(np.sin(phi * t))
    if nu == 3:
        wp = np.eye(6) - kappa * csw * np.kron(PAULI[mu], s)
        wm = np.eye(6) + kappa * csw * np.kron(PAULI[mu], s)
    else:
        k = {(0, 1): 2, (1, 2): 0, (0, 2): 1}[plane]
        sgn = -1.0 if plane == (0, 2) else 1.0  # sigma_13 = -sigma_31 = +diag(s2,s2)
        wp = wm = np.eye(6) + sgn * kappa * csw * np.kron(PAULI[k], s)
    assert np.abs(A[:, 0] - wp[None]).max() < 1e-15
    assert np.abs(A[:, 1] - wm[None]).max() < 1e-15


def test_P6_antiperiodic_equivalence():
    # theta_4 = pi distributed over all time links == (-1) on the wrap link after psi -> exp(i pi x4/L4) psi
    L = (4, 4, 4, 6)
    V = synth.vol(L)
    kappa = 0.125
    U = synth.haar_gauge(L, 61)
    psi = synth.gaussian_spinor(L, 62)
    A = oracle.clover_blocks(L, U, kappa, 1.0)
    x4 = np.arange(V) // (L[0] * L[1] * L[2])
    ph = np.exp(1j * math.pi * x4 / L[3])[:, None, None]
    Uw = U.copy()
    Uw[x4 == L[3] - 1, 3] *= -1.0
    lhs = oracle.dw(L, U, psi, kappa, Ablk=A, theta=(0, 0, 0, math.pi))
    rhs = oracle.dw(L, Uw, ph * psi, kappa, Ablk=A) / ph
    assert rel(lhs, rhs) < 1e-14


@pytest.mark.parametrize("bc,phiT", BCS[1:])
def test_P7_dirichlet_structure(bc, phiT):
    L = (4, 4, 4, 8)
    V = synth.vol(L)
    kappa, csw = 0.1365, 1.9
    theta = (0.5, 0.5, 0.5, 0.0)
    U = synth.smooth_gauge(L, 71)
    if bc == oracle.BC_SF_ORBI:
        U = synth.apply_sf_boundary(L, U)
    inter = interior_mask(L, bc)
    x4 = np.arange(V) // (L[0] * L[1] * L[2])
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=phiT)
    assert np.array_equal(A[~inter], np.tile(np.eye(6, dtype=complex), ((~inter).sum(), 2, 1, 1)))
    psi = synth.gaussian_spinor(L, 72)
    out = oracle.dw(L, U, psi, kappa, Ablk=A, bc=bc, theta=theta)
    assert np.all(out[~inter] == 0)
    # NaN on the frozen slices of the input must not leak
    bad = psi.copy()
    bad[~inter] = np.nan
    assert np.array_equal(oracle.dw(L, U, bad, kappa, Ablk=A, bc=bc, theta=theta), out)
    assert np.array_equal(oracle.dw(L, U, bad, kappa, Ablk=A, bc=bc, theta=theta, dagger=True),
                          oracle.dw(L, U, psi, kappa, Ablk=A, bc=bc, theta=theta, dagger=True))
    Un = U.copy()
    Un[x4 == L[3] - 1, 3] = np.nan
    if bc == oracle.BC_OPEN:
        # wrap-around time links are never used: neither by H nor by the leaves
        An = oracle.clover_blocks(L, Un, kappa, csw, bc=bc)
        assert np.array_equal(An, A)
        assert np.array_equal(oracle.dw(L, Un, psi, kappa, Ablk=An, bc=bc, theta=theta), out)
    else:
        # SF: the stored time links on the last slice ARE used, but only by the leaves at x4 = L4-1
        An = oracle.clover_blocks(L, Un, kappa, csw, bc=bc, phiT=phiT)
        changed = np.isnan(An).any(axis=(1, 2, 3))
        assert changed.any() and np.all(x4[changed] == L[3] - 1)
        assert np.array_equal(oracle.dw(L, Un, psi, kappa, Ablk=A, bc=bc, theta=theta), out)
        # changing phiT changes A only on the last slice
        A2 = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=(0.3, -0.1, -0.2))
        diff = np.abs(A2 - A).max(axis=(1, 2, 3)) > 0
        assert diff.any() and np.all(x4[diff] == L[3] - 1)
        # equivalence SF(L4) == Dirichlet on L4+1 slices whose last slice carries W' (R8)
        L5 = (L[0], L[1], L[2], L[3] + 1)
        n3 = L[0] * L[1] * L[2]
        U5 = np.concatenate([U, np.tile(np.eye(3, dtype=complex), (n3, 4, 1, 1))])
        for mu in range(3):
            U5[V:, mu] = synth.sf_boundary_links(L, phiT, mu)
        A5 = oracle.clover_blocks(L5, U5, kappa, csw, bc=oracle.BC_OPEN)
        assert np.abs(A5[:V] - A).max() < 1e-15
        psi5 = np.concatenate([psi, np.zeros((n3, 4, 3))])
        th5 = tuple(theta[mu] * L5[mu] / L[mu] for mu in range(4))
        out5 = oracle.dw(L5, U5, psi5, kappa, Ablk=A5, bc=oracle.BC_OPEN, theta=th5)
        assert rel(out5[:V], out) < 1e-15
    # D^+D positive definite on the interior: CG converges, solution exactly 0 on frozen slices
    b = synth.point_source(L, (0, 0, 0, L[3] // 2), 1, 2)
    x, it, rn, rt = oracle.cg(L, U, b, kappa, Ablk=A, bc=bc, theta=theta, tol=1e-10, maxiter=5000)
    assert it > 0 and rn < 2e-10
    assert np.all(x[~inter] == 0)


def test_R10_ct_term_linear():
    # ct = 1 is absent; the term is 2 kappa (ct-1) on the slices next to frozen ones ("parity unpinned"
    # beyond this structure: the paper only names cF)
    L = (4, 4, 4, 6)
    kappa = 0.13
    U = synth.smooth_gauge(L, 81)
    x4 = np.arange(synth.vol(L)) // 64
    A1 = oracle.clover_blocks(L, U, kappa, 1.5, bc=oracle.BC_OPEN, ct=1.0)
    A2 = oracle.clover_blocks(L, U, kappa, 1.5, bc=oracle.BC_OPEN, ct=1.25)
    d = A2 - A1
    want = np.zeros_like(d)
    want[(x4 == 1) | (x4 == L[3] - 2)] = 2 * kappa * 0.25 * np.eye(6)
    assert np.abs(d - want).max() < 1e-15


@pytest.mark.parametrize("bc,phiT", BCS)
def test_P10_even_odd_equals_full(bc, phiT):
    L = (4, 4, 4, 4) if bc == oracle.BC_PERIODIC else (4, 4, 4, 8)
    kappa, csw = 0.1355, 1.8
    theta = (0.5, 0.5, 0.5, 0.0)
    U = synth.smooth_gauge(L, 91)
    if bc == oracle.BC_SF_ORBI:
        U = synth.apply_sf_boundary(L, U)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=phiT)
    Ai = oracle.clover_inverse(L, A)
    assert np.abs(np.einsum("ncij,ncjk->ncik", A, Ai) - np.eye(6)).max() < 1e-13
    b = synth.gaussian_spinor(L, 92)
    inter = interior_mask(L, bc)
    x_full, it_f, _, rt_f = oracle.cg(L, U, b, kappa, Ablk=A, bc=bc, theta=theta, tol=1e-12)
    x_eo, it_e, _, rt_e = oracle.cg_eo(L, U, b, kappa, A, Ai, bc=bc, theta=theta, tol=1e-12)
    assert it_f > 0 and it_e > 0 and it_e < it_f
    assert rel(x_eo[inter], x_full[inter]) < 1e-10
    assert rt_e < 1e-10
    # D^ is gamma5-hermitian on the even sublattice
    psi = synth.gaussian_spinor(L, 93)
    chi = synth.gaussian_spinor(L, 94)
    n = np.arange(synth.vol(L))
    par = (n % L[0] + (n // L[0]) % L[1] + (n // (L[0] * L[1])) % L[2] + n // (L[0] * L[1] * L[2])) % 2
    psi[par == 1] = 0
    chi[par == 1] = 0
    lhs = inner(chi, oracle.dhat(L, U, psi, kappa, A, Ai, bc=bc, theta=theta))
    rhs = inner(oracle.dhat(L, U, chi, kappa, A, Ai, bc=bc, theta=theta, dagger=True), psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13


def test_dw_at_sites_matches_field():
    L = (4, 4, 6, 8)
    kappa, csw = 0.137, 1.9
    theta = (0.1, 0.2, 0.3, 0.4)
    U = synth.smooth_gauge(L, 95)
    psi = synth.gaussian_spinor(L, 96)
    A = oracle.clover_blocks(L, U, kappa, csw)
    sites = np.array([0, 1, 17, synth.vol(L) - 1, 300, 301], dtype=np.int64)
    for dagger in (False, True):
        full = oracle.dw(L, U, psi, kappa, Ablk=A, theta=theta, dagger=dagger)
        some = oracle.dw_at_sites(L, U, psi, sites, kappa, csw, theta=theta, dagger=dagger)
        assert np.array_equal(some, full[sites])


def test_P12_free_field_pseudoscalar_correlator():
    """NEXT-2 pin: on U = 1 the point-source propagator is the inverse lattice Fourier transform of
    D(p)^-1 = [(1 - 2k sum cos p) - 2k i sum gamma sin p] / [(1 - 2k sum cos p)^2 + 4 k^2 sum sin^2 p] (P1), so
    C(x4) = sum_xvec Tr S^+ S is known in closed form: it pins point source + CG + contraction together
    (theta_4 = pi: antiperiodic in time, the momenta shift by theta/L)."""
    L = (4, 4, 4, 8)
    V = synth.vol(L)
    kappa = 0.115
    theta = (0.0, 0.0, 0.0, math.pi)
    U = np.tile(np.eye(3, dtype=complex), (V, 4, 1, 1))
    # momentum-space propagator on the grid p_mu = (2 pi n_mu + theta_mu) / L_mu, array index order [n4, n3, n2, n1]
    grids = np.meshgrid(*[(2 * math.pi * np.arange(L[mu]) + theta[mu]) / L[mu] for mu in (3, 2, 1, 0)], indexing="ij")
    p = {3: grids[0], 2: grids[1], 1: grids[2], 0: grids[3]}
    a = 1 - 2 * kappa * sum(np.cos(p[mu]) for mu in range(4))
    den = a ** 2 + 4 * kappa ** 2 * sum(np.sin(p[mu]) ** 2 for mu in range(4))
    Sp = a[..., None, None] * np.eye(4) - 2j * kappa * sum(np.sin(p[mu])[..., None, None] * GAMMA[mu] for mu in range(4))
    Sp = Sp / den[..., None, None]
    # S(x) = (1/V) sum_p e^{i p x} S(p);  the theta part of p is the twist phase e^{i theta_mu x_mu / L_mu}
    Sx = np.fft.ifftn(Sp, axes=(0, 1, 2, 3))
    x4 = np.arange(L[3]).reshape(-1, 1, 1, 1)
    Sx = Sx * np.exp(1j * theta[3] * x4 / L[3])[..., None, None]
    want = 3.0 * (np.abs(Sx) ** 2).sum(axis=(1, 2, 3, 4, 5))     # 3 colours x spin trace, per time slice
    cols = []
    for spin in range(4):
        for colour in range(3):
            b = synth.point_source(L, (0, 0, 0, 0), spin, colour)
            x, it, _, _ = oracle.cg(L, U, b, kappa, None, theta=theta, tol=1e-13)
            assert it > 0
            cols.append(x)
    got = oracle.correlator_ps(L, np.array(cols))
    assert np.max(np.abs(got - want) / want) < 1e-9
    assert got[0] > got[1] > got[2] > got[3] > got[4]            # decays away from the source, symmetric in time
    assert np.allclose(got[1:4], got[:4:-1][:3], rtol=1e-9)


def test_correlator_slice_mapping_and_sum_rule():
    """x4 is the slowest canonical index (D1): a field living on one time slice contributes to that entry only;
    sum_t C(t) = sum of the squared norms of the columns."""
    L = (4, 6, 2, 8)
    V = synth.vol(L)
    V3 = L[0] * L[1] * L[2]
    rng = np.random.default_rng(7)
    cols = rng.standard_normal((3, V, 4, 3)) + 1j * rng.standard_normal((3, V, 4, 3))
    C = oracle.correlator_ps(L, cols)
    assert abs(C.sum() - np.linalg.norm(cols) ** 2) / C.sum() < 1e-14
    one = np.zeros_like(cols)
    one[:, 5 * V3:6 * V3] = cols[:, 5 * V3:6 * V3]
    C1 = oracle.correlator_ps(L, one)
    assert C1[5] == C[5] and np.count_nonzero(C1) == 1


@pytest.mark.parametrize("mu", [0.05, -0.3])
def test_P13_twisted_mass(mu):
    """NEXT-4 pin ("mu is the twisted mass"): D = A + 2 i kappa mu gamma5 - kappa H.
    Free field: D(p) = a + 2 i kappa (gamma.sin p) + 2 i kappa mu gamma5 and D^+ D = a^2 + 4 k^2 sum sin^2 + (2 k mu)^2
    (gamma5 anticommutes with every gamma_mu, so the cross terms cancel); D(mu)^+ = gamma5 D(-mu) gamma5 on an
    interacting field; and the term is exactly the difference to mu = 0."""
    L = (4, 4, 6, 4)
    V = synth.vol(L)
    kappa = 0.124
    U1 = np.tile(np.eye(3, dtype=complex), (V, 4, 1, 1))
    n = np.arange(V)
    xs = [n % L[0], (n // L[0]) % L[1], (n // (L[0] * L[1])) % L[2], n // (L[0] * L[1] * L[2])]
    rng = np.random.default_rng(5)
    for mom in [(0, 0, 0, 0), (1, 3, 2, 1), (2, 0, 5, 3)]:
        p = [2 * math.pi * mom[m] / L[m] for m in range(4)]
        u = rng.standard_normal(12) + 1j * rng.standard_normal(12)
        phase = np.exp(1j * sum(p[m] * xs[m] for m in range(4)))
        psi = (phase[:, None] * u[None, :]).reshape(V, 4, 3)
        a = 1 - 2 * kappa * sum(math.cos(t) for t in p)
        gs = sum(math.sin(p[m]) * GAMMA[m] for m in range(4))
        Dm = np.kron(a * np.eye(4) + 2j * kappa * gs + 2j * kappa * mu * GAMMA5, np.eye(3))
        want = (phase[:, None] * (Dm @ u)[None, :]).reshape(V, 4, 3)
        got = oracle.dw(L, U1, psi, kappa, mu=mu)
        assert np.linalg.norm(got - want) / np.linalg.norm(psi) < 1e-14
        wantd = (phase[:, None] * (Dm.conj().T @ u)[None, :]).reshape(V, 4, 3)
        assert np.linalg.norm(oracle.dw(L, U1, psi, kappa, mu=mu, dagger=True) - wantd) / np.linalg.norm(psi) < 1e-14
        dd = a ** 2 + 4 * kappa ** 2 * sum(math.sin(t) ** 2 for t in p) + (2 * kappa * mu) ** 2
        assert np.linalg.norm(oracle.dw(L, U1, got, kappa, mu=mu, dagger=True) - dd * psi) / np.linalg.norm(psi) < 1e-14
    # interacting field with clover term
    U = synth.smooth_gauge(L, 97)
    A = oracle.clover_blocks(L, U, kappa, 1.6)
    psi = synth.gaussian_spinor(L, 98)
    chi = synth.gaussian_spinor(L, 99)
    g5 = lambda v: v * np.array([1, 1, -1, -1])[None, :, None]
    lhs = oracle.dw(L, U, psi, kappa, A, mu=mu, dagger=True)
    rhs = g5(oracle.dw(L, U, g5(psi), kappa, A, mu=-mu))
    assert np.linalg.norm(lhs - rhs) / np.linalg.norm(rhs) < 1e-14
    # <chi, D psi> = <D^+ chi, psi>
    a1 = np.vdot(chi, oracle.dw(L, U, psi, kappa, A, mu=mu))
    a2 = np.vdot(oracle.dw(L, U, chi, kappa, A, mu=mu, dagger=True), psi)
    assert abs(a1 - a2) / abs(a1) < 1e-13
    diff = oracle.dw(L, U, psi, kappa, A, mu=mu) - oracle.dw(L, U, psi, kappa, A)
    assert np.linalg.norm(diff - 2j * kappa * mu * g5(psi)) / np.linalg.norm(psi) < 1e-15
    # CG on the normal equations of the twisted operator
    x, it, rn, rt = oracle.cg(L, U, psi, kappa, A, tol=1e-11, mu=mu)
    assert it > 0 and np.linalg.norm(oracle.dw(L, U, x, kappa, A, mu=mu) - psi) / np.linalg.norm(psi) < 1e-9
