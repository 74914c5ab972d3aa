"""Pins for the N-colour oracle of the SU(2) fundamental representation (oracle/lqcd_oracle_sun.cpp).

Two kinds.  (a) Its N = 3 instance against the separately pinned SU(3) oracle (lqcd_oracle.cpp, pins P1-P13): the two
files share no code, so agreement to rounding pins every index, sign and factor of the generic loops.  (b) The N = 2
instance against what the theory fixes, typed out in numpy here: Cayley-Dickson form, free-field closed form,
gamma5-hermiticity, SU(2) gauge covariance, a dense matrix built from the element formula on 2^4 with its inverse
against CG, np.roll plaquette leaves, and the constant-flux closed form with t = diag(1, -1).  No GPU.
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
GAMMA = [np.block([[Z2, -1j * s], [1j * s, Z2]]) for s in PAULI] + [np.block([[Z2, I2], [I2, Z2]])]   # D2
GAMMA5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(complex)
NC = 2


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def dg(a):
    return np.conj(np.swapaxes(a, -1, -2))


def sh(a, mu, d):
    return np.roll(a, -d, axis=3 - mu)


def fhat_numpy(L, U, mu, nu, nc):
    u = U.reshape((L[3], L[2], L[1], L[0], 4, nc, nc))
    Um, Un = u[..., mu, :, :], u[..., nu, :, :]
    l1 = Um @ sh(Un, mu, 1) @ dg(sh(Um, nu, 1)) @ dg(Un)
    l2 = Un @ dg(sh(sh(Um, mu, -1), nu, 1)) @ dg(sh(Un, mu, -1)) @ sh(Um, mu, -1)
    l3 = dg(sh(Um, mu, -1)) @ dg(sh(sh(Un, mu, -1), nu, -1)) @ sh(sh(Um, mu, -1), nu, -1) @ sh(Un, nu, -1)
    l4 = dg(sh(Un, nu, -1)) @ sh(Um, nu, -1) @ sh(sh(Un, mu, 1), nu, -1) @ dg(Um)
    Q = l1 + l2 + l3 + l4
    return ((Q - dg(Q)) / 8.0).reshape(-1, nc, nc)


def clover_numpy(L, U, kappa, csw, nc):
    V = synth.vol(L)
    A = np.tile(np.eye(4 * nc, dtype=complex), (V, 1, 1))
    for mu in range(4):
        for nu in range(4):
            if mu != nu:
                sig = 0.5j * (GAMMA[mu] @ GAMMA[nu] - GAMMA[nu] @ GAMMA[mu])
                A += kappa * csw * 0.5j * np.einsum("st,nab->nsatb", sig, fhat_numpy(L, U, mu, nu, nc)).reshape(V, 4 * nc, 4 * nc)
    return A


def dense_dirac(L, U, kappa, theta, nc, A=None):
    V, D = synth.vol(L), 4 * nc
    M = np.zeros((D * V, D * V), dtype=complex)
    th = [np.exp(1j * theta[mu] / L[mu]) for mu in range(4)]
    for n in range(V):
        x = [n % L[0], (n // L[0]) % L[1], (n // (L[0] * L[1])) % L[2], n // (L[0] * L[1] * L[2])]
        M[D * n:D * n + D, D * n:D * n + D] += np.eye(D) if A is None else A[n]
        for mu in range(4):
            xp, xm = list(x), list(x)
            xp[mu] = (x[mu] + 1) % L[mu]
            xm[mu] = (x[mu] - 1) % L[mu]
            npl, nmi = synth.site_index(L, xp), synth.site_index(L, xm)
            M[D * n:D * n + D, D * npl:D * npl + D] += -kappa * th[mu] * np.kron(np.eye(4) - GAMMA[mu], U[n, mu])
            M[D * n:D * n + D, D * nmi:D * nmi + D] += -kappa * np.conj(th[mu]) * np.kron(np.eye(4) + GAMMA[mu], U[nmi, mu].conj().T)
    return M


# ------------------------------------------------------------------------------------------------ (a) N = 3 == the SU(3) oracle
@pytest.mark.parametrize("bc", [oracle.BC_PERIODIC, oracle.BC_OPEN])
def test_generic_loops_equal_su3_oracle(bc):
    L = (4, 2, 6, 8)
    kappa, csw, theta = 0.131, 1.6, (0.5, -0.3, 0.2, 0.9)
    U = synth.haar_gauge(L, 901)
    psi = synth.gaussian_spinor(L, 902)
    A3 = oracle.clover_blocks(L, U, kappa, csw, bc=bc)
    An = oracle.sun_clover_blocks(3, L, U, kappa, csw, bc=bc)
    assert np.abs(An - A3).max() < 1e-14
    for dagger in (False, True):
        want = oracle.dw(L, U, psi, kappa, A3, bc=bc, theta=theta, dagger=dagger)
        got = oracle.sun_dw(3, L, U, psi, kappa, An, bc=bc, theta=theta, dagger=dagger)
        assert np.abs(got - want).max() < 1e-13
        assert np.abs(oracle.sun_dw(3, L, U, psi, kappa, None, bc=bc, theta=theta, dagger=dagger)
                      - oracle.dw(L, U, psi, kappa, None, bc=bc, theta=theta, dagger=dagger)).max() < 1e-13
    if bc == oracle.BC_PERIODIC:
        assert np.abs(oracle.sun_hop(3, L, U, psi, theta=theta) - oracle.hop(L, U, psi, theta=theta)).max() < 1e-13
        for (mu, nu) in itertools.permutations(range(4), 2):
            x = (1, 1, 5, 7)
            assert np.abs(oracle.sun_fhat_site(3, L, U, x, mu, nu) - oracle.fhat_site(L, U, x, mu, nu)).max() < 1e-15


def test_generic_cg_equals_su3_oracle():
    L, kappa, csw = (4, 4, 4, 8), 0.125, 1.0
    U = synth.smooth_gauge(L, 903)
    b = synth.point_source(L, (1, 2, 3, 4), 2, 1)
    for bc in (oracle.BC_PERIODIC, oracle.BC_OPEN):
        A = oracle.clover_blocks(L, U, kappa, csw, bc=bc)
        x3, it3, rn3, rt3 = oracle.cg(L, U, b, kappa, A, bc=bc, tol=1e-11)
        xn, itn, rnn, rtn = oracle.sun_cg(3, L, U, b, kappa, A, bc=bc, tol=1e-11)
        assert it3 > 0 and abs(itn - it3) <= 1
        assert rel(xn, x3) < 1e-9
        assert abs(rtn - rt3) <= 0.2 * rt3 + 1e-15


# ------------------------------------------------------------------------------------------------ (b) N = 2
def test_cayley_dickson_and_generators():
    L = (4, 4, 4, 4)
    for z in (synth.haar_su2_cd(L, 911), synth.smooth_su2_cd(L, 912)):
        assert np.allclose(np.abs(z[..., 0]) ** 2 + np.abs(z[..., 1]) ** 2, 1.0, atol=1e-14)
        W = oracle.su2_from_cayley_dickson(z).reshape(-1, 2, 2)
        assert np.array_equal(W, synth.su2_matrices(z).reshape(-1, 2, 2))
        assert np.allclose(W @ dg(W), np.eye(2), atol=1e-14)
        assert np.allclose(np.linalg.det(W), 1.0, atol=1e-14)
    # the smooth generator: U = exp(i eps H) against the matrix exponential by eigendecomposition; plaquette ~ 0.6
    rng = np.random.Generator(np.random.PCG64(912))
    h = rng.standard_normal((synth.vol(L) * 4, 3))[:5]
    for k in range(5):
        H = sum(h[k, a] * PAULI[a] / 2 for a in range(3))
        w, v = np.linalg.eigh(H)
        want = v @ np.diag(np.exp(1j * 0.55 * w)) @ v.conj().T
        assert np.abs(synth.su2_matrices(synth.smooth_su2_cd(L, 912)).reshape(-1, 2, 2)[k] - want).max() < 1e-14
    U = synth.su2_matrices(synth.smooth_su2_cd((8, 8, 8, 8), 913))
    u = U.reshape(8, 8, 8, 8, 4, 2, 2)
    plaq = np.mean([np.trace(u[..., m, :, :] @ sh(u[..., n, :, :], m, 1) @ dg(sh(u[..., m, :, :], n, 1)) @ dg(u[..., n, :, :]),
                             axis1=-2, axis2=-1).real.mean() / 2 for m in range(4) for n in range(m + 1, 4)])
    assert abs(plaq - 0.6) < 0.03


@pytest.mark.parametrize("theta", [(0.0, 0.0, 0.0, 0.0), (0.5, 0.5, 0.5, math.pi)])
def test_P1_free_field_su2(theta):
    L = (4, 6, 4, 8)
    V, kappa = synth.vol(L), 0.124
    U = np.tile(np.eye(2, dtype=complex), (V, 4, 1, 1))
    assert np.abs(oracle.sun_clover_blocks(NC, L, U, kappa, 1.7) - np.eye(4)).max() == 0.0
    rng = np.random.default_rng(3)
    n = np.arange(V)
    xs = [n % L[0], (n // L[0]) % L[1], (n // (L[0] * L[1])) % L[2], n // (L[0] * L[1] * L[2])]
    for mom in [(0, 0, 0, 0), (1, 0, 0, 0), (0, 2, 0, 0), (0, 0, 1, 0), (0, 0, 0, 3), (1, 5, 2, 7)]:
        p = [2 * math.pi * mom[mu] / L[mu] for mu in range(4)]
        pt = [p[mu] + theta[mu] / L[mu] for mu in range(4)]
        u = rng.standard_normal(8) + 1j * rng.standard_normal(8)
        phase = np.exp(1j * sum(p[mu] * xs[mu] for mu in range(4)))
        psi = (phase[:, None] * u[None, :]).reshape(V, 4, 2)
        scal = 1 - 2 * kappa * sum(math.cos(t) for t in pt)
        gs = sum(math.sin(pt[mu]) * GAMMA[mu] for mu in range(4))
        Dm = np.kron(scal * np.eye(4) + 2j * kappa * gs, np.eye(2))
        npsi = np.linalg.norm(psi)
        want = (phase[:, None] * (Dm @ u)[None, :]).reshape(V, 4, 2)
        assert np.linalg.norm(oracle.sun_dw(NC, L, U, psi, kappa, theta=theta) - want) / npsi < 1e-14
        wantd = (phase[:, None] * (Dm.conj().T @ u)[None, :]).reshape(V, 4, 2)
        assert np.linalg.norm(oracle.sun_dw(NC, L, U, psi, kappa, theta=theta, dagger=True) - wantd) / npsi < 1e-14


@pytest.mark.parametrize("bc", [oracle.BC_PERIODIC, oracle.BC_OPEN])
def test_P2_P3_hermiticity_and_covariance_su2(bc):
    L = (4, 4, 2, 6)
    V, kappa, csw, theta = synth.vol(L), 0.13, 1.8, (0.5, 0.5, 0.5, 0.3)
    U = synth.su2_matrices(synth.haar_su2_cd(L, 921))
    psi, chi = synth.gaussian_spinor_nc(L, 922, 2), synth.gaussian_spinor_nc(L, 923, 2)
    x4 = np.arange(V) // (L[0] * L[1] * L[2])
    inside = np.ones(V, dtype=bool) if bc == oracle.BC_PERIODIC else (x4 != 0) & (x4 != L[3] - 1)
    psi[~inside] = 0
    chi[~inside] = 0
    A = oracle.sun_clover_blocks(NC, L, U, kappa, csw, bc=bc)
    assert np.abs(A - dg(A)).max() < 1e-15                                    # Hermitian blocks
    lhs = np.vdot(chi, oracle.sun_dw(NC, L, U, psi, kappa, A, bc=bc, theta=theta))
    rhs = np.vdot(oracle.sun_dw(NC, L, U, chi, kappa, A, bc=bc, theta=theta, dagger=True), psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-14                                   # P2
    out = oracle.sun_dw(NC, L, U, psi, kappa, A, bc=bc, theta=theta)
    assert np.all(out[~inside] == 0)
    # P3: U'_mu(x) = g(x) U_mu(x) g(x+mu)^+, psi' = g psi  =>  D[U'] psi' = g D[U] psi
    g = synth.su2_matrices(synth.haar_su2_cd(L, 924)[:, 0])
    gl = g.reshape(L[3], L[2], L[1], L[0], 2, 2)
    Ug = np.empty_like(U)
    for mu in range(4):
        Ug[:, mu] = (gl @ U[:, mu].reshape(gl.shape) @ dg(sh(gl, mu, 1))).reshape(V, 2, 2)
    psig = np.einsum("nab,nsb->nsa", g, psi)
    Ag = oracle.sun_clover_blocks(NC, L, Ug, kappa, csw, bc=bc)
    outg = oracle.sun_dw(NC, L, Ug, psig, kappa, Ag, bc=bc, theta=theta)
    assert rel(outg, np.einsum("nab,nsb->nsa", g, out)) < 1e-14


@pytest.mark.parametrize("csw", [0.0, 1.3])
def test_P4_dense_matrix_2to4_su2(csw):
    L, kappa, theta = (2, 2, 2, 2), 0.125, (0.0, 0.0, 0.0, math.pi)
    U = synth.su2_matrices(synth.haar_su2_cd(L, 931))
    A8 = clover_numpy(L, U, kappa, csw, 2)
    M = dense_dirac(L, U, kappa, theta, 2, A8)
    A = oracle.sun_clover_blocks(NC, L, U, kappa, csw)
    # the chiral blocks are the diagonal blocks of the dense numpy matrix, the off-diagonal ones vanish
    assert np.abs(A[:, 0] - A8[:, :4, :4]).max() < 1e-14 and np.abs(A[:, 1] - A8[:, 4:, 4:]).max() < 1e-14
    assert np.abs(A8[:, :4, 4:]).max() < 1e-15
    psi = synth.gaussian_spinor_nc(L, 932, 2)
    assert rel(oracle.sun_dw(NC, L, U, psi, kappa, A, theta=theta).reshape(-1), M @ psi.reshape(-1)) < 1e-14
    assert rel(oracle.sun_dw(NC, L, U, psi, kappa, A, theta=theta, dagger=True).reshape(-1), M.conj().T @ psi.reshape(-1)) < 1e-14
    G5 = np.kron(np.eye(16), np.kron(GAMMA5, np.eye(2)))
    assert np.abs(G5 @ M @ G5 - M.conj().T).max() < 1e-14
    b = synth.gaussian_spinor_nc(L, 933, 2)
    want = np.linalg.solve(M, b.reshape(-1))
    x, it, rn, rt = oracle.sun_cg(NC, L, U, b, kappa, A, theta=theta, tol=1e-13, maxiter=2000)
    assert it > 0 and rel(x.reshape(-1), want) < 10 * np.linalg.cond(M) * 1e-13


def test_fhat_vs_numpy_rolls_su2():
    L = (4, 6, 4, 4)
    U = synth.su2_matrices(synth.haar_su2_cd(L, 941))
    for mu, nu in itertools.permutations(range(4), 2):
        F = fhat_numpy(L, U, mu, nu, 2)
        for x in [(0, 0, 0, 0), (3, 5, 3, 3), (1, 2, 3, 0)]:
            assert np.abs(oracle.sun_fhat_site(NC, L, U, x, mu, nu) - F[synth.site_index(L, x)]).max() < 1e-14


@pytest.mark.parametrize("plane", [(0, 1), (0, 2), (1, 2), (0, 3), (1, 3), (2, 3)])
def test_P5_constant_flux_su2(plane):
    """As pin P5 of the SU(3) oracle with the traceless generator t = diag(1, -1): every mu-nu plaquette is exp(i phi t),
    F^_{mu nu} = i sin(phi t), A = 1 - kappa csw sigma_{mu nu} (x) sin(phi t)."""
    mu, nu = plane
    L = (4, 6, 4, 8)
    V = synth.vol(L)
    phi = 2 * math.pi / (L[mu] * L[nu])
    t = np.array([1.0, -1.0])
    n = np.arange(V)
    xs = [n % L[0], (n // L[0]) % L[1], (n // (L[0] * L[1])) % L[2], n // (L[0] * L[1] * L[2])]
    U = np.tile(np.eye(2, dtype=complex), (V, 4, 1, 1))
    for a in range(2):
        U[:, mu, a, a] = np.exp(-1j * phi * xs[nu] * t[a])
        U[:, nu, a, a] = np.where(xs[nu] == L[nu] - 1, np.exp(1j * phi * L[nu] * xs[mu] * t[a]), 1.0)
    kappa, csw = 0.137, 1.9
    for x in [(0, 0, 0, 0), (3, 5, 3, 7)]:
        assert np.abs(oracle.sun_fhat_site(NC, L, U, x, mu, nu) - np.diag(1j * np.sin(phi * t))).max() < 1e-15
    s = np.diag(np.sin(phi * t))
    A = oracle.sun_clover_blocks(NC, L, U, kappa, csw)
    if nu == 3:
        wp, wm = np.eye(4) - kappa * csw * np.kron(PAULI[mu], s), np.eye(4) + kappa * csw * np.kron(PAULI[mu], s)
    else:
        k = {(0, 1): 2, (1, 2): 0, (0, 2): 1}[plane]
        sgn = -1.0 if plane == (0, 2) else 1.0
        wp = wm = np.eye(4) + sgn * kappa * csw * np.kron(PAULI[k], s)
    assert np.abs(A[:, 0] - wp[None]).max() < 1e-15 and np.abs(A[:, 1] - wm[None]).max() < 1e-15
