"""-m gpu parity of the time-direction domain decomposition: the lattice is cut into
P time slabs, each with its own LQCD_BC_SLAB geometry, fields, clover term (built from the slab plus a one-slice
gauge halo) and face buffers, exactly as P ranks would hold them; the slabs run one after the other on the one GPU
(no kernel waits on another), the faces are moved between them by plain copies in the pattern slab.FaceExchange uses
between ranks (tests/test_slab_dist.py checks that pattern over gloo).  The assembled result must be the oracle's D
(D^+) on the whole lattice, to north_star's per-site tolerances."""
import numpy as np
import pytest
import torch

import oracle
from paper_2503_16994_b200 import binding as B
from paper_2503_16994_b200 import slab, synth

from gpu_util import f32_storage_err, round_f32, site_rel_err, to_dev

pytestmark = pytest.mark.gpu

TOL = {B.F64: 1e-12, B.F32: 2e-6}


@pytest.fixture
def mode(request):
    B.set_option("dw_mode", request.param)
    yield request.param
    B.set_option("dw_mode", "pipe")


class Rank:
    """What one rank of the decomposition holds."""

    def __init__(self, L, P, r, theta, U, kappa, csw, prec, recon, bc=B.BC_PERIODIC, ct=1.0, phiT=None):
        self.T = slab.slab_extent(L[3], P)
        self.ns = L[0] * L[1] * L[2]
        self.lo, self.hi = r * self.T * self.ns, (r + 1) * self.T * self.ns   # canonical site range (time slowest)
        self.g = slab.slab_geom_create(L, P, theta, rank=r, bc=bc, phiT=phiT)
        self.nbr = slab.ring_neighbours(P, r, bc == B.BC_PERIODIC)
        Uc = to_dev(U[self.lo:self.hi])
        self.U64 = B.alloc_field(self.g, B.FIELD_GAUGE, B.F64, recon)
        B.gauge_import(self.g, Uc, self.U64, B.F64, recon)
        self.U = self.U64
        if prec == B.F32:
            self.U = B.alloc_field(self.g, B.FIELD_GAUGE, prec, recon)
            B.gauge_import(self.g, Uc, self.U, prec, recon)
        V = U.shape[0]
        below = np.arange(self.lo - self.ns, self.lo) % V
        above = np.arange(self.hi, self.hi + self.ns) % V
        self.A = B.alloc_field(self.g, B.FIELD_CLOVER, prec)
        B.clover_build_slab(self.g, kappa, csw, self.U64, to_dev(U[below]) if self.nbr[0] is not None else None,
                            to_dev(U[above]) if self.nbr[1] is not None else None, self.A, None, recon, prec, ct=ct)
        self.send_lo, self.send_hi, self.recv_lo, self.recv_hi = (B.alloc_field(self.g, B.FIELD_FACE, prec) for _ in range(4))
        self.src = B.alloc_field(self.g, B.FIELD_SPINOR, prec)
        self.dst = B.alloc_field(self.g, B.FIELD_SPINOR, prec)


def slab_dw(ranks, kappa, psi, prec, recon, dagger, clover=True, mu=0.0):
    P = len(ranks)
    for R in ranks:
        B.spinor_import(R.g, to_dev(psi[R.lo:R.hi]), R.src, prec)
        R.dst.fill_(0x7F)
        B.dw_slab_pack(R.g, kappa, R.U, R.src, R.send_lo, R.send_hi, dagger, prec, recon)
    for R in ranks:   # the ring: send_lo -> below's recv_hi, send_hi -> above's recv_lo (nothing across an open boundary)
        if R.nbr[0] is not None:
            ranks[R.nbr[0]].recv_hi.copy_(R.send_lo)
        if R.nbr[1] is not None:
            ranks[R.nbr[1]].recv_lo.copy_(R.send_hi)
    out = np.empty_like(psi)
    for R in ranks:
        fn = B.dwdag_apply if dagger else B.dw_apply
        fn(R.g, kappa, R.U, R.A if clover else None, R.src, R.dst, prec, recon, mu=mu)
        B.dw_slab_faces(R.g, kappa, R.U, R.recv_lo, R.recv_hi, R.dst, dagger, prec, recon)
        o = torch.empty((R.hi - R.lo, 4, 3), dtype=torch.complex128, device="cuda")
        B.spinor_export(R.g, R.dst, o, prec)
        torch.cuda.synchronize()
        out[R.lo:R.hi] = o.cpu().numpy()
    return out


@pytest.mark.parametrize("mode", ["pipe", "stream", "split", "direct"], indirect=True)
@pytest.mark.parametrize("L,P,theta", [
    ((8, 4, 4, 8), 2, (0.3, -0.2, 0.1, np.pi)),     # two slabs of 4^4 tiles, antiperiodic in time
    ((4, 8, 4, 12), 3, None),                        # three slabs
    ((6, 4, 10, 8), 1, (0.5, 0.5, 0.5, 1.0)),        # one slab = the periodic lattice through its own faces; no 4^4 tiles
    ((4, 4, 4, 16), 2, (0, 0, 0, np.pi)),            # slabs of two tiles in time
])
@pytest.mark.parametrize("prec,recon", [(B.F64, B.RECON_18), (B.F64, B.RECON_12), (B.F32, B.RECON_18)])
def test_slab_dw_equals_whole_lattice(mode, L, P, theta, prec, recon):
    kappa, csw = 0.137, 1.9
    U = synth.smooth_gauge(L, 101)
    psi = synth.gaussian_spinor(L, 102)
    A = oracle.clover_blocks(L, U, kappa, csw)
    Uo, psio, Ao = (round_f32(U), round_f32(psi), round_f32(A)) if prec == B.F32 else (U, psi, A)
    ranks = [Rank(L, P, r, theta, U, kappa, csw, prec, recon) for r in range(P)]
    # the clover term of each slab is the whole lattice's (fp64 build, rounded once)
    for R in ranks:
        got = torch.empty((R.hi - R.lo, 2, 6, 6), dtype=torch.complex128, device="cuda")
        B.clover_export(R.g, R.A, got, prec)
        torch.cuda.synchronize()
        if prec == B.F64:
            assert np.max(np.abs(got.cpu().numpy() - A[R.lo:R.hi])) <= 2e-14
        else:   # fp32 storage: the fp64 build rounded once (same rule as tests/test_gpu_dw.py::test_clover_build)
            assert f32_storage_err(got.cpu().numpy(), A[R.lo:R.hi]) <= 0
    for dagger in (False, True):
        ref = oracle.dw(L, Uo, psio, kappa, Ao, theta=theta, dagger=dagger)
        assert site_rel_err(slab_dw(ranks, kappa, psi, prec, recon, dagger), ref) <= TOL[prec]
    ref = oracle.dw(L, Uo, psio, kappa, None, theta=theta)
    assert site_rel_err(slab_dw(ranks, kappa, psi, prec, recon, False, clover=False), ref) <= TOL[prec]
    ref = oracle.dw(L, Uo, psio, kappa, Ao, theta=theta, dagger=True, mu=0.3)
    assert site_rel_err(slab_dw(ranks, kappa, psi, prec, recon, True, mu=0.3), ref) <= TOL[prec]
    for R in ranks:
        B.geom_destroy(R.g)


@pytest.mark.parametrize("mode", ["pipe", "stream"], indirect=True)
@pytest.mark.parametrize("L,P", [((8, 4, 4, 8), 2), ((4, 8, 4, 12), 3), ((4, 4, 4, 8), 1), ((6, 4, 4, 8), 2)])
@pytest.mark.parametrize("prec", [B.F64, B.F32])
def test_slab_dw_open_boundaries(mode, L, P, prec):
    """A lattice with open time boundaries cut into slabs: the first / last rank carry the frozen slice (D7) and the
    c~_t term next to it, nothing is exchanged across the open boundary; one slab with both edges open is the open
    lattice itself.  Against the oracle's open-BC operator on the whole lattice."""
    kappa, csw, ct, theta, recon = 0.1365, 1.9, 1.2, (0.5, 0.5, 0.5, 0.0), B.RECON_18
    U = synth.smooth_gauge(L, 121)
    psi = synth.gaussian_spinor(L, 122)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=B.BC_OPEN, ct=ct)
    Uo, psio, Ao = (round_f32(U), round_f32(psi), round_f32(A)) if prec == B.F32 else (U, psi, A)
    ranks = [Rank(L, P, r, theta, U, kappa, csw, prec, recon, bc=B.BC_OPEN, ct=ct) for r in range(P)]
    t = np.arange(psi.shape[0]) // (L[0] * L[1] * L[2])
    mask = (t >= 1) & (t <= L[3] - 2)
    for R in ranks:
        got = torch.empty((R.hi - R.lo, 2, 6, 6), dtype=torch.complex128, device="cuda")
        B.clover_export(R.g, R.A, got, prec)
        torch.cuda.synchronize()
        if prec == B.F64:
            assert np.max(np.abs(got.cpu().numpy() - A[R.lo:R.hi])) <= 2e-14
        else:   # fp32 storage: the fp64 build rounded once (same rule as tests/test_gpu_dw.py::test_clover_build)
            assert f32_storage_err(got.cpu().numpy(), A[R.lo:R.hi]) <= 0
    for dagger in (False, True):
        ref = oracle.dw(L, Uo, psio, kappa, Ao, bc=B.BC_OPEN, theta=theta, dagger=dagger)
        got = slab_dw(ranks, kappa, psi, prec, recon, dagger)
        assert site_rel_err(got, ref, mask) <= TOL[prec]
        assert np.all(got[~mask] == 0)
    for R in ranks:
        B.geom_destroy(R.g)


@pytest.mark.parametrize("mode", ["pipe", "stream"], indirect=True)
@pytest.mark.parametrize("L,P", [((4, 4, 4, 8), 2), ((4, 8, 4, 12), 3), ((4, 4, 4, 8), 1)])
@pytest.mark.parametrize("prec", [B.F64, B.F32])
def test_slab_dw_sf_boundaries(mode, L, P, prec):
    """Schroedinger-functional lattice in slabs: frozen slice x4 = 0 on the first rank, boundary field W' (phiT) above
    the last rank's top slice in the clover term, c~_t on both ends.  Against the oracle's SF operator."""
    kappa, csw, ct, theta, recon, bc = 0.1355, 1.8, 1.1, (0.5, 0.5, 0.5, 0.0), B.RECON_18, B.BC_SF_ORBI
    U = synth.apply_sf_boundary(L, synth.smooth_gauge(L, 131))
    psi = synth.gaussian_spinor(L, 132)
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc, phiT=synth.SF_PHIT, ct=ct)
    Uo, psio, Ao = (round_f32(U), round_f32(psi), round_f32(A)) if prec == B.F32 else (U, psi, A)
    ranks = [Rank(L, P, r, theta, U, kappa, csw, prec, recon, bc=bc, ct=ct, phiT=synth.SF_PHIT) for r in range(P)]
    t = np.arange(psi.shape[0]) // (L[0] * L[1] * L[2])
    mask = t >= 1
    for R in ranks:
        got = torch.empty((R.hi - R.lo, 2, 6, 6), dtype=torch.complex128, device="cuda")
        B.clover_export(R.g, R.A, got, prec)
        torch.cuda.synchronize()
        if prec == B.F64:
            assert np.max(np.abs(got.cpu().numpy() - A[R.lo:R.hi])) <= 2e-14
        else:   # fp32 storage: the fp64 build rounded once (same rule as tests/test_gpu_dw.py::test_clover_build)
            assert f32_storage_err(got.cpu().numpy(), A[R.lo:R.hi]) <= 0
    for dagger in (False, True):
        ref = oracle.dw(L, Uo, psio, kappa, Ao, bc=bc, theta=theta, dagger=dagger)
        got = slab_dw(ranks, kappa, psi, prec, recon, dagger)
        assert site_rel_err(got, ref, mask) <= TOL[prec]
        assert np.all(got[~mask] == 0)
    for R in ranks:
        B.geom_destroy(R.g)


def test_slab_without_faces_differs_and_unsupported_calls_fail():
    """The slab stencil alone must NOT be the periodic operator (the faces are really needed), and the calls that
    would ignore the faces are refused."""
    L, kappa = (4, 4, 4, 8), 0.13
    U = synth.smooth_gauge(L, 103)
    psi = synth.gaussian_spinor(L, 104)
    R = Rank(L, 1, 0, None, U, kappa, 1.0, B.F64, B.RECON_18)
    B.spinor_import(R.g, to_dev(psi), R.src, B.F64)
    B.dw_apply(R.g, kappa, R.U, R.A, R.src, R.dst)
    o = torch.empty((psi.shape[0], 4, 3), dtype=torch.complex128, device="cuda")
    B.spinor_export(R.g, R.dst, o, B.F64)
    torch.cuda.synchronize()
    ref = oracle.dw(L, U, psi, kappa, oracle.clover_blocks(L, U, kappa, 1.0))
    err = np.linalg.norm((o.cpu().numpy() - ref).reshape(psi.shape[0], -1), axis=1)
    t = np.arange(psi.shape[0]) // (4 * 4 * 4)
    assert np.all(err[(t > 0) & (t < 7)] < 1e-12) and np.all(err[(t == 0) | (t == 7)] > 1e-3)
    ws = B.alloc_field(R.g, B.FIELD_WORKSPACE)
    for call in (lambda: B.cg_solve(R.g, kappa, R.U, R.A, R.src, R.dst, ws),
                 lambda: B.clover_build(R.g, kappa, 1.0, R.U, R.A),
                 lambda: B.dw_eo_apply(R.g, kappa, R.U, R.A, R.A, R.src, R.dst, ws)):
        with pytest.raises(B.LqcdError) as e:
            call()
        assert e.value.status == B.EUNSUPPORTED
    per = B.geom_create(L)
    with pytest.raises(B.LqcdError):   # the face kernels want a slab geometry
        B.dw_slab_pack(per, kappa, R.U, R.src, R.send_lo, R.send_hi)
    B.geom_destroy(per)
    B.geom_destroy(R.g)


def test_slab_dirac_driver_single_rank():
    """slab.SlabDirac (pack -> exchange on a side stream || stencil -> faces) with one rank: the periodic lattice."""
    L, kappa, csw, theta = (8, 8, 4, 8), 0.135, 1.7, (0, 0, 0, np.pi)
    U = synth.smooth_gauge(L, 105)
    psi = synth.gaussian_spinor(L, 106)
    A = oracle.clover_blocks(L, U, kappa, csw)
    R = Rank(L, 1, 0, theta, U, kappa, csw, B.F64, B.RECON_18)
    D = slab.SlabDirac(R.g, kappa, R.U, R.A)
    B.spinor_import(R.g, to_dev(psi), R.src, B.F64)
    for dagger in (False, True):
        D.apply(R.src, R.dst, dagger)
        o = torch.empty((psi.shape[0], 4, 3), dtype=torch.complex128, device="cuda")
        B.spinor_export(R.g, R.dst, o, B.F64)
        torch.cuda.synchronize()
        assert site_rel_err(o.cpu().numpy(), oracle.dw(L, U, psi, kappa, A, theta=theta, dagger=dagger)) <= 1e-12
    B.geom_destroy(R.g)


class ThreadRing:
    """Test stand-in for slab.FaceExchange between P 'ranks' that are threads of this process sharing the one GPU and
    its default stream: host barriers order the enqueues, stream order and events order the work, so no kernel ever
    spins on another.
    Same interface and the same who-gets-what as FaceExchange."""

    def __init__(self, P, periodic=True):
        import threading
        self.P = P
        self.periodic = periodic
        self.barrier = threading.Barrier(P, timeout=120)
        self.faces = [None] * P
        self.scal = [None] * P
        self.tmp = [None] * P

    def view(self, r):
        ring = self

        class View:
            world, rank = ring.P, r
            below, above = slab.ring_neighbours(ring.P, r, ring.periodic)

            def start(self, send_lo, send_hi, recv_lo, recv_hi):
                ring.faces[r] = (send_lo, send_hi)
                main, cur = torch.cuda.default_stream(), torch.cuda.current_stream()
                ring.barrier.wait()                      # every rank's pack kernel is enqueued on the main stream
                cur.wait_stream(main)                    # (the communicator calls this on its own side stream)
                if self.above is not None:
                    recv_hi.copy_(ring.faces[self.above][0])
                if self.below is not None:
                    recv_lo.copy_(ring.faces[self.below][1])
                main.wait_stream(cur)                    # nobody's next pack may overtake these copies
                ring.barrier.wait()                      # every copy is enqueued before anyone packs again
                return []

            @staticmethod
            def finish(reqs):
                pass

            def __call__(self, *a):
                self.finish(self.start(*a))

            def allreduce_sum(self, t):
                ring.scal[r] = t
                ring.barrier.wait()
                acc = ring.scal[0].clone()
                for k in range(1, ring.P):               # same order on every rank: identical bits everywhere
                    acc += ring.scal[k]
                ring.tmp[r] = acc
                ring.barrier.wait()
                t.copy_(acc)
                ring.barrier.wait()
                return t

        return View()


@pytest.mark.timeout(600)
@pytest.mark.parametrize("mixed", [False, True])
@pytest.mark.parametrize("L,P,theta,bc", [((8, 4, 4, 8), 2, (0, 0, 0, np.pi), B.BC_PERIODIC), ((4, 4, 4, 12), 3, None, B.BC_PERIODIC),
                                          ((4, 4, 4, 8), 1, None, B.BC_PERIODIC), ((4, 4, 4, 12), 3, (0.5, 0.5, 0.5, 0), B.BC_OPEN)])
def test_cg_over_slabs(L, P, theta, bc, mixed):
    """lqcd_cg_solve_slab on P slabs (P threads, one per 'rank', all calling the library together as P processes
    would) against the oracle's CG on the whole lattice: solution, iteration count, residuals."""
    import threading

    kappa, csw = 0.125, 1.0
    U = synth.smooth_gauge(L, 111)
    b = synth.gaussian_spinor(L, 112)
    if bc == B.BC_OPEN:   # the solve lives on the interior (D7): a source without support on the frozen slices
        tt = np.arange(b.shape[0]) // (L[0] * L[1] * L[2])
        b[(tt == 0) | (tt == L[3] - 1)] = 0
    A = oracle.clover_blocks(L, U, kappa, csw, bc=bc)
    ranks = [Rank(L, P, r, theta, U, kappa, csw, B.F64, B.RECON_18, bc=bc) for r in range(P)]
    ring = ThreadRing(P, periodic=(bc == B.BC_PERIODIC))
    out = np.empty_like(b)
    infos, errors = [None] * P, []

    def run(r):
        try:
            R = ranks[r]
            B.spinor_import(R.g, to_dev(b[R.lo:R.hi]), R.src, B.F64)
            comm = slab.SlabCommunicator(R.g, ring.view(r))
            ws = B.alloc_field(R.g, B.FIELD_WORKSPACE)
            kw = {}
            if mixed:   # fp32 copies of this rank's slab for the inner solve
                U32 = B.alloc_field(R.g, B.FIELD_GAUGE, B.F32)
                A32 = B.alloc_field(R.g, B.FIELD_CLOVER, B.F32)
                B.field_to_f32(R.g, B.FIELD_GAUGE, B.RECON_18, R.U, U32)
                B.field_to_f32(R.g, B.FIELD_CLOVER, B.RECON_18, R.A, A32)
                kw = dict(U32=U32, clover32=A32, mixed=True)
            infos[r] = slab.cg_solve_slab(R.g, kappa, R.U, R.A, R.src, R.dst, ws, comm, tol=1e-10, maxiter=4000, **kw)
            o = torch.empty((R.hi - R.lo, 4, 3), dtype=torch.complex128, device="cuda")
            B.spinor_export(R.g, R.dst, o, B.F64)
            torch.cuda.synchronize()
            out[R.lo:R.hi] = o.cpu().numpy()
        except Exception as e:   # noqa: BLE001
            errors.append(e)
            ring.barrier.abort()

    threads = [threading.Thread(target=run, args=(r,)) for r in range(P)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(500)
    assert not errors, errors
    xo, it_o, _, _ = oracle.cg(L, U, b, kappa, A, bc=bc, theta=theta, tol=1e-10)
    assert np.linalg.norm(out - xo) / np.linalg.norm(xo) <= 1e-8
    for info in infos:
        assert info["status"] == B.OK and (mixed or abs(info["iters"] - it_o) <= 2)
        assert info["rel_resid_normal"] <= 2e-10 and info["rel_resid_true"] <= 1e-8
        assert (info["outer"] >= 2) == mixed
        assert info["iters"] == infos[0]["iters"]          # lockstep
    tt = np.arange(b.shape[0]) // (L[0] * L[1] * L[2])
    live = (tt >= 1) & (tt <= L[3] - 2) if bc == B.BC_OPEN else np.ones(b.shape[0], dtype=bool)
    r = (oracle.dw(L, U, out, kappa, A, bc=bc, theta=theta) - b)[live]
    assert np.linalg.norm(r) / np.linalg.norm(b[live]) <= 1e-8
    for R in ranks:
        B.geom_destroy(R.g)


@pytest.mark.timeout(600)
def test_propagator_and_correlator_over_slabs():
    """The paper's end product on a decomposed lattice: 12 point-source columns by
    lqcd_cg_solve_slab on two slabs (threads as ranks), then C(x4) assembled from the slabs' own time slices, against
    the oracle's CG + correlator on the whole lattice.  The source sits in the second slab."""
    import threading

    L, P, kappa, csw, theta, y = (4, 4, 4, 8), 2, 0.125, 1.0, (0, 0, 0, np.pi), (1, 2, 3, 5)
    U = synth.smooth_gauge(L, 141)
    A = oracle.clover_blocks(L, U, kappa, csw)
    ranks = [Rank(L, P, r, theta, U, kappa, csw, B.F64, B.RECON_18) for r in range(P)]
    ring = ThreadRing(P)
    V = synth.vol(L)
    got_cols = np.empty((12, V, 4, 3), dtype=np.complex128)
    corr, errors = [None] * P, []

    def run(r):
        try:
            R = ranks[r]
            comm = slab.SlabCommunicator(R.g, ring.view(r))
            ws = B.alloc_field(R.g, B.FIELD_WORKSPACE)
            fb = B.field_bytes(R.g, B.FIELD_SPINOR)
            cols = torch.empty(12 * fb, dtype=torch.uint8, device="cuda")
            infos = slab.propagator_slab(R.g, L, P, r, kappa, R.U, R.A, y, cols, ws, comm, tol=1e-12, maxiter=4000)
            assert all(i["status"] == B.OK for i in infos)
            corr[r] = slab.correlator_ps_slab(R.g, L, P, r, cols, 12, ws, comm)
            o = torch.empty((R.hi - R.lo, 4, 3), dtype=torch.complex128, device="cuda")
            for c in range(12):
                B.spinor_export(R.g, cols[c * fb:(c + 1) * fb], o)
                torch.cuda.synchronize()
                got_cols[c, R.lo:R.hi] = o.cpu().numpy()
        except Exception as e:   # noqa: BLE001
            errors.append(e)
            ring.barrier.abort()

    threads = [threading.Thread(target=run, args=(r,)) for r in range(P)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(500)
    assert not errors, errors
    ref_cols = []
    for c in range(12):
        b = synth.point_source(L, y, c // 3, c % 3)
        ref_cols.append(oracle.cg(L, U, b, kappa, A, theta=theta, tol=1e-12)[0])
    ref_cols = np.array(ref_cols)
    assert np.linalg.norm(got_cols - ref_cols) / np.linalg.norm(ref_cols) <= 1e-8
    ref = oracle.correlator_ps(L, ref_cols)
    for r in range(P):
        assert np.max(np.abs(np.array(corr[r]) - ref) / ref) <= 1e-8
    assert int(np.argmax(ref)) == y[3]
    for R in ranks:
        B.geom_destroy(R.g)
