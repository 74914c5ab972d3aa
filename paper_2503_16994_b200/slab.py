"""Time-direction domain decomposition over torch.distributed.

One process per GPU; rank r owns the time slab [r*T, (r+1)*T) of the lattice (T = L4 / world).  The lattice may be
periodic in time (antiperiodic = theta4 = pi), open, or Schroedinger-functional: on an open / SF lattice the first
and last rank carry the physical boundary (lqcd_geom_desc.slab_edges) and the chain of ranks is not closed.
Every step of the arithmetic runs in the library's kernels (lqcd_dw_slab_pack, lqcd_dw_apply / lqcd_dwdag_apply on the
LQCD_BC_SLAB geometry, lqcd_dw_slab_faces, lqcd_clover_build_slab, lqcd_cg_solve_slab); this module only decides who owns what and moves the two half-spinor
faces per application between ring neighbours (NCCL send/recv over NVLink on GPUs; gloo in the CPU tests of the
exchange logic).  The exchange runs on its own stream and overlaps the interior stencil kernel.

Traffic per application and rank: 2 faces x 6 complex x L1 L2 L3 sites sent and received
(48^3, fp64: 2 x 10.6 MB against 16.3 GB / world of HBM traffic for the slab's stencil).
"""
from . import binding as B


def slab_extent(L4, world):
    """Time extent of one slab; every rank owns the same number of slices (even, >= 4: R13 and the stencil's needs)."""
    L4, world = int(L4), int(world)
    if world < 1 or L4 % world != 0:
        raise ValueError("L4=%d is not divisible by the number of ranks %d" % (L4, world))
    T = L4 // world
    if T < 4 or T % 2 != 0:
        raise ValueError("slab extent %d must be even and >= 4" % T)
    return T


def slab_origin(L4, world, rank):
    return int(rank) * slab_extent(L4, world)


def slab_theta(theta, L4, world):
    """The slab geometry's angles: the per-link phase exp(i theta4 / L4) of the whole lattice, expressed over T links."""
    th = [0.0, 0.0, 0.0, 0.0] if theta is None else [float(v) for v in theta]
    th[3] = th[3] * slab_extent(L4, world) / int(L4)
    return th


def ring_neighbours(world, rank, periodic=True):
    """(rank below, rank above) along time; None across an open boundary of the lattice."""
    below, above = (rank - 1) % world, (rank + 1) % world
    if not periodic:
        below = None if rank == 0 else below
        above = None if rank == world - 1 else above
    return below, above


def slab_edges(world, rank, bc=B.BC_PERIODIC):
    """lqcd_geom_desc.slab_edges of this rank: which of its faces are open boundaries of the lattice."""
    if bc == B.BC_PERIODIC:
        return 0
    if bc not in (B.BC_OPEN, B.BC_SF_ORBI, B.BC_SF_AFWB):
        raise ValueError("bad time boundary condition %r" % (bc,))
    top = B.SLAB_OPEN_HI if bc == B.BC_OPEN else B.SLAB_SF_HI   # SF: no frozen slice at the top, boundary field W'
    return (B.SLAB_OPEN_LO if rank == 0 else 0) | (top if rank == world - 1 else 0)


def slab_geom_create(L, world, theta=None, device=0, rank=0, bc=B.BC_PERIODIC, phiT=None):
    """Geometry handle of one rank's slab of the lattice L (bc: periodic in time -- antiperiodic = theta4 = pi --,
    open: the first and last rank get a frozen outer slice, or SF: frozen slice x4 = 0 on the first rank, boundary
    field W' = exp(i phiT / L_k) above the last rank's top slice)."""
    T = slab_extent(L[3], world)
    return B.geom_create((L[0], L[1], L[2], T), B.BC_SLAB, slab_theta(theta, L[3], world), phiT=phiT, device=device,
                         slab_edges=slab_edges(world, rank, bc))


class FaceExchange:
    """send_lo -> the rank below (lands in its recv_hi), send_hi -> the rank above (lands in its recv_lo).

    world == 1, periodic: the slab is its own neighbour on both sides (the periodic lattice).  periodic=False (open
    lattice): the first rank has nobody below, the last nobody above; those faces are left alone.  Tensors of any
    device / dtype; the two directions carry different tags so that world == 2 (both neighbours are the same peer)
    cannot mix them.
    """
    TAG_DOWN, TAG_UP = 11, 12

    def __init__(self, group=None, periodic=True):
        import torch.distributed as dist

        self.dist = dist
        self.group = group
        self.periodic = periodic
        active = dist.is_available() and dist.is_initialized()
        self.world = dist.get_world_size(group) if active else 1
        self.rank = dist.get_rank(group) if active else 0
        self.below, self.above = ring_neighbours(self.world, self.rank, periodic)

    def start(self, send_lo, send_hi, recv_lo, recv_hi):
        if self.world == 1:
            if self.periodic:
                recv_hi.copy_(send_lo)
                recv_lo.copy_(send_hi)
            return []
        d = self.dist
        ops = []
        if self.below is not None:
            ops.append(d.P2POp(d.isend, send_lo, self.below, self.group, self.TAG_DOWN))
        if self.above is not None:
            ops.append(d.P2POp(d.isend, send_hi, self.above, self.group, self.TAG_UP))
            ops.append(d.P2POp(d.irecv, recv_hi, self.above, self.group, self.TAG_DOWN))
        if self.below is not None:
            ops.append(d.P2POp(d.irecv, recv_lo, self.below, self.group, self.TAG_UP))
        return d.batch_isend_irecv(ops) if ops else []

    @staticmethod
    def finish(reqs):
        for r in reqs:
            r.wait()

    def __call__(self, send_lo, send_hi, recv_lo, recv_hi):
        self.finish(self.start(send_lo, send_hi, recv_lo, recv_hi))

    def allreduce_sum(self, t):
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)
        return t


class SlabDirac:
    """D and D^+ on this rank's slab: pack -> (exchange || interior stencil) -> faces."""

    def __init__(self, g, kappa, U, clover, prec=B.F64, recon=B.RECON_18, mu=0.0, exchange=None):
        import torch

        self.torch = torch
        self.g, self.kappa, self.U, self.A, self.prec, self.recon, self.mu = g, kappa, U, clover, prec, recon, mu
        self.xch = exchange if exchange is not None else FaceExchange()
        self.send_lo, self.send_hi, self.recv_lo, self.recv_hi = (B.alloc_field(g, B.FIELD_FACE, prec) for _ in range(4))
        self.comm_stream = torch.cuda.Stream()

    def apply(self, psi_in, psi_out, dagger=False):
        torch = self.torch
        main = torch.cuda.current_stream()
        B.dw_slab_pack(self.g, self.kappa, self.U, psi_in, self.send_lo, self.send_hi, dagger, self.prec, self.recon)
        self.comm_stream.wait_stream(main)
        with torch.cuda.stream(self.comm_stream):
            reqs = self.xch.start(self.send_lo, self.send_hi, self.recv_lo, self.recv_hi)
            self.xch.finish(reqs)
        fn = B.dwdag_apply if dagger else B.dw_apply
        fn(self.g, self.kappa, self.U, self.A, psi_in, psi_out, self.prec, self.recon, mu=self.mu)
        main.wait_stream(self.comm_stream)
        B.dw_slab_faces(self.g, self.kappa, self.U, self.recv_lo, self.recv_hi, psi_out, dagger, self.prec, self.recon)


def gauge_halo_exchange(U_canon_slab, L, exchange=None):
    """The two time slices the clover builder needs from the ring neighbours (once per configuration).

    U_canon_slab: this rank's links, canonical layout [T * L1 L2 L3, 4, 3, 3] complex128 (time slowest).
    Returns (halo_lo, halo_hi): the slice below the slab's first and the slice above its last (None across an open
    boundary)."""
    import torch

    xch = exchange if exchange is not None else FaceExchange()
    ns = int(L[0]) * int(L[1]) * int(L[2])
    first = U_canon_slab[:ns].contiguous()
    last = U_canon_slab[-ns:].contiguous()
    halo_lo, halo_hi = torch.empty_like(last), torch.empty_like(first)
    # my first slice is the halo_hi of the rank below; my last slice the halo_lo of the rank above
    xch(first, last, halo_lo, halo_hi)
    # across an open boundary there is no neighbour (and lqcd_clover_build_slab wants no halo there)
    return (halo_lo if xch.below is not None else None), (halo_hi if xch.above is not None else None)


class SlabCommunicator:
    """One rank's lqcd_slab_comm: fp64 face buffers, the all-reduce payload and the three host callbacks that
    lqcd_cg_solve_slab calls.  Call the solver with stream=None (torch's current stream): the callbacks order their
    work against that stream.  The face exchange runs on a stream of its own and overlaps the interior stencil."""

    def __init__(self, g, exchange=None):
        import ctypes
        import sys
        import traceback

        import torch

        xch = exchange if exchange is not None else FaceExchange()
        self.exchange = xch
        self.send_lo, self.send_hi, self.recv_lo, self.recv_hi = (B.alloc_field(g, B.FIELD_FACE, B.F64) for _ in range(4))
        self.scalars = torch.zeros(4, dtype=torch.float64, device=self.send_lo.device)
        self.comm_stream = torch.cuda.Stream()

        def guarded(fn):
            def wrapper(*a):
                try:
                    fn(*a)
                    return 0
                except Exception:   # an exception must not unwind through the C frames
                    traceback.print_exc(file=sys.stderr)
                    return 1
            return wrapper

        def start(_ctx, nbytes):   # fp32 faces use the first half of the buffers
            self.comm_stream.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(self.comm_stream):
                xch.finish(xch.start(self.send_lo[:nbytes], self.send_hi[:nbytes], self.recv_lo[:nbytes], self.recv_hi[:nbytes]))

        def wait(_ctx):
            torch.cuda.current_stream().wait_stream(self.comm_stream)

        def allreduce(_ctx, n):
            xch.allreduce_sum(self.scalars[:n])

        # keep the CFUNCTYPE objects alive as long as the struct
        self._cbs = (B.SLAB_CALLBACK_BYTES(guarded(start)), B.SLAB_CALLBACK(guarded(wait)), B.SLAB_CALLBACK_N(guarded(allreduce)))
        self.struct = B.SlabComm(self.send_lo.data_ptr(), self.send_hi.data_ptr(), self.recv_lo.data_ptr(),
                                 self.recv_hi.data_ptr(), self.scalars.data_ptr(), self._cbs[0], self._cbs[1],
                                 self._cbs[2], ctypes.c_void_p(None))


def cg_solve_slab(g, kappa, U64, clover64, b, x, workspace, communicator, **kw):
    """D x = b on the decomposed lattice; every rank calls this with its slab.  Returns lqcd_cg_solve's info dict."""
    return B.cg_solve_slab(g, kappa, U64, clover64, b, x, workspace, communicator.struct, **kw)


def propagator_slab(g, L, world, rank, kappa, U64, clover64, y, columns, workspace, communicator, **kw):
    """propagator! point-source method on the decomposed lattice: for column = 3*spin + colour solve
    D x = delta_y e_column with lqcd_cg_solve_slab.  y: source position on the WHOLE lattice (only the rank whose slab
    holds y[3] has a non-zero source); columns: 12 consecutive internal fp64 spinor fields of this rank's slab.
    Returns the 12 info dicts."""
    T = slab_extent(L[3], world)
    t0 = slab_origin(L[3], world, rank)
    mine = t0 <= int(y[3]) < t0 + T
    fb = B.field_bytes(g, B.FIELD_SPINOR, B.F64)
    src = B.alloc_field(g, B.FIELD_SPINOR, B.F64)
    infos = []
    for col in range(12):
        if mine:
            B.point_source(g, (y[0], y[1], y[2], int(y[3]) - t0), col // 3, col % 3, src)
        else:
            src.zero_()
        infos.append(B.cg_solve_slab(g, kappa, U64, clover64, src, columns[col * fb:(col + 1) * fb], workspace,
                                     communicator.struct, **kw))
    return infos


def correlator_ps_slab(g, L, world, rank, columns, ncol, workspace, communicator, prec=B.F64):
    """C(x4) for all x4 of the whole lattice on every rank: each rank reduces its own time slices
    (lqcd_correlator_ps), the slices are put in place in a zero vector of length L4 and summed over the ranks."""
    import torch

    T = slab_extent(L[3], world)
    t0 = slab_origin(L[3], world, rank)
    local = B.correlator_ps(g, columns, ncol, workspace, T, prec)
    C = torch.zeros(int(L[3]), dtype=torch.float64, device=columns.device)
    C[t0:t0 + T] = torch.tensor(list(local), dtype=torch.float64, device=columns.device)
    communicator.exchange.allreduce_sum(C)
    return C.cpu().tolist()
