"""Thin ctypes binding of include/lqcd.h (liblqcd_b200.so): argument marshalling only.

Every function has the name of its C entry point minus the `lqcd_` prefix; every step of the path
runs in the CUDA kernels behind the C-ABI.  torch is used for device memory and streams only.
There is no CPU fallback: if the library is missing or no CUDA device is present, calls raise.
"""
import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "liblqcd_b200.so")

# enums of include/lqcd.h
OK, EINVAL, ENOMEM, ECUDA, ENOTCONV, EBREAKDOWN, EUNSUPPORTED = 0, -1, -2, -3, -4, -5, -6
BC_PERIODIC, BC_OPEN, BC_SF_ORBI, BC_SF_AFWB, BC_SLAB = 0, 1, 2, 3, 4
F64, F32 = 0, 1
SLAB_OPEN_LO, SLAB_OPEN_HI, SLAB_SF_HI = 1, 2, 4
RECON_18, RECON_12 = 18, 12
FIELD_GAUGE, FIELD_SPINOR, FIELD_CLOVER, FIELD_WORKSPACE, FIELD_FACE = 0, 1, 2, 3, 4

EXPORTS = [
    "lqcd_geom_create", "lqcd_geom_destroy", "lqcd_geom_info", "lqcd_field_bytes",
    "lqcd_gauge_import", "lqcd_gauge_export", "lqcd_spinor_import", "lqcd_spinor_export",
    "lqcd_clover_export", "lqcd_field_to_f32", "lqcd_clover_build", "lqcd_dw_apply", "lqcd_dwdag_apply",
    "lqcd_dw_eo_apply", "lqcd_point_source", "lqcd_cg_solve", "lqcd_cg_solve_multi", "lqcd_cg_multi_workspace_bytes", "lqcd_propagator_batched", "lqcd_propagator", "lqcd_spinor_norm2",
    "lqcd_spinor_dot", "lqcd_dw_apply_host", "lqcd_host_cache_release", "lqcd_last_error", "lqcd_launch_count", "lqcd_dw_plan",
    "lqcd_set_option", "lqcd_dw_apply_multi", "lqcd_correlator_ps", "lqcd_correlator_ps_static", "lqcd_dw_slab_pack", "lqcd_dw_slab_faces",
    "lqcd_clover_build_slab", "lqcd_cg_solve_slab",
    "lqcd_su2_field_bytes", "lqcd_su2_gauge_import", "lqcd_su2_gauge_export", "lqcd_su2_spinor_import",
    "lqcd_su2_spinor_export", "lqcd_su2_clover_build", "lqcd_su2_clover_export", "lqcd_su2_dw_apply", "lqcd_su2_cg_solve",
]


class LqcdError(RuntimeError):
    def __init__(self, status, msg):
        RuntimeError.__init__(self, "lqcd status %d: %s" % (status, msg))
        self.status = status


class GeomDesc(ctypes.Structure):
    _fields_ = [("L", ctypes.c_int * 4), ("bc", ctypes.c_int), ("theta", ctypes.c_double * 4),
                ("phi0", ctypes.c_double * 3), ("phiT", ctypes.c_double * 3), ("device", ctypes.c_int),
                ("slab_edges", ctypes.c_int)]


class Dirac(ctypes.Structure):
    _fields_ = [("kappa", ctypes.c_double), ("csw", ctypes.c_double), ("ct", ctypes.c_double),
                ("mu", ctypes.c_double)]


class CgParm(ctypes.Structure):
    _fields_ = [("tol", ctypes.c_double), ("maxiter", ctypes.c_int), ("mixed", ctypes.c_int), ("eo", ctypes.c_int),
                ("inner_tol", ctypes.c_double), ("check_every", ctypes.c_int)]


class CgInfo(ctypes.Structure):
    _fields_ = [("iters", ctypes.c_int), ("outer", ctypes.c_int), ("rel_resid_normal", ctypes.c_double),
                ("rel_resid_true", ctypes.c_double), ("seconds", ctypes.c_double)]


class CgFields(ctypes.Structure):
    _fields_ = [("U64", ctypes.c_void_p), ("clover64", ctypes.c_void_p), ("clover_inv64", ctypes.c_void_p),
                ("U32", ctypes.c_void_p), ("clover32", ctypes.c_void_p), ("clover_inv32", ctypes.c_void_p)]


_lib = None


def lib():
    """Load liblqcd_b200.so (built by paper_2503_16994_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s not found: run `python -m paper_2503_16994_b200.build` (there is no CPU fallback)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        L.lqcd_last_error.restype = ctypes.c_char_p
        L.lqcd_launch_count.restype = ctypes.c_longlong
        L.lqcd_field_bytes.restype = ctypes.c_size_t
        L.lqcd_field_bytes.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        _lib = L
    return _lib


def _check(st):
    if st != OK:
        raise LqcdError(st, lib().lqcd_last_error().decode())


def _ptr(t):
    """device (or host) pointer of a torch tensor / numpy array / int / None"""
    if t is None:
        return ctypes.c_void_p(None)
    if isinstance(t, int):
        return ctypes.c_void_p(t)
    if hasattr(t, "data_ptr"):
        return ctypes.c_void_p(t.data_ptr())
    if hasattr(t, "ctypes"):
        return ctypes.c_void_p(t.ctypes.data)
    raise TypeError("cannot take a pointer of %r" % type(t))


def _stream(stream):
    if stream is None:
        import torch
        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return ctypes.c_void_p(stream)
    return ctypes.c_void_p(stream.cuda_stream)


def _dirac(kappa, csw=0.0, ct=1.0, mu=0.0):
    return Dirac(float(kappa), float(csw), float(ct), float(mu))


def geom_desc(L, bc=BC_PERIODIC, theta=None, phi0=None, phiT=None, device=0, slab_edges=0):
    d = GeomDesc()
    for i in range(4):
        d.L[i] = int(L[i])
        d.theta[i] = float(theta[i]) if theta is not None else 0.0
    d.bc = int(bc)
    for i in range(3):
        d.phi0[i] = float(phi0[i]) if phi0 is not None else 0.0
        d.phiT[i] = float(phiT[i]) if phiT is not None else 0.0
    d.device = int(device)
    d.slab_edges = int(slab_edges)
    return d


def geom_create(L, bc=BC_PERIODIC, theta=None, phi0=None, phiT=None, device=0, slab_edges=0):
    d = geom_desc(L, bc, theta, phi0, phiT, device, slab_edges)
    g = ctypes.c_void_p()
    _check(lib().lqcd_geom_create(ctypes.byref(d), ctypes.byref(g)))
    return g


def geom_destroy(g):
    _check(lib().lqcd_geom_destroy(g))


def geom_info(g):
    tile, nt, chunk = (ctypes.c_int * 4)(), (ctypes.c_int * 4)(), (ctypes.c_int * 2)()
    _check(lib().lqcd_geom_info(g, tile, nt, chunk))
    return list(tile), list(nt), list(chunk)


def field_bytes(g, kind, prec=F64, recon=RECON_18):
    return int(lib().lqcd_field_bytes(g, kind, prec, recon))


def alloc_field(g, kind, prec=F64, recon=RECON_18, device="cuda"):
    """Device memory for one internal field (torch allocation: plumbing only)."""
    import torch
    return torch.empty(field_bytes(g, kind, prec, recon), dtype=torch.uint8, device=device)


def gauge_import(g, canon, U, prec=F64, recon=RECON_18, stream=None):
    _check(lib().lqcd_gauge_import(g, _ptr(canon), _ptr(U), prec, recon, _stream(stream)))


def gauge_export(g, U, canon, prec=F64, recon=RECON_18, stream=None):
    _check(lib().lqcd_gauge_export(g, _ptr(U), _ptr(canon), prec, recon, _stream(stream)))


def spinor_import(g, canon, psi, prec=F64, stream=None):
    _check(lib().lqcd_spinor_import(g, _ptr(canon), _ptr(psi), prec, _stream(stream)))


def spinor_export(g, psi, canon, prec=F64, stream=None):
    _check(lib().lqcd_spinor_export(g, _ptr(psi), _ptr(canon), prec, _stream(stream)))


def clover_export(g, clover, canon, prec=F64, stream=None):
    _check(lib().lqcd_clover_export(g, _ptr(clover), _ptr(canon), prec, _stream(stream)))


def field_to_f32(g, kind, recon, src64, dst32, stream=None):
    _check(lib().lqcd_field_to_f32(g, kind, recon, _ptr(src64), _ptr(dst32), _stream(stream)))


def clover_build(g, kappa, csw, U64, clover, clover_inv=None, recon=RECON_18, out_prec=F64, ct=1.0, stream=None):
    d = _dirac(kappa, csw, ct)
    _check(lib().lqcd_clover_build(g, ctypes.byref(d), _ptr(U64), recon, _ptr(clover), _ptr(clover_inv), out_prec,
                                   _stream(stream)))


def clover_build_slab(g, kappa, csw, U64, halo_lo, halo_hi, clover, clover_inv=None, recon=RECON_18, out_prec=F64,
                      stream=None, ct=1.0):
    """Csw! on a time slab (BC_SLAB); halo_lo / halo_hi: the neighbour ranks' adjacent time slices, canonical fp64
    (None on a face that is an open boundary)."""
    d = _dirac(kappa, csw, ct)
    _check(lib().lqcd_clover_build_slab(g, ctypes.byref(d), _ptr(U64), recon, _ptr(halo_lo), _ptr(halo_hi), _ptr(clover),
                                        _ptr(clover_inv), out_prec, _stream(stream)))


def dw_slab_pack(g, kappa, U, psi_in, send_lo, send_hi, dagger=False, prec=F64, recon=RECON_18, stream=None):
    d = _dirac(kappa)
    _check(lib().lqcd_dw_slab_pack(g, ctypes.byref(d), _ptr(U), _ptr(psi_in), _ptr(send_lo), _ptr(send_hi),
                                   1 if dagger else 0, prec, recon, _stream(stream)))


def dw_slab_faces(g, kappa, U, recv_lo, recv_hi, psi_out, dagger=False, prec=F64, recon=RECON_18, stream=None):
    d = _dirac(kappa)
    _check(lib().lqcd_dw_slab_faces(g, ctypes.byref(d), _ptr(U), _ptr(recv_lo), _ptr(recv_hi), _ptr(psi_out),
                                    1 if dagger else 0, prec, recon, _stream(stream)))


def dw_apply(g, kappa, U, clover, psi_in, psi_out, prec=F64, recon=RECON_18, stream=None, mu=0.0):
    d = _dirac(kappa, mu=mu)
    _check(lib().lqcd_dw_apply(g, ctypes.byref(d), _ptr(U), _ptr(clover), _ptr(psi_in), _ptr(psi_out), prec, recon,
                               _stream(stream)))


def dwdag_apply(g, kappa, U, clover, psi_in, psi_out, prec=F64, recon=RECON_18, stream=None, mu=0.0):
    d = _dirac(kappa, mu=mu)
    _check(lib().lqcd_dwdag_apply(g, ctypes.byref(d), _ptr(U), _ptr(clover), _ptr(psi_in), _ptr(psi_out), prec, recon,
                                  _stream(stream)))


def dw_eo_apply(g, kappa, U, clover, clover_inv, in_e, out_e, tmp, dagger=False, prec=F64, recon=RECON_18, stream=None):
    d = _dirac(kappa)
    _check(lib().lqcd_dw_eo_apply(g, ctypes.byref(d), _ptr(U), _ptr(clover), _ptr(clover_inv), _ptr(in_e), _ptr(out_e),
                                  _ptr(tmp), 1 if dagger else 0, prec, recon, _stream(stream)))


def point_source(g, y, spin, colour, b, prec=F64, stream=None):
    yy = (ctypes.c_int * 4)(*[int(v) for v in y])
    _check(lib().lqcd_point_source(g, yy, int(spin), int(colour), _ptr(b), prec, _stream(stream)))


def _cg_args(U64, clover64, clover_inv64, U32, clover32, clover_inv32, tol, maxiter, mixed, eo, inner_tol, check_every):
    f = CgFields(_ptr(U64), _ptr(clover64), _ptr(clover_inv64), _ptr(U32), _ptr(clover32), _ptr(clover_inv32))
    p = CgParm(float(tol), int(maxiter), 1 if mixed else 0, 1 if eo else 0, float(inner_tol), int(check_every))
    return f, p


def _info_dict(info, status):
    return {"iters": info.iters, "outer": info.outer, "rel_resid_normal": info.rel_resid_normal,
            "rel_resid_true": info.rel_resid_true, "seconds": info.seconds, "status": status}


def cg_solve(g, kappa, U64, clover64, b, x, workspace, tol=1e-10, maxiter=10000, clover_inv64=None, U32=None,
             clover32=None, clover_inv32=None, mixed=False, eo=False, inner_tol=1e-4, check_every=16,
             recon=RECON_18, stream=None, raise_on_notconv=True, mu=0.0):
    """Returns a dict (iters, outer, rel_resid_normal, rel_resid_true, seconds, status)."""
    d = _dirac(kappa, mu=mu)
    f, p = _cg_args(U64, clover64, clover_inv64, U32, clover32, clover_inv32, tol, maxiter, mixed, eo, inner_tol, check_every)
    info = CgInfo()
    st = lib().lqcd_cg_solve(g, ctypes.byref(d), ctypes.byref(f), _ptr(b), _ptr(x), _ptr(workspace), ctypes.byref(p),
                             ctypes.byref(info), recon, _stream(stream))
    if st != OK and not (st == ENOTCONV and not raise_on_notconv):
        _check(st)
    return _info_dict(info, st)


SLAB_CALLBACK = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p)
SLAB_CALLBACK_N = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_int)
SLAB_CALLBACK_BYTES = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_size_t)


class SlabComm(ctypes.Structure):
    """lqcd_slab_comm: face buffers, the all-reduce payload and the three host callbacks."""
    _fields_ = [("send_lo", ctypes.c_void_p), ("send_hi", ctypes.c_void_p), ("recv_lo", ctypes.c_void_p),
                ("recv_hi", ctypes.c_void_p), ("scalars", ctypes.c_void_p), ("exchange_start", SLAB_CALLBACK_BYTES),
                ("exchange_wait", SLAB_CALLBACK), ("allreduce_sum", SLAB_CALLBACK_N), ("ctx", ctypes.c_void_p)]


def cg_solve_slab(g, kappa, U64, clover64, b, x, workspace, comm, tol=1e-10, maxiter=10000, U32=None, clover32=None,
                  mixed=False, inner_tol=1e-4, check_every=16, recon=RECON_18, stream=None, raise_on_notconv=True, mu=0.0):
    """lqcd_cg_solve_slab; comm: a SlabComm (paper_2503_16994_b200.slab.SlabCommunicator builds one)."""
    d = _dirac(kappa, mu=mu)
    f, p = _cg_args(U64, clover64, None, U32, clover32, None, tol, maxiter, mixed, False, inner_tol, check_every)
    info = CgInfo()
    st = lib().lqcd_cg_solve_slab(g, ctypes.byref(d), ctypes.byref(f), _ptr(b), _ptr(x), _ptr(workspace),
                                  ctypes.byref(p), ctypes.byref(info), ctypes.byref(comm), recon, _stream(stream))
    if st != OK and not (st == ENOTCONV and not raise_on_notconv):
        _check(st)
    return _info_dict(info, st)


def propagator(g, kappa, U64, clover64, y, columns, workspace, tol=1e-10, maxiter=10000, clover_inv64=None, U32=None,
               clover32=None, clover_inv32=None, mixed=False, eo=False, inner_tol=1e-4, check_every=16,
               recon=RECON_18, stream=None, mu=0.0):
    """12 point-source columns (spin-major: column = 3*spin + colour) into `columns` (12 internal fp64 spinors)."""
    d = _dirac(kappa, mu=mu)
    f, p = _cg_args(U64, clover64, clover_inv64, U32, clover32, clover_inv32, tol, maxiter, mixed, eo, inner_tol, check_every)
    infos = (CgInfo * 12)()
    yy = (ctypes.c_int * 4)(*[int(v) for v in y])
    st = lib().lqcd_propagator(g, ctypes.byref(d), ctypes.byref(f), yy, _ptr(columns), _ptr(workspace), ctypes.byref(p),
                               infos, recon, _stream(stream))
    _check(st)
    return [_info_dict(infos[i], st) for i in range(12)]


def cg_multi_workspace_bytes(g, nrhs):
    lib().lqcd_cg_multi_workspace_bytes.restype = ctypes.c_size_t
    lib().lqcd_cg_multi_workspace_bytes.argtypes = [ctypes.c_void_p, ctypes.c_int]
    return int(lib().lqcd_cg_multi_workspace_bytes(g, int(nrhs)))


def cg_solve_multi(g, kappa, U64, clover64, b, x, nrhs, workspace, tol=1e-10, maxiter=10000, clover_inv64=None, U32=None,
                   clover32=None, clover_inv32=None, mixed=False, eo=False, inner_tol=1e-4, check_every=16,
                   recon=RECON_18, stream=None, raise_on_notconv=True, mu=0.0):
    """nrhs systems D x_n = b_n in lock step (b, x: nrhs internal fp64 spinor fields back to back); workspace of
    cg_multi_workspace_bytes(g, nrhs) bytes.  Returns a list of info dicts."""
    d = _dirac(kappa, mu=mu)
    f, p = _cg_args(U64, clover64, clover_inv64, U32, clover32, clover_inv32, tol, maxiter, mixed, eo, inner_tol, check_every)
    infos = (CgInfo * int(nrhs))()
    st = lib().lqcd_cg_solve_multi(g, ctypes.byref(d), ctypes.byref(f), _ptr(b), _ptr(x), int(nrhs), _ptr(workspace),
                                   ctypes.byref(p), infos, recon, _stream(stream))
    if st != OK and not (st == ENOTCONV and not raise_on_notconv):
        _check(st)
    return [_info_dict(infos[i], st) for i in range(int(nrhs))]


def propagator_batched(g, kappa, U64, clover64, y, columns, sources, workspace, tol=1e-10, maxiter=10000, check_every=16,
                       recon=RECON_18, stream=None, mu=0.0):
    """The 12 point-source columns through cg_solve_multi (plain fp64); sources: scratch of 12 spinor fields,
    workspace: cg_multi_workspace_bytes(g, 12) bytes."""
    d = _dirac(kappa, mu=mu)
    f, p = _cg_args(U64, clover64, None, None, None, None, tol, maxiter, False, False, 1e-4, check_every)
    infos = (CgInfo * 12)()
    yy = (ctypes.c_int * 4)(*[int(v) for v in y])
    st = lib().lqcd_propagator_batched(g, ctypes.byref(d), ctypes.byref(f), yy, _ptr(columns), _ptr(sources), _ptr(workspace),
                                       ctypes.byref(p), infos, recon, _stream(stream))
    _check(st)
    return [_info_dict(infos[i], st) for i in range(12)]


def spinor_norm2(g, v, workspace, half=False, prec=F64, stream=None):
    r = ctypes.c_double(0)
    _check(lib().lqcd_spinor_norm2(g, _ptr(v), 1 if half else 0, prec, _ptr(workspace), ctypes.byref(r), _stream(stream)))
    return r.value


def spinor_dot(g, u, v, workspace, half=False, prec=F64, stream=None):
    r = (ctypes.c_double * 2)()
    _check(lib().lqcd_spinor_dot(g, _ptr(u), _ptr(v), 1 if half else 0, prec, _ptr(workspace), r, _stream(stream)))
    return complex(r[0], r[1])


def dw_apply_host(L, kappa, csw, U_canon, psi_canon, out_canon, bc=BC_PERIODIC, theta=None, phi0=None, phiT=None,
                  dagger=False, prec=F64, recon=RECON_18, ct=1.0, device=0, mu=0.0):
    """End to end over HOST buffers (numpy complex128, canonical layout); copies are inside the call."""
    desc = geom_desc(L, bc, theta, phi0, phiT, device)
    d = _dirac(kappa, csw, ct, mu)
    _check(lib().lqcd_dw_apply_host(ctypes.byref(desc), ctypes.byref(d), _ptr(U_canon), _ptr(psi_canon), _ptr(out_canon),
                                    1 if dagger else 0, prec, recon))


def host_cache_release():
    """Free the device scratch lqcd_dw_apply_host keeps between calls."""
    _check(lib().lqcd_host_cache_release())


def dw_apply_multi(g, kappa, U, clover, src, dst, nrhs, prec=F64, recon=RECON_18, dagger=False, stream=None, mu=0.0):
    """D (or D^+) on nrhs spinor fields stored back to back in src / dst."""
    d = _dirac(kappa, mu=mu)
    _check(lib().lqcd_dw_apply_multi(g, ctypes.byref(d), _ptr(U), _ptr(clover), _ptr(src), _ptr(dst), int(nrhs),
                                     1 if dagger else 0, prec, recon, _stream(stream)))


def correlator_ps(g, columns, ncol, workspace, L4, prec=F64, stream=None):
    """C(x4) = sum_xvec sum_{columns, spin, colour} |S|^2 as a list of L4 floats."""
    C = (ctypes.c_double * int(L4))()
    _check(lib().lqcd_correlator_ps(g, _ptr(columns), int(ncol), prec, _ptr(workspace), C, _stream(stream)))
    return list(C)


CORRELATOR_STATIC_MAX_DOUBLES = 196608   # include/lqcd.h: LQCD_CORRELATOR_STATIC_MAX_DOUBLES


def correlator_ps_static(g, columns, ncol, L4, prec=F64, stream=None):
    """lqcd_correlator_ps without a workspace and without any allocation: the scratch is a static device array of the
    library (lattices up to ntiles * b4 + L4 <= CORRELATOR_STATIC_MAX_DOUBLES; calls must not overlap on the GPU)."""
    C = (ctypes.c_double * int(L4))()
    _check(lib().lqcd_correlator_ps_static(g, _ptr(columns), int(ncol), prec, C, _stream(stream)))
    return list(C)


def launch_count():
    return int(lib().lqcd_launch_count())


def dw_plan(g, prec=F64, recon=RECON_18, has_clover=True, parity=-1):
    """One line naming the stencil kernel and launch configuration lqcd_dw_apply would use."""
    buf = ctypes.create_string_buffer(512)
    _check(lib().lqcd_dw_plan(g, prec, recon, 1 if has_clover else 0, parity, buf, 512))
    return buf.value.decode()


def set_option(key, value):
    _check(lib().lqcd_set_option(key.encode(), value.encode()))


# ---- SU(2) fundamental representation (NEXT-4; include/lqcd.h "The SU(2) fundamental representation") ---------------
def su2_alloc_field(g, kind, prec=F64):
    import torch
    lib().lqcd_su2_field_bytes.restype = ctypes.c_size_t
    n = lib().lqcd_su2_field_bytes(g, kind, prec)
    return torch.empty(n, dtype=torch.uint8, device="cuda")


def su2_gauge_import(g, canon, U, prec=F64, stream=None):
    _check(lib().lqcd_su2_gauge_import(g, _ptr(canon), _ptr(U), prec, _stream(stream)))


def su2_gauge_export(g, U, canon, prec=F64, stream=None):
    _check(lib().lqcd_su2_gauge_export(g, _ptr(U), _ptr(canon), prec, _stream(stream)))


def su2_spinor_import(g, canon, psi, prec=F64, stream=None):
    _check(lib().lqcd_su2_spinor_import(g, _ptr(canon), _ptr(psi), prec, _stream(stream)))


def su2_spinor_export(g, psi, canon, prec=F64, stream=None):
    _check(lib().lqcd_su2_spinor_export(g, _ptr(psi), _ptr(canon), prec, _stream(stream)))


def su2_clover_build(g, kappa, csw, U64, clover, prec=F64, stream=None):
    d = _dirac(kappa, csw)
    _check(lib().lqcd_su2_clover_build(g, ctypes.byref(d), _ptr(U64), _ptr(clover), prec, _stream(stream)))


def su2_clover_export(g, clover, canon, prec=F64, stream=None):
    _check(lib().lqcd_su2_clover_export(g, _ptr(clover), _ptr(canon), prec, _stream(stream)))


def su2_dw_apply(g, kappa, U, clover, src, dst, dagger=False, prec=F64, stream=None):
    d = _dirac(kappa)
    _check(lib().lqcd_su2_dw_apply(g, ctypes.byref(d), _ptr(U), _ptr(clover), _ptr(src), _ptr(dst), 1 if dagger else 0, prec,
                                   _stream(stream)))


def su2_cg_solve(g, kappa, U64, clover64, b, x, workspace, tol=1e-10, maxiter=10000, check_every=16, stream=None,
                 raise_on_notconv=True):
    d = _dirac(kappa)
    f, p = _cg_args(U64, clover64, None, None, None, None, tol, maxiter, False, False, 1e-4, check_every)
    info = CgInfo()
    st = lib().lqcd_su2_cg_solve(g, ctypes.byref(d), _ptr(U64), _ptr(clover64), _ptr(b), _ptr(x), _ptr(workspace), ctypes.byref(p),
                                 ctypes.byref(info), _stream(stream))
    if st != OK and not (st == ENOTCONV and not raise_on_notconv):
        _check(st)
    return _info_dict(info, st)
