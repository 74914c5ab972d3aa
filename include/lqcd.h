/* lqcd.h -- C-ABI of the B200-native clover Wilson-Dirac / CG library (liblqcd_b200.so).
 *
 * What is computed is fixed by DESIGN.md ("Definitions D1-D8", restating SURVEY.md 8(c)); the paper
 * (arxiv 2503.16994, LatticeGPU.jl) names the operations and their arguments:
 *   SpaceParm  : lattice extents with time last, boundary conditions          PAPER.md:41-60  (sec. 2.1)
 *   DiracParam : m0 <-> kappa, csw, theta (boundary phases), cF = c~_t
 *   Dw!, g5Dw!, DwdagDw!(pso,U,psi,...) : out-of-place operator application
 *   Csw!(dws,U,gp,lp) : clover term stored in a workspace field, used by Dw
 *   CG!, propagator!(psi,U,dpar,dws,lp,maxiter,tol,...) -> iteration count
 *   GaugeParm phi : SF boundary links exp(i phi/L)
 *
 * Conventions
 *  - Every call returns lqcd_status (0 = OK, negative = error); nothing throws or aborts;
 *    lqcd_last_error() returns a thread-local message for the last failing call.
 *  - All field pointers are DEVICE pointers owned by the caller (e.g. torch allocations), at least
 *    lqcd_field_bytes() long and 16-byte aligned.  `stream` is a cudaStream_t cast to void* (NULL =
 *    default stream).  Calls are asynchronous on `stream`, except lqcd_cg_solve / lqcd_propagator /
 *    the *_host convenience calls, which synchronise before returning.
 *  - Inputs are const and left bit-unchanged; outputs must not alias inputs (LQCD_EINVAL).
 *  - There is no CPU fallback: without a CUDA device every compute call returns LQCD_ECUDA.
 *  - "canonical" (interchange) layout, always fp64 complex (re,im), site n = x1 + L1*(x2 + L2*(x3 + L3*x4)),
 *    x4 = time:   gauge  [n][mu=0..3][row][col]   (18 reals per link, mu=3 is time)
 *                 spinor [n][spin=0..3][colour=0..2]
 *                 clover [n][chirality=0..1][6][6]  dense Hermitian blocks, row = 3*s + a
 *  - "internal" layout: private, tile-blocked even-odd structure of arrays;
 *    only this library reads or writes it.  A full internal field is [even half | odd half]; the
 *    even-odd operator works on the even half (first lqcd_field_bytes/2 bytes of a spinor).
 *  - gamma basis, sign and normalisation conventions: DESIGN.md D2-D6.  D = A - kappa*H,
 *    kappa = 1/(2(m0+4)), D_paper = D/(2 kappa).
 */
#ifndef LQCD_H
#define LQCD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  LQCD_OK = 0,
  LQCD_EINVAL = -1,      /* bad argument (odd extent, aliasing, NULL pointer, bad enum)            */
  LQCD_ENOMEM = -2,
  LQCD_ECUDA = -3,       /* CUDA runtime error or no device                                         */
  LQCD_ENOTCONV = -4,    /* CG hit maxiter; x holds the last iterate                                */
  LQCD_EBREAKDOWN = -5,  /* CG saw a NaN or a non-positive <p, D^+D p>                              */
  LQCD_EUNSUPPORTED = -6
} lqcd_status;

typedef enum {
  LQCD_BC_PERIODIC = 0, LQCD_BC_OPEN = 1, LQCD_BC_SF_ORBI = 2, LQCD_BC_SF_AFWB = 3,
  LQCD_BC_SLAB = 4   /* one time slab of a lattice periodic in time: see "Time-direction domain decomposition" below */
} lqcd_bc;
typedef enum { LQCD_F64 = 0, LQCD_F32 = 1 } lqcd_prec;
typedef enum { LQCD_RECON_18 = 18, LQCD_RECON_12 = 12 } lqcd_recon;
typedef enum {
  LQCD_FIELD_GAUGE = 0, LQCD_FIELD_SPINOR = 1, LQCD_FIELD_CLOVER = 2, LQCD_FIELD_WORKSPACE = 3,
  LQCD_FIELD_FACE = 4   /* one half-spinor time face of a slab: 6 complex numbers x L[0] L[1] L[2] sites */
} lqcd_field_kind;

/* Geometry (the paper's SpaceParm, plus the fermion phases of DiracParam, :119). */
typedef struct {
  int L[4];            /* extents, L[3] = time; all even and >= 2; >= 4 in time for open/SF */
  lqcd_bc bc;          /* PAPER.md:53-58.  SF_ORBI and SF_AFWB are the same for the fermion path (R9)     */
  double theta[4];     /* ANGLES: every link of direction mu carries exp(i*theta[mu]/L[mu]) (R6)          */
  double phi0[3];      /* SF only, informational: phases of the x4=0 boundary links, which the caller     */
                       /* stores in the gauge array itself (R8)                                          */
  double phiT[3];      /* SF only: phases of the x4=T boundary links W'_k = exp(i*phiT/L_k) */
  int device;          /* CUDA ordinal                                                                   */
  int slab_edges;      /* LQCD_BC_SLAB only: bit 0 (LQCD_SLAB_OPEN_LO) / bit 1 (LQCD_SLAB_OPEN_HI) = the slab's lower /  */
                       /* upper time face is an OPEN boundary of the lattice (first / last rank of a lattice with  */
                       /* open BC): that slice is frozen (D7) and nothing is exchanged through it.  0 = periodic.  */
} lqcd_geom_desc;
enum { LQCD_SLAB_OPEN_LO = 1, LQCD_SLAB_OPEN_HI = 2,
       LQCD_SLAB_SF_HI = 4 };   /* the upper face is the SF boundary x4 = T (last rank of an SF lattice; its first rank */
                                /* sets LQCD_SLAB_OPEN_LO: the frozen slice x4 = 0): no slice of the slab is frozen   */
                                /* there, nothing is exchanged, and Csw! takes the boundary field W' from phiT      */

/* Dirac parameters: kappa = 1/(2(m0+4)); csw; ct = c~_t (paper's cF), 1 = absent; mu = twisted
 * mass: D = A + 2 i kappa mu gamma5 - kappa H, D^+ = gamma5 D(-mu) gamma5; 0 = absent.
 * mu != 0 is supported by lqcd_dw_apply / lqcd_dwdag_apply / lqcd_dw_apply_multi / lqcd_dw_apply_host and by the
 * plain (not even-odd) lqcd_cg_solve / lqcd_propagator; the even-odd paths return LQCD_EINVAL for mu != 0. */
typedef struct { double kappa, csw, ct, mu; } lqcd_dirac;

typedef struct lqcd_geom lqcd_geom;   /* opaque, library-owned */

lqcd_status lqcd_geom_create(const lqcd_geom_desc* desc, lqcd_geom** out);
lqcd_status lqcd_geom_destroy(lqcd_geom* g);
/* tile shape (4 ints), tiles per direction (4 ints) and L2 chunking (2 ints) chosen for this lattice */
lqcd_status lqcd_geom_info(const lqcd_geom* g, int tile[4], int ntiles[4], int chunk[2]);

/* Bytes of one internal field.  WORKSPACE: what lqcd_cg_solve / lqcd_propagator need (prec = LQCD_F64
 * covers the mixed-precision solver too). */
size_t lqcd_field_bytes(const lqcd_geom* g, lqcd_field_kind kind, lqcd_prec prec, lqcd_recon recon);

/* canonical (fp64) <-> internal.  Import rounds once to `prec` (R14). */
lqcd_status lqcd_gauge_import(const lqcd_geom* g, const void* canon, void* U, lqcd_prec prec, lqcd_recon recon, void* stream);
lqcd_status lqcd_gauge_export(const lqcd_geom* g, const void* U, void* canon, lqcd_prec prec, lqcd_recon recon, void* stream);
lqcd_status lqcd_spinor_import(const lqcd_geom* g, const void* canon, void* psi, lqcd_prec prec, void* stream);
lqcd_status lqcd_spinor_export(const lqcd_geom* g, const void* psi, void* canon, lqcd_prec prec, void* stream);
lqcd_status lqcd_clover_export(const lqcd_geom* g, const void* clover, void* canon, lqcd_prec prec, void* stream);
/* internal fp64 spinor/clover/gauge -> internal fp32 (round to nearest), same geometry */
lqcd_status lqcd_field_to_f32(const lqcd_geom* g, lqcd_field_kind kind, lqcd_recon recon, const void* src64, void* dst32, void* stream);

/* Csw! (D4, D5): A(x) = 1 + kappa*csw*(i/2) sum sigma_{mu nu} F^_{mu nu}(x) as two packed 6x6
 * Hermitian blocks per site; F^ = (Q - Q^+)/8 from the four plaquette leaves.  Always evaluated in fp64
 * from fp64 links `U64` (R14) and stored in `out_prec`.  clover_inv (may be NULL) receives A^{-1}. */
lqcd_status lqcd_clover_build(const lqcd_geom* g, const lqcd_dirac* d, const void* U64, lqcd_recon recon,
                              void* clover, void* clover_inv, lqcd_prec out_prec, void* stream);

/* Dw! (D6): out = A in - kappa H in.  clover == NULL => A = 1 (csw term absent until Csw!
 * has been called).  lqcd_dwdag_apply: out = gamma5 D gamma5 in. */
lqcd_status lqcd_dw_apply(const lqcd_geom* g, const lqcd_dirac* d, const void* U, const void* clover,
                          const void* in, void* out, lqcd_prec prec, lqcd_recon recon, void* stream);
lqcd_status lqcd_dwdag_apply(const lqcd_geom* g, const lqcd_dirac* d, const void* U, const void* clover,
                             const void* in, void* out, lqcd_prec prec, lqcd_recon recon, void* stream);
/* Even-odd preconditioned operator (D8) on even-site half fields:
 * out_e = A_ee in_e - kappa^2 H_eo A_oo^{-1} H_oe in_e (dagger: gamma5 . gamma5).  tmp: one spinor field. */
lqcd_status lqcd_dw_eo_apply(const lqcd_geom* g, const lqcd_dirac* d, const void* U, const void* clover,
                             const void* clover_inv, const void* in_e, void* out_e, void* tmp, int dagger,
                             lqcd_prec prec, lqcd_recon recon, void* stream);

/* b = delta_{x,y} e_{spin,colour} in the internal layout (propagator! point-source method). */
lqcd_status lqcd_point_source(const lqcd_geom* g, const int y[4], int spin, int colour, void* b, lqcd_prec prec, void* stream);

/* CG! on the normal equations (algorithm and stopping rule: DESIGN.md R11):
 *   solves D x = b via D^+D x = D^+ b from x0 = 0 until |r| <= tol*|D^+ b| (recursive residual).
 *   eo != 0   : even-odd preconditioned (D8), needs clover and clover_inv.
 *   mixed != 0: defect correction, fp32 inner CG to inner_tol, fp64 outer; needs the *32 fields. */
typedef struct { double tol; int maxiter; int mixed; int eo; double inner_tol; int check_every; } lqcd_cg_parm;
typedef struct { int iters; int outer; double rel_resid_normal; double rel_resid_true; double seconds; } lqcd_cg_info;
typedef struct {
  const void* U64; const void* clover64; const void* clover_inv64;   /* fp64 internal fields             */
  const void* U32; const void* clover32; const void* clover_inv32;   /* fp32 copies (mixed only, else NULL) */
} lqcd_cg_fields;
lqcd_status lqcd_cg_solve(const lqcd_geom* g, const lqcd_dirac* d, const lqcd_cg_fields* f, const void* b,
                          void* x, void* workspace, const lqcd_cg_parm* parm, lqcd_cg_info* info,
                          lqcd_recon recon, void* stream);

/* propagator! point-source method: for column = 3*spin + colour = 0..11 solve D x = delta_y e_column
 * with lqcd_cg_solve's parameters.  `columns`: 12 consecutive internal fp64 spinor fields (caller-owned, out);
 * infos[12] filled per column.  Stops at the first column that fails and returns its status. */
lqcd_status lqcd_propagator(const lqcd_geom* g, const lqcd_dirac* d, const lqcd_cg_fields* f, const int y[4],
                            void* columns, void* workspace, const lqcd_cg_parm* parm, lqcd_cg_info infos[12],
                            lqcd_recon recon, void* stream);

/* BLAS-1 used by the solver, exported for tests: |v|^2 and <u,v> over a full (or even-half) spinor. */
lqcd_status lqcd_spinor_norm2(const lqcd_geom* g, const void* v, int half, lqcd_prec prec, void* workspace, double* result_host, void* stream);
lqcd_status lqcd_spinor_dot(const lqcd_geom* g, const void* u, const void* v, int half, lqcd_prec prec, void* workspace, double* result_host /* re, im */, void* stream);

/* SURVEY.md 8(f) NEXT-1 carried into the solver (the 12 colour-spin sources of propagator!):
 * nrhs (1..64) independent systems D x_n = b_n solved by CG on the normal equations IN LOCK STEP -- every stencil
 * pass is one lqcd_dw_apply_multi over all columns (links and clover blocks are fetched once per tile for all of
 * them) with the |t|^2 / r -= alpha q / |r|^2 epilogues fused per column; alpha, beta, the iteration count and the
 * convergence flag are kept per column on the device, and a column that has converged is frozen (alpha = 0) while
 * the others go on.  Per column the arithmetic is that of lqcd_cg_solve (same iterates, same iteration count).
 *   b, x      : DEVICE, nrhs internal fp64 spinor fields back to back (lqcd_field_bytes(SPINOR) apart), caller-owned,
 *               not overlapping; components of b on frozen time slices are ignored (D7)
 *   workspace : DEVICE, lqcd_cg_multi_workspace_bytes(g, nrhs) bytes (4 nrhs spinor fields + reduction scratch)
 *   infos     : HOST, nrhs entries; `seconds` is the time of the whole call in every entry
 * Plain fp64 only: with parm->eo or parm->mixed set, with nrhs == 1, or on a lattice the pipeline kernel does not
 * serve (tiles other than 4^4), the columns are solved one after the other by lqcd_cg_solve (same results; the fields
 * those modes need must then be in `f`).  Errors: as lqcd_cg_solve; LQCD_ENOTCONV / LQCD_EBREAKDOWN if any column
 * failed (lqcd_last_error names the first / the broken one), all infos are filled.
 * lqcd_propagator_batched: the 12 point-source columns of lqcd_propagator through lqcd_cg_solve_multi; `sources`:
 * DEVICE scratch for the 12 source fields (12 spinor fields, caller-owned). */
size_t lqcd_cg_multi_workspace_bytes(const lqcd_geom* g, int nrhs);
lqcd_status lqcd_cg_solve_multi(const lqcd_geom* g, const lqcd_dirac* d, const lqcd_cg_fields* f, const void* b, void* x,
                                int nrhs, void* workspace, const lqcd_cg_parm* parm, lqcd_cg_info* infos, lqcd_recon recon,
                                void* stream);
lqcd_status lqcd_propagator_batched(const lqcd_geom* g, const lqcd_dirac* d, const lqcd_cg_fields* f, const int y[4],
                                    void* columns, void* sources, void* workspace, const lqcd_cg_parm* parm,
                                    lqcd_cg_info infos[12], lqcd_recon recon, void* stream);

/* SURVEY.md 8(f) NEXT-2 (PAPER.md:11 "fermionic two point functions", :125 the columns of propagator!): the
 * pseudoscalar two-point function of ncol propagator columns,
 *   C(x4) = sum over x1,x2,x3 of sum over columns, spin, colour of |S(x)|^2      ( = sum_xvec Tr S^+ S ),
 * accumulated in fp64 in a fixed order.  columns: DEVICE array of ncol internal spinor fields stored back to back
 * (as lqcd_propagator writes them); workspace: DEVICE, lqcd_field_bytes(WORKSPACE); C_host: HOST array of L4
 * doubles, valid on return (the call synchronises the stream).  A noise-source propagator (the other method of
 * propagator!) is lqcd_cg_solve on a caller-supplied Gaussian source: random numbers are inputs of this library. */
lqcd_status lqcd_correlator_ps(const lqcd_geom* g, const void* columns, int ncol, lqcd_prec prec, void* workspace,
                               double* C_host, void* stream);

/* The same for callers that cannot allocate device memory or provide a
 * workspace -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The scratch
 * (ntiles * tile extent in time + L4 doubles) is a static array of LQCD_CORRELATOR_STATIC_MAX_DOUBLES doubles
 * (1.5 MiB) in the device memory of every GPU that loads the library, held until the process exits; the call itself
 * makes no cudaMalloc / cudaFree and calls no allocating library routine.  Same kernels as lqcd_correlator_ps: the
 * result is bit-identical.  columns: DEVICE, ncol internal spinor fields back to back; C_host: HOST, L4 doubles, valid
 * on return (the call synchronises the stream).  Errors: LQCD_EINVAL for NULL / bad enum / ncol outside 1..4096, and
 * for a lattice whose scratch does not fit (e.g. 64^3 x 128; 48^3 x 96 fits) -- use lqcd_correlator_ps then.
 * All calls on a device share the array (nothing in it needs clearing: every element read is written earlier in the
 * same call), so calls that overlap on the GPU -- other streams, other host threads -- race: serialise them. */
#define LQCD_CORRELATOR_STATIC_MAX_DOUBLES 196608
lqcd_status lqcd_correlator_ps_static(const lqcd_geom* g, const void* columns, int ncol, lqcd_prec prec, double* C_host,
                                      void* stream);

/* End-to-end call over HOST buffers in the canonical layout (SURVEY.md 8(b), 8(d) "e2e"; Csw! then
 * Dw! on a configuration that lives on the host).  U_canon_host [V][4][3][3], in_canon_host / out_canon_host [V][4][3],
 * complex fp64, HOST memory (pinned memory makes the copies asynchronous; pageable memory works).  The gauge field is
 * copied in time slabs through two device staging buffers; each slab is converted to the internal layout and the
 * clover term of the time slices whose neighbours have arrived is built while the next slab crosses PCIe; then the
 * spinor is imported, D (dagger = 0) or D^+ applied in `prec`, the result exported and copied back.  The call returns
 * when out_canon_host is valid.  Device scratch, streams and the geometry are kept by the library between calls and
 * reused when desc, prec and recon are unchanged (one cached context per process, mutex-guarded);
 * lqcd_host_cache_release() frees them.  Errors: LQCD_EINVAL (NULL, bad enum, kappa <= 0, LQCD_BC_SLAB),
 * LQCD_ECUDA / LQCD_ENOMEM (the cache is released). */
lqcd_status lqcd_dw_apply_host(const lqcd_geom_desc* desc, const lqcd_dirac* d, const void* U_canon_host,
                               const void* in_canon_host, void* out_canon_host, int dagger, lqcd_prec prec,
                               lqcd_recon recon);
lqcd_status lqcd_host_cache_release(void);

/* Time-direction domain decomposition (the volume one GPU holds
 * is the paper's stated limit).  A rank owns the slab x4 in [t0, t0 + L[3]) of a lattice periodic in time and creates
 * its geometry with bc = LQCD_BC_SLAB, L[3] = the slab's extent and theta[3] = theta4 * L[3] / L4 (the per-link
 * phase exp(i theta4 / L4) of the whole lattice; an antiperiodic lattice is theta4 = pi).  One application of D:
 *   1. lqcd_dw_slab_pack   : in -> send_lo, send_hi (DEVICE, caller-owned, lqcd_field_bytes(LQCD_FIELD_FACE) each):
 *                            half spinors of the first / last slice; the backward hop's link multiply is done here.
 *   2. the caller moves send_lo to the rank below (its recv_hi) and send_hi to the rank above (its recv_lo); with one
 *      rank the two are swapped in place, which reproduces the periodic lattice;
 *   3. lqcd_dw_apply / lqcd_dwdag_apply on the slab (the hops through the two time faces are left out; it may run
 *      while the faces travel);
 *   4. lqcd_dw_slab_faces  : out -= kappa * (the two missing hops) from recv_lo, recv_hi.  Call after 3 on `out`.
 * Step 3 + 4 equal the whole-lattice operator restricted to the slab (rounding order of the last additions aside).
 * A lattice with OPEN time boundaries is decomposed the same way: its first / last rank set slab_edges; their outer
 * slice is frozen as in LQCD_BC_OPEN, the pack / face kernels leave that face alone and the ring is not closed
 * (theta[3] plays no role across an open boundary).  An SF lattice: first rank LQCD_SLAB_OPEN_LO, last rank
 * LQCD_SLAB_SF_HI (with phiT in its geometry descriptor).
 * lqcd_clover_build_slab: Csw! on the slab; halo_lo / halo_hi = the time slice just below / above the slab, DEVICE,
 * canonical fp64 layout [L0 L1 L2][4][3][3] (a one-off exchange per configuration).  On a SLAB geometry the solver,
 * the even-odd operator and lqcd_clover_build return LQCD_EUNSUPPORTED (they would ignore the faces). */
lqcd_status lqcd_dw_slab_pack(const lqcd_geom* g, const lqcd_dirac* d, const void* U, const void* in, void* send_lo,
                              void* send_hi, int dagger, lqcd_prec prec, lqcd_recon recon, void* stream);
lqcd_status lqcd_dw_slab_faces(const lqcd_geom* g, const lqcd_dirac* d, const void* U, const void* recv_lo,
                               const void* recv_hi, void* out, int dagger, lqcd_prec prec, lqcd_recon recon, void* stream);
lqcd_status lqcd_clover_build_slab(const lqcd_geom* g, const lqcd_dirac* d, const void* U64, lqcd_recon recon,
                                   const void* halo_lo, const void* halo_hi, void* clover, void* clover_inv,
                                   lqcd_prec out_prec, void* stream);

/* CG! on the slabs of a decomposed lattice (8(e)(ii): "CG adds two scalar all-reduces per iteration"): the algorithm
 * of lqcd_cg_solve (plain fp64, not even-odd) with D applied as pack / exchange / stencil / faces and every inner
 * product summed over the ranks.  All ranks call it together with their slab's fields.  The library does no
 * communication itself: the caller supplies three host callbacks, each called while the library enqueues work on
 * `stream`, each returning 0 on success (nonzero aborts the solve with LQCD_ECUDA on that rank):
 *   exchange_start(ctx, nbytes): the first nbytes of send_lo / send_hi have been written by work already enqueued on
 *                        `stream`; start moving them into the rank below's recv_hi and the rank above's recv_lo
 *                        (ordered after `stream`'s current tail, e.g. on a second stream so that the transfer overlaps
 *                        the stencil kernel).  nbytes = lqcd_field_bytes(LQCD_FIELD_FACE) of the precision at work;
 *   exchange_wait(ctx) : make `stream` wait until recv_lo / recv_hi have arrived;
 *   allreduce_sum(ctx, n): sum scalars[0..n) (DEVICE doubles, written by work enqueued on `stream`) over all ranks,
 *                        in place, ordered on `stream`.
 * Face buffers (fp64-sized) and scalars (>= 4 doubles): DEVICE, caller-owned.  b, x: this rank's slab of the source /
 * solution.  f, parm, info as lqcd_cg_solve (residuals of the whole lattice); parm->mixed != 0 runs the fp32 inner CG
 * on the slabs too (fp32 faces, half the bytes); parm->eo must be 0. */
typedef struct {
  void* send_lo; void* send_hi; void* recv_lo; void* recv_hi;
  double* scalars;
  int (*exchange_start)(void* ctx, size_t nbytes);
  int (*exchange_wait)(void* ctx);
  int (*allreduce_sum)(void* ctx, int n);
  void* ctx;
} lqcd_slab_comm;
lqcd_status lqcd_cg_solve_slab(const lqcd_geom* g, const lqcd_dirac* d, const lqcd_cg_fields* f, const void* b, void* x,
                               void* workspace, const lqcd_cg_parm* parm, lqcd_cg_info* info,
                               const lqcd_slab_comm* comm, lqcd_recon recon, void* stream);

/* SURVEY.md 8(f) NEXT-1 (the 12 colour-spin sources of propagator! share one gauge field): D or D^+
 * (dagger != 0) applied to nrhs (1..64) spinor fields in one pass.  in / out: DEVICE arrays of nrhs internal spinor
 * fields stored back to back (lqcd_field_bytes(SPINOR) apart), caller-owned, not overlapping.  Links and clover
 * blocks are fetched from HBM once per tile and serve all right-hand sides (the 2nd..nth come out of L2), i.e.
 * 144 + 48 nrhs reals per site instead of 192 nrhs.  Same result, bit for bit, as nrhs separate calls. */
lqcd_status lqcd_dw_apply_multi(const lqcd_geom* g, const lqcd_dirac* d, const void* U, const void* clover,
                                const void* in, void* out, int nrhs, int dagger, lqcd_prec prec, lqcd_recon recon,
                                void* stream);

/* Which kernel lqcd_dw_apply / lqcd_dwdag_apply (parity = -1) or one half-lattice pass of lqcd_dw_eo_apply
 * (parity = 0/1) launches for this geometry, precision, link format and clover flag, with its launch
 * configuration, written as one line of text into buf (at most len bytes, always terminated).  Host only;
 * for bench.py and the tests.  The choice follows the option "dw_mode" (below) and the tile shape. */
lqcd_status lqcd_dw_plan(const lqcd_geom* g, lqcd_prec prec, lqcd_recon recon, int has_clover, int parity,
                         char* buf, int len);
/* Process-wide options (host strings).  "dw_mode": which stencil kernel serves the full-lattice operator --
 * "pipe" (default: the warp-specialised shared-memory pipeline where the tile shape allows it), "stream"
 * (persistent one-thread-per-site CTAs), "split" (one parity of a tile per CTA), "direct" (one CTA per tile).
 * All four compute the same operator; the environment variable LQCD_DW_MODE sets the initial value.
 * "host_slab": decimal string n >= 0, time slices per staged gauge slab of lqcd_dw_apply_host (0 = automatic: about
 * 1/12 of the lattice, at least 64 MB).  "pipe_grid": decimal string n >= 0, at most n CTAs for the pipeline kernel (0 = default, one per SM) -- a test hook:
 * with one or two CTAs each of them walks hundreds of tiles and wraps its mbarrier rings many times.
 * LQCD_EINVAL for an unknown key or value. */
lqcd_status lqcd_set_option(const char* key, const char* value);

const char* lqcd_last_error(void);
/* number of kernels launched by this library since load (for bench.py's gpu_launches) */
long long lqcd_launch_count(void);

/* ---------------------------------------------------------------------------------------------------------------
 * The SU(2) fundamental representation (section 2.2: gauge fields in SU2{T},
 * stored in the Cayley-Dickson form g = (z1, z2), |z1|^2 + |z2|^2 = 1; fermion fields Spinor{4, SU2fund}).
 * Same geometry handle, same definitions D1-D8 with two colours, same tile-blocked layout; per site 8 complex numbers
 * of links (4 directions x (z1, z2); U = [[z1, z2], [-conj z2, conj z1]]), 8 of spinor (index 2*spin + colour) and 16
 * of clover term (two packed Hermitian 4x4 blocks, row index 2*s + a).  Canonical (interchange) layouts, DEVICE
 * memory, complex fp64: gauge [V][4][2][2] (full matrices; import keeps the first row), spinor [V][4][2], blocks
 * [V][2][4][4].  Periodic and open time boundaries (LQCD_EUNSUPPORTED-like LQCD_EINVAL otherwise); mu = 0, ct = 1;
 * no even-odd or mixed-precision solver.  One-thread-per-site kernels (the shared-memory pipeline is SU(3) only).
 * lqcd_su2_field_bytes: GAUGE | SPINOR | CLOVER | WORKSPACE (of lqcd_su2_cg_solve).  All calls are asynchronous on
 * `stream` except lqcd_su2_cg_solve (PAPER.md:125 CG!, :171-172: maxiter, tol, iteration count), which follows
 * lqcd_cg_solve: x0 = 0, stop when |r| <= tol |D^+ b| (recursive residual), true residuals in `info`, LQCD_ENOTCONV
 * with the last iterate in x when maxiter is hit, components of b on frozen slices ignored. */
size_t lqcd_su2_field_bytes(const lqcd_geom* g, lqcd_field_kind kind, lqcd_prec prec);
lqcd_status lqcd_su2_gauge_import(const lqcd_geom* g, const void* canon, void* U, lqcd_prec prec, void* stream);
lqcd_status lqcd_su2_gauge_export(const lqcd_geom* g, const void* U, void* canon, lqcd_prec prec, void* stream);
lqcd_status lqcd_su2_spinor_import(const lqcd_geom* g, const void* canon, void* psi, lqcd_prec prec, void* stream);
lqcd_status lqcd_su2_spinor_export(const lqcd_geom* g, const void* psi, void* canon, lqcd_prec prec, void* stream);
/* Csw! from the fp64 links; the blocks are rounded once to out_prec (R14) */
lqcd_status lqcd_su2_clover_build(const lqcd_geom* g, const lqcd_dirac* d, const void* U64, void* clover, lqcd_prec out_prec,
                                  void* stream);
lqcd_status lqcd_su2_clover_export(const lqcd_geom* g, const void* clover, void* canon, lqcd_prec prec, void* stream);
/* Dw!: out = D in (dagger = 0) or D^+ in; clover = NULL means csw = 0; out must not alias an input */
lqcd_status lqcd_su2_dw_apply(const lqcd_geom* g, const lqcd_dirac* d, const void* U, const void* clover, const void* in,
                              void* out, int dagger, lqcd_prec prec, void* stream);
lqcd_status lqcd_su2_cg_solve(const lqcd_geom* g, const lqcd_dirac* d, const void* U64, const void* clover64, const void* b,
                              void* x, void* workspace, const lqcd_cg_parm* parm, lqcd_cg_info* info, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* LQCD_H */
