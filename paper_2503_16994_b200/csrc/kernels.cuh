// kernels.cuh -- host-callable launchers of layout.cu, clover.cu and blas.cu.
#pragma once
#include "dw.cuh"

namespace lqcd {

// layout.cu
template <typename T> cudaError_t gauge_import(const Geom& g, const void* canon, void* U, int recon, cudaStream_t s);
// the time slab t_lo <= x4 < t_hi only; canon_slab points at the first site of slice t_lo
template <typename T> cudaError_t gauge_import_slab(const Geom& g, const void* canon_slab, void* U, int recon, int t_lo, int t_hi, cudaStream_t s);
template <typename T> cudaError_t gauge_export(const Geom& g, const void* U, void* canon, int recon, cudaStream_t s);
template <typename T> cudaError_t spinor_import(const Geom& g, const void* canon, void* psi, cudaStream_t s);
template <typename T> cudaError_t spinor_export(const Geom& g, const void* psi, void* canon, cudaStream_t s);
template <typename T> cudaError_t clover_export(const Geom& g, const void* A, void* canon, cudaStream_t s);
template <typename T> cudaError_t point_source(const Geom& g, const int y[4], int spin, int colour, void* b, cudaStream_t s);
cudaError_t to_f32(const void* src, void* dst, size_t ncomplex, cudaStream_t s);

// clover.cu
struct CloverParm {
  double kappa, csw, ct;
  double phiT[3];
  int t_lo = 0, t_hi = 1 << 30;   // only sites with t_lo <= x4 < t_hi are built (the host path builds time slabs as they arrive)
};
// halo_lo / halo_hi: LQCD_BC_SLAB only (the neighbour ranks' adjacent time slices, canonical fp64 layout)
cudaError_t clover_build(const Geom& g, const CloverParm& cp, const void* U64, int recon, void* clover, void* clover_inv,
                         int out_prec, cudaStream_t s, const void* halo_lo = nullptr, const void* halo_hi = nullptr);

// slab.cu (NEXT-3): half-spinor faces of a time slab; [6][L1 L2 L3] complex numbers each
}  // namespace lqcd
struct lqcd_geom;
namespace lqcd {
// su2.cu -- the SU(2) fundamental representation (NEXT-4): Cayley-Dickson links (8 complex per site), 4 x 2 spinors (8),
// two packed Hermitian 4x4 blocks (16)
template <typename T> cudaError_t su2_gauge_import(const Geom& g, const void* canon, void* U, cudaStream_t s);
template <typename T> cudaError_t su2_gauge_export(const Geom& g, const void* U, void* canon, cudaStream_t s);
template <typename T> cudaError_t su2_spinor_import(const Geom& g, const void* canon, void* psi, cudaStream_t s);
template <typename T> cudaError_t su2_spinor_export(const Geom& g, const void* psi, void* canon, cudaStream_t s);
template <typename T> cudaError_t su2_clover_build(const Geom& g, double kappa, double csw, const void* U64, void* A, cudaStream_t s);
template <typename T> cudaError_t su2_clover_export(const Geom& g, const void* A, void* canon, cudaStream_t s);
template <typename T> cudaError_t su2_dw(const lqcd_geom* h, double kappa, const void* U, const void* A, const void* in, void* out, bool dagger, cudaStream_t s);
template <typename T> cudaError_t su2_mask_frozen(const Geom& g, void* psi, cudaStream_t s);
}  // namespace lqcd
namespace lqcd {
template <typename T> cudaError_t slab_pack(const lqcd_geom* h, bool dagger, const void* U, int recon, const void* in,
                                            void* send_lo, void* send_hi, cudaStream_t s);
template <typename T> cudaError_t slab_faces(const lqcd_geom* h, double kappa, bool dagger, const void* U, int recon,
                                             const void* recv_lo, const void* recv_hi, void* out, cudaStream_t s);

// blas.cu -- CG scalars live on the device
struct CgState {
  double rho, rho0, alpha, beta, tt, rho_new, tol2;
  int done;       // 0 running, 2 converged this iteration (x update pending), 1 finished
  int iters;
  int breakdown;
  int pad;
};
int reduce_blocks(size_t ncomplex);  // grid size used by the norm/dot kernels (partial buffer length)
int reduce_blocks_max();             // its upper bound: 8 CTAs per SM of the device
void set_reduce_sm_count(int sms);   // called by lqcd_geom_create with the device's SM count
template <typename T> cudaError_t norm2_partial(const void* v, size_t ncomplex, double* partial, cudaStream_t s);
template <typename T> cudaError_t dot_partial(const void* u, const void* v, size_t ncomplex, double* partial, cudaStream_t s);
cudaError_t final_sum(const double* partial, int n, int nvals, double* result, cudaStream_t s);
// CG bookkeeping kernels (single CTA; partial sums reduced in fixed order)
cudaError_t cg_init_state(CgState* st, const double* partial, int n, double tol, cudaStream_t s);
cudaError_t cg_reduce_alpha(CgState* st, const double* partial, int n, cudaStream_t s);
cudaError_t cg_reduce_beta(CgState* st, const double* partial, int n, cudaStream_t s);
// the same for nrhs columns in lock step (partial sums of column c at partial + c * n; flags: {all finished, ticket})
cudaError_t cg_init_state_multi(CgState* st, int nrhs, const double* partial, int n, double tol, int* flags, cudaStream_t s);
cudaError_t cg_reduce_alpha_multi(CgState* st, int nrhs, const double* partial, int n, int* flags, cudaStream_t s);
cudaError_t cg_reduce_beta_multi(CgState* st, int nrhs, const double* partial, int n, cudaStream_t s);
template <typename T>
cudaError_t cg_update_xp_multi(const CgState* st, int nrhs, void* x, void* p, const void* r, size_t n, size_t stride, cudaStream_t s);
// x += alpha p ; p = r + beta p   (skips according to st->done)
template <typename T> cudaError_t cg_update_xp(const CgState* st, void* x, void* p, const void* r, size_t ncomplex, cudaStream_t s);
// r -= st->alpha * q, |r|^2 partials (reduce_blocks(ncomplex) of them); skipped once st->done is set
template <typename T> cudaError_t cg_raxpy_norm(const CgState* st, const void* q, void* r, size_t ncomplex, double* partial, cudaStream_t s);
// y = a*x + y  /  y = x + a*y  / copy / zero with host scalar a
template <typename T> cudaError_t axpy(double a, const void* x, void* y, size_t ncomplex, cudaStream_t s);
template <typename T> cudaError_t xmy(const void* x, const void* y, void* z, size_t ncomplex, cudaStream_t s);  // z = x - y
cudaError_t add_f32_to_f64(const void* e32, void* x64, size_t ncomplex, cudaStream_t s);                          // x += e
// NEXT-2: C(x4) of ncol spinor fields stored back to back; partial >= ntiles*b3 doubles, C_dev >= L4 doubles
template <typename T> cudaError_t correlator_ps(const Geom& g, const void* cols, int ncol, double* partial, double* C_dev, cudaStream_t s);
// zero the frozen time slices of a spinor (D7: the solve lives on the interior)
template <typename T> cudaError_t mask_frozen(const Geom& g, void* psi, cudaStream_t s);

}  // namespace lqcd
