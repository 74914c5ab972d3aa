// cg.cuh -- operator abstraction (full D or even-odd D^) and the CG loop on the normal equations.
#pragma once
#include "kernels.cuh"

namespace lqcd {

template <typename T>
struct Op {
  const lqcd_geom* geom;
  const void* U;
  const void* A;      // packed clover blocks or NULL (full operator only)
  const void* Ainv;   // even-odd only
  void* tmp;          // even-odd only: one full spinor field (its odd half is used)
  double kappa;
  double mu = 0.0;    // twisted mass (full operator only)
  int recon;
  bool eo;
  size_t ncomplex() const { return (size_t)(eo ? 1 : 2) * geom->g.Vh * 12; }
  // out = M in or M^+ in, with the fused epilogue `epi` (dw.cuh)
  cudaError_t apply(const void* in, void* out, bool dagger, int epi, void* r, const double* alpha, double* partial,
                    const int* skip, cudaStream_t s) const;
  // full operator on nrhs spinor fields stored back to back (in[n], out[n] one full field apart), EPI_STORE
  cudaError_t apply_multi(const void* in, void* out, int nrhs, bool dagger, cudaStream_t s) const;
  // the same with a fused epilogue per right-hand side (pipeline kernel only: check multi_fused_ok() first):
  // partial[n * ntiles + tile], alpha of column n at alpha[n * alpha_stride], r an array like in / out
  cudaError_t apply_multi_epi(const void* in, void* out, int nrhs, bool dagger, int epi, void* r, const double* alpha,
                              int alpha_stride, double* partial, const int* skip, cudaStream_t s) const;
  bool multi_fused_ok() const;
  cudaError_t hop_xpay(const void* in, const void* self, void* out, double k, int parity, cudaStream_t s) const;
};

struct CgVectors {
  void* r;
  void* p;
  void* t;
  double* partial;   // >= max(ntiles, 2*reduce_blocks) doubles
  CgState* state;    // device
  unsigned int* sched_pool = nullptr;   // device, zeroed: SCHED_POOL_PAIRS pairs of tile-scheduler counters of this solve
};
enum { SCHED_POOL_PAIRS = 128 };

// Solve M^+ M x = bprime from x = 0 (bprime = M^+ b already formed).  Leaves the final state in *host_state.
template <typename T>
cudaError_t cg_normal(const Op<T>& M, const void* bprime, void* x, const CgVectors& v, double tol, int maxiter,
                      int check_every, CgState* host_state, cudaStream_t s);

// nrhs independent solves M^+ M x_n = bprime_n in lock step (full operator, pipeline kernel): every stencil pass takes
// all columns (links and clover blocks shared, lqcd_dw_apply_multi), scalars and convergence flags per column on the
// device.  r, p, t, x, bprime: nrhs fields back to back.  states: nrhs CgState on the device, host_states: nrhs on the
// host (final states).  partial: >= nrhs * ntiles doubles; flags: 2 ints on the device (all-done flag, ticket counter).
template <typename T>
cudaError_t cg_normal_multi(const Op<T>& M, int nrhs, const void* bprime, void* x, void* r, void* p, void* t, double* partial,
                            CgState* states, int* flags, double tol, int maxiter, int check_every, CgState* host_states,
                            cudaStream_t s);

template <typename T>
cudaError_t device_norm2(const void* vec, size_t n, double* partial, double* scratch_dev, double* host, cudaStream_t s);

}  // namespace lqcd
