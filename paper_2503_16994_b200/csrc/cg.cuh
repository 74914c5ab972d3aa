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
  cudaError_t hop_xpay(const void* in, const void* self, void* out, double k, int parity, cudaStream_t s) const;
};

struct CgVectors {
  void* r;
  void* p;
  void* t;
  double* partial;   // >= max(ntiles, 2*reduce_blocks) doubles
  CgState* state;    // device
};

// Solve M^+ M x = bprime from x = 0 (bprime = M^+ b already formed).  Leaves the final state in *host_state.
template <typename T>
cudaError_t cg_normal(const Op<T>& M, const void* bprime, void* x, const CgVectors& v, double tol, int maxiter,
                      int check_every, CgState* host_state, cudaStream_t s);

template <typename T>
cudaError_t device_norm2(const void* vec, size_t n, double* partial, double* scratch_dev, double* host, cudaStream_t s);

}  // namespace lqcd
