// cg.cu -- CG! on the normal equations and the solves built on it (algorithm
// and stopping rule: SURVEY.md 8(c) "Algorithm CG", R11; even-odd: D8; mixed precision: defect correction).
//
// One CG iteration is three big kernels:  t = M p with |t|^2 fused (EPI_STORE_NORM);  r -= alpha M^+ t with
// |r|^2 fused, M^+ t never written (EPI_AXPY_NORM);  x += alpha p, p = r + beta p.  Two single-CTA kernels
// turn the per-CTA partial sums into alpha, beta and the convergence flag on the device; the host reads
// the 80-byte state back only every `check_every` iterations, and all kernels become no-ops once the flag
// is set, so the iteration count is exact.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include "cg.cuh"

namespace lqcd {

template <typename T> using T2 = typename vec2<T>::type;

#define CK(e) do { cudaError_t _e = (e); if (_e != cudaSuccess) return _e; } while (0)

template <typename T>
cudaError_t Op<T>::apply(const void* in, void* out, bool dagger, int epi, void* r, const double* alpha, double* partial,
                         const int* skip, cudaStream_t s) const {
  DwArgs<T> a;
  memset(&a, 0, sizeof(a));
  a.U = (const T2<T>*)U;
  a.r = (T2<T>*)r;
  a.alpha = alpha;
  a.partial = partial;
  a.skip = skip;
  a.has_theta = geom->has_theta;
  for (int d = 0; d < 4; d++) a.theta[d] = cx<T>((T)geom->th_re[d], (T)geom->th_im[d]);
  a.dagger = dagger ? 1 : 0;
  if (!eo) {
    a.A = (const T2<T>*)A;
    a.in = (const T2<T>*)in;
    a.self = (const T2<T>*)in;
    a.out = (T2<T>*)out;
    a.k = (T)kappa;
    a.tm = (T)(2.0 * kappa * (dagger ? -mu : mu));
    a.parity = -1;
    a.epi = epi;
    return launch_dw<T>(geom->g, a, recon, A ? DIAG_PRE : DIAG_ONE, s);
  }
  // D^ = A_ee - kappa^2 H_eo A_oo^{-1} H_oe  (D8): tmp_o = A_oo^{-1} H_oe in_e ; out_e = A_ee in_e - kappa^2 H_eo tmp_o
  a.A = (const T2<T>*)Ainv;
  a.in = (const T2<T>*)in;
  a.self = (const T2<T>*)in;
  a.out = (T2<T>*)tmp;
  a.k = (T)0;
  a.parity = 1;
  a.epi = EPI_STORE;
  CK(launch_dw<T>(geom->g, a, recon, DIAG_POST, s));
  a.A = (const T2<T>*)A;
  a.in = (const T2<T>*)tmp;
  a.self = (const T2<T>*)in;
  a.out = (T2<T>*)out;
  a.k = (T)(kappa * kappa);
  a.parity = 0;
  a.epi = epi;
  return launch_dw<T>(geom->g, a, recon, DIAG_PRE, s);
}

template <typename T>
cudaError_t Op<T>::apply_multi(const void* in, void* out, int nrhs, bool dagger, cudaStream_t s) const {
  DwArgs<T> a;
  memset(&a, 0, sizeof(a));
  a.U = (const T2<T>*)U;
  a.A = (const T2<T>*)A;
  a.in = (const T2<T>*)in;
  a.self = (const T2<T>*)in;
  a.out = (T2<T>*)out;
  a.k = (T)kappa;
  a.tm = (T)(2.0 * kappa * (dagger ? -mu : mu));
  a.has_theta = geom->has_theta;
  for (int d = 0; d < 4; d++) a.theta[d] = cx<T>((T)geom->th_re[d], (T)geom->th_im[d]);
  a.dagger = dagger ? 1 : 0;
  a.parity = -1;
  a.epi = EPI_STORE;
  a.nrhs = nrhs;
  a.rhs_stride = (long long)2 * geom->g.Vh * 12;
  return launch_dw<T>(geom->g, a, recon, A ? DIAG_PRE : DIAG_ONE, s);
}

template <typename T>
bool Op<T>::multi_fused_ok() const {
  return !eo && dw_uses_pipe<T>(geom->g, recon, A ? DIAG_PRE : DIAG_ONE, -1);
}

template <typename T>
cudaError_t Op<T>::apply_multi_epi(const void* in, void* out, int nrhs, bool dagger, int epi, void* r, const double* alpha,
                                   int alpha_stride, double* partial, const int* skip, cudaStream_t s) const {
  DwArgs<T> a;
  memset(&a, 0, sizeof(a));
  a.U = (const T2<T>*)U;
  a.A = (const T2<T>*)A;
  a.in = (const T2<T>*)in;
  a.self = (const T2<T>*)in;
  a.out = (T2<T>*)out;
  a.r = (T2<T>*)r;
  a.alpha = alpha;
  a.alpha_stride = alpha_stride;
  a.partial = partial;
  a.skip = skip;
  a.k = (T)kappa;
  a.tm = (T)(2.0 * kappa * (dagger ? -mu : mu));
  a.has_theta = geom->has_theta;
  for (int d = 0; d < 4; d++) a.theta[d] = cx<T>((T)geom->th_re[d], (T)geom->th_im[d]);
  a.dagger = dagger ? 1 : 0;
  a.parity = -1;
  a.epi = epi;
  a.nrhs = nrhs;
  a.rhs_stride = (long long)2 * geom->g.Vh * 12;
  return launch_dw<T>(geom->g, a, recon, A ? DIAG_PRE : DIAG_ONE, s);
}

// out(parity) = self - k * H in   (no clover), used by the even-odd source preparation / reconstruction
template <typename T>
cudaError_t Op<T>::hop_xpay(const void* in, const void* self, void* out, double k, int parity, cudaStream_t s) const {
  DwArgs<T> a;
  memset(&a, 0, sizeof(a));
  a.U = (const T2<T>*)U;
  a.in = (const T2<T>*)in;
  a.self = (const T2<T>*)self;
  a.out = (T2<T>*)out;
  a.k = (T)k;
  a.has_theta = geom->has_theta;
  for (int d = 0; d < 4; d++) a.theta[d] = cx<T>((T)geom->th_re[d], (T)geom->th_im[d]);
  a.parity = parity;
  a.epi = EPI_STORE;
  return launch_dw<T>(geom->g, a, recon, DIAG_ONE, s);
}

template <typename T>
cudaError_t cg_normal(const Op<T>& M, const void* bprime, void* x, const CgVectors& v, double tol, int maxiter,
                      int check_every, CgState* host_state, cudaStream_t s) {
  const size_t n = M.ncomplex();
  const size_t bytes = n * sizeof(T2<T>);
  const int nt = M.eo ? dw_num_partials<T>(M.geom->g, M.recon, DIAG_PRE, 0)
                      : dw_num_partials<T>(M.geom->g, M.recon, M.A ? DIAG_PRE : DIAG_ONE, -1);
  CK(cudaMemsetAsync(x, 0, bytes, s));
  CK(cudaMemcpyAsync(v.r, bprime, bytes, cudaMemcpyDeviceToDevice, s));
  CK(cudaMemcpyAsync(v.p, bprime, bytes, cudaMemcpyDeviceToDevice, s));
  CK(norm2_partial<T>(v.r, n, v.partial, s));
  CK(cg_init_state(v.state, v.partial, reduce_blocks(n), tol, s));
  if (check_every < 1) check_every = 1;
  auto iterations = [&](int count, cudaStream_t st) -> cudaError_t {
    for (int it = 0; it < count; it++) {
      CK(M.apply(v.p, v.t, false, EPI_STORE_NORM, nullptr, nullptr, v.partial, &v.state->done, st));
      CK(cg_reduce_alpha(v.state, v.partial, nt, st));
      CK(M.apply(v.t, nullptr, true, EPI_AXPY_NORM, v.r, &v.state->alpha, v.partial, &v.state->done, st));
      CK(cg_reduce_beta(v.state, v.partial, nt, st));
      CK(cg_update_xp<T>(v.state, x, v.p, v.r, n, st));
    }
    return cudaSuccess;
  };
  // The check_every iterations between two looks at the state are captured once as a CUDA graph and replayed, which
  // closes the launch gaps between the five to seven dependent kernels of an iteration (1-3 % of a solve on the
  // 24^3 x 48 and 32^3 x 64 lattices; LQCD_CG_GRAPH=0 launches them one by one; so does any failure to capture).
  // Capture needs a real stream: on the legacy default stream the graph runs on a blocking stream of its own, which
  // the legacy stream's implicit synchronisation keeps in order with the caller's work.
  static const bool want_graph = [] { const char* e = getenv("LQCD_CG_GRAPH"); return !(e && e[0] == '0'); }();
  cudaGraphExec_t gexec = nullptr;
  cudaStream_t gs = s, own = nullptr;
  // the captured launches keep their tile-scheduler counters for every replay: give them this solve's own
  struct PoolGuard {
    explicit PoolGuard(unsigned int* p) { if (p) dw_set_sched_pool(p, SCHED_POOL_PAIRS); }
    ~PoolGuard() { dw_set_sched_pool(nullptr, 0); }
  } pool_guard(v.sched_pool);
  if (want_graph && maxiter >= check_every) {
    if (s == nullptr) { CK(cudaStreamCreate(&own)); gs = own; }
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamBeginCapture(gs, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
      const cudaError_t e1 = iterations(check_every, gs);
      const cudaError_t e2 = cudaStreamEndCapture(gs, &graph);
      e = e1 != cudaSuccess ? e1 : e2;
    }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&gexec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (e != cudaSuccess) { gexec = nullptr; (void)cudaGetLastError(); }   // fall back to plain launches
  }
  int launched = 0;
  cudaError_t rc = cudaSuccess;
  for (;;) {
    rc = cudaMemcpyAsync(host_state, v.state, sizeof(CgState), cudaMemcpyDeviceToHost, s);
    if (rc != cudaSuccess) break;
    rc = cudaStreamSynchronize(s);
    if (rc != cudaSuccess) break;
    if (host_state->done || launched >= maxiter) break;
    int batch = check_every;
    if (launched + batch > maxiter) batch = maxiter - launched;
    if (gexec && batch == check_every) {
      rc = cudaGraphLaunch(gexec, gs);
      if (rc == cudaSuccess && gs != s) rc = cudaStreamSynchronize(gs);
    } else {
      rc = iterations(batch, s);
    }
    if (rc != cudaSuccess) break;
    launched += batch;
  }
  if (gexec) cudaGraphExecDestroy(gexec);
  if (own) cudaStreamDestroy(own);
  return rc;
}

template <typename T>
cudaError_t cg_normal_multi(const Op<T>& M, int nrhs, const void* bprime, void* x, void* r, void* p, void* t, double* partial,
                            CgState* states, int* flags, double tol, int maxiter, int check_every, CgState* host_states,
                            cudaStream_t s) {
  const size_t n = M.ncomplex();
  const size_t bytes = (size_t)nrhs * n * sizeof(T2<T>);
  const int nt = M.geom->g.ntiles;
  const int np = reduce_blocks(n);
  CK(cudaMemsetAsync(x, 0, bytes, s));
  CK(cudaMemcpyAsync(r, bprime, bytes, cudaMemcpyDeviceToDevice, s));
  CK(cudaMemcpyAsync(p, bprime, bytes, cudaMemcpyDeviceToDevice, s));
  for (int c = 0; c < nrhs; c++) CK(norm2_partial<T>((const T2<T>*)r + (size_t)c * n, n, partial + (size_t)c * np, s));
  CK(cg_init_state_multi(states, nrhs, partial, np, tol, flags, s));
  if (check_every < 1) check_every = 1;
  const int astride = (int)(sizeof(CgState) / sizeof(double));
  int launched = 0;
  for (;;) {
    CK(cudaMemcpyAsync(host_states, states, (size_t)nrhs * sizeof(CgState), cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    bool all = true;
    for (int c = 0; c < nrhs; c++) all = all && host_states[c].done != 0;
    if (all || launched >= maxiter) break;
    int batch = check_every;
    if (launched + batch > maxiter) batch = maxiter - launched;
    for (int it = 0; it < batch; it++) {
      CK(M.apply_multi_epi(p, t, nrhs, false, EPI_STORE_NORM, nullptr, nullptr, 0, partial, flags, s));
      CK(cg_reduce_alpha_multi(states, nrhs, partial, nt, flags, s));
      CK(M.apply_multi_epi(t, nullptr, nrhs, true, EPI_AXPY_NORM, r, &states->alpha, astride, partial, flags, s));
      CK(cg_reduce_beta_multi(states, nrhs, partial, nt, s));
      CK(cg_update_xp_multi<T>(states, nrhs, x, p, r, n, n, s));
    }
    launched += batch;
  }
  return cudaSuccess;
}

template <typename T>
cudaError_t device_norm2(const void* vec, size_t n, double* partial, double* scratch_dev, double* host, cudaStream_t s) {
  CK(norm2_partial<T>(vec, n, partial, s));
  CK(final_sum(partial, reduce_blocks(n), 1, scratch_dev, s));
  CK(cudaMemcpyAsync(host, scratch_dev, sizeof(double), cudaMemcpyDeviceToHost, s));
  return cudaStreamSynchronize(s);
}

template struct Op<double>;
template struct Op<float>;
template cudaError_t cg_normal<double>(const Op<double>&, const void*, void*, const CgVectors&, double, int, int, CgState*, cudaStream_t);
template cudaError_t cg_normal<float>(const Op<float>&, const void*, void*, const CgVectors&, double, int, int, CgState*, cudaStream_t);
template cudaError_t cg_normal_multi<double>(const Op<double>&, int, const void*, void*, void*, void*, void*, double*, CgState*, int*, double, int, int, CgState*, cudaStream_t);
template cudaError_t cg_normal_multi<float>(const Op<float>&, int, const void*, void*, void*, void*, void*, double*, CgState*, int*, double, int, int, CgState*, cudaStream_t);
template cudaError_t device_norm2<double>(const void*, size_t, double*, double*, double*, cudaStream_t);
template cudaError_t device_norm2<float>(const void*, size_t, double*, double*, double*, cudaStream_t);

}  // namespace lqcd
