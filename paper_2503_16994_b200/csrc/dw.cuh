// dw.cuh -- arguments of the stencil kernel (dw.cu) and of the BLAS-1 / reduction kernels (blas.cu).
#pragma once
#include "lqcd_internal.cuh"

namespace lqcd {

enum { DIAG_ONE = 0, DIAG_PRE = 1, DIAG_POST = 2 };
enum { EPI_STORE = 0, EPI_STORE_NORM = 1, EPI_AXPY_NORM = 2 };

template <typename T>
struct DwArgs {
  const typename vec2<T>::type* U;     // internal gauge field
  const typename vec2<T>::type* A;     // packed clover blocks (DIAG_PRE: A, DIAG_POST: A^{-1}); unused for DIAG_ONE
  const typename vec2<T>::type* in;    // field whose neighbours are hopped (base of a full field)
  const typename vec2<T>::type* self;  // field supplying the site-diagonal term (base of a full field)
  typename vec2<T>::type* out;         // base of a full field (only the output parity is written)
  typename vec2<T>::type* r;           // EPI_AXPY_NORM: r -= alpha * result
  const double* alpha;                 // device scalar
  double* partial;                     // one partial sum per CTA
  const int* skip;                     // device flag: if non-NULL and *skip != 0 the kernel does nothing
  T k;                                 // kappa (or kappa^2 for the even-odd operator)
  T tm;                                // twisted mass term: + i tm gamma5 self added to the result (2 kappa mu; -2 kappa mu
                                       // for D^+); 0 = absent.  Full-lattice operator only.
  cx<T> theta[4];
  int has_theta;
  int dagger;
  int parity;                          // -1: both parities; 0/1: only this output parity
  int epi;
  unsigned int* sched;                 // pipeline kernel: {next tile, finished CTAs} of its tile scheduler (NULL: static)
  int nrhs;                            // > 1: in / out are arrays of nrhs spinor fields rhs_stride complex numbers apart
  long long rhs_stride;                //      (several right-hand sides share the links and the clover term)
  int alpha_stride;                    //      in doubles: right-hand side n takes its alpha from alpha[n * alpha_stride] (0: one alpha for all)
  int nsplit;                          //      pipeline kernel: a tile's right-hand sides are shared out over nsplit work units (set by launch_pipe)
};

// number of per-CTA partial sums an EPI_*_NORM launch with these arguments writes to DwArgs::partial
template <typename T>
int dw_num_partials(const Geom& g, int recon, int diag, int parity);

// does launch_dw run these arguments on the pipeline kernel (dw_pipe_kernel)?  Only then may nrhs > 1 be combined with
// a reducing epilogue (partial[n * ntiles + tile], alpha[n * alpha_stride])
template <typename T>
bool dw_uses_pipe(const Geom& g, int recon, int diag, int parity);

// one-line description of the kernel launch_dw would use (lqcd_dw_plan); dw_set_mode: lqcd_set_option("dw_mode")
template <typename T>
void dw_describe(const Geom& g, int recon, int diag, int parity, char* buf, int len);
bool dw_set_mode(const char* name);
bool dw_set_pipe_grid(int n);
// Tile-scheduler counters for the pipeline-kernel launches of the CALLING THREAD: while set (base != NULL), launches
// take their {next tile, finished CTAs} pair from these npairs zeroed pairs (round robin) instead of the geometry's
// pool.  A solver that replays its launches as a CUDA graph sets this to counters of its own (in its workspace), so
// that two solves on one geometry running on different streams can never share a counter.
void dw_set_sched_pool(unsigned int* base, int npairs);

template <typename T>
cudaError_t launch_dw(const Geom& g, const DwArgs<T>& a, int recon, int diag, cudaStream_t s);
// out(x) = B(x) in(x) on sites of `parity` (-1: all), zero on frozen slices; B = packed 6x6 blocks
template <typename T>
cudaError_t launch_diag(const Geom& g, const void* B, const void* in, void* out, int parity, cudaStream_t s);

}  // namespace lqcd
