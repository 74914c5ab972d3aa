// noalloc.cu -- lqcd_correlator_ps_static: the pseudoscalar two-point function (lqcd_correlator_ps, SURVEY.md 8(f)
// NEXT-2) for callers that can neither allocate device memory nor hand over a workspace: code under
// CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The scratch the two kernels need -- one
// partial sum per tile and local time coordinate, then the L4 sums -- lives in a file-scope array in device memory of
// a fixed, stated size; every GPU that loads the library holds it until the process exits.
//
// This call allocates nothing: no cudaMalloc / cudaFree, no allocating library routine, no geometry or context object
// of its own.  It launches the same two kernels as lqcd_correlator_ps (blas.cu: corr_ps_tile_kernel,
// corr_ps_final_kernel), so the result is bit-identical to the existing path.
//
// Sharing: every call on a device uses the same array.  Nothing in it has to start at zero -- the tile kernel writes
// every partial sum the final kernel reads, and the final kernel writes every C(x4) that is copied out, in the same
// call -- so no clearing is needed and the previous call's contents are simply overwritten; but two calls that overlap
// on the GPU (different streams, or different host threads) race on it.  Serialise them.
#include <stdio.h>

#include <mutex>

#include "kernels.cuh"

namespace lqcd {

// 196608 doubles = 1.5 MiB per GPU: enough for ntiles * b4 + L4 <= 196608, e.g. 48^3 x 96 (165 984 with 4^4 tiles);
// 64^3 x 128 (524 416) is rejected.
enum { CORR_STATIC_MAX = LQCD_CORRELATOR_STATIC_MAX_DOUBLES };
static __device__ __align__(256) double g_corr_scratch[CORR_STATIC_MAX];

// Keeps the array alive in the device image whatever the compiler thinks of a variable that only host code names, and
// is the one place where device code names it directly.
__global__ void corr_static_touch_kernel(double* where) {
  if (where == nullptr) g_corr_scratch[0] = 0.0;
}

// In host code `g_corr_scratch` is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, once per device, with that device current.
static cudaError_t corr_static_ptr(int dev, double** out) {
  enum { MAX_DEV = 64 };
  static std::mutex mu;
  static double* ptr[MAX_DEV] = {};
  if (dev < 0 || dev >= MAX_DEV) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(mu);
  if (ptr[dev] == nullptr) {
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_corr_scratch);
    if (e != cudaSuccess) return e;
    if (p == nullptr) return cudaErrorInvalidSymbol;
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return cudaSuccess;
}

}  // namespace lqcd

using namespace lqcd;

extern "C" lqcd_status lqcd_correlator_ps_static(const lqcd_geom* h, const void* columns, int ncol, lqcd_prec prec,
                                                 double* C_host, void* stream) {
  if (!h || !columns || !C_host) {
    set_error("lqcd_correlator_ps_static: NULL argument");
    return LQCD_EINVAL;
  }
  if ((prec != LQCD_F64 && prec != LQCD_F32) || ncol < 1 || ncol > 4096) {
    set_error("lqcd_correlator_ps_static: bad precision or column count");
    return LQCD_EINVAL;
  }
  const Geom& g = h->g;
  const size_t npartial = (size_t)g.ntiles * g.b[3];
  const size_t need = npartial + (size_t)g.L[3];
  if (need > (size_t)CORR_STATIC_MAX) {
    set_error("lqcd_correlator_ps_static: this lattice needs %zu doubles of scratch (tiles x tile extent in time + L4), "
              "the static scratch holds %d; use lqcd_correlator_ps with a caller-owned workspace",
              need, (int)CORR_STATIC_MAX);
    return LQCD_EINVAL;
  }
  int prev = -1;
  const int dev = h->desc.device;
  bool switched = false;
  if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  lqcd_status st = LQCD_OK;
  double* scratch = nullptr;
  cudaStream_t s = (cudaStream_t)stream;
  do {
    if (!cuda_ok(corr_static_ptr(dev, &scratch), "lqcd_correlator_ps_static: cudaGetSymbolAddress")) { st = LQCD_ECUDA; break; }
    double* C_dev = scratch + npartial;
    const cudaError_t e = prec == LQCD_F64 ? correlator_ps<double>(g, columns, ncol, scratch, C_dev, s)
                                           : correlator_ps<float>(g, columns, ncol, scratch, C_dev, s);
    if (!cuda_ok(e, "lqcd_correlator_ps_static: correlator kernel")) { st = LQCD_ECUDA; break; }
    if (!cuda_ok(cudaMemcpyAsync(C_host, C_dev, (size_t)g.L[3] * sizeof(double), cudaMemcpyDeviceToHost, s),
                 "lqcd_correlator_ps_static: memcpy")) { st = LQCD_ECUDA; break; }
    if (!cuda_ok(cudaStreamSynchronize(s), "lqcd_correlator_ps_static: sync")) { st = LQCD_ECUDA; break; }
  } while (0);
  if (switched) cudaSetDevice(prev);
  return st;
}
