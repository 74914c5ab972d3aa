// blas.cu -- BLAS-1 and reductions of the CG driver that are not fused into the stencil
// (SURVEY.md 8(a) row a6): warp-shuffle trees, one partial per CTA, fixed-order final pass in a single
// CTA (bit-reproducible run to run); fp64 accumulation in both precisions.  CG scalars stay on the device.
#include "kernels.cuh"

namespace lqcd {

template <typename T> using T2 = typename vec2<T>::type;

static const int RB_THREADS = 256;
// SMs of the device the geometry was created on (lqcd_geom_create); 148 = B200 until a geometry exists
static int g_reduce_sms = 148;
void set_reduce_sm_count(int sms) { if (sms > 0) g_reduce_sms = sms; }
int reduce_blocks_max() { return g_reduce_sms * 8; }
int reduce_blocks(size_t ncomplex) {
  size_t b = (ncomplex + (size_t)RB_THREADS * 8 - 1) / ((size_t)RB_THREADS * 8);
  if (b < 1) b = 1;
  if (b > (size_t)reduce_blocks_max()) b = (size_t)reduce_blocks_max();
  return (int)b;
}

__device__ __forceinline__ double block_sum(double v, double* s_red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
  __syncthreads();
  double s = 0;
  if (threadIdx.x == 0) {
    const int nw = (blockDim.x + 31) >> 5;
    for (int w = 0; w < nw; w++) s += s_red[w];
  }
  return s;  // valid in thread 0
}

template <typename T>
__global__ void norm2_kernel(const T2<T>* __restrict__ v, size_t n, double* partial) {
  __shared__ double s_red[32];
  double acc = 0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    T2<T> a = v[i];
    acc += (double)a.x * (double)a.x + (double)a.y * (double)a.y;
  }
  double s = block_sum(acc, s_red);
  if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

template <typename T>
__global__ void dot_kernel(const T2<T>* __restrict__ u, const T2<T>* __restrict__ v, size_t n, double* partial) {
  __shared__ double s_red[32];
  double re = 0, im = 0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    T2<T> a = u[i], b = v[i];  // conj(a) * b
    re += (double)a.x * (double)b.x + (double)a.y * (double)b.y;
    im += (double)a.x * (double)b.y - (double)a.y * (double)b.x;
  }
  double s = block_sum(re, s_red);
  if (threadIdx.x == 0) partial[blockIdx.x] = s;
  s = block_sum(im, s_red);
  if (threadIdx.x == 0) partial[gridDim.x + blockIdx.x] = s;
}

// fixed-order sum of partial[0..n): thread t adds elements t, t+256, ... then a fixed tree
__device__ double ordered_sum(const double* partial, int n, double* s_red) {
  double acc = 0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) acc += partial[i];
  return block_sum(acc, s_red);
}

__global__ void final_sum_kernel(const double* partial, int n, int nvals, double* result) {
  __shared__ double s_red[32];
  for (int k = 0; k < nvals; k++) {
    double s = ordered_sum(partial + (size_t)k * n, n, s_red);
    if (threadIdx.x == 0) result[k] = s;
  }
}

__global__ void cg_init_kernel(CgState* st, const double* partial, int n, double tol) {
  __shared__ double s_red[32];
  double s = ordered_sum(partial, n, s_red);
  if (threadIdx.x == 0) {
    st->rho = s; st->rho0 = s; st->alpha = 0; st->beta = 0; st->tt = 0; st->rho_new = s;
    st->tol2 = tol * tol;
    st->iters = 0; st->breakdown = 0;
    st->done = (s == 0.0) ? 1 : 0;
    if (!(s == s)) { st->done = 1; st->breakdown = 1; }
  }
}

// after t = M p:  alpha = rho / |t|^2
__global__ void cg_alpha_kernel(CgState* st, const double* partial, int n) {
  __shared__ double s_red[32];
  if (st->done == 2) { if (threadIdx.x == 0) st->done = 1; return; }
  if (st->done) return;
  double s = ordered_sum(partial, n, s_red);
  if (threadIdx.x == 0) {
    st->tt = s;
    if (!(s > 0.0)) { st->breakdown = 1; st->done = 1; st->alpha = 0; }
    else st->alpha = st->rho / s;
  }
}

// after r -= alpha M^+ t:  rho' = |r|^2, convergence test, beta = rho'/rho
__global__ void cg_beta_kernel(CgState* st, const double* partial, int n) {
  __shared__ double s_red[32];
  if (st->done) return;
  double s = ordered_sum(partial, n, s_red);
  if (threadIdx.x == 0) {
    st->rho_new = s;
    st->iters += 1;
    if (!(s == s)) { st->breakdown = 1; st->done = 2; st->alpha = 0; }
    else if (s <= st->tol2 * st->rho0) st->done = 2;  // x += alpha p still pending
    st->beta = s / st->rho;
    st->rho = s;
  }
}

// ---- the same bookkeeping for nrhs solves in lock step (cg_normal_multi): CTA c serves column c -----------------
// flags[0]: all columns finished (the stencil launches then return at once), flags[1]: ticket counter of the alpha kernel
__global__ void cg_init_multi_kernel(CgState* st, const double* partial, int n, double tol, int* flags) {
  __shared__ double s_red[32];
  st += blockIdx.x;
  double s = ordered_sum(partial + (size_t)blockIdx.x * n, n, s_red);
  if (threadIdx.x == 0) {
    st->rho = s; st->rho0 = s; st->alpha = 0; st->beta = 0; st->tt = 0; st->rho_new = s;
    st->tol2 = tol * tol;
    st->iters = 0; st->breakdown = 0;
    st->done = (s == 0.0) ? 1 : 0;
    if (!(s == s)) { st->done = 1; st->breakdown = 1; }
    if (blockIdx.x == 0) { flags[0] = 0; flags[1] = 0; }
  }
}
// A finished column keeps taking part in the stencil passes (they are per tile, not per column) with alpha = 0, which
// leaves its r alone; its x and p are no longer touched.  The last CTA to arrive sets the all-finished flag.
__global__ void cg_alpha_multi_kernel(CgState* st0, const double* partial, int n, int* flags) {
  __shared__ double s_red[32];
  CgState* st = st0 + blockIdx.x;
  if (st->done == 2) { if (threadIdx.x == 0) st->done = 1; }
  __syncthreads();
  if (st->done) {
    if (threadIdx.x == 0) st->alpha = 0;
  } else {
    double s = ordered_sum(partial + (size_t)blockIdx.x * n, n, s_red);
    if (threadIdx.x == 0) {
      st->tt = s;
      if (!(s > 0.0)) { st->breakdown = 1; st->done = 1; st->alpha = 0; }
      else st->alpha = st->rho / s;
    }
  }
  if (threadIdx.x == 0) {
    __threadfence();
    if (atomicAdd(flags + 1, 1) == (int)gridDim.x - 1) {
      __threadfence();
      int all = 1;
      for (unsigned c = 0; c < gridDim.x; c++) all &= (((volatile CgState*)st0)[c].done == 1);
      flags[0] = all;
      flags[1] = 0;
    }
  }
}
__global__ void cg_beta_multi_kernel(CgState* st, const double* partial, int n) {
  __shared__ double s_red[32];
  st += blockIdx.x;
  if (st->done) return;
  double s = ordered_sum(partial + (size_t)blockIdx.x * n, n, s_red);
  if (threadIdx.x == 0) {
    st->rho_new = s;
    st->iters += 1;
    if (!(s == s)) { st->breakdown = 1; st->done = 2; st->alpha = 0; }
    else if (s <= st->tol2 * st->rho0) st->done = 2;  // x += alpha p still pending
    st->beta = s / st->rho;
    st->rho = s;
  }
}
// blockIdx.y: column; x, p, r: arrays of fields `stride` complex numbers apart
template <typename T>
__global__ void cg_update_xp_multi_kernel(const CgState* st, T2<T>* x, T2<T>* p, const T2<T>* __restrict__ r, size_t n, size_t stride) {
  st += blockIdx.y;
  const int done = st->done;
  if (done == 1) return;
  x += blockIdx.y * stride; p += blockIdx.y * stride; r += blockIdx.y * stride;
  const T al = (T)st->alpha, be = (T)st->beta;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    T2<T> xv = x[i], pv = p[i];
    xv.x = fma(al, pv.x, xv.x);
    xv.y = fma(al, pv.y, xv.y);
    x[i] = xv;
    if (done == 0) {
      T2<T> rv = r[i];
      pv.x = fma(be, pv.x, rv.x);
      pv.y = fma(be, pv.y, rv.y);
      p[i] = pv;
    }
  }
}

template <typename T>
__global__ void cg_update_xp_kernel(const CgState* st, T2<T>* x, T2<T>* p, const T2<T>* __restrict__ r, size_t n) {
  const int done = st->done;
  if (done == 1) return;
  const T al = (T)st->alpha, be = (T)st->beta;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    T2<T> xv = x[i], pv = p[i];
    xv.x = fma(al, pv.x, xv.x);
    xv.y = fma(al, pv.y, xv.y);
    x[i] = xv;
    if (done == 0) {
      T2<T> rv = r[i];
      pv.x = fma(be, pv.x, rv.x);
      pv.y = fma(be, pv.y, rv.y);
      p[i] = pv;
    }
  }
}

// r -= alpha q with alpha on the device, |r|^2 partial per CTA (the unfused form of EPI_AXPY_NORM, used by the slab
// solver, whose operator result is complete only after the face kernel); does nothing once st->done is set
template <typename T>
__global__ void cg_raxpy_norm_kernel(const CgState* st, const T2<T>* __restrict__ q, T2<T>* r, size_t n, double* partial) {
  __shared__ double s_red[32];
  if (st->done) return;
  const T al = (T)st->alpha;
  double acc = 0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    T2<T> qv = q[i], rv = r[i];
    rv.x = fma(-al, qv.x, rv.x);
    rv.y = fma(-al, qv.y, rv.y);
    r[i] = rv;
    acc += (double)rv.x * (double)rv.x + (double)rv.y * (double)rv.y;
  }
  double s = block_sum(acc, s_red);
  if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

template <typename T>
__global__ void axpy_kernel(T a, const T2<T>* __restrict__ x, T2<T>* y, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    T2<T> xv = x[i], yv = y[i];
    yv.x = fma(a, xv.x, yv.x);
    yv.y = fma(a, xv.y, yv.y);
    y[i] = yv;
  }
}
template <typename T>
__global__ void xmy_kernel(const T2<T>* __restrict__ x, const T2<T>* __restrict__ y, T2<T>* z, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    T2<T> xv = x[i], yv = y[i];
    xv.x -= yv.x; xv.y -= yv.y;
    z[i] = xv;
  }
}
__global__ void add32_kernel(const float2* __restrict__ e, double2* x, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    float2 ev = e[i];
    double2 xv = x[i];
    xv.x += (double)ev.x; xv.y += (double)ev.y;
    x[i] = xv;
  }
}

template <typename T>
__global__ void mask_frozen_kernel(const Geom g, T2<T>* psi) {
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 2 * g.Vh) return;
  int p = (int)(idx / g.Vh);
  long long rem = idx - (long long)p * g.Vh;
  int tile = (int)(rem / g.TV);
  int j = (int)(rem - (long long)tile * g.TV);
  int Tc[4], l[4];
  tile_coords(g, tile, Tc);
  local_coords(g, j, p, l);
  if (!frozen_slice(g, Tc[3] * g.b[3] + l[3])) return;
  T2<T> z; z.x = 0; z.y = 0;
  for (int c = 0; c < 12; c++) psi[field_offset(g, 12, p, tile, c, j)] = z;
}

static unsigned ew_blocks(size_t n) {
  size_t b = (n + 1023) / 1024;
  if (b < 1) b = 1;
  if (b > 148 * 16) b = 148 * 16;
  return (unsigned)b;
}

template <typename T> cudaError_t norm2_partial(const void* v, size_t n, double* partial, cudaStream_t s) {
  norm2_kernel<T><<<reduce_blocks(n), RB_THREADS, 0, s>>>((const T2<T>*)v, n, partial);
  count_launch();
  return cudaGetLastError();
}
template <typename T> cudaError_t dot_partial(const void* u, const void* v, size_t n, double* partial, cudaStream_t s) {
  dot_kernel<T><<<reduce_blocks(n), RB_THREADS, 0, s>>>((const T2<T>*)u, (const T2<T>*)v, n, partial);
  count_launch();
  return cudaGetLastError();
}
cudaError_t final_sum(const double* partial, int n, int nvals, double* result, cudaStream_t s) {
  final_sum_kernel<<<1, 1024, 0, s>>>(partial, n, nvals, result);
  count_launch();
  return cudaGetLastError();
}
cudaError_t cg_init_state(CgState* st, const double* partial, int n, double tol, cudaStream_t s) {
  cg_init_kernel<<<1, 1024, 0, s>>>(st, partial, n, tol);
  count_launch();
  return cudaGetLastError();
}
cudaError_t cg_reduce_alpha(CgState* st, const double* partial, int n, cudaStream_t s) {
  cg_alpha_kernel<<<1, 1024, 0, s>>>(st, partial, n);
  count_launch();
  return cudaGetLastError();
}
cudaError_t cg_reduce_beta(CgState* st, const double* partial, int n, cudaStream_t s) {
  cg_beta_kernel<<<1, 1024, 0, s>>>(st, partial, n);
  count_launch();
  return cudaGetLastError();
}
template <typename T> cudaError_t cg_update_xp(const CgState* st, void* x, void* p, const void* r, size_t n, cudaStream_t s) {
  cg_update_xp_kernel<T><<<ew_blocks(n), 256, 0, s>>>(st, (T2<T>*)x, (T2<T>*)p, (const T2<T>*)r, n);
  count_launch();
  return cudaGetLastError();
}
cudaError_t cg_init_state_multi(CgState* st, int nrhs, const double* partial, int n, double tol, int* flags, cudaStream_t s) {
  cg_init_multi_kernel<<<nrhs, 1024, 0, s>>>(st, partial, n, tol, flags);
  count_launch();
  return cudaGetLastError();
}
cudaError_t cg_reduce_alpha_multi(CgState* st, int nrhs, const double* partial, int n, int* flags, cudaStream_t s) {
  cg_alpha_multi_kernel<<<nrhs, 1024, 0, s>>>(st, partial, n, flags);
  count_launch();
  return cudaGetLastError();
}
cudaError_t cg_reduce_beta_multi(CgState* st, int nrhs, const double* partial, int n, cudaStream_t s) {
  cg_beta_multi_kernel<<<nrhs, 1024, 0, s>>>(st, partial, n);
  count_launch();
  return cudaGetLastError();
}
template <typename T>
cudaError_t cg_update_xp_multi(const CgState* st, int nrhs, void* x, void* p, const void* r, size_t n, size_t stride, cudaStream_t s) {
  unsigned bx = (unsigned)ew_blocks(n);
  if (nrhs > 1 && bx > 2048) bx = 2048;   // nrhs columns share the machine
  cg_update_xp_multi_kernel<T><<<dim3(bx, (unsigned)nrhs), 256, 0, s>>>(st, (T2<T>*)x, (T2<T>*)p, (const T2<T>*)r, n, stride);
  count_launch();
  return cudaGetLastError();
}
template <typename T> cudaError_t cg_raxpy_norm(const CgState* st, const void* q, void* r, size_t n, double* partial, cudaStream_t s) {
  cg_raxpy_norm_kernel<T><<<reduce_blocks(n), RB_THREADS, 0, s>>>(st, (const T2<T>*)q, (T2<T>*)r, n, partial);
  count_launch();
  return cudaGetLastError();
}
template <typename T> cudaError_t axpy(double a, const void* x, void* y, size_t n, cudaStream_t s) {
  axpy_kernel<T><<<ew_blocks(n), 256, 0, s>>>((T)a, (const T2<T>*)x, (T2<T>*)y, n);
  count_launch();
  return cudaGetLastError();
}
template <typename T> cudaError_t xmy(const void* x, const void* y, void* z, size_t n, cudaStream_t s) {
  xmy_kernel<T><<<ew_blocks(n), 256, 0, s>>>((const T2<T>*)x, (const T2<T>*)y, (T2<T>*)z, n);
  count_launch();
  return cudaGetLastError();
}
cudaError_t add_f32_to_f64(const void* e32, void* x64, size_t n, cudaStream_t s) {
  add32_kernel<<<ew_blocks(n), 256, 0, s>>>((const float2*)e32, (double2*)x64, n);
  count_launch();
  return cudaGetLastError();
}
template <typename T> cudaError_t mask_frozen(const Geom& g, void* psi, cudaStream_t s) {
  if (g.bc == LQCD_BC_PERIODIC) return cudaSuccess;
  mask_frozen_kernel<T><<<(unsigned)((2 * g.Vh + 255) / 256), 256, 0, s>>>(g, (T2<T>*)psi);
  count_launch();
  return cudaGetLastError();
}

#define INST(T)                                                                                     \
  template cudaError_t norm2_partial<T>(const void*, size_t, double*, cudaStream_t);                \
  template cudaError_t dot_partial<T>(const void*, const void*, size_t, double*, cudaStream_t);     \
  template cudaError_t cg_update_xp<T>(const CgState*, void*, void*, const void*, size_t, cudaStream_t); \
  template cudaError_t cg_update_xp_multi<T>(const CgState*, int, void*, void*, const void*, size_t, size_t, cudaStream_t); \
  template cudaError_t axpy<T>(double, const void*, void*, size_t, cudaStream_t);                   \
  template cudaError_t cg_raxpy_norm<T>(const CgState*, const void*, void*, size_t, double*, cudaStream_t); \
  template cudaError_t xmy<T>(const void*, const void*, void*, size_t, cudaStream_t);               \
  template cudaError_t mask_frozen<T>(const Geom&, void*, cudaStream_t);
INST(double)
INST(float)
#undef INST

// ---- NEXT-2: pseudoscalar two-point function C(x4) = sum_{xvec} sum_{columns, spin, colour} |S|^2 ---------------
// (SURVEY.md 8(f)).  One CTA per tile, one thread per site; a site's |S|^2 over all columns is
// accumulated in fp64, then summed per local time coordinate in a fixed order; the second kernel adds the tiles of
// each time slice with a fixed assignment of tiles to threads and a fixed reduction tree, so the result is deterministic.
template <typename T>
__global__ void __launch_bounds__(256) corr_ps_tile_kernel(const Geom g, const T2<T>* __restrict__ cols, const int ncol,
                                                           const long long col_stride, double* __restrict__ partial) {
  __shared__ double s_val[256];
  const int TV = g.TV;
  const int tid = threadIdx.x;
  const int tile = blockIdx.x;
  double acc = 0.0;
  int l3 = -1;
  if (tid < 2 * TV) {
    const int p = tid >= TV ? 1 : 0;
    const int j = tid - p * TV;
    int l[4];
    local_coords(g, j, p, l);
    l3 = l[3];
    const size_t off = field_offset(g, 12, p, tile, 0, j);
    for (int c = 0; c < ncol; c++) {
      const T2<T>* v = cols + (size_t)c * col_stride + off;
#pragma unroll
      for (int k = 0; k < 12; k++) {
        const T2<T> w = __ldg(v + (size_t)k * TV);
        acc += (double)w.x * (double)w.x + (double)w.y * (double)w.y;
      }
    }
  }
  s_val[tid] = acc;
  __syncthreads();
  if (tid < g.b[3]) {   // thread t adds the sites with local time t, in thread order
    double s = 0.0;
    const int st3 = (g.b[0] >> 1) << (g.lb[1] + g.lb[2]);   // j stride of l3
    for (int p = 0; p < 2; p++)
      for (int jj = 0; jj < st3; jj++) s += s_val[p * TV + tid * st3 + jj];
    partial[(size_t)tile * g.b[3] + tid] = s;
  }
}
__global__ void __launch_bounds__(256) corr_ps_final_kernel(const Geom g, const double* __restrict__ partial,
                                                            double* __restrict__ C) {
  __shared__ double s_red[32];
  const int x4 = blockIdx.x;   // one CTA per time slice
  const int origin = (x4 / g.b[3]) * g.b[3], l3 = x4 - origin;
  double acc = 0.0;
  for (int t = threadIdx.x; t < g.ntiles; t += blockDim.x)   // thread i: tiles i, i+256, ... in order
    if (__ldg(g.tile_tab + (size_t)t * TILE_TAB + 8) == origin) acc += partial[(size_t)t * g.b[3] + l3];
  const double s = block_sum(acc, s_red);
  if (threadIdx.x == 0) C[x4] = s;
}
template <typename T>
cudaError_t correlator_ps(const Geom& g, const void* cols, int ncol, double* partial, double* C_dev, cudaStream_t s) {
  const int threads = ((2 * g.TV + 31) / 32) * 32;
  corr_ps_tile_kernel<T><<<g.ntiles, threads, 0, s>>>(g, (const T2<T>*)cols, ncol, (long long)2 * g.Vh * 12, partial);
  count_launch();
  corr_ps_final_kernel<<<g.L[3], 256, 0, s>>>(g, partial, C_dev);
  count_launch();
  return cudaGetLastError();
}
template cudaError_t correlator_ps<double>(const Geom&, const void*, int, double*, double*, cudaStream_t);
template cudaError_t correlator_ps<float>(const Geom&, const void*, int, double*, double*, cudaStream_t);

}  // namespace lqcd
