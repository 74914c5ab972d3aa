// layout.cu -- canonical (interchange, fp64 AoS) <-> internal (tile-blocked even-odd SoA) conversion,
// precision conversion and point sources.
#include "kernels.cuh"

namespace lqcd {

// one thread per internal site: idx -> (parity, tile, j) -> coordinates -> canonical site index
struct SiteId {
  int p, tile, j;
  int x[4];
  long long n;  // canonical index
};
__device__ __forceinline__ bool site_from_thread(const Geom& g, SiteId& s) {
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 2 * g.Vh) return false;
  s.p = (int)(idx / g.Vh);
  long long rem = idx - (long long)s.p * g.Vh;
  s.tile = (int)(rem / g.TV);
  s.j = (int)(rem - (long long)s.tile * g.TV);
  int T[4], l[4];
  tile_coords(g, s.tile, T);
  local_coords(g, s.j, s.p, l);
  for (int i = 0; i < 4; i++) s.x[i] = T[i] * g.b[i] + l[i];
  s.n = s.x[0] + (long long)g.L[0] * (s.x[1] + (long long)g.L[1] * (s.x[2] + (long long)g.L[2] * s.x[3]));
  return true;
}

template <typename T>
__global__ void gauge_import_kernel(const Geom g, const double2* __restrict__ canon, typename vec2<T>::type* U, int recon,
                                    const int t_lo, const int t_hi) {
  SiteId s;
  if (!site_from_thread(g, s)) return;
  if (s.x[3] < t_lo || s.x[3] >= t_hi) return;
  s.n -= (long long)t_lo * g.L[0] * g.L[1] * g.L[2];   // canon starts at slice t_lo
  const int NCU = recon == 12 ? 6 : 9;
  for (int mu = 0; mu < 4; mu++)
    for (int c = 0; c < NCU; c++) {
      double2 v = canon[(s.n * 4 + mu) * 9 + c];
      typename vec2<T>::type w;
      w.x = (T)v.x; w.y = (T)v.y;
      U[field_offset(g, 4 * NCU, s.p, s.tile, mu * NCU + c, s.j)] = w;
    }
}

template <typename T>
__global__ void gauge_export_kernel(const Geom g, const typename vec2<T>::type* __restrict__ U, double2* canon, int recon) {
  SiteId s;
  if (!site_from_thread(g, s)) return;
  const int NCU = recon == 12 ? 6 : 9;
  for (int mu = 0; mu < 4; mu++) {
    double2 m[9];
    for (int c = 0; c < NCU; c++) {
      typename vec2<T>::type w = U[field_offset(g, 4 * NCU, s.p, s.tile, mu * NCU + c, s.j)];
      m[c] = make_double2((double)w.x, (double)w.y);
    }
    if (recon == 12) {  // row 3 = conj(row 1 x row 2)
      for (int k = 0; k < 3; k++) {
        int k1 = (k + 1) % 3, k2 = (k + 2) % 3;
        double re = (m[k1].x * m[3 + k2].x - m[k1].y * m[3 + k2].y) - (m[k2].x * m[3 + k1].x - m[k2].y * m[3 + k1].y);
        double im = (m[k1].x * m[3 + k2].y + m[k1].y * m[3 + k2].x) - (m[k2].x * m[3 + k1].y + m[k2].y * m[3 + k1].x);
        m[6 + k] = make_double2(re, -im);
      }
    }
    for (int c = 0; c < 9; c++) canon[(s.n * 4 + mu) * 9 + c] = m[c];
  }
}

template <typename T>
__global__ void spinor_import_kernel(const Geom g, const double2* __restrict__ canon, typename vec2<T>::type* psi) {
  SiteId s;
  if (!site_from_thread(g, s)) return;
  for (int c = 0; c < 12; c++) {
    double2 v = canon[s.n * 12 + c];
    typename vec2<T>::type w;
    w.x = (T)v.x; w.y = (T)v.y;
    psi[field_offset(g, 12, s.p, s.tile, c, s.j)] = w;
  }
}

template <typename T>
__global__ void spinor_export_kernel(const Geom g, const typename vec2<T>::type* __restrict__ psi, double2* canon) {
  SiteId s;
  if (!site_from_thread(g, s)) return;
  for (int c = 0; c < 12; c++) {
    typename vec2<T>::type w = psi[field_offset(g, 12, s.p, s.tile, c, s.j)];
    canon[s.n * 12 + c] = make_double2((double)w.x, (double)w.y);
  }
}

// packed Hermitian blocks -> dense [n][2][6][6]
template <typename T>
__global__ void clover_export_kernel(const Geom g, const typename vec2<T>::type* __restrict__ A, double2* canon) {
  SiteId s;
  if (!site_from_thread(g, s)) return;
  for (int ch = 0; ch < 2; ch++) {
    double2* o = canon + (s.n * 2 + ch) * 36;
    for (int k = 0; k < 3; k++) {
      typename vec2<T>::type d = A[field_offset(g, 36, s.p, s.tile, 18 * ch + k, s.j)];
      o[(2 * k) * 6 + 2 * k] = make_double2((double)d.x, 0.0);
      o[(2 * k + 1) * 6 + 2 * k + 1] = make_double2((double)d.y, 0.0);
    }
    for (int i = 1; i < 6; i++)
      for (int jj = 0; jj < i; jj++) {
        typename vec2<T>::type l = A[field_offset(g, 36, s.p, s.tile, 18 * ch + 3 + i * (i - 1) / 2 + jj, s.j)];
        o[i * 6 + jj] = make_double2((double)l.x, (double)l.y);
        o[jj * 6 + i] = make_double2((double)l.x, -(double)l.y);
      }
  }
}

__global__ void to_f32_kernel(const double2* __restrict__ src, float2* dst, size_t n) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (; i < n; i += stride) {
    double2 v = src[i];
    dst[i] = make_float2((float)v.x, (float)v.y);
  }
}

template <typename T>
__global__ void point_source_kernel(typename vec2<T>::type* b, size_t off) {
  typename vec2<T>::type one;
  one.x = (T)1; one.y = (T)0;
  b[off] = one;
}

static inline unsigned site_blocks(const Geom& g) { return (unsigned)((2 * g.Vh + 255) / 256); }

template <typename T>
cudaError_t gauge_import(const Geom& g, const void* canon, void* U, int recon, cudaStream_t s) {
  gauge_import_kernel<T><<<site_blocks(g), 256, 0, s>>>(g, (const double2*)canon, (typename vec2<T>::type*)U, recon, 0, g.L[3]);
  count_launch();
  return cudaGetLastError();
}
template <typename T>
cudaError_t gauge_import_slab(const Geom& g, const void* canon_slab, void* U, int recon, int t_lo, int t_hi, cudaStream_t s) {
  gauge_import_kernel<T><<<site_blocks(g), 256, 0, s>>>(g, (const double2*)canon_slab, (typename vec2<T>::type*)U, recon, t_lo, t_hi);
  count_launch();
  return cudaGetLastError();
}
template <typename T>
cudaError_t gauge_export(const Geom& g, const void* U, void* canon, int recon, cudaStream_t s) {
  gauge_export_kernel<T><<<site_blocks(g), 256, 0, s>>>(g, (const typename vec2<T>::type*)U, (double2*)canon, recon);
  count_launch();
  return cudaGetLastError();
}
template <typename T>
cudaError_t spinor_import(const Geom& g, const void* canon, void* psi, cudaStream_t s) {
  spinor_import_kernel<T><<<site_blocks(g), 256, 0, s>>>(g, (const double2*)canon, (typename vec2<T>::type*)psi);
  count_launch();
  return cudaGetLastError();
}
template <typename T>
cudaError_t spinor_export(const Geom& g, const void* psi, void* canon, cudaStream_t s) {
  spinor_export_kernel<T><<<site_blocks(g), 256, 0, s>>>(g, (const typename vec2<T>::type*)psi, (double2*)canon);
  count_launch();
  return cudaGetLastError();
}
template <typename T>
cudaError_t clover_export(const Geom& g, const void* A, void* canon, cudaStream_t s) {
  clover_export_kernel<T><<<site_blocks(g), 256, 0, s>>>(g, (const typename vec2<T>::type*)A, (double2*)canon);
  count_launch();
  return cudaGetLastError();
}
cudaError_t to_f32(const void* src, void* dst, size_t ncomplex, cudaStream_t s) {
  unsigned blocks = (unsigned)((ncomplex + 1023) / 1024);
  if (blocks > 148u * 16u) blocks = 148u * 16u;
  if (blocks == 0) blocks = 1;
  to_f32_kernel<<<blocks, 256, 0, s>>>((const double2*)src, (float2*)dst, ncomplex);
  count_launch();
  return cudaGetLastError();
}
template <typename T>
cudaError_t point_source(const Geom& g, const int y[4], int spin, int colour, void* b, cudaStream_t s) {
  cudaError_t e = cudaMemsetAsync(b, 0, (size_t)2 * g.Vh * 12 * sizeof(typename vec2<T>::type), s);
  if (e != cudaSuccess) return e;
  int p, tile, j;
  site_locate(g, y, p, tile, j);
  point_source_kernel<T><<<1, 1, 0, s>>>((typename vec2<T>::type*)b, field_offset(g, 12, p, tile, 3 * spin + colour, j));
  count_launch();
  return cudaGetLastError();
}

#define INST(T)                                                                                  \
  template cudaError_t gauge_import<T>(const Geom&, const void*, void*, int, cudaStream_t);      \
  template cudaError_t gauge_import_slab<T>(const Geom&, const void*, void*, int, int, int, cudaStream_t); \
  template cudaError_t gauge_export<T>(const Geom&, const void*, void*, int, cudaStream_t);      \
  template cudaError_t spinor_import<T>(const Geom&, const void*, void*, cudaStream_t);          \
  template cudaError_t spinor_export<T>(const Geom&, const void*, void*, cudaStream_t);          \
  template cudaError_t clover_export<T>(const Geom&, const void*, void*, cudaStream_t);          \
  template cudaError_t point_source<T>(const Geom&, const int*, int, int, void*, cudaStream_t);
INST(double)
INST(float)
#undef INST

}  // namespace lqcd
