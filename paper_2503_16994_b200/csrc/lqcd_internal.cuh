// lqcd_internal.cuh -- geometry, internal layout and small complex helpers shared by the kernels.
//
// Internal layout.  The lattice is cut into 4-D tiles of
// b[0] x b[1] x b[2] x b[3] sites (all powers of two, b[0] >= 2).  Sites are split by parity
// p = (x1+x2+x3+x4) & 1; inside a tile a site has the checkerboard index
//   j = l0/2 + (b0/2) * (l1 + b1 * (l2 + b2 * l3)),          l = x - tile origin,
// and TV = (b0/2)*b1*b2*b3 is the number of sites of one parity in a tile.  A field with NC complex
// numbers per site is stored as   [parity][tile][component c][j]   in units of one complex number
// (double2 / float2): component-major inside the tile so that the 32 lanes of a warp (consecutive j)
// read 32 consecutive complex numbers = 512 B (fp64) / 256 B (fp32) per load instruction, and
// tile-major outside so that one tile's data is one contiguous block of memory.
// Tiles are ordered so that a linear sweep over the tile index walks one direction inside a chunk of
// (c1 x c2) tiles in the other two of (x2,x3,x4): the working set between the first and last use of a
// spinor or link then fits the 126 MB L2 (SURVEY.md section 7 "hard parts").
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/lqcd.h"

namespace lqcd {

struct Geom {
  int L[4];       // extents
  int b[4];       // tile extents (powers of two)
  int lb[4];      // log2: lb[0] = log2(b0/2), lb[1..3] = log2(b[1..3])
  int nt[4];      // tiles per direction
  int sw, da, db; // tile order: direction swept inside a chunk, and the two chunked directions (a permutation of 1,2,3)
  int c1, c2;     // L2 chunk, in tiles, along directions da and db
  int TV;         // sites of one parity per tile
  int ntiles;
  int bc;         // lqcd_bc
  int edges;      // LQCD_BC_SLAB: LQCD_SLAB_OPEN_LO | LQCD_SLAB_OPEN_HI (faces that are open boundaries of the lattice)
  long long Vh;   // sites of one parity
  // device table, TILE_TAB ints per tile: linear index of the 8 neighbour tiles (2*mu + (0: +mu, 1: -mu)),
  // then the time coordinate of the tile origin and its three space coordinates (library-owned, built by lqcd_geom_create)
  const int* tile_tab;
  unsigned int* sched;   // SCHED_SLOTS pairs of counters for the pipeline kernel's tile scheduler (library-owned, zeroed)
  int sm_count;     // host-side launch configuration (SMs, opt-in shared memory per CTA)
  int smem_optin;
};
enum { TILE_TAB = 12, SCHED_SLOTS = 64 };

// ---- tile order: [Tb hi][Ta hi][Ts][Tb lo][Ta lo][T0] ----------------------------------------------
// (sw, da, db) is a permutation of the directions (1, 2, 3): a linear sweep over the tile index walks direction sw
// inside a chunk of c1 x c2 tiles along (da, db); direction 0 is always whole.  The faces cut by chunk borders are
// those of da and db only -- the sweep direction's neighbours are one layer away -- so da and db are chosen among the
// directions whose tile faces are contiguous runs in memory.
__host__ __device__ inline int tile_linear(const Geom& g, int T0, int T1, int T2, int T3) {
  const int T[4] = {T0, T1, T2, T3};
  const int Ta = T[g.da], Tb = T[g.db], Ts = T[g.sw];
  int Tahi = Ta / g.c1, Talo = Ta - Tahi * g.c1;
  int Tbhi = Tb / g.c2, Tblo = Tb - Tbhi * g.c2;
  int nahi = g.nt[g.da] / g.c1;
  return T0 + g.nt[0] * (Talo + g.c1 * (Tblo + g.c2 * (Ts + g.nt[g.sw] * (Tahi + nahi * Tbhi))));
}
__host__ __device__ inline void tile_coords(const Geom& g, int t, int T[4]) {
  int nahi = g.nt[g.da] / g.c1;
  T[0] = t % g.nt[0]; t /= g.nt[0];
  int Talo = t % g.c1; t /= g.c1;
  int Tblo = t % g.c2; t /= g.c2;
  T[g.sw] = t % g.nt[g.sw]; t /= g.nt[g.sw];
  int Tahi = t % nahi; t /= nahi;
  int Tbhi = t;
  T[g.da] = Tahi * g.c1 + Talo;
  T[g.db] = Tbhi * g.c2 + Tblo;
}

// local coordinates of checkerboard index j, parity p, inside a tile (tile origins are even)
__host__ __device__ inline void local_coords(const Geom& g, int j, int p, int l[4]) {
  int l0h = j & ((g.b[0] >> 1) - 1);
  int r = j >> g.lb[0];
  l[1] = r & (g.b[1] - 1); r >>= g.lb[1];
  l[2] = r & (g.b[2] - 1); r >>= g.lb[2];
  l[3] = r;
  l[0] = 2 * l0h + ((p + l[1] + l[2] + l[3]) & 1);
}
__host__ __device__ inline int local_index(const Geom& g, const int l[4]) {
  return (l[0] >> 1) + ((l[1] + ((l[2] + (l[3] << g.lb[2])) << g.lb[1])) << g.lb[0]);
}

// full coordinates -> (parity, tile, j)
__host__ __device__ inline void site_locate(const Geom& g, const int x[4], int& p, int& tile, int& j) {
  int T[4], l[4];
  for (int i = 0; i < 4; i++) { T[i] = x[i] / g.b[i]; l[i] = x[i] - T[i] * g.b[i]; }
  p = (x[0] + x[1] + x[2] + x[3]) & 1;
  tile = tile_linear(g, T[0], T[1], T[2], T[3]);
  j = local_index(g, l);
}

// D7: frozen time slices
__host__ __device__ inline bool frozen_slice(const Geom& g, int x3) {
  if (g.bc == LQCD_BC_OPEN) return x3 == 0 || x3 == g.L[3] - 1;
  if (g.bc == LQCD_BC_SF_ORBI || g.bc == LQCD_BC_SF_AFWB) return x3 == 0;
  if (g.bc == LQCD_BC_SLAB) return ((g.edges & LQCD_SLAB_OPEN_LO) && x3 == 0) || ((g.edges & LQCD_SLAB_OPEN_HI) && x3 == g.L[3] - 1);
  return false;
}

// Is the time hop out of slice x3 (fwd: to x3 + 1, else to x3 - 1, wrapping) NOT taken by the stencil kernels?
// open / SF: hops onto frozen slices (D7).  Slab: hops across the slab's two time
// faces -- the face kernels of slab.cu add them from the exchanged half spinors.
__host__ __device__ inline bool time_hop_blocked(const Geom& g, int x3, bool fwd) {
  if (g.bc == LQCD_BC_SLAB && (fwd ? (x3 + 1 == g.L[3]) : (x3 == 0))) return true;
  const int xn = fwd ? ((x3 + 1 == g.L[3]) ? 0 : x3 + 1) : ((x3 == 0) ? g.L[3] - 1 : x3 - 1);
  return frozen_slice(g, xn);
}

// element offset (in complex numbers) of component c, site j of tile `tile`, parity p, NC comps/site
__host__ __device__ inline size_t field_offset(const Geom& g, int NC, int p, int tile, int c, int j) {
  return ((size_t)p * g.Vh + (size_t)tile * g.TV) * NC + (size_t)c * g.TV + j;
}

// ---- complex helpers ---------------------------------------------------------------------------
template <typename T> struct vec2;
template <> struct vec2<double> { typedef double2 type; };
template <> struct vec2<float> { typedef float2 type; };

template <typename T>
struct cx {
  T re, im;
  __host__ __device__ cx() {}
  __host__ __device__ cx(T r, T i) : re(r), im(i) {}
};
template <typename T> __device__ __forceinline__ cx<T> operator+(cx<T> a, cx<T> b) { return cx<T>(a.re + b.re, a.im + b.im); }
template <typename T> __device__ __forceinline__ cx<T> operator-(cx<T> a, cx<T> b) { return cx<T>(a.re - b.re, a.im - b.im); }
template <typename T> __device__ __forceinline__ cx<T> operator*(cx<T> a, cx<T> b) {
  return cx<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <typename T> __device__ __forceinline__ cx<T> operator*(T s, cx<T> a) { return cx<T>(s * a.re, s * a.im); }
template <typename T> __device__ __forceinline__ cx<T> conj(cx<T> a) { return cx<T>(a.re, -a.im); }
// a*b + c, conj(a)*b + c
template <typename T> __device__ __forceinline__ cx<T> cfma(cx<T> a, cx<T> b, cx<T> c) {
  return cx<T>(fma(a.re, b.re, fma(-a.im, b.im, c.re)), fma(a.re, b.im, fma(a.im, b.re, c.im)));
}
template <typename T> __device__ __forceinline__ cx<T> cfma_conj(cx<T> a, cx<T> b, cx<T> c) {
  return cx<T>(fma(a.re, b.re, fma(a.im, b.im, c.re)), fma(a.re, b.im, fma(-a.im, b.re, c.im)));
}
// multiply by +i / -i
template <typename T> __device__ __forceinline__ cx<T> mul_i(cx<T> a) { return cx<T>(-a.im, a.re); }
template <typename T> __device__ __forceinline__ cx<T> mul_mi(cx<T> a) { return cx<T>(a.im, -a.re); }

template <typename T> __device__ __forceinline__ cx<T> ld(const typename vec2<T>::type* p) {
  typename vec2<T>::type v = __ldg(p);
  return cx<T>(v.x, v.y);
}
template <typename T> __device__ __forceinline__ void st(typename vec2<T>::type* p, cx<T> a) {
  typename vec2<T>::type v;
  v.x = a.re; v.y = a.im;
  *p = v;
}

// ---- host side -----------------------------------------------------------------------------------
void set_error(const char* fmt, ...);
bool cuda_ok(cudaError_t e, const char* what);
void count_launch(int n = 1);
void set_host_slab(int n);

}  // namespace lqcd

struct lqcd_geom {
  lqcd::Geom g;
  lqcd_geom_desc desc;
  double th_re[4], th_im[4];   // per-link phase factors exp(i theta/L)
  bool has_theta;
  int sm_count;
  int smem_optin;   // max dynamic shared memory per CTA (opt-in)
};
