// slab.cu -- time-direction domain decomposition (the paper names the volume one
// GPU can hold as its limit).
//
// A rank owns the slab x4 in [t0, t0 + L[3]) of a lattice that is periodic in time (geometry bc = LQCD_BC_SLAB).
// The stencil kernels of dw.cu run on the slab unchanged, except that the two hops that leave it through a time
// face are not taken (time_hop_blocked).  The two kernels here supply them:
//
//   slab_pack_kernel   reads the slab's first and last time slice of `in` and writes two face buffers of spin-projected
//                      half spinors, 6 complex numbers per spatial site (half of a spinor: D2):
//                        send_lo[c][n] = P(m) in(x, 0)                                   -> rank below, its recv_hi
//                        send_hi[c][n] = theta4^* U_4(x, L3-1)^+ P(-m) in(x, L3-1)        -> rank above, its recv_lo
//                      with P(m): h0 = p0 - m p2, h1 = p1 - m p3 (gamma_4 row of hop_dir), m = +1 for D, -1 for D^+;
//   slab_faces_kernel  adds the missing hops to `out` after the stencil kernel has run:
//                        out(x, L3-1) -= k R(m)  theta4 U_4(x, L3-1) recv_hi          (forward hop)
//                        out(x, 0)    -= k R(-m) recv_lo                               (backward hop)
//                      with R(m): rows 0,1 += y0, y1; rows 2,3 += -m y0, -m y1.
// The link multiply of the backward hop is done by the sender, which owns U_4(x - 4^): no gauge halo is needed.
// Face buffers: [6][Ns] complex numbers of the working precision, n = x1 + L1 (x2 + L2 x3) (canonical spatial
// order), so that a face is one contiguous message.  With one rank, send_lo -> recv_hi and send_hi -> recv_lo of the
// same slab reproduce the periodic lattice.
#include "kernels.cuh"

namespace lqcd {

template <typename T> using T2 = typename vec2<T>::type;

template <typename T>
struct SlabArgs {
  const T2<T>* U;
  const T2<T>* in;
  T2<T>* out;
  T2<T>* lo;   // pack: send_lo; faces: recv_lo
  T2<T>* hi;   // pack: send_hi; faces: recv_hi
  T k;
  T m;         // +1: D, -1: D^+
  cx<T> th;    // exp(i theta4 / L4) per link
  int has_theta;
  int ns;      // spatial sites
};

template <typename T, int RECON>
__device__ __forceinline__ void load_u4(const Geom& g, const T2<T>* U, int p, int tile, int j, cx<T> (&u)[3][3]) {
  constexpr int NCU = RECON == 12 ? 6 : 9;
  const T2<T>* up = U + field_offset(g, 4 * NCU, p, tile, 3 * NCU, j);
#pragma unroll
  for (int i = 0; i < (RECON == 12 ? 2 : 3); i++)
#pragma unroll
    for (int k = 0; k < 3; k++) u[i][k] = ld<T>(up + (size_t)(3 * i + k) * g.TV);
  if (RECON == 12) {   // row 3 = conj(row 1 x row 2) (R16)
    u[2][0] = conj(u[0][1] * u[1][2] - u[0][2] * u[1][1]);
    u[2][1] = conj(u[0][2] * u[1][0] - u[0][0] * u[1][2]);
    u[2][2] = conj(u[0][0] * u[1][1] - u[0][1] * u[1][0]);
  }
}

__device__ __forceinline__ void spatial_site(const Geom& g, int n, int t, int (&x)[4]) {
  x[0] = n % g.L[0];
  n /= g.L[0];
  x[1] = n % g.L[1];
  x[2] = n / g.L[1];
  x[3] = t;
}

template <typename T, int RECON>
__global__ void __launch_bounds__(128) slab_pack_kernel(const Geom g, const SlabArgs<T> a) {
  const int id = blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= 2 * a.ns) return;
  const bool upper = id >= a.ns;   // upper face: slice L3-1 -> send_hi
  if (g.edges & (upper ? (LQCD_SLAB_OPEN_HI | LQCD_SLAB_SF_HI) : LQCD_SLAB_OPEN_LO)) return;   // open / SF boundary: nothing crosses it
  const int n = upper ? id - a.ns : id;
  int x[4], p, tile, j;
  spatial_site(g, n, upper ? g.L[3] - 1 : 0, x);
  site_locate(g, x, p, tile, j);
  const T2<T>* ps = a.in + field_offset(g, 12, p, tile, 0, j);
  const T m = upper ? -a.m : a.m;
  cx<T> h[2][3];
#pragma unroll
  for (int c = 0; c < 3; c++) {
    const cx<T> p0 = ld<T>(ps + (size_t)(0 + c) * g.TV), p1 = ld<T>(ps + (size_t)(3 + c) * g.TV);
    const cx<T> p2 = ld<T>(ps + (size_t)(6 + c) * g.TV), p3 = ld<T>(ps + (size_t)(9 + c) * g.TV);
    h[0][c] = cx<T>(fma(-m, p2.re, p0.re), fma(-m, p2.im, p0.im));
    h[1][c] = cx<T>(fma(-m, p3.re, p1.re), fma(-m, p3.im, p1.im));
  }
  T2<T>* dst = upper ? a.hi : a.lo;
  if (upper) {   // y = theta4^* U^+ h
    cx<T> u[3][3];
    load_u4<T, RECON>(g, a.U, p, tile, j, u);
    const cx<T> ph = conj(a.th);
#pragma unroll
    for (int s = 0; s < 2; s++) {
      cx<T> y[3];
#pragma unroll
      for (int c = 0; c < 3; c++) {
        cx<T> t = conj(u[0][c]) * h[s][0];
        t = cfma_conj(u[1][c], h[s][1], t);
        y[c] = cfma_conj(u[2][c], h[s][2], t);
        if (a.has_theta) y[c] = ph * y[c];
      }
#pragma unroll
      for (int c = 0; c < 3; c++) st<T>(dst + (size_t)(3 * s + c) * a.ns + n, y[c]);
    }
  } else {
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
      for (int c = 0; c < 3; c++) st<T>(dst + (size_t)(3 * s + c) * a.ns + n, h[s][c]);
  }
}

template <typename T, int RECON>
__global__ void __launch_bounds__(128) slab_faces_kernel(const Geom g, const SlabArgs<T> a) {
  const int id = blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= 2 * a.ns) return;
  const bool upper = id >= a.ns;   // upper face: forward hop of slice L3-1 from recv_hi
  if (g.edges & (upper ? (LQCD_SLAB_OPEN_HI | LQCD_SLAB_SF_HI) : LQCD_SLAB_OPEN_LO)) return;   // open / SF boundary: no hop
  const int n = upper ? id - a.ns : id;
  int x[4], p, tile, j;
  spatial_site(g, n, upper ? g.L[3] - 1 : 0, x);
  site_locate(g, x, p, tile, j);
  const T2<T>* src = upper ? a.hi : a.lo;
  cx<T> y[2][3];
#pragma unroll
  for (int s = 0; s < 2; s++)
#pragma unroll
    for (int c = 0; c < 3; c++) y[s][c] = ld<T>(src + (size_t)(3 * s + c) * a.ns + n);
  if (upper) {   // y = theta4 U h
    cx<T> u[3][3];
    load_u4<T, RECON>(g, a.U, p, tile, j, u);
#pragma unroll
    for (int s = 0; s < 2; s++) {
      cx<T> w[3];
#pragma unroll
      for (int c = 0; c < 3; c++) {
        cx<T> t = u[c][0] * y[s][0];
        t = cfma(u[c][1], y[s][1], t);
        w[c] = cfma(u[c][2], y[s][2], t);
        if (a.has_theta) w[c] = a.th * w[c];
      }
#pragma unroll
      for (int c = 0; c < 3; c++) y[s][c] = w[c];
    }
  }
  const T m = upper ? a.m : -a.m;
  T2<T>* op = a.out + field_offset(g, 12, p, tile, 0, j);
#pragma unroll
  for (int s = 0; s < 2; s++)
#pragma unroll
    for (int c = 0; c < 3; c++) {
      T2<T>* o_up = op + (size_t)(3 * s + c) * g.TV;       // rows 0,1: + y
      T2<T>* o_dn = op + (size_t)(6 + 3 * s + c) * g.TV;   // rows 2,3: - m y
      T2<T> v = *o_up, w = *o_dn;
      st<T>(o_up, cx<T>(fma(-a.k, y[s][c].re, v.x), fma(-a.k, y[s][c].im, v.y)));
      st<T>(o_dn, cx<T>(fma(a.k * m, y[s][c].re, w.x), fma(a.k * m, y[s][c].im, w.y)));
    }
}

template <typename T>
static SlabArgs<T> slab_args(const lqcd_geom* h, double kappa, bool dagger, const void* U, const void* in, void* out,
                             void* lo, void* hi) {
  SlabArgs<T> a;
  a.U = (const T2<T>*)U;
  a.in = (const T2<T>*)in;
  a.out = (T2<T>*)out;
  a.lo = (T2<T>*)lo;
  a.hi = (T2<T>*)hi;
  a.k = (T)kappa;
  a.m = dagger ? (T)-1 : (T)1;
  a.th = cx<T>((T)h->th_re[3], (T)h->th_im[3]);
  a.has_theta = h->has_theta ? 1 : 0;
  a.ns = h->g.L[0] * h->g.L[1] * h->g.L[2];
  return a;
}

template <typename T>
cudaError_t slab_pack(const lqcd_geom* h, bool dagger, const void* U, int recon, const void* in, void* send_lo,
                      void* send_hi, cudaStream_t s) {
  SlabArgs<T> a = slab_args<T>(h, 0.0, dagger, U, in, nullptr, send_lo, send_hi);
  const unsigned blocks = (unsigned)((2 * a.ns + 127) / 128);
  if (recon == 12) slab_pack_kernel<T, 12><<<blocks, 128, 0, s>>>(h->g, a);
  else slab_pack_kernel<T, 18><<<blocks, 128, 0, s>>>(h->g, a);
  count_launch();
  return cudaGetLastError();
}

template <typename T>
cudaError_t slab_faces(const lqcd_geom* h, double kappa, bool dagger, const void* U, int recon, const void* recv_lo,
                       const void* recv_hi, void* out, cudaStream_t s) {
  SlabArgs<T> a = slab_args<T>(h, kappa, dagger, U, nullptr, out, (void*)recv_lo, (void*)recv_hi);
  const unsigned blocks = (unsigned)((2 * a.ns + 127) / 128);
  if (recon == 12) slab_faces_kernel<T, 12><<<blocks, 128, 0, s>>>(h->g, a);
  else slab_faces_kernel<T, 18><<<blocks, 128, 0, s>>>(h->g, a);
  count_launch();
  return cudaGetLastError();
}

template cudaError_t slab_pack<double>(const lqcd_geom*, bool, const void*, int, const void*, void*, void*, cudaStream_t);
template cudaError_t slab_pack<float>(const lqcd_geom*, bool, const void*, int, const void*, void*, void*, cudaStream_t);
template cudaError_t slab_faces<double>(const lqcd_geom*, double, bool, const void*, int, const void*, const void*, void*, cudaStream_t);
template cudaError_t slab_faces<float>(const lqcd_geom*, double, bool, const void*, int, const void*, const void*, void*, cudaStream_t);

}  // namespace lqcd
