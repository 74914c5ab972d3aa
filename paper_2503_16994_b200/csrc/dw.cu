// dw.cu -- the Wilson-clover stencil kernel (fused pieces of a6).
//
//   DIAG_ONE : out(x) = self(x)      - k * (H in)(x)            D with csw = 0       (D3, D6)
//   DIAG_PRE : out(x) = A(x) self(x) - k * (H in)(x)            D (k = kappa), and the second half of the
//                                                              even-odd operator (k = kappa^2)   (D6, D8)
//   DIAG_POST: out(x) = B(x) (H in)(x)                          A_oo^{-1} H_oe, first half of D^      (D8)
// with (H in)(x) = sum_mu [ theta_mu (1 - gamma_mu) U_mu(x) in(x+mu) + theta_mu^* (1 + gamma_mu) U_mu(x-mu)^+ in(x-mu) ]
// and the projector signs swapped for the gamma5-conjugate (D^+ = gamma5 D gamma5; A commutes with gamma5).
// Spin projection to half spinors before the SU(3) multiply (D2); one thread per site; a CTA owns one
// tile (both parities for the full operator) so that neighbour spinors and backward links are reused
// out of L1; all loads are 128-bit (fp64) / 64-bit (fp32) and coalesced over the tile-local site index.
// Epilogues (CG fusion): EPI_STORE, EPI_STORE_NORM (|out|^2 partial per CTA),
// EPI_AXPY_NORM (r -= alpha*out, |r|^2 partial; out itself is never written).
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <atomic>

#include "dw.cuh"
#include "pipe.cuh"

namespace lqcd {

template <typename T> using T2 = typename vec2<T>::type;

// LDG = true: read-only global load (ld.global.nc); false: generic load (the pointer may be shared or global)
template <typename T, bool LDG>
__device__ __forceinline__ cx<T> ldx(const T2<T>* p) {
  if (LDG) return ld<T>(p);
  T2<T> v = *p;
  return cx<T>(v.x, v.y);
}

// ---- one hopping direction -------------------------------------------------------------------------
// m = +1 selects (1 - gamma_mu), m = -1 selects (1 + gamma_mu) (D2):
//   mu=0: h0 = p0 + m i p3, h1 = p1 + m i p2; low2 = -m i y1, low3 = -m i y0
//   mu=1: h0 = p0 + m p3,   h1 = p1 - m p2;   low2 = -m y1,   low3 = +m y0
//   mu=2: h0 = p0 + m i p2, h1 = p1 - m i p3; low2 = -m i y0, low3 = +m i y1
//   mu=3: h0 = p0 - m p2,   h1 = p1 - m p3;   low2 = -m y0,   low3 = -m y1
template <typename T, int RECON, int MU, bool FWD, bool LDG = true>
__device__ __forceinline__ void hop_dir(const T2<T>* __restrict__ psi, const T2<T>* __restrict__ u, const int SP,
                                        const int SU, const T m, const bool has_theta, const cx<T> th,
                                        cx<T> (&acc)[12]) {
  cx<T> h[2][3];
#pragma unroll
  for (int a = 0; a < 3; a++) {
    cx<T> p0 = ldx<T, LDG>(psi + (0 + a) * SP), p1 = ldx<T, LDG>(psi + (3 + a) * SP);
    cx<T> p2 = ldx<T, LDG>(psi + (6 + a) * SP), p3 = ldx<T, LDG>(psi + (9 + a) * SP);
    if (MU == 0) {
      h[0][a] = cx<T>(fma(-m, p3.im, p0.re), fma(m, p3.re, p0.im));
      h[1][a] = cx<T>(fma(-m, p2.im, p1.re), fma(m, p2.re, p1.im));
    } else if (MU == 1) {
      h[0][a] = cx<T>(fma(m, p3.re, p0.re), fma(m, p3.im, p0.im));
      h[1][a] = cx<T>(fma(-m, p2.re, p1.re), fma(-m, p2.im, p1.im));
    } else if (MU == 2) {
      h[0][a] = cx<T>(fma(-m, p2.im, p0.re), fma(m, p2.re, p0.im));
      h[1][a] = cx<T>(fma(m, p3.im, p1.re), fma(-m, p3.re, p1.im));
    } else {
      h[0][a] = cx<T>(fma(-m, p2.re, p0.re), fma(-m, p2.im, p0.im));
      h[1][a] = cx<T>(fma(-m, p3.re, p1.re), fma(-m, p3.im, p1.im));
    }
  }
  cx<T> U[3][3];
#pragma unroll
  for (int i = 0; i < (RECON == 12 ? 2 : 3); i++)
#pragma unroll
    for (int k = 0; k < 3; k++) U[i][k] = ldx<T, LDG>(u + (3 * i + k) * SU);
  if (RECON == 12) {  // row 3 = conj(row 1 x row 2) (R16)
    U[2][0] = conj(U[0][1] * U[1][2] - U[0][2] * U[1][1]);
    U[2][1] = conj(U[0][2] * U[1][0] - U[0][0] * U[1][2]);
    U[2][2] = conj(U[0][0] * U[1][1] - U[0][1] * U[1][0]);
  }
  cx<T> y[2][3];
#pragma unroll
  for (int s = 0; s < 2; s++)
#pragma unroll
    for (int a = 0; a < 3; a++) {
      if (FWD) {  // y = U h
        cx<T> t = U[a][0] * h[s][0];
        t = cfma(U[a][1], h[s][1], t);
        y[s][a] = cfma(U[a][2], h[s][2], t);
      } else {  // y = U^+ h
        cx<T> t = conj(U[0][a]) * h[s][0];
        t = cfma_conj(U[1][a], h[s][1], t);
        y[s][a] = cfma_conj(U[2][a], h[s][2], t);
      }
    }
  if (has_theta) {
    const cx<T> ph = FWD ? th : conj(th);
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
      for (int a = 0; a < 3; a++) y[s][a] = ph * y[s][a];
  }
#pragma unroll
  for (int a = 0; a < 3; a++) {
    acc[0 + a] = acc[0 + a] + y[0][a];
    acc[3 + a] = acc[3 + a] + y[1][a];
    if (MU == 0) {  // low2 = -m i y1, low3 = -m i y0
      acc[6 + a] = cx<T>(fma(m, y[1][a].im, acc[6 + a].re), fma(-m, y[1][a].re, acc[6 + a].im));
      acc[9 + a] = cx<T>(fma(m, y[0][a].im, acc[9 + a].re), fma(-m, y[0][a].re, acc[9 + a].im));
    } else if (MU == 1) {  // low2 = -m y1, low3 = +m y0
      acc[6 + a] = cx<T>(fma(-m, y[1][a].re, acc[6 + a].re), fma(-m, y[1][a].im, acc[6 + a].im));
      acc[9 + a] = cx<T>(fma(m, y[0][a].re, acc[9 + a].re), fma(m, y[0][a].im, acc[9 + a].im));
    } else if (MU == 2) {  // low2 = -m i y0, low3 = +m i y1
      acc[6 + a] = cx<T>(fma(m, y[0][a].im, acc[6 + a].re), fma(-m, y[0][a].re, acc[6 + a].im));
      acc[9 + a] = cx<T>(fma(-m, y[1][a].im, acc[9 + a].re), fma(m, y[1][a].re, acc[9 + a].im));
    } else {  // low2 = -m y0, low3 = -m y1
      acc[6 + a] = cx<T>(fma(-m, y[0][a].re, acc[6 + a].re), fma(-m, y[0][a].im, acc[6 + a].im));
      acc[9 + a] = cx<T>(fma(-m, y[1][a].re, acc[9 + a].re), fma(-m, y[1][a].im, acc[9 + a].im));
    }
  }
}

#ifndef PIPE_NHB32
#define PIPE_NHB32 4
#endif
#ifndef PIPE_NSPB32
#define PIPE_NSPB32 2
#endif

// ---- packed Hermitian 6x6 block times 6-vector, both chiralities (D5) ------------------------------
// per chirality 18 complex slots: (d0,d1) (d2,d3) (d4,d5), then the strict lower triangle row by row.
template <typename T>
__device__ __forceinline__ void clover_mul(const T2<T>* __restrict__ A, const int TV, const cx<T> (&v)[12],
                                           cx<T> (&out)[12]) {
#pragma unroll
  for (int ch = 0; ch < 2; ch++) {
    const T2<T>* B = A + (size_t)(18 * ch) * TV;
    cx<T> o[6];
#pragma unroll
    for (int k = 0; k < 3; k++) {
      cx<T> d = ld<T>(B + k * TV);
      o[2 * k] = d.re * v[6 * ch + 2 * k];
      o[2 * k + 1] = d.im * v[6 * ch + 2 * k + 1];
    }
#pragma unroll
    for (int i = 1; i < 6; i++)
#pragma unroll
      for (int jj = 0; jj < i; jj++) {
        cx<T> l = ld<T>(B + (3 + i * (i - 1) / 2 + jj) * TV);
        o[i] = cfma(l, v[6 * ch + jj], o[i]);
        o[jj] = cfma_conj(l, v[6 * ch + i], o[jj]);
      }
#pragma unroll
    for (int i = 0; i < 6; i++) out[6 * ch + i] = o[i];
  }
}

// One thread per site, one tile (both parities for the full operator) per CTA at a time; CTA b works through
// tiles b, b + gridDim.x, ... (gridDim.x == ntiles gives the plain one-tile-per-CTA launch).
// twisted mass (NEXT-4): o += i t gamma5 v, gamma5 = diag(1,1,-1,-1) in the chiral basis (components 0..5 / 6..11)
template <typename T, int C0, int C1>
__device__ __forceinline__ void add_twist(const T t, const cx<T> (&v)[12], cx<T> (&o)[12]) {
#pragma unroll
  for (int c = C0; c < C1; c++) {
    const T tc = (c < 6) ? t : -t;
    o[c] = cx<T>(fma(-tc, v[c].im, o[c].re), fma(tc, v[c].re, o[c].im));
  }
}

template <typename T, int RECON, int DIAG, bool SPLIT>
__device__ __forceinline__ void dw_body(const Geom& g, const DwArgs<T>& a) {
  constexpr int NCU = (RECON == 12) ? 6 : 9;
  __shared__ double s_red[8];
  if (a.skip != nullptr && *a.skip != 0) return;  // CG finished: uniform early exit
  const int TV = g.TV;
  const int tid = threadIdx.x;
  // SPLIT: the full operator with one PARITY of a tile per CTA (work item = 2*tile + parity, TV threads): three
  // 128-thread CTAs fit an SM where one 256-thread CTA did, i.e. 12 warps of loads in flight instead of 8.
  const int npar = (!SPLIT && a.parity < 0) ? 2 : 1;
  const bool active = tid < npar * TV;
  const int pidx = SPLIT ? (int)(blockIdx.x & 1) : ((tid >= TV) ? 1 : 0);
  const int j = SPLIT ? tid : tid - pidx * TV;
  const int p = (a.parity < 0) ? pidx : a.parity;
  const int q = 1 - p;
  double nrm = 0.0;
  int l[4];
  local_coords(g, j, p, l);
  const bool nonper = (g.bc != LQCD_BC_PERIODIC);
  const T sg = a.dagger ? T(-1) : T(1);
  const int bh0 = g.b[0] >> 1;
  const int l0h = l[0] >> 1;
  const int st1 = bh0, st2 = bh0 << g.lb[1], st3 = st2 << g.lb[2];
  const int tstep = SPLIT ? (int)(gridDim.x >> 1) : (int)gridDim.x;   // SPLIT needs an even grid
  for (int tile = SPLIT ? (int)(blockIdx.x >> 1) : (int)blockIdx.x; tile < g.ntiles; tile += tstep) {
    const int* __restrict__ tab = g.tile_tab + (size_t)tile * TILE_TAB;
    if (active) {
      const int x3 = __ldg(tab + 8) + l[3];
      const bool fz = nonper && frozen_slice(g, x3);
      cx<T> res[12];
      if (fz) {
#pragma unroll
        for (int c = 0; c < 12; c++) res[c] = cx<T>(0, 0);
      } else {
        cx<T> acc[12];
#pragma unroll
        for (int c = 0; c < 12; c++) acc[c] = cx<T>(0, 0);
        const size_t ubase_self = field_offset(g, 4 * NCU, p, tile, 0, j);
        // direction 0
        {
          bool cr = (l[0] + 1 == g.b[0]);
          int jn = j - l0h + (cr ? 0 : ((l[0] + 1) >> 1));
          int tn = cr ? __ldg(tab + 0) : tile;
          hop_dir<T, RECON, 0, true>(a.in + field_offset(g, 12, q, tn, 0, jn), a.U + ubase_self + (size_t)(0 * NCU) * TV,
                                     TV, TV, sg, a.has_theta, a.theta[0], acc);
          cr = (l[0] == 0);
          jn = j - l0h + (cr ? bh0 - 1 : ((l[0] - 1) >> 1));
          tn = cr ? __ldg(tab + 1) : tile;
          hop_dir<T, RECON, 0, false>(a.in + field_offset(g, 12, q, tn, 0, jn),
                                      a.U + field_offset(g, 4 * NCU, q, tn, 0 * NCU, jn), TV, TV, -sg, a.has_theta,
                                      a.theta[0], acc);
        }
        // direction 1
        {
          bool cr = (l[1] + 1 == g.b[1]);
          int jn = cr ? j - (g.b[1] - 1) * st1 : j + st1;
          int tn = cr ? __ldg(tab + 2) : tile;
          hop_dir<T, RECON, 1, true>(a.in + field_offset(g, 12, q, tn, 0, jn), a.U + ubase_self + (size_t)(1 * NCU) * TV,
                                     TV, TV, sg, a.has_theta, a.theta[1], acc);
          cr = (l[1] == 0);
          jn = cr ? j + (g.b[1] - 1) * st1 : j - st1;
          tn = cr ? __ldg(tab + 3) : tile;
          hop_dir<T, RECON, 1, false>(a.in + field_offset(g, 12, q, tn, 0, jn),
                                      a.U + field_offset(g, 4 * NCU, q, tn, 1 * NCU, jn), TV, TV, -sg, a.has_theta,
                                      a.theta[1], acc);
        }
        // direction 2
        {
          bool cr = (l[2] + 1 == g.b[2]);
          int jn = cr ? j - (g.b[2] - 1) * st2 : j + st2;
          int tn = cr ? __ldg(tab + 4) : tile;
          hop_dir<T, RECON, 2, true>(a.in + field_offset(g, 12, q, tn, 0, jn), a.U + ubase_self + (size_t)(2 * NCU) * TV,
                                     TV, TV, sg, a.has_theta, a.theta[2], acc);
          cr = (l[2] == 0);
          jn = cr ? j + (g.b[2] - 1) * st2 : j - st2;
          tn = cr ? __ldg(tab + 5) : tile;
          hop_dir<T, RECON, 2, false>(a.in + field_offset(g, 12, q, tn, 0, jn),
                                      a.U + field_offset(g, 4 * NCU, q, tn, 2 * NCU, jn), TV, TV, -sg, a.has_theta,
                                      a.theta[2], acc);
        }
        // direction 3 (time): hops onto frozen slices are skipped, never multiplied by zero (D7, P7)
        {
          bool cr = (l[3] + 1 == g.b[3]);
          int jn = cr ? j - (g.b[3] - 1) * st3 : j + st3;
          int tn = cr ? __ldg(tab + 6) : tile;
          if (!(nonper && time_hop_blocked(g, x3, true)))
            hop_dir<T, RECON, 3, true>(a.in + field_offset(g, 12, q, tn, 0, jn),
                                       a.U + ubase_self + (size_t)(3 * NCU) * TV, TV, TV, sg, a.has_theta, a.theta[3], acc);
          cr = (l[3] == 0);
          jn = cr ? j + (g.b[3] - 1) * st3 : j - st3;
          tn = cr ? __ldg(tab + 7) : tile;
          if (!(nonper && time_hop_blocked(g, x3, false)))
            hop_dir<T, RECON, 3, false>(a.in + field_offset(g, 12, q, tn, 0, jn),
                                        a.U + field_offset(g, 4 * NCU, q, tn, 3 * NCU, jn), TV, TV, -sg, a.has_theta,
                                        a.theta[3], acc);
        }
        // site-diagonal part
        if (DIAG == DIAG_POST) {
          clover_mul<T>(a.A + field_offset(g, 36, p, tile, 0, j), TV, acc, res);
        } else {
          cx<T> v[12];
          const T2<T>* sp = a.self + field_offset(g, 12, p, tile, 0, j);
#pragma unroll
          for (int c = 0; c < 12; c++) v[c] = ld<T>(sp + c * TV);
          if (DIAG == DIAG_PRE) {
            cx<T> av[12];
            clover_mul<T>(a.A + field_offset(g, 36, p, tile, 0, j), TV, v, av);
#pragma unroll
            for (int c = 0; c < 12; c++) res[c] = cx<T>(fma(-a.k, acc[c].re, av[c].re), fma(-a.k, acc[c].im, av[c].im));
          } else {
#pragma unroll
            for (int c = 0; c < 12; c++) res[c] = cx<T>(fma(-a.k, acc[c].re, v[c].re), fma(-a.k, acc[c].im, v[c].im));
          }
          if (a.tm != T(0)) add_twist<T, 0, 12>(a.tm, v, res);
        }
      }
      // epilogue
      const size_t ooff = field_offset(g, 12, p, tile, 0, j);
      if (a.epi == EPI_AXPY_NORM) {
        const T al = (T)(*a.alpha);
        T2<T>* rp = a.r + ooff;
#pragma unroll
        for (int c = 0; c < 12; c++) {
          T2<T> rv = rp[c * TV];
          cx<T> w(fma(-al, res[c].re, rv.x), fma(-al, res[c].im, rv.y));
          st<T>(rp + c * TV, w);
          nrm += (double)w.re * (double)w.re + (double)w.im * (double)w.im;
        }
      } else {
        T2<T>* op = a.out + ooff;
#pragma unroll
        for (int c = 0; c < 12; c++) st<T>(op + c * TV, res[c]);
        if (a.epi == EPI_STORE_NORM) {
#pragma unroll
          for (int c = 0; c < 12; c++) nrm += (double)res[c].re * (double)res[c].re + (double)res[c].im * (double)res[c].im;
        }
      }
    }
  }
  if (a.epi != EPI_STORE) {  // fixed-order CTA reduction: shuffle tree, then warp sums in warp order
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nrm += __shfl_xor_sync(0xffffffffu, nrm, o);
    if ((tid & 31) == 0) s_red[tid >> 5] = nrm;
    __syncthreads();
    if (tid == 0) {
      double s = 0;
      const int nw = (blockDim.x + 31) >> 5;
      for (int w = 0; w < nw; w++) s += s_red[w];
      a.partial[blockIdx.x] = s;
    }
  }
}

template <typename T, int RECON, int DIAG>
__global__ void __launch_bounds__(256) dw_kernel(const Geom g, const DwArgs<T> a) {
  dw_body<T, RECON, DIAG, false>(g, a);
}
// 128-thread CTAs (one parity of a tile): three resident per SM
template <typename T, int RECON, int DIAG, bool SPLIT>
__global__ void __launch_bounds__(128, 3) dw_kernel_h(const Geom g, const DwArgs<T> a) {
  dw_body<T, RECON, DIAG, SPLIT>(g, a);
}


// =====================================================================================================
// Persistent, warp-specialised version of the full-lattice operator (parity = -1, self == in).
//
// The one-thread-per-site kernel above is latency-bound: 184 registers per thread in fp64 allow 8 warps per SM
// and every hop is a dependent round trip to L2/DRAM.  Here NO consumer thread ever touches global memory
// for its operands; three kinds of warps share a CTA:
//   * warp 8, one lane: 1-D bulk-asynchronous copies (cp.async.bulk, SASS UBLKCP) stream what a tile reads
//     from HBM exactly once -- its links (4 stages of NCU components x both parities), its clover blocks
//     (36/NCU stages) and its spinor -- into a shared-memory ring of `nslot` stage buffers guarded by
//     full/empty mbarriers.  The tile-blocked layout makes every stage a pair of contiguous blocks, so no
//     tensor map is needed, and the bytes in flight per SM no longer depend on resident warps.
//   * warps 9-11: the halo of direction mu -- the spinors on the two faces of the neighbour tiles and the
//     links U_mu(x - mu) leaving the backward face -- is gathered element by element with per-thread
//     asynchronous copies (cp.async, SASS LDGSTS; they complete on an mbarrier, occupy no registers) into a
//     double-buffered halo area; the stage order (below) gives every halo two (fp64) or three (fp32) stages of lead.
//   * warps 0-7: 2*TV consumer threads, one per site (both parities of the tile), run the spin-projected
//     hops and the clover multiply purely out of shared memory.
// =====================================================================================================

// packed Hermitian block, one component at a time, ACCUMULATED into o: c in [0,36), chirality c/18; slot
// c%18 < 3 holds two real diagonal entries, slot 3 + i(i-1)/2 + jj the element (i,jj) of the strict lower
// triangle (D5).
template <typename T, int C>
__device__ __forceinline__ void clover_comp(const cx<T> l, const cx<T> (&v)[12], cx<T> (&o)[12]) {
  constexpr int ch = C / 18, s = C % 18;
  if (s < 3) {   // o += diag * v
    o[6 * ch + 2 * s] = cx<T>(fma(l.re, v[6 * ch + 2 * s].re, o[6 * ch + 2 * s].re), fma(l.re, v[6 * ch + 2 * s].im, o[6 * ch + 2 * s].im));
    o[6 * ch + 2 * s + 1] =
        cx<T>(fma(l.im, v[6 * ch + 2 * s + 1].re, o[6 * ch + 2 * s + 1].re), fma(l.im, v[6 * ch + 2 * s + 1].im, o[6 * ch + 2 * s + 1].im));
  } else {
    constexpr int t = s - 3;
    constexpr int i = (t >= 10) ? 5 : (t >= 6) ? 4 : (t >= 3) ? 3 : (t >= 1) ? 2 : 1;
    constexpr int jj = t - i * (i - 1) / 2;
    o[6 * ch + i] = cfma(l, v[6 * ch + jj], o[6 * ch + i]);
    o[6 * ch + jj] = cfma_conj(l, v[6 * ch + i], o[6 * ch + jj]);
  }
}
template <typename T, int C0, int N>
struct CloverStage {
  static __device__ __forceinline__ void run(const T2<T>* __restrict__ b, const int TV, const cx<T> (&v)[12], cx<T> (&o)[12]) {
    T2<T> w = *b;
    clover_comp<T, C0>(cx<T>(w.x, w.y), v, o);
    CloverStage<T, C0 + 1, N - 1>::run(b + TV, TV, v, o);
  }
};
template <typename T, int C0>
struct CloverStage<T, C0, 0> {
  static __device__ __forceinline__ void run(const T2<T>*, const int, const cx<T> (&)[12], cx<T> (&)[12]) {}
};

// The pipeline kernel is written for 4x4x4x4 tiles: TV = 128 sites of one parity, every face 2*TV/4 = 64 columns.
// With both fixed at compile time every shared-memory access of the arithmetic warps is an immediate offset from
// one base register, and a pair of halo buffers interleaves into rows of 2*PIPE_NF = PIPE_TV columns, i.e. halo rows
// have the same stride as tile rows and a hop needs no stride select.
// Spinor-tile buffers of the pipeline kernels.  With one buffer the next tile's spinor can only be requested once the
// arithmetic warps are done with the hops of this one, and its trip from DRAM is covered by the clover stages alone;
// fp32 has the shared memory for a second buffer (fp64 does not), and the request then goes out a whole tile ahead.
template <typename T> __host__ __device__ constexpr int pipe_nspb() { return sizeof(T) == 4 ? PIPE_NSPB32 : 1; }
// Halo buffers of the full-lattice kernel: pairs of them interleave into rows of PIPE_TV columns (so halo rows have the
// stride of tile rows), one pair in fp64 (all that fits), two pairs in fp32: a halo can then be gathered a whole tile
// ahead (profile: 11 % of the arithmetic warps' samples were waits for the halos of the third and fourth hop; Dw fp32 at
// 48^3 x 96 with 2 / 3 / 4 buffers: 1.562 / 1.512 / 1.502 ms).
template <typename T> __host__ __device__ constexpr int pipe_nhb() { return sizeof(T) == 4 ? PIPE_NHB32 : 2; }
// Clover stages placed between the two pairs of hop stages (the rest follows the last hop).  fp32: half of them, so that
// every halo has three stages of lead.  fp64, with its single spinor buffer: one -- the spinor tile is released after
// the last hop, and the more stages follow it the more time the next tile's spinor has to arrive from DRAM; the halos,
// which mostly come out of L2, make do with two stages of lead (measured: 2.948 -> 2.914 ms at 48^3 x 96; none early:
// 3.003 ms; fp32 with one early stage: 1.573 -> 1.593 ms).
template <typename T> __host__ __device__ constexpr int pipe_early_stages(int nstc) { return sizeof(T) == 8 ? (nstc > 0 ? 1 : 0) : nstc / 2; }
enum { PIPE_CONS_WARPS = 8, PIPE_HALO_THREADS = 96, PIPE_THREADS = 384, PIPE_MAX_SLOTS = 12, PIPE_TV = 128, PIPE_NF = 64,
       PIPE_TQ = 4 };
struct PipeBars {
  uint64_t full_sp[2], empty_sp[2];   // spinor tile buffer(s): one in fp64, two in fp32 (pipe_nspb)
  uint64_t full_h[4], empty_h[4];   // two halo buffers (full lattice), three or four (half lattice)
  uint64_t full[PIPE_MAX_SLOTS], empty[PIPE_MAX_SLOTS];
  uint64_t tq_full[PIPE_TQ], tq_empty[PIPE_TQ];   // tile queue: the producer lane tells the other warps which tile is next
  int tq[PIPE_TQ];
};

// ---- tile scheduler ------------------------------------------------------------------------------------------
// A CTA starts with tile blockIdx.x and then draws tiles gridDim.x, gridDim.x + 1, ... from a global counter
// (DwArgs::sched[0]), so that at any moment the CTAs of the grid work on (nearly) consecutive tile indices no matter
// how their speeds differ: with a static assignment b, b + grid, ... the CTAs drift apart over the hundreds of tiles
// each of them walks, and the neighbour tiles a halo gathers are no longer the ones that just went through L2.
// Only the producer lane draws; it hands every tile index to the halo and arithmetic warps through a small
// shared-memory queue (negative index: no more tiles).
__device__ __forceinline__ void tq_push(PipeBars* bars, const int kt, const int tile) {
  const int q = kt & (PIPE_TQ - 1);
  mbar_wait_relaxed(&bars->tq_empty[q], (uint32_t)(((kt / PIPE_TQ) & 1) ^ 1));
  *(volatile int*)&bars->tq[q] = tile;
  mbar_arrive(&bars->tq_full[q]);   // release: the index is visible to whoever sees the phase complete
}
__device__ __forceinline__ int tq_pop(PipeBars* bars, const int kt, const int lane) {
  const int q = kt & (PIPE_TQ - 1);
  mbar_wait(&bars->tq_full[q], (uint32_t)((kt / PIPE_TQ) & 1));
  const int tile = *(volatile int*)&bars->tq[q];
  __syncwarp();
  if (lane == 0) mbar_arrive(&bars->tq_empty[q]);
  return tile;
}
__device__ __forceinline__ int next_tile(const int nunits, unsigned int* sched, const int tile) {
  const int n = sched ? (int)(gridDim.x + atomicAdd(sched, 1u)) : tile + (int)gridDim.x;
  return n < nunits ? n : -1;
}

struct RingPos {
  int slot;
  uint32_t ph;
  __device__ __forceinline__ void advance(const int nslot) {
    if (++slot == nslot) { slot = 0; ph ^= 1u; }
  }
};

template <typename T, int NCU, int S, int NS>
struct CloverPipe {
  static __device__ __forceinline__ void run(PipeBars* bars, const T2<T>* ring, RingPos& rp, const int nslot, const int TV,
                                             const int own, const bool live, const int lane, const cx<T> (&v)[12],
                                             cx<T> (&o)[12]) {
    mbar_wait(&bars->full[rp.slot], rp.ph);
    if (live) CloverStage<T, S * NCU, NCU>::run(ring + (size_t)rp.slot * 2 * NCU * TV + own, TV, v, o);
    __syncwarp();
    if (lane == 0) mbar_arrive(&bars->empty[rp.slot]);
    rp.advance(nslot);
    CloverPipe<T, NCU, S + 1, NS>::run(bars, ring, rp, nslot, TV, own, live, lane, v, o);
  }
};
template <typename T, int NCU, int NS>
struct CloverPipe<T, NCU, NS, NS> {
  static __device__ __forceinline__ void run(PipeBars*, const T2<T>*, RingPos&, const int, const int, const int, const bool,
                                             const int, const cx<T> (&)[12], cx<T> (&)[12]) {}
};

// ---- faces of a tile ------------------------------------------------------------------------------------
// The sites of one parity on the face l_mu = const of a tile are numbered by their other three coordinates:
//   mu = 0 : fidx = (l1 >> 1) + (b1/2) * (l2 + b2 * l3)      (l1's low bit is fixed by the parity)
//   mu >= 1: fidx = l0h + (b0/2) * (la + ba * lb),  (a, b) = the two directions of {1,2,3} other than mu
// TV / b_mu sites per parity.  A halo buffer for direction mu holds, with Nf = 2*TV/b_mu columns (parity-major):
//   F [12][Nf]  spinors of the +mu neighbour tile on its face l_mu = 0        (forward hops leaving the tile)
//   B [12][Nf]  spinors of the -mu neighbour tile on its face l_mu = b_mu - 1 (backward hops leaving the tile)
//   BU[NCU][Nf] links U_mu on that backward face
// stored as rows of PIPE_TV columns: buffer 0 in columns [0, Nf), buffer 1 in columns [Nf, 2 Nf).
template <int MU>
__device__ __forceinline__ int face_index(const int (&l)[4]) {   // 4x4x4x4 tile
  const int l0h = l[0] >> 1;
  if (MU == 0) return (l[1] >> 1) + 2 * (l[2] + 4 * l[3]);
  if (MU == 1) return l0h + 2 * (l[2] + 4 * l[3]);
  if (MU == 2) return l0h + 2 * (l[1] + 4 * l[3]);
  return l0h + 2 * (l[1] + 4 * l[2]);
}
// inverse: tile-local checkerboard index j of the face site (parity P, face index fidx, l_mu = lmu), 4x4x4x4 tile
__device__ __forceinline__ int face_site(const int mu, const int P, const int fidx, const int lmu) {
  const int lo = fidx & 1, mid = (fidx >> 1) & 3, hi = fidx >> 3;
  int l0, l1, l2, l3;
  if (mu == 0) {
    l2 = mid; l3 = hi; l0 = lmu;
    l1 = 2 * lo + ((P + l2 + l3 + lmu) & 1);
  } else {
    if (mu == 1) { l1 = lmu; l2 = mid; l3 = hi; }
    else if (mu == 2) { l1 = mid; l2 = lmu; l3 = hi; }
    else { l1 = mid; l2 = hi; l3 = lmu; }
    l0 = 2 * lo + ((P + l1 + l2 + l3) & 1);
  }
  return (l0 >> 1) + 2 * (l1 + 4 * (l2 + 4 * l3));
}

// both hops of direction MU for one site: links of the tile in ring stage `ub`, spinor tile `sp`, halo buffer `hb`
template <typename T, int RECON, int MU>
__device__ __forceinline__ void hop_pair(const Geom& g, const DwArgs<T>& a, const T2<T>* sp, const T2<T>* ub,
                                         const T2<T>* hb, const int p, const int j, const int (&l)[4], const int x3,
                                         const bool nonper, const T sg, cx<T> (&acc)[12]) {
  constexpr int NCU = (RECON == 12) ? 6 : 9;
  constexpr int TV = PIPE_TV, Nh = PIPE_NF / 2;
  const int q = 1 - p;
  const int l0h = l[0] >> 1;
  const int fq = q * Nh + face_index<MU>(l);
  constexpr int stride = MU == 1 ? 2 : (MU == 2 ? 8 : 32);   // index stride of direction MU (MU >= 1)
  // ---- forward: theta (1 - gamma_mu) U_mu(x) psi(x + mu)
  {
    const bool cr = (l[MU] == 3);
    int jn;
    if (MU == 0) jn = j - l0h + ((l[0] + 1) >> 1);
    else jn = j + stride;
    bool on = true;
    if (MU == 3 && nonper) on = !time_hop_blocked(g, x3, true);
    if (on) {
      const T2<T>* ps = cr ? hb + fq : sp + (q * 12) * TV + jn;
      hop_dir<T, RECON, MU, true, false>(ps, ub + (p * NCU) * TV + j, TV, TV, sg, a.has_theta, a.theta[MU], acc);
    }
  }
  // ---- backward: theta^* (1 + gamma_mu) U_mu(x - mu)^+ psi(x - mu)
  {
    const bool cr = (l[MU] == 0);
    int jn;
    if (MU == 0) jn = j - l0h + ((l[0] - 1) >> 1);
    else jn = j - stride;
    bool on = true;
    if (MU == 3 && nonper) on = !time_hop_blocked(g, x3, false);
    if (on) {
      const T2<T>* ps = cr ? hb + 12 * TV + fq : sp + (q * 12) * TV + jn;
      const T2<T>* us = cr ? hb + 24 * TV + fq : ub + (q * NCU) * TV + jn;
      hop_dir<T, RECON, MU, false, false>(ps, us, TV, TV, -sg, a.has_theta, a.theta[MU], acc);
    }
  }
}

template <typename T> __device__ __forceinline__ void cp_async_elem(T2<T>* dst, const T2<T>* src);
template <> __device__ __forceinline__ void cp_async_elem<double>(double2* dst, const double2* src) { cp_async_16(dst, src); }
template <> __device__ __forceinline__ void cp_async_elem<float>(float2* dst, const float2* src) { cp_async_8(dst, src); }

// halo of direction mu of the tile whose table row is `tab` -> buffer hb (layout above); lt = index of this
// loader thread.
template <typename T, int NCU>
__device__ __forceinline__ void halo_load(const Geom& g, const DwArgs<T>& a, const T2<T>* __restrict__ in,
                                          const int* __restrict__ tab, const int mu, T2<T>* hb, const int lt) {
  constexpr int TV = PIPE_TV, Nf = PIPE_NF, Nh = PIPE_NF / 2;
  const int tf = __ldg(tab + 2 * mu), tb = __ldg(tab + 2 * mu + 1);
  for (int u = lt; u < 3 * Nf; u += PIPE_HALO_THREADS) {
    const int kind = u / Nf;           // 0: F, 1: B, 2: BU
    const int f = u - kind * Nf;       // column: parity-major
    const int P = f >= Nh ? 1 : 0;
    const int jn = face_site(mu, P, f - P * Nh, kind == 0 ? 0 : 3);
    if (kind < 2) {
      const T2<T>* src = in + field_offset(g, 12, P, kind == 0 ? tf : tb, 0, jn);
      T2<T>* dst = hb + kind * 12 * TV + f;
#pragma unroll
      for (int c = 0; c < 12; c++) cp_async_elem<T>(dst + c * TV, src + c * TV);
    } else {
      const T2<T>* src = a.U + field_offset(g, 4 * NCU, P, tb, mu * NCU, jn);
      T2<T>* dst = hb + 24 * TV + f;
#pragma unroll
      for (int c = 0; c < NCU; c++) cp_async_elem<T>(dst + c * TV, src + c * TV);
    }
  }
}

template <typename T, int RECON, int DIAG>
__global__ void __launch_bounds__(PIPE_THREADS, 1)
dw_pipe_kernel(const Geom g, const DwArgs<T> a, const int nslot) {
  constexpr int nhb = pipe_nhb<T>();   // halo buffers: columns [0, PIPE_NF) and [PIPE_NF, PIPE_TV) of the rows of a pair
  constexpr int NCU = (RECON == 12) ? 6 : 9;
  constexpr int NSTC = (DIAG == DIAG_PRE) ? 36 / NCU : 0;   // clover stages per tile
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ double s_red[2][PIPE_CONS_WARPS];
  if (a.skip != nullptr && *a.skip != 0) return;  // CG finished: uniform early exit
  constexpr int TV = PIPE_TV;
  const int tid = threadIdx.x;
  const int lane = tid & 31;
  const int warp = tid >> 5;
  constexpr int NSPB = pipe_nspb<T>();
  T2<T>* sp0 = reinterpret_cast<T2<T>*>(smem_raw);  // NSPB x [2][12][TV] spinor tile
  T2<T>* ring = sp0 + NSPB * 24 * TV;               // nslot x [2][NCU][TV]
  T2<T>* halo = ring + nslot * 2 * NCU * TV;        // [24 + NCU][PIPE_TV]: both halo buffers
  PipeBars* bars = reinterpret_cast<PipeBars*>(halo + ((nhb + 1) / 2) * (24 + NCU) * TV);
  if (tid == 0) {
    for (int i = 0; i < NSPB; i++) {
      mbar_init(&bars->full_sp[i], 1);
      mbar_init(&bars->empty_sp[i], PIPE_CONS_WARPS);
    }
    for (int i = 0; i < nhb; i++) {
      mbar_init(&bars->full_h[i], PIPE_HALO_THREADS);
      mbar_init(&bars->empty_h[i], PIPE_CONS_WARPS);
    }
    for (int i = 0; i < nslot; i++) {
      mbar_init(&bars->full[i], 1);
      mbar_init(&bars->empty[i], PIPE_CONS_WARPS);
    }
    for (int i = 0; i < PIPE_TQ; i++) {
      mbar_init(&bars->tq_full[i], 1);
      mbar_init(&bars->tq_empty[i], PIPE_CONS_WARPS + PIPE_HALO_THREADS / 32);
    }
    mbar_fence_init();
  }
  __syncthreads();
  double nrm = 0.0;
  const int nrhs = a.nrhs > 1 ? a.nrhs : 1;
  // work unit u = (tile u / nsplit, right-hand sides [(u % nsplit) nper, + nper)): units of one tile are drawn one after
  // the other, so the CTAs that share a tile's links and clover blocks read them at about the same time (L2)
  const int nsplit = (a.nrhs > 1 && a.nsplit > 1) ? a.nsplit : 1;
  const int nper = nrhs / nsplit;
  const int NUNITS = g.ntiles * nsplit;
  const uint32_t stage_bytes = (uint32_t)(NCU * TV * sizeof(T2<T>));
  const uint32_t sp_bytes = (uint32_t)(12 * TV * sizeof(T2<T>));

  if (warp >= PIPE_CONS_WARPS) {
    setmaxnreg_dec<56>();
    if (warp == PIPE_CONS_WARPS) {
      // ------------------------------ producer: one lane feeds the ring ------------------------------
      if (lane == 0) {
        const uint64_t pol_once = policy_evict_first();
        RingPos rp = {0, 0u};
        int k = 0, kt = 0;
        int tile = blockIdx.x;   // a work unit; the host keeps gridDim.x <= the number of units
        int tile_after = next_tile(NUNITS, a.sched, tile);
        tq_push(bars, kt++, tile);
        while (tile >= 0) {
        // the halo warps run half a tile ahead of the arithmetic warps: they get the next index (or the end marker) now,
        // and the draw for the tile after that is in flight while this tile is streamed
        tq_push(bars, kt++, tile_after);
        const int tile_after2 = tile_after >= 0 ? next_tile(NUNITS, a.sched, tile_after) : -1;
        const int unit = tile, r0 = (unit % nsplit) * nper;
        {
        const int tile = unit / nsplit;
        for (int rhs = r0; rhs < r0 + nper; rhs++, k++) {   // the unit's right-hand sides back to back: links and clover
                                                       // blocks of the 2nd..nth pass come out of L2
          // spinor of pass kk (buffer kk % NSPB): its previous occupant, pass kk - NSPB, must have been released
          auto request_spinor = [&](const int kk, const int t, const int r) {
            const int b = kk % NSPB;
            if (kk >= NSPB) mbar_wait_relaxed(&bars->empty_sp[b], (uint32_t)((kk / NSPB - 1) & 1));
            mbar_arrive_expect_tx(&bars->full_sp[b], 2 * sp_bytes);
            for (int p = 0; p < 2; p++)
              bulk_g2s(sp0 + (b * 24 + p * 12) * TV, a.in + r * a.rhs_stride + field_offset(g, 12, p, t, 0, 0), sp_bytes,
                       &bars->full_sp[b]);
          };
          int next = tile, nr = rhs + 1;
          if (nr == r0 + nper) {
            next = tile_after >= 0 ? tile_after / nsplit : -1;
            nr = tile_after >= 0 ? (tile_after % nsplit) * nper : 0;
          }
          if (k == 0) request_spinor(0, tile, rhs);
          if (NSPB > 1 && next >= 0) request_spinor(k + 1, next, nr);   // a whole pass ahead
#pragma unroll 1
          for (int st = 0; st < 4 + NSTC; st++) {   // stage order: L0 L1 [H clover stages] L2 L3 [the rest]  (consumer loop below)
            constexpr int H = pipe_early_stages<T>(NSTC);
            int mu = -1, cs = -1;
            if (st < 2) mu = st;
            else if (st < 2 + H) cs = st - 2;
            else if (st < 4 + H) mu = st - H;
            else cs = st - 4;
            mbar_wait_relaxed(&bars->empty[rp.slot], rp.ph ^ 1u);
            mbar_arrive_expect_tx(&bars->full[rp.slot], 2 * stage_bytes);
            T2<T>* dst = ring + rp.slot * 2 * NCU * TV;
            for (int p = 0; p < 2; p++) {
              if (mu >= 0)
                bulk_g2s(dst + (p * NCU) * TV, a.U + field_offset(g, 4 * NCU, p, tile, mu * NCU, 0), stage_bytes,
                         &bars->full[rp.slot]);
              else if (rhs + 1 < r0 + nper)
                bulk_g2s(dst + (p * NCU) * TV, a.A + field_offset(g, 36, p, tile, cs * NCU, 0), stage_bytes,
                         &bars->full[rp.slot]);
              else   // clover blocks are read for the last time: evict-first keeps them from displacing spinors and links in L2
                bulk_g2s_hint(dst + (p * NCU) * TV, a.A + field_offset(g, 36, p, tile, cs * NCU, 0), stage_bytes,
                              &bars->full[rp.slot], pol_once);
            }
            rp.advance(nslot);
          }
          // one buffer: the spinor of the next pass is requested when this pass's hops have released the buffer
          if (NSPB == 1 && next >= 0) request_spinor(k + 1, next, nr);
        }
        }
        tile = tile_after;
        tile_after = tile_after2;
        }
      }
    } else {
      // ------------------------------ halo loaders: LDGSTS one stage ahead ----------------------------
      const int lt = tid - (PIPE_CONS_WARPS + 1) * 32;
      RingPos hp = {0, 0u};   // halo buffer ring
      for (int kt = 0;; kt++) {
      const int unit = tq_pop(bars, kt, lane);
      if (unit < 0) break;
      const int tile = unit / nsplit, r0 = (unit % nsplit) * nper;
      for (int rhs = r0; rhs < r0 + nper; rhs++) {
        const int* tab = g.tile_tab + (size_t)tile * TILE_TAB;
        const T2<T>* in_r = a.in + rhs * a.rhs_stride;
        for (int mu = 0; mu < 4; mu++) {
          mbar_wait_relaxed(&bars->empty_h[hp.slot], hp.ph ^ 1u);
          halo_load<T, NCU>(g, a, in_r, tab, mu, halo + (hp.slot >> 1) * (24 + NCU) * TV + (hp.slot & 1) * PIPE_NF, lt);
          cp_async_arrive_noinc(&bars->full_h[hp.slot]);
          hp.advance(nhb);
        }
      }
      }
    }
  } else {
    // ------------------------------ consumers: one thread per site ---------------------------------
    setmaxnreg_inc<216>();
    const int p = (tid >= TV) ? 1 : 0;
    const int j = tid - p * TV;
    int l[4];   // 4x4x4x4 tile: j = l0/2 + 2 (l1 + 4 (l2 + 4 l3))
    l[1] = (j >> 1) & 3;
    l[2] = (j >> 3) & 3;
    l[3] = j >> 5;
    l[0] = 2 * (j & 1) + ((p + l[1] + l[2] + l[3]) & 1);
    const bool nonper = (g.bc != LQCD_BC_PERIODIC);
    const T sg = a.dagger ? T(-1) : T(1);
    RingPos rp = {0, 0u};
    RingPos hp = {0, 0u};
    int k = 0;
    for (int kt = 0;; kt++) {
    const int unit = tq_pop(bars, kt, lane);
    if (unit < 0) break;
    const int tile = unit / nsplit, r0 = (unit % nsplit) * nper;
    for (int rhs = r0; rhs < r0 + nper; rhs++, k++) {
      // the time coordinate matters only where time is not periodic: no load (and no wait for it) on periodic lattices
      const int x3 = nonper ? __ldg(g.tile_tab + (size_t)tile * TILE_TAB + 8) + l[3] : 0;
      const bool live = !(nonper && frozen_slice(g, x3));
      cx<T> acc[12], v[12], res[12];
#pragma unroll
      for (int c = 0; c < 12; c++) acc[c] = cx<T>(0, 0);
      const T2<T>* sp = sp0 + (k % NSPB) * 24 * TV;
      mbar_wait(&bars->full_sp[k % NSPB], (uint32_t)((k / NSPB) & 1));
#define LQCD_HOP_STAGE(MU)                                                                                       \
      {                                                                                                          \
        const int b = hp.slot;                                                                                   \
        mbar_wait(&bars->full_h[b], hp.ph);                                                                      \
        mbar_wait(&bars->full[rp.slot], rp.ph);                                                                  \
        if (live)                                                                                                \
          hop_pair<T, RECON, MU>(g, a, sp, ring + rp.slot * 2 * NCU * TV, halo + (b >> 1) * (24 + NCU) * TV + (b & 1) * PIPE_NF, p, j, l, x3, \
                                 nonper, sg, acc);                                                               \
        __syncwarp();                                                                                            \
        if (lane == 0) {                                                                                         \
          mbar_arrive(&bars->empty[rp.slot]);                                                                    \
          mbar_arrive(&bars->empty_h[b]);                                                                        \
        }                                                                                                        \
        rp.advance(nslot);                                                                                       \
        hp.advance(nhb);                                                                                         \
      }
      // Stage order H0 H1 [early clover stages] H2 H3 [the other clover stages] (pipe_early_stages): clover stages
      // between the hop pairs give the halos lead, clover stages after the last hop give the next spinor tile lead.
      // With the clover term ONE accumulator serves both: acc = sum of hops - (1/k) A psi, result = -k acc,
      // so that no second 12-component register set is live during the hops.
      const T2<T>* sv = sp + (p * 12) * TV + j;
      LQCD_HOP_STAGE(0)
      LQCD_HOP_STAGE(1)
      if (DIAG == DIAG_PRE) {
        const T s = T(-1) / a.k;
        if (live) {
#pragma unroll
          for (int c = 0; c < 6; c++) {
            T2<T> w = sv[c * TV];
            v[c] = cx<T>(s * w.x, s * w.y);
          }
          if (a.tm != T(0)) add_twist<T, 0, 6>(a.tm, v, acc);   // acc carries -(1/k) (A + i tm gamma5) psi
        }
        CloverPipe<T, NCU, 0, pipe_early_stages<T>(NSTC)>::run(bars, ring, rp, nslot, TV, (p * NCU) * TV + j, live, lane, v, acc);
      }
      LQCD_HOP_STAGE(2)
      LQCD_HOP_STAGE(3)
#undef LQCD_HOP_STAGE
      if (live) {
        if (DIAG == DIAG_PRE) {
          const T s = T(-1) / a.k;
#pragma unroll
          for (int c = 6; c < 12; c++) {
            T2<T> w = sv[c * TV];
            v[c] = cx<T>(s * w.x, s * w.y);
          }
          if (a.tm != T(0)) add_twist<T, 6, 12>(a.tm, v, acc);
        } else {
#pragma unroll
          for (int c = 0; c < 12; c++) {
            T2<T> w = sv[c * TV];
            v[c] = cx<T>(w.x, w.y);
          }
        }
      }
      // (pipe.cuh: release_fence.  The ring and halo releases above go without it: their refills come from DRAM / L2 a
      // microsecond after the arrive, and every value loaded from a slot feeds the stage's own arithmetic; a fence per
      // stage costs 1.2 % at 48^3 x 96.)
      release_fence();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->empty_sp[k % NSPB]);   // spinor tile no longer needed: the next but NSPB-1 may land
      if (DIAG == DIAG_PRE) {
        CloverPipe<T, NCU, pipe_early_stages<T>(NSTC), NSTC>::run(bars, ring, rp, nslot, TV, (p * NCU) * TV + j, live, lane, v, acc);
        if (live) {
#pragma unroll
          for (int c = 0; c < 12; c++) res[c] = cx<T>(-a.k * acc[c].re, -a.k * acc[c].im);
        }
      } else if (live) {
#pragma unroll
        for (int c = 0; c < 12; c++) res[c] = cx<T>(fma(-a.k, acc[c].re, v[c].re), fma(-a.k, acc[c].im, v[c].im));
        if (a.tm != T(0)) add_twist<T, 0, 12>(a.tm, v, res);
      }
      if (!live) {
#pragma unroll
        for (int c = 0; c < 12; c++) res[c] = cx<T>(0, 0);
      }
      // epilogue (same three variants as dw_kernel)
      const size_t ooff = field_offset(g, 12, p, tile, 0, j) + (size_t)(rhs * a.rhs_stride);
      if (a.epi == EPI_AXPY_NORM) {
        const T al = (T)a.alpha[(size_t)rhs * a.alpha_stride];
        T2<T>* rq = a.r + ooff;
#pragma unroll
        for (int c = 0; c < 12; c++) {
          T2<T> rv = rq[c * TV];
          cx<T> w(fma(-al, res[c].re, rv.x), fma(-al, res[c].im, rv.y));
          st<T>(rq + c * TV, w);
          nrm += (double)w.re * (double)w.re + (double)w.im * (double)w.im;
        }
      } else {
        T2<T>* op = a.out + ooff;
#pragma unroll
        for (int c = 0; c < 12; c++) st<T>(op + c * TV, res[c]);
        if (a.epi == EPI_STORE_NORM) {
#pragma unroll
          for (int c = 0; c < 12; c++) nrm += (double)res[c].re * (double)res[c].re + (double)res[c].im * (double)res[c].im;
        }
      }
      if (a.epi != EPI_STORE) {
        // one partial sum per (right-hand side, tile), reduced in a fixed order: the result does not depend on which
        // CTA happened to draw the tile.  s_red alternates between two rows, so one named barrier per pass is enough.
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nrm += __shfl_xor_sync(0xffffffffu, nrm, o);
        if (lane == 0) s_red[k & 1][warp] = nrm;
        asm volatile("bar.sync 1, %0;" ::"n"(PIPE_CONS_WARPS * 32) : "memory");
        if (tid == 0) {
          double s = 0;
          for (int w = 0; w < PIPE_CONS_WARPS; w++) s += s_red[k & 1][w];
          a.partial[(size_t)rhs * g.ntiles + tile] = s;
        }
        nrm = 0.0;
      }
    }
    }
  }
  if (a.sched != nullptr) {   // the last CTA to finish puts the scheduler's counters back to zero for the next launch
    if (tid == 0) {           // (thread 0 has seen the end-of-tiles marker, so this CTA's last draw is behind it)
      __threadfence();
      if (atomicAdd(a.sched + 1, 1u) == gridDim.x - 1) {
        a.sched[0] = 0u;
        a.sched[1] = 0u;
        __threadfence();
      }
    }
  }
}

// =====================================================================================================
// Half-lattice version of the pipeline kernel (output parity P = a.parity): the two passes of the even-odd operator
// (D8:  tmp_o = A_oo^-1 H_oe in_e  [DIAG_POST],   out_e = A_ee in_e - kappa^2 H_eo tmp_o  [DIAG_PRE]).
// A tile has only 128 output sites, so the eight arithmetic warps split the WORK of a site instead of the sites:
//   * hops: warps 0-3 ("group F") take the forward hop of every direction, warps 4-7 ("group B") the backward hop of
//     the same site -- disjoint operands (U_mu(x), psi(x+mu) against U_mu(x-mu), psi(x-mu)), twelve accumulators each;
//   * after the last hop the groups swap halves through the (then dead) input-spinor buffer: F ends up with the
//     complete upper chirality (components 0-5), B with the lower one (6-11);
//   * the packed 6x6 blocks are block-diagonal in chirality: F multiplies with A+ (clover stages 0, 1), B with A-
//     (stages 2, 3), and each group writes its six components.  No further exchange.
// Stage order L0 L1 L2 L3 C C C C (DIAG_POST needs the complete hop sum before the block multiply); three halo buffers of
// 32 columns (only the input parity's face sites are needed) give every halo two stages of lead.  Per tile the kernel
// streams both parities of the links (all of them are used: forward hops take the links of the output parity, backward
// hops those of the input parity), one parity of the input spinor, of the self spinor (DIAG_PRE) and of the blocks.
// =====================================================================================================
#ifndef HALF_NHB32
#define HALF_NHB32 4
#endif
enum { HALF_NF = 32, HALF_CLV_ROWS = 9 };
// halo buffers of the half-lattice kernel (32 columns each): three in fp64 (all that fits), four in fp32 -- every halo
// then has three stages of lead and halo rows have the stride of tile rows (D^ fp32 at 32^3 x 64 with 3 / 4 / 5 / 6
// buffers: 0.441 / 0.422 / 0.437 / 0.434 ms)
template <typename T> __host__ __device__ constexpr int half_nhb() { return sizeof(T) == 4 ? HALF_NHB32 : 3; }
template <typename T> __host__ __device__ constexpr int half_hs() { return half_nhb<T>() * HALF_NF; }

template <typename T, int NCU>
__device__ __forceinline__ void halo_load_half(const Geom& g, const DwArgs<T>& a, const int* __restrict__ tab, const int mu,
                                               const int q, T2<T>* hb, const int lt) {
  constexpr int TV = PIPE_TV;
  const int tf = __ldg(tab + 2 * mu), tb = __ldg(tab + 2 * mu + 1);
  for (int u = lt; u < 3 * HALF_NF; u += PIPE_HALO_THREADS) {
    const int kind = u / HALF_NF;      // 0: F, 1: B, 2: BU
    const int f = u - kind * HALF_NF;  // face index of the parity-q site
    const int jn = face_site(mu, q, f, kind == 0 ? 0 : 3);
    if (kind < 2) {
      const T2<T>* src = a.in + field_offset(g, 12, q, kind == 0 ? tf : tb, 0, jn);
      T2<T>* dst = hb + kind * 12 * half_hs<T>() + f;
#pragma unroll
      for (int c = 0; c < 12; c++) cp_async_elem<T>(dst + c * half_hs<T>(), src + c * TV);
    } else {
      const T2<T>* src = a.U + field_offset(g, 4 * NCU, q, tb, mu * NCU, jn);
      T2<T>* dst = hb + 24 * half_hs<T>() + f;
#pragma unroll
      for (int c = 0; c < NCU; c++) cp_async_elem<T>(dst + c * half_hs<T>(), src + c * TV);
    }
  }
}

// one hop of direction MU for one output site: FWD (group F) or backward (group B)
template <typename T, int RECON, int MU, bool FWD>
__device__ __forceinline__ void hop_one(const Geom& g, const DwArgs<T>& a, const T2<T>* sp_in, const T2<T>* ub, const T2<T>* hb,
                                        const int p, const int j, const int (&l)[4], const int x3, const bool nonper, const T sg,
                                        cx<T> (&acc)[12]) {
  constexpr int NCU = (RECON == 12) ? 6 : 9;
  constexpr int TV = PIPE_TV;
  const int q = 1 - p;
  const int l0h = l[0] >> 1;
  const int fidx = face_index<MU>(l);
  constexpr int stride = MU == 1 ? 2 : (MU == 2 ? 8 : 32);
  if (MU == 3 && nonper && time_hop_blocked(g, x3, FWD)) return;
  if (FWD) {
    const bool cr = (l[MU] == 3);
    int jn;
    if (MU == 0) jn = j - l0h + ((l[0] + 1) >> 1);
    else jn = j + stride;
    const T2<T>* ps = cr ? hb + fidx : sp_in + jn;
    hop_dir<T, RECON, MU, true, false>(ps, ub + (p * NCU) * TV + j, cr ? half_hs<T>() : TV, TV, sg, a.has_theta, a.theta[MU], acc);
  } else {
    const bool cr = (l[MU] == 0);
    int jn;
    if (MU == 0) jn = j - l0h + ((l[0] - 1) >> 1);
    else jn = j - stride;
    const T2<T>* ps = cr ? hb + 12 * half_hs<T>() + fidx : sp_in + jn;
    const T2<T>* us = cr ? hb + 24 * half_hs<T>() + fidx : ub + (q * NCU) * TV + jn;
    hop_dir<T, RECON, MU, false, false>(ps, us, cr ? half_hs<T>() : TV, cr ? half_hs<T>() : TV, -sg, a.has_theta, a.theta[MU], acc);
  }
}

template <typename T, int RECON, int DIAG>
__global__ void __launch_bounds__(PIPE_THREADS, 1)
dw_pipe_half_kernel(const Geom g, const DwArgs<T> a, const int nslot) {
  constexpr int NCU = (RECON == 12) ? 6 : 9;
  constexpr int NSTC = (DIAG == DIAG_ONE) ? 0 : 4;          // block stages per tile: two per chirality, 9 rows each
  constexpr bool SELF = (DIAG != DIAG_POST);                // the self spinor is staged too
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ double s_red[2][PIPE_CONS_WARPS];
  if (a.skip != nullptr && *a.skip != 0) return;  // CG finished: uniform early exit
  constexpr int TV = PIPE_TV;
  const int tid = threadIdx.x;
  const int lane = tid & 31;
  const int warp = tid >> 5;
  const int p = a.parity, q = 1 - p;
  constexpr int NSPB = pipe_nspb<T>();                      // spinor buffers (fp32: two)
  constexpr int SPW = SELF ? 24 : 12;                       // rows of one spinor buffer:
  T2<T>* sp_base = reinterpret_cast<T2<T>*>(smem_raw);      //   [12][TV] input spinor, parity q; exchange area after the hops
                                                            //   [12][TV] self spinor, parity p (SELF)
  T2<T>* ring = sp_base + NSPB * SPW * TV;                  // nslot x [2][NCU][TV] (block stages use the first 9 rows)
  T2<T>* halo = ring + nslot * 2 * NCU * TV;                // [24 + NCU][half_hs<T>()]: halo buffers of 32 columns
  PipeBars* bars = reinterpret_cast<PipeBars*>(halo + (24 + NCU) * half_hs<T>());
  if (tid == 0) {
    for (int i = 0; i < NSPB; i++) {
      mbar_init(&bars->full_sp[i], 1);
      mbar_init(&bars->empty_sp[i], PIPE_CONS_WARPS);
    }
    for (int i = 0; i < half_nhb<T>(); i++) {
      mbar_init(&bars->full_h[i], PIPE_HALO_THREADS);
      mbar_init(&bars->empty_h[i], PIPE_CONS_WARPS);
    }
    for (int i = 0; i < nslot; i++) {
      mbar_init(&bars->full[i], 1);
      mbar_init(&bars->empty[i], PIPE_CONS_WARPS);
    }
    for (int i = 0; i < PIPE_TQ; i++) {
      mbar_init(&bars->tq_full[i], 1);
      mbar_init(&bars->tq_empty[i], PIPE_CONS_WARPS + PIPE_HALO_THREADS / 32);
    }
    mbar_fence_init();
  }
  __syncthreads();
  const int NUNITS = g.ntiles;
  const uint32_t link_bytes = (uint32_t)(NCU * TV * sizeof(T2<T>));
  const uint32_t clv_bytes = (uint32_t)(HALF_CLV_ROWS * TV * sizeof(T2<T>));
  const uint32_t sp_bytes = (uint32_t)(12 * TV * sizeof(T2<T>));

  if (warp >= PIPE_CONS_WARPS) {
    setmaxnreg_dec<56>();
    if (warp == PIPE_CONS_WARPS) {
      // ------------------------------ producer ------------------------------
      if (lane == 0) {
        const uint64_t pol_once = policy_evict_first();
        RingPos rp = {0, 0u};
        int k = 0, kt = 0;
        int tile = blockIdx.x;
        int tile_after = next_tile(NUNITS, a.sched, tile);
        tq_push(bars, kt++, tile);
        // spinors of the kk-th tile of this CTA (buffer kk % NSPB): the buffer's previous occupant, tile kk - NSPB, must
        // have been released (after its exchange)
        auto load_spinors = [&](const int kk, const int t) {
          const int b = kk % NSPB;
          if (kk >= NSPB) mbar_wait_relaxed(&bars->empty_sp[b], (uint32_t)((kk / NSPB - 1) & 1));
          T2<T>* sp_in = sp_base + b * SPW * TV;
          mbar_arrive_expect_tx(&bars->full_sp[b], (SELF ? 2 : 1) * sp_bytes);
          bulk_g2s(sp_in, a.in + field_offset(g, 12, q, t, 0, 0), sp_bytes, &bars->full_sp[b]);
          if (SELF) bulk_g2s(sp_in + 12 * TV, a.self + field_offset(g, 12, p, t, 0, 0), sp_bytes, &bars->full_sp[b]);
        };
        load_spinors(0, tile);
        while (tile >= 0) {
          tq_push(bars, kt++, tile_after);
          const int tile_after2 = tile_after >= 0 ? next_tile(NUNITS, a.sched, tile_after) : -1;
          if (NSPB > 1 && tile_after >= 0) load_spinors(k + 1, tile_after);   // a whole tile ahead
#pragma unroll 1
          for (int st = 0; st < 4 + NSTC; st++) {   // L0 L1 L2 L3 C0 C1 C2 C3
            mbar_wait_relaxed(&bars->empty[rp.slot], rp.ph ^ 1u);
            T2<T>* dst = ring + rp.slot * 2 * NCU * TV;
            if (st < 4) {
              mbar_arrive_expect_tx(&bars->full[rp.slot], 2 * link_bytes);
              for (int pp = 0; pp < 2; pp++)
                bulk_g2s(dst + (pp * NCU) * TV, a.U + field_offset(g, 4 * NCU, pp, tile, st * NCU, 0), link_bytes, &bars->full[rp.slot]);
            } else {   // blocks are read exactly once per application: evict-first
              mbar_arrive_expect_tx(&bars->full[rp.slot], clv_bytes);
              bulk_g2s_hint(dst, a.A + field_offset(g, 36, p, tile, (st - 4) * HALF_CLV_ROWS, 0), clv_bytes, &bars->full[rp.slot], pol_once);
            }
            rp.advance(nslot);
          }
          if (NSPB == 1 && tile_after >= 0) load_spinors(k + 1, tile_after);   // one buffer: once this tile has released it
          k++;
          tile = tile_after;
          tile_after = tile_after2;
        }
      }
    } else {
      // ------------------------------ halo loaders ----------------------------
      const int lt = tid - (PIPE_CONS_WARPS + 1) * 32;
      RingPos hp = {0, 0u};
      for (int kt = 0;; kt++) {
        const int tile = tq_pop(bars, kt, lane);
        if (tile < 0) break;
        const int* tab = g.tile_tab + (size_t)tile * TILE_TAB;
        for (int mu = 0; mu < 4; mu++) {
          mbar_wait_relaxed(&bars->empty_h[hp.slot], hp.ph ^ 1u);
          halo_load_half<T, NCU>(g, a, tab, mu, q, halo + hp.slot * HALF_NF, lt);
          cp_async_arrive_noinc(&bars->full_h[hp.slot]);
          hp.advance(half_nhb<T>());
        }
      }
    }
  } else {
    // ------------------------------ arithmetic ---------------------------------
    setmaxnreg_inc<216>();
    const int grp = warp >> 2;          // 0: forward hops, upper chirality; 1: backward hops, lower chirality
    const int j = tid & (TV - 1);
    int l[4];
    l[1] = (j >> 1) & 3;
    l[2] = (j >> 3) & 3;
    l[3] = j >> 5;
    l[0] = 2 * (j & 1) + ((p + l[1] + l[2] + l[3]) & 1);
    const bool nonper = (g.bc != LQCD_BC_PERIODIC);
    const T sg = a.dagger ? T(-1) : T(1);
    RingPos rp = {0, 0u};
    RingPos hp = {0, 0u};
    double nrm = 0.0;
    int k = 0;
    for (int kt = 0;; kt++, k++) {
      const int tile = tq_pop(bars, kt, lane);
      if (tile < 0) break;
      const int x3 = nonper ? __ldg(g.tile_tab + (size_t)tile * TILE_TAB + 8) + l[3] : 0;   // (see dw_pipe_kernel)
      const bool live = !(nonper && frozen_slice(g, x3));
      cx<T> acc[12];
#pragma unroll
      for (int c = 0; c < 12; c++) acc[c] = cx<T>(0, 0);
      T2<T>* sp_in = sp_base + (k % NSPB) * SPW * TV;
      const T2<T>* sp_self = sp_in + 12 * TV;
      mbar_wait(&bars->full_sp[k % NSPB], (uint32_t)((k / NSPB) & 1));
#define LQCD_HALF_HOP(MU)                                                                                              \
      {                                                                                                                \
        const int b = hp.slot;                                                                                         \
        mbar_wait(&bars->full_h[b], hp.ph);                                                                            \
        mbar_wait(&bars->full[rp.slot], rp.ph);                                                                        \
        if (live) {                                                                                                    \
          if (grp == 0) hop_one<T, RECON, MU, true>(g, a, sp_in, ring + rp.slot * 2 * NCU * TV, halo + b * HALF_NF, p, j, l, x3, nonper, sg, acc);  \
          else hop_one<T, RECON, MU, false>(g, a, sp_in, ring + rp.slot * 2 * NCU * TV, halo + b * HALF_NF, p, j, l, x3, nonper, sg, acc);          \
        }                                                                                                              \
        release_fence();                                                                                               \
        __syncwarp();                                                                                                  \
        if (lane == 0) {                                                                                               \
          mbar_arrive(&bars->empty[rp.slot]);                                                                          \
          mbar_arrive(&bars->empty_h[b]);                                                                              \
        }                                                                                                              \
        rp.advance(nslot);                                                                                             \
        hp.advance(half_nhb<T>());                                                                                          \
      }
      LQCD_HALF_HOP(0)
      LQCD_HALF_HOP(1)
      LQCD_HALF_HOP(2)
      LQCD_HALF_HOP(3)
#undef LQCD_HALF_HOP
      // swap halves through the input-spinor buffer (no hop reads it any more): rows 0-5 <- F's lower components,
      // rows 6-11 <- B's upper components; then F adds B's upper half, B adds F's lower half.  From here on a thread
      // holds ITS chirality in elements 0-5 of its arrays (register arrays want compile-time indices; the group only
      // enters through addresses and selects).
      cx<T> m[12], v[12];   // m: hop sums, later the accumulator of the block multiply; v: the vector the blocks act on
      asm volatile("bar.sync 2, %0;" ::"n"(PIPE_CONS_WARPS * 32) : "memory");
      {
        T2<T>* x = sp_in + (grp == 0 ? 0 : 6) * TV + j;
#pragma unroll
        for (int c = 0; c < 6; c++) {
          const cx<T> send(grp == 0 ? acc[6 + c].re : acc[c].re, grp == 0 ? acc[6 + c].im : acc[c].im);
          m[c] = cx<T>(grp == 0 ? acc[c].re : acc[6 + c].re, grp == 0 ? acc[c].im : acc[6 + c].im);
          st<T>(x + c * TV, send);
        }
      }
      // these generic-proxy stores share their addresses with the next tile's bulk copy (async proxy): without the
      // proxy fence the copy may overtake them (seen as a few garbage tiles per launch on a full grid)
      fence_proxy_async();
      asm volatile("bar.sync 2, %0;" ::"n"(PIPE_CONS_WARPS * 32) : "memory");
      {
        const T2<T>* x = sp_in + (grp == 0 ? 6 : 0) * TV + j;
#pragma unroll
        for (int c = 0; c < 6; c++) {
          const T2<T> w = x[c * TV];
          m[c] = cx<T>(m[c].re + w.x, m[c].im + w.y);
        }
      }
      // this group's six components of the self spinor (before the buffers are released)
      if (SELF) {
        const T sc = (DIAG == DIAG_PRE) ? T(-1) / a.k : T(1);
        const T2<T>* sv = sp_self + (grp == 0 ? 0 : 6) * TV + j;
#pragma unroll
        for (int c = 0; c < 6; c++) {
          const T2<T> w = sv[c * TV];
          v[c] = cx<T>(sc * w.x, sc * w.y);
        }
      }
      release_fence();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->empty_sp[k % NSPB]);   // both spinor buffers may be overwritten
      if (NSTC > 0) {
        // DIAG_PRE: m = hops - (1/k) A self, result = -k m;  DIAG_POST: result = B (hops)
        if (DIAG == DIAG_POST) {
#pragma unroll
          for (int c = 0; c < 6; c++) { v[c] = m[c]; m[c] = cx<T>(0, 0); }
        }
        // the packing of the two chiral blocks is the same: the stage of this group's chirality is processed as
        // "chirality 0" on elements 0-5
#define LQCD_HALF_CLV(S)                                                                                               \
        {                                                                                                              \
          mbar_wait(&bars->full[rp.slot], rp.ph);                                                                      \
          if (live && grp == (S) / 2) CloverStage<T, ((S) & 1) * HALF_CLV_ROWS, HALF_CLV_ROWS>::run(ring + rp.slot * 2 * NCU * TV + j, TV, v, m);  \
          release_fence();                                                                                             \
          __syncwarp();                                                                                                \
          if (lane == 0) mbar_arrive(&bars->empty[rp.slot]);                                                           \
          rp.advance(nslot);                                                                                           \
        }
        LQCD_HALF_CLV(0)
        LQCD_HALF_CLV(1)
        LQCD_HALF_CLV(2)
        LQCD_HALF_CLV(3)
#undef LQCD_HALF_CLV
      }
      cx<T> res[6];
#pragma unroll
      for (int c = 0; c < 6; c++) {
        if (!live) res[c] = cx<T>(0, 0);
        else if (DIAG == DIAG_PRE) res[c] = cx<T>(-a.k * m[c].re, -a.k * m[c].im);
        else if (DIAG == DIAG_POST) res[c] = m[c];
        else res[c] = cx<T>(fma(-a.k, m[c].re, v[c].re), fma(-a.k, m[c].im, v[c].im));
      }
      // epilogue on this group's six components
      const size_t ooff = field_offset(g, 12, p, tile, grp == 0 ? 0 : 6, j);
      if (a.epi == EPI_AXPY_NORM) {
        const T al = (T)(*a.alpha);
        T2<T>* rq = a.r + ooff;
#pragma unroll
        for (int c = 0; c < 6; c++) {
          T2<T> rv = rq[c * TV];
          cx<T> w(fma(-al, res[c].re, rv.x), fma(-al, res[c].im, rv.y));
          st<T>(rq + c * TV, w);
          nrm += (double)w.re * (double)w.re + (double)w.im * (double)w.im;
        }
      } else {
        T2<T>* op = a.out + ooff;
#pragma unroll
        for (int c = 0; c < 6; c++) {
          st<T>(op + c * TV, res[c]);
          if (a.epi == EPI_STORE_NORM) nrm += (double)res[c].re * (double)res[c].re + (double)res[c].im * (double)res[c].im;
        }
      }
      if (a.epi != EPI_STORE) {   // one partial sum per tile, fixed order (see dw_pipe_kernel)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nrm += __shfl_xor_sync(0xffffffffu, nrm, o);
        if (lane == 0) s_red[k & 1][warp] = nrm;
        asm volatile("bar.sync 1, %0;" ::"n"(PIPE_CONS_WARPS * 32) : "memory");
        if (tid == 0) {
          double s = 0;
          for (int w = 0; w < PIPE_CONS_WARPS; w++) s += s_red[k & 1][w];
          a.partial[tile] = s;
        }
        nrm = 0.0;
      }
    }
  }
  if (a.sched != nullptr) {
    if (tid == 0) {
      __threadfence();
      if (atomicAdd(a.sched + 1, 1u) == gridDim.x - 1) {
        a.sched[0] = 0u;
        a.sched[1] = 0u;
        __threadfence();
      }
    }
  }
}

// LQCD_DW_MODE selects the kernel of the full-lattice operator: stream = persistent one-thread-per-site CTAs;
// split = the same with one parity of a tile per 128-thread CTA; direct = one CTA per tile (hardware scheduling);
// pipe = the warp-specialised shared-memory pipeline where it applies.
enum { MODE_STREAM = 0, MODE_DIRECT = 1, MODE_PIPE = 2, MODE_SPLIT = 3 };
static int g_mode = -1;
static int mode_from_name(const char* e) {
  if (!e) return -1;
  if (!strcmp(e, "pipe")) return MODE_PIPE;
  if (!strcmp(e, "stream")) return MODE_STREAM;
  if (!strcmp(e, "split")) return MODE_SPLIT;
  if (!strcmp(e, "direct")) return MODE_DIRECT;
  return -1;
}
static int dw_mode() {
  if (g_mode < 0) {
    g_mode = mode_from_name(getenv("LQCD_DW_MODE"));
    // default: the pipeline where it applies (full lattice, 128-site tiles), else persistent one-thread-per-site
    if (g_mode < 0) g_mode = MODE_PIPE;
  }
  return g_mode;
}
// lqcd_set_option("pipe_grid", n): at most n CTAs for the pipeline kernel (0 = one per SM).  A test hook: with one or
// two CTAs every CTA walks hundreds of tiles, i.e. every slot and phase of its mbarrier rings many times over.
static int g_pipe_grid = 0;
bool dw_set_pipe_grid(int n) {
  if (n < 0) return false;
  g_pipe_grid = n;
  return true;
}
bool dw_set_mode(const char* name) {
  const int m = mode_from_name(name);
  if (m < 0) return false;
  g_mode = m;
  return true;
}
static int env_int(const char* name, int dflt) {
  const char* e = getenv(name);
  return e ? atoi(e) : dflt;
}
// LQCD_SCHED=static: tiles b, b + grid, ... per CTA instead of the global tile counter (an experiment switch)
static bool pipe_dynamic() {
  static int dyn = -1;
  if (dyn < 0) {
    const char* e = getenv("LQCD_SCHED");
    dyn = (e && !strcmp(e, "static")) ? 0 : 1;
  }
  return dyn == 1;
}
// ---- host side: configuration of the persistent kernel ------------------------------------------------
struct PipeCfg {
  bool use;
  int grid, nslot;
  size_t smem;
};
template <typename T>
static PipeCfg pipe_config(const Geom& g, int recon, int diag, int parity) {
  PipeCfg c = {false, 0, 0, 0};
  if (dw_mode() != MODE_PIPE || parity >= 0 || diag == DIAG_POST) return c;
  if (g.b[0] != 4 || g.b[1] != 4 || g.b[2] != 4 || g.b[3] != 4 || g.tile_tab == nullptr) return c;   // PIPE_TV, PIPE_NF
  const int ncu = recon == 12 ? 6 : 9;
  const size_t sp = (size_t)pipe_nspb<T>() * 24 * g.TV * sizeof(T2<T>);
  const size_t slot = (size_t)2 * ncu * g.TV * sizeof(T2<T>);
  const size_t halo = (size_t)((pipe_nhb<T>() + 1) / 2) * (24 + ncu) * PIPE_TV * sizeof(T2<T>);   // pairs of buffers
  const size_t budget = (size_t)g.smem_optin - 256;   // 256 B: the kernel's static shared memory
  if (budget < sp + halo + sizeof(PipeBars) + 2 * slot) return c;
  int nslot = (int)((budget - sp - halo - sizeof(PipeBars)) / slot);
  if (nslot > 4) nslot = 4;   // measured: a deeper ring only lets the stream run further ahead of the halos (fp32, with two
                              // spinor buffers: 4 / 6 / 8 slots 1.58 / 1.68 / 1.74 ms at 48^3 x 96)
  const int e = env_int("LQCD_NSLOT", nslot);
  if (e >= 2 && e <= nslot) nslot = e;
  c.use = true;
  c.nslot = nslot;
  c.smem = sp + (size_t)nslot * slot + halo + sizeof(PipeBars);
  c.grid = g.sm_count;
  if (g_pipe_grid > 0 && g_pipe_grid < c.grid) c.grid = g_pipe_grid;
  if (c.grid > g.ntiles) c.grid = g.ntiles;
  return c;
}

// half-lattice pipeline (even-odd passes): DIAG_PRE / DIAG_POST on 4x4x4x4 tiles
template <typename T>
static PipeCfg pipe_half_config(const Geom& g, int recon, int diag, int parity) {
  PipeCfg c = {false, 0, 0, 0};
  if (dw_mode() != MODE_PIPE || parity < 0 || diag == DIAG_ONE) return c;
  if (g.b[0] != 4 || g.b[1] != 4 || g.b[2] != 4 || g.b[3] != 4 || g.tile_tab == nullptr) return c;
  if (env_int("LQCD_EO_PIPE", 1) == 0) return c;   // experiment switch: the one-thread-per-site kernel instead
  const int ncu = recon == 12 ? 6 : 9;
  const size_t sp = (size_t)pipe_nspb<T>() * (diag == DIAG_POST ? 12 : 24) * g.TV * sizeof(T2<T>);
  const size_t slot = (size_t)2 * ncu * g.TV * sizeof(T2<T>);
  const size_t halo = (size_t)(24 + ncu) * half_hs<T>() * sizeof(T2<T>);
  const size_t budget = (size_t)g.smem_optin - 256;
  if (budget < sp + halo + sizeof(PipeBars) + 2 * slot) return c;
  int nslot = (int)((budget - sp - halo - sizeof(PipeBars)) / slot);
  // ring depth: with two spinor buffers (fp32) the producer is no longer held back by the spinor release and a deeper
  // ring pays: D^ fp32 at 32^3 x 64 with 4 / 5 / 6 / 7 / 8 slots 0.462 / 0.440 / 0.439 / 0.454 / 0.458 ms
  { const int cap = pipe_nspb<T>() > 1 ? 6 : 4; if (nslot > cap) nslot = cap; }
  const int e = env_int("LQCD_NSLOT", nslot);
  if (e >= 2 && e <= nslot) nslot = e;
  c.use = true;
  c.nslot = nslot;
  c.smem = sp + (size_t)nslot * slot + halo + sizeof(PipeBars);
  c.grid = g.sm_count;
  if (g_pipe_grid > 0 && g_pipe_grid < c.grid) c.grid = g_pipe_grid;
  if (c.grid > g.ntiles) c.grid = g.ntiles;
  return c;
}

static thread_local unsigned int* t_sched_base = nullptr;
static thread_local int t_sched_pairs = 0, t_sched_next = 0;
void dw_set_sched_pool(unsigned int* base, int npairs) {
  t_sched_base = npairs > 0 ? base : nullptr;
  t_sched_pairs = npairs;
  t_sched_next = 0;
}
static unsigned int* sched_slot(const Geom& g) {
  if (t_sched_base != nullptr && g.sched != nullptr && pipe_dynamic()) return t_sched_base + 2 * (t_sched_next++ % t_sched_pairs);
  static std::atomic<unsigned> launch_no(0);
  // one pair of scheduler counters per launch in flight (a pool of SCHED_SLOTS pairs owned by the geometry, handed out
  // round-robin): launches of the same geometry running concurrently on different streams do not share a counter
  return (g.sched != nullptr && pipe_dynamic()) ? g.sched + 2 * (launch_no++ % SCHED_SLOTS) : nullptr;
}

template <typename T, int RECON, int DIAG>
static cudaError_t launch_pipe_half(const Geom& g, const DwArgs<T>& a, const PipeCfg& c, cudaStream_t s) {
  cudaError_t e = cudaFuncSetAttribute(dw_pipe_half_kernel<T, RECON, DIAG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);
  if (e != cudaSuccess) return e;
  DwArgs<T> b = a;
  b.sched = sched_slot(g);
  dw_pipe_half_kernel<T, RECON, DIAG><<<c.grid, PIPE_THREADS, c.smem, s>>>(g, b, c.nslot);
  count_launch();
  return cudaGetLastError();
}

template <typename T, int RECON, int DIAG>
static cudaError_t launch_pipe(const Geom& g, const DwArgs<T>& a, const PipeCfg& c, cudaStream_t s) {
  // the attribute is per function AND per device: set it on every launch (a host-side call of about a microsecond) rather
  // than cache it in a process-wide variable that another device or thread would not see
  cudaError_t e = cudaFuncSetAttribute(dw_pipe_kernel<T, RECON, DIAG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);
  if (e != cudaSuccess) return e;
  DwArgs<T> b = a;
  b.sched = sched_slot(g);
  // several right-hand sides: every tile becomes nsplit work units of nrhs / nsplit columns each.  148 CTAs each on a
  // tile of its own keep 65 MB of links and clover blocks in flight between the passes, more than L2 holds next to the
  // spinor streams (measured: 12.5 GB of DRAM reads per column, 0 % gain); with the columns of a tile shared out over
  // neighbouring CTAs the set shrinks by nsplit and a tile's links come from DRAM once.
  int grid = c.grid;
  b.nsplit = 1;
  if (a.nrhs > 1) {
    int want = env_int("LQCD_NSPLIT", 4);
    if (want < 1) want = 1;
    while (want > 1 && a.nrhs % want != 0) want--;
    b.nsplit = want;
    const long long units = (long long)g.ntiles * want;
    grid = g.sm_count;
    if (g_pipe_grid > 0 && g_pipe_grid < grid) grid = g_pipe_grid;
    if (grid > units) grid = (int)units;
  }
  dw_pipe_kernel<T, RECON, DIAG><<<grid, PIPE_THREADS, c.smem, s>>>(g, b, c.nslot);
  count_launch();
  return cudaGetLastError();
}

// ---- host side: configuration of the one-thread-per-site kernel ------------------------------------------
enum { KIND_FULL = 0, KIND_HALF = 1, KIND_SPLIT = 2 };   // dw_kernel / dw_kernel_h<false> / dw_kernel_h<true>
struct DirectCfg {
  int grid, threads, kind;
};
template <typename T, int RECON, int DIAG>
static DirectCfg direct_config_t(const Geom& g, int parity) {
  DirectCfg c;
  const int mode = dw_mode();
  const int npar = parity < 0 ? 2 : 1;
  c.kind = KIND_FULL;
  if (parity < 0 && mode == MODE_SPLIT) c.kind = KIND_SPLIT;
  else if (npar * g.TV <= 128) c.kind = KIND_HALF;
  c.threads = c.kind == KIND_SPLIT ? ((g.TV + 31) / 32) * 32 : ((npar * g.TV + 31) / 32) * 32;
  const int items = c.kind == KIND_SPLIT ? 2 * g.ntiles : g.ntiles;
  c.grid = items;
  if (mode == MODE_DIRECT) return c;
  // resident CTAs per SM of this instantiation on the current device for this CTA size (queried per call: the
  // answer depends on the device and on c.threads, and the query is a host-side table lookup)
  int occ = 0;
  {
    cudaError_t e;
    if (c.kind == KIND_FULL) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, dw_kernel<T, RECON, DIAG>, c.threads, 0);
    else if (c.kind == KIND_HALF) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, dw_kernel_h<T, RECON, DIAG, false>, c.threads, 0);
    else e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, dw_kernel_h<T, RECON, DIAG, true>, c.threads, 0);
    if (e != cudaSuccess || occ < 1) occ = 1;
    if (occ > 8) occ = 8;   // partial_len() (api.cu) sizes the per-CTA partial sums for at most 8 CTAs per SM
  }
  int ctas = env_int("LQCD_CTAS_PER_SM", occ);
  if (ctas < 1 || ctas > occ) ctas = occ;
  c.grid = g.sm_count * ctas;
  if (c.grid > items) c.grid = items;
  if (c.kind == KIND_SPLIT) c.grid &= ~1;   // both parities of a tile sit in neighbouring CTAs
  return c;
}
template <typename T>
static DirectCfg direct_config(const Geom& g, int recon, int diag, int parity) {
  if (recon == 12) {
    if (diag == DIAG_ONE) return direct_config_t<T, 12, DIAG_ONE>(g, parity);
    if (diag == DIAG_PRE) return direct_config_t<T, 12, DIAG_PRE>(g, parity);
    return direct_config_t<T, 12, DIAG_POST>(g, parity);
  }
  if (diag == DIAG_ONE) return direct_config_t<T, 18, DIAG_ONE>(g, parity);
  if (diag == DIAG_PRE) return direct_config_t<T, 18, DIAG_PRE>(g, parity);
  return direct_config_t<T, 18, DIAG_POST>(g, parity);
}

template <typename T>
void dw_describe(const Geom& g, int recon, int diag, int parity, char* buf, int len) {
  const PipeCfg pc = pipe_config<T>(g, recon, diag, parity);
  const char* tn = sizeof(T) == 8 ? "double" : "float";
  const PipeCfg hc = pipe_half_config<T>(g, recon, diag, parity);
  if (hc.use) {
    snprintf(buf, (size_t)len, "dw_pipe_half_kernel<%s,%d,%d> grid=%d threads=%d smem=%zu ring_slots=%d halo_buffers=%d tile=%dx%dx%dx%d sweep=%d chunk=%dx%d",
             tn, recon, diag, hc.grid, (int)PIPE_THREADS, hc.smem, hc.nslot, half_nhb<T>(), g.b[0], g.b[1], g.b[2], g.b[3], g.sw, g.c1, g.c2);
    return;
  }
  if (pc.use) {
    snprintf(buf, (size_t)len, "dw_pipe_kernel<%s,%d,%d> grid=%d threads=%d smem=%zu ring_slots=%d halo_buffers=%d tile=%dx%dx%dx%d sweep=%d chunk=%dx%d",
             tn, recon, diag, pc.grid, (int)PIPE_THREADS, pc.smem, pc.nslot, pipe_nhb<T>(), g.b[0], g.b[1], g.b[2], g.b[3], g.sw, g.c1, g.c2);
    return;
  }
  const DirectCfg dc = direct_config<T>(g, recon, diag, parity);
  snprintf(buf, (size_t)len, "%s<%s,%d,%d%s> grid=%d threads=%d smem=0 tile=%dx%dx%dx%d sweep=%d chunk=%dx%d",
           dc.kind == KIND_FULL ? "dw_kernel" : "dw_kernel_h", tn, recon, diag,
           dc.kind == KIND_FULL ? "" : (dc.kind == KIND_SPLIT ? ",split" : ",half"), dc.grid, dc.threads, g.b[0], g.b[1],
           g.b[2], g.b[3], g.sw, g.c1, g.c2);
}
template void dw_describe<double>(const Geom&, int, int, int, char*, int);
template void dw_describe<float>(const Geom&, int, int, int, char*, int);

template <typename T>
int dw_num_partials(const Geom& g, int recon, int diag, int parity) {
  PipeCfg c = pipe_config<T>(g, recon, diag, parity);
  if (!c.use) c = pipe_half_config<T>(g, recon, diag, parity);
  return c.use ? g.ntiles : direct_config<T>(g, recon, diag, parity).grid;   // pipeline: one partial sum per tile
}
template <typename T>
bool dw_uses_pipe(const Geom& g, int recon, int diag, int parity) { return pipe_config<T>(g, recon, diag, parity).use; }
template bool dw_uses_pipe<double>(const Geom&, int, int, int);
template bool dw_uses_pipe<float>(const Geom&, int, int, int);
template int dw_num_partials<double>(const Geom&, int, int, int);
template int dw_num_partials<float>(const Geom&, int, int, int);

template <typename T>
__global__ void __launch_bounds__(256) diag_kernel(const Geom g, const T2<T>* __restrict__ B, const T2<T>* __restrict__ in,
                                                   T2<T>* out, const int parity) {
  const int TV = g.TV;
  const int tid = threadIdx.x;
  const int tile = blockIdx.x;
  const int npar = (parity < 0) ? 2 : 1;
  if (tid >= npar * TV) return;
  const int pidx = (tid >= TV) ? 1 : 0;
  const int j = tid - pidx * TV;
  const int p = (parity < 0) ? pidx : parity;
  int Tc[4], l[4];
  tile_coords(g, tile, Tc);
  local_coords(g, j, p, l);
  const size_t off = field_offset(g, 12, p, tile, 0, j);
  cx<T> v[12], o[12];
  if ((g.bc != LQCD_BC_PERIODIC) && frozen_slice(g, Tc[3] * g.b[3] + l[3])) {
#pragma unroll
    for (int c = 0; c < 12; c++) o[c] = cx<T>(0, 0);
  } else {
#pragma unroll
    for (int c = 0; c < 12; c++) v[c] = ld<T>(in + off + (size_t)c * TV);
    clover_mul<T>(B + field_offset(g, 36, p, tile, 0, j), TV, v, o);
  }
#pragma unroll
  for (int c = 0; c < 12; c++) st<T>(out + off + (size_t)c * TV, o[c]);
}

template <typename T>
cudaError_t launch_diag(const Geom& g, const void* B, const void* in, void* out, int parity, cudaStream_t s) {
  int npar = parity < 0 ? 2 : 1;
  int threads = ((npar * g.TV + 31) / 32) * 32;
  diag_kernel<T><<<g.ntiles, threads, 0, s>>>(g, (const T2<T>*)B, (const T2<T>*)in, (T2<T>*)out, parity);
  count_launch();
  return cudaGetLastError();
}
template cudaError_t launch_diag<double>(const Geom&, const void*, const void*, void*, int, cudaStream_t);
template cudaError_t launch_diag<float>(const Geom&, const void*, const void*, void*, int, cudaStream_t);

template <typename T, int RECON, int DIAG>
static cudaError_t launch_one(const Geom& g, const DwArgs<T>& a, cudaStream_t s) {
  const DirectCfg c = direct_config_t<T, RECON, DIAG>(g, a.parity);
  if (c.kind == KIND_FULL) dw_kernel<T, RECON, DIAG><<<c.grid, c.threads, 0, s>>>(g, a);
  else if (c.kind == KIND_HALF) dw_kernel_h<T, RECON, DIAG, false><<<c.grid, c.threads, 0, s>>>(g, a);
  else dw_kernel_h<T, RECON, DIAG, true><<<c.grid, c.threads, 0, s>>>(g, a);
  count_launch();
  return cudaGetLastError();
}

template <typename T>
cudaError_t launch_dw(const Geom& g, const DwArgs<T>& a, int recon, int diag, cudaStream_t s) {
  if (a.self == a.in) {
    const PipeCfg c = pipe_config<T>(g, recon, diag, a.parity);
    if (c.use) {
      if (recon == 12) return diag == DIAG_ONE ? launch_pipe<T, 12, DIAG_ONE>(g, a, c, s) : launch_pipe<T, 12, DIAG_PRE>(g, a, c, s);
      return diag == DIAG_ONE ? launch_pipe<T, 18, DIAG_ONE>(g, a, c, s) : launch_pipe<T, 18, DIAG_PRE>(g, a, c, s);
    }
  }
  if (a.parity >= 0 && a.nrhs <= 1) {
    const PipeCfg c = pipe_half_config<T>(g, recon, diag, a.parity);
    if (c.use) {
      if (recon == 12) return diag == DIAG_PRE ? launch_pipe_half<T, 12, DIAG_PRE>(g, a, c, s) : launch_pipe_half<T, 12, DIAG_POST>(g, a, c, s);
      return diag == DIAG_PRE ? launch_pipe_half<T, 18, DIAG_PRE>(g, a, c, s) : launch_pipe_half<T, 18, DIAG_POST>(g, a, c, s);
    }
  }
  if (a.nrhs > 1) {   // the one-thread-per-site kernels take one right-hand side per launch
    for (int n = 0; n < a.nrhs; n++) {
      DwArgs<T> b = a;
      b.nrhs = 0;
      b.in = a.in + n * a.rhs_stride;
      b.self = (a.self == a.in) ? b.in : a.self + n * a.rhs_stride;
      b.out = a.out + n * a.rhs_stride;
      if (a.r) b.r = a.r + n * a.rhs_stride;
      cudaError_t e = launch_dw<T>(g, b, recon, diag, s);
      if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
  }
  if (recon == 12) {
    if (diag == DIAG_ONE) return launch_one<T, 12, DIAG_ONE>(g, a, s);
    if (diag == DIAG_PRE) return launch_one<T, 12, DIAG_PRE>(g, a, s);
    return launch_one<T, 12, DIAG_POST>(g, a, s);
  }
  if (diag == DIAG_ONE) return launch_one<T, 18, DIAG_ONE>(g, a, s);
  if (diag == DIAG_PRE) return launch_one<T, 18, DIAG_PRE>(g, a, s);
  return launch_one<T, 18, DIAG_POST>(g, a, s);
}

template cudaError_t launch_dw<double>(const Geom&, const DwArgs<double>&, int, int, cudaStream_t);
template cudaError_t launch_dw<float>(const Geom&, const DwArgs<float>&, int, int, cudaStream_t);

}  // namespace lqcd
