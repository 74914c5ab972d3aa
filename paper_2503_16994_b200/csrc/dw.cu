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
#include <stdlib.h>

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
__device__ __forceinline__ void hop_dir(const T2<T>* __restrict__ psi, const T2<T>* __restrict__ u, const int TV,
                                        const T m, const bool has_theta, const cx<T> th, cx<T> (&acc)[12]) {
  cx<T> h[2][3];
#pragma unroll
  for (int a = 0; a < 3; a++) {
    cx<T> p0 = ldx<T, LDG>(psi + (0 + a) * TV), p1 = ldx<T, LDG>(psi + (3 + a) * TV);
    cx<T> p2 = ldx<T, LDG>(psi + (6 + a) * TV), p3 = ldx<T, LDG>(psi + (9 + a) * TV);
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
    for (int k = 0; k < 3; k++) U[i][k] = ldx<T, LDG>(u + (3 * i + k) * TV);
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

template <typename T, int RECON, int DIAG>
__global__ void __launch_bounds__(256) dw_kernel(const Geom g, const DwArgs<T> a) {
  constexpr int NCU = (RECON == 12) ? 6 : 9;
  __shared__ int s_nbr[8];
  __shared__ double s_red[8];
  if (a.skip != nullptr && *a.skip != 0) return;  // CG finished: uniform early exit
  const int TV = g.TV;
  const int tid = threadIdx.x;
  const int tile = blockIdx.x;
  int Tc[4];
  tile_coords(g, tile, Tc);
  if (tid < 8) {
    int mu = tid >> 1, d = (tid & 1) ? -1 : +1;
    int Tn[4] = {Tc[0], Tc[1], Tc[2], Tc[3]};
    Tn[mu] += d;
    if (Tn[mu] < 0) Tn[mu] += g.nt[mu];
    if (Tn[mu] >= g.nt[mu]) Tn[mu] -= g.nt[mu];
    s_nbr[tid] = tile_linear(g, Tn[0], Tn[1], Tn[2], Tn[3]);
  }
  __syncthreads();

  const int npar = (a.parity < 0) ? 2 : 1;
  const bool active = tid < npar * TV;
  const int pidx = (tid >= TV) ? 1 : 0;
  const int j = tid - pidx * TV;
  const int p = (a.parity < 0) ? pidx : a.parity;
  double nrm = 0.0;

  if (active) {
    int l[4];
    local_coords(g, j, p, l);
    const int x3 = Tc[3] * g.b[3] + l[3];
    const bool nonper = (g.bc != LQCD_BC_PERIODIC);
    const bool fz = nonper && frozen_slice(g, x3);
    cx<T> res[12];
    if (fz) {
#pragma unroll
      for (int c = 0; c < 12; c++) res[c] = cx<T>(0, 0);
    } else {
      cx<T> acc[12];
#pragma unroll
      for (int c = 0; c < 12; c++) acc[c] = cx<T>(0, 0);
      const T sg = a.dagger ? T(-1) : T(1);
      const int bh0 = g.b[0] >> 1;
      const int l0h = l[0] >> 1;
      const int st1 = bh0, st2 = bh0 << g.lb[1], st3 = st2 << g.lb[2];
      const size_t ubase_self = field_offset(g, 4 * NCU, p, tile, 0, j);
      const int q = 1 - p;
      // direction 0
      {
        bool cr = (l[0] + 1 == g.b[0]);
        int jn = j - l0h + (cr ? 0 : ((l[0] + 1) >> 1));
        int tn = cr ? s_nbr[0] : tile;
        hop_dir<T, RECON, 0, true>(a.in + field_offset(g, 12, q, tn, 0, jn), a.U + ubase_self + (size_t)(0 * NCU) * TV,
                                   TV, sg, a.has_theta, a.theta[0], acc);
        cr = (l[0] == 0);
        jn = j - l0h + (cr ? bh0 - 1 : ((l[0] - 1) >> 1));
        tn = cr ? s_nbr[1] : tile;
        hop_dir<T, RECON, 0, false>(a.in + field_offset(g, 12, q, tn, 0, jn),
                                    a.U + field_offset(g, 4 * NCU, q, tn, 0 * NCU, jn), TV, -sg, a.has_theta,
                                    a.theta[0], acc);
      }
      // direction 1
      {
        bool cr = (l[1] + 1 == g.b[1]);
        int jn = cr ? j - (g.b[1] - 1) * st1 : j + st1;
        int tn = cr ? s_nbr[2] : tile;
        hop_dir<T, RECON, 1, true>(a.in + field_offset(g, 12, q, tn, 0, jn), a.U + ubase_self + (size_t)(1 * NCU) * TV,
                                   TV, sg, a.has_theta, a.theta[1], acc);
        cr = (l[1] == 0);
        jn = cr ? j + (g.b[1] - 1) * st1 : j - st1;
        tn = cr ? s_nbr[3] : tile;
        hop_dir<T, RECON, 1, false>(a.in + field_offset(g, 12, q, tn, 0, jn),
                                    a.U + field_offset(g, 4 * NCU, q, tn, 1 * NCU, jn), TV, -sg, a.has_theta,
                                    a.theta[1], acc);
      }
      // direction 2
      {
        bool cr = (l[2] + 1 == g.b[2]);
        int jn = cr ? j - (g.b[2] - 1) * st2 : j + st2;
        int tn = cr ? s_nbr[4] : tile;
        hop_dir<T, RECON, 2, true>(a.in + field_offset(g, 12, q, tn, 0, jn), a.U + ubase_self + (size_t)(2 * NCU) * TV,
                                   TV, sg, a.has_theta, a.theta[2], acc);
        cr = (l[2] == 0);
        jn = cr ? j + (g.b[2] - 1) * st2 : j - st2;
        tn = cr ? s_nbr[5] : tile;
        hop_dir<T, RECON, 2, false>(a.in + field_offset(g, 12, q, tn, 0, jn),
                                    a.U + field_offset(g, 4 * NCU, q, tn, 2 * NCU, jn), TV, -sg, a.has_theta,
                                    a.theta[2], acc);
      }
      // direction 3 (time): hops onto frozen slices are skipped, never multiplied by zero (D7, P7)
      {
        bool cr = (l[3] + 1 == g.b[3]);
        int jn = cr ? j - (g.b[3] - 1) * st3 : j + st3;
        int tn = cr ? s_nbr[6] : tile;
        int xn = (x3 + 1 == g.L[3]) ? 0 : x3 + 1;
        if (!(nonper && frozen_slice(g, xn)))
          hop_dir<T, RECON, 3, true>(a.in + field_offset(g, 12, q, tn, 0, jn),
                                     a.U + ubase_self + (size_t)(3 * NCU) * TV, TV, sg, a.has_theta, a.theta[3], acc);
        cr = (l[3] == 0);
        jn = cr ? j + (g.b[3] - 1) * st3 : j - st3;
        tn = cr ? s_nbr[7] : tile;
        xn = (x3 == 0) ? g.L[3] - 1 : x3 - 1;
        if (!(nonper && frozen_slice(g, xn)))
          hop_dir<T, RECON, 3, false>(a.in + field_offset(g, 12, q, tn, 0, jn),
                                      a.U + field_offset(g, 4 * NCU, q, tn, 3 * NCU, jn), TV, -sg, a.has_theta,
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


// =====================================================================================================
// Persistent, warp-specialised version of the full-lattice operator (parity = -1, self == in).
//
// The direct-load kernel above is latency-bound (184 registers -> 8 warps/SM, every hop a round trip to
// L2/DRAM).  Here the operands that are streamed from HBM exactly once -- the tile's own links (4 stages of
// NCU components x both parities), its clover blocks (36/NCU stages) and its spinor -- are fetched by ONE
// producer lane with 1-D bulk-asynchronous copies (cp.async.bulk, SASS UBLKCP) into a shared-memory ring of
// `nslot` stage buffers guarded by full/empty mbarriers, so the bytes in flight per SM (nslot-1 stages, ~110 KB
// in fp64) no longer depend on resident warps.  2*TV consumer threads (one per site, both parities of the
// tile) run the spin-projected hops and the clover multiply out of shared memory; only neighbours outside
// the tile and their backward links are read from global memory (L2 hits thanks to the tile order).
// The tile-blocked layout makes every stage a pair of contiguous blocks, so no tensor map is needed.
// =====================================================================================================

// packed Hermitian block, one component at a time: c in [0,36), chirality c/18; slot c%18 < 3 holds two real
// diagonal entries, slot 3 + i(i-1)/2 + jj the element (i,jj) of the strict lower triangle (D5).
template <typename T, int C>
__device__ __forceinline__ void clover_comp(const cx<T> l, const cx<T> (&v)[12], cx<T> (&o)[12]) {
  constexpr int ch = C / 18, s = C % 18;
  if (s < 3) {
    o[6 * ch + 2 * s] = l.re * v[6 * ch + 2 * s];
    o[6 * ch + 2 * s + 1] = l.im * v[6 * ch + 2 * s + 1];
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

struct PipeBars {
  uint64_t full_sp, empty_sp;
  uint64_t full[8], empty[8];
};

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

// both hops of direction MU for one site, links of the tile in ring stage `ub`, spinor tile in `sp`
template <typename T, int RECON, int MU>
__device__ __forceinline__ void hop_pair(const Geom& g, const DwArgs<T>& a, const T2<T>* sp, const T2<T>* ub,
                                         const int* __restrict__ tab, const int tile, const int p, const int j,
                                         const int (&l)[4], const int x3, const bool nonper, const T sg,
                                         cx<T> (&acc)[12]) {
  constexpr int NCU = (RECON == 12) ? 6 : 9;
  const int TV = g.TV;
  const int q = 1 - p;
  const int bh0 = g.b[0] >> 1;
  const int l0h = l[0] >> 1;
  int stride = bh0;                       // index stride of direction MU (MU >= 1)
  if (MU >= 2) stride <<= g.lb[1];
  if (MU >= 3) stride <<= g.lb[2];
  // ---- forward: theta (1 - gamma_mu) U_mu(x) psi(x + mu)
  {
    const bool cr = (l[MU] + 1 == g.b[MU]);
    int jn;
    if (MU == 0) jn = j - l0h + (cr ? 0 : ((l[0] + 1) >> 1));
    else jn = cr ? j - (g.b[MU] - 1) * stride : j + stride;
    bool on = true;
    if (MU == 3 && nonper) on = !frozen_slice(g, (x3 + 1 == g.L[3]) ? 0 : x3 + 1);
    if (on) {
      const T2<T>* ps = cr ? a.in + field_offset(g, 12, q, __ldg(tab + 2 * MU), 0, jn) : sp + (size_t)(q * 12) * TV + jn;
      hop_dir<T, RECON, MU, true, false>(ps, ub + (size_t)(p * NCU) * TV + j, TV, sg, a.has_theta, a.theta[MU], acc);
    }
  }
  // ---- backward: theta^* (1 + gamma_mu) U_mu(x - mu)^+ psi(x - mu)
  {
    const bool cr = (l[MU] == 0);
    int jn;
    if (MU == 0) jn = j - l0h + (cr ? bh0 - 1 : ((l[0] - 1) >> 1));
    else jn = cr ? j + (g.b[MU] - 1) * stride : j - stride;
    bool on = true;
    if (MU == 3 && nonper) on = !frozen_slice(g, (x3 == 0) ? g.L[3] - 1 : x3 - 1);
    if (on) {
      const T2<T>* ps;
      const T2<T>* us;
      if (cr) {
        const int tn = __ldg(tab + 2 * MU + 1);
        ps = a.in + field_offset(g, 12, q, tn, 0, jn);
        us = a.U + field_offset(g, 4 * NCU, q, tn, MU * NCU, jn);
      } else {
        ps = sp + (size_t)(q * 12) * TV + jn;
        us = ub + (size_t)(q * NCU) * TV + jn;
      }
      hop_dir<T, RECON, MU, false, false>(ps, us, TV, -sg, a.has_theta, a.theta[MU], acc);
    }
  }
}

template <typename T, int RECON, int DIAG>
__global__ void __launch_bounds__(288, (sizeof(T) == 4) ? 2 : 1)
dw_pipe_kernel(const Geom g, const DwArgs<T> a, const int nslot) {
  constexpr int NCU = (RECON == 12) ? 6 : 9;
  constexpr int NSTC = (DIAG == DIAG_PRE) ? 36 / NCU : 0;   // clover stages per tile
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ double s_red[9];
  if (a.skip != nullptr && *a.skip != 0) return;  // CG finished: uniform early exit
  const int TV = g.TV;
  const int tid = threadIdx.x;
  const int lane = tid & 31;
  const int ncons = 2 * TV;                         // consumer threads (multiple of 32)
  T2<T>* sp = reinterpret_cast<T2<T>*>(smem_raw);   // [2][12][TV] spinor tile
  T2<T>* ring = sp + (size_t)24 * TV;               // nslot x [2][NCU][TV]
  PipeBars* bars = reinterpret_cast<PipeBars*>(ring + (size_t)nslot * 2 * NCU * TV);
  if (tid == 0) {
    mbar_init(&bars->full_sp, 1);
    mbar_init(&bars->empty_sp, ncons >> 5);
    for (int i = 0; i < nslot; i++) {
      mbar_init(&bars->full[i], 1);
      mbar_init(&bars->empty[i], ncons >> 5);
    }
    mbar_fence_init();
  }
  __syncthreads();
  double nrm = 0.0;
  const uint32_t stage_bytes = (uint32_t)(NCU * TV * sizeof(T2<T>));
  const uint32_t sp_bytes = (uint32_t)(12 * TV * sizeof(T2<T>));

  if (tid >= ncons) {
    // ------------------------------ producer: one lane feeds the ring ------------------------------
    if (tid == ncons) {
      const uint64_t pol_once = policy_evict_first();
      RingPos rp = {0, 0u};
      int k = 0;
      for (int tile = blockIdx.x; tile < g.ntiles; tile += gridDim.x, k++) {
        if (k == 0) {
          mbar_arrive_expect_tx(&bars->full_sp, 2 * sp_bytes);
          for (int p = 0; p < 2; p++)
            bulk_g2s(sp + (size_t)(p * 12) * TV, a.in + field_offset(g, 12, p, tile, 0, 0), sp_bytes, &bars->full_sp);
        }
#pragma unroll 1
        for (int st = 0; st < 4 + NSTC; st++) {
          mbar_wait(&bars->empty[rp.slot], rp.ph ^ 1u);
          mbar_arrive_expect_tx(&bars->full[rp.slot], 2 * stage_bytes);
          T2<T>* dst = ring + (size_t)rp.slot * 2 * NCU * TV;
          for (int p = 0; p < 2; p++) {
            if (st < 4)
              bulk_g2s(dst + (size_t)(p * NCU) * TV, a.U + field_offset(g, 4 * NCU, p, tile, st * NCU, 0), stage_bytes,
                       &bars->full[rp.slot]);
            else
              bulk_g2s_hint(dst + (size_t)(p * NCU) * TV, a.A + field_offset(g, 36, p, tile, (st - 4) * NCU, 0),
                            stage_bytes, &bars->full[rp.slot], pol_once);
          }
          rp.advance(nslot);
        }
        const int next = tile + gridDim.x;
        if (next < g.ntiles) {  // spinor of the next tile: its buffer is released after this tile's hops
          mbar_wait(&bars->empty_sp, (uint32_t)(k & 1));
          mbar_arrive_expect_tx(&bars->full_sp, 2 * sp_bytes);
          for (int p = 0; p < 2; p++)
            bulk_g2s(sp + (size_t)(p * 12) * TV, a.in + field_offset(g, 12, p, next, 0, 0), sp_bytes, &bars->full_sp);
        }
      }
    }
  } else {
    // ------------------------------ consumers: one thread per site ---------------------------------
    const int p = (tid >= TV) ? 1 : 0;
    const int j = tid - p * TV;
    int l[4];
    local_coords(g, j, p, l);
    const bool nonper = (g.bc != LQCD_BC_PERIODIC);
    const T sg = a.dagger ? T(-1) : T(1);
    RingPos rp = {0, 0u};
    int k = 0;
    for (int tile = blockIdx.x; tile < g.ntiles; tile += gridDim.x, k++) {
      const int* tab = g.tile_tab + (size_t)tile * TILE_TAB;
      const int x3 = __ldg(tab + 8) + l[3];
      const bool live = !(nonper && frozen_slice(g, x3));
      cx<T> acc[12], v[12], res[12];
#pragma unroll
      for (int c = 0; c < 12; c++) acc[c] = cx<T>(0, 0);
      mbar_wait(&bars->full_sp, (uint32_t)(k & 1));
#define LQCD_HOP_STAGE(MU)                                                                                       \
      mbar_wait(&bars->full[rp.slot], rp.ph);                                                                    \
      if (live)                                                                                                  \
        hop_pair<T, RECON, MU>(g, a, sp, ring + (size_t)rp.slot * 2 * NCU * TV, tab, tile, p, j, l, x3, nonper, sg, acc); \
      __syncwarp();                                                                                              \
      if (lane == 0) mbar_arrive(&bars->empty[rp.slot]);                                                         \
      rp.advance(nslot);
      LQCD_HOP_STAGE(0)
      LQCD_HOP_STAGE(1)
      LQCD_HOP_STAGE(2)
      LQCD_HOP_STAGE(3)
#undef LQCD_HOP_STAGE
      if (live) {
        const T2<T>* sv = sp + (size_t)(p * 12) * TV + j;
#pragma unroll
        for (int c = 0; c < 12; c++) {
          T2<T> w = sv[c * TV];
          v[c] = cx<T>(w.x, w.y);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->empty_sp);   // spinor tile no longer needed: next tile's may land
      if (DIAG == DIAG_PRE) {
        cx<T> av[12];
        CloverPipe<T, NCU, 0, NSTC>::run(bars, ring, rp, nslot, TV, (p * NCU) * TV + j, live, lane, v, av);
        if (live) {
#pragma unroll
          for (int c = 0; c < 12; c++) res[c] = cx<T>(fma(-a.k, acc[c].re, av[c].re), fma(-a.k, acc[c].im, av[c].im));
        }
      } else if (live) {
#pragma unroll
        for (int c = 0; c < 12; c++) res[c] = cx<T>(fma(-a.k, acc[c].re, v[c].re), fma(-a.k, acc[c].im, v[c].im));
      }
      if (!live) {
#pragma unroll
        for (int c = 0; c < 12; c++) res[c] = cx<T>(0, 0);
      }
      // epilogue (same three variants as dw_kernel)
      const size_t ooff = field_offset(g, 12, p, tile, 0, j);
      if (a.epi == EPI_AXPY_NORM) {
        const T al = (T)(*a.alpha);
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
    }
  }
  if (a.epi != EPI_STORE) {  // fixed-order CTA reduction over everything this CTA produced
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nrm += __shfl_xor_sync(0xffffffffu, nrm, o);
    if (lane == 0) s_red[tid >> 5] = nrm;
    __syncthreads();
    if (tid == 0) {
      double s = 0;
      const int nw = (int)(blockDim.x >> 5);
      for (int w = 0; w < nw; w++) s += s_red[w];
      a.partial[blockIdx.x] = s;
    }
  }
}

// ---- host side: configuration of the persistent kernel ------------------------------------------------
struct PipeCfg {
  bool use;
  int grid, threads, nslot;
  size_t smem;
};
template <typename T>
static PipeCfg pipe_config(const Geom& g, int recon, int diag, int parity) {
  PipeCfg c = {false, 0, 0, 0, 0};
  static const bool disabled = getenv("LQCD_NO_PIPE") != nullptr;
  if (disabled || parity >= 0 || diag == DIAG_POST) return c;
  if (g.TV < 32 || g.TV > 128 || (g.TV & 15) || g.tile_tab == nullptr) return c;
  const int ncu = recon == 12 ? 6 : 9;
  const int per_sm = sizeof(T) == 4 ? 2 : 1;
  const size_t sp = (size_t)24 * g.TV * sizeof(T2<T>);
  const size_t slot = (size_t)2 * ncu * g.TV * sizeof(T2<T>);
  size_t budget = (size_t)g.smem_optin - 256;                            // 256 B: the kernel's static shared memory
  if (per_sm == 2) budget = ((size_t)g.smem_optin + 1024) / 2 - 1024 - 256;   // 1 KB per CTA is reserved by the system
  if (budget < sp + sizeof(PipeBars) + 3 * slot) return c;
  int nslot = (int)((budget - sp - sizeof(PipeBars)) / slot);
  if (nslot > 8) nslot = 8;
  const char* e = getenv("LQCD_NSLOT");
  if (e && atoi(e) >= 2 && atoi(e) <= nslot) nslot = atoi(e);
  c.use = true;
  c.nslot = nslot;
  c.smem = sp + (size_t)nslot * slot + sizeof(PipeBars);
  c.threads = 2 * g.TV + 32;
  c.grid = g.sm_count * per_sm;
  if (c.grid > g.ntiles) c.grid = g.ntiles;
  return c;
}

template <typename T, int RECON, int DIAG>
static cudaError_t launch_pipe(const Geom& g, const DwArgs<T>& a, const PipeCfg& c, cudaStream_t s) {
  static size_t attr_smem = 0;   // the attribute is per function; raise it when a launch needs more
  if (c.smem > attr_smem) {
    cudaError_t e = cudaFuncSetAttribute(dw_pipe_kernel<T, RECON, DIAG>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)c.smem);
    if (e != cudaSuccess) return e;
    attr_smem = c.smem;
  }
  dw_pipe_kernel<T, RECON, DIAG><<<c.grid, c.threads, c.smem, s>>>(g, a, c.nslot);
  count_launch();
  return cudaGetLastError();
}

template <typename T>
int dw_num_partials(const Geom& g, int recon, int diag, int parity) {
  PipeCfg c = pipe_config<T>(g, recon, diag, parity);
  return c.use ? c.grid : g.ntiles;
}
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
  int npar = a.parity < 0 ? 2 : 1;
  int threads = ((npar * g.TV + 31) / 32) * 32;
  dw_kernel<T, RECON, DIAG><<<g.ntiles, threads, 0, s>>>(g, a);
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
