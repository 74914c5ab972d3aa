// su2.cu -- the SU(2) fundamental representation: gauge links stored as
// Cayley-Dickson pairs (z1, z2), U = [[z1, z2], [-conj z2, conj z1]], spinors with 4 x 2 components,
// the clover term as two packed Hermitian 4x4 chiral blocks.  Same definitions as the SU(3) path (D1-D8 with two
// colours), same tile-blocked even-odd SoA layout with 8 (links), 8 (spinor) and 16 (blocks) complex numbers per
// site.  One thread per site, direct global loads: a first, plain version (the shared-memory pipeline is SU(3) only).
// Periodic and open time boundaries; no even-odd, no twisted mass, c~_t = 1.
#include <math.h>
#include <string.h>

#include "kernels.cuh"

namespace lqcd {

template <typename T> using T2 = typename vec2<T>::type;
enum { SU2_NG = 8, SU2_NS = 8, SU2_NA = 16, SU2_THREADS = 128 };

// ---- sites and neighbours through the tile table (any tile shape) --------------------------------------------
struct Site2 {
  int p, tile, j, x3;
  int l[4];
};
__device__ __forceinline__ bool site2_from_thread(const Geom& g, Site2& s) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 2 * g.Vh) return false;
  // a CTA (128 threads) takes runs of JC = min(64, TV) consecutive checkerboard indices of BOTH parities of a tile
  // (4^4 tiles: a 4x4x4x2 slab), so that most neighbours of a site are fetched by the same CTA and hit in L1
  const int JC = g.TV < 64 ? g.TV : 64;
  const long long unit = idx / (2 * JC);
  const int r = (int)(idx - unit * (2 * JC));
  const int cpt = g.TV / JC;   // runs per tile
  s.tile = (int)(unit / cpt);
  s.p = r / JC;
  s.j = (int)(unit - (long long)s.tile * cpt) * JC + (r - s.p * JC);
  local_coords(g, s.j, s.p, s.l);
  s.x3 = __ldg(g.tile_tab + (size_t)s.tile * TILE_TAB + 8) + s.l[3];
  return true;
}
__device__ __forceinline__ Site2 step2(const Geom& g, const Site2& s, const int mu, const int d) {
  Site2 n = s;
  n.p = 1 - s.p;
  n.l[mu] += d;
  if (n.l[mu] < 0) {
    n.l[mu] += g.b[mu];
    n.tile = __ldg(g.tile_tab + (size_t)s.tile * TILE_TAB + 2 * mu + 1);
  } else if (n.l[mu] >= g.b[mu]) {
    n.l[mu] -= g.b[mu];
    n.tile = __ldg(g.tile_tab + (size_t)s.tile * TILE_TAB + 2 * mu);
  }
  n.j = local_index(g, n.l);
  n.x3 = __ldg(g.tile_tab + (size_t)n.tile * TILE_TAB + 8) + n.l[3];
  return n;
}
__device__ __forceinline__ long long canon_index(const Geom& g, const Site2& s) {
  int T[4];
  tile_coords(g, s.tile, T);
  long long n = 0;
  for (int i = 3; i >= 0; i--) n = n * g.L[i] + (T[i] * g.b[i] + s.l[i]);
  return n;
}

// ---- layout conversion -------------------------------------------------------------------------------------------
// canonical gauge [n][mu][2][2] (full matrices); the stored pair is the first row
template <typename T>
__global__ void su2_gauge_import_kernel(const Geom g, const double2* __restrict__ canon, T2<T>* U) {
  Site2 s;
  if (!site2_from_thread(g, s)) return;
  const long long n = canon_index(g, s);
  for (int mu = 0; mu < 4; mu++)
    for (int k = 0; k < 2; k++) {
      const double2 v = canon[(n * 4 + mu) * 4 + k];
      T2<T> w;
      w.x = (T)v.x; w.y = (T)v.y;
      U[field_offset(g, SU2_NG, s.p, s.tile, 2 * mu + k, s.j)] = w;
    }
}
template <typename T>
__global__ void su2_gauge_export_kernel(const Geom g, const T2<T>* __restrict__ U, double2* canon) {
  Site2 s;
  if (!site2_from_thread(g, s)) return;
  const long long n = canon_index(g, s);
  for (int mu = 0; mu < 4; mu++) {
    const T2<T> a = U[field_offset(g, SU2_NG, s.p, s.tile, 2 * mu, s.j)], b = U[field_offset(g, SU2_NG, s.p, s.tile, 2 * mu + 1, s.j)];
    double2* o = canon + (n * 4 + mu) * 4;
    o[0] = make_double2((double)a.x, (double)a.y);
    o[1] = make_double2((double)b.x, (double)b.y);
    o[2] = make_double2(-(double)b.x, (double)b.y);
    o[3] = make_double2((double)a.x, -(double)a.y);
  }
}
// canonical [n][NC] <-> internal, NC complex numbers per site
template <typename T, bool IMPORT>
__global__ void su2_field_kernel(const Geom g, double2* canon, T2<T>* f, const int NC) {
  Site2 s;
  if (!site2_from_thread(g, s)) return;
  const long long n = canon_index(g, s);
  for (int c = 0; c < NC; c++) {
    const size_t off = field_offset(g, NC, s.p, s.tile, c, s.j);
    if (IMPORT) {
      const double2 v = canon[n * NC + c];
      T2<T> w;
      w.x = (T)v.x; w.y = (T)v.y;
      f[off] = w;
    } else {
      const T2<T> w = f[off];
      canon[n * NC + c] = make_double2((double)w.x, (double)w.y);
    }
  }
}

// ---- 2x2 complex matrices for the clover builder (fp64 always, R14) ------------------------------------------------
struct m2 { double2 e[2][2]; };
__device__ __forceinline__ double2 cm(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 ca(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ m2 mmul(const m2& a, const m2& b) {
  m2 c;
  for (int i = 0; i < 2; i++)
    for (int j = 0; j < 2; j++) c.e[i][j] = ca(cm(a.e[i][0], b.e[0][j]), cm(a.e[i][1], b.e[1][j]));
  return c;
}
__device__ __forceinline__ m2 mdag(const m2& a) {
  m2 c;
  for (int i = 0; i < 2; i++)
    for (int j = 0; j < 2; j++) c.e[i][j] = make_double2(a.e[j][i].x, -a.e[j][i].y);
  return c;
}
__device__ __forceinline__ m2 link2(const Geom& g, const double2* __restrict__ U, const Site2& s, const int mu) {
  const double2 a = __ldg(U + field_offset(g, SU2_NG, s.p, s.tile, 2 * mu, s.j)), b = __ldg(U + field_offset(g, SU2_NG, s.p, s.tile, 2 * mu + 1, s.j));
  m2 r;
  r.e[0][0] = a; r.e[0][1] = b;
  r.e[1][0] = make_double2(-b.x, b.y);
  r.e[1][1] = make_double2(a.x, -a.y);
  return r;
}
// i F^_{mu nu}(x) (Hermitian 2x2) from the four leaves (D4)
__device__ __forceinline__ m2 i_fhat2(const Geom& g, const double2* __restrict__ U, const Site2& x, const int mu, const int nu) {
  const Site2 xpm = step2(g, x, mu, +1), xpn = step2(g, x, nu, +1), xmm = step2(g, x, mu, -1), xmn = step2(g, x, nu, -1);
  const Site2 xmmpn = step2(g, xmm, nu, +1), xmmmn = step2(g, xmm, nu, -1), xpmmn = step2(g, xpm, nu, -1);
  const m2 q1 = mmul(mmul(link2(g, U, x, mu), link2(g, U, xpm, nu)), mmul(mdag(link2(g, U, xpn, mu)), mdag(link2(g, U, x, nu))));
  const m2 q2 = mmul(mmul(link2(g, U, x, nu), mdag(link2(g, U, xmmpn, mu))), mmul(mdag(link2(g, U, xmm, nu)), link2(g, U, xmm, mu)));
  const m2 q3 = mmul(mmul(mdag(link2(g, U, xmm, mu)), mdag(link2(g, U, xmmmn, nu))), mmul(link2(g, U, xmmmn, mu), link2(g, U, xmn, nu)));
  const m2 q4 = mmul(mmul(mdag(link2(g, U, xmn, nu)), link2(g, U, xmn, mu)), mmul(link2(g, U, xpmmn, nu), mdag(link2(g, U, x, mu))));
  m2 f;
  for (int i = 0; i < 2; i++)
    for (int j = 0; j < 2; j++) {
      const double2 q = ca(ca(q1.e[i][j], q2.e[i][j]), ca(q3.e[i][j], q4.e[i][j]));
      const double2 p = ca(ca(q1.e[j][i], q2.e[j][i]), ca(q3.e[j][i], q4.e[j][i]));
      // (Q - Q^+)/8, times i:  i (a + i b) = -b + i a
      const double re = (q.x - p.x) * 0.125, im = (q.y + p.y) * 0.125;
      f.e[i][j] = make_double2(-im, re);
    }
  return f;
}

// packed Hermitian 4x4 block: slot 0 = (d0, d1), slot 1 = (d2, d3), slots 2..7 = (1,0) (2,0) (2,1) (3,0) (3,1) (3,2)
__device__ __forceinline__ int su2_slot(int i, int k) { return 2 + i * (i - 1) / 2 + k; }

template <typename T>
__global__ void __launch_bounds__(SU2_THREADS) su2_clover_kernel(const Geom g, const double2* __restrict__ U, const double kc, T2<T>* A) {
  Site2 s;
  if (!site2_from_thread(g, s)) return;
  const bool fz = (g.bc != LQCD_BC_PERIODIC) && frozen_slice(g, s.x3);
  m2 E[3], Bm[3];
  if (!fz && kc != 0.0) {
    for (int k = 0; k < 3; k++) {
      E[k] = i_fhat2(g, U, s, k, 3);                       // i E_k = i F^_{k4}
      Bm[k] = i_fhat2(g, U, s, (k + 1) % 3, (k + 2) % 3);  // i B_k = i F^_{k+1,k+2}
    }
  }
  for (int ch = 0; ch < 2; ch++) {
    double2 blk[4][4];
    for (int i = 0; i < 4; i++)
      for (int k = 0; k < 4; k++) blk[i][k] = make_double2(i == k ? 1.0 : 0.0, 0.0);
    if (!fz && kc != 0.0) {
      const double se = ch == 0 ? kc : -kc;
      m2 G[3];   // kappa csw i(+-E_k - B_k)
      for (int k = 0; k < 3; k++)
        for (int a = 0; a < 2; a++)
          for (int b = 0; b < 2; b++) G[k].e[a][b] = make_double2(se * E[k].e[a][b].x - kc * Bm[k].e[a][b].x, se * E[k].e[a][b].y - kc * Bm[k].e[a][b].y);
      // 1 + [[G_3, G_1 - i G_2], [G_1 + i G_2, -G_3]]   (row index 2*s + a; D5 with two colours)
      for (int a = 0; a < 2; a++)
        for (int b = 0; b < 2; b++) {
          const double2 g1 = G[0].e[a][b], g2 = G[1].e[a][b], g3 = G[2].e[a][b];
          blk[a][b] = ca(blk[a][b], g3);
          blk[2 + a][2 + b] = ca(blk[2 + a][2 + b], make_double2(-g3.x, -g3.y));
          blk[a][2 + b] = make_double2(g1.x + g2.y, g1.y - g2.x);
          blk[2 + a][b] = make_double2(g1.x - g2.y, g1.y + g2.x);
        }
    }
    T2<T>* out = A + field_offset(g, SU2_NA, s.p, s.tile, 8 * ch, s.j);
    T2<T> d;
    d.x = (T)blk[0][0].x; d.y = (T)blk[1][1].x;
    out[0] = d;
    d.x = (T)blk[2][2].x; d.y = (T)blk[3][3].x;
    out[(size_t)g.TV] = d;
    for (int i = 1; i < 4; i++)
      for (int k = 0; k < i; k++) {
        T2<T> w;
        w.x = (T)blk[i][k].x; w.y = (T)blk[i][k].y;
        out[(size_t)su2_slot(i, k) * g.TV] = w;
      }
  }
}
template <typename T>
__global__ void su2_clover_export_kernel(const Geom g, const T2<T>* __restrict__ A, double2* canon) {
  Site2 s;
  if (!site2_from_thread(g, s)) return;
  const long long n = canon_index(g, s);
  for (int ch = 0; ch < 2; ch++) {
    const T2<T>* in = A + field_offset(g, SU2_NA, s.p, s.tile, 8 * ch, s.j);
    double2* o = canon + (n * 2 + ch) * 16;
    const T2<T> d0 = in[0], d1 = in[(size_t)g.TV];
    o[0] = make_double2((double)d0.x, 0.0);
    o[5] = make_double2((double)d0.y, 0.0);
    o[10] = make_double2((double)d1.x, 0.0);
    o[15] = make_double2((double)d1.y, 0.0);
    for (int i = 1; i < 4; i++)
      for (int k = 0; k < i; k++) {
        const T2<T> w = in[(size_t)su2_slot(i, k) * g.TV];
        o[i * 4 + k] = make_double2((double)w.x, (double)w.y);
        o[k * 4 + i] = make_double2((double)w.x, -(double)w.y);
      }
  }
}

// ---- the operator ----------------------------------------------------------------------------------------------
// one hop: m = +1 selects (1 - gamma_mu), -1 selects (1 + gamma_mu); the projections are those of dw.cu (D2) with
// two colours; y = U h (forward) or U^+ h (backward) with U = [[z1, z2], [-conj z2, conj z1]]
template <typename T, int MU, bool FWD>
__device__ __forceinline__ void hop_su2(const T2<T>* __restrict__ psi, const T2<T>* __restrict__ u, const size_t TV, const T m,
                                        const bool has_theta, const cx<T> th, cx<T> (&acc)[8]) {
  cx<T> h[2][2];
#pragma unroll
  for (int a = 0; a < 2; a++) {
    const cx<T> p0 = ld<T>(psi + (0 + a) * TV), p1 = ld<T>(psi + (2 + a) * TV), p2 = ld<T>(psi + (4 + a) * TV), p3 = ld<T>(psi + (6 + a) * TV);
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
  const cx<T> z1 = ld<T>(u), z2 = ld<T>(u + TV);
  cx<T> y[2][2];
#pragma unroll
  for (int s = 0; s < 2; s++) {
    if (FWD) {
      y[s][0] = cfma(z2, h[s][1], z1 * h[s][0]);
      y[s][1] = cfma_conj(z1, h[s][1], cx<T>(0, 0) - conj(z2) * h[s][0]);
    } else {
      y[s][0] = conj(z1) * h[s][0] - z2 * h[s][1];
      y[s][1] = cfma(z1, h[s][1], conj(z2) * h[s][0]);
    }
  }
  if (has_theta) {
    const cx<T> ph = FWD ? th : conj(th);
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
      for (int a = 0; a < 2; a++) y[s][a] = ph * y[s][a];
  }
#pragma unroll
  for (int a = 0; a < 2; a++) {
    acc[0 + a] = acc[0 + a] + y[0][a];
    acc[2 + a] = acc[2 + a] + y[1][a];
    if (MU == 0) {   // low2 = -m i y1, low3 = -m i y0
      acc[4 + a] = cx<T>(fma(m, y[1][a].im, acc[4 + a].re), fma(-m, y[1][a].re, acc[4 + a].im));
      acc[6 + a] = cx<T>(fma(m, y[0][a].im, acc[6 + a].re), fma(-m, y[0][a].re, acc[6 + a].im));
    } else if (MU == 1) {   // low2 = -m y1, low3 = +m y0
      acc[4 + a] = cx<T>(fma(-m, y[1][a].re, acc[4 + a].re), fma(-m, y[1][a].im, acc[4 + a].im));
      acc[6 + a] = cx<T>(fma(m, y[0][a].re, acc[6 + a].re), fma(m, y[0][a].im, acc[6 + a].im));
    } else if (MU == 2) {   // low2 = -m i y0, low3 = +m i y1
      acc[4 + a] = cx<T>(fma(m, y[0][a].im, acc[4 + a].re), fma(-m, y[0][a].re, acc[4 + a].im));
      acc[6 + a] = cx<T>(fma(-m, y[1][a].im, acc[6 + a].re), fma(m, y[1][a].re, acc[6 + a].im));
    } else {   // low2 = -m y0, low3 = -m y1
      acc[4 + a] = cx<T>(fma(-m, y[0][a].re, acc[4 + a].re), fma(-m, y[0][a].im, acc[4 + a].im));
      acc[6 + a] = cx<T>(fma(-m, y[1][a].re, acc[6 + a].re), fma(-m, y[1][a].im, acc[6 + a].im));
    }
  }
}

struct Su2Args {
  double k;
  double th_re[4], th_im[4];
  int has_theta, dagger;
};

template <typename T, int MU>
__device__ __forceinline__ void hop_both(const Geom& g, const Su2Args& a, const T2<T>* __restrict__ U, const T2<T>* __restrict__ in,
                                         const Site2& s, const bool nonper, const T sg, cx<T> (&acc)[8]) {
  const size_t TV = g.TV;
  const cx<T> th((T)a.th_re[MU], (T)a.th_im[MU]);
  if (!(MU == 3 && nonper && time_hop_blocked(g, s.x3, true))) {
    const Site2 n = step2(g, s, MU, +1);
    hop_su2<T, MU, true>(in + field_offset(g, SU2_NS, n.p, n.tile, 0, n.j), U + field_offset(g, SU2_NG, s.p, s.tile, 2 * MU, s.j), TV, sg,
                         a.has_theta != 0, th, acc);
  }
  if (!(MU == 3 && nonper && time_hop_blocked(g, s.x3, false))) {
    const Site2 n = step2(g, s, MU, -1);
    hop_su2<T, MU, false>(in + field_offset(g, SU2_NS, n.p, n.tile, 0, n.j), U + field_offset(g, SU2_NG, n.p, n.tile, 2 * MU, n.j), TV, -sg,
                          a.has_theta != 0, th, acc);
  }
}

// out = A in - kappa H in (or its gamma5 conjugate); A = NULL means csw = 0
// A latency-bound gather kernel: resident warps are what counts.  Measured at 48^3 x 96 (one gpurun call each): fp64
// 140 registers / 3 CTAs per SM 1.74 ms, 128 / 4 CTAs 1.46 ms, 96 / 5 CTAs (spills) 1.67 ms; fp32 80 registers / 6 CTAs
// 0.91 ms, 64 / 8 CTAs 0.84 ms.
enum { SU2_MINB64 = 4, SU2_MINB32 = 8 };
template <typename T>
__global__ void __launch_bounds__(SU2_THREADS, sizeof(T) == 8 ? SU2_MINB64 : SU2_MINB32) su2_dw_kernel(const Geom g, const Su2Args a, const T2<T>* __restrict__ U,
                                                             const T2<T>* __restrict__ A, const T2<T>* __restrict__ in, T2<T>* out) {
  Site2 s;
  if (!site2_from_thread(g, s)) return;
  const size_t TV = g.TV;
  const bool nonper = g.bc != LQCD_BC_PERIODIC;
  T2<T>* op = out + field_offset(g, SU2_NS, s.p, s.tile, 0, s.j);
  if (nonper && frozen_slice(g, s.x3)) {
#pragma unroll
    for (int c = 0; c < 8; c++) st<T>(op + c * TV, cx<T>(0, 0));
    return;
  }
  const T sg = a.dagger ? T(-1) : T(1);
  cx<T> acc[8], v[8], res[8];
#pragma unroll
  for (int c = 0; c < 8; c++) acc[c] = cx<T>(0, 0);
  hop_both<T, 0>(g, a, U, in, s, nonper, sg, acc);
  hop_both<T, 1>(g, a, U, in, s, nonper, sg, acc);
  hop_both<T, 2>(g, a, U, in, s, nonper, sg, acc);
  hop_both<T, 3>(g, a, U, in, s, nonper, sg, acc);
  const T2<T>* sp = in + field_offset(g, SU2_NS, s.p, s.tile, 0, s.j);
#pragma unroll
  for (int c = 0; c < 8; c++) v[c] = ld<T>(sp + c * TV);
  if (A != nullptr) {
#pragma unroll
    for (int ch = 0; ch < 2; ch++) {
      const T2<T>* B = A + field_offset(g, SU2_NA, s.p, s.tile, 8 * ch, s.j);
      cx<T> o[4];
      const cx<T> d0 = ld<T>(B), d1 = ld<T>(B + TV);
      o[0] = d0.re * v[4 * ch + 0];
      o[1] = d0.im * v[4 * ch + 1];
      o[2] = d1.re * v[4 * ch + 2];
      o[3] = d1.im * v[4 * ch + 3];
#pragma unroll
      for (int i = 1; i < 4; i++)
#pragma unroll
        for (int k = 0; k < i; k++) {
          const cx<T> l = ld<T>(B + (size_t)(2 + i * (i - 1) / 2 + k) * TV);
          o[i] = cfma(l, v[4 * ch + k], o[i]);
          o[k] = cfma_conj(l, v[4 * ch + i], o[k]);
        }
#pragma unroll
      for (int i = 0; i < 4; i++) res[4 * ch + i] = o[i];
    }
  } else {
#pragma unroll
    for (int c = 0; c < 8; c++) res[c] = v[c];
  }
  const T k = (T)a.k;
#pragma unroll
  for (int c = 0; c < 8; c++) st<T>(op + c * TV, cx<T>(fma(-k, acc[c].re, res[c].re), fma(-k, acc[c].im, res[c].im)));
}

// zero the frozen slices of an SU(2) spinor (D7)
template <typename T>
__global__ void su2_mask_kernel(const Geom g, T2<T>* psi) {
  Site2 s;
  if (!site2_from_thread(g, s)) return;
  if (!frozen_slice(g, s.x3)) return;
  for (int c = 0; c < 8; c++) st<T>(psi + field_offset(g, SU2_NS, s.p, s.tile, c, s.j), cx<T>(0, 0));
}

static unsigned su2_blocks(const Geom& g) { return (unsigned)((2 * g.Vh + SU2_THREADS - 1) / SU2_THREADS); }

// ---- host-callable launchers (declared in kernels.cuh) -----------------------------------------------------------
template <typename T> cudaError_t su2_gauge_import(const Geom& g, const void* canon, void* U, cudaStream_t s) {
  su2_gauge_import_kernel<T><<<su2_blocks(g), SU2_THREADS, 0, s>>>(g, (const double2*)canon, (T2<T>*)U);
  count_launch();
  return cudaGetLastError();
}
template <typename T> cudaError_t su2_gauge_export(const Geom& g, const void* U, void* canon, cudaStream_t s) {
  su2_gauge_export_kernel<T><<<su2_blocks(g), SU2_THREADS, 0, s>>>(g, (const T2<T>*)U, (double2*)canon);
  count_launch();
  return cudaGetLastError();
}
template <typename T> cudaError_t su2_spinor_import(const Geom& g, const void* canon, void* psi, cudaStream_t s) {
  su2_field_kernel<T, true><<<su2_blocks(g), SU2_THREADS, 0, s>>>(g, (double2*)canon, (T2<T>*)psi, SU2_NS);
  count_launch();
  return cudaGetLastError();
}
template <typename T> cudaError_t su2_spinor_export(const Geom& g, const void* psi, void* canon, cudaStream_t s) {
  su2_field_kernel<T, false><<<su2_blocks(g), SU2_THREADS, 0, s>>>(g, (double2*)canon, (T2<T>*)psi, SU2_NS);
  count_launch();
  return cudaGetLastError();
}
template <typename T> cudaError_t su2_clover_build(const Geom& g, double kappa, double csw, const void* U64, void* A, cudaStream_t s) {
  su2_clover_kernel<T><<<su2_blocks(g), SU2_THREADS, 0, s>>>(g, (const double2*)U64, kappa * csw, (T2<T>*)A);
  count_launch();
  return cudaGetLastError();
}
template <typename T> cudaError_t su2_clover_export(const Geom& g, const void* A, void* canon, cudaStream_t s) {
  su2_clover_export_kernel<T><<<su2_blocks(g), SU2_THREADS, 0, s>>>(g, (const T2<T>*)A, (double2*)canon);
  count_launch();
  return cudaGetLastError();
}
template <typename T>
cudaError_t su2_dw(const lqcd_geom* h, double kappa, const void* U, const void* A, const void* in, void* out, bool dagger, cudaStream_t s) {
  Su2Args a;
  a.k = kappa;
  for (int d = 0; d < 4; d++) { a.th_re[d] = h->th_re[d]; a.th_im[d] = h->th_im[d]; }
  a.has_theta = h->has_theta ? 1 : 0;
  a.dagger = dagger ? 1 : 0;
  su2_dw_kernel<T><<<su2_blocks(h->g), SU2_THREADS, 0, s>>>(h->g, a, (const T2<T>*)U, (const T2<T>*)A, (const T2<T>*)in, (T2<T>*)out);
  count_launch();
  return cudaGetLastError();
}
template <typename T> cudaError_t su2_mask_frozen(const Geom& g, void* psi, cudaStream_t s) {
  su2_mask_kernel<T><<<su2_blocks(g), SU2_THREADS, 0, s>>>(g, (T2<T>*)psi);
  count_launch();
  return cudaGetLastError();
}

#define INST(T)                                                                                                     \
  template cudaError_t su2_gauge_import<T>(const Geom&, const void*, void*, cudaStream_t);                          \
  template cudaError_t su2_gauge_export<T>(const Geom&, const void*, void*, cudaStream_t);                          \
  template cudaError_t su2_spinor_import<T>(const Geom&, const void*, void*, cudaStream_t);                         \
  template cudaError_t su2_spinor_export<T>(const Geom&, const void*, void*, cudaStream_t);                         \
  template cudaError_t su2_clover_build<T>(const Geom&, double, double, const void*, void*, cudaStream_t);          \
  template cudaError_t su2_clover_export<T>(const Geom&, const void*, void*, cudaStream_t);                         \
  template cudaError_t su2_dw<T>(const lqcd_geom*, double, const void*, const void*, const void*, void*, bool, cudaStream_t); \
  template cudaError_t su2_mask_frozen<T>(const Geom&, void*, cudaStream_t);
INST(double)
INST(float)
#undef INST

}  // namespace lqcd
