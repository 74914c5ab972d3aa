// clover.cu -- Csw!: the Sheikholeslami-Wohlert term from the four plaquette leaves
// (definitions D4, D5, D7).
//
//   Q_{mu nu}(x) = sum of the four leaves in the mu-nu plane,  F^ = (Q - Q^+)/8  (no trace subtraction, R3)
//   E_k = F^_{k4},  B_1 = F^_{23}, B_2 = F^_{31}, B_3 = F^_{12}
//   A+ = 1 + kappa csw sum_k sigma_k (x) i(E_k - B_k),   A- = 1 - kappa csw sum_k sigma_k (x) i(E_k + B_k)
// i.e. with the Hermitian 3x3 matrices G_k = i(+-E_k - B_k) each chiral block is
//   1 + kappa csw [[G_3, G_1 - i G_2], [G_1 + i G_2, -G_3]]          (row index 3*s + a)
// stored packed (6 real diagonal entries + 15 complex below the diagonal).  Always evaluated in fp64
// (R14); the result is rounded once to the requested precision.  One thread per site.
#include "kernels.cuh"

namespace lqcd {

struct m3 { double2 e[3][3]; };

__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) { return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }  // a*conj(b)
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }

__device__ m3 mmul(const m3& a, const m3& b) {
  m3 c;
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) {
      double2 s = cmul(a.e[i][0], b.e[0][j]);
      s = cadd(s, cmul(a.e[i][1], b.e[1][j]));
      s = cadd(s, cmul(a.e[i][2], b.e[2][j]));
      c.e[i][j] = s;
    }
  return c;
}
__device__ m3 mdag(const m3& a) {
  m3 c;
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) c.e[i][j] = make_double2(a.e[j][i].x, -a.e[j][i].y);
  return c;
}

struct CloverCtx {
  Geom g;
  const double2* U;
  int recon;
  double phiT[3];
};

// U_mu at the point x (coordinates may be one or two steps outside the box).
// Spatial directions wrap; time wraps for periodic BC; SF: slice x4 = L4 is the fixed boundary field W' (D7).
__device__ m3 link_at(const CloverCtx& c, const int xin[4], int mu) {
  const Geom& g = c.g;
  int x[4];
  for (int i = 0; i < 3; i++) {
    x[i] = xin[i];
    if (x[i] < 0) x[i] += g.L[i];
    if (x[i] >= g.L[i]) x[i] -= g.L[i];
  }
  x[3] = xin[3];
  m3 r;
  const bool sf = (g.bc == LQCD_BC_SF_ORBI || g.bc == LQCD_BC_SF_AFWB);
  if (sf && x[3] == g.L[3]) {
    for (int i = 0; i < 3; i++)
      for (int j = 0; j < 3; j++) r.e[i][j] = make_double2(0.0, 0.0);
    if (mu < 3)
      for (int i = 0; i < 3; i++) {
        double s, co;
        sincos(c.phiT[i] / g.L[mu], &s, &co);
        r.e[i][i] = make_double2(co, s);
      }
    return r;
  }
  if (x[3] < 0) x[3] += g.L[3];
  if (x[3] >= g.L[3]) x[3] -= g.L[3];
  int p, tile, j;
  site_locate(g, x, p, tile, j);
  const int NCU = c.recon == 12 ? 6 : 9;
  for (int k = 0; k < NCU; k++) r.e[k / 3][k % 3] = __ldg(c.U + field_offset(g, 4 * NCU, p, tile, mu * NCU + k, j));
  if (c.recon == 12) {
    for (int k = 0; k < 3; k++) {
      int k1 = (k + 1) % 3, k2 = (k + 2) % 3;
      double2 v = csub(cmul(r.e[0][k1], r.e[1][k2]), cmul(r.e[0][k2], r.e[1][k1]));
      r.e[2][k] = make_double2(v.x, -v.y);
    }
  }
  return r;
}

__device__ __forceinline__ void shifted(const int x[4], int mu, int d, int y[4]) {
  for (int i = 0; i < 4; i++) y[i] = x[i];
  y[mu] += d;
}

// i * F^_{mu nu}(x)  (Hermitian)
__device__ m3 i_fhat(const CloverCtx& c, const int x[4], int mu, int nu) {
  int xpm[4], xpn[4], xmm[4], xmn[4], xmmpn[4], xmmmn[4], xpmmn[4];
  shifted(x, mu, +1, xpm);
  shifted(x, nu, +1, xpn);
  shifted(x, mu, -1, xmm);
  shifted(x, nu, -1, xmn);
  shifted(xmm, nu, +1, xmmpn);
  shifted(xmm, nu, -1, xmmmn);
  shifted(xpm, nu, -1, xpmmn);
  m3 Q;
  {  // U_mu(x) U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+
    m3 a = mmul(link_at(c, x, mu), link_at(c, xpm, nu));
    m3 b = mmul(link_at(c, x, nu), link_at(c, xpn, mu));
    Q = mmul(a, mdag(b));
  }
  {  // U_nu(x) U_mu(x-mu+nu)^+ U_nu(x-mu)^+ U_mu(x-mu)
    m3 a = mmul(link_at(c, x, nu), mdag(link_at(c, xmmpn, mu)));
    m3 b = mmul(mdag(link_at(c, xmm, nu)), link_at(c, xmm, mu));
    m3 l = mmul(a, b);
    for (int i = 0; i < 3; i++)
      for (int j = 0; j < 3; j++) Q.e[i][j] = cadd(Q.e[i][j], l.e[i][j]);
  }
  {  // U_mu(x-mu)^+ U_nu(x-mu-nu)^+ U_mu(x-mu-nu) U_nu(x-nu)
    m3 a = mmul(link_at(c, xmmmn, nu), link_at(c, xmm, mu));
    m3 b = mmul(link_at(c, xmmmn, mu), link_at(c, xmn, nu));
    m3 l = mmul(mdag(a), b);
    for (int i = 0; i < 3; i++)
      for (int j = 0; j < 3; j++) Q.e[i][j] = cadd(Q.e[i][j], l.e[i][j]);
  }
  {  // U_nu(x-nu)^+ U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^+
    m3 a = mmul(mdag(link_at(c, xmn, nu)), link_at(c, xmn, mu));
    m3 b = mmul(link_at(c, xpmmn, nu), mdag(link_at(c, x, mu)));
    m3 l = mmul(a, b);
    for (int i = 0; i < 3; i++)
      for (int j = 0; j < 3; j++) Q.e[i][j] = cadd(Q.e[i][j], l.e[i][j]);
  }
  // i (Q - Q^+)/8 :  (Q - Q^+)_{ij} = Q_ij - conj(Q_ji) ;  i*(a + ib) = -b + ia
  m3 F;
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) {
      double re = (Q.e[i][j].x - Q.e[j][i].x) * 0.125;
      double im = (Q.e[i][j].y + Q.e[j][i].y) * 0.125;
      F.e[i][j] = make_double2(-im, re);
    }
  return F;
}

// in-place inverse of a Hermitian positive-definite 6x6 (Gauss-Jordan, no pivoting needed for HPD)
__device__ void invert6(double2 (&a)[6][6]) {
  for (int c = 0; c < 6; c++) {
    double piv = 1.0 / a[c][c].x;  // diagonal of an HPD Schur complement is real
    a[c][c] = make_double2(1.0, 0.0);
    for (int j = 0; j < 6; j++) a[c][j] = make_double2(a[c][j].x * piv, a[c][j].y * piv);
    for (int r = 0; r < 6; r++) {
      if (r == c) continue;
      double2 f = a[r][c];
      a[r][c] = make_double2(0.0, 0.0);
      for (int j = 0; j < 6; j++) a[r][j] = csub(a[r][j], cmul(f, a[c][j]));
    }
  }
}

template <typename T>
__device__ void store_packed(const Geom& g, typename vec2<T>::type* out, int p, int tile, int j, int ch, const double2 (&a)[6][6]) {
  for (int k = 0; k < 3; k++) {
    typename vec2<T>::type d;
    d.x = (T)a[2 * k][2 * k].x;
    d.y = (T)a[2 * k + 1][2 * k + 1].x;
    out[field_offset(g, 36, p, tile, 18 * ch + k, j)] = d;
  }
  for (int i = 1; i < 6; i++)
    for (int jj = 0; jj < i; jj++) {
      typename vec2<T>::type l;
      l.x = (T)a[i][jj].x;
      l.y = (T)a[i][jj].y;
      out[field_offset(g, 36, p, tile, 18 * ch + 3 + i * (i - 1) / 2 + jj, j)] = l;
    }
}

template <typename T>
__global__ void __launch_bounds__(128) clover_kernel(const CloverCtx c, const CloverParm cp, typename vec2<T>::type* A,
                                                     typename vec2<T>::type* Ainv) {
  const Geom& g = c.g;
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 2 * g.Vh) return;
  // thread -> site in internal order (stores are coalesced over j)
  int p = (int)(idx / g.Vh);
  long long rem = idx - (long long)p * g.Vh;
  int tile = (int)(rem / g.TV);
  int j = (int)(rem - (long long)tile * g.TV);
  int Tc[4], l[4], x[4];
  tile_coords(g, tile, Tc);
  local_coords(g, j, p, l);
  for (int i = 0; i < 4; i++) x[i] = Tc[i] * g.b[i] + l[i];

  double2 blk[2][6][6];
  for (int ch = 0; ch < 2; ch++)
    for (int i = 0; i < 6; i++)
      for (int k = 0; k < 6; k++) blk[ch][i][k] = make_double2(i == k ? 1.0 : 0.0, 0.0);

  const bool fz = (g.bc != LQCD_BC_PERIODIC) && frozen_slice(g, x[3]);
  if (!fz) {
    const double cc = cp.kappa * cp.csw;
    if (cc != 0.0) {
      for (int k = 0; k < 3; k++) {
        const int k1 = (k + 1) % 3, k2 = (k + 2) % 3;
        m3 E = i_fhat(c, x, k, 3);    // i E_k = i F^_{k4}
        m3 B = i_fhat(c, x, k1, k2);  // i B_k = i F^_{k1 k2}  (23, 31, 12)
        for (int ch = 0; ch < 2; ch++) {
          const double se = (ch == 0) ? 1.0 : -1.0;
          for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) {
              // G = i(+-E - B)
              double2 G = make_double2(se * E.e[a][b].x - B.e[a][b].x, se * E.e[a][b].y - B.e[a][b].y);
              G.x *= cc; G.y *= cc;
              if (k == 2) {  // sigma_3: +G on (0,0), -G on (1,1)
                blk[ch][a][b] = cadd(blk[ch][a][b], G);
                blk[ch][3 + a][3 + b] = csub(blk[ch][3 + a][3 + b], G);
              } else if (k == 0) {  // sigma_1: G on (0,1) and (1,0)
                blk[ch][a][3 + b] = cadd(blk[ch][a][3 + b], G);
                blk[ch][3 + a][b] = cadd(blk[ch][3 + a][b], G);
              } else {  // sigma_2: -i G on (0,1), +i G on (1,0)
                blk[ch][a][3 + b] = cadd(blk[ch][a][3 + b], make_double2(G.y, -G.x));
                blk[ch][3 + a][b] = cadd(blk[ch][3 + a][b], make_double2(-G.y, G.x));
              }
            }
        }
      }
    }
    if (g.bc != LQCD_BC_PERIODIC && cp.ct != 1.0) {  // R10: + 2 kappa (ct - 1) next to the frozen slices
      const int last = (g.bc == LQCD_BC_OPEN) ? g.L[3] - 2 : g.L[3] - 1;
      double add = 0.0;
      if (x[3] == 1) add += 2.0 * cp.kappa * (cp.ct - 1.0);
      if (x[3] == last) add += 2.0 * cp.kappa * (cp.ct - 1.0);
      for (int ch = 0; ch < 2; ch++)
        for (int i = 0; i < 6; i++) blk[ch][i][i].x += add;
    }
  }
  for (int ch = 0; ch < 2; ch++) store_packed<T>(g, A, p, tile, j, ch, blk[ch]);
  if (Ainv) {
    for (int ch = 0; ch < 2; ch++) {
      invert6(blk[ch]);
      store_packed<T>(g, Ainv, p, tile, j, ch, blk[ch]);
    }
  }
}

cudaError_t clover_build(const Geom& g, const CloverParm& cp, const void* U64, int recon, void* clover, void* clover_inv,
                         int out_prec, cudaStream_t s) {
  CloverCtx c;
  c.g = g;
  c.U = (const double2*)U64;
  c.recon = recon;
  for (int i = 0; i < 3; i++) c.phiT[i] = cp.phiT[i];
  unsigned blocks = (unsigned)((2 * g.Vh + 127) / 128);
  if (out_prec == LQCD_F64)
    clover_kernel<double><<<blocks, 128, 0, s>>>(c, cp, (double2*)clover, (double2*)clover_inv);
  else
    clover_kernel<float><<<blocks, 128, 0, s>>>(c, cp, (float2*)clover, (float2*)clover_inv);
  count_launch();
  return cudaGetLastError();
}

}  // namespace lqcd
