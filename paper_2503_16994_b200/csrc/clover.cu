// clover.cu -- Csw!: the Sheikholeslami-Wohlert term from the four plaquette leaves
// (definitions D4, D5, D7).
//
//   Q_{mu nu}(x) = sum of the four leaves in the mu-nu plane,  F^ = (Q - Q^+)/8  (no trace subtraction, R3)
//   E_k = F^_{k4},  B_1 = F^_{23}, B_2 = F^_{31}, B_3 = F^_{12}
//   A+ = 1 + kappa csw sum_k sigma_k (x) i(E_k - B_k),   A- = 1 - kappa csw sum_k sigma_k (x) i(E_k + B_k)
// i.e. with the Hermitian 3x3 matrices G_k = i(+-E_k - B_k) each chiral block is
//   1 + kappa csw [[G_3, G_1 - i G_2], [G_1 + i G_2, -G_3]]          (row index 3*s + a)
// stored packed (6 real diagonal entries + 15 complex below the diagonal).  Always evaluated in fp64
// (R14); the result is rounded once to the requested precision.
#include "kernels.cuh"

namespace lqcd {

// Kernel structure: one thread per site.  The six Hermitian matrices i F^_{mu nu} are computed one plane at a time
// in a rolled loop (4 leaves x 3 SU(3) products per plane, leaf loop rolled too) and parked in shared memory
// as 9 reals each (54 doubles per thread, [component][thread]: conflict-free); the two chiral blocks are then
// assembled entry by entry straight into the packed output, so no 6x6 array is ever live unless the inverse is
// requested.  Arithmetic bound: 72 products x 198 flop = 14.3 kflop fp64 per site against 1152 bytes moved.

struct m3 { double2 e[3][3]; };

__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cfma(double2 a, double2 b, double2 s) {  // s + a*b
  return make_double2(fma(a.x, b.x, fma(-a.y, b.y, s.x)), fma(a.x, b.y, fma(a.y, b.x, s.y)));
}

// c = a b
__device__ __forceinline__ m3 mul_nn(const m3& a, const m3& b) {
  m3 c;
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) c.e[i][j] = cfma(a.e[i][2], b.e[2][j], cfma(a.e[i][1], b.e[1][j], cmul(a.e[i][0], b.e[0][j])));
  return c;
}
// q += a b
__device__ __forceinline__ void acc_nn(m3& q, const m3& a, const m3& b) {
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) q.e[i][j] = cfma(a.e[i][2], b.e[2][j], cfma(a.e[i][1], b.e[1][j], cfma(a.e[i][0], b.e[0][j], q.e[i][j])));
}

struct CloverCtx {
  Geom g;
  const double2* U;
  double phiT[3];
  // LQCD_BC_SLAB (NEXT-3): the time slices just below and just above the slab, canonical layout [n][4][3][3]
  const double2* halo_lo;
  const double2* halo_hi;
};

// The site a thread works on: tile, local coordinates, parity, global time coordinate.
struct SitePos {
  int tile, par, x3;
  int l[4];
};

// W = U_dir (dag == 0) or U_dir^+ (dag != 0) at the point x + dm mu^ + dn nu^ (|dm|, |dn| <= 1).
// The neighbour is found from the local coordinates: a step out of the tile follows the neighbour-tile table
// (periodic in every direction), so no division by a run-time extent is needed.  SF: the slice x4 = L4 is the
// fixed boundary field W' (D7) and is never read from memory.
// mu, nu, dir are run-time values: coordinates are shifted by comparison, never by indexing a register array.
template <int RECON>
__device__ __forceinline__ m3 link_at(const CloverCtx& c, const SitePos& sp, int mu, int dm, int nu, int dn, int dir, int dag) {
  const Geom& g = c.g;
  constexpr int NCU = RECON == 12 ? 6 : 9;
  m3 r;
  const bool sf = (g.bc == LQCD_BC_SF_ORBI || g.bc == LQCD_BC_SF_AFWB) || (g.bc == LQCD_BC_SLAB && (g.edges & LQCD_SLAB_SF_HI));
  const int x3 = sp.x3 + (mu == 3 ? dm : 0) + (nu == 3 ? dn : 0);
  if (sf && x3 == g.L[3]) {   // diagonal: its own transpose; dagger = conjugate
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
      for (int j = 0; j < 3; j++) r.e[i][j] = make_double2(0.0, 0.0);
    if (dir < 3) {
      const int Ld = dir == 0 ? g.L[0] : (dir == 1 ? g.L[1] : g.L[2]);
#pragma unroll
      for (int i = 0; i < 3; i++) {
        double s, co;
        sincos(c.phiT[i] / Ld, &s, &co);
        r.e[i][i] = make_double2(co, dag ? -s : s);
      }
    }
    return r;
  }
  int l[4];
  int t = sp.tile;
#pragma unroll
  for (int i = 0; i < 4; i++) {
    l[i] = sp.l[i] + (i == mu ? dm : 0) + (i == nu ? dn : 0);
    if (l[i] < 0) {
      l[i] += g.b[i];
      t = __ldg(g.tile_tab + (size_t)t * TILE_TAB + 2 * i + 1);
    } else if (l[i] >= g.b[i]) {
      l[i] -= g.b[i];
      t = __ldg(g.tile_tab + (size_t)t * TILE_TAB + 2 * i);
    }
  }
  const int p = (sp.par + dm + dn) & 1;
  m3 u;
  if (g.bc == LQCD_BC_SLAB && (x3 < 0 || x3 >= g.L[3])) {   // neighbour rank's slice: from the gauge halo
    int Tc[4];
    tile_coords(g, t, Tc);
    const int n = (Tc[0] * g.b[0] + l[0]) + g.L[0] * ((Tc[1] * g.b[1] + l[1]) + g.L[1] * (Tc[2] * g.b[2] + l[2]));
    const double2* hp = (x3 < 0 ? c.halo_lo : c.halo_hi) + ((size_t)n * 4 + dir) * 9;
#pragma unroll
    for (int k = 0; k < 9; k++) u.e[k / 3][k % 3] = __ldg(hp + k);
  } else {
    const double2* up = c.U + field_offset(g, 4 * NCU, p, t, dir * NCU, local_index(g, l));
#pragma unroll
    for (int k = 0; k < NCU; k++) u.e[k / 3][k % 3] = __ldg(up + (size_t)k * g.TV);
  }
  if (RECON == 12) {
#pragma unroll
    for (int k = 0; k < 3; k++) {
      const int k1 = (k + 1) % 3, k2 = (k + 2) % 3;
      double2 v = csub(cmul(u.e[0][k1], u.e[1][k2]), cmul(u.e[0][k2], u.e[1][k1]));
      u.e[2][k] = make_double2(v.x, -v.y);
    }
  }
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) r.e[i][j] = dag ? make_double2(u.e[j][i].x, -u.e[j][i].y) : u.e[i][j];
  return r;
}

// The four leaves of Q_{mu nu}(x), each a closed path of four oriented links starting and ending at x:
// per link (dm, dn, direction: 0 = mu / 1 = nu, dagger)
//   1: U_mu(x) U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+
//   2: U_nu(x) U_mu(x-mu+nu)^+ U_nu(x-mu)^+ U_mu(x-mu)
//   3: U_mu(x-mu)^+ U_nu(x-mu-nu)^+ U_mu(x-mu-nu) U_nu(x-nu)
//   4: U_nu(x-nu)^+ U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^+
__constant__ signed char LEAF[4][4][4] = {
    {{0, 0, 0, 0}, {+1, 0, 1, 0}, {0, +1, 0, 1}, {0, 0, 1, 1}},
    {{0, 0, 1, 0}, {-1, +1, 0, 1}, {-1, 0, 1, 1}, {-1, 0, 0, 0}},
    {{-1, 0, 0, 1}, {-1, -1, 1, 1}, {-1, -1, 0, 0}, {0, -1, 1, 0}},
    {{0, -1, 1, 1}, {0, -1, 0, 0}, {+1, -1, 1, 0}, {0, 0, 0, 1}},
};

// i * F^_{mu nu}(x)  (Hermitian), as 9 reals: diagonal, then (re, im) of [1][0], [2][0], [2][1].
// The leaf loop stays rolled (3 products + 4 link fetches of code): the unrolled body does not fit the
// instruction cache and the kernel then stalls on instruction fetch.
template <int RECON>
__device__ __forceinline__ void i_fhat(const CloverCtx& c, const SitePos& sp, int mu, int nu, double (&h)[9]) {
  m3 Q;
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) Q.e[i][j] = make_double2(0.0, 0.0);
#pragma unroll 1
  for (int lf = 0; lf < 4; lf++) {
#define LQCD_W(s) link_at<RECON>(c, sp, mu, LEAF[lf][s][0], nu, LEAF[lf][s][1], LEAF[lf][s][2] ? nu : mu, LEAF[lf][s][3])
    m3 t = mul_nn(LQCD_W(0), LQCD_W(1));
    m3 t2 = mul_nn(t, LQCD_W(2));
    acc_nn(Q, t2, LQCD_W(3));
#undef LQCD_W
  }
  // i (Q - Q^+)/8 :  (Q - Q^+)_{ij} = Q_ij - conj(Q_ji) ;  i*(a + ib) = -b + ia
#pragma unroll
  for (int i = 0; i < 3; i++) h[i] = -0.25 * Q.e[i][i].y;
  h[3] = -(Q.e[1][0].y + Q.e[0][1].y) * 0.125;  h[4] = (Q.e[1][0].x - Q.e[0][1].x) * 0.125;
  h[5] = -(Q.e[2][0].y + Q.e[0][2].y) * 0.125;  h[6] = (Q.e[2][0].x - Q.e[0][2].x) * 0.125;
  h[7] = -(Q.e[2][1].y + Q.e[1][2].y) * 0.125;  h[8] = (Q.e[2][1].x - Q.e[1][2].x) * 0.125;
}

// element (a, b) of a Hermitian 3x3 held as 9 reals (layout of i_fhat)
__device__ __forceinline__ double2 herm_at(const double (&h)[9], int a, int b) {
  if (a == b) return make_double2(h[a], 0.0);
  const int hi = a > b ? a : b, lo = a > b ? b : a;
  const int o = 3 + 2 * (hi * (hi - 1) / 2 + lo);
  return make_double2(h[o], a > b ? h[o + 1] : -h[o + 1]);
}

// in-place inverse of a Hermitian positive-definite 6x6 (Gauss-Jordan, no pivoting needed for HPD)
__device__ __forceinline__ void invert6(double2 (&a)[6][6]) {
#pragma unroll
  for (int c = 0; c < 6; c++) {
    const double piv = 1.0 / a[c][c].x;  // diagonal of an HPD Schur complement is real
    a[c][c] = make_double2(1.0, 0.0);
#pragma unroll
    for (int j = 0; j < 6; j++) a[c][j] = make_double2(a[c][j].x * piv, a[c][j].y * piv);
#pragma unroll
    for (int r = 0; r < 6; r++) {
      if (r == c) continue;
      const double2 f = a[r][c];
      a[r][c] = make_double2(0.0, 0.0);
#pragma unroll
      for (int j = 0; j < 6; j++) a[r][j] = csub(a[r][j], cmul(f, a[c][j]));
    }
  }
}

template <typename T>
__device__ __forceinline__ void store_packed(typename vec2<T>::type* out, size_t TV, const double2 (&a)[6][6]) {
#pragma unroll
  for (int k = 0; k < 3; k++) {
    typename vec2<T>::type d;
    d.x = (T)a[2 * k][2 * k].x;
    d.y = (T)a[2 * k + 1][2 * k + 1].x;
    out[k * TV] = d;
  }
#pragma unroll
  for (int i = 1; i < 6; i++)
#pragma unroll
    for (int jj = 0; jj < i; jj++) {
      typename vec2<T>::type l;
      l.x = (T)a[i][jj].x;
      l.y = (T)a[i][jj].y;
      out[(3 + i * (i - 1) / 2 + jj) * TV] = l;
    }
}

constexpr int CLV_THREADS = 128;
#ifndef CLV_MINB
#define CLV_MINB 3
#endif

template <typename T, int RECON, bool INV>
__global__ void __launch_bounds__(CLV_THREADS, CLV_MINB) clover_kernel(const CloverCtx c, const CloverParm cp, typename vec2<T>::type* A,
                                                             typename vec2<T>::type* Ainv) {
  extern __shared__ double sF[];   // [6 planes][9][CLV_THREADS]
  const Geom& g = c.g;
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 2 * g.Vh) return;
  // thread -> site: a CTA takes runs of JC = min(64, TV) consecutive checkerboard indices of BOTH parities of a
  // tile (for 4^4 tiles: a 4x4x4x2 slab), so that the links a site shares with its neighbours are fetched by
  // the same CTA at the same time and hit in L1; stores stay coalesced over j in runs of JC.
  const int JC = g.TV < 64 ? g.TV : 64;
  const long long unit = idx / (2 * JC);
  const int r = (int)(idx - unit * (2 * JC));
  const int cpt = g.TV / JC;   // runs per tile
  const int tile = (int)(unit / cpt);
  const int p = r / JC;
  const int j = (int)(unit - (long long)tile * cpt) * JC + (r - p * JC);
  SitePos sp;
  sp.tile = tile;
  sp.par = p;
  local_coords(g, j, p, sp.l);
  sp.x3 = __ldg(g.tile_tab + (size_t)tile * TILE_TAB + 8) + sp.l[3];
  const int x3 = sp.x3;
  if (x3 < cp.t_lo || x3 >= cp.t_hi) return;   // no barrier in this kernel: threads may leave on their own

  const bool fz = (g.bc != LQCD_BC_PERIODIC) && frozen_slice(g, x3);
  const double cc = cp.kappa * cp.csw;
  const bool have_f = !fz && cc != 0.0;
  double* myF = sF + threadIdx.x;
  if (have_f) {
    // planes 0..2: E_k = F^_{k4};  planes 3..5: B_k = F^_{k1 k2} = (23, 31, 12)
#pragma unroll 1
    for (int pl = 0; pl < 6; pl++) {
      const int k = pl < 3 ? pl : pl - 3;
      const int mu = pl < 3 ? k : (k + 1) % 3;
      const int nu = pl < 3 ? 3 : (k + 2) % 3;
      double h[9];
      i_fhat<RECON>(c, sp, mu, nu, h);
#pragma unroll
      for (int r = 0; r < 9; r++) myF[(pl * 9 + r) * CLV_THREADS] = h[r];
    }
  }
  double dadd = 0.0;
  if (!fz && g.bc != LQCD_BC_PERIODIC && cp.ct != 1.0) {  // R10: + 2 kappa (ct - 1) next to the frozen slices
    const bool slab = g.bc == LQCD_BC_SLAB;   // a slab has the term only next to its open faces
    const int last = (g.bc == LQCD_BC_OPEN || (slab && (g.edges & LQCD_SLAB_OPEN_HI))) ? g.L[3] - 2 : g.L[3] - 1;
    if (x3 == 1 && (!slab || (g.edges & LQCD_SLAB_OPEN_LO))) dadd += 2.0 * cp.kappa * (cp.ct - 1.0);
    if (x3 == last && (!slab || (g.edges & (LQCD_SLAB_OPEN_HI | LQCD_SLAB_SF_HI)))) dadd += 2.0 * cp.kappa * (cp.ct - 1.0);
  }
  const size_t TV = g.TV;
#pragma unroll 1
  for (int ch = 0; ch < 2; ch++) {
    // G_k = i(+-E_k - B_k), scaled by kappa csw
    double G[3][9];
    const double se = (ch == 0) ? cc : -cc;
#pragma unroll
    for (int k = 0; k < 3; k++)
#pragma unroll
      for (int r = 0; r < 9; r++)
        G[k][r] = have_f ? se * myF[(k * 9 + r) * CLV_THREADS] - cc * myF[((3 + k) * 9 + r) * CLV_THREADS] : 0.0;
    // block = 1 + [[G_3, G_1 - i G_2], [G_1 + i G_2, -G_3]]   (row index 3*s + a)
    double2 blk[6][6];
#pragma unroll
    for (int a = 0; a < 3; a++)
#pragma unroll
      for (int b = 0; b < 3; b++) {
        const double2 g1 = herm_at(G[0], a, b), g2 = herm_at(G[1], a, b), g3 = herm_at(G[2], a, b);
        const double one = (a == b) ? 1.0 + dadd : 0.0;
        blk[a][b] = make_double2(one + g3.x, g3.y);
        blk[3 + a][3 + b] = make_double2(one - g3.x, -g3.y);
        blk[a][3 + b] = make_double2(g1.x + g2.y, g1.y - g2.x);
        blk[3 + a][b] = make_double2(g1.x - g2.y, g1.y + g2.x);
      }
    const size_t off = field_offset(g, 36, p, tile, 18 * ch, j);
    store_packed<T>(A + off, TV, blk);
    if (INV) {
      invert6(blk);
      store_packed<T>(Ainv + off, TV, blk);
    }
  }
}

template <typename T, int RECON, bool INV>
static cudaError_t clover_launch(const CloverCtx& c, const CloverParm& cp, void* clover, void* clover_inv, cudaStream_t s) {
  typedef typename vec2<T>::type T2;
  const size_t smem = (size_t)54 * CLV_THREADS * sizeof(double);
  cudaError_t e = cudaFuncSetAttribute(clover_kernel<T, RECON, INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  unsigned blocks = (unsigned)((2 * c.g.Vh + CLV_THREADS - 1) / CLV_THREADS);
  clover_kernel<T, RECON, INV><<<blocks, CLV_THREADS, smem, s>>>(c, cp, (T2*)clover, (T2*)clover_inv);
  count_launch();
  return cudaGetLastError();
}

cudaError_t clover_build(const Geom& g, const CloverParm& cp, const void* U64, int recon, void* clover, void* clover_inv,
                         int out_prec, cudaStream_t s, const void* halo_lo, const void* halo_hi) {
  CloverCtx c;
  c.g = g;
  c.U = (const double2*)U64;
  c.halo_lo = (const double2*)halo_lo;
  c.halo_hi = (const double2*)halo_hi;
  for (int i = 0; i < 3; i++) c.phiT[i] = cp.phiT[i];
  const bool f64 = out_prec == LQCD_F64, r12 = recon == 12, inv = clover_inv != nullptr;
#define LQCD_CLV(T, R, I) return clover_launch<T, R, I>(c, cp, clover, clover_inv, s)
  if (f64) {
    if (r12) { if (inv) LQCD_CLV(double, 12, true); else LQCD_CLV(double, 12, false); }
    else     { if (inv) LQCD_CLV(double, 18, true); else LQCD_CLV(double, 18, false); }
  } else {
    if (r12) { if (inv) LQCD_CLV(float, 12, true); else LQCD_CLV(float, 12, false); }
    else     { if (inv) LQCD_CLV(float, 18, true); else LQCD_CLV(float, 18, false); }
  }
#undef LQCD_CLV
}

}  // namespace lqcd
