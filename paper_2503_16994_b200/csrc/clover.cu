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
#include <stdlib.h>

#include <algorithm>
#include <mutex>
#include <utility>
#include <vector>

#include "kernels.cuh"
#include "pipe.cuh"

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

// =====================================================================================================================
// Tile kernel (4^4 tiles).  The kernel above fetches every link of every leaf from L1/L2 (16 links x 6 planes per
// site = 13.8 kB per site through the L2 -> SM path, which is what bounds it).  Here a CTA owns a 4x4x4x2 slab of a
// tile (both parities, 128 sites, one thread each) and works plane by plane: the links of U_mu and U_nu that the
// slab's four leaves touch form two boxes (the slab grown by [-1, 0] along the link's own direction and by [-1, +1]
// along the other one), at most 630 links = 91 kB, which are copied into shared memory once (16-byte cp.async, no
// registers in flight) and then read from there: 3.7 kB per site through L2 instead of 13.8, and 13 instead of 16
// link reads per plane because consecutive leaves share a link.  Two CTAs are resident per SM, so one stages while
// the other multiplies.  The planes are taken in the order (E_3, B_3), (E_1, B_1), (E_2, B_2): the first pair gives
// the diagonal 3x3 blocks of both chiral blocks, which are written at once; the second pair is parked in shared
// memory (18 reals per thread) and combined with the third into the off-diagonal blocks -- so no more than one
// i F^ beside the running product is ever held in registers.
//
// Staged layout: [row k of the link][site r], r = c1 + E1 (c2 + E2 c3) + S0 c0 with c the box coordinate and
// S0 = E1 E2 E3 rounded up to 2 mod 4.  A quarter warp is 2 (x1 pairs) x 4 (x2) sites of one parity, i.e. its x1
// coordinates alternate between {a, a+2} and {a+-1, a+-1+2} from one x2 to the next; with x2 contiguous and the x1
// stride 2 or 6 mod 8 the eight 16-byte words fall into eight different bank groups for every leaf offset
// (x1 fastest, or the parity-split layout of the global fields, cannot achieve that for offsets along x1).

constexpr int CT_THREADS = 128;
constexpr int CT_TV = 128;       // sites of one parity in a 4^4 tile: compile-time, so that row offsets are immediates
constexpr int CT_NR = 632;        // staged links per plane (largest: plane (1,4), 330 + 300 with padding)
constexpr size_t CT_SMEM = (size_t)9 * CT_NR * sizeof(double2) + (size_t)18 * CT_THREADS * sizeof(double) + 81 * sizeof(int) + 12;

// s + (a or a^*) (b or b^*)
template <bool CA, bool CB>
__device__ __forceinline__ double2 cfma_c(double2 a, double2 b, double2 s) {
  const double ai = CA ? -a.y : a.y, bi = CB ? -b.y : b.y;
  return make_double2(fma(a.x, b.x, fma(-ai, bi, s.x)), fma(a.x, bi, fma(ai, b.x, s.y)));
}
// q (+)= op(a) op(b),  op = identity or Hermitian conjugate
template <bool DA, bool DB, bool ACC>
__device__ __forceinline__ void mul_op(m3& q, const m3& a, const m3& b) {
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) {
      double2 s = ACC ? q.e[i][j] : make_double2(0.0, 0.0);
#pragma unroll
      for (int k = 0; k < 3; k++) s = cfma_c<DA, DB>(DA ? a.e[k][i] : a.e[i][k], DB ? b.e[j][k] : b.e[k][j], s);
      q.e[i][j] = s;
    }
}

// one staged box: the links U_dir on the slab grown along mu and nu
struct StageBox {
  int E[4];   // extents
  int o[4];   // box coordinate of the slab's first site
  int S[4];   // strides in the staged array
  int n;      // links to stage
  int size;   // words taken in the staged array (with the padding of S[0])
};
__host__ __device__ inline StageBox make_box(int mu, int nu, bool is_nu) {
  StageBox b;
  for (int d = 0; d < 4; d++) {
    const int e = d == 3 ? 2 : 4;
    const int grow = d == mu ? (is_nu ? 2 : 1) : (d == nu ? (is_nu ? 1 : 2) : 0);
    b.E[d] = e + grow;
    b.o[d] = grow ? 1 : 0;
  }
  b.S[1] = 1;
  b.S[2] = b.E[1];
  b.S[3] = b.E[1] * b.E[2];
  const int n123 = b.S[3] * b.E[3];
  b.S[0] = n123 + ((2 - n123) & 3);
  b.n = n123 * b.E[0];
  b.size = b.S[0] * b.E[0];
  return b;
}

// Every thread brings in the two links of its own site (U_mu(x), U_nu(x): 256 of the ~600 links of a plane) through
// registers; the rest -- the fringe of the two boxes, at most 374 links -- is listed in a table.  Where a fringe link
// comes from and goes to depends only on the plane and on which half of the tile the slab is, not on the lattice: one
// 32-bit word per link, built on the host at first use (ct_table_upload):
//   bits 0-9 index r in the staged array, 10-16 neighbour tile (index into sNb), 17-23 checkerboard index j in that
//   tile, 24 parity, 25 box (0: U_mu, 1: U_nu), 26-28 time offset from the slab's first slice plus one; ~0 = none
#ifndef CT_REG
#define CT_REG 2            // table slots (of 128 links) that go through registers (see ct_table_build)
#endif
constexpr int CT_NIT = CT_REG + 2;   // two more slots for cp.async
__device__ uint32_t ct_table[2][6][CT_NIT * CT_THREADS];

// plane number pl = 2 * step + half of the kernel's loop -> (mu, nu)
__host__ __device__ inline void ct_plane(int pl, int& mu, int& nu) {
  const int step = pl >> 1, k = step == 0 ? 2 : step - 1;
  mu = (pl & 1) ? (k + 1) % 3 : k;
  nu = (pl & 1) ? (k + 2) % 3 : 3;
}

static void ct_table_build(uint32_t* tab) {
  for (int s = 0; s < 2; s++)
    for (int pl = 0; pl < 6; pl++) {
      int mu, nu;
      ct_plane(pl, mu, nu);
      const StageBox ba = make_box(mu, nu, false), bb = make_box(mu, nu, true);
      uint32_t* t = tab + (size_t)(s * 6 + pl) * CT_NIT * CT_THREADS;
      for (int i = 0; i < CT_NIT * CT_THREADS; i++) t[i] = ~0u;
      // fringe links whose x1 and x2 coordinates lie inside the slab come in whole runs of 8 consecutive j
      // (128 bytes per row): time slices next to the slab, x3 layers, their corners.  Sorted by address they fill the
      // first CT_REG slots, which go through registers; everything else (and what does not fit) is copied by cp.async.
      std::vector<std::pair<uint32_t, uint32_t>> runs;   // (sort key, word)
      int n = CT_REG * CT_THREADS;
      for (int idx = 0; idx < ba.n + bb.n; idx++) {
        const bool isb = idx >= ba.n;
        const StageBox& b = isb ? bb : ba;
        int q = isb ? idx - ba.n : idx, cc[4], l[4], rel[4];
        cc[0] = q % b.E[0]; q /= b.E[0];
        cc[1] = q % b.E[1]; q /= b.E[1];
        cc[2] = q % b.E[2];
        cc[3] = q / b.E[2];
        const int r = (isb ? ba.size : 0) + cc[1] + b.S[2] * cc[2] + b.S[3] * cc[3] + b.S[0] * cc[0];
        int nb = 0;
        bool own = true;
        for (int d = 3; d >= 0; d--) {
          rel[d] = cc[d] - b.o[d];   // coordinate relative to the slab
          own = own && rel[d] >= 0 && rel[d] < (d == 3 ? 2 : 4);
          l[d] = rel[d] + (d == 3 ? 2 * s : 0);
          nb = nb * 3 + (l[d] < 0 ? 0 : (l[d] >= 4 ? 2 : 1));
          l[d] &= 3;
        }
        if (own) continue;
        const int j = (l[0] >> 1) + 2 * (l[1] + 4 * (l[2] + 4 * l[3]));
        const int p = (l[0] + l[1] + l[2] + l[3]) & 1;
        const uint32_t word = (uint32_t)r | (uint32_t)nb << 10 | (uint32_t)j << 17 | (uint32_t)p << 24 | (uint32_t)isb << 25 |
                              (uint32_t)(rel[3] + 1) << 26;
        if (rel[0] >= 0 && rel[0] < 4 && rel[1] >= 0 && rel[1] < 4) {
          runs.push_back(std::make_pair((uint32_t)isb << 16 | (uint32_t)nb << 8 | (uint32_t)p << 7 | (uint32_t)j, word));
          continue;
        }
        if (n >= CT_NIT * CT_THREADS) abort();   // cannot happen (see the counts in DESIGN.md)
        t[n++] = word;
      }
      std::sort(runs.begin(), runs.end());
      for (size_t i = 0; i < runs.size(); i++) {
        if (i < (size_t)CT_REG * CT_THREADS) t[i] = runs[i].second;
        else {
          if (n >= CT_NIT * CT_THREADS) abort();
          t[n++] = runs[i].second;
        }
      }
    }
}

// Copies the links of both boxes of a plane into sU[k][r] (box A = U_mu from 0, box B = U_nu from ba.size).
// A 16-byte cp.async costs one shared-memory wavefront per LANE (32 per instruction; with every link staged that way
// the copies alone were 2.4 G wavefronts = 8.4 ms of the load/store pipe at 48^3 x 96, next to 0.94 G for the reads of
// the arithmetic), a 16-byte load into a register plus a 16-byte store costs a quarter of that but holds registers and
// exposes its round trip.  So: what a warp can load in whole 128-byte lines goes through registers, all of it in
// flight together -- the thread's own two links, and CT_REG table slots of fringe links that come in runs of eight
// consecutive j -- and the scattered rest of the fringe (x1 and x2 faces: 16- and 32-byte pieces) is copied by
// cp.async while those loads are under way.  Scattered links through registers, or more than one batch of register
// loads, were measured slower (profiles/r02_notes.md, section 12).  RECON 12: the third row is rebuilt in registers,
// or in shared memory once the copies have landed.
template <int RECON>
__device__ __forceinline__ void recon_row3(double2 (&v)[9]) {
  if (RECON == 12) {
#pragma unroll
    for (int k = 0; k < 3; k++) {
      const int k1 = (k + 1) % 3, k2 = (k + 2) % 3;
      const double2 w = csub(cmul(v[k1], v[3 + k2]), cmul(v[k2], v[3 + k1]));
      v[6 + k] = make_double2(w.x, -w.y);
    }
  }
}

// own: the thread's own links, element offset of row 0 of U_0(x) in the gauge field; ra / rb: where they go
template <int RECON>
__device__ __forceinline__ void stage_plane(const CloverCtx& c, double2* sU, const int* sNb, const uint32_t* tb, int mu, int nu,
                                            const double2* own, int ra, int rb, m3& Umu) {
  const Geom& g = c.g;
  constexpr int NCU = RECON == 12 ? 6 : 9;
  double2 va[9], vb[9];
#pragma unroll
  for (int k = 0; k < NCU; k++) va[k] = __ldg(own + (size_t)(mu * NCU + k) * CT_TV);
#pragma unroll
  for (int k = 0; k < NCU; k++) vb[k] = __ldg(own + (size_t)(nu * NCU + k) * CT_TV);
  uint32_t ent[CT_NIT];
#pragma unroll
  for (int it = 0; it < CT_NIT; it++) ent[it] = __ldg(tb + threadIdx.x + it * CT_THREADS);
  double2 vf[CT_REG][9];
#pragma unroll
  for (int it = 0; it < CT_NIT; it++) {
    if (ent[it] == ~0u) continue;
    const uint32_t en = ent[it];
    const int t = sNb[(en >> 10) & 127], j = (en >> 17) & 127, p = (en >> 24) & 1;
    const int dir = (en >> 25) & 1 ? nu : mu;
    const double2* src = c.U + field_offset(g, 4 * NCU, p, t, dir * NCU, j);
    double2* dst = sU + (en & 1023);
    if (it < CT_REG) {
#pragma unroll
      for (int k = 0; k < NCU; k++) vf[it < CT_REG ? it : 0][k] = __ldg(src + (size_t)k * CT_TV);
    } else {
#pragma unroll
      for (int k = 0; k < NCU; k++) cp_async_16(dst + k * CT_NR, src + (size_t)k * CT_TV);
    }
  }
  recon_row3<RECON>(va);
  recon_row3<RECON>(vb);
#pragma unroll
  for (int k = 0; k < 9; k++) sU[k * CT_NR + ra] = va[k];
#pragma unroll
  for (int k = 0; k < 9; k++) Umu.e[k / 3][k % 3] = va[k];   // stays in registers: first and last link of the leaf chain
#pragma unroll
  for (int k = 0; k < 9; k++) sU[k * CT_NR + rb] = vb[k];
#pragma unroll
  for (int it = 0; it < CT_REG; it++) {
    if (ent[it] == ~0u) continue;
    recon_row3<RECON>(vf[it]);
    double2* dst = sU + (ent[it] & 1023);
#pragma unroll
    for (int k = 0; k < 9; k++) dst[k * CT_NR] = vf[it][k];
  }
  asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
  if (RECON == 12) {
#pragma unroll
    for (int it = CT_REG; it < CT_NIT; it++) {
      if (ent[it] == ~0u) continue;
      double2* dst = sU + (ent[it] & 1023);
      double2 v[9];
#pragma unroll
      for (int k = 0; k < 6; k++) v[k] = dst[k * CT_NR];
      recon_row3<RECON>(v);
#pragma unroll
      for (int k = 6; k < 9; k++) dst[k * CT_NR] = v[k];
    }
  }
}

// The same for the planes of a slab that reach past the lattice in time: SF, the slice x4 = L4 is the boundary
// field W' (D7); LQCD_BC_SLAB, slices outside the slab come from the gauge halos.  One link at a time.
template <int RECON>
__device__ __forceinline__ void stage_plane_edge(const CloverCtx& c, double2* sU, const int* sNb, const uint32_t* tb, int mu, int nu, int t0,
                                              const double2* own, int ra, int rb, m3& Umu) {
  const Geom& g = c.g;
  constexpr int NCU = RECON == 12 ? 6 : 9;
#pragma unroll 1
  for (int w = 0; w < 2; w++) {   // the thread's own two links (always inside the lattice)
    double2 v[9];
#pragma unroll
    for (int k = 0; k < NCU; k++) v[k] = __ldg(own + (size_t)((w ? nu : mu) * NCU + k) * CT_TV);
    recon_row3<RECON>(v);
#pragma unroll
    for (int k = 0; k < 9; k++) sU[k * CT_NR + (w ? rb : ra)] = v[k];
    if (w == 0) {
#pragma unroll
      for (int k = 0; k < 9; k++) Umu.e[k / 3][k % 3] = v[k];
    }
  }
  const bool sf = (g.bc == LQCD_BC_SF_ORBI || g.bc == LQCD_BC_SF_AFWB) || (g.bc == LQCD_BC_SLAB && (g.edges & LQCD_SLAB_SF_HI));
#pragma unroll 1
  for (int it = 0; it < CT_NIT; it++) {
    const uint32_t ent = __ldg(tb + threadIdx.x + it * CT_THREADS);
    if (ent == ~0u) continue;   // slots are filled from the front, but not to the end
    const int t = sNb[(ent >> 10) & 127], j = (ent >> 17) & 127, p = (ent >> 24) & 1;
    const int dir = (ent >> 25) & 1 ? nu : mu;
    const int x3 = t0 + (int)((ent >> 26) & 7) - 1;
    double2* dst = sU + (ent & 1023);
    double2 v[9];
#pragma unroll
    for (int k = 0; k < 9; k++) v[k] = make_double2(0.0, 0.0);
    if (sf && x3 == g.L[3]) {
      if (dir < 3) {
        const int Ld = dir == 0 ? g.L[0] : (dir == 1 ? g.L[1] : g.L[2]);
#pragma unroll
        for (int i = 0; i < 3; i++) {
          double sn, co;
          sincos(c.phiT[i] / Ld, &sn, &co);
          v[4 * i] = make_double2(co, sn);
        }
      }
    } else if (g.bc == LQCD_BC_SLAB && (x3 < 0 || x3 >= g.L[3])) {
      int l[4];
      local_coords(g, j, p, l);
      const int* org = g.tile_tab + (size_t)t * TILE_TAB + 9;   // space coordinates of the tile origin
      const int n = (__ldg(org) + l[0]) + g.L[0] * ((__ldg(org + 1) + l[1]) + g.L[1] * (__ldg(org + 2) + l[2]));
      const double2* hb = x3 < 0 ? c.halo_lo : c.halo_hi;   // NULL at an open face: only the frozen slice asks
      if (hb) {
#pragma unroll
        for (int k = 0; k < 9; k++) v[k] = __ldg(hb + ((size_t)n * 4 + dir) * 9 + k);
      }
    } else {
      const double2* src = c.U + field_offset(g, 4 * NCU, p, t, dir * NCU, j);
#pragma unroll
      for (int k = 0; k < NCU; k++) v[k] = __ldg(src + (size_t)k * CT_TV);
      recon_row3<RECON>(v);
    }
#pragma unroll
    for (int k = 0; k < 9; k++) dst[k * CT_NR] = v[k];
  }
}

__device__ __forceinline__ m3 lds_link(const double2* sU, int r) {
  m3 w;
#pragma unroll
  for (int k = 0; k < 9; k++) w.e[k / 3][k % 3] = sU[k * CT_NR + r];
  return w;
}

// i F^_{mu nu} of the thread's site from the staged boxes: ra / rb = the site's index in the U_mu / U_nu box,
// (am, an) / (bm, bn) = the strides of a step along mu / nu in them.  Consecutive leaves share a link: 11 reads.
__device__ __forceinline__ void i_fhat_staged(const double2* sU, const m3& Umu, int ra, int am, int an, int rb, int bm, int bn,
                                              double (&h)[9]) {
  m3 Q, t, t2, W, H;
  W = lds_link(sU, rb + bm);                 // U_nu(x+mu)
  mul_op<false, false, false>(t, Umu, W);       // U_mu(x) (the thread's own link, kept in registers by the staging)
  W = lds_link(sU, ra + an);                 // U_mu(x+nu)^+
  mul_op<false, true, false>(t2, t, W);
  H = lds_link(sU, rb);                      // U_nu(x)^+ ... and first of leaf 2
  mul_op<false, true, false>(Q, t2, H);
  W = lds_link(sU, ra - am + an);            // U_mu(x-mu+nu)^+
  mul_op<false, true, false>(t, H, W);
  W = lds_link(sU, rb - bm);                 // U_nu(x-mu)^+
  mul_op<false, true, false>(t2, t, W);
  H = lds_link(sU, ra - am);                 // U_mu(x-mu) ... and (daggered) first of leaf 3
  mul_op<false, false, true>(Q, t2, H);
  W = lds_link(sU, rb - bm - bn);            // U_mu(x-mu)^+ U_nu(x-mu-nu)^+ = (U_nu(x-mu-nu) U_mu(x-mu))^+
  mul_op<false, false, false>(t, W, H);
  W = lds_link(sU, ra - am - an);            // U_mu(x-mu-nu)
  mul_op<true, false, false>(t2, t, W);
  H = lds_link(sU, rb - bn);                 // U_nu(x-nu) ... and (daggered) first of leaf 4
  mul_op<false, false, true>(Q, t2, H);
  W = lds_link(sU, ra - an);                 // U_mu(x-nu)
  mul_op<true, false, false>(t, H, W);
  W = lds_link(sU, rb + bm - bn);            // U_nu(x+mu-nu)
  mul_op<false, false, false>(t2, t, W);
  mul_op<false, true, true>(Q, t2, Umu);        // U_mu(x)^+
#pragma unroll
  for (int i = 0; i < 3; i++) h[i] = -0.25 * Q.e[i][i].y;
  h[3] = -(Q.e[1][0].y + Q.e[0][1].y) * 0.125;  h[4] = (Q.e[1][0].x - Q.e[0][1].x) * 0.125;
  h[5] = -(Q.e[2][0].y + Q.e[0][2].y) * 0.125;  h[6] = (Q.e[2][0].x - Q.e[0][2].x) * 0.125;
  h[7] = -(Q.e[2][1].y + Q.e[1][2].y) * 0.125;  h[8] = (Q.e[2][1].x - Q.e[1][2].x) * 0.125;
}

template <typename T, int RECON>
__global__ void __launch_bounds__(CT_THREADS, 2) clover_tile_kernel(const CloverCtx c, const CloverParm cp, typename vec2<T>::type* A) {
  extern __shared__ __align__(16) unsigned char ct_smem[];
  double2* sU = (double2*)ct_smem;                  // [9][CT_NR]
  double* sG = (double*)(sU + 9 * CT_NR) + threadIdx.x;   // [18][CT_THREADS]
  int* sNb = (int*)((double*)(sU + 9 * CT_NR) + 18 * CT_THREADS);   // [3][3][3][3] neighbour tiles, direction 0 fastest
  const Geom& g = c.g;
  const int tile = blockIdx.x >> 1, s = blockIdx.x & 1;
  const int t0 = __ldg(g.tile_tab + (size_t)tile * TILE_TAB + 8) + 2 * s;
  if (t0 + 1 < cp.t_lo || t0 >= cp.t_hi) return;   // whole slab outside the requested slices (uniform over the CTA)
  if (threadIdx.x < 81) {   // tiles at offsets (-1, 0, +1) in every direction; a plane needs those with at most two steps
    int q = threadIdx.x, t = tile, steps = 0, st[4];
#pragma unroll
    for (int d = 0; d < 4; d++) { st[d] = q % 3; q /= 3; steps += st[d] != 1; }
    if (steps <= 2) {
#pragma unroll
      for (int d = 0; d < 4; d++)
        if (st[d] != 1) t = __ldg(g.tile_tab + (size_t)t * TILE_TAB + 2 * d + (st[d] == 0 ? 1 : 0));
    }
    sNb[threadIdx.x] = t;
  }
  const int p = threadIdx.x >> 6, j = 64 * s + (threadIdx.x & 63);
  int l[4];
  local_coords(g, j, p, l);
  l[3] -= 2 * s;
  const int x3 = t0 + l[3];
  // does the slab's time neighbourhood leave the lattice where that needs special links?
  const bool edge = (g.bc == LQCD_BC_SF_ORBI || g.bc == LQCD_BC_SF_AFWB || g.bc == LQCD_BC_SLAB) && (t0 == 0 || t0 + 2 >= g.L[3]);
  const bool wr = x3 >= cp.t_lo && x3 < cp.t_hi;
  const bool fz = (g.bc != LQCD_BC_PERIODIC) && frozen_slice(g, x3);
  const double cc = fz ? 0.0 : cp.kappa * cp.csw;
  double one = 1.0;
  if (!fz && g.bc != LQCD_BC_PERIODIC && cp.ct != 1.0) {  // R10: + 2 kappa (ct - 1) next to the frozen slices
    const bool slab = g.bc == LQCD_BC_SLAB;
    const int last = (g.bc == LQCD_BC_OPEN || (slab && (g.edges & LQCD_SLAB_OPEN_HI))) ? g.L[3] - 2 : g.L[3] - 1;
    if (x3 == 1 && (!slab || (g.edges & LQCD_SLAB_OPEN_LO))) one += 2.0 * cp.kappa * (cp.ct - 1.0);
    if (x3 == last && (!slab || (g.edges & (LQCD_SLAB_OPEN_HI | LQCD_SLAB_SF_HI)))) one += 2.0 * cp.kappa * (cp.ct - 1.0);
  }
  typedef typename vec2<T>::type T2;
  T2* out0 = A + field_offset(g, 36, p, tile, 0, j);
  const double2* own = c.U + field_offset(g, RECON == 12 ? 24 : 36, p, tile, 0, j);
  constexpr size_t TV = CT_TV;
  auto put = [&](int ch, int idx, double x, double y) {
    if (wr) {
      T2 v;
      v.x = (T)x; v.y = (T)y;
      out0[(size_t)(18 * ch + idx) * TV] = v;
    }
  };

#pragma unroll 1
  for (int step = 0; step < 3; step++) {
    double e[9], h[9];
#pragma unroll 1
    for (int half = 0; half < 2; half++) {
      int mu, nu;
      ct_plane(2 * step + half, mu, nu);
      const StageBox ba = make_box(mu, nu, false), bb = make_box(mu, nu, true);
      const uint32_t* tb = ct_table[s][2 * step + half];
      int ra = 0, rb = ba.size, am = 0, an = 0, bm = 0, bn = 0;
#pragma unroll
      for (int d = 0; d < 4; d++) {
        ra += ba.S[d] * (l[d] + ba.o[d]);
        rb += bb.S[d] * (l[d] + bb.o[d]);
        if (d == mu) { am = ba.S[d]; bm = bb.S[d]; }
        if (d == nu) { an = ba.S[d]; bn = bb.S[d]; }
      }
      m3 Umu;
      __syncthreads();   // the previous plane has been read by every thread
      if (edge && nu == 3) stage_plane_edge<RECON>(c, sU, sNb, tb, mu, nu, t0, own, ra, rb, Umu);
      else stage_plane<RECON>(c, sU, sNb, tb, mu, nu, own, ra, rb, Umu);
      __syncthreads();
      if (half == 0) {
        i_fhat_staged(sU, Umu, ra, am, an, rb, bm, bn, e);
      } else {
        i_fhat_staged(sU, Umu, ra, am, an, rb, bm, bn, h);
      }
    }
    // e = i E_k, h = i B_k;  G_k = kappa csw i(+-E_k - B_k) for the two chiral blocks
    if (step == 0) {          // G_3: the diagonal 3x3 blocks  1 + G_3  and  1 - G_3
#pragma unroll
      for (int ch = 0; ch < 2; ch++) {
        double G[9];
#pragma unroll
        for (int r = 0; r < 9; r++) G[r] = cc * ((ch == 0 ? e[r] : -e[r]) - h[r]);
        put(ch, 0, one + G[0], one + G[1]);
        put(ch, 1, one + G[2], one - G[0]);
        put(ch, 2, one - G[1], one - G[2]);
        put(ch, 3, G[3], G[4]);     // (1,0)
        put(ch, 4, G[5], G[6]);     // (2,0)
        put(ch, 5, G[7], G[8]);     // (2,1)
        put(ch, 12, -G[3], -G[4]);  // (4,3)
        put(ch, 16, -G[5], -G[6]);  // (5,3)
        put(ch, 17, -G[7], -G[8]);  // (5,4)
      }
    } else if (step == 1) {   // G_1: parked
#pragma unroll
      for (int r = 0; r < 9; r++) { sG[r * CT_THREADS] = e[r]; sG[(9 + r) * CT_THREADS] = h[r]; }
    } else {                  // G_2: lower-left block G_1 + i G_2, rows 3 + a, columns b
#pragma unroll
      for (int ch = 0; ch < 2; ch++) {
        double G1[9], G2[9];
#pragma unroll
        for (int r = 0; r < 9; r++) {
          const double e1 = sG[r * CT_THREADS], b1 = sG[(9 + r) * CT_THREADS];
          G1[r] = cc * ((ch == 0 ? e1 : -e1) - b1);
          G2[r] = cc * ((ch == 0 ? e[r] : -e[r]) - h[r]);
        }
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
          for (int b = 0; b < 3; b++) {
            const double2 g1 = herm_at(G1, a, b), g2 = herm_at(G2, a, b);
            put(ch, 3 + (3 + a) * (2 + a) / 2 + b, g1.x - g2.y, g1.y + g2.x);
          }
      }
    }
  }
}

// A^-1 from the packed blocks (one thread per site and chirality)
template <typename T>
__global__ void __launch_bounds__(128) clover_invert_kernel(const Geom g, const typename vec2<T>::type* A, typename vec2<T>::type* Ainv) {
  typedef typename vec2<T>::type T2;
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 4 * g.Vh) return;
  const int j = (int)(idx % g.TV);
  long long q = idx / g.TV;
  const int ch = (int)(q & 1);
  q >>= 1;   // parity * ntiles + tile
  const size_t off = ((size_t)q * 36 + 18 * ch) * g.TV + j;
  double2 a[6][6];
#pragma unroll
  for (int k = 0; k < 3; k++) {
    const T2 d = A[off + (size_t)k * g.TV];
    a[2 * k][2 * k] = make_double2((double)d.x, 0.0);
    a[2 * k + 1][2 * k + 1] = make_double2((double)d.y, 0.0);
  }
#pragma unroll
  for (int i = 1; i < 6; i++)
#pragma unroll
    for (int jj = 0; jj < i; jj++) {
      const T2 v = A[off + (size_t)(3 + i * (i - 1) / 2 + jj) * g.TV];
      a[i][jj] = make_double2((double)v.x, (double)v.y);
      a[jj][i] = make_double2((double)v.x, -(double)v.y);
    }
  invert6(a);
  store_packed<T>(Ainv + off, g.TV, a);
}

// LQCD_CLOVER_TILE=0 keeps the one-thread-per-site kernel for every geometry (A/B runs)
static bool tile_kernel_enabled() {
  static const bool on = [] {
    const char* e = getenv("LQCD_CLOVER_TILE");
    return !(e && e[0] == '0');
  }();
  return on;
}

// the table lives in a __device__ array, one copy per device: uploaded on a device's first build
static cudaError_t ct_table_upload(cudaStream_t s) {
  static std::mutex mu;
  static std::vector<uint32_t> host;
  static bool done[64] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lk(mu);
  if (dev < 64 && done[dev]) return cudaSuccess;
  if (host.empty()) {
    host.resize((size_t)2 * 6 * CT_NIT * CT_THREADS);
    ct_table_build(host.data());
  }
  e = cudaMemcpyToSymbolAsync(ct_table, host.data(), host.size() * sizeof(uint32_t), 0, cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess) return e;
  e = cudaStreamSynchronize(s);   // pageable source: keep it simple, this happens once per device
  if (e == cudaSuccess && dev < 64) done[dev] = true;
  return e;
}

template <typename T, int RECON>
static cudaError_t clover_tile_launch(const CloverCtx& c, const CloverParm& cp, void* clover, void* clover_inv, cudaStream_t s) {
  typedef typename vec2<T>::type T2;
  cudaError_t e = ct_table_upload(s);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(clover_tile_kernel<T, RECON>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CT_SMEM);
  if (e != cudaSuccess) return e;
  clover_tile_kernel<T, RECON><<<2u * (unsigned)c.g.ntiles, CT_THREADS, CT_SMEM, s>>>(c, cp, (T2*)clover);
  count_launch();
  if (clover_inv) {
    const unsigned blocks = (unsigned)((4 * c.g.Vh + 127) / 128);
    clover_invert_kernel<T><<<blocks, 128, 0, s>>>(c.g, (const T2*)clover, (T2*)clover_inv);
    count_launch();
  }
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
  // 4^4 tiles: the staged kernel.  The inverse is then taken from the stored blocks, which is only the same as
  // inverting before rounding when the blocks are stored in fp64; a partial build (t_lo / t_hi) has no inverse.
  const bool tiles4 = g.b[0] == 4 && g.b[1] == 4 && g.b[2] == 4 && g.b[3] == 4 && (size_t)g.smem_optin >= CT_SMEM;
  if (tiles4 && tile_kernel_enabled() && (!inv || (f64 && cp.t_lo <= 0 && cp.t_hi >= g.L[3]))) {
    if (f64) return r12 ? clover_tile_launch<double, 12>(c, cp, clover, clover_inv, s) : clover_tile_launch<double, 18>(c, cp, clover, clover_inv, s);
    return r12 ? clover_tile_launch<float, 12>(c, cp, clover, clover_inv, s) : clover_tile_launch<float, 18>(c, cp, clover, clover_inv, s);
  }
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
