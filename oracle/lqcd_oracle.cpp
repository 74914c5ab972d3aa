// lqcd_oracle.cpp -- CPU ORACLE (test infrastructure, NOT the product).
//
// Plain, slow, fp64 implementation of the hot path of arxiv 2503.16994 (LatticeGPU.jl):
// the O(a)-improved Wilson-Dirac operator `Dw!`, the clover term `Csw!`
// (PAPER.md:123), `CG!` on the normal equations and `propagator!`.
// The paper prints no formula for any of them; the definitions used here are the readings
// D1-D8 / R1-R16 of SURVEY.md section 8(c), restated in DESIGN.md.  Every function below is the
// definition written out with dense 4x4 gamma matrices and naive loops; nothing is blocked,
// spin-projected, fused or reordered.  OpenMP appears on outer site loops only.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
// this library.  It shares no code, header, table or constant with paper_2503_16994_b200/csrc.
//
// Pins (tests/test_oracle_pins.py): free-field closed form (P1), gamma5-hermiticity (P2), gauge
// covariance (P3), dense 2^4 matrix built from the element formula in numpy (P4), constant abelian
// flux closed form for the clover term (P5), antiperiodic equivalence (P6), Dirichlet structure
// (P7), CG = dense inverse (P8), even-odd = full (P10), plaquette of the generator (P11), free-field
// pseudoscalar correlator from the momentum-space propagator (P12: point source + CG + contraction).
// Parity unpinned: the value dependence of the c~_t boundary term (R10) beyond "ct=1 is absent and
// the term is linear in (ct-1)".
//
// Canonical layouts: site n = x1 + L1*(x2 + L2*(x3 + L3*x4)), x4 = time;
// gauge [n][mu][row][col] complex; spinor [n][spin][colour] complex; clover blocks
// [n][chirality][6][6] complex with row index 3*s + a (s = spin inside the chirality, a = colour).

#include <complex>
#include <cmath>
#include <cstring>
#include <cstdlib>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;
static const cd I_(0.0, 1.0);

enum { BC_PERIODIC = 0, BC_OPEN = 1, BC_SF_ORBI = 2, BC_SF_AFWB = 3 };

struct Lat {
    int L[4];
    int bc;
    long V;
    cd theta[4];      // per-link phase factor exp(i*angle/L_mu)   (D3, R6)
    double phiT[3];   // SF boundary phases at x4 = T               (D7, R8)
    double mu;        // twisted mass ("mu is the twisted mass"): D = A + 2 i kappa mu gamma5 - kappa H
};
// NEXT-4: the twisted mass is a state of this library (oracle_set_twisted_mass), read when a lattice is set up;
// the Python wrapper sets it before and clears it after each call.  Even-odd routines do not support it.
static double g_twisted_mu = 0.0;

// ----------------------------------------------------------------------------------------------
// D2: gamma matrices, chiral basis.  gamma_k = [[0,-i sigma_k],[+i sigma_k,0]], gamma_4 = [[0,1],[1,0]]
// ----------------------------------------------------------------------------------------------
static cd GAM[4][4][4];      // GAM[mu][s][s']
static cd GAM5[4][4];
static cd SIG[4][4][4][4];   // SIG[mu][nu] = (i/2) [gamma_mu, gamma_nu]
static bool gam_ready = false;

static void init_gamma() {
    if (gam_ready) return;
    cd pauli[3][2][2] = {
        {{0, 1}, {1, 0}},
        {{0, -I_}, {I_, 0}},
        {{1, 0}, {0, -1}}};
    memset(GAM, 0, sizeof(GAM));
    for (int k = 0; k < 3; k++)
        for (int a = 0; a < 2; a++)
            for (int b = 0; b < 2; b++) {
                GAM[k][a][2 + b] = -I_ * pauli[k][a][b];
                GAM[k][2 + a][b] = +I_ * pauli[k][a][b];
            }
    for (int a = 0; a < 2; a++) {
        GAM[3][a][2 + a] = 1.0;
        GAM[3][2 + a][a] = 1.0;
    }
    // gamma5 = gamma1 gamma2 gamma3 gamma4
    cd t1[4][4], t2[4][4];
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            t1[i][j] = 0;
            for (int k = 0; k < 4; k++) t1[i][j] += GAM[0][i][k] * GAM[1][k][j];
        }
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            t2[i][j] = 0;
            for (int k = 0; k < 4; k++) t2[i][j] += t1[i][k] * GAM[2][k][j];
        }
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            GAM5[i][j] = 0;
            for (int k = 0; k < 4; k++) GAM5[i][j] += t2[i][k] * GAM[3][k][j];
        }
    for (int mu = 0; mu < 4; mu++)
        for (int nu = 0; nu < 4; nu++)
            for (int i = 0; i < 4; i++)
                for (int j = 0; j < 4; j++) {
                    cd ab = 0, ba = 0;
                    for (int k = 0; k < 4; k++) {
                        ab += GAM[mu][i][k] * GAM[nu][k][j];
                        ba += GAM[nu][i][k] * GAM[mu][k][j];
                    }
                    SIG[mu][nu][i][j] = 0.5 * I_ * (ab - ba);
                }
    gam_ready = true;
}

// ----------------------------------------------------------------------------------------------
// D1: geometry
// ----------------------------------------------------------------------------------------------
static inline long site_index(const Lat& g, const int x[4]) {
    return x[0] + (long)g.L[0] * (x[1] + (long)g.L[1] * (x[2] + (long)g.L[2] * x[3]));
}
static inline void site_coords(const Lat& g, long n, int x[4]) {
    x[0] = (int)(n % g.L[0]); n /= g.L[0];
    x[1] = (int)(n % g.L[1]); n /= g.L[1];
    x[2] = (int)(n % g.L[2]); n /= g.L[2];
    x[3] = (int)n;
}
// D7: frozen time slices (psi == 0 there; output of D is 0 there)
static inline bool frozen(const Lat& g, int x4) {
    if (g.bc == BC_OPEN) return x4 == 0 || x4 == g.L[3] - 1;
    if (g.bc == BC_SF_ORBI || g.bc == BC_SF_AFWB) return x4 == 0;
    return false;
}
static inline int wrap(int c, int L) { return ((c % L) + L) % L; }

static Lat make_lat(const int L[4], int bc, const double theta[4], const double phiT[3]) {
    Lat g;
    for (int i = 0; i < 4; i++) g.L[i] = L[i];
    g.bc = bc;
    g.V = (long)L[0] * L[1] * L[2] * L[3];
    for (int i = 0; i < 4; i++) {
        double ang = theta ? theta[i] / L[i] : 0.0;
        g.theta[i] = cd(cos(ang), sin(ang));
    }
    for (int i = 0; i < 3; i++) g.phiT[i] = phiT ? phiT[i] : 0.0;
    g.mu = g_twisted_mu;
    init_gamma();
    return g;
}

// ----------------------------------------------------------------------------------------------
// 3x3 helpers
// ----------------------------------------------------------------------------------------------
struct M3 { cd m[3][3]; };
static inline M3 mul(const M3& a, const M3& b) {
    M3 c;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            c.m[i][j] = 0;
            for (int k = 0; k < 3; k++) c.m[i][j] += a.m[i][k] * b.m[k][j];
        }
    return c;
}
static inline M3 dag(const M3& a) {
    M3 c;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) c.m[i][j] = std::conj(a.m[j][i]);
    return c;
}
static inline M3 add(const M3& a, const M3& b) {
    M3 c;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) c.m[i][j] = a.m[i][j] + b.m[i][j];
    return c;
}

// Link U_mu(x) for a point x that may lie one or two steps outside the stored box.
// Spatial directions always wrap.  Time: periodic wraps; SF: slice x4 == L4 (= T) is the fixed
// boundary W'_k = exp(i diag(phiT)/L_k) (D7, R8; form of W: PAPER.md:84); open: never outside.
static M3 link(const Lat& g, const cd* U, const int xin[4], int mu) {
    int x[4];
    for (int i = 0; i < 3; i++) x[i] = wrap(xin[i], g.L[i]);
    x[3] = xin[3];
    bool sf = (g.bc == BC_SF_ORBI || g.bc == BC_SF_AFWB);
    if (g.bc == BC_PERIODIC) x[3] = wrap(x[3], g.L[3]);
    if (sf && x[3] == g.L[3]) {
        M3 w;
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) w.m[i][j] = 0;
        if (mu < 3)
            for (int i = 0; i < 3; i++) {
                double a = g.phiT[i] / g.L[mu];
                w.m[i][i] = cd(cos(a), sin(a));
            }
        else  // a time link starting on slice T is never part of any leaf of an interior site
            for (int i = 0; i < 3; i++) w.m[i][i] = cd(NAN, NAN);
        return w;
    }
    if (x[3] < 0 || x[3] >= g.L[3]) {  // not reachable from interior sites (D7); poison it
        M3 w;
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) w.m[i][j] = cd(NAN, NAN);
        return w;
    }
    M3 r;
    const cd* p = U + (site_index(g, x) * 4 + mu) * 9;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) r.m[i][j] = p[i * 3 + j];
    return r;
}

static inline void shift(const int x[4], int mu, int d, int y[4]) {
    for (int i = 0; i < 4; i++) y[i] = x[i];
    y[mu] += d;
}

// D4: F^_{mu nu}(x) = (Q - Q^dagger)/8, Q = sum of the four plaquette leaves in the mu-nu plane,
// all starting and ending at x, counter-clockwise; trace not subtracted (R3), theta not included.
static M3 fhat(const Lat& g, const cd* U, const int x[4], int mu, int nu) {
    int xpm[4], xpn[4], xmm[4], xmn[4], xmmpn[4], xmmmn[4], xpmmn[4];
    shift(x, mu, +1, xpm);
    shift(x, nu, +1, xpn);
    shift(x, mu, -1, xmm);
    shift(x, nu, -1, xmn);
    shift(xmm, nu, +1, xmmpn);
    shift(xmm, nu, -1, xmmmn);
    shift(xpm, nu, -1, xpmmn);
    // leaf 1: U_mu(x) U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+
    M3 l1 = mul(mul(link(g, U, x, mu), link(g, U, xpm, nu)),
                mul(dag(link(g, U, xpn, mu)), dag(link(g, U, x, nu))));
    // leaf 2: U_nu(x) U_mu(x-mu+nu)^+ U_nu(x-mu)^+ U_mu(x-mu)
    M3 l2 = mul(mul(link(g, U, x, nu), dag(link(g, U, xmmpn, mu))),
                mul(dag(link(g, U, xmm, nu)), link(g, U, xmm, mu)));
    // leaf 3: U_mu(x-mu)^+ U_nu(x-mu-nu)^+ U_mu(x-mu-nu) U_nu(x-nu)
    M3 l3 = mul(mul(dag(link(g, U, xmm, mu)), dag(link(g, U, xmmmn, nu))),
                mul(link(g, U, xmmmn, mu), link(g, U, xmn, nu)));
    // leaf 4: U_nu(x-nu)^+ U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^+
    M3 l4 = mul(mul(dag(link(g, U, xmn, nu)), link(g, U, xmn, mu)),
                mul(link(g, U, xpmmn, nu), dag(link(g, U, x, mu))));
    M3 Q = add(add(l1, l2), add(l3, l4));
    M3 Qd = dag(Q);
    M3 F;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) F.m[i][j] = (Q.m[i][j] - Qd.m[i][j]) / 8.0;
    return F;
}

// D5: A(x) = 1 + kappa*csw*(i/2) sum_{mu,nu} sigma_{mu nu} (x) F^_{mu nu}(x)  as a dense 12x12
// matrix, index 3*spin + colour.  On frozen slices A = 1 (D7).  R10: + 2 kappa (ct-1) on the
// slices next to a frozen slice.
static void clover_site_dense(const Lat& g, const cd* U, const int x[4], double kappa, double csw,
                              double ct, cd A[12][12]) {
    for (int i = 0; i < 12; i++)
        for (int j = 0; j < 12; j++) A[i][j] = (i == j) ? 1.0 : 0.0;
    if (frozen(g, x[3])) return;
    if (csw != 0.0) {
        for (int mu = 0; mu < 4; mu++)
            for (int nu = 0; nu < 4; nu++) {
                if (mu == nu) continue;
                M3 F = fhat(g, U, x, mu, nu);
                for (int s = 0; s < 4; s++)
                    for (int sp = 0; sp < 4; sp++)
                        for (int a = 0; a < 3; a++)
                            for (int b = 0; b < 3; b++)
                                A[3 * s + a][3 * sp + b] +=
                                    kappa * csw * 0.5 * I_ * SIG[mu][nu][s][sp] * F.m[a][b];
            }
    }
    if (g.bc != BC_PERIODIC && ct != 1.0) {
        int last = (g.bc == BC_OPEN) ? g.L[3] - 2 : g.L[3] - 1;
        double add_ = 0.0;
        if (x[3] == 1) add_ += 2.0 * kappa * (ct - 1.0);
        if (x[3] == last) add_ += 2.0 * kappa * (ct - 1.0);
        for (int i = 0; i < 12; i++) A[i][i] += add_;
    }
}

// Spinor at a (possibly out-of-box) point: spatial wrap; time wrap for periodic; zero on frozen
// slices and outside the box (D7: mask, never multiply, so NaNs stored there cannot leak).
// g5in: read gamma5*psi instead of psi (for D^dagger = gamma5 D gamma5).
static inline void psi_at(const Lat& g, const cd* psi, const int xin[4], bool g5in, cd out[12]) {
    int x[4];
    for (int i = 0; i < 3; i++) x[i] = wrap(xin[i], g.L[i]);
    x[3] = wrap(xin[3], g.L[3]);
    if (g.bc != BC_PERIODIC && (xin[3] < 0 || xin[3] >= g.L[3] || frozen(g, x[3]))) {
        for (int i = 0; i < 12; i++) out[i] = 0;
        return;
    }
    const cd* p = psi + site_index(g, x) * 12;
    for (int s = 0; s < 4; s++)
        for (int a = 0; a < 3; a++) {
            cd v = 0;
            if (g5in) {
                for (int sp = 0; sp < 4; sp++) v += GAM5[s][sp] * p[3 * sp + a];
            } else
                v = p[3 * s + a];
            out[3 * s + a] = v;
        }
}

// D3: (H psi)(x) = sum_mu [ theta_mu (1-gamma_mu) U_mu(x) psi(x+mu) + theta_mu^* (1+gamma_mu) U_mu(x-mu)^+ psi(x-mu) ]
static void hop_site(const Lat& g, const cd* U, const cd* psi, const int x[4], bool g5in, cd out[12]) {
    for (int i = 0; i < 12; i++) out[i] = 0;
    for (int mu = 0; mu < 4; mu++) {
        int xp[4], xm[4];
        shift(x, mu, +1, xp);
        shift(x, mu, -1, xm);
        cd pf[12], pb[12];
        psi_at(g, psi, xp, g5in, pf);
        psi_at(g, psi, xm, g5in, pb);
        bool fzero = true, bzero = true;
        for (int i = 0; i < 12; i++) {
            if (pf[i] != 0.0) fzero = false;
            if (pb[i] != 0.0) bzero = false;
        }
        if (!fzero) {  // forward: theta (1-gamma) U_mu(x) psi(x+mu)
            M3 u = link(g, U, x, mu);
            for (int s = 0; s < 4; s++)
                for (int a = 0; a < 3; a++) {
                    cd acc = 0;
                    for (int sp = 0; sp < 4; sp++) {
                        cd pr = ((s == sp) ? 1.0 : 0.0) - GAM[mu][s][sp];
                        if (pr == 0.0) continue;
                        for (int b = 0; b < 3; b++) acc += pr * u.m[a][b] * pf[3 * sp + b];
                    }
                    out[3 * s + a] += g.theta[mu] * acc;
                }
        }
        if (!bzero) {  // backward: theta^* (1+gamma) U_mu(x-mu)^+ psi(x-mu)
            M3 u = dag(link(g, U, xm, mu));
            for (int s = 0; s < 4; s++)
                for (int a = 0; a < 3; a++) {
                    cd acc = 0;
                    for (int sp = 0; sp < 4; sp++) {
                        cd pr = ((s == sp) ? 1.0 : 0.0) + GAM[mu][s][sp];
                        if (pr == 0.0) continue;
                        for (int b = 0; b < 3; b++) acc += pr * u.m[a][b] * pb[3 * sp + b];
                    }
                    out[3 * s + a] += std::conj(g.theta[mu]) * acc;
                }
        }
    }
}

// D6 at one site: (D psi)(x) = A(x) psi(x) - kappa (H psi)(x); zero on frozen slices.
// Ablk = [2][6][6] chiral blocks of A(x), or NULL => A = 1 (csw = 0, "once Csw! is
// called the term is added").  g5: apply gamma5 to input and output (D^dagger = gamma5 D gamma5).
static void dw_site(const Lat& g, const cd* U, const cd* Ablk, const cd* psi, const int x[4],
                    double kappa, bool g5, cd out[12]) {
    if (frozen(g, x[3])) {
        for (int i = 0; i < 12; i++) out[i] = 0;
        return;
    }
    cd h[12], p[12], r[12];
    hop_site(g, U, psi, x, g5, h);
    psi_at(g, psi, x, g5, p);
    for (int i = 0; i < 12; i++) r[i] = p[i];
    if (Ablk) {
        for (int c = 0; c < 2; c++)
            for (int i = 0; i < 6; i++) {
                cd acc = 0;
                for (int j = 0; j < 6; j++) acc += Ablk[(c * 6 + i) * 6 + j] * p[6 * c + j];
                r[6 * c + i] = acc;
            }
    }
    for (int i = 0; i < 12; i++) r[i] -= kappa * h[i];
    if (g.mu != 0.0) {
        // + 2 i kappa mu gamma5 psi; D^dagger = gamma5 D(-mu) gamma5, so the conjugated path (g5) carries -mu
        const double m = 2.0 * kappa * (g5 ? -g.mu : g.mu);
        for (int s = 0; s < 4; s++)
            for (int a = 0; a < 3; a++) {
                cd v = 0;
                for (int sp = 0; sp < 4; sp++) v += GAM5[s][sp] * p[3 * sp + a];
                r[3 * s + a] += I_ * m * v;
            }
    }
    if (g5) {
        for (int s = 0; s < 4; s++)
            for (int a = 0; a < 3; a++) {
                cd v = 0;
                for (int sp = 0; sp < 4; sp++) v += GAM5[s][sp] * r[3 * sp + a];
                out[3 * s + a] = v;
            }
    } else
        for (int i = 0; i < 12; i++) out[i] = r[i];
}

// ----------------------------------------------------------------------------------------------
// field-level routines
// ----------------------------------------------------------------------------------------------
static void clover_blocks(const Lat& g, const cd* U, double kappa, double csw, double ct, cd* Ablk) {
#pragma omp parallel for schedule(static)
    for (long n = 0; n < g.V; n++) {
        int x[4];
        site_coords(g, n, x);
        cd A[12][12];
        clover_site_dense(g, U, x, kappa, csw, ct, A);
        for (int c = 0; c < 2; c++)
            for (int i = 0; i < 6; i++)
                for (int j = 0; j < 6; j++) Ablk[((n * 2 + c) * 6 + i) * 6 + j] = A[6 * c + i][6 * c + j];
    }
}

static void dw_field(const Lat& g, const cd* U, const cd* Ablk, const cd* in, cd* out, double kappa,
                     bool dagger) {
#pragma omp parallel for schedule(static)
    for (long n = 0; n < g.V; n++) {
        int x[4];
        site_coords(g, n, x);
        dw_site(g, U, Ablk ? Ablk + n * 72 : nullptr, in, x, kappa, dagger, out + n * 12);
    }
}

static double norm2(const cd* v, long n) {
    double s = 0;
#pragma omp parallel for reduction(+ : s) schedule(static)
    for (long i = 0; i < n; i++) s += std::norm(v[i]);
    return s;
}

// 6x6 complex inverse by Gauss-Jordan with partial pivoting (plain definition of A^{-1})
static void inv6(const cd* a, cd* inv) {
    cd m[6][12];
    for (int i = 0; i < 6; i++)
        for (int j = 0; j < 6; j++) {
            m[i][j] = a[i * 6 + j];
            m[i][6 + j] = (i == j) ? 1.0 : 0.0;
        }
    for (int c = 0; c < 6; c++) {
        int piv = c;
        for (int r = c + 1; r < 6; r++)
            if (std::abs(m[r][c]) > std::abs(m[piv][c])) piv = r;
        if (piv != c)
            for (int j = 0; j < 12; j++) std::swap(m[c][j], m[piv][j]);
        cd d = 1.0 / m[c][c];
        for (int j = 0; j < 12; j++) m[c][j] *= d;
        for (int r = 0; r < 6; r++) {
            if (r == c) continue;
            cd f = m[r][c];
            for (int j = 0; j < 12; j++) m[r][j] -= f * m[c][j];
        }
    }
    for (int i = 0; i < 6; i++)
        for (int j = 0; j < 6; j++) inv[i * 6 + j] = m[i][6 + j];
}

static inline int parity_of(const int x[4]) { return (x[0] + x[1] + x[2] + x[3]) & 1; }

// out(x) = (H in)(x) on sites of parity `par`, 0 elsewhere (D8: H_eo / H_oe with the D7 masks)
static void hop_field_parity(const Lat& g, const cd* U, const cd* in, cd* out, int par) {
#pragma omp parallel for schedule(static)
    for (long n = 0; n < g.V; n++) {
        int x[4];
        site_coords(g, n, x);
        cd* o = out + n * 12;
        if (parity_of(x) != par || frozen(g, x[3])) {
            for (int i = 0; i < 12; i++) o[i] = 0;
            continue;
        }
        hop_site(g, U, in, x, false, o);
    }
}
// out(x) = B(x) in(x) on sites of parity par (B = [V][2][6][6] blocks), 0 elsewhere / frozen
static void blk_field_parity(const Lat& g, const cd* B, const cd* in, cd* out, int par) {
#pragma omp parallel for schedule(static)
    for (long n = 0; n < g.V; n++) {
        int x[4];
        site_coords(g, n, x);
        cd* o = out + n * 12;
        if (parity_of(x) != par || frozen(g, x[3])) {
            for (int i = 0; i < 12; i++) o[i] = 0;
            continue;
        }
        for (int c = 0; c < 2; c++)
            for (int i = 0; i < 6; i++) {
                cd acc = 0;
                for (int j = 0; j < 6; j++) acc += B[((n * 2 + c) * 6 + i) * 6 + j] * in[n * 12 + 6 * c + j];
                o[6 * c + i] = acc;
            }
    }
}
static void gamma5_field(const Lat& g, const cd* in, cd* out) {
#pragma omp parallel for schedule(static)
    for (long n = 0; n < g.V; n++)
        for (int s = 0; s < 4; s++)
            for (int a = 0; a < 3; a++) {
                cd v = 0;
                for (int sp = 0; sp < 4; sp++) v += GAM5[s][sp] * in[n * 12 + 3 * sp + a];
                out[n * 12 + 3 * s + a] = v;
            }
}

// D8: D^ psi_e = A_ee psi_e - kappa^2 H_eo A_oo^{-1} H_oe psi_e  (full-lattice arrays, odd part 0)
static void dhat_field(const Lat& g, const cd* U, const cd* Ablk, const cd* Ainv, const cd* in,
                       cd* out, double kappa, bool dagger) {
    long N = g.V * 12;
    std::vector<cd> src(N), t1(N), t2(N), t3(N), t4(N);
    if (dagger) gamma5_field(g, in, src.data());
    else memcpy(src.data(), in, N * sizeof(cd));
    // keep the even part only
    for (long n = 0; n < g.V; n++) {
        int x[4];
        site_coords(g, n, x);
        if (parity_of(x) != 0 || frozen(g, x[3]))
            for (int i = 0; i < 12; i++) src[n * 12 + i] = 0;
    }
    hop_field_parity(g, U, src.data(), t1.data(), 1);       // H_oe psi_e
    blk_field_parity(g, Ainv, t1.data(), t2.data(), 1);     // A_oo^{-1} .
    hop_field_parity(g, U, t2.data(), t3.data(), 0);        // H_eo .
    blk_field_parity(g, Ablk, src.data(), t4.data(), 0);    // A_ee psi_e
    for (long i = 0; i < N; i++) t4[i] -= kappa * kappa * t3[i];
    if (dagger) gamma5_field(g, t4.data(), out);
    else memcpy(out, t4.data(), N * sizeof(cd));
}

// ----------------------------------------------------------------------------------------------
// CG on the normal equations, step by step as in SURVEY.md 8(c) "Algorithm CG" (R11):
//   b' = M^+ b; x = 0; r = b'; p = r; rho = |r|^2; rho0 = rho;
//   repeat { t = M p; alpha = rho/|t|^2; x += alpha p; r -= alpha M^+ t; rho' = |r|^2;
//            if rho' <= tol^2 rho0 stop; p = r + (rho'/rho) p; rho = rho' }
// M is passed as a callback so the same loop serves D and D^.
// ----------------------------------------------------------------------------------------------
template <class Op>
static int cg_normal(long N, Op M, const cd* b, cd* x, double tol, int maxiter, double* rel_normal,
                     double* rel_true) {
    std::vector<cd> bp(N), r(N), p(N), t(N), q(N);
    M(b, bp.data(), true);
    for (long i = 0; i < N; i++) { x[i] = 0; r[i] = bp[i]; p[i] = bp[i]; }
    double rho = norm2(r.data(), N), rho0 = rho;
    int it = 0;
    bool conv = (rho0 == 0.0);
    while (!conv && it < maxiter) {
        M(p.data(), t.data(), false);
        double alpha = rho / norm2(t.data(), N);
        M(t.data(), q.data(), true);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < N; i++) { x[i] += alpha * p[i]; r[i] -= alpha * q[i]; }
        double rhop = norm2(r.data(), N);
        it++;
        if (rhop <= tol * tol * rho0) { conv = true; break; }
        double beta = rhop / rho;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < N; i++) p[i] = r[i] + beta * p[i];
        rho = rhop;
    }
    // true residuals with fresh operator applications
    M(x, t.data(), false);
    for (long i = 0; i < N; i++) t[i] = b[i] - t[i];
    double nb = norm2(b, N);
    if (rel_true) *rel_true = nb > 0 ? sqrt(norm2(t.data(), N) / nb) : 0.0;
    M(t.data(), q.data(), true);
    if (rel_normal) *rel_normal = rho0 > 0 ? sqrt(norm2(q.data(), N) / rho0) : 0.0;
    return conv ? it : -it - 1;
}

// ----------------------------------------------------------------------------------------------
// C-ABI
// ----------------------------------------------------------------------------------------------
extern "C" {

void oracle_set_twisted_mass(double mu) { g_twisted_mu = mu; }

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}

// gamma_mu (mu = 0..3) and gamma5 (mu = 4) as 4x4 complex, row-major: lets tests check D2's algebra
void oracle_gamma(int mu, cd* out) {
    init_gamma();
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) out[i * 4 + j] = (mu < 4) ? GAM[mu][i][j] : GAM5[i][j];
}
void oracle_sigma(int mu, int nu, cd* out) {
    init_gamma();
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) out[i * 4 + j] = SIG[mu][nu][i][j];
}

// average plaquette (1/3) Re Tr over all sites and the 6 planes (periodic wrap in all directions)
double oracle_plaquette(const int L[4], const cd* U) {
    Lat g = make_lat(L, BC_PERIODIC, nullptr, nullptr);
    double s = 0;
#pragma omp parallel for reduction(+ : s) schedule(static)
    for (long n = 0; n < g.V; n++) {
        int x[4];
        site_coords(g, n, x);
        for (int mu = 0; mu < 4; mu++)
            for (int nu = mu + 1; nu < 4; nu++) {
                int xpm[4], xpn[4];
                shift(x, mu, 1, xpm);
                shift(x, nu, 1, xpn);
                M3 P = mul(mul(link(g, U, x, mu), link(g, U, xpm, nu)),
                           mul(dag(link(g, U, xpn, mu)), dag(link(g, U, x, nu))));
                s += (P.m[0][0] + P.m[1][1] + P.m[2][2]).real() / 3.0;
            }
    }
    return s / (6.0 * g.V);
}

// F^_{mu nu}(x) at one site (3x3 complex, row-major)
void oracle_fhat_site(const int L[4], int bc, const double phiT[3], const cd* U, const int x[4], int mu,
                      int nu, cd* out) {
    Lat g = make_lat(L, bc, nullptr, phiT);
    M3 F = fhat(g, U, x, mu, nu);
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) out[i * 3 + j] = F.m[i][j];
}

// dense 12x12 A(x) for every site: A12 = [V][12][12]
void oracle_clover_dense(const int L[4], int bc, const double phiT[3], double kappa, double csw, double ct,
                         const cd* U, cd* A12) {
    Lat g = make_lat(L, bc, nullptr, phiT);
#pragma omp parallel for schedule(static)
    for (long n = 0; n < g.V; n++) {
        int x[4];
        site_coords(g, n, x);
        cd A[12][12];
        clover_site_dense(g, U, x, kappa, csw, ct, A);
        for (int i = 0; i < 12; i++)
            for (int j = 0; j < 12; j++) A12[(n * 12 + i) * 12 + j] = A[i][j];
    }
}

// chiral 6x6 blocks of A(x): Ablk = [V][2][6][6]
void oracle_clover_blocks(const int L[4], int bc, const double phiT[3], double kappa, double csw, double ct,
                          const cd* U, cd* Ablk) {
    Lat g = make_lat(L, bc, nullptr, phiT);
    clover_blocks(g, U, kappa, csw, ct, Ablk);
}

// block-wise inverse: Ainv = [V][2][6][6]
void oracle_clover_inverse(const int L[4], const cd* Ablk, cd* Ainv) {
    long V = (long)L[0] * L[1] * L[2] * L[3];
#pragma omp parallel for schedule(static)
    for (long n = 0; n < 2 * V; n++) inv6(Ablk + n * 36, Ainv + n * 36);
}

// out = D in (dagger = 0) or D^+ in = gamma5 D gamma5 in (dagger = 1).  Ablk may be NULL (A = 1).
void oracle_dw(const int L[4], int bc, const double theta[4], double kappa, const cd* U, const cd* Ablk,
               const cd* in, cd* out, int dagger) {
    Lat g = make_lat(L, bc, theta, nullptr);
    dw_field(g, U, Ablk, in, out, kappa, dagger != 0);
}

// out = H in (hopping term alone, D3 with the D7 masks) -- for pins
void oracle_hop(const int L[4], int bc, const double theta[4], const cd* U, const cd* in, cd* out) {
    Lat g = make_lat(L, bc, theta, nullptr);
#pragma omp parallel for schedule(static)
    for (long n = 0; n < g.V; n++) {
        int x[4];
        site_coords(g, n, x);
        if (frozen(g, x[3]))
            for (int i = 0; i < 12; i++) out[n * 12 + i] = 0;
        else
            hop_site(g, U, in, x, false, out + n * 12);
    }
}

// (D in)(x) or (D^+ in)(x) at listed sites only, clover computed on the fly from the links
// (O(1) extra memory: for the 48^3x96 / 64^3x128 sampled parity checks).  out = [nsites][12]
void oracle_dw_at_sites(const int L[4], int bc, const double theta[4], const double phiT[3], double kappa,
                        double csw, double ct, const cd* U, const cd* in, int dagger, long nsites,
                        const long* sites, cd* out) {
    Lat g = make_lat(L, bc, theta, phiT);
#pragma omp parallel for schedule(dynamic)
    for (long k = 0; k < nsites; k++) {
        int x[4];
        site_coords(g, sites[k], x);
        cd A[12][12], blk[72];
        clover_site_dense(g, U, x, kappa, csw, ct, A);
        for (int c = 0; c < 2; c++)
            for (int i = 0; i < 6; i++)
                for (int j = 0; j < 6; j++) blk[(c * 6 + i) * 6 + j] = A[6 * c + i][6 * c + j];
        dw_site(g, U, blk, in, x, kappa, dagger != 0, out + k * 12);
    }
}

// even-odd Schur operator D^ (D8) on full-lattice arrays (odd part of in ignored, of out zero)
void oracle_dhat(const int L[4], int bc, const double theta[4], double kappa, const cd* U, const cd* Ablk,
                 const cd* Ainv, const cd* in, cd* out, int dagger) {
    Lat g = make_lat(L, bc, theta, nullptr);
    dhat_field(g, U, Ablk, Ainv, in, out, kappa, dagger != 0);
}

// CG for D^+ D x = D^+ b (R11).  Returns iterations (>= 0) or -(iterations)-1 if maxiter was hit.
int oracle_cg(const int L[4], int bc, const double theta[4], double kappa, const cd* U, const cd* Ablk,
              const cd* b, cd* x, double tol, int maxiter, double* rel_normal, double* rel_true) {
    Lat g = make_lat(L, bc, theta, nullptr);
    auto M = [&](const cd* in, cd* out, bool dagger) { dw_field(g, U, Ablk, in, out, kappa, dagger); };
    return cg_normal(g.V * 12, M, b, x, tol, maxiter, rel_normal, rel_true);
}

// Even-odd preconditioned solve of D x = b (D8):
//   b^_e = b_e + kappa H_eo A_oo^{-1} b_o ; CG on D^^+ D^ x_e = D^^+ b^_e ; x_o = A_oo^{-1}(b_o + kappa H_oe x_e)
int oracle_cg_eo(const int L[4], int bc, const double theta[4], double kappa, const cd* U, const cd* Ablk,
                 const cd* Ainv, const cd* b, cd* x, double tol, int maxiter, double* rel_normal,
                 double* rel_true) {
    Lat g = make_lat(L, bc, theta, nullptr);
    long N = g.V * 12;
    std::vector<cd> bm(N), bo(N), t1(N), t2(N), bh(N), xe(N);
    // D7: the solve lives on the interior; mask b on frozen slices
    for (long n = 0; n < g.V; n++) {
        int xx[4];
        site_coords(g, n, xx);
        bool fz = frozen(g, xx[3]);
        int par = parity_of(xx);
        for (int i = 0; i < 12; i++) {
            cd v = fz ? cd(0) : b[n * 12 + i];
            bm[n * 12 + i] = v;
            bo[n * 12 + i] = (par == 1) ? v : cd(0);
        }
    }
    blk_field_parity(g, Ainv, bo.data(), t1.data(), 1);
    hop_field_parity(g, U, t1.data(), t2.data(), 0);
    for (long n = 0; n < g.V; n++) {
        int xx[4];
        site_coords(g, n, xx);
        for (int i = 0; i < 12; i++)
            bh[n * 12 + i] = (parity_of(xx) == 0) ? bm[n * 12 + i] + kappa * t2[n * 12 + i] : cd(0);
    }
    auto M = [&](const cd* in, cd* out, bool dagger) { dhat_field(g, U, Ablk, Ainv, in, out, kappa, dagger); };
    double rn = 0;
    int it = cg_normal(N, M, bh.data(), xe.data(), tol, maxiter, &rn, nullptr);
    if (rel_normal) *rel_normal = rn;
    hop_field_parity(g, U, xe.data(), t1.data(), 1);
    for (long i = 0; i < N; i++) t1[i] = bo[i] + kappa * t1[i];
    blk_field_parity(g, Ainv, t1.data(), t2.data(), 1);
    for (long i = 0; i < N; i++) x[i] = xe[i] + t2[i];
    if (rel_true) {
        dw_field(g, U, Ablk, x, t1.data(), kappa, false);
        for (long i = 0; i < N; i++) t1[i] = bm[i] - t1[i];
        double nb = norm2(bm.data(), N);
        *rel_true = nb > 0 ? sqrt(norm2(t1.data(), N) / nb) : 0.0;
    }
    return it;
}

// NEXT-2 (SURVEY.md 8(f); PAPER.md:11 "different fermionic two point functions", :125 the propagator columns):
// pseudoscalar two-point function from ncol propagator columns S_c(x) (canonical spinors [V][4][3]),
//   C(x4) = sum over x1,x2,x3 of sum_c sum_{spin, colour} |S_c(x)|^2     ( = sum_xvec Tr S(x)^+ S(x) for the 12 columns
// of a point source, since gamma5-hermiticity turns Tr[gamma5 S gamma5 S^+] into it).  Plain loops, x4 slowest (D1).
void oracle_correlator_ps(const int L[4], const cd* cols, int ncol, double* C) {
    const long V = (long)L[0] * L[1] * L[2] * L[3];
    const long V3 = (long)L[0] * L[1] * L[2];
    for (int t = 0; t < L[3]; t++) {
        double s = 0.0;
        for (int c = 0; c < ncol; c++)
            for (long n = (long)t * V3; n < (long)(t + 1) * V3; n++)
                for (int k = 0; k < 12; k++) s += std::norm(cols[((long)c * V + n) * 12 + k]);
        C[t] = s;
    }
}

}  // extern "C"
