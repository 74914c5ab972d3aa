// lqcd_oracle_sun.cpp -- CPU ORACLE for the SU(2) fundamental representation (test infrastructure, NOT the product).
//
// PAPER.md:66-70 (section 2.2): gauge fields take values in SU3{T} or SU2{T}, SU(2) elements are stored in the
// Cayley-Dickson form g = (z1, z2), |z1|^2 + |z2|^2 = 1, and fermion fields are Spinor{4, REP} with REP = SU2fund or
// SU3fund.  The operators are the ones of lqcd_oracle.cpp (definitions D1-D8 of SURVEY.md 8(c), restated in DESIGN.md)
// with N colours instead of three:
//   (H psi)(x) = sum_mu [ theta_mu (1 - gamma_mu) U_mu(x) psi(x+mu) + theta_mu^* (1 + gamma_mu) U_mu(x-mu)^+ psi(x-mu) ]   (D3)
//   Q_{mu nu}(x) = sum of the four plaquette leaves, F^ = (Q - Q^+)/8                                               (D4)
//   A(x) = 1 + kappa csw (i/2) sum_{mu nu} sigma_{mu nu} (x) F^_{mu nu}(x), chirally block diagonal: two Hermitian
//          2N x 2N blocks, row index N*s + a (s = spin inside the chirality, a = colour)                            (D5)
//   D = A - kappa H,   D^+ = gamma5 D gamma5                                                                        (D6)
//   time boundaries: periodic, or open (psi = 0 on the first and last stored slice, D = P D P)                      (D7)
//   CG on D^+ D x = D^+ b from x = 0, stop when |r| <= tol |D^+ b|                                                  (CG, R11)
// Everything is the definition written out with dense gamma matrices and naive loops, templated on the number of
// colours N.  N = 2 is the representation under test.  N = 3 exists only so that this file can be pinned against the
// separately pinned SU(3) oracle (tests/test_oracle_su2_pins.py): the two share no code, so agreement of the N = 3
// instance with lqcd_oracle.cpp to rounding pins every index, sign and factor of the generic loops; the N = 2
// instance is pinned on its own by the free-field closed form, gamma5-hermiticity, SU(2) gauge covariance, a dense
// matrix built from the element formula in numpy, and the constant-flux closed form with t = diag(1, -1).
//
// Only tests/ and bench.py's cpu_baseline leg may load this library; it shares nothing with paper_2503_16994_b200/csrc.
// Canonical layouts: site n = x1 + L1*(x2 + L2*(x3 + L3*x4)); gauge [n][mu][N][N] complex (full matrices; the
// Cayley-Dickson pair of an SU(2) link is its first row); spinor [n][4][N]; blocks [n][2][2N][2N].

#include <complex>
#include <cmath>
#include <cstring>
#include <vector>

typedef std::complex<double> cd;
static const cd I_(0.0, 1.0);
enum { BC_PERIODIC = 0, BC_OPEN = 1 };

// D2: gamma_k = [[0, -i sigma_k], [+i sigma_k, 0]], gamma_4 = [[0, 1], [1, 0]], gamma5 = diag(1, 1, -1, -1)
static cd GAM[4][4][4], SIG[4][4][4][4];
static double G5[4] = {1.0, 1.0, -1.0, -1.0};
static bool ready = false;
static void init_gamma() {
    if (ready) return;
    const cd s[3][2][2] = {{{0, 1}, {1, 0}}, {{0, -I_}, {I_, 0}}, {{1, 0}, {0, -1}}};
    memset(GAM, 0, sizeof(GAM));
    for (int k = 0; k < 3; k++)
        for (int a = 0; a < 2; a++)
            for (int b = 0; b < 2; b++) {
                GAM[k][a][2 + b] = -I_ * s[k][a][b];
                GAM[k][2 + a][b] = I_ * s[k][a][b];
            }
    for (int a = 0; a < 2; a++) { GAM[3][a][2 + a] = 1.0; GAM[3][2 + a][a] = 1.0; }
    for (int m = 0; m < 4; m++)
        for (int n = 0; n < 4; n++)
            for (int a = 0; a < 4; a++)
                for (int b = 0; b < 4; b++) {
                    cd c = 0;
                    for (int e = 0; e < 4; e++) c += GAM[m][a][e] * GAM[n][e][b] - GAM[n][a][e] * GAM[m][e][b];
                    SIG[m][n][a][b] = 0.5 * I_ * c;
                }
    ready = true;
}

struct Lat {
    int L[4];
    int bc;
    long V;
    cd theta[4];
};
static Lat make_lat(const int* L, int bc, const double* theta) {
    Lat l;
    l.V = 1;
    for (int i = 0; i < 4; i++) { l.L[i] = L[i]; l.V *= L[i]; }
    l.bc = bc;
    for (int i = 0; i < 4; i++) l.theta[i] = theta ? std::exp(I_ * (theta[i] / L[i])) : cd(1.0, 0.0);
    return l;
}
static long site(const Lat& l, const int x[4]) { return x[0] + (long)l.L[0] * (x[1] + (long)l.L[1] * (x[2] + (long)l.L[2] * x[3])); }
static void coords(const Lat& l, long n, int x[4]) {
    for (int i = 0; i < 4; i++) { x[i] = (int)(n % l.L[i]); n /= l.L[i]; }
}
static bool frozen(const Lat& l, int x3) { return l.bc == BC_OPEN && (x3 == 0 || x3 == l.L[3] - 1); }
// x + d mu^, periodic wrap in every direction (the open lattice never uses a wrapped time neighbour: its slices are frozen)
static void shift(const Lat& l, const int x[4], int mu, int d, int y[4]) {
    for (int i = 0; i < 4; i++) y[i] = x[i];
    y[mu] = ((x[mu] + d) % l.L[mu] + l.L[mu]) % l.L[mu];
}

template <int N>
struct Mat {
    cd e[N][N];
};
template <int N>
static Mat<N> link(const Lat& l, const cd* U, const int x[4], int mu) {
    Mat<N> m;
    const cd* p = U + ((size_t)site(l, x) * 4 + mu) * N * N;
    for (int a = 0; a < N; a++)
        for (int b = 0; b < N; b++) m.e[a][b] = p[a * N + b];
    return m;
}
template <int N>
static Mat<N> mul(const Mat<N>& a, const Mat<N>& b) {
    Mat<N> c;
    for (int i = 0; i < N; i++)
        for (int j = 0; j < N; j++) {
            cd s = 0;
            for (int k = 0; k < N; k++) s += a.e[i][k] * b.e[k][j];
            c.e[i][j] = s;
        }
    return c;
}
template <int N>
static Mat<N> dag(const Mat<N>& a) {
    Mat<N> c;
    for (int i = 0; i < N; i++)
        for (int j = 0; j < N; j++) c.e[i][j] = std::conj(a.e[j][i]);
    return c;
}

// D4: the four leaves of the mu-nu plane, each starting and ending at x, counter-clockwise
template <int N>
static Mat<N> fhat(const Lat& l, const cd* U, const int x[4], int mu, int nu) {
    int xpm[4], xpn[4], xmm[4], xmn[4], xmmpn[4], xmmmn[4], xpmmn[4];
    shift(l, x, mu, +1, xpm);
    shift(l, x, nu, +1, xpn);
    shift(l, x, mu, -1, xmm);
    shift(l, x, nu, -1, xmn);
    shift(l, xmm, nu, +1, xmmpn);
    shift(l, xmm, nu, -1, xmmmn);
    shift(l, xpm, nu, -1, xpmmn);
    Mat<N> q1 = mul(mul(link<N>(l, U, x, mu), link<N>(l, U, xpm, nu)), mul(dag(link<N>(l, U, xpn, mu)), dag(link<N>(l, U, x, nu))));
    Mat<N> q2 = mul(mul(link<N>(l, U, x, nu), dag(link<N>(l, U, xmmpn, mu))), mul(dag(link<N>(l, U, xmm, nu)), link<N>(l, U, xmm, mu)));
    Mat<N> q3 = mul(mul(dag(link<N>(l, U, xmm, mu)), dag(link<N>(l, U, xmmmn, nu))), mul(link<N>(l, U, xmmmn, mu), link<N>(l, U, xmn, nu)));
    Mat<N> q4 = mul(mul(dag(link<N>(l, U, xmn, nu)), link<N>(l, U, xmn, mu)), mul(link<N>(l, U, xpmmn, nu), dag(link<N>(l, U, x, mu))));
    Mat<N> f;
    for (int i = 0; i < N; i++)
        for (int j = 0; j < N; j++) {
            cd q = q1.e[i][j] + q2.e[i][j] + q3.e[i][j] + q4.e[i][j];
            cd qd = std::conj(q1.e[j][i] + q2.e[j][i] + q3.e[j][i] + q4.e[j][i]);
            f.e[i][j] = (q - qd) / 8.0;
        }
    return f;
}

// D5: the dense (4N) x (4N) site-diagonal matrix, index N*spin + colour
template <int N>
static void clover_dense(const Lat& l, const cd* U, const int x[4], double kappa, double csw, cd* A /*[4N][4N]*/) {
    const int D = 4 * N;
    for (int i = 0; i < D * D; i++) A[i] = 0;
    for (int i = 0; i < D; i++) A[i * D + i] = 1.0;
    if (frozen(l, x[3]) || csw == 0.0) return;
    for (int mu = 0; mu < 4; mu++)
        for (int nu = 0; nu < 4; nu++) {
            if (mu == nu) continue;
            Mat<N> f = fhat<N>(l, U, x, mu, nu);
            for (int s = 0; s < 4; s++)
                for (int t = 0; t < 4; t++)
                    for (int a = 0; a < N; a++)
                        for (int b = 0; b < N; b++) A[(N * s + a) * D + (N * t + b)] += kappa * csw * 0.5 * I_ * SIG[mu][nu][s][t] * f.e[a][b];
        }
}

// (H psi)(x), dense (1 -+ gamma_mu) (x) U
template <int N>
static void hop_site(const Lat& l, const cd* U, const cd* psi, const int x[4], cd* out /*[4][N]*/) {
    for (int i = 0; i < 4 * N; i++) out[i] = 0;
    for (int mu = 0; mu < 4; mu++) {
        int xp[4], xm[4];
        shift(l, x, mu, +1, xp);
        shift(l, x, mu, -1, xm);
        const bool fwd_ok = !(mu == 3 && l.bc == BC_OPEN && frozen(l, xp[3]));   // a hop onto a frozen slice is not taken
        const bool bwd_ok = !(mu == 3 && l.bc == BC_OPEN && frozen(l, xm[3]));
        Mat<N> Uf = link<N>(l, U, x, mu), Ub = dag(link<N>(l, U, xm, mu));
        const cd* pf = psi + (size_t)site(l, xp) * 4 * N;
        const cd* pb = psi + (size_t)site(l, xm) * 4 * N;
        for (int s = 0; s < 4; s++)
            for (int a = 0; a < N; a++) {
                cd acc = 0;
                for (int t = 0; t < 4; t++) {
                    const cd pm = (s == t ? 1.0 : 0.0) - GAM[mu][s][t], pp = (s == t ? 1.0 : 0.0) + GAM[mu][s][t];
                    for (int b = 0; b < N; b++) {
                        if (fwd_ok) acc += l.theta[mu] * pm * Uf.e[a][b] * pf[t * N + b];
                        if (bwd_ok) acc += std::conj(l.theta[mu]) * pp * Ub.e[a][b] * pb[t * N + b];
                    }
                }
                out[s * N + a] += acc;
            }
    }
}

// D6 with the blocks given (or A = 1): out = D psi or gamma5 D gamma5 psi
template <int N>
static void dw(const Lat& l, double kappa, const cd* U, const cd* Ablk, const cd* psi, cd* out, int dagger) {
    const int B = 2 * N;
    std::vector<cd> in((size_t)l.V * 4 * N);
    for (long n = 0; n < l.V; n++)
        for (int s = 0; s < 4; s++)
            for (int a = 0; a < N; a++) in[(size_t)n * 4 * N + s * N + a] = (dagger ? G5[s] : 1.0) * psi[(size_t)n * 4 * N + s * N + a];
#pragma omp parallel for
    for (long n = 0; n < l.V; n++) {
        int x[4];
        coords(l, n, x);
        cd* o = out + (size_t)n * 4 * N;
        if (frozen(l, x[3])) {
            for (int i = 0; i < 4 * N; i++) o[i] = 0;
            continue;
        }
        cd h[4 * 3];
        hop_site<N>(l, U, in.data(), x, h);
        for (int s = 0; s < 4; s++)
            for (int a = 0; a < N; a++) {
                cd d = in[(size_t)n * 4 * N + s * N + a];
                if (Ablk) {   // chirality ch = s / 2, row N*(s%2) + a of the block
                    const int ch = s / 2;
                    const cd* blk = Ablk + ((size_t)n * 2 + ch) * B * B;
                    d = 0;
                    for (int t = 0; t < 2; t++)
                        for (int b = 0; b < N; b++) d += blk[(N * (s % 2) + a) * B + (N * t + b)] * in[(size_t)n * 4 * N + (2 * ch + t) * N + b];
                }
                o[s * N + a] = (dagger ? G5[s] : 1.0) * (d - kappa * h[s * N + a]);
            }
    }
}

template <int N>
static void clover_blocks(const Lat& l, double kappa, double csw, const cd* U, cd* out) {
    const int D = 4 * N, B = 2 * N;
#pragma omp parallel for
    for (long n = 0; n < l.V; n++) {
        int x[4];
        coords(l, n, x);
        cd A[12 * 12];
        clover_dense<N>(l, U, x, kappa, csw, A);
        for (int ch = 0; ch < 2; ch++)
            for (int i = 0; i < B; i++)
                for (int j = 0; j < B; j++) out[(((size_t)n * 2 + ch) * B + i) * B + j] = A[(B * ch + i) * D + (B * ch + j)];
    }
}

static double norm2(const std::vector<cd>& v) {
    double s = 0;
    for (size_t i = 0; i < v.size(); i++) s += std::norm(v[i]);
    return s;
}

// CG on the normal equations, step by step (SURVEY.md 8(c) "Algorithm CG")
template <int N>
static int cg(const Lat& l, double kappa, const cd* U, const cd* Ablk, const cd* b, cd* x, double tol, int maxiter, double* rn, double* rt) {
    const size_t n = (size_t)l.V * 4 * N;
    std::vector<cd> bm(b, b + n), bp(n), r(n), p(n), t(n), q(n);
    for (long s = 0; s < l.V; s++) {   // D7: components of b on frozen slices are ignored
        int xx[4];
        coords(l, s, xx);
        if (frozen(l, xx[3]))
            for (int i = 0; i < 4 * N; i++) bm[(size_t)s * 4 * N + i] = 0;
    }
    dw<N>(l, kappa, U, Ablk, bm.data(), bp.data(), 1);
    for (size_t i = 0; i < n; i++) x[i] = 0;
    r = bp;
    p = r;
    double rho = norm2(r);
    const double rho0 = rho;
    int it = 0;
    bool conv = (rho0 == 0.0);
    while (!conv && it < maxiter) {
        dw<N>(l, kappa, U, Ablk, p.data(), t.data(), 0);
        const double alpha = rho / norm2(t);
        for (size_t i = 0; i < n; i++) x[i] += alpha * p[i];
        dw<N>(l, kappa, U, Ablk, t.data(), q.data(), 1);
        for (size_t i = 0; i < n; i++) r[i] -= alpha * q[i];
        const double rho_new = norm2(r);
        it++;
        if (rho_new <= tol * tol * rho0) { conv = true; break; }
        const double beta = rho_new / rho;
        for (size_t i = 0; i < n; i++) p[i] = r[i] + beta * p[i];
        rho = rho_new;
    }
    // true residuals with fresh operator applications
    dw<N>(l, kappa, U, Ablk, x, t.data(), 0);
    for (size_t i = 0; i < n; i++) t[i] = bm[i] - t[i];
    dw<N>(l, kappa, U, Ablk, t.data(), q.data(), 1);
    const double nb = norm2(bm);
    *rt = nb > 0 ? std::sqrt(norm2(t) / nb) : 0.0;
    *rn = rho0 > 0 ? std::sqrt(norm2(q) / rho0) : 0.0;
    return conv ? it : -it;
}

extern "C" {

// the Cayley-Dickson pair (z1, z2) of an SU(2) element, as the matrix [[z1, z2], [-conj(z2), conj(z1)]]
void oracle_su2_from_cayley_dickson(long n, const cd* z, cd* U) {
    for (long i = 0; i < n; i++) {
        U[4 * i + 0] = z[2 * i];
        U[4 * i + 1] = z[2 * i + 1];
        U[4 * i + 2] = -std::conj(z[2 * i + 1]);
        U[4 * i + 3] = std::conj(z[2 * i]);
    }
}

int oracle_sun_dw(int nc, const int* L, int bc, const double* theta, double kappa, const cd* U, const cd* Ablk, const cd* psi, cd* out, int dagger) {
    init_gamma();
    Lat l = make_lat(L, bc, theta);
    if (nc == 2) dw<2>(l, kappa, U, Ablk, psi, out, dagger);
    else if (nc == 3) dw<3>(l, kappa, U, Ablk, psi, out, dagger);
    else return -1;
    return 0;
}

int oracle_sun_hop(int nc, const int* L, int bc, const double* theta, const cd* U, const cd* psi, cd* out) {
    init_gamma();
    Lat l = make_lat(L, bc, theta);
    for (long n = 0; n < l.V; n++) {
        int x[4];
        coords(l, n, x);
        if (nc == 2) hop_site<2>(l, U, psi, x, out + (size_t)n * 8);
        else if (nc == 3) hop_site<3>(l, U, psi, x, out + (size_t)n * 12);
        else return -1;
    }
    return 0;
}

int oracle_sun_fhat_site(int nc, const int* L, const cd* U, const int* x, int mu, int nu, cd* out) {
    init_gamma();
    Lat l = make_lat(L, BC_PERIODIC, nullptr);
    if (nc == 2) { Mat<2> f = fhat<2>(l, U, x, mu, nu); memcpy(out, f.e, sizeof(f.e)); }
    else if (nc == 3) { Mat<3> f = fhat<3>(l, U, x, mu, nu); memcpy(out, f.e, sizeof(f.e)); }
    else return -1;
    return 0;
}

int oracle_sun_clover_blocks(int nc, const int* L, int bc, double kappa, double csw, const cd* U, cd* out) {
    init_gamma();
    Lat l = make_lat(L, bc, nullptr);
    if (nc == 2) clover_blocks<2>(l, kappa, csw, U, out);
    else if (nc == 3) clover_blocks<3>(l, kappa, csw, U, out);
    else return -1;
    return 0;
}

int oracle_sun_cg(int nc, const int* L, int bc, const double* theta, double kappa, const cd* U, const cd* Ablk, const cd* b, cd* x, double tol,
                  int maxiter, double* rn, double* rt) {
    init_gamma();
    Lat l = make_lat(L, bc, theta);
    if (nc == 2) return cg<2>(l, kappa, U, Ablk, b, x, tol, maxiter, rn, rt);
    if (nc == 3) return cg<3>(l, kappa, U, Ablk, b, x, tol, maxiter, rn, rt);
    return 0;
}

}  // extern "C"
