// lgf_oracle.cpp -- CPU ORACLE for Fourier-accelerated Landau gauge fixing (arXiv 1301.3460).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
// cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
// header, table or helper with the CUDA path under paper_1301_3460_b200/, and neither imports the other.
//
// Plain, slow, literal: full 3x3 std::complex<double> matrices, array-of-structs, all nine entries
// of Delta Fourier transformed separately (no packing), a naive separable DFT straight from the
// definition, no 12-real tricks except the explicit storage-mode emulation (step O6).
//
// What it follows (PAPER.md = /root/reference/PAPER.md; NS = BASELINE.json "north_star";
// readings A1..A21 = SURVEY.md section 8(c), restated in DESIGN.md):
//   O1  measure   A(x) = sum_mu [U_mu(x-mu) - U_mu(x)];  D = A - A^dag;  Delta = D - (Tr D/3) 1
//                 theta = (1/(N_c V)) sum_x Tr[Delta Delta^dag]                     [NS step 1]
//                 F = (1/(N_d N_c V)) sum_x sum_mu Re Tr U_mu(x)   [PAPER.md:39, g absorbed in U]
//   O2  stop when theta < theta_tol (strict)                                        [PAPER.md:47]
//   O3  X = IDFT[ (p2max/p2(n)) DFT[Delta] ],  p2 = sum_mu 4 sin^2(pi n_mu/L_mu),
//       p2max = 4 N_d = 16, zero mode -> 0, unnormalised forward e^{-i..}, 1/V on inverse
//                                                      [NS step 2; Fourier acceleration PAPER.md:41]
//   O4  g(x) = rowGramSchmidt(1 + (alpha/2) X(x)), third row = conj(u x v)          [NS step 3]
//   O5  U_mu(x) <- g(x) U_mu(x) g(x+mu)^dag, all (x,mu) simultaneously              [NS step 4; PAPER.md:39]
//   O6  12-real storage: row 2 of every U <- conj(row0 x row1)                      [PAPER.md:45,51]
//
// Pins (tests/test_oracle_pins.py, CPU only): brute-force 4-D DFT on 4^4 and numpy.fft, Parseval,
// Delta traceless anti-Hermitian and sum_x Delta = 0, theta_0 -> 128/9 for Haar links, dF/dalpha closed
// form, linearised rate (1-16 alpha)^2, unitarity/det, plaquette invariance, translation and axis
// permutation covariance, the Abelian special case against an independent scalar numpy code, the
// pure-gauge fixed point F = 1, F_U[g] evaluated literally from PAPER.md:39.  Nothing on this path is
// "parity unpinned".
//
// Build: g++ -O2 -fopenmp -shared -fPIC (see oracle/build.py).  OpenMP only parallelises loops over
// sites/lines; every reduction is a serial compensated sum in site order, so results do not depend on
// the thread count.

#include <complex>
#include <vector>
#include <cmath>
#include <cstring>
#include <cstdint>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;

namespace {

struct Mat { cd m[3][3]; };

inline Mat mat_zero() { Mat r; for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) r.m[i][j] = cd(0, 0); return r; }
inline Mat mat_id() { Mat r = mat_zero(); for (int i = 0; i < 3; i++) r.m[i][i] = cd(1, 0); return r; }
inline Mat mat_mul(const Mat& a, const Mat& b) {
    Mat r = mat_zero();
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) { cd s(0, 0); for (int k = 0; k < 3; k++) s += a.m[i][k] * b.m[k][j]; r.m[i][j] = s; }
    return r;
}
inline Mat mat_dag(const Mat& a) { Mat r; for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) r.m[i][j] = std::conj(a.m[j][i]); return r; }
inline Mat mat_add(const Mat& a, const Mat& b) { Mat r; for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) r.m[i][j] = a.m[i][j] + b.m[i][j]; return r; }
inline Mat mat_sub(const Mat& a, const Mat& b) { Mat r; for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) r.m[i][j] = a.m[i][j] - b.m[i][j]; return r; }
inline cd mat_tr(const Mat& a) { return a.m[0][0] + a.m[1][1] + a.m[2][2]; }

// third row from the first two: row2 = conj(row0 x row1)   [PAPER.md:45 "12 real number representation"]
inline void third_row(Mat& u) {
    u.m[2][0] = std::conj(u.m[0][1] * u.m[1][2] - u.m[0][2] * u.m[1][1]);
    u.m[2][1] = std::conj(u.m[0][2] * u.m[1][0] - u.m[0][0] * u.m[1][2]);
    u.m[2][2] = std::conj(u.m[0][0] * u.m[1][1] - u.m[0][1] * u.m[1][0]);
}

// Neumaier compensated sum, serial, in index order.
inline double csum(const std::vector<double>& v) {
    double s = 0.0, c = 0.0;
    for (size_t i = 0; i < v.size(); i++) {
        double t = s + v[i];
        if (std::fabs(s) >= std::fabs(v[i])) c += (s - t) + v[i]; else c += (v[i] - t) + s;
        s = t;
    }
    return s + c;
}

struct Geometry {
    int L[4]; long V;
    long stride[4];
    void set(const int* d) { V = 1; for (int k = 0; k < 4; k++) { L[k] = d[k]; stride[k] = V; V *= d[k]; } }
    inline void coords(long x, int c[4]) const { for (int k = 0; k < 4; k++) { c[k] = (int)(x % L[k]); x /= L[k]; } }
    inline long fwd(long x, int mu) const { int c = (int)((x / stride[mu]) % L[mu]); return (c == L[mu] - 1) ? x - (long)(L[mu] - 1) * stride[mu] : x + stride[mu]; }
    inline long bwd(long x, int mu) const { int c = (int)((x / stride[mu]) % L[mu]); return (c == 0) ? x + (long)(L[mu] - 1) * stride[mu] : x - stride[mu]; }
};

// exp(sign * 2 pi i k / L), k = 0..L-1, evaluated in long double at the exact argument
std::vector<cd> twiddles(int L, int sign) {
    std::vector<cd> w(L);
    const long double twopi = 6.283185307179586476925286766559005768L;
    for (int k = 0; k < L; k++) {
        long double a = twopi * (long double)k / (long double)L;
        w[k] = cd((double)cosl(a), (double)(sign * sinl(a)));
    }
    // exact values on the axes
    for (int k = 0; k < L; k++) {
        if ((4 * k) % L == 0) { int q = (4 * k) / L; static const double cr[4] = {1, 0, -1, 0}, ci[4] = {0, 1, 0, -1}; w[k] = cd(cr[q], sign * ci[q]); }
    }
    return w;
}

// One line, the definition:  out[n] = sum_x in[x] exp(sign 2 pi i n x / L)
void dft_line_naive(const cd* in, cd* out, int L, const std::vector<cd>& w) {
    for (int n = 0; n < L; n++) {
        cd s(0, 0);
        for (int x = 0; x < L; x++) s += in[x] * w[(int)(((long)n * x) % L)];
        out[n] = s;
    }
}

// Textbook iterative radix-2 Cooley-Tukey (bit reversal + butterflies); L must be a power of two.
// Used only when fft_mode = 1 (timed CPU baseline and long trajectories); checked against the
// naive DFT in tests.
void fft_line_radix2(const cd* in, cd* out, int L, const std::vector<cd>& w) {
    int lg = 0; while ((1 << lg) < L) lg++;
    for (int i = 0; i < L; i++) { int r = 0; for (int b = 0; b < lg; b++) if (i & (1 << b)) r |= 1 << (lg - 1 - b); out[r] = in[i]; }
    for (int len = 2; len <= L; len <<= 1) {
        int half = len >> 1, step = L / len;
        for (int base = 0; base < L; base += len)
            for (int j = 0; j < half; j++) {
                cd t = out[base + j + half] * w[j * step];
                cd u = out[base + j];
                out[base + j] = u + t;
                out[base + j + half] = u - t;
            }
    }
}

// Separable 4-D DFT of one complex field f[x] (x0 fastest), in place, no normalisation.
void dft4(const Geometry& G, std::vector<cd>& f, int sign, int fft_mode) {
    for (int ax = 0; ax < 4; ax++) {
        const int L = G.L[ax];
        const long st = G.stride[ax];
        const std::vector<cd> w = twiddles(L, sign);
        const long nlines = G.V / L;
        const bool pow2 = (L & (L - 1)) == 0;
#pragma omp parallel
        {
            std::vector<cd> a(L), b(L);
#pragma omp for schedule(static)
            for (long l = 0; l < nlines; l++) {
                long lo = l % st, hi = l / st;
                long base = lo + hi * st * L;
                for (int x = 0; x < L; x++) a[x] = f[base + x * st];
                if (fft_mode == 1 && pow2) fft_line_radix2(a.data(), b.data(), L, w);
                else dft_line_naive(a.data(), b.data(), L, w);
                for (int x = 0; x < L; x++) f[base + x * st] = b[x];
            }
        }
    }
}

// w(n) = p2max / p2(n), p2max = 4 N_d = 16, w(0) = 0      [NS step 2]
// nd = 4: Landau gauge (the paper).  nd = 3: Coulomb gauge (the variant of PAPER.md:41
// refs [1],[2] with the sum over mu restricted to the spatial directions): p2 runs over axes 0..2, p2max = 4*3 = 12,
// and the weight vanishes on the zero spatial momentum of every time slice (n0 = n1 = n2 = 0, any n3).  The weight
// then does not depend on n3, so the 4-D transform pair acts as a 3-D transform pair on every time slice.
std::vector<double> fa_weights(const Geometry& G, int accel, int nd = 4) {
    std::vector<double> w(G.V);
    const double pi = 3.14159265358979323846264338327950288;
    for (long n = 0; n < G.V; n++) {
        if (!accel) { w[n] = 1.0; continue; }
        int c[4]; G.coords(n, c);
        double p2 = 0;
        bool zero = true;
        for (int k = 0; k < nd; k++) { double s = std::sin(pi * (double)c[k] / (double)G.L[k]); p2 += 4.0 * s * s; zero = zero && c[k] == 0; }
        w[n] = zero ? 0.0 : (4.0 * nd) / p2;
    }
    return w;
}

}  // namespace

struct orc_ctx {
    Geometry G;
    int storage;    // 12 or 18
    int fft_mode;   // 0 naive DFT (definition), 1 radix-2 FFT
    int accel;      // 1 Fourier accelerated (paper), 0 plain steepest descent (pin P8 only)
    int exp_sign;   // -1: forward e^{-i..} (default); +1: swapped convention (pin P7 only)
    int nd;         // directions in the gauge condition: 4 Landau (the paper), 3 Coulomb (mu = 0..2)
    std::vector<Mat> U;  // U[x*4+mu]
    bool loaded;
};

namespace {

// O1, per site
inline Mat delta_site(const orc_ctx* c, long x) {
    Mat A = mat_zero();
    for (int mu = 0; mu < c->nd; mu++) {
        long xb = c->G.bwd(x, mu);
        A = mat_add(A, mat_sub(c->U[xb * 4 + mu], c->U[x * 4 + mu]));
    }
    Mat D = mat_sub(A, mat_dag(A));
    cd t = mat_tr(D) / 3.0;
    for (int i = 0; i < 3; i++) D.m[i][i] -= t;
    return D;
}

void delta_field(const orc_ctx* c, std::vector<Mat>& D) {
    D.resize(c->G.V);
#pragma omp parallel for schedule(static)
    for (long x = 0; x < c->G.V; x++) D[x] = delta_site(c, x);
}

void measure(const orc_ctx* c, const std::vector<Mat>& D, double* F, double* theta) {
    const long V = c->G.V;
    std::vector<double> th(V), fs(V);
#pragma omp parallel for schedule(static)
    for (long x = 0; x < V; x++) {
        double s = 0;
        for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) s += std::norm(D[x].m[i][j]);   // Tr[Delta Delta^dag]
        th[x] = s;
        double f = 0;
        for (int mu = 0; mu < c->nd; mu++) f += mat_tr(c->U[x * 4 + mu]).real();
        fs[x] = f;
    }
    *theta = csum(th) / (3.0 * (double)V);
    *F = csum(fs) / (3.0 * (double)c->nd * (double)V);
}

// O3
void fa_field(const orc_ctx* c, const std::vector<Mat>& D, std::vector<Mat>& X) {
    const Geometry& G = c->G;
    const long V = G.V;
    X.resize(V);
    std::vector<double> w = fa_weights(G, c->accel, c->nd);
    std::vector<cd> f(V);
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) {
        for (long x = 0; x < V; x++) f[x] = D[x].m[i][j];
        dft4(G, f, c->exp_sign, c->fft_mode);
        for (long n = 0; n < V; n++) f[n] *= w[n];
        dft4(G, f, -c->exp_sign, c->fft_mode);
        const double inv = 1.0 / (double)V;
        for (long x = 0; x < V; x++) X[x].m[i][j] = f[x] * inv;
    }
}

// O4: row Gram-Schmidt of M = 1 + (alpha/2) X; <a,b> = sum_j conj(a_j) b_j
inline Mat g_site(const Mat& Xx, double alpha) {
    Mat M = mat_id();
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) M.m[i][j] += (alpha / 2.0) * Xx.m[i][j];
    Mat g;
    double n0 = 0; for (int j = 0; j < 3; j++) n0 += std::norm(M.m[0][j]);
    n0 = std::sqrt(n0);
    for (int j = 0; j < 3; j++) g.m[0][j] = M.m[0][j] / n0;
    cd ip(0, 0); for (int j = 0; j < 3; j++) ip += std::conj(g.m[0][j]) * M.m[1][j];
    cd v[3]; double n1 = 0;
    for (int j = 0; j < 3; j++) { v[j] = M.m[1][j] - ip * g.m[0][j]; n1 += std::norm(v[j]); }
    n1 = std::sqrt(n1);
    for (int j = 0; j < 3; j++) g.m[1][j] = v[j] / n1;
    third_row(g);
    return g;
}

void g_field(const std::vector<Mat>& X, double alpha, std::vector<Mat>& g) {
    g.resize(X.size());
#pragma omp parallel for schedule(static)
    for (long x = 0; x < (long)X.size(); x++) g[x] = g_site(X[x], alpha);
}

// O5 + O6
void update_links(orc_ctx* c, const std::vector<Mat>& g) {
    const long V = c->G.V;
#pragma omp parallel for schedule(static)
    for (long x = 0; x < V; x++)
        for (int mu = 0; mu < 4; mu++) {
            long xf = c->G.fwd(x, mu);
            Mat r = mat_mul(mat_mul(g[x], c->U[x * 4 + mu]), mat_dag(g[xf]));
            if (c->storage == 12) third_row(r);
            c->U[x * 4 + mu] = r;
        }
}

void one_update(orc_ctx* c, const std::vector<Mat>& D, double alpha) {
    std::vector<Mat> X, g;
    fa_field(c, D, X);
    g_field(X, alpha, g);
    update_links(c, g);
}

void mats_out(const std::vector<Mat>& a, double* out) { std::memcpy(out, a.data(), a.size() * sizeof(Mat)); }

}  // namespace

extern "C" {

orc_ctx* orc_create(const int dims[4], int storage, int fft_mode) {
    if (storage != 12 && storage != 18) return nullptr;
    for (int k = 0; k < 4; k++) if (dims[k] < 1) return nullptr;
    orc_ctx* c = new orc_ctx;
    c->G.set(dims); c->storage = storage; c->fft_mode = fft_mode; c->accel = 1; c->exp_sign = -1; c->nd = 4; c->loaded = false;
    return c;
}
void orc_destroy(orc_ctx* c) { delete c; }
void orc_set_variant(orc_ctx* c, int accel, int exp_sign) { c->accel = accel; c->exp_sign = exp_sign; }
void orc_set_gauge(orc_ctx* c, int nd) { c->nd = (nd == 3) ? 3 : 4; }

// links: [V][4][3][3][2] doubles, x0 fastest.  Stored as given (no reprojection, reading A9);
// in 12-real mode row 2 is dropped and rebuilt from rows 0,1.
void orc_load(orc_ctx* c, const double* links) {
    const long n = c->G.V * 4;
    c->U.resize(n);
    std::memcpy(c->U.data(), links, n * sizeof(Mat));
    if (c->storage == 12) for (long i = 0; i < n; i++) third_row(c->U[i]);
    c->loaded = true;
}
void orc_get(const orc_ctx* c, double* links) { std::memcpy(links, c->U.data(), c->U.size() * sizeof(Mat)); }

void orc_measure(const orc_ctx* c, double* F, double* theta) {
    std::vector<Mat> D; delta_field(c, D); measure(c, D, F, theta);
}
void orc_delta(const orc_ctx* c, double* delta) { std::vector<Mat> D; delta_field(c, D); mats_out(D, delta); }
// X(x) for the current links (O1 then O3)
void orc_fa_field(const orc_ctx* c, double* X) {
    std::vector<Mat> D, Xf; delta_field(c, D); fa_field(c, D, Xf); mats_out(Xf, X);
}
// g(x) for the current links and alpha (O1, O3, O4)
void orc_g_field(const orc_ctx* c, double alpha, double* g) {
    std::vector<Mat> D, Xf, gf; delta_field(c, D); fa_field(c, D, Xf); g_field(Xf, alpha, gf); mats_out(gf, g);
}
// F_U[g] evaluated literally from PAPER.md:39 for given g (links unchanged)
double orc_F_of_g(const orc_ctx* c, const double* g_in) {
    const long V = c->G.V;
    const Mat* g = reinterpret_cast<const Mat*>(g_in);
    std::vector<double> fs(V);
    for (long x = 0; x < V; x++) {
        double f = 0;
        for (int mu = 0; mu < c->nd; mu++) f += mat_tr(mat_mul(mat_mul(g[x], c->U[x * 4 + mu]), mat_dag(g[c->G.fwd(x, mu)]))).real();
        fs[x] = f;
    }
    return csum(fs) / (3.0 * (double)c->nd * (double)V);
}

// iterate(n): (O1, O3-O6) n times, then O1 once more; returns F, theta of the links after the n-th update (A5)
void orc_iterate(orc_ctx* c, int n, double alpha, double* F, double* theta) {
    std::vector<Mat> D;
    for (int k = 0; k < n; k++) { delta_field(c, D); one_update(c, D, alpha); }
    delta_field(c, D); measure(c, D, F, theta);
}

// fix: loop O1, O2, O3-O6.  Returns 0 if converged, 100 if max_iter reached.  hist (optional) receives
// (F_k, theta_k) of every O1, k = 0..n_iter, so hist must hold 2*(max_iter+1) doubles.
int orc_fix(orc_ctx* c, double alpha, double theta_tol, int max_iter, int* n_iter, double* F, double* theta, double* hist) {
    std::vector<Mat> D;
    int k = 0;
    for (;;) {
        delta_field(c, D); measure(c, D, F, theta);
        if (hist) { hist[2 * k] = *F; hist[2 * k + 1] = *theta; }
        if (*theta < theta_tol) { *n_iter = k; return 0; }
        if (k == max_iter) { *n_iter = k; return 100; }
        one_update(c, D, alpha);
        k++;
    }
}

// average plaquette (1/(6V)) sum_x sum_{mu<nu} (1/3) Re Tr[U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag]
double orc_plaquette(const orc_ctx* c) {
    const long V = c->G.V;
    std::vector<double> ps(V);
#pragma omp parallel for schedule(static)
    for (long x = 0; x < V; x++) {
        double p = 0;
        for (int mu = 0; mu < 4; mu++) for (int nu = mu + 1; nu < 4; nu++) {
            Mat P = mat_mul(mat_mul(c->U[x * 4 + mu], c->U[c->G.fwd(x, mu) * 4 + nu]),
                            mat_mul(mat_dag(c->U[c->G.fwd(x, nu) * 4 + mu]), mat_dag(c->U[x * 4 + nu])));
            p += mat_tr(P).real() / 3.0;
        }
        ps[x] = p;
    }
    return csum(ps) / (6.0 * (double)V);
}

// max over links of ||U U^dag - 1||_max and |det U - 1|
void orc_unitarity(const orc_ctx* c, double* max_uudag, double* max_det) {
    double a = 0, b = 0;
    for (size_t i = 0; i < c->U.size(); i++) {
        const Mat& u = c->U[i];
        Mat p = mat_mul(u, mat_dag(u));
        for (int r = 0; r < 3; r++) for (int s = 0; s < 3; s++) a = std::fmax(a, std::abs(p.m[r][s] - cd(r == s ? 1.0 : 0.0, 0)));
        cd det = u.m[0][0] * (u.m[1][1] * u.m[2][2] - u.m[1][2] * u.m[2][1]) - u.m[0][1] * (u.m[1][0] * u.m[2][2] - u.m[1][2] * u.m[2][0]) +
                 u.m[0][2] * (u.m[1][0] * u.m[2][1] - u.m[1][1] * u.m[2][0]);
        b = std::fmax(b, std::abs(det - cd(1, 0)));
    }
    *max_uudag = a; *max_det = b;
}

// Stand-alone separable 4-D DFT of a complex field [V][2] (x0 fastest), out = sum_x in e^{sign 2 pi i n.x/L}.
void orc_dft4(const int dims[4], const double* in, double* out, int sign, int fft_mode) {
    Geometry G; G.set(dims);
    std::vector<cd> f(G.V);
    std::memcpy(f.data(), in, G.V * sizeof(cd));
    dft4(G, f, sign, fft_mode);
    std::memcpy(out, f.data(), G.V * sizeof(cd));
}
// w(n) table
void orc_fa_weights(const int dims[4], double* w) {
    Geometry G; G.set(dims);
    std::vector<double> t = fa_weights(G, 1);
    std::memcpy(w, t.data(), G.V * sizeof(double));
}
// g = rowGramSchmidt(1 + (alpha/2) X) for a given X field [V][3][3][2]
void orc_project(long n, const double* X_in, double alpha, double* g_out) {
    const Mat* X = reinterpret_cast<const Mat*>(X_in);
    Mat* g = reinterpret_cast<Mat*>(g_out);
    for (long x = 0; x < n; x++) g[x] = g_site(X[x], alpha);
}

int orc_num_threads(void) {
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        n = omp_get_num_threads();
    }
#endif
    return n;
}

}  // extern "C"
