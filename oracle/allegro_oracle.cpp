/*
 * allegro_oracle.cpp -- float64, single-threaded CPU oracle of the Allegro tensor-product
 * hot path (env-embedding, CG contraction, first derivative, forces).
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT (see allegro_oracle.h).  Shares no code with the CUDA
 * path; only tests/, __graft_entry__.smoke() and bench.py's CPU-baseline legs load it.
 *
 * The method reaches exactly (up to rounding order) a result with a plain definition
 * (a sparse evaluation of a dense contraction), so each function below is that
 * definition written out: dense loops, CSR order, no blocking, no fusion.
 * Parity pins (tests/test_oracle_*.py): sympy clebsch_gordan, scipy sph_harm_y, closed
 * forms for l <= 3, CG orthonormality, Gaunt relation, Wigner-D equivariance (proper and
 * improper), finite differences of the energy, adjoint identities, sum F = 0.  No function
 * here is "parity unpinned".
 */
#include "allegro_oracle.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdlib>
#include <cstring>
#include <vector>

namespace {

typedef std::complex<double> cplx;
const double kPi = 3.14159265358979323846264338327950288;

double fact(int n) {
    static double tab[64];
    static bool init = false;
    if (!init) {
        tab[0] = 1.0;
        for (int i = 1; i < 64; ++i) tab[i] = tab[i - 1] * (double)i;
        init = true;
    }
    return (n < 0 || n >= 64) ? NAN : tab[n];
}

/* Racah's closed form (BASELINE.json:north_star "CG coefficients from the Racah closed form").
 * <j1 m1 j2 m2 | J M> = delta(M, m1+m2)
 *   sqrt[(2J+1) (J+j1-j2)! (J-j1+j2)! (j1+j2-J)! / (j1+j2+J+1)!]
 *   sqrt[(J+M)! (J-M)! (j1-m1)! (j1+m1)! (j2-m2)! (j2+m2)!]
 *   sum_k (-1)^k / [k! (j1+j2-J-k)! (j1-m1-k)! (j2+m2-k)! (J-j2+m1+k)! (J-j1-m2+k)!]     */
double cg_racah(int j1, int m1, int j2, int m2, int J, int M) {
    if (m1 + m2 != M) return 0.0;
    if (J < std::abs(j1 - j2) || J > j1 + j2) return 0.0;
    if (std::abs(m1) > j1 || std::abs(m2) > j2 || std::abs(M) > J) return 0.0;
    double pre = std::sqrt((2.0 * J + 1.0) * fact(J + j1 - j2) * fact(J - j1 + j2) * fact(j1 + j2 - J) /
                           fact(j1 + j2 + J + 1));
    pre *= std::sqrt(fact(J + M) * fact(J - M) * fact(j1 - m1) * fact(j1 + m1) * fact(j2 - m2) *
                     fact(j2 + m2));
    int kmin = std::max(0, std::max(j2 - J - m1, j1 - J + m2));
    int kmax = std::min(j1 + j2 - J, std::min(j1 - m1, j2 + m2));
    double s = 0.0;
    for (int k = kmin; k <= kmax; ++k) {
        double d = fact(k) * fact(j1 + j2 - J - k) * fact(j1 - m1 - k) * fact(j2 + m2 - k) *
                   fact(J - j2 + m1 + k) * fact(J - j1 - m2 + k);
        s += ((k & 1) ? -1.0 : 1.0) / d;
    }
    return pre * s;
}

/* complex -> real change of basis, reading A1/A2 (real = U complex; rows m, columns mu):
 *   m = 0 : U[0,0] = 1
 *   m > 0 : U[m,-m] = 1/sqrt2,  U[m,+m] = (-1)^m / sqrt2
 *   m < 0 : a = |m|, U[m,-a] = i/sqrt2, U[m,+a] = -i (-1)^a / sqrt2                       */
cplx Umat(int m, int mu) {
    const double r = 1.0 / std::sqrt(2.0);
    if (m == 0) return (mu == 0) ? cplx(1.0, 0.0) : cplx(0.0, 0.0);
    int a = std::abs(m);
    double sgn = (a & 1) ? -1.0 : 1.0;
    if (m > 0) {
        if (mu == -a) return cplx(r, 0.0);
        if (mu == a) return cplx(sgn * r, 0.0);
        return cplx(0.0, 0.0);
    }
    if (mu == -a) return cplx(0.0, r);
    if (mu == a) return cplx(0.0, -sgn * r);
    return cplx(0.0, 0.0);
}

/* T[m1][m2][M] = sum conj(U1[m1,mu1]) conj(U2[m2,mu2]) U3[M,mu3] <l1 mu1 l2 mu2 | l3 mu3>
 * C := Re T + Im T   (T is purely real for even l1+l2+l3, purely imaginary for odd).      */
void cg_real(int l1, int l2, int l3, std::vector<double>& C, double* max_re, double* max_im) {
    int d1 = 2 * l1 + 1, d2 = 2 * l2 + 1, d3 = 2 * l3 + 1;
    C.assign((size_t)d1 * d2 * d3, 0.0);
    double mre = 0.0, mim = 0.0;
    for (int m1 = -l1; m1 <= l1; ++m1)
        for (int m2 = -l2; m2 <= l2; ++m2)
            for (int M = -l3; M <= l3; ++M) {
                cplx t(0.0, 0.0);
                for (int mu1 = -l1; mu1 <= l1; ++mu1)
                    for (int mu2 = -l2; mu2 <= l2; ++mu2) {
                        int mu3 = mu1 + mu2;
                        if (std::abs(mu3) > l3) continue;
                        double c = cg_racah(l1, mu1, l2, mu2, l3, mu3);
                        if (c == 0.0) continue;
                        t += std::conj(Umat(m1, mu1)) * std::conj(Umat(m2, mu2)) * Umat(M, mu3) * c;
                    }
                mre = std::max(mre, std::fabs(t.real()));
                mim = std::max(mim, std::fabs(t.imag()));
                C[((size_t)(m1 + l1) * d2 + (m2 + l2)) * d3 + (M + l3)] = t.real() + t.imag();
            }
    if (max_re) *max_re = mre;
    if (max_im) *max_im = mim;
}

inline int off_feat(int l, int p) { return 2 * l * l + (p ? 2 * l + 1 : 0); }

struct Path {
    int l1, p1, l2, l3, p3, off1, off2, off3;
    std::vector<double> C; /* [2l1+1][2l2+1][2l3+1] */
};

/* reading A3: all triangle-allowed (l1,p1) x l2 -> l3 <= lmax, p3 = p1 (-1)^l2 */
std::vector<Path> build_paths(int lmax) {
    std::vector<Path> P;
    for (int l1 = 0; l1 <= lmax; ++l1)
        for (int p1 = 0; p1 <= 1; ++p1)
            for (int l2 = 0; l2 <= lmax; ++l2)
                for (int l3 = std::abs(l1 - l2); l3 <= std::min(l1 + l2, lmax); ++l3) {
                    Path q;
                    q.l1 = l1; q.p1 = p1; q.l2 = l2; q.l3 = l3;
                    q.p3 = p1 ^ (l2 & 1);
                    q.off1 = off_feat(l1, p1);
                    q.off2 = l2 * l2;
                    q.off3 = off_feat(l3, q.p3);
                    cg_real(l1, l2, l3, q.C, nullptr, nullptr);
                    P.push_back(q);
                }
    return P;
}

const std::vector<Path>& paths_for(int lmax) {
    static std::vector<Path> cache[8];
    static bool have[8] = {false, false, false, false, false, false, false, false};
    if (!have[lmax]) { cache[lmax] = build_paths(lmax); have[lmax] = true; }
    return cache[lmax];
}

struct Nz { int path, i, j, k; double c; };

const std::vector<Nz>& nz_for(int lmax) {
    static std::vector<Nz> cache[8];
    static bool have[8] = {false, false, false, false, false, false, false, false};
    if (!have[lmax]) {
        const std::vector<Path>& P = paths_for(lmax);
        std::vector<Nz> L;
        for (size_t p = 0; p < P.size(); ++p) {
            const Path& q = P[p];
            int d1 = 2 * q.l1 + 1, d2 = 2 * q.l2 + 1, d3 = 2 * q.l3 + 1;
            for (int a = 0; a < d1; ++a)
                for (int b = 0; b < d2; ++b)
                    for (int c = 0; c < d3; ++c) {
                        double v = q.C[((size_t)a * d2 + b) * d3 + c];
                        if (std::fabs(v) > 1e-12) {
                            Nz z; z.path = (int)p; z.i = q.off1 + a; z.j = q.off2 + b; z.k = q.off3 + c; z.c = v;
                            L.push_back(z);
                        }
                    }
        }
        cache[lmax] = L; have[lmax] = true; /* loop order already gives (path,i,j,k) order */
    }
    return cache[lmax];
}

/* forward-mode number: value and partials w.r.t. the unit-vector components (x,y,z) */
struct D3 {
    double v, d[3];
    D3() : v(0.0) { d[0] = d[1] = d[2] = 0.0; }
    explicit D3(double c) : v(c) { d[0] = d[1] = d[2] = 0.0; }
};
inline D3 operator+(const D3& a, const D3& b) { D3 r; r.v = a.v + b.v; for (int i = 0; i < 3; ++i) r.d[i] = a.d[i] + b.d[i]; return r; }
inline D3 operator-(const D3& a, const D3& b) { D3 r; r.v = a.v - b.v; for (int i = 0; i < 3; ++i) r.d[i] = a.d[i] - b.d[i]; return r; }
inline D3 operator*(const D3& a, const D3& b) { D3 r; r.v = a.v * b.v; for (int i = 0; i < 3; ++i) r.d[i] = a.d[i] * b.v + a.v * b.d[i]; return r; }
inline D3 operator*(double s, const D3& a) { D3 r; r.v = s * a.v; for (int i = 0; i < 3; ++i) r.d[i] = s * a.d[i]; return r; }

/* Step 1 (reading A1): real spherical harmonics by the explicit recursion.
 *   (x,y,z) = r/|r|;  c_0 = 1, s_0 = 0, c_m = x c_{m-1} - y s_{m-1}, s_m = x s_{m-1} + y c_{m-1}
 *   Q_m^m = (2m-1)!!, Q_{m+1}^m = (2m+1) z Q_m^m,
 *   Q_l^m = ((2l-1) z Q_{l-1}^m - (l+m-1) Q_{l-2}^m) / (l-m)
 *   K_lm = sqrt((2l+1) (l-m)!/(l+m)!)
 *   Y_{l,0} = K_l0 Q_l^0, Y_{l,+m} = sqrt2 K_lm Q_l^m c_m, Y_{l,-m} = sqrt2 K_lm Q_l^m s_m
 * Derivative: forward mode through the same recursion with x,y,z independent (J~), then
 *   dY/dr = J~ (I - rhat rhat^T) / |r|.                                                    */
void sph_harm(int lmax, const double* r, double* Y, double* dYdr) {
    double rn = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
    double u[3] = {r[0] / rn, r[1] / rn, r[2] / rn};
    D3 x(u[0]), y(u[1]), z(u[2]);
    x.d[0] = 1.0; y.d[1] = 1.0; z.d[2] = 1.0;
    int L = lmax;
    std::vector<D3> c(L + 1), s(L + 1);
    c[0] = D3(1.0); s[0] = D3(0.0);
    for (int m = 1; m <= L; ++m) {
        c[m] = x * c[m - 1] - y * s[m - 1];
        s[m] = x * s[m - 1] + y * c[m - 1];
    }
    /* Q[l][m] */
    std::vector<std::vector<D3> > Q(L + 1, std::vector<D3>(L + 1));
    for (int m = 0; m <= L; ++m) {
        double dfact = 1.0;
        for (int t = 2 * m - 1; t > 1; t -= 2) dfact *= (double)t;
        Q[m][m] = D3(dfact);
        if (m + 1 <= L) Q[m + 1][m] = (2.0 * m + 1.0) * (z * Q[m][m]);
        for (int l = m + 2; l <= L; ++l) {
            D3 a = (2.0 * l - 1.0) * (z * Q[l - 1][m]);
            D3 b = (double)(l + m - 1) * Q[l - 2][m];
            Q[l][m] = (1.0 / (double)(l - m)) * (a - b);
        }
    }
    int dE = (L + 1) * (L + 1);
    std::vector<D3> Yd(dE);
    for (int l = 0; l <= L; ++l) {
        for (int m = 0; m <= l; ++m) {
            double K = std::sqrt((2.0 * l + 1.0) * fact(l - m) / fact(l + m));
            if (m == 0) {
                Yd[l * l + l] = K * Q[l][0];
            } else {
                Yd[l * l + l + m] = (std::sqrt(2.0) * K) * (Q[l][m] * c[m]);
                Yd[l * l + l - m] = (std::sqrt(2.0) * K) * (Q[l][m] * s[m]);
            }
        }
    }
    for (int j = 0; j < dE; ++j) {
        if (Y) Y[j] = Yd[j].v;
        if (dYdr) {
            double dot = Yd[j].d[0] * u[0] + Yd[j].d[1] * u[1] + Yd[j].d[2] * u[2];
            for (int a = 0; a < 3; ++a) dYdr[j * 3 + a] = (Yd[j].d[a] - dot * u[a]) / rn;
        }
    }
}

/* Wigner's small-d formula,
 * d^j_{m'm}(b) = sum_s (-1)^{m'-m+s} sqrt((j+m')!(j-m')!(j+m)!(j-m)!)
 *                / ((j+m-s)! s! (m'-m+s)! (j-m'-s)!) cos(b/2)^{2j+m-m'-2s} sin(b/2)^{m'-m+2s} */
double wigner_small_d(int j, int mp, int m, double beta) {
    double cb = std::cos(beta / 2.0), sb = std::sin(beta / 2.0);
    double pre = std::sqrt(fact(j + mp) * fact(j - mp) * fact(j + m) * fact(j - m));
    double sum = 0.0;
    int smin = std::max(0, m - mp), smax = std::min(j + m, j - mp);
    for (int s = smin; s <= smax; ++s) {
        double den = fact(j + m - s) * fact(s) * fact(mp - m + s) * fact(j - mp - s);
        double sg = ((mp - m + s) & 1) ? -1.0 : 1.0;
        sum += sg / den * std::pow(cb, 2 * j + m - mp - 2 * s) * std::pow(sb, mp - m + 2 * s);
    }
    return pre * sum;
}

inline void centre_range_edges(const int32_t* row_ptr, int c_lo, int c_hi, int64_t* e0, int64_t* e1) {
    *e0 = row_ptr[c_lo];
    *e1 = row_ptr[c_hi];
}

}  // namespace

extern "C" {

int orc_dim_v(int lmax) { return 2 * (lmax + 1) * (lmax + 1); }
int orc_dim_e(int lmax) { return (lmax + 1) * (lmax + 1); }

double orc_cg_complex(int j1, int m1, int j2, int m2, int j3, int m3) { return cg_racah(j1, m1, j2, m2, j3, m3); }

void orc_cg_real(int l1, int l2, int l3, double* C, double* max_re, double* max_im) {
    std::vector<double> c;
    cg_real(l1, l2, l3, c, max_re, max_im);
    std::memcpy(C, c.data(), c.size() * sizeof(double));
}

int orc_num_paths(int lmax) { return (int)paths_for(lmax).size(); }

void orc_paths(int lmax, int32_t* l1, int32_t* p1, int32_t* l2, int32_t* l3, int32_t* p3, int32_t* off1,
               int32_t* off2, int32_t* off3) {
    const std::vector<Path>& P = paths_for(lmax);
    for (size_t p = 0; p < P.size(); ++p) {
        l1[p] = P[p].l1; p1[p] = P[p].p1; l2[p] = P[p].l2; l3[p] = P[p].l3; p3[p] = P[p].p3;
        off1[p] = P[p].off1; off2[p] = P[p].off2; off3[p] = P[p].off3;
    }
}

int64_t orc_nnz(int lmax) { return (int64_t)nz_for(lmax).size(); }

void orc_cg_list(int lmax, int32_t* path, int32_t* i, int32_t* j, int32_t* k, double* coef) {
    const std::vector<Nz>& L = nz_for(lmax);
    for (size_t t = 0; t < L.size(); ++t) {
        path[t] = L[t].path; i[t] = L[t].i; j[t] = L[t].j; k[t] = L[t].k; coef[t] = L[t].c;
    }
}

void orc_sph_harm(int lmax, const double* r, double* Y, double* dYdr) { sph_harm(lmax, r, Y, dYdr); }

void orc_rotation_matrix(double al, double be, double ga, double* R) {
    double ca = std::cos(al), sa = std::sin(al), cb = std::cos(be), sb = std::sin(be), cg = std::cos(ga), sg = std::sin(ga);
    double Rza[9] = {ca, -sa, 0, sa, ca, 0, 0, 0, 1};
    double Ryb[9] = {cb, 0, sb, 0, 1, 0, -sb, 0, cb};
    double Rzg[9] = {cg, -sg, 0, sg, cg, 0, 0, 0, 1};
    double T[9];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double s = 0;
            for (int k = 0; k < 3; ++k) s += Rza[i * 3 + k] * Ryb[k * 3 + j];
            T[i * 3 + j] = s;
        }
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double s = 0;
            for (int k = 0; k < 3; ++k) s += T[i * 3 + k] * Rzg[k * 3 + j];
            R[i * 3 + j] = s;
        }
}

/* Complex harmonics obey Y_mu(R r) = sum_mu' conj(D^l_{mu mu'}(R)) Y_mu'(r) with
 * D^l_{mu' mu}(a,b,g) = exp(-i mu' a) d^l_{mu' mu}(b) exp(-i mu g), R = Rz(a) Ry(b) Rz(g).
 * Real basis: D_real = U conj(D) U^dagger.                                                 */
void orc_wigner_D_real(int l, double al, double be, double ga, double* D) {
    int d = 2 * l + 1;
    std::vector<cplx> Dc((size_t)d * d), tmp((size_t)d * d);
    for (int mp = -l; mp <= l; ++mp)
        for (int m = -l; m <= l; ++m) {
            cplx v = std::exp(cplx(0.0, -mp * al)) * wigner_small_d(l, mp, m, be) * std::exp(cplx(0.0, -m * ga));
            Dc[(size_t)(mp + l) * d + (m + l)] = std::conj(v);
        }
    for (int a = -l; a <= l; ++a)
        for (int m = -l; m <= l; ++m) {
            cplx s(0.0, 0.0);
            for (int mu = -l; mu <= l; ++mu) s += Umat(a, mu) * Dc[(size_t)(mu + l) * d + (m + l)];
            tmp[(size_t)(a + l) * d + (m + l)] = s;
        }
    for (int a = -l; a <= l; ++a)
        for (int b = -l; b <= l; ++b) {
            cplx s(0.0, 0.0);
            for (int mu = -l; mu <= l; ++mu) s += tmp[(size_t)(a + l) * d + (mu + l)] * std::conj(Umat(b, mu));
            D[(size_t)(a + l) * d + (b + l)] = s.real();
        }
}

/* Step 0 (readings A5, A8): x = r/rc; B_b = sqrt(2/rc) sin(b pi x)/r, b = 1..nb;
 * u(x) = 1 - 28 x^6 + 48 x^7 - 21 x^8 (p = 6 polynomial cutoff);
 * w[n] = sum_b Wr[n][b] B_b u.                                                             */
void orc_radial(int n, int nb, double rc, const double* Wr, int64_t E, const double* rvec, double* w,
                double* dwdr) {
    std::vector<double> B(nb), dB(nb);
    for (int64_t e = 0; e < E; ++e) {
        const double* r = rvec + 3 * e;
        double rn = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
        double x = rn / rc;
        double x2 = x * x, x5 = x2 * x2 * x, x6 = x5 * x, x7 = x6 * x, x8 = x7 * x;
        double u = 1.0 - 28.0 * x6 + 48.0 * x7 - 21.0 * x8;
        double du = (-168.0 * x5 + 336.0 * x6 - 168.0 * x7) / rc;
        if (x >= 1.0) { u = 0.0; du = 0.0; }
        double pre = std::sqrt(2.0 / rc);
        for (int b = 1; b <= nb; ++b) {
            double k = b * kPi / rc;
            double sn = std::sin(k * rn), cs = std::cos(k * rn);
            double Bv = pre * sn / rn;
            double dBv = pre * (k * cs / rn - sn / (rn * rn));
            B[b - 1] = Bv * u;
            dB[b - 1] = dBv * u + Bv * du;
        }
        for (int c = 0; c < n; ++c) {
            double s = 0.0, ds = 0.0;
            for (int b = 0; b < nb; ++b) { s += Wr[c * nb + b] * B[b]; ds += Wr[c * nb + b] * dB[b]; }
            if (w) w[e * n + c] = s;
            if (dwdr) dwdr[e * n + c] = ds;
        }
    }
}

void orc_radial_backward(int n, int64_t E, const double* rvec, const double* g_w, const double* dwdr,
                         double* g_rvec) {
    for (int64_t e = 0; e < E; ++e) {
        const double* r = rvec + 3 * e;
        double rn = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
        double s = 0.0;
        for (int c = 0; c < n; ++c) s += g_w[e * n + c] * dwdr[e * n + c];
        for (int a = 0; a < 3; ++a) g_rvec[3 * e + a] += s * r[a] / rn;
    }
}

/* reading A16 */
int64_t orc_segments(const int32_t* row_ptr, int N, int T, int32_t* items, int64_t cap) {
    int64_t cnt = 0;
    for (int i = 0; i < N; ++i) {
        int a = row_ptr[i], b = row_ptr[i + 1];
        if (a == b) {
            if (items && cnt < cap) { items[3 * cnt] = i; items[3 * cnt + 1] = a; items[3 * cnt + 2] = a; }
            ++cnt;
            continue;
        }
        for (int e0 = a; e0 < b; e0 += T) {
            int e1 = std::min(e0 + T, b);
            if (items && cnt < cap) { items[3 * cnt] = i; items[3 * cnt + 1] = e0; items[3 * cnt + 2] = e1; }
            ++cnt;
        }
    }
    return cnt;
}

/* Step 3: Eenv[i][n][j] = scale sum_{e in row i, CSR order} w[e][n] Y_j(rhat_e) */
void orc_env_embed(int lmax, int n, int N, const int32_t* row_ptr, const double* rvec, const double* w,
                   double scale, double* Eenv) {
    int dE = orc_dim_e(lmax);
    std::vector<double> Y(dE);
    for (int i = 0; i < N; ++i) {
        double* Ei = Eenv + (size_t)i * n * dE;
        for (int t = 0; t < n * dE; ++t) Ei[t] = 0.0;
        for (int e = row_ptr[i]; e < row_ptr[i + 1]; ++e) {
            sph_harm(lmax, rvec + 3 * (size_t)e, Y.data(), nullptr);
            for (int c = 0; c < n; ++c)
                for (int j = 0; j < dE; ++j) Ei[c * dE + j] += w[(size_t)e * n + c] * Y[j];
        }
        for (int t = 0; t < n * dE; ++t) Ei[t] *= scale;
    }
}

/* Step 3, brute force over the dense real-CG blocks.
 * scalar: out[e][n][off3+M] = sum_p w_p sum_{m1 m2} C^p[m1][m2][M] V[e][n][off1+m1] Eenv[c][n][off2+m2]
 * dense : t[e][n][p][M] = inner sum; out[e][n'][off3+M] = sum_p sum_n W[p][n'][n] t[e][n][p][M] */
void orc_tp_forward_dense(int lmax, int n, int wmode, int N, const int32_t* row_ptr, int c_lo, int c_hi,
                          const double* V, const double* Eenv, const double* path_w, double* out) {
    (void)N;
    const std::vector<Path>& P = paths_for(lmax);
    int dV = orc_dim_v(lmax), dE = orc_dim_e(lmax);
    std::vector<double> t((size_t)n * 16);
    for (int c = c_lo; c < c_hi; ++c)
        for (int e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
            const double* Ve = V + (size_t)e * n * dV;
            const double* Ec = Eenv + (size_t)c * n * dE;
            double* oe = out + (size_t)e * n * dV;
            for (int q = 0; q < n * dV; ++q) oe[q] = 0.0;
            for (size_t p = 0; p < P.size(); ++p) {
                const Path& pa = P[p];
                int d1 = 2 * pa.l1 + 1, d2 = 2 * pa.l2 + 1, d3 = 2 * pa.l3 + 1;
                for (int ch = 0; ch < n; ++ch)
                    for (int M = 0; M < d3; ++M) {
                        double s = 0.0;
                        for (int m1 = 0; m1 < d1; ++m1)
                            for (int m2 = 0; m2 < d2; ++m2)
                                s += pa.C[((size_t)m1 * d2 + m2) * d3 + M] * Ve[ch * dV + pa.off1 + m1] *
                                     Ec[ch * dE + pa.off2 + m2];
                        t[(size_t)ch * 16 + M] = s;
                    }
                if (wmode == 0) {
                    for (int ch = 0; ch < n; ++ch)
                        for (int M = 0; M < d3; ++M) oe[ch * dV + pa.off3 + M] += path_w[p] * t[(size_t)ch * 16 + M];
                } else {
                    const double* W = path_w + p * (size_t)n * n;
                    for (int co = 0; co < n; ++co)
                        for (int M = 0; M < d3; ++M) {
                            double s = 0.0;
                            for (int ci = 0; ci < n; ++ci) s += W[(size_t)co * n + ci] * t[(size_t)ci * 16 + M];
                            oe[co * dV + pa.off3 + M] += s;
                        }
                }
            }
        }
}

/* Same result from the compressed sparse list ("compressed sparse format"); this
 * is the variant the CPU baseline times. */
void orc_tp_forward_sparse(int lmax, int n, int wmode, int N, const int32_t* row_ptr, int c_lo, int c_hi,
                           const double* V, const double* Eenv, const double* path_w, double* out) {
    (void)N;
    const std::vector<Path>& P = paths_for(lmax);
    const std::vector<Nz>& L = nz_for(lmax);
    int dV = orc_dim_v(lmax), dE = orc_dim_e(lmax);
    int nP = (int)P.size();
    std::vector<double> t;
    if (wmode == 1) t.resize((size_t)nP * 7 * n);
    for (int c = c_lo; c < c_hi; ++c)
        for (int e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
            const double* Ve = V + (size_t)e * n * dV;
            const double* Ec = Eenv + (size_t)c * n * dE;
            double* oe = out + (size_t)e * n * dV;
            for (int q = 0; q < n * dV; ++q) oe[q] = 0.0;
            if (wmode == 0) {
                for (int ch = 0; ch < n; ++ch)
                    for (size_t z = 0; z < L.size(); ++z)
                        oe[ch * dV + L[z].k] += path_w[L[z].path] * L[z].c * Ve[ch * dV + L[z].i] * Ec[ch * dE + L[z].j];
            } else {
                std::fill(t.begin(), t.end(), 0.0);
                for (int ch = 0; ch < n; ++ch)
                    for (size_t z = 0; z < L.size(); ++z) {
                        int M = L[z].k - P[L[z].path].off3;
                        t[((size_t)L[z].path * 7 + M) * n + ch] += L[z].c * Ve[ch * dV + L[z].i] * Ec[ch * dE + L[z].j];
                    }
                for (int p = 0; p < nP; ++p) {
                    const double* W = path_w + (size_t)p * n * n;
                    int d3 = 2 * P[p].l3 + 1;
                    for (int M = 0; M < d3; ++M)
                        for (int co = 0; co < n; ++co) {
                            double s = 0.0;
                            for (int ci = 0; ci < n; ++ci) s += W[(size_t)co * n + ci] * t[((size_t)p * 7 + M) * n + ci];
                            oe[co * dV + P[p].off3 + M] += s;
                        }
                }
            }
        }
}

/* Step 4 ("its first derivative"): VJP for cotangent G.
 * scalar: gV[e][n][i]  = sum w_p C[i][j][k] Eenv[c][n][j] G[e][n][k]
 *         gE[c][n][j]  = sum_{e in row c} sum w_p C[i][j][k] V[e][n][i] G[e][n][k]
 *         g_w[p]      += sum_e sum_n sum_{(i,j,k) in p} C V Eenv G
 * dense : gt[e][n][p][M] = sum_n' W[p][n'][n] G[e][n'][off3+M], then as above with unit weights;
 *         g_W[p][n'][n] += sum_e sum_M G[e][n'][off3+M] t[e][n][p][M]                          */
void orc_tp_backward(int lmax, int n, int wmode, int N, const int32_t* row_ptr, int c_lo, int c_hi,
                     const double* G, const double* V, const double* Eenv, const double* path_w, double* gV,
                     double* gEenv, double* g_path_w) {
    (void)N;
    const std::vector<Path>& P = paths_for(lmax);
    const std::vector<Nz>& L = nz_for(lmax);
    int dV = orc_dim_v(lmax), dE = orc_dim_e(lmax);
    int nP = (int)P.size();
    std::vector<double> gt, t;
    if (wmode == 1) { gt.resize((size_t)nP * 7 * n); t.resize((size_t)nP * 7 * n); }
    for (int c = c_lo; c < c_hi; ++c) {
        double* gEc = gEenv + (size_t)c * n * dE;
        for (int q = 0; q < n * dE; ++q) gEc[q] = 0.0;
        const double* Ec = Eenv + (size_t)c * n * dE;
        for (int e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
            const double* Ve = V + (size_t)e * n * dV;
            const double* Ge = G + (size_t)e * n * dV;
            double* gVe = gV ? gV + (size_t)e * n * dV : nullptr;
            if (gVe) for (int q = 0; q < n * dV; ++q) gVe[q] = 0.0;
            if (wmode == 0) {
                for (int ch = 0; ch < n; ++ch)
                    for (size_t z = 0; z < L.size(); ++z) {
                        double cw = path_w[L[z].path] * L[z].c;
                        double v = Ve[ch * dV + L[z].i], en = Ec[ch * dE + L[z].j], g = Ge[ch * dV + L[z].k];
                        if (gVe) gVe[ch * dV + L[z].i] += cw * en * g;
                        gEc[ch * dE + L[z].j] += cw * v * g;
                        if (g_path_w) g_path_w[L[z].path] += L[z].c * v * en * g;
                    }
            } else {
                for (int p = 0; p < nP; ++p) {
                    const double* W = path_w + (size_t)p * n * n;
                    int d3 = 2 * P[p].l3 + 1;
                    for (int M = 0; M < d3; ++M)
                        for (int ci = 0; ci < n; ++ci) {
                            double s = 0.0;
                            for (int co = 0; co < n; ++co) s += W[(size_t)co * n + ci] * Ge[co * dV + P[p].off3 + M];
                            gt[((size_t)p * 7 + M) * n + ci] = s;
                        }
                }
                if (g_path_w) std::fill(t.begin(), t.end(), 0.0);
                for (int ch = 0; ch < n; ++ch)
                    for (size_t z = 0; z < L.size(); ++z) {
                        int M = L[z].k - P[L[z].path].off3;
                        double g = gt[((size_t)L[z].path * 7 + M) * n + ch];
                        double v = Ve[ch * dV + L[z].i], en = Ec[ch * dE + L[z].j];
                        if (gVe) gVe[ch * dV + L[z].i] += L[z].c * en * g;
                        gEc[ch * dE + L[z].j] += L[z].c * v * g;
                        if (g_path_w) t[((size_t)L[z].path * 7 + M) * n + ch] += L[z].c * v * en;
                    }
                if (g_path_w)
                    for (int p = 0; p < nP; ++p) {
                        double* gW = g_path_w + (size_t)p * n * n;
                        int d3 = 2 * P[p].l3 + 1;
                        for (int co = 0; co < n; ++co)
                            for (int ci = 0; ci < n; ++ci) {
                                double s = 0.0;
                                for (int M = 0; M < d3; ++M)
                                    s += Ge[co * dV + P[p].off3 + M] * t[((size_t)p * 7 + M) * n + ci];
                                gW[(size_t)co * n + ci] += s;
                            }
                    }
            }
        }
    }
}

/* g_w[e][n] = scale sum_j gE[c][n][j] Y_e[j];  gY_e[j] = scale sum_n gE[c][n][j] w[e][n];
 * g_r[e] = (dY/dr)^T gY_e                                                                   */
void orc_env_embed_backward(int lmax, int n, int N, const int32_t* row_ptr, int c_lo, int c_hi,
                            const double* gEenv, const double* rvec, const double* w, double scale,
                            double* g_rvec, double* g_w) {
    (void)N;
    int dE = orc_dim_e(lmax);
    std::vector<double> Y(dE), dY((size_t)dE * 3), gY(dE);
    for (int c = c_lo; c < c_hi; ++c) {
        const double* gEc = gEenv + (size_t)c * n * dE;
        for (int e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
            sph_harm(lmax, rvec + 3 * (size_t)e, Y.data(), dY.data());
            for (int j = 0; j < dE; ++j) gY[j] = 0.0;
            for (int ch = 0; ch < n; ++ch) {
                double s = 0.0;
                for (int j = 0; j < dE; ++j) {
                    s += gEc[ch * dE + j] * Y[j];
                    gY[j] += gEc[ch * dE + j] * w[(size_t)e * n + ch];
                }
                if (g_w) g_w[(size_t)e * n + ch] = scale * s;
            }
            for (int a = 0; a < 3; ++a) {
                double s = 0.0;
                for (int j = 0; j < dE; ++j) s += dY[j * 3 + a] * gY[j];
                g_rvec[3 * (size_t)e + a] = scale * s;
            }
        }
    }
}

/* Second derivative of the tensor product ("the additional kernels required for training are left for future work";
   SURVEY 8.f2: VJP-of-VJP for a force-matching loss).  The first derivative (scalar weights, Wc = sum_p w_p C^p) is
       gV[e,n,i] = sum_{jk} Wc[ijk] E[c,n,j] G[e,n,k],      gE[c,n,j] = sum_{e in row c} sum_{ik} Wc[ijk] V[e,n,i] G[e,n,k].
   For cotangents aV (of gV) and bE (of gE) the scalar S = <aV, gV> + <bE, gE> has the gradients written out below, term by term
   over the non-zero list (reading A26: S is trilinear in (aV | bE, V | E, G) and linear in w):
       dG[e,n,k] = sum_{ij} Wc[ijk] (aV[e,n,i] E[c,n,j] + V[e,n,i] bE[c,n,j])
       dV[e,n,i] = sum_{jk} Wc[ijk] bE[c,n,j] G[e,n,k]
       dE[c,n,j] = sum_{e in row c} sum_{ik} Wc[ijk] aV[e,n,i] G[e,n,k]
       dw[p]     = sum_{e,n} sum_{(ijk) in p} C^p[ijk] G[e,n,k] (aV[e,n,i] E[c,n,j] + V[e,n,i] bE[c,n,j])                       */
void orc_tp_double_backward(int lmax, int n, int N, const int32_t* row_ptr, const double* G, const double* V, const double* Eenv,
                            const double* path_w, const double* aV, const double* bE, double* dG, double* dV_, double* dE_, double* dw) {
    const std::vector<Path>& P = paths_for(lmax);
    const std::vector<Nz>& L = nz_for(lmax);
    int dV = orc_dim_v(lmax), dE = orc_dim_e(lmax);
    for (size_t p = 0; p < P.size(); ++p) dw[p] = 0.0;
    for (int c = 0; c < N; ++c) {
        const double* Ec = Eenv + (size_t)c * n * dE;
        const double* bc = bE + (size_t)c * n * dE;
        double* dEc = dE_ + (size_t)c * n * dE;
        for (int q = 0; q < n * dE; ++q) dEc[q] = 0.0;
        for (int e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
            const double* Ve = V + (size_t)e * n * dV;
            const double* Ge = G + (size_t)e * n * dV;
            const double* ae = aV + (size_t)e * n * dV;
            double* dGe = dG + (size_t)e * n * dV;
            double* dVe = dV_ + (size_t)e * n * dV;
            for (int q = 0; q < n * dV; ++q) { dGe[q] = 0.0; dVe[q] = 0.0; }
            for (int ch = 0; ch < n; ++ch)
                for (size_t z = 0; z < L.size(); ++z) {
                    const double cw = path_w[L[z].path] * L[z].c;
                    const int i = ch * dV + L[z].i, j = ch * dE + L[z].j, k = ch * dV + L[z].k;
                    const double mix = ae[i] * Ec[j] + Ve[i] * bc[j];
                    dGe[k] += cw * mix;
                    dVe[i] += cw * bc[j] * Ge[k];
                    dEc[j] += cw * ae[i] * Ge[k];
                    dw[L[z].path] += L[z].c * Ge[k] * mix;
                }
        }
    }
}

/* F[a] = sum_{e in row a} (g_r[e] - g_r[rev[e]])  (r_e = x_nbr - x_centre + shift, F = -dE/dx) */
void orc_force_gather(int N, const int32_t* row_ptr, const int32_t* rev, const double* g_rvec, double* F) {
    for (int a = 0; a < N; ++a) {
        double f[3] = {0.0, 0.0, 0.0};
        for (int e = row_ptr[a]; e < row_ptr[a + 1]; ++e)
            for (int d = 0; d < 3; ++d) f[d] += g_rvec[3 * (size_t)e + d] - g_rvec[3 * (size_t)rev[e] + d];
        for (int d = 0; d < 3; ++d) F[3 * (size_t)a + d] = f[d];
    }
}

/* Virial of an energy that depends on the positions only through the edge vectors (reading A25): under the homogeneous
   deformation r_e -> (I + eps) r_e,  dE/d eps[a][b] = sum_e g_rvec[e][a] * r_e[b] =: W[a][b] (sum over DIRECTED edges: each is its
   own term of E_tot).  Pressure = -trace(W) / (3 volume).  (the MD integration consumes forces; stress is the
   companion quantity for constant-pressure MD.) */
void orc_virial(int64_t E, const double* rvec, const double* g_rvec, double* W) {
    for (int i = 0; i < 9; ++i) W[i] = 0.0;
    for (int64_t e = 0; e < E; ++e)
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) W[3 * a + b] += g_rvec[3 * (size_t)e + a] * rvec[3 * (size_t)e + b];
}

void orc_edge_energy(int lmax, int n, int64_t E, const double* out, const double* q, double kappa,
                     double* e_edge, double* G) {
    int dV = orc_dim_v(lmax);
    for (int64_t e = 0; e < E; ++e) {
        double s = 0.0;
        for (int ch = 0; ch < n; ++ch) {
            const double* o = out + ((size_t)e * n + ch) * dV;
            double sq = 0.0;
            for (int k = 0; k < dV; ++k) sq += o[k] * o[k];
            s += q[ch] * o[0] + 0.5 * kappa * sq;
            if (G) {
                double* g = G + ((size_t)e * n + ch) * dV;
                for (int k = 0; k < dV; ++k) g[k] = kappa * o[k];
                g[0] += q[ch];
            }
        }
        if (e_edge) e_edge[e] = s;
    }
}

void orc_segment_sum(const int32_t* ptr, int nseg, const double* vals, double* out) {
    for (int s = 0; s < nseg; ++s) {
        double a = 0.0;
        for (int i = ptr[s]; i < ptr[s + 1]; ++i) a += vals[i];
        out[s] = a;
    }
}

}  // extern "C"
