// plan.cpp -- CG-table / path-plan / segment-plan builder of the product library (host only).
//
// PAPER.md:71 (Sec. II.D): "compressed sparse format to represent the combined tensor of Wigner 3-j
// contraction coefficients".  The table built here is that compressed sparse tensor; gen_tp.cpp
// unrolls it into straight-line CUDA at build time and the kernels fold the run-time path weights in.
//
// Independent of oracle/ by construction: complex Clebsch-Gordan coefficients come from the
// ladder-operator recursion (highest-weight state from J+|JJ> = 0, then repeated J-), not from the
// Racah closed form the oracle uses.  The real-basis convention (reading A1/A2) is a definition and is
// restated, not shared.
#include "plan.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdlib>

namespace allegro {

static inline double a_plus(int j, int m) { return std::sqrt((double)(j * (j + 1) - m * (m + 1))); }
static inline double a_minus(int j, int m) { return std::sqrt((double)(j * (j + 1) - m * (m - 1))); }

void cg_complex_ladder(int j1, int j2, int J, std::vector<double>& table) {
    const int d1 = 2 * j1 + 1, d2 = 2 * j2 + 1, d3 = 2 * J + 1;
    table.assign((size_t)d1 * d2 * d3, 0.0);
    if (J < std::abs(j1 - j2) || J > j1 + j2) return;
    auto at = [&](int m1, int m2, int M) -> double& { return table[((size_t)(m1 + j1) * d2 + (m2 + j2)) * d3 + (M + J)]; };
    // highest weight: |J J> = sum_{m1} c(m1) |m1, J-m1>,  J+ |J J> = 0
    //   c(mu1-1) a+(j1,mu1-1) + c(mu1) a+(j2, J-mu1) = 0
    const int m1_lo = std::max(-j1, J - j2);
    std::vector<double> c(d1, 0.0);
    c[j1 + j1] = 1.0;
    for (int mu1 = j1; mu1 > m1_lo; --mu1) c[mu1 - 1 + j1] = -c[mu1 + j1] * a_plus(j2, J - mu1) / a_plus(j1, mu1 - 1);
    double nrm = 0.0;
    for (int m1 = m1_lo; m1 <= j1; ++m1) nrm += c[m1 + j1] * c[m1 + j1];
    nrm = 1.0 / std::sqrt(nrm);  // c(j1) > 0: Condon-Shortley
    for (int m1 = m1_lo; m1 <= j1; ++m1) at(m1, J - m1, J) = c[m1 + j1] * nrm;
    // lowering: |J M-1> = J- |J M> / a-(J,M),  J- = J1- + J2-
    for (int M = J; M > -J; --M) {
        const double inv = 1.0 / a_minus(J, M);
        for (int m1 = -j1; m1 <= j1; ++m1) {
            int m2 = M - m1;
            if (m2 < -j2 || m2 > j2) continue;
            double v = at(m1, m2, M);
            if (v == 0.0) continue;
            if (m1 - 1 >= -j1) at(m1 - 1, m2, M - 1) += v * a_minus(j1, m1) * inv;
            if (m2 - 1 >= -j2) at(m1, m2 - 1, M - 1) += v * a_minus(j2, m2) * inv;
        }
    }
}

// real index m -> its (at most two) complex components: real_m = sum_t coef[t] * complex_{mu[t]}
struct RealRow {
    int cnt;
    int mu[2];
    std::complex<double> coef[2];
};
static RealRow real_row(int m) {
    RealRow r;
    const double s = std::sqrt(0.5);
    if (m == 0) {
        r.cnt = 1; r.mu[0] = 0; r.coef[0] = {1.0, 0.0};
        return r;
    }
    const int a = std::abs(m);
    const double sg = (a % 2) ? -1.0 : 1.0;
    r.cnt = 2; r.mu[0] = -a; r.mu[1] = a;
    if (m > 0) { r.coef[0] = {s, 0.0}; r.coef[1] = {sg * s, 0.0}; }
    else       { r.coef[0] = {0.0, s}; r.coef[1] = {0.0, -sg * s}; }
    return r;
}

void cg_real_block(int l1, int l2, int l3, std::vector<double>& C) {
    std::vector<double> cc;
    cg_complex_ladder(l1, l2, l3, cc);
    const int d1 = 2 * l1 + 1, d2 = 2 * l2 + 1, d3 = 2 * l3 + 1;
    C.assign((size_t)d1 * d2 * d3, 0.0);
    for (int m1 = -l1; m1 <= l1; ++m1) {
        RealRow r1 = real_row(m1);
        for (int m2 = -l2; m2 <= l2; ++m2) {
            RealRow r2 = real_row(m2);
            for (int M = -l3; M <= l3; ++M) {
                RealRow r3 = real_row(M);
                std::complex<double> t(0.0, 0.0);
                for (int a = 0; a < r1.cnt; ++a)
                    for (int b = 0; b < r2.cnt; ++b)
                        for (int c = 0; c < r3.cnt; ++c) {
                            if (r1.mu[a] + r2.mu[b] != r3.mu[c]) continue;
                            double g = cc[((size_t)(r1.mu[a] + l1) * d2 + (r2.mu[b] + l2)) * d3 + (r3.mu[c] + l3)];
                            t += std::conj(r1.coef[a]) * std::conj(r2.coef[b]) * r3.coef[c] * g;
                        }
                // purely real (l1+l2+l3 even) or purely imaginary (odd): keep the non-zero part
                C[((size_t)(m1 + l1) * d2 + (m2 + l2)) * d3 + (M + l3)] = t.real() + t.imag();
            }
        }
    }
}

static inline int feat_off(int l, int p) { return 2 * l * l + (p ? 2 * l + 1 : 0); }

void build_tables(int l_max, PlanTables& t) {
    t.l_max = l_max;
    t.dV = 2 * (l_max + 1) * (l_max + 1);
    t.dE = (l_max + 1) * (l_max + 1);
    t.paths.clear();
    t.nnz.clear();
    std::vector<double> C;
    for (int l1 = 0; l1 <= l_max; ++l1)
        for (int p1 = 0; p1 < 2; ++p1)
            for (int l2 = 0; l2 <= l_max; ++l2)
                for (int l3 = std::abs(l1 - l2); l3 <= std::min(l1 + l2, l_max); ++l3) {
                    PathInfo q{l1, p1, l2, l3, p1 ^ (l2 & 1), feat_off(l1, p1), l2 * l2, feat_off(l3, p1 ^ (l2 & 1))};
                    const int pid = (int)t.paths.size();
                    t.paths.push_back(q);
                    cg_real_block(l1, l2, l3, C);
                    const int d2 = 2 * l2 + 1, d3 = 2 * l3 + 1;
                    for (int a = 0; a < 2 * l1 + 1; ++a)
                        for (int b = 0; b < d2; ++b)
                            for (int c = 0; c < d3; ++c) {
                                double v = C[((size_t)a * d2 + b) * d3 + c];
                                if (std::fabs(v) > 1e-12) t.nnz.push_back(NonZero{pid, q.off1 + a, q.off2 + b, q.off3 + c, v});
                            }
                }
}

long build_segments(const int32_t* row_ptr, int n_atoms, int tile_edges, int32_t* items, long cap) {
    long cnt = 0;
    for (int i = 0; i < n_atoms; ++i) {
        const int a = row_ptr[i], b = row_ptr[i + 1];
        int e0 = a;
        do {
            const int e1 = std::min(e0 + tile_edges, b);
            if (items && cnt < cap) { items[3 * cnt] = i; items[3 * cnt + 1] = e0; items[3 * cnt + 2] = e1; }
            ++cnt;
            e0 = e1;
        } while (e0 < b);
    }
    return cnt;
}

}  // namespace allegro
