/*
 * allegro_oracle.h -- C API of the float64 CPU oracle.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this library.  The
 * product path (paper_2504_16068_b200/, include/) never links, imports or calls
 * anything in oracle/, and shares no source, table or generator with it.
 *
 * What it computes: the Allegro per-edge equivariant tensor product with its
 * environment embedding and first derivative, as a plain definition in float64,
 * single-threaded, no blocking / fusion / reordering.
 *   PAPER.md:65-71  (Sec. II.D "Optimized Tensor Product Kernel": the tensor product
 *                    and its first derivative; combined Wigner-3j tensor; no outer
 *                    product intermediates)
 *   PAPER.md:170    (App. A: embedding = radial basis x spherical harmonics)
 *   BASELINE.json:north_star (the formulas; CG from the Racah closed form, Y_lm from
 *                    the explicit recursion)
 * The paper prints no equations; every convention is a DESIGN.md reading (A1..A21)
 * and is cited beside the function that applies it.
 *
 * All arrays are row-major, caller-owned host memory.  Feature layout
 *   V / out / G / gV : [E][n][dV],  dV = 2 (lmax+1)^2, component index
 *                      off(l,p) + (m + l),  off(l,p) = 2 l^2 + (p == odd ? 2l+1 : 0)
 *   Eenv / gEenv     : [N][n][dE],  dE = (lmax+1)^2, component index l^2 + l + m
 * (reading A3).
 */
#ifndef ALLEGRO_ORACLE_H
#define ALLEGRO_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* ---- tables ------------------------------------------------------------------ */
int     orc_dim_v(int lmax);
int     orc_dim_e(int lmax);
/* complex Clebsch-Gordan <j1 m1 j2 m2 | j3 m3>, Racah closed form, Condon-Shortley */
double  orc_cg_complex(int j1, int m1, int j2, int m2, int j3, int m3);
/* real-basis CG block C[m1][m2][M] (sizes 2l+1), reading A2: C = Re T + Im T.
 * max_re / max_im receive max|Re T|, max|Im T| (one of them is ~0). */
void    orc_cg_real(int l1, int l2, int l3, double* C, double* max_re, double* max_im);
/* path plan, reading A3: lexicographic (l1, p1 [even<odd], l2, l3); parity 0=even 1=odd */
int     orc_num_paths(int lmax);
void    orc_paths(int lmax, int32_t* l1, int32_t* p1, int32_t* l2, int32_t* l3, int32_t* p3,
                  int32_t* off1, int32_t* off2, int32_t* off3);
/* sparse list of all paths' non-zeros (|c| > 1e-12), sorted (path, i, j, k);
 * i indexes V comps, j indexes Eenv comps, k indexes out comps */
int64_t orc_nnz(int lmax);
void    orc_cg_list(int lmax, int32_t* path, int32_t* i, int32_t* j, int32_t* k, double* coef);

/* ---- spherical harmonics / rotations ------------------------------------------- */
/* Y[dE] = real component-normalised Y_lm(r/|r|) (reading A1), dYdr[dE][3] = dY/dr */
void    orc_sph_harm(int lmax, const double* r, double* Y, double* dYdr);
/* R = Rz(alpha) Ry(beta) Rz(gamma), row-major 3x3 */
void    orc_rotation_matrix(double alpha, double beta, double gamma, double* R);
/* real-basis Wigner matrix with Y(R r) = D Y(r); D is (2l+1)x(2l+1) row-major */
void    orc_wigner_D_real(int l, double alpha, double beta, double gamma, double* D);

/* ---- radial weights (step 0, readings A5/A8) -------------------------------------- */
/* w[e][n] = sum_b Wr[n][b] B_b(|r_e|) u(|r_e|/rc),  dwdr[e][n] = d w / d |r| */
void    orc_radial(int n, int nb, double rc, const double* Wr, int64_t E, const double* rvec,
                   double* w, double* dwdr);
/* g_rvec[e] += (sum_n g_w[e][n] dwdr[e][n]) r_e/|r_e| */
void    orc_radial_backward(int n, int64_t E, const double* rvec, const double* g_w,
                            const double* dwdr, double* g_rvec);

/* ---- segment plan (reading A16) ------------------------------------------------------ */
int64_t orc_segments(const int32_t* row_ptr, int N, int T, int32_t* items, int64_t cap);

/* ---- the path ---------------------------------------------------------------------- */
void    orc_env_embed(int lmax, int n, int N, const int32_t* row_ptr, const double* rvec,
                      const double* w, double scale, double* Eenv);
/* wmode 0: path_w[P]; wmode 1: path_w[P][n][n] (out channel, in channel).
 * centre[e] is derived from row_ptr. c_lo..c_hi restricts the work to those centres' edges
 * (other rows of out are left untouched). */
void    orc_tp_forward_dense(int lmax, int n, int wmode, int N, const int32_t* row_ptr,
                             int c_lo, int c_hi, const double* V, const double* Eenv,
                             const double* path_w, double* out);
void    orc_tp_forward_sparse(int lmax, int n, int wmode, int N, const int32_t* row_ptr,
                              int c_lo, int c_hi, const double* V, const double* Eenv,
                              const double* path_w, double* out);
/* VJP.  gV nullable; g_path_w nullable (accumulated into, caller zeroes);
 * gEenv rows c_lo..c_hi are overwritten. */
void    orc_tp_backward(int lmax, int n, int wmode, int N, const int32_t* row_ptr,
                        int c_lo, int c_hi, const double* G, const double* V, const double* Eenv,
                        const double* path_w, double* gV, double* gEenv, double* g_path_w);
void    orc_env_embed_backward(int lmax, int n, int N, const int32_t* row_ptr, int c_lo, int c_hi,
                               const double* gEenv, const double* rvec, const double* w,
                               double scale, double* g_rvec, double* g_w);
void    orc_force_gather(int N, const int32_t* row_ptr, const int32_t* rev, const double* g_rvec,
                         double* F);
/* reading A12: e_edge[e] = sum_n ( q[n] out[e][n][0] + kappa/2 sum_k out[e][n][k]^2 ),
 * G = q (x) delta_{k,0} + kappa out.  e_edge, G nullable. */
void    orc_edge_energy(int lmax, int n, int64_t E, const double* out, const double* q,
                        double kappa, double* e_edge, double* G);
/* out[s] = sum_{i = ptr[s]}^{ptr[s+1]-1} vals[i], sequential */
void    orc_segment_sum(const int32_t* ptr, int nseg, const double* vals, double* out);
/* gradients of S = <aV, gV> + <bE, gE> of orc_tp_backward's outputs (scalar weights) with respect to G, V, Eenv, path_w (reading A26) */
void    orc_tp_double_backward(int lmax, int n, int N, const int32_t* row_ptr, const double* G, const double* V, const double* Eenv,
                               const double* path_w, const double* aV, const double* bE, double* dG, double* dV, double* dE, double* dw);
/* W[a][b] = sum_e g_rvec[e][a] rvec[e][b]  (reading A25: dE/d(strain), directed edges) */
void    orc_virial(int64_t E, const double* rvec, const double* g_rvec, double* W);


#ifdef __cplusplus
}
#endif
#endif
