// env_kernels.cuh -- real spherical harmonics fused with the environment embedding and its VJP
// (north_star; "embedding of edge vectors ... to a radial-chemical and spherical harmonics basis").
//
// Y_lm is never stored: every kernel re-evaluates it from r_e (3 numbers per edge).  The harmonics here
// are the explicit Cartesian polynomials for l <= 3 in the convention of reading A1 (real,
// component-normalised, m = -l..l, Y_1 = sqrt3 (y, z, x)); the oracle uses the Legendre recursion
// instead, so the two share neither code nor algorithm.
#pragma once
#include "common.cuh"
#include "launch.h"
#include "radial.cuh"

namespace allegro {

// Y[DE] at the unit vector (x,y,z)
template <typename T, int L>
__device__ __forceinline__ void sph_harm(T x, T y, T z, T (&Y)[(L + 1) * (L + 1)]) {
    Y[0] = T(1);
    if constexpr (L >= 1) {
        const T s3 = T(1.7320508075688772935);
        Y[1] = s3 * y; Y[2] = s3 * z; Y[3] = s3 * x;
    }
    if constexpr (L >= 2) {
        const T s15 = T(3.8729833462074168852), s5h = T(1.1180339887498948482);
        Y[4] = s15 * x * y;
        Y[5] = s15 * y * z;
        Y[6] = s5h * (T(3) * z * z - T(1));
        Y[7] = s15 * x * z;
        Y[8] = T(0.5) * s15 * (x * x - y * y);
    }
    if constexpr (L >= 3) {
        const T a = T(2.0916500663351888699);   // sqrt(35/8)
        const T b = T(10.246950765959598383);   // sqrt(105)
        const T c = T(1.6201851746019651310);   // sqrt(21/8)
        const T d = T(1.3228756555322952953);   // sqrt(7)/2
        const T x2 = x * x, y2 = y * y, z2 = z * z;
        Y[9] = a * y * (T(3) * x2 - y2);
        Y[10] = b * x * y * z;
        Y[11] = c * y * (T(5) * z2 - T(1));
        Y[12] = d * z * (T(5) * z2 - T(3));
        Y[13] = c * x * (T(5) * z2 - T(1));
        Y[14] = T(0.5) * b * z * (x2 - y2);
        Y[15] = a * x * (x2 - T(3) * y2);
    }
}

// g[a] = sum_j gY[j] dY_j/du_a with (x,y,z) treated as independent variables (J~^T gY).  Any other
// polynomial extension off the sphere differs by a radial term that the projection below removes.
template <typename T, int L>
__device__ __forceinline__ void sph_harm_vjp(T x, T y, T z, const T (&gY)[(L + 1) * (L + 1)], T (&g)[3]) {
    g[0] = g[1] = g[2] = T(0);
    if constexpr (L >= 1) {
        const T s3 = T(1.7320508075688772935);
        g[1] += s3 * gY[1]; g[2] += s3 * gY[2]; g[0] += s3 * gY[3];
    }
    if constexpr (L >= 2) {
        const T s15 = T(3.8729833462074168852), s5 = T(2.2360679774997896964);
        g[0] += s15 * (y * gY[4] + z * gY[7] + x * gY[8]);
        g[1] += s15 * (x * gY[4] + z * gY[5] - y * gY[8]);
        g[2] += s15 * (y * gY[5] + x * gY[7]) + T(3) * s5 * z * gY[6];
    }
    if constexpr (L >= 3) {
        const T a = T(2.0916500663351888699), b = T(10.246950765959598383), c = T(1.6201851746019651310), d = T(1.3228756555322952953);
        const T x2 = x * x, y2 = y * y, z2 = z * z;
        const T f = T(5) * z2 - T(1);
        g[0] += a * (T(6) * x * y * gY[9] + T(3) * (x2 - y2) * gY[15]) + b * (y * z * gY[10] + x * z * gY[14]) + c * f * gY[13];
        g[1] += a * (T(3) * (x2 - y2) * gY[9] - T(6) * x * y * gY[15]) + b * (x * z * gY[10] - y * z * gY[14]) + c * f * gY[11];
        g[2] += b * (x * y * gY[10] + T(0.5) * (x2 - y2) * gY[14]) + c * T(10) * z * (y * gY[11] + x * gY[13]) + d * (T(15) * z2 - T(3)) * gY[12];
    }
}

// ------------------------------------------------------------------------------------------------
// Eenv[i][ch][j] = scale * sum_{e in item, CSR order per slot} w[e][ch] Y_j(rhat_e); slots combined in slot order.
// One CTA per item; thread <-> (edge slot, channel).  With `by_item` the row goes to the item's partial row.
template <typename T, int L, int THREADS>
__global__ void __launch_bounds__(THREADS) env_embed_kernel(int n, const int* __restrict__ row_ptr, const int* __restrict__ items,
                                                             const T* __restrict__ rvec, const T* __restrict__ w, T scale,
                                                             T* __restrict__ dst, int by_item) {
    constexpr int DE = (L + 1) * (L + 1);
    __shared__ T red[THREADS * DE];
    const int tid = threadIdx.x;
    const int nslots = THREADS / n;
    const int slot = tid / n, ch = tid - slot * n;
    const bool active = slot < nslots;
    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    T acc[DE];
#pragma unroll
    for (int j = 0; j < DE; ++j) acc[j] = T(0);
    if (active) {
        for (int e = e0 + slot; e < e1; e += nslots) {
            const T rx = rvec[3 * (size_t)e], ry = rvec[3 * (size_t)e + 1], rz = rvec[3 * (size_t)e + 2];
            const T wv = w[(size_t)e * n + ch];
            const T inv = T(1) / sqrt(rx * rx + ry * ry + rz * rz);
            T Y[DE];
            sph_harm<T, L>(rx * inv, ry * inv, rz * inv, Y);
#pragma unroll
            for (int j = 0; j < DE; ++j) acc[j] = fma(wv, Y[j], acc[j]);
        }
#pragma unroll
        for (int j = 0; j < DE; ++j) red[((size_t)slot * n + ch) * DE + j] = acc[j];
    }
    __syncthreads();
    if (slot == 0) {
        T* o = dst + ((size_t)(by_item ? (long)blockIdx.x : (long)c) * n + ch) * DE;
#pragma unroll
        for (int j = 0; j < DE; ++j) {
            T s = red[(size_t)ch * DE + j];
            for (int sl = 1; sl < nslots; ++sl) s += red[((size_t)sl * n + ch) * DE + j];
            o[j] = scale * s;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Sum 16 per-lane values over the 32 lanes of a warp with 16 shuffles instead of 80: at each step a lane
// hands one half of its live values to its partner and keeps the other half (recursive halving).  On
// return v[0] of lane l holds the total of input index (l >> 1) & 15.  Fixed shape -> deterministic.
template <typename T>
__device__ __forceinline__ void warp_reduce16(T (&v)[16], int lane) {
#pragma unroll
    for (int h = 8, bit = 16; h >= 1; h >>= 1, bit >>= 1) {
        const bool up = (lane & bit) != 0;
#pragma unroll
        for (int i = 0; i < h; ++i) {
            const T send = up ? v[i] : v[i + h];
            const T keep = up ? v[i + h] : v[i];
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, bit);
        }
    }
    v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
}

// VJP of the embedding.  One CTA (8 warps) per centre; warp <-> edge, lane <-> channels lane, lane+32, ...
// (CPL per lane), so w[e][:] and g_w[e][:] are read / written as whole coalesced rows and the centre's gEenv
// rows (times scale) stay in registers for the whole segment.  No block barrier.
//   g_w[e][ch] = sum_j gE[ch][j] Y_j(e)
//   gY_e[j]   = sum_ch gE[ch][j] w[e][ch]   -- lane-local over the lane's channels, then warp_reduce16
//   g_r[e]    = (1/|r|)(I - rhat rhat^T) J~^T gY_e
template <typename T, int L, int CPL>
__global__ void __launch_bounds__(256) env_embed_bwd_kernel(int n, const int* __restrict__ row_ptr, const T* __restrict__ gEenv,
                                                             const T* __restrict__ rvec, const T* __restrict__ w, T scale,
                                                             T* __restrict__ g_rvec, T* __restrict__ g_w) {
    constexpr int DE = (L + 1) * (L + 1);
    static_assert(DE <= 16, "warp_reduce16 handles l_max <= 3");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int c = blockIdx.x;
    const int e0 = row_ptr[c], e1 = row_ptr[c + 1];
    T gE[CPL][DE];
#pragma unroll
    for (int q = 0; q < CPL; ++q) {
        const int ch = lane + 32 * q;
#pragma unroll
        for (int j = 0; j < DE; ++j) gE[q][j] = ch < n ? scale * gEenv[((size_t)c * n + ch) * DE + j] : T(0);
    }
    for (int e = e0 + warp; e < e1; e += 8) {
        const T rx = rvec[3 * (size_t)e], ry = rvec[3 * (size_t)e + 1], rz = rvec[3 * (size_t)e + 2];
        const T inv = T(1) / sqrt(rx * rx + ry * ry + rz * rz);
        const T x = rx * inv, y = ry * inv, z = rz * inv;
        T Y[DE];
        sph_harm<T, L>(x, y, z, Y);
        T part[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) part[j] = T(0);
#pragma unroll
        for (int q = 0; q < CPL; ++q) {
            const int ch = lane + 32 * q;
            const T wv = ch < n ? w[(size_t)e * n + ch] : T(0);
            T gw = T(0);
#pragma unroll
            for (int j = 0; j < DE; ++j) { gw = fma(gE[q][j], Y[j], gw); part[j] = fma(gE[q][j], wv, part[j]); }
            if (g_w && ch < n) g_w[(size_t)e * n + ch] = gw;
        }
        warp_reduce16<T>(part, lane);
        T gY[DE];
#pragma unroll
        for (int j = 0; j < DE; ++j) gY[j] = __shfl_sync(0xffffffffu, part[0], 2 * j);
        if (lane == 0) {
            T g[3];
            sph_harm_vjp<T, L>(x, y, z, gY, g);
            const T dot = g[0] * x + g[1] * y + g[2] * z;
            g_rvec[3 * (size_t)e] = (g[0] - dot * x) * inv;
            g_rvec[3 * (size_t)e + 1] = (g[1] - dot * y) * inv;
            g_rvec[3 * (size_t)e + 2] = (g[2] - dot * z) * inv;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Fused geometry kernels: radial weights (A8) + Y_lm + environment embedding in one pass, and the matching VJP
// (embedding VJP + radial chain rule) in one pass.  w[E][n] and g_w[E][n] need not exist in HBM (both are optional
// outputs): per edge the kernels read r_e (12 bytes) only.  Arithmetic is the same as radial_fwd/bwd_kernel +
// env_embed(_bwd)_kernel: basis and W_r dot products in double, w rounded once to T, Y_lm and the sums in T.
// Mapping: CTA per item; chunks of kGeoChunk edges: phase 1, thread per edge -> basis, Y_lm, unit vector into
// shared memory; phase 2, warp per edge, lane <-> channels lane, lane+32, ... with their W_r rows in registers.
constexpr int kGeoChunk = 128;

template <typename T, int L, int NB>
struct GeoSmem {
    static constexpr int DE = (L + 1) * (L + 1);
    double Bs[kGeoChunk][NB];
    double dBs[kGeoChunk][NB];
    double rh[kGeoChunk][3];
    T Ys[kGeoChunk][DE];
    T geo[kGeoChunk][4];  // unit vector, 1/|r|
};

template <typename T, int L, int NB, bool WANT_D>
__device__ __forceinline__ void geo_phase1(GeoSmem<T, L, NB>& sm, int le, const T* __restrict__ rvec, size_t e, double rc, int nb) {
    constexpr int DE = (L + 1) * (L + 1);
    const T rx = rvec[3 * e], ry = rvec[3 * e + 1], rz = rvec[3 * e + 2];
    const double dx = (double)rx, dy = (double)ry, dz = (double)rz;
    const double rr = sqrt(dx * dx + dy * dy + dz * dz);
    double Bu[kMaxBasis], dBu[kMaxBasis];
    radial_basis<WANT_D>(rr, rc, nb, Bu, dBu);
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        sm.Bs[le][b] = b < nb ? Bu[b] : 0.0;
        if (WANT_D) sm.dBs[le][b] = b < nb ? dBu[b] : 0.0;
    }
    if (WANT_D) { sm.rh[le][0] = dx / rr; sm.rh[le][1] = dy / rr; sm.rh[le][2] = dz / rr; }
    const T inv = T(1) / sqrt(rx * rx + ry * ry + rz * rz);
    const T x = rx * inv, y = ry * inv, z = rz * inv;
    T Y[DE];
    sph_harm<T, L>(x, y, z, Y);
#pragma unroll
    for (int j = 0; j < DE; ++j) sm.Ys[le][j] = Y[j];
    sm.geo[le][0] = x; sm.geo[le][1] = y; sm.geo[le][2] = z; sm.geo[le][3] = inv;
}

template <typename T, int L, int CPL, int NB>
__global__ void __launch_bounds__(256) env_radial_fwd_kernel(int n, int nb, double rc, const T* __restrict__ rc_edge, const int* __restrict__ row_ptr, const int* __restrict__ items,
                                                              const T* __restrict__ rvec, const T* __restrict__ W_r, T scale,
                                                              T* __restrict__ w_out, T* __restrict__ dst, int by_item) {
    constexpr int DE = (L + 1) * (L + 1);
    extern __shared__ __align__(16) unsigned char geo_raw[];
    GeoSmem<T, L, NB>& sm = *reinterpret_cast<GeoSmem<T, L, NB>*>(geo_raw);
    T* red = reinterpret_cast<T*>(geo_raw + sizeof(GeoSmem<T, L, NB>));  // [32 * CPL][DE]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    double Wd[CPL][NB];
#pragma unroll
    for (int q = 0; q < CPL; ++q)
#pragma unroll
        for (int b = 0; b < NB; ++b) Wd[q][b] = (lane + 32 * q < n && b < nb) ? (double)W_r[(lane + 32 * q) * nb + b] : 0.0;
    T acc[CPL][DE];
#pragma unroll
    for (int q = 0; q < CPL; ++q)
#pragma unroll
        for (int j = 0; j < DE; ++j) acc[q][j] = T(0);

    for (int cb = e0; cb < e1; cb += kGeoChunk) {
        const int cnt = min(kGeoChunk, e1 - cb);
        if (tid < cnt) geo_phase1<T, L, NB, false>(sm, tid, rvec, (size_t)(cb + tid), rc_edge ? (double)rc_edge[(size_t)(cb + tid)] : rc, nb);
        __syncthreads();
        for (int le = warp; le < cnt; le += 8) {
            double Bv[NB];
#pragma unroll
            for (int b = 0; b < NB; ++b) Bv[b] = sm.Bs[le][b];
            T Y[DE];
#pragma unroll
            for (int j = 0; j < DE; ++j) Y[j] = sm.Ys[le][j];
#pragma unroll
            for (int q = 0; q < CPL; ++q) {
                double s = 0.0;
#pragma unroll
                for (int b = 0; b < NB; ++b) s = fma(Wd[q][b], Bv[b], s);
                const T wv = (T)s;
                if (w_out && lane + 32 * q < n) w_out[(size_t)(cb + le) * n + lane + 32 * q] = wv;
#pragma unroll
                for (int j = 0; j < DE; ++j) acc[q][j] = fma(wv, Y[j], acc[q][j]);
            }
        }
        __syncthreads();
    }
    // warps folded in warp order through one [n][DE] buffer
    for (int wv = 0; wv < 8; ++wv) {
        if (warp == wv) {
#pragma unroll
            for (int q = 0; q < CPL; ++q) {
                const int ch = lane + 32 * q;
                if (ch < n) {
#pragma unroll
                    for (int j = 0; j < DE; ++j) red[ch * DE + j] = (wv == 0 ? T(0) : red[ch * DE + j]) + acc[q][j];
                }
            }
        }
        __syncthreads();
    }
    T* o = dst + (size_t)(by_item ? (long)blockIdx.x : (long)c) * n * DE;
    for (int idx = tid; idx < n * DE; idx += 256) o[idx] = scale * red[idx];
}

template <typename T, int L, int CPL, int NB>
__global__ void __launch_bounds__(256) env_radial_bwd_kernel(int n, int nb, double rc, const T* __restrict__ rc_edge, const int* __restrict__ row_ptr, const T* __restrict__ gEenv,
                                                              const T* __restrict__ rvec, const T* __restrict__ W_r, T scale,
                                                              T* __restrict__ g_rvec, T* __restrict__ g_w) {
    constexpr int DE = (L + 1) * (L + 1);
    static_assert(DE <= 16, "warp_reduce16 handles l_max <= 3");
    extern __shared__ __align__(16) unsigned char geo_raw[];
    GeoSmem<T, L, NB>& sm = *reinterpret_cast<GeoSmem<T, L, NB>*>(geo_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int c = blockIdx.x;
    const int e0 = row_ptr[c], e1 = row_ptr[c + 1];
    double Wd[CPL][NB];
#pragma unroll
    for (int q = 0; q < CPL; ++q)
#pragma unroll
        for (int b = 0; b < NB; ++b) Wd[q][b] = (lane + 32 * q < n && b < nb) ? (double)W_r[(lane + 32 * q) * nb + b] : 0.0;
    T gE[CPL][DE];
#pragma unroll
    for (int q = 0; q < CPL; ++q) {
        const int ch = lane + 32 * q;
#pragma unroll
        for (int j = 0; j < DE; ++j) gE[q][j] = ch < n ? scale * gEenv[((size_t)c * n + ch) * DE + j] : T(0);
    }
    for (int cb = e0; cb < e1; cb += kGeoChunk) {
        const int cnt = min(kGeoChunk, e1 - cb);
        if (tid < cnt) geo_phase1<T, L, NB, true>(sm, tid, rvec, (size_t)(cb + tid), rc_edge ? (double)rc_edge[(size_t)(cb + tid)] : rc, nb);
        __syncthreads();
        for (int le = warp; le < cnt; le += 8) {
            const size_t e = (size_t)(cb + le);
            double Bv[NB], dBv[NB];
#pragma unroll
            for (int b = 0; b < NB; ++b) { Bv[b] = sm.Bs[le][b]; dBv[b] = sm.dBs[le][b]; }
            T Y[DE];
#pragma unroll
            for (int j = 0; j < DE; ++j) Y[j] = sm.Ys[le][j];
            T part[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) part[j] = T(0);
            double rad = 0.0;
#pragma unroll
            for (int q = 0; q < CPL; ++q) {
                double s = 0.0, ds = 0.0;
#pragma unroll
                for (int b = 0; b < NB; ++b) { s = fma(Wd[q][b], Bv[b], s); ds = fma(Wd[q][b], dBv[b], ds); }
                const T wv = (T)s;
                T gw = T(0);
#pragma unroll
                for (int j = 0; j < DE; ++j) { gw = fma(gE[q][j], Y[j], gw); part[j] = fma(gE[q][j], wv, part[j]); }
                if (g_w && lane + 32 * q < n) g_w[e * n + lane + 32 * q] = gw;
                rad = fma((double)gw, ds, rad);
            }
            warp_reduce16<T>(part, lane);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) rad += __shfl_xor_sync(0xffffffffu, rad, o);
            T gY[DE];
#pragma unroll
            for (int j = 0; j < DE; ++j) gY[j] = __shfl_sync(0xffffffffu, part[0], 2 * j);
            if (lane == 0) {
                const T x = sm.geo[le][0], y = sm.geo[le][1], z = sm.geo[le][2], inv = sm.geo[le][3];
                T g[3];
                sph_harm_vjp<T, L>(x, y, z, gY, g);
                const T dot = g[0] * x + g[1] * y + g[2] * z;
                g_rvec[3 * e] = (T)((double)((g[0] - dot * x) * inv) + rad * sm.rh[le][0]);
                g_rvec[3 * e + 1] = (T)((double)((g[1] - dot * y) * inv) + rad * sm.rh[le][1]);
                g_rvec[3 * e + 2] = (T)((double)((g[2] - dot * z) * inv) + rad * sm.rh[le][2]);
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// Factorised geometry kernels, used when w / g_w are not requested.  The radial weights are LINEAR in the small basis,
// w[e][ch] = sum_b W_r[ch][b] Bu_e[b], so the sums over a centre's edges and over channels can be regrouped exactly:
//   Eenv[c][ch][j] = scale sum_b W_r[ch][b] S_c[b][j],            S_c[b][j] = sum_{e in row c} Bu_e[b] Y_j(e)     (NB x DE per centre)
//   gY_e[j]        = sum_b Bu_e[b] M_c[b][j],                     M_c[b][j] = scale sum_ch gE[c][ch][j] W_r[ch][b]
//   sum_ch g_w[e][ch] dw[e][ch]/dr = sum_j Y_j(e) sum_b dBu_e[b] M_c[b][j]
// Per-edge work no longer scales with the channel count (72 FMAs instead of n x 17), and everything is in double.
template <typename T, int L, int NB>
__global__ void __launch_bounds__(kGeoChunk) env_radial_fwd_fact_kernel(int n, int nb, double rc, const T* __restrict__ rc_edge, const int* __restrict__ row_ptr,
                                                                         const int* __restrict__ items, const T* __restrict__ rvec,
                                                                         const T* __restrict__ W_r, double scale, T* __restrict__ dst, int by_item) {
    constexpr int DE = (L + 1) * (L + 1);
    extern __shared__ __align__(16) unsigned char geo_raw[];
    GeoSmem<T, L, NB>& sm = *reinterpret_cast<GeoSmem<T, L, NB>*>(geo_raw);
    double* S = reinterpret_cast<double*>(geo_raw + sizeof(GeoSmem<T, L, NB>));  // [NB][DE]
    const int tid = threadIdx.x;
    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    constexpr int R = (NB * DE + kGeoChunk - 1) / kGeoChunk;  // (basis, component) pairs per thread
    double sacc[R];
#pragma unroll
    for (int r = 0; r < R; ++r) sacc[r] = 0.0;
    for (int cb = e0; cb < e1; cb += kGeoChunk) {
        const int cnt = min(kGeoChunk, e1 - cb);
        if (tid < cnt) geo_phase1<T, L, NB, false>(sm, tid, rvec, (size_t)(cb + tid), rc_edge ? (double)rc_edge[(size_t)(cb + tid)] : rc, nb);
        __syncthreads();
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int t = tid + r * kGeoChunk;
            if (t < NB * DE) {
                const int b = t / DE, j = t - b * DE;
                for (int le = 0; le < cnt; ++le) sacc[r] = fma(sm.Bs[le][b], (double)sm.Ys[le][j], sacc[r]);
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < R; ++r)
        if (tid + r * kGeoChunk < NB * DE) S[tid + r * kGeoChunk] = sacc[r];
    __syncthreads();
    T* o = dst + (size_t)(by_item ? (long)blockIdx.x : (long)c) * n * DE;
    for (int idx = tid; idx < n * DE; idx += kGeoChunk) {
        const int ch = idx / DE, jj = idx - ch * DE;
        double acc = 0.0;
        for (int bb = 0; bb < nb; ++bb) acc = fma((double)W_r[ch * nb + bb], S[bb * DE + jj], acc);
        o[idx] = (T)(scale * acc);
    }
}

template <typename T, int L, int NB>
__global__ void __launch_bounds__(kGeoChunk) env_radial_bwd_fact_kernel(int n, int nb, double rc, const T* __restrict__ rc_edge, const int* __restrict__ row_ptr,
                                                                         const T* __restrict__ gEenv, const T* __restrict__ rvec,
                                                                         const T* __restrict__ W_r, double scale, T* __restrict__ g_rvec) {
    constexpr int DE = (L + 1) * (L + 1);
    __shared__ double Ms[NB * DE];
    extern __shared__ __align__(16) unsigned char geo_raw[];
    T* gEs = reinterpret_cast<T*>(geo_raw);  // [n][DE] the centre's gEenv rows
    T* Wrs = gEs + (size_t)n * DE;           // [n][nb]
    const int tid = threadIdx.x;
    const int c = blockIdx.x;
    const int e0 = row_ptr[c], e1 = row_ptr[c + 1];
    for (int idx = tid; idx < n * DE; idx += kGeoChunk) gEs[idx] = gEenv[(size_t)c * n * DE + idx];
    for (int idx = tid; idx < n * nb; idx += kGeoChunk) Wrs[idx] = W_r[idx];
    __syncthreads();
    for (int t = tid; t < NB * DE; t += kGeoChunk) {
        const int b = t / DE, j = t - b * DE;
        double m = 0.0;
        if (b < nb)
            for (int ch = 0; ch < n; ++ch) m = fma((double)gEs[ch * DE + j], (double)Wrs[ch * nb + b], m);
        Ms[t] = scale * m;
    }
    __syncthreads();
    for (int e = e0 + tid; e < e1; e += kGeoChunk) {
        const T rx = rvec[3 * (size_t)e], ry = rvec[3 * (size_t)e + 1], rz = rvec[3 * (size_t)e + 2];
        const double dx = (double)rx, dy = (double)ry, dz = (double)rz;
        const double rr = sqrt(dx * dx + dy * dy + dz * dz);
        double Bu[kMaxBasis], dBu[kMaxBasis];
        radial_basis<true>(rr, rc_edge ? (double)rc_edge[e] : rc, nb, Bu, dBu);
        const T inv = T(1) / sqrt(rx * rx + ry * ry + rz * rz);
        const T x = rx * inv, y = ry * inv, z = rz * inv;
        T Y[DE], gY[DE];
        sph_harm<T, L>(x, y, z, Y);
        double rad = 0.0;
#pragma unroll
        for (int j = 0; j < DE; ++j) {
            double gy = 0.0, dj = 0.0;
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                if (b < nb) { gy = fma(Bu[b], Ms[b * DE + j], gy); dj = fma(dBu[b], Ms[b * DE + j], dj); }
            }
            gY[j] = (T)gy;
            rad = fma((double)Y[j], dj, rad);
        }
        T g[3];
        sph_harm_vjp<T, L>(x, y, z, gY, g);
        const T dot = g[0] * x + g[1] * y + g[2] * z;
        g_rvec[3 * (size_t)e] = (T)((double)((g[0] - dot * x) * inv) + rad * dx / rr);
        g_rvec[3 * (size_t)e + 1] = (T)((double)((g[1] - dot * y) * inv) + rad * dy / rr);
        g_rvec[3 * (size_t)e + 2] = (T)((double)((g[2] - dot * z) * inv) + rad * dz / rr);
    }
}

// ------------------------------------------------------------------------------------------------
// Layer-0 edge embedding of the two-layer model (reading A19; BASELINE.json:configs[2]):
//   b_e = [B_b(r_e) u(r_e/r_c)],  x0[e][ch] = sum_b W_x0[ch][b] b_e[b],
//   V0[e][ch][(l, (-1)^l), m] = (sum_b W_v0[ch][b] b_e[b]) Y_lm(rhat_e), other-parity slots 0.
// CTA per kGeoChunk edges: phase 1 thread per edge (basis in double, Y_lm), phase 2 warp per edge, lanes over channels.
template <int L>
__device__ __forceinline__ constexpr int natural_slot(int j) {  // Eenv-style index l^2+l+m -> feature index of (l, (-1)^l, m)
    int l = 0;
    while ((l + 1) * (l + 1) <= j) ++l;
    return 2 * l * l + ((l & 1) ? 2 * l + 1 : 0) + (j - l * l);
}

// Feature rows of 32 consecutive channels of one edge are ONE contiguous byte range in HBM: they are staged per warp in shared
// memory and cross HBM as 16-byte vectors, lanes consecutive (a lane's own 72-byte row written or read directly costs nine
// strided 8-byte requests per warp: 4x the transactions).
template <typename T>
__device__ __forceinline__ void warp_copy(T* __restrict__ dst, const T* __restrict__ src, int nelem, int lane) {
    const bool vec = ((reinterpret_cast<uintptr_t>(dst) | reinterpret_cast<uintptr_t>(src)) & 15u) == 0 && (nelem * (int)sizeof(T)) % 16 == 0;
    if (vec) {
        const int nv = nelem * (int)sizeof(T) / 16;
        for (int i = lane; i < nv; i += 32) reinterpret_cast<int4*>(dst)[i] = reinterpret_cast<const int4*>(src)[i];
    } else {
        for (int i = lane; i < nelem; i += 32) dst[i] = src[i];
    }
}

template <typename T, int L, int NB>
__global__ void __launch_bounds__(256) edge_embed_kernel(int n, int nb, double rc, long E, const T* __restrict__ rvec, const T* __restrict__ W_x0,
                                                          const T* __restrict__ W_v0, T* __restrict__ x0, T* __restrict__ V0, T* __restrict__ v0_out) {
    constexpr int DE = (L + 1) * (L + 1), DV = 2 * DE;
    extern __shared__ __align__(16) unsigned char geo_raw[];
    GeoSmem<T, L, NB>& sm = *reinterpret_cast<GeoSmem<T, L, NB>*>(geo_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long cb = (long)blockIdx.x * kGeoChunk;
    const int cnt = (int)min((long)kGeoChunk, E - cb);
    T* stg = reinterpret_cast<T*>(geo_raw + ((sizeof(GeoSmem<T, L, NB>) + 15) / 16) * 16) + (size_t)warp * 32 * DV;   // [32 channels][DV] per warp
    // the two weight matrices transposed to [b][ch] in double: lanes run over channels, so the reads below are conflict-free (read
    // from global memory as W[ch][b] they cost 32 sectors per request)
    double* Wxs = reinterpret_cast<double*>(geo_raw + ((sizeof(GeoSmem<T, L, NB>) + 15) / 16) * 16 + (size_t)8 * 32 * DV * sizeof(T));
    double* Wvs = Wxs + (size_t)nb * n;
    for (int idx = tid; idx < n * nb; idx += 256) {
        const int ch = idx / nb, b = idx - ch * nb;
        Wxs[b * n + ch] = (double)W_x0[idx];
        Wvs[b * n + ch] = (double)W_v0[idx];
    }
    if (tid < cnt) geo_phase1<T, L, NB, false>(sm, tid, rvec, (size_t)(cb + tid), rc, nb);
    __syncthreads();
    // n <= 64: the weights of the lane's (at most two) channels live in registers for all of the warp's edges -- read from shared memory
    // per edge they are 4 wavefronts per basis function and the kernel is bound by the shared-memory pipe
    const bool wreg = n <= 64;
    double wx[2][NB], wv[2][NB];
#pragma unroll
    for (int g = 0; g < 2; ++g)
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const int ch = 32 * g + lane;
            const bool ok = wreg && ch < n && b < nb;
            wx[g][b] = ok ? Wxs[b * n + ch] : 0.0;
            wv[g][b] = ok ? Wvs[b * n + ch] : 0.0;
        }
    for (int le = warp; le < cnt; le += 8) {
        const size_t e = (size_t)(cb + le);
        double bus[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) bus[b] = b < nb ? sm.Bs[le][b] : 0.0;
        for (int ch0 = 0; ch0 < n; ch0 += 32) {
            const int ch = ch0 + lane;
            if (ch < n) {
                double sx = 0.0, sv = 0.0;
                if (wreg) {
                    const int g = ch0 >> 5;
#pragma unroll
                    for (int b = 0; b < NB; ++b) {
                        sx = fma(g ? wx[1][b] : wx[0][b], bus[b], sx);
                        sv = fma(g ? wv[1][b] : wv[0][b], bus[b], sv);
                    }
                } else {
                    for (int b = 0; b < nb; ++b) {      // (sm.Bs, not bus[b]: a run-time index would put bus into local memory)
                        const double bu = sm.Bs[le][b];
                        sx = fma(Wxs[b * n + ch], bu, sx);
                        sv = fma(Wvs[b * n + ch], bu, sv);
                    }
                }
                x0[e * n + ch] = (T)sx;
                const T v0 = (T)sv;
                if (v0_out != nullptr) v0_out[e * n + ch] = v0;      // the factor alone (V0 = v0 (x) Y is generated on chip by its consumer)
                if (V0 != nullptr) {
                    T row[DV];
#pragma unroll
                    for (int k = 0; k < DV; ++k) row[k] = T(0);
#pragma unroll
                    for (int j = 0; j < DE; ++j) row[natural_slot<L>(j)] = v0 * sm.Ys[le][j];
                    row_store<T, DV>(stg + lane * DV, row);
                }
            }
            if (V0 != nullptr) {
                __syncwarp();
                warp_copy<T>(V0 + (e * n + ch0) * DV, stg, min(32, n - ch0) * DV, lane);
                __syncwarp();
            }
        }
    }
}

// VJP of the edge embedding: g_rvec[e] += d/dr_e of ( <g_x0[e], x0[e]> + <gV0[e], V0[e]> )
template <typename T, int L, int NB>
__global__ void __launch_bounds__(256) edge_embed_bwd_kernel(int n, int nb, double rc, long E, const T* __restrict__ rvec,
                                                              const T* __restrict__ W_x0, const T* __restrict__ W_v0, const T* __restrict__ g_x0,
                                                              const T* __restrict__ gV0, T* __restrict__ g_rvec, const T* __restrict__ g_v0c,
                                                              const T* __restrict__ gYc) {
    // gV0 == NULL: the cotangent of V0 = v0 (x) Y arrives already contracted (allegro_tp_backward_outer): g_v0c[e][ch] = <gV0[e][ch], Y>,
    // gYc[e][j] = sum_ch gV0[e][ch][slot j] v0[e][ch]
    constexpr int DE = (L + 1) * (L + 1), DV = 2 * DE;
    static_assert(DE <= 16 && NB <= 16, "warp_reduce16");
    extern __shared__ __align__(16) unsigned char geo_raw[];
    GeoSmem<T, L, NB>& sm = *reinterpret_cast<GeoSmem<T, L, NB>*>(geo_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long cb = (long)blockIdx.x * kGeoChunk;
    const int cnt = (int)min((long)kGeoChunk, E - cb);
    T* stg = reinterpret_cast<T*>(geo_raw + ((sizeof(GeoSmem<T, L, NB>) + 15) / 16) * 16) + (size_t)warp * 32 * DV;   // [32 channels][DV] per warp
    double* Wxs = reinterpret_cast<double*>(geo_raw + ((sizeof(GeoSmem<T, L, NB>) + 15) / 16) * 16 + (size_t)8 * 32 * DV * sizeof(T));   // [b][ch]
    double* Wvs = Wxs + (size_t)nb * n;
    for (int idx = tid; idx < n * nb; idx += 256) {
        const int ch = idx / nb, b = idx - ch * nb;
        Wxs[b * n + ch] = (double)W_x0[idx];
        Wvs[b * n + ch] = (double)W_v0[idx];
    }
    if (tid < cnt) geo_phase1<T, L, NB, true>(sm, tid, rvec, (size_t)(cb + tid), rc, nb);
    __syncthreads();
    for (int le = warp; le < cnt; le += 8) {
        const size_t e = (size_t)(cb + le);
        T gYp[16];
        double gbp[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) { gYp[j] = T(0); gbp[j] = 0.0; }
        for (int ch0 = 0; ch0 < n; ch0 += 32) {
            T gv0 = T(0);
            const int ch = ch0 + lane;
            if (gV0 != nullptr) {
                __syncwarp();
                warp_copy<T>(stg, gV0 + (e * n + ch0) * DV, min(32, n - ch0) * DV, lane);
                __syncwarp();
                if (ch >= n) continue;
                T row[DV];
                row_load<T, DV>(stg + lane * DV, row);
                double sv = 0.0;
                for (int b = 0; b < nb; ++b) sv = fma(Wvs[b * n + ch], sm.Bs[le][b], sv);
                const T v0 = (T)sv;
#pragma unroll
                for (int j = 0; j < DE; ++j) {
                    const T gj = row[natural_slot<L>(j)];
                    gv0 = fma(gj, sm.Ys[le][j], gv0);
                    gYp[j] = fma(gj, v0, gYp[j]);
                }
            } else {
                if (ch >= n) continue;
                gv0 = g_v0c[e * n + ch];
            }
            const double gx = (double)g_x0[e * n + ch];
#pragma unroll
            for (int b = 0; b < NB; ++b)
                if (b < nb) gbp[b] += gx * Wxs[b * n + ch] + (double)gv0 * Wvs[b * n + ch];
        }
        warp_reduce16<T>(gYp, lane);
        warp_reduce16<double>(gbp, lane);
        T gY[DE];
#pragma unroll
        for (int j = 0; j < DE; ++j) gY[j] = __shfl_sync(0xffffffffu, gYp[0], 2 * j);
        if (gV0 == nullptr) {
#pragma unroll
            for (int j = 0; j < DE; ++j) gY[j] = gYc[e * DE + j];
        }
        double rad = 0.0;
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const double gb = __shfl_sync(0xffffffffu, gbp[0], 2 * b);
            rad = fma(gb, sm.dBs[le][b], rad);
        }
        if (lane == 0) {
            const T x = sm.geo[le][0], y = sm.geo[le][1], z = sm.geo[le][2], inv = sm.geo[le][3];
            T g[3];
            sph_harm_vjp<T, L>(x, y, z, gY, g);
            const T dot = g[0] * x + g[1] * y + g[2] * z;
            g_rvec[3 * e] = (T)((double)g_rvec[3 * e] + (double)((g[0] - dot * x) * inv) + rad * sm.rh[le][0]);
            g_rvec[3 * e + 1] = (T)((double)g_rvec[3 * e + 1] + (double)((g[1] - dot * y) * inv) + rad * sm.rh[le][1]);
            g_rvec[3 * e + 2] = (T)((double)g_rvec[3 * e + 2] + (double)((g[2] - dot * z) * inv) + rad * sm.rh[le][2]);
        }
    }
}

// VJP of the edge embedding from the FACTORS of the cotangent of V0 = v0 (x) Y (allegro_edge_embed_factors_backward): thread per edge,
//   g_b[b] = sum_ch ( g_x0[e][ch] W_x0[ch][b] + g_v0[e][ch] W_v0[ch][b] ),   g_rvec[e] += (sum_b g_b dBu_b/dr) rhat_e + proj(J^T gY[e]) / |r_e|
// with the weights broadcast from shared memory ([b][ch], double); no cross-lane reduction at all.
template <typename T, int L, int NB>
__global__ void __launch_bounds__(kGeoChunk) edge_embed_factors_bwd_kernel(int n, int nb, double rc, long E, const T* __restrict__ rvec,
                                                                           const T* __restrict__ W_x0, const T* __restrict__ W_v0,
                                                                           const T* __restrict__ g_x0, const T* __restrict__ g_v0,
                                                                           const T* __restrict__ gYc, T* __restrict__ g_rvec) {
    constexpr int DE = (L + 1) * (L + 1);
    extern __shared__ __align__(16) unsigned char geo_raw[];
    double* Wxs = reinterpret_cast<double*>(geo_raw);   // [ch][NB] (ch-major: one thread walks ch, all threads read the same address)
    double* Wvs = Wxs + (size_t)n * NB;
    const int tid = threadIdx.x;
    for (int idx = tid; idx < n * NB; idx += kGeoChunk) {
        const int ch = idx / NB, b = idx - ch * NB;
        Wxs[idx] = b < nb ? (double)W_x0[ch * nb + b] : 0.0;
        Wvs[idx] = b < nb ? (double)W_v0[ch * nb + b] : 0.0;
    }
    const long cb = (long)blockIdx.x * kGeoChunk;
    const long e = cb + tid;
    const bool live = e < E;
    const int cnt = (int)min((long)kGeoChunk, E - cb);
    // the chunk's cotangent rows, 32 channels at a time: loaded with lanes along the channels (coalesced), read back one ROW per thread
    // from rows padded to 33 words (conflict-free).  Read straight from global memory a thread walks its own 256-byte row: one sector
    // per lane and load, 32 wavefronts per request
    T* xs = reinterpret_cast<T*>(Wvs + (size_t)n * NB);     // [chunk][33]
    T* vs = xs + kGeoChunk * 33;
    const T rx = live ? rvec[3 * e] : T(1), ry = live ? rvec[3 * e + 1] : T(0), rz = live ? rvec[3 * e + 2] : T(0);
    const double dx = (double)rx, dy = (double)ry, dz = (double)rz;
    const double rr = sqrt(dx * dx + dy * dy + dz * dz);
    double Bu[kMaxBasis], dBu[kMaxBasis];
    radial_basis<true>(rr, rc, nb, Bu, dBu);
    double gb[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) gb[b] = 0.0;
    for (int c0 = 0; c0 < n; c0 += 32) {
        const int cw = min(32, n - c0);
        __syncthreads();
        for (int idx = tid; idx < cnt * 32; idx += kGeoChunk) {
            const int le = idx >> 5, cc = idx & 31;
            if (cc < cw) {
                xs[le * 33 + cc] = g_x0[(size_t)(cb + le) * n + c0 + cc];
                vs[le * 33 + cc] = g_v0[(size_t)(cb + le) * n + c0 + cc];
            }
        }
        __syncthreads();
        if (live) {
            for (int cc = 0; cc < cw; ++cc) {
                const double a = (double)xs[tid * 33 + cc], c = (double)vs[tid * 33 + cc];
                const int ch = c0 + cc;
#pragma unroll
                for (int b = 0; b < NB; ++b) gb[b] = fma(a, Wxs[ch * NB + b], fma(c, Wvs[ch * NB + b], gb[b]));
            }
        }
    }
    if (!live) return;
    double rad = 0.0;
#pragma unroll
    for (int b = 0; b < NB; ++b)
        if (b < nb) rad = fma(gb[b], dBu[b], rad);
    const T inv = T(1) / sqrt(rx * rx + ry * ry + rz * rz);
    const T x = rx * inv, y = ry * inv, z = rz * inv;
    T gY[DE], g[3];
#pragma unroll
    for (int j = 0; j < DE; ++j) gY[j] = gYc[(size_t)e * DE + j];
    sph_harm_vjp<T, L>(x, y, z, gY, g);
    const T dot = g[0] * x + g[1] * y + g[2] * z;
    g_rvec[3 * e] = (T)((double)g_rvec[3 * e] + (double)((g[0] - dot * x) * inv) + rad * (dx / rr));
    g_rvec[3 * e + 1] = (T)((double)g_rvec[3 * e + 1] + (double)((g[1] - dot * y) * inv) + rad * (dy / rr));
    g_rvec[3 * e + 2] = (T)((double)g_rvec[3 * e + 2] + (double)((g[2] - dot * z) * inv) + rad * (dz / rr));
}

}  // namespace allegro
