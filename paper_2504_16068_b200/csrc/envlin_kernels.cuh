// envlin_kernels.cuh -- environment embedding of LINEAR per-edge weights, w[e][n] = sum_m W[n][m] x[e][m] (the per-edge linear
// map of the stacked model, reading A19), without ever forming w: the sums over edges and over m commute, so per centre c
//   forward : S_c[m][j] = sum_{e in row c} x[e][m] Y_j(rhat_e)              (n_in x dE),   Eenv[c][n][j] = scale sum_m W[n][m] S_c[m][j]
//   VJP     : M_c[m][j] = scale sum_n W[n][m] gEenv[c][n][j]                (n_in x dE)
//             g_x[e][m]  (+)= sum_j M_c[m][j] Y_j(rhat_e)                    (= sum_n W[n][m] g_w[e][n])
//             gY_e[j]      = sum_m M_c[m][j] x[e][m],   g_rvec[e] (+)= (I - rhat rhat^T) J^T gY_e / |r_e|
// The per-edge n_in x n GEMM (and its transpose in the VJP) becomes one n x n_in x dE product per CENTRE: ~deg / dE times fewer
// FMAs, and neither w[E][n] nor g_w[E][n] crosses HBM.  One CTA (256 threads) per centre; every sum has a fixed order.
// Included by inst_env.cu once per (ALLEGRO_T, ALLEGRO_L).
#pragma once
#include "common.cuh"
#include "launch.h"

namespace allegro {

constexpr int kEnvLinThreads = 256, kEnvLinChunk = 128;

template <typename T, int L>
__global__ void __launch_bounds__(kEnvLinThreads) env_linear_fwd_kernel(int n_atoms, int n_out, int n_in, const int* __restrict__ row_ptr, const T* __restrict__ rvec,
                                                                         const T* __restrict__ x, const T* __restrict__ W, T scale,
                                                                         T* __restrict__ Eenv) {
    constexpr int DE = (L + 1) * (L + 1);
    extern __shared__ __align__(16) unsigned char envlin_raw[];
    T* Ys = reinterpret_cast<T*>(envlin_raw);                 // [chunk][DE]
    T* red = Ys + kEnvLinChunk * DE;                           // [threads][DE] per-slot partial sums, then S[n_in][DE] in its first rows
    T* Wt = red + kEnvLinThreads * DE;                         // [n_in][n_out + 1]: W transposed, rows padded (conflict-free both ways)
    const int tid = threadIdx.x;
    const int ldw = n_out + 1;
    T* part = Wt + (size_t)n_in * ldw;                         // [threads / n_out][n_out][DE]: partial sums of the per-centre product
    const int nslots = kEnvLinThreads / n_in;
    const int slot = tid / n_in, m = tid - slot * n_in;
    const bool active = slot < nslots;
    for (int idx = tid; idx < n_out * n_in; idx += kEnvLinThreads) {     // once per CTA: the CTA walks centres blockIdx.x, + gridDim.x, ...
        const int n = idx / n_in, mm = idx - n * n_in;
        Wt[mm * ldw + n] = W[idx];
    }
    for (int c = blockIdx.x; c < n_atoms; c += gridDim.x) {
    const int e0 = row_ptr[c], e1 = row_ptr[c + 1];
    T acc[DE];
#pragma unroll
    for (int j = 0; j < DE; ++j) acc[j] = T(0);
    for (int cb = e0; cb < e1; cb += kEnvLinChunk) {
        const int cnt = min(kEnvLinChunk, e1 - cb);
        __syncthreads();
        if (tid < cnt) {
            const size_t e = (size_t)(cb + tid);
            const T rx = rvec[3 * e], ry = rvec[3 * e + 1], rz = rvec[3 * e + 2];
            const T inv = T(1) / sqrt(rx * rx + ry * ry + rz * rz);
            T Y[DE];
            sph_harm<T, L>(rx * inv, ry * inv, rz * inv, Y);
#pragma unroll
            for (int j = 0; j < DE; ++j) Ys[tid * DE + j] = Y[j];
        }
        __syncthreads();
        if (active) {
            int le = slot;
            for (; le + 3 * nslots < cnt; le += 4 * nslots) {      // four rows in flight: the loop is bound by the latency of the x loads
                T xv[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) xv[u] = x[(size_t)(cb + le + u * nslots) * n_in + m];
#pragma unroll
                for (int u = 0; u < 4; ++u)
#pragma unroll
                    for (int j = 0; j < DE; ++j) acc[j] = fma(xv[u], Ys[(le + u * nslots) * DE + j], acc[j]);
            }
            for (; le < cnt; le += nslots) {
                const T xv = x[(size_t)(cb + le) * n_in + m];
#pragma unroll
                for (int j = 0; j < DE; ++j) acc[j] = fma(xv, Ys[le * DE + j], acc[j]);
            }
        }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < DE; ++j) red[tid * DE + j] = acc[j];
    __syncthreads();
    if (slot == 0) {     // S[m][j]: slots in slot order (into the first n_in rows; thread m only touches row m and rows sl * n_in + m)
#pragma unroll
        for (int j = 0; j < DE; ++j) {
            T s = red[m * DE + j];
            for (int sl = 1; sl < nslots; ++sl) s += red[(sl * n_in + m) * DE + j];
            acc[j] = s;
        }
    }
    __syncthreads();
    if (slot == 0) {
#pragma unroll
        for (int j = 0; j < DE; ++j) red[m * DE + j] = acc[j];
    }
    __syncthreads();
    // Eenv[c][n][j] = scale sum_m W[n][m] S[m][j]: thread (q, n) holds the DE sums of output channel n over the q-th part of the m
    // range (one W load and DE broadcast loads of S per DE FMAs); the parts are then added in q order
    {
        const int nq = kEnvLinThreads / n_out;                    // parts of the m range (4 at n = 64); n_out <= 256
        const int q = tid / n_out, n = tid - q * n_out;
        if (q < nq) {
            const int m0 = (int)((long)n_in * q / nq), m1 = (int)((long)n_in * (q + 1) / nq);
            T s[DE];
#pragma unroll
            for (int j = 0; j < DE; ++j) s[j] = T(0);
            for (int mm = m0; mm < m1; ++mm) {
                const T w = Wt[mm * ldw + n];
#pragma unroll
                for (int j = 0; j < DE; ++j) s[j] = fma(w, red[mm * DE + j], s[j]);
            }
#pragma unroll
            for (int j = 0; j < DE; ++j) part[((size_t)q * n_out + n) * DE + j] = s[j];
        }
        __syncthreads();
        for (int idx = tid; idx < n_out * DE; idx += kEnvLinThreads) {     // idx = n * DE + j: the store is contiguous
            T t = part[idx];
            for (int qq = 1; qq < nq; ++qq) t += part[(size_t)qq * n_out * DE + idx];
            Eenv[(size_t)c * n_out * DE + idx] = scale * t;
        }
    }
    __syncthreads();     // red / Ys / part are rewritten by the next centre
    }
}

template <typename T, int L>
__global__ void __launch_bounds__(kEnvLinThreads) env_linear_bwd_kernel(int n_out, int n_in, const int* __restrict__ row_ptr, const T* __restrict__ gEenv,
                                                                         const T* __restrict__ rvec, const T* __restrict__ x, const T* __restrict__ W,
                                                                         T scale, T* __restrict__ g_rvec, int acc_g_rvec, T* __restrict__ g_x, int acc_g_x,
                                                                         int stage_x) {
    constexpr int DE = (L + 1) * (L + 1);
    extern __shared__ __align__(16) unsigned char envlin_raw[];
    T* Ys = reinterpret_cast<T*>(envlin_raw);                 // [chunk][DE]
    T* geo = Ys + kEnvLinChunk * DE;                           // [chunk][4]: unit vector, 1/|r|
    T* gEs = geo + kEnvLinChunk * 4;                           // [n_out][DE]
    T* Ms = gEs + n_out * DE;                                  // [n_in][DE]
    T* part = Ms + n_in * DE;                                  // [chunk][DE]: the second half-sum of gY
    // [chunk][n_in + 1] (stage_x): the chunk's x rows, loaded with lanes along m (coalesced).  The gY sum walks a ROW per thread:
    // from global memory that is one 32-byte sector per lane and load (32 L1 wavefronts per request), from the padded rows here
    // it is conflict-free
    T* mpart = part + kEnvLinChunk * DE;                       // [threads / n_in][n_in][DE]: partial sums of M
    T* xs = mpart + kEnvLinThreads * DE;
    const int ldx = n_in + 1;
    const int tid = threadIdx.x;
    const int c = blockIdx.x;
    const int e0 = row_ptr[c], e1 = row_ptr[c + 1];
    const int nslots = kEnvLinThreads / n_in;
    const int slot = tid / n_in, m = tid - slot * n_in;
    const bool active = slot < nslots;
    for (int idx = tid; idx < n_out * DE; idx += kEnvLinThreads) gEs[idx] = gEenv[(size_t)c * n_out * DE + idx];
    __syncthreads();
    // M[m][j] = scale sum_n W[n][m] gE[n][j]: thread (q, m) holds the DE sums of row m over the q-th part of the n range (lanes run
    // over m: coalesced rows of W, one load per DE FMAs); the parts are added in q order.
    {
        const int nq = kEnvLinThreads / n_in;
        const int q = tid / n_in, mm = tid - q * n_in;
        if (q < nq) {
            const int n0 = (int)((long)n_out * q / nq), n1 = (int)((long)n_out * (q + 1) / nq);
            T sacc[DE];
#pragma unroll
            for (int j = 0; j < DE; ++j) sacc[j] = T(0);
            for (int n = n0; n < n1; ++n) {
                const T w = W[(size_t)n * n_in + mm];
#pragma unroll
                for (int j = 0; j < DE; ++j) sacc[j] = fma(w, gEs[n * DE + j], sacc[j]);
            }
#pragma unroll
            for (int j = 0; j < DE; ++j) mpart[((size_t)q * n_in + mm) * DE + j] = sacc[j];
        }
        __syncthreads();
        for (int idx = tid; idx < n_in * DE; idx += kEnvLinThreads) {
            T t = mpart[idx];
            for (int qq = 1; qq < nq; ++qq) t += mpart[(size_t)qq * n_in * DE + idx];
            Ms[idx] = scale * t;
        }
    }
    for (int cb = e0; cb < e1; cb += kEnvLinChunk) {
        const int cnt = min(kEnvLinChunk, e1 - cb);
        __syncthreads();
        if (tid < cnt) {
            const size_t e = (size_t)(cb + tid);
            const T rx = rvec[3 * e], ry = rvec[3 * e + 1], rz = rvec[3 * e + 2];
            const T inv = T(1) / sqrt(rx * rx + ry * ry + rz * rz);
            const T ux = rx * inv, uy = ry * inv, uz = rz * inv;
            T Y[DE];
            sph_harm<T, L>(ux, uy, uz, Y);
#pragma unroll
            for (int j = 0; j < DE; ++j) Ys[tid * DE + j] = Y[j];
            geo[tid * 4] = ux; geo[tid * 4 + 1] = uy; geo[tid * 4 + 2] = uz; geo[tid * 4 + 3] = inv;
        }
        if (stage_x) {
            for (int idx = tid; idx < cnt * n_in; idx += kEnvLinThreads) {
                const int le = idx / n_in, mm = idx - le * n_in;
                xs[le * ldx + mm] = x[(size_t)cb * n_in + idx];
            }
        }
        __syncthreads();
        if (active) {        // g_x[e][m] = sum_j M[m][j] Y_j(e)
            T Mr[DE];
#pragma unroll
            for (int j = 0; j < DE; ++j) Mr[j] = Ms[m * DE + j];
            int le = slot;
            for (; le + 3 * nslots < cnt; le += 4 * nslots) {      // four rows in flight (the accumulate variant waits on its loads)
                T* dst = g_x + (size_t)(cb + le) * n_in + m;
                const size_t st = (size_t)nslots * n_in;
                T old[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) old[u] = acc_g_x ? dst[u * st] : T(0);
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    T sv = T(0);
#pragma unroll
                    for (int j = 0; j < DE; ++j) sv = fma(Mr[j], Ys[(le + u * nslots) * DE + j], sv);
                    dst[u * st] = old[u] + sv;
                }
            }
            for (; le < cnt; le += nslots) {
                T sv = T(0);
#pragma unroll
                for (int j = 0; j < DE; ++j) sv = fma(Mr[j], Ys[le * DE + j], sv);
                T* dst = g_x + (size_t)(cb + le) * n_in + m;
                *dst = acc_g_x ? *dst + sv : sv;
            }
        }
        {   // gY_e[j] = sum_m M[m][j] x[e][m]: thread (half, edge) sums one half of the m range; halves added in order
            const int half = tid / kEnvLinChunk, le = tid - half * kEnvLinChunk;
            const int m0 = half ? n_in / 2 : 0, m1 = half ? n_in : n_in / 2;
            T gYh[DE];
#pragma unroll
            for (int j = 0; j < DE; ++j) gYh[j] = T(0);
            if (le < cnt) {
                const T* xr = stage_x ? xs + le * ldx : x + (size_t)(cb + le) * n_in;
                for (int mm = m0; mm < m1; ++mm) {
                    const T xv = xr[mm];
#pragma unroll
                    for (int j = 0; j < DE; ++j) gYh[j] = fma(Ms[mm * DE + j], xv, gYh[j]);
                }
                if (half) {
#pragma unroll
                    for (int j = 0; j < DE; ++j) part[le * DE + j] = gYh[j];
                }
            }
            __syncthreads();
            if (half == 0 && le < cnt) {
#pragma unroll
                for (int j = 0; j < DE; ++j) gYh[j] += part[le * DE + j];
            }
            if (half != 0 || le >= cnt) continue;
            const size_t e = (size_t)(cb + tid);
            T gY[DE];
#pragma unroll
            for (int j = 0; j < DE; ++j) gY[j] = gYh[j];
            const T ux = geo[tid * 4], uy = geo[tid * 4 + 1], uz = geo[tid * 4 + 2], inv = geo[tid * 4 + 3];
            T g[3];
            sph_harm_vjp<T, L>(ux, uy, uz, gY, g);
            const T dot = g[0] * ux + g[1] * uy + g[2] * uz;
            const T r0 = (g[0] - dot * ux) * inv, r1 = (g[1] - dot * uy) * inv, r2 = (g[2] - dot * uz) * inv;
            T* dst = g_rvec + 3 * e;
            if (acc_g_rvec) { dst[0] += r0; dst[1] += r1; dst[2] += r2; } else { dst[0] = r0; dst[1] = r1; dst[2] = r2; }
        }
    }
}

}  // namespace allegro
