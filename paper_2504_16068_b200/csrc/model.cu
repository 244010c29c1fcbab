// model.cu -- dtype-only pieces of the two-layer model of BASELINE.json:configs[2] (reading A19) that are not part
// of the tensor-product hot path: the per-edge linear maps (w = W_w x and its transpose), the scalar latent update
// x' = u(r/r_c) SiLU(A [x ; V[:,0e]]) with its VJP, and an in-place add.  Small-K GEMMs ([E x 64] x [64 x 64..128]) in the
// method's own precision (fp32 / fp64 FMA): register-tiled, both operands K-major in shared memory.
#include "common.cuh"
#include "launch.h"

namespace allegro {

// ---------------------------------------------------------------------------------------------- register-tiled small GEMM
// All three maps are [E x K] . [K x n_out] products with K, n_out in {64, 128}: HBM-light, FMA-heavy.  One CTA (256 threads) owns
// a tile of TILE_E = 128 edges and walks the outputs in chunks of 64; thread (ty, tx) = (tid / 16, tid % 16) accumulates 8 edges
// (8 ty .. 8 ty + 7) x 4 outputs (4 tx .. 4 tx + 3) in registers.  Both operands sit in shared memory K-major -- xs[k][128 edges],
// Ws[k][64 outputs] -- so one k step is two 128-bit loads of x (a broadcast inside each half-warp), one of W and 32 FMAs.
constexpr int kTileE = 128, kTileO = 64;

template <typename T>
__device__ __forceinline__ void tile_mac(const T* __restrict__ xs, const T* __restrict__ Ws, int K, int ty, int tx, T (&acc)[8][4]) {
#pragma unroll 4
    for (int k = 0; k < K; ++k) {
        T xv[8], wv[4];
#pragma unroll
        for (int i = 0; i < 8; ++i) xv[i] = xs[k * kTileE + 8 * ty + i];
#pragma unroll
        for (int j = 0; j < 4; ++j) wv[j] = Ws[k * kTileO + 4 * tx + j];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j] = fma(xv[i], wv[j], acc[i][j]);
    }
}
// Ws[k][o] = W[o0 + o][k] (transpose_w == 0, W [n_out][ldw = K]) or W[k][o0 + o] (transpose_w == 1, W [K][ldw = n_out]); columns beyond
// n_out are zero
template <typename T>
__device__ __forceinline__ void tile_load_w(T* __restrict__ Ws, const T* __restrict__ W, int K, int n_out, int o0, int transpose_w, int tid) {
    for (int idx = tid; idx < K * kTileO; idx += 256) {
        int k, o;
        if (transpose_w) { k = idx / kTileO; o = idx - k * kTileO; } else { o = idx / K; k = idx - o * K; }
        const int og = o0 + o;
        Ws[k * kTileO + o] = og < n_out ? (transpose_w ? W[(size_t)k * n_out + og] : W[(size_t)og * K + k]) : T(0);
    }
}
// xs[k][le] = x[eb + le][k] for k < K (rows beyond E are zero): lanes run over edges, so the shared-memory writes are conflict-free
template <typename T>
__device__ __forceinline__ void tile_load_x(T* __restrict__ xs, const T* __restrict__ x, long E, long eb, int K, int k0, int ldx, int kstride, int tid) {
    for (int idx = tid; idx < K * kTileE; idx += 256) {
        const int k = idx / kTileE, le = idx - k * kTileE;
        xs[(k0 + k) * kTileE + le] = eb + le < E ? x[(size_t)(eb + le) * ldx + (size_t)k * kstride] : T(0);
    }
}

// y[e][o] (+)= sum_i x[e][i] Wm[o][i]            (transpose_w == 0, Wm = W [n_out][n_in])
// y[e][o] (+)= sum_i x[e][i] W[i][o]             (transpose_w == 1, W [n_in][n_out]: the VJP of the map above)
template <typename T>
__global__ void __launch_bounds__(256) linear_kernel(long E, int n_out, int n_in, const T* __restrict__ x, const T* __restrict__ W, int transpose_w,
                                                      int accumulate, T* __restrict__ y) {
    extern __shared__ __align__(16) unsigned char lin_raw[];
    T* xs = reinterpret_cast<T*>(lin_raw);            // [n_in][128]
    T* Ws = xs + (size_t)n_in * kTileE;               // [n_in][64]
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
    const int nchunk = (n_out + kTileO - 1) / kTileO;
    for (long eb = (long)blockIdx.x * kTileE; eb < E; eb += (long)gridDim.x * kTileE) {
        __syncthreads();
        tile_load_x<T>(xs, x, E, eb, n_in, 0, n_in, 1, tid);
        for (int c = 0; c < nchunk; ++c) {
            if (c > 0 || nchunk > 1 || eb == (long)blockIdx.x * kTileE) {   // one output chunk: W stays resident over the tiles
                __syncthreads();
                tile_load_w<T>(Ws, W, n_in, n_out, c * kTileO, transpose_w, tid);
            }
            __syncthreads();
            T acc[8][4];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = T(0);
            tile_mac<T>(xs, Ws, n_in, ty, tx, acc);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const long e = eb + 8 * ty + i;
                if (e >= E) continue;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int o = c * kTileO + 4 * tx + j;
                    if (o < n_out) {
                        T* dst = y + (size_t)e * n_out + o;
                        *dst = accumulate ? *dst + acc[i][j] : acc[i][j];
                    }
                }
            }
        }
    }
}

template <typename T>
__device__ __forceinline__ T cutoff_u(T xr, T& du) {  // u(x) = 1 - 28x^6 + 48x^7 - 21x^8 and du/dx (reading A8)
    const T x2 = xr * xr, x5 = x2 * x2 * xr, x6 = x5 * xr, x7 = x6 * xr, x8 = x7 * xr;
    du = T(-168) * x5 + T(336) * x6 - T(168) * x7;
    T u = T(1) - T(28) * x6 + T(48) * x7 - T(21) * x8;
    if (xr >= T(1)) { u = T(0); du = T(0); }
    return u;
}

// z[e][o] = sum_i A[o][i] x[e][i] + sum_i A[o][n+i] V[e][i][0];  x_new = u(|r_e|/r_c) SiLU(z)
template <typename T>
__global__ void __launch_bounds__(256) latent_fwd_kernel(long E, int n, int dV, T rc, const T* __restrict__ rvec, const T* __restrict__ x,
                                                          const T* __restrict__ V, const T* __restrict__ A, T* __restrict__ z, T* __restrict__ x_new) {
    extern __shared__ __align__(16) unsigned char lin_raw[];
    const int K = 2 * n;
    T* xs = reinterpret_cast<T*>(lin_raw);            // [2n][128]: rows 0..n-1 = x, rows n..2n-1 = V[:, :, 0]
    T* Ws = xs + (size_t)K * kTileE;                  // [2n][64]
    T* us = Ws + (size_t)K * kTileO;                  // [128] cutoff u(|r|/rc)
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
    const int nchunk = (n + kTileO - 1) / kTileO;
    for (long eb = (long)blockIdx.x * kTileE; eb < E; eb += (long)gridDim.x * kTileE) {
        __syncthreads();
        tile_load_x<T>(xs, x, E, eb, n, 0, n, 1, tid);
        tile_load_x<T>(xs, V, E, eb, n, n, n * dV, dV, tid);   // V[e][k][0]
        if (tid < kTileE) {
            const long e = eb + tid;
            T du, u = T(0);
            if (e < E) {
                const T rx = rvec[3 * e], ry = rvec[3 * e + 1], rz = rvec[3 * e + 2];
                u = cutoff_u<T>(sqrt(rx * rx + ry * ry + rz * rz) / rc, du);
            }
            us[tid] = u;
        }
        for (int c = 0; c < nchunk; ++c) {
            if (c > 0 || nchunk > 1 || eb == (long)blockIdx.x * kTileE) {
                __syncthreads();
                tile_load_w<T>(Ws, A, K, n, c * kTileO, 0, tid);
            }
            __syncthreads();
            T acc[8][4];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = T(0);
            tile_mac<T>(xs, Ws, K, ty, tx, acc);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const long e = eb + 8 * ty + i;
                if (e >= E) continue;
                const T u = us[8 * ty + i];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int o = c * kTileO + 4 * tx + j;
                    if (o < n) {
                        const T a = acc[i][j];
                        const T sg = T(1) / (T(1) + exp(-a));
                        z[(size_t)e * n + o] = a;
                        x_new[(size_t)e * n + o] = u * a * sg;
                    }
                }
            }
        }
    }
}
// VJP: g_z = g_xnew u SiLU'(z);  g_x[e][i] = sum_o g_z[o] A[o][i] (overwritten);  gV[e][i][0] += sum_o g_z[o] A[o][n+i];
//      g_rvec[e] += (sum_o g_xnew[o] SiLU(z[o])) u'(x)/r_c rhat_e
template <typename T>
__global__ void __launch_bounds__(256) latent_bwd_kernel(long E, int n, int dV, T rc, const T* __restrict__ rvec, const T* __restrict__ z,
                                                          const T* __restrict__ g_xnew, const T* __restrict__ A, T* __restrict__ g_x,
                                                          T* __restrict__ gV, T* __restrict__ g_rvec) {
    extern __shared__ __align__(16) unsigned char lin_raw[];
    T* xs = reinterpret_cast<T*>(lin_raw);            // [n][128]: g_z, K-major (K = the n outputs of the forward map)
    T* Ws = xs + (size_t)n * kTileE;                  // [n][64]: A[o][chunk of the 2n inputs]
    T* us = Ws + (size_t)n * kTileO;                  // [128] u, [128] u'/rc/|r|, [2][128] partial radial sums
    T* dus = us + kTileE;
    T* rs = dus + kTileE;
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
    const int nchunk = (2 * n + kTileO - 1) / kTileO;
    for (long eb = (long)blockIdx.x * kTileE; eb < E; eb += (long)gridDim.x * kTileE) {
        __syncthreads();
        if (tid < kTileE) {
            const long e = eb + tid;
            T u = T(0), du = T(0), r = T(1);
            if (e < E) {
                const T rx = rvec[3 * e], ry = rvec[3 * e + 1], rz = rvec[3 * e + 2];
                r = sqrt(rx * rx + ry * ry + rz * rz);
                u = cutoff_u<T>(r / rc, du);
            }
            us[tid] = u;
            dus[tid] = du / rc / r;
        }
        __syncthreads();
        {   // g_z = g_xnew u SiLU'(z) -> xs[o][le]; this thread's edge le = tid % 128 is the same in every iteration
            const int le = tid & (kTileE - 1);
            const long e = eb + le;
            T part = T(0);
            for (int o = tid >> 7; o < n; o += 2) {
                T gzv = T(0);
                if (e < E) {
                    const T zz = z[(size_t)e * n + o], g = g_xnew[(size_t)e * n + o];
                    const T sg = T(1) / (T(1) + exp(-zz));
                    gzv = g * us[le] * (sg * (T(1) + zz * (T(1) - sg)));
                    part += g * zz * sg;
                }
                xs[o * kTileE + le] = gzv;
            }
            rs[(tid >> 7) * kTileE + le] = part;
        }
        for (int c = 0; c < nchunk; ++c) {
            __syncthreads();
            tile_load_w<T>(Ws, A, n, 2 * n, c * kTileO, 1, tid);
            __syncthreads();
            T acc[8][4];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = T(0);
            tile_mac<T>(xs, Ws, n, ty, tx, acc);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const long e = eb + 8 * ty + i;
                if (e >= E) continue;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int o = c * kTileO + 4 * tx + j;
                    if (o < n) g_x[(size_t)e * n + o] = acc[i][j];
                    else if (o < 2 * n) gV[((size_t)e * n + (o - n)) * dV] += acc[i][j];
                }
            }
        }
        if (tid < kTileE && eb + tid < E) {   // radial term: rs was written before the first barrier of the chunk loop
            const long e = eb + tid;
            const T sc = (rs[tid] + rs[kTileE + tid]) * dus[tid];
            g_rvec[3 * e] += sc * rvec[3 * e];
            g_rvec[3 * e + 1] += sc * rvec[3 * e + 1];
            g_rvec[3 * e + 2] += sc * rvec[3 * e + 2];
        }
    }
}

template <typename T>
__global__ void add_inplace_kernel(long count, T* __restrict__ y, const T* __restrict__ x) {
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (long)gridDim.x * blockDim.x) y[i] += x[i];
}

// ------------------------------------------------------------------------------------------------ launchers
static inline unsigned model_grid(long E) {
    const long want = (E + kTileE - 1) / kTileE;
    return (unsigned)(want < 148 * 2 ? (want < 1 ? 1 : want) : 148 * 2);
}

template <typename T>
allegro_status_t launch_linear(long E, int n_out, int n_in, const void* x, const void* W, int transpose_w, int accumulate, void* y, cudaStream_t st) {
    if (n_out > 1024 || n_in > 256) { set_error("linear: n_out = %d, n_in = %d unsupported (<= 1024, <= 256)", n_out, n_in); return ALLEGRO_EUNSUPPORTED; }
    if (E == 0) return ALLEGRO_OK;
    const size_t smem = (size_t)n_in * (kTileE + kTileO) * sizeof(T);
    ALLEGRO_CUDA(cudaFuncSetAttribute(linear_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    linear_kernel<T><<<model_grid(E), 256, smem, st>>>(E, n_out, n_in, (const T*)x, (const T*)W, transpose_w, accumulate, (T*)y);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
template <typename T>
allegro_status_t launch_latent_forward(long E, int n, int dV, double rc, const void* rvec, const void* x, const void* V, const void* A, void* z,
                                       void* x_new, cudaStream_t st) {
    if (n > 128 || n < 1) { set_error("latent_forward: n = %d unsupported (1 <= n <= 128)", n); return ALLEGRO_EUNSUPPORTED; }
    if (E == 0) return ALLEGRO_OK;
    const size_t smem = ((size_t)2 * n * (kTileE + kTileO) + kTileE) * sizeof(T);
    ALLEGRO_CUDA(cudaFuncSetAttribute(latent_fwd_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    latent_fwd_kernel<T><<<model_grid(E), 256, smem, st>>>(E, n, dV, (T)rc, (const T*)rvec, (const T*)x, (const T*)V, (const T*)A, (T*)z, (T*)x_new);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
template <typename T>
allegro_status_t launch_latent_backward(long E, int n, int dV, double rc, const void* rvec, const void* z, const void* g_xnew, const void* A,
                                        void* g_x, void* gV, void* g_rvec, cudaStream_t st) {
    if (n > 256 || n < 1) { set_error("latent_backward: n = %d unsupported (1 <= n <= 256)", n); return ALLEGRO_EUNSUPPORTED; }
    if (E == 0) return ALLEGRO_OK;
    const size_t smem = ((size_t)n * (kTileE + kTileO) + 4 * kTileE) * sizeof(T);
    ALLEGRO_CUDA(cudaFuncSetAttribute(latent_bwd_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    latent_bwd_kernel<T><<<model_grid(E), 256, smem, st>>>(E, n, dV, (T)rc, (const T*)rvec, (const T*)z, (const T*)g_xnew, (const T*)A, (T*)g_x,
                                                          (T*)gV, (T*)g_rvec);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
template <typename T>
allegro_status_t launch_add_inplace(long count, void* y, const void* x, cudaStream_t st) {
    if (count == 0) return ALLEGRO_OK;
    add_inplace_kernel<T><<<(unsigned)((count + 255) / 256 < 148 * 16 ? (count + 255) / 256 : 148 * 16), 256, 0, st>>>(count, (T*)y, (const T*)x);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

#define ALLEGRO_INST_MODEL(T)                                                                                                         \
    template allegro_status_t launch_linear<T>(long, int, int, const void*, const void*, int, int, void*, cudaStream_t);               \
    template allegro_status_t launch_latent_forward<T>(long, int, int, double, const void*, const void*, const void*, const void*, void*, void*, cudaStream_t); \
    template allegro_status_t launch_latent_backward<T>(long, int, int, double, const void*, const void*, const void*, const void*, void*, void*, void*, cudaStream_t); \
    template allegro_status_t launch_add_inplace<T>(long, void*, const void*, cudaStream_t);
ALLEGRO_INST_MODEL(float)
ALLEGRO_INST_MODEL(double)

}  // namespace allegro
