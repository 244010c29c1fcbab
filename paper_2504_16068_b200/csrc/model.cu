// model.cu -- dtype-only pieces of the two-layer model of BASELINE.json:configs[2] (reading A19) that are not part
// of the tensor-product hot path: the per-edge linear maps (w = W_w x and its transpose), the scalar latent update
// x' = u(r/r_c) SiLU(A [x ; V[:,0e]]) with its VJP, and an in-place add.  Small-K GEMMs ([E x 64] x [64 x 64..128]) in the
// method's own precision (fp32 / fp64 FMA): register-tiled, operands in shared memory.
#include <initializer_list>

#include "common.cuh"
#include "launch.h"

namespace allegro {

// ---------------------------------------------------------------------------------------------- register-tiled small GEMM
// All three maps are [E x K] . [K x n_out] products with K, n_out in {64, 128}: HBM-light, FMA-heavy.  One CTA (256 threads) owns
// a tile of kTileE = 128 edges and walks the outputs in chunks of 64; thread (ty, tx) = (tid / 16, tid % 16) accumulates 8 edges
// (ty + 16 i) x 4 outputs (4 tx .. 4 tx + 3) in registers.  The x tile sits in shared memory ROW-major, xs[edge][Kp + VEC] (Kp = K
// rounded up to the 16-byte vector width VEC, the pad columns zero): global rows are read with lanes running along K (fully
// coalesced, conflict-free stores), and the multiply loop reads one 16-byte vector of VEC consecutive k per edge -- the two
// edges of a warp are adjacent rows, Kp + VEC words apart, so their vectors fall into different banks, and the 16 tx lanes
// share the address (broadcast).  W sits K-major, Ws[k][64 outputs].  One step of VEC k's: 8 + VEC vector loads, 32 VEC FMAs.
constexpr int kTileE = 128, kTileO = 64;

template <typename T> struct TileVec { static constexpr int N = 16 / (int)sizeof(T); };
__host__ __device__ static inline int tile_kp(int K, int vec) { return (K + vec - 1) / vec * vec; }

template <typename T>
__device__ __forceinline__ void tile_mac(const T* __restrict__ xs, const T* __restrict__ Ws, int Kp, int ty, int tx, T (&acc)[8][4]) {
    constexpr int VEC = TileVec<T>::N;
    constexpr int WV = 4 / VEC;                       // 16-byte vectors per 4 outputs: 1 (float) or 2 (double)
    const int ld = Kp + VEC;
    for (int k = 0; k < Kp; k += VEC) {
        T xv[8][VEC], wv[VEC][4];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int4 v = *reinterpret_cast<const int4*>(xs + (size_t)(ty + 16 * i) * ld + k);
            const T* sv = reinterpret_cast<const T*>(&v);
#pragma unroll
            for (int q = 0; q < VEC; ++q) xv[i][q] = sv[q];
        }
#pragma unroll
        for (int q = 0; q < VEC; ++q) {
            const T* wrow = Ws + (size_t)(k + q) * kTileO + 4 * tx;
#pragma unroll
            for (int h = 0; h < WV; ++h) {
                const int4 v = *reinterpret_cast<const int4*>(wrow + h * VEC);
                const T* sv = reinterpret_cast<const T*>(&v);
#pragma unroll
                for (int jj = 0; jj < VEC; ++jj) wv[q][h * VEC + jj] = sv[jj];
            }
        }
#pragma unroll
        for (int q = 0; q < VEC; ++q)
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int jj = 0; jj < 4; ++jj) acc[i][jj] = fma(xv[i][q], wv[q][jj], acc[i][jj]);
    }
}
// Ws[k][o] = W[o0 + o][k] (transpose_w == 0, W [n_out][K]) or W[k][o0 + o] (transpose_w == 1, W [K][n_out]); rows k >= K and columns
// beyond n_out are zero
template <typename T>
__device__ __forceinline__ void tile_load_w(T* __restrict__ Ws, const T* __restrict__ W, int K, int Kp, int n_out, int o0, int transpose_w, int tid) {
    for (int idx = tid; idx < Kp * kTileO; idx += 256) {
        int k, o;
        if (transpose_w) { k = idx / kTileO; o = idx - k * kTileO; } else { o = idx / Kp; k = idx - o * Kp; }
        const int og = o0 + o;
        Ws[k * kTileO + o] = (og < n_out && k < K) ? (transpose_w ? W[(size_t)k * n_out + og] : W[(size_t)og * K + k]) : T(0);
    }
}
// xs[le][k0 + k] = x[(eb + le) * ldx + k * kstride] for k < K (rows beyond E are zero): lanes run along k
template <typename T>
__device__ __forceinline__ void tile_load_x(T* __restrict__ xs, int ld, const T* __restrict__ x, long E, long eb, int K, int k0, size_t ldx, int kstride,
                                            int tid) {
    for (int idx = tid; idx < K * kTileE; idx += 256) {
        const int le = idx / K, k = idx - le * K;
        xs[(size_t)le * ld + k0 + k] = eb + le < E ? x[(size_t)(eb + le) * ldx + (size_t)k * kstride] : T(0);
    }
}
// store 4 consecutive outputs of one edge: one 16-byte vector when the row allows it (float, n_out % 4 == 0), else scalars
template <typename T>
__device__ __forceinline__ void tile_store4(T* __restrict__ dst, const T (&v)[4], int o, int n_out, bool vec) {
    if (vec) {
        if constexpr (sizeof(T) == 4) {
            *reinterpret_cast<float4*>(dst) = make_float4(v[0], v[1], v[2], v[3]);
        } else {
            *reinterpret_cast<double2*>(dst) = make_double2(v[0], v[1]);
            *reinterpret_cast<double2*>(dst + 2) = make_double2(v[2], v[3]);
        }
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) if (o + j < n_out) dst[j] = v[j];
    }
}
// zero the pad columns [K, ld) of every row (once per CTA: the tile loads never touch them)
template <typename T>
__device__ __forceinline__ void tile_zero_pad(T* __restrict__ xs, int ld, int K, int tid) {
    const int w = ld - K;
    for (int idx = tid; idx < w * kTileE; idx += 256) xs[(size_t)(idx / w) * ld + K + idx % w] = T(0);
}

// y[e][o] (+)= sum_i x[e][i] Wm[o][i]            (transpose_w == 0, Wm = W [n_out][n_in])
// y[e][o] (+)= sum_i x[e][i] W[i][o]             (transpose_w == 1, W [n_in][n_out]: the VJP of the map above)
template <typename T>
__global__ void __launch_bounds__(256) linear_kernel(long E, int n_out, int n_in, const T* __restrict__ x, const T* __restrict__ W, int transpose_w,
                                                      int accumulate, T* __restrict__ y) {
    constexpr int VEC = TileVec<T>::N;
    extern __shared__ __align__(16) unsigned char lin_raw[];
    const int Kp = tile_kp(n_in, VEC), ld = Kp + VEC;
    T* xs = reinterpret_cast<T*>(lin_raw);            // [128][ld]
    T* Ws = xs + (size_t)kTileE * ld;                 // [Kp][64]
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
    const int nchunk = (n_out + kTileO - 1) / kTileO;
    const bool vec_out = n_out % 4 == 0 && (reinterpret_cast<uintptr_t>(y) & 15u) == 0;
    tile_zero_pad<T>(xs, ld, n_in, tid);
    for (long eb = (long)blockIdx.x * kTileE; eb < E; eb += (long)gridDim.x * kTileE) {
        __syncthreads();
        tile_load_x<T>(xs, ld, x, E, eb, n_in, 0, (size_t)n_in, 1, tid);
        for (int c = 0; c < nchunk; ++c) {
            if (c > 0 || nchunk > 1 || eb == (long)blockIdx.x * kTileE) {   // one output chunk: W stays resident over the tiles
                __syncthreads();
                tile_load_w<T>(Ws, W, n_in, Kp, n_out, c * kTileO, transpose_w, tid);
            }
            __syncthreads();
            T acc[8][4];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = T(0);
            tile_mac<T>(xs, Ws, Kp, ty, tx, acc);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const long e = eb + ty + 16 * i;
                const int o = c * kTileO + 4 * tx;
                if (e >= E || o >= n_out) continue;
                T* dst = y + (size_t)e * n_out + o;
                if (accumulate) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) if (o + j < n_out) acc[i][j] += dst[j];
                }
                tile_store4<T>(dst, acc[i], o, n_out, vec_out);
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
    constexpr int VEC = TileVec<T>::N;
    const int K = 2 * n, Kp = tile_kp(K, VEC), ld = Kp + VEC;
    T* xs = reinterpret_cast<T*>(lin_raw);            // [128][ld]: columns 0..n-1 = x, n..2n-1 = V[:, :, 0]
    T* Ws = xs + (size_t)kTileE * ld;                 // [Kp][64]
    T* us = Ws + (size_t)Kp * kTileO;                 // [128] cutoff u(|r|/rc)
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
    const int nchunk = (n + kTileO - 1) / kTileO;
    const bool vec_out = n % 4 == 0 && ((reinterpret_cast<uintptr_t>(z) | reinterpret_cast<uintptr_t>(x_new)) & 15u) == 0;
    tile_zero_pad<T>(xs, ld, K, tid);
    for (long eb = (long)blockIdx.x * kTileE; eb < E; eb += (long)gridDim.x * kTileE) {
        __syncthreads();
        tile_load_x<T>(xs, ld, x, E, eb, n, 0, (size_t)n, 1, tid);
        tile_load_x<T>(xs, ld, V, E, eb, n, n, (size_t)n * dV, dV, tid);   // V[e][k][0]
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
                tile_load_w<T>(Ws, A, K, Kp, n, c * kTileO, 0, tid);
            }
            __syncthreads();
            T acc[8][4];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = T(0);
            tile_mac<T>(xs, Ws, Kp, ty, tx, acc);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const long e = eb + ty + 16 * i;
                if (e >= E) continue;
                const T u = us[ty + 16 * i];
                const int o = c * kTileO + 4 * tx;
                if (o >= n) continue;
                T xn[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const T a = acc[i][j];
                    xn[j] = u * a * (T(1) / (T(1) + exp(-a)));
                }
                tile_store4<T>(z + (size_t)e * n + o, acc[i], o, n, vec_out);
                tile_store4<T>(x_new + (size_t)e * n + o, xn, o, n, vec_out);
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
    constexpr int VEC = TileVec<T>::N;
    const int Kp = tile_kp(n, VEC), ld = Kp + VEC, ld2 = n + 1;
    T* xs = reinterpret_cast<T*>(lin_raw);            // [128][ld]: g_z, row-major (K = the n outputs of the forward map)
    T* Ws = xs + (size_t)kTileE * ld;                 // [Kp][64]: A[o][chunk of the 2n inputs]
    T* ss = Ws + (size_t)Kp * kTileO;                 // [128][n + 1]: g_xnew SiLU(z), summed over o per edge for the radial term
    T* us = ss + (size_t)kTileE * ld2;                // [128] u, [128] u'/rc/|r|
    T* dus = us + kTileE;
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
    const int nchunk = (2 * n + kTileO - 1) / kTileO;
    const bool vec_out = n % 4 == 0 && ((reinterpret_cast<uintptr_t>(g_x) | reinterpret_cast<uintptr_t>(gV)) & 15u) == 0;
    tile_zero_pad<T>(xs, ld, n, tid);
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
        // g_z = g_xnew u SiLU'(z) -> xs[le][o], g_xnew SiLU(z) -> ss[le][o]; lanes run along o (coalesced)
        for (int idx = tid; idx < n * kTileE; idx += 256) {
            const int le = idx / n, o = idx - le * n;
            const long e = eb + le;
            T gzv = T(0), sv = T(0);
            if (e < E) {
                const T zz = z[(size_t)e * n + o], g = g_xnew[(size_t)e * n + o];
                const T sg = T(1) / (T(1) + exp(-zz));
                gzv = g * us[le] * (sg * (T(1) + zz * (T(1) - sg)));
                sv = g * zz * sg;
            }
            xs[(size_t)le * ld + o] = gzv;
            ss[(size_t)le * ld2 + o] = sv;
        }
        for (int c = 0; c < nchunk; ++c) {
            __syncthreads();
            tile_load_w<T>(Ws, A, n, Kp, 2 * n, c * kTileO, 1, tid);
            __syncthreads();
            T acc[8][4];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = T(0);
            tile_mac<T>(xs, Ws, Kp, ty, tx, acc);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const long e = eb + ty + 16 * i;
                if (e >= E) continue;
                const int o0 = c * kTileO + 4 * tx;
                if (vec_out && o0 + 3 < n) {
                    tile_store4<T>(g_x + (size_t)e * n + o0, acc[i], o0, n, true);
                } else if (vec_out && dV == 1 && o0 >= n && o0 + 3 < 2 * n) {      // compact scalar cotangent: contiguous
                    T* dst = gV + (size_t)e * n + (o0 - n);
#pragma unroll
                    for (int j = 0; j < 4; ++j) acc[i][j] += dst[j];
                    tile_store4<T>(dst, acc[i], o0 - n, n, true);
                } else {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int o = o0 + j;
                        if (o < n) g_x[(size_t)e * n + o] = acc[i][j];
                        else if (o < 2 * n) gV[((size_t)e * n + (o - n)) * dV] += acc[i][j];
                    }
                }
            }
        }
        if (tid < kTileE && eb + tid < E) {   // radial term: ss was written before the first barrier of the chunk loop; o in order
            const long e = eb + tid;
            T tot = T(0);
            for (int o = 0; o < n; ++o) tot += ss[(size_t)tid * ld2 + o];
            const T sc = tot * dus[tid];
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

allegro_status_t launch_linear64_tc(long E, const void* x, const void* W, int transpose_w, int accumulate, void* y, cudaStream_t st);

template <typename T>
allegro_status_t launch_linear(long E, int n_out, int n_in, const void* x, const void* W, int transpose_w, int accumulate, void* y, cudaStream_t st) {
    if (n_out > 1024 || n_in > 256) { set_error("linear: n_out = %d, n_in = %d unsupported (<= 1024, <= 256)", n_out, n_in); return ALLEGRO_EUNSUPPORTED; }
    if (E == 0) return ALLEGRO_OK;
    if (sizeof(T) == 4 && n_out == 64 && n_in == 64 && aligned16(x) && aligned16(y)) return launch_linear64_tc(E, x, W, transpose_w, accumulate, y, st);
    const int vec = TileVec<T>::N, Kp = tile_kp(n_in, vec);
    const size_t smem = ((size_t)kTileE * (Kp + vec) + (size_t)Kp * kTileO) * sizeof(T);
    ALLEGRO_CUDA(cudaFuncSetAttribute(linear_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    linear_kernel<T><<<model_grid(E), 256, smem, st>>>(E, n_out, n_in, (const T*)x, (const T*)W, transpose_w, accumulate, (T*)y);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
// tclin.cu: fp32, n = 64, compact scalars (dV == 1), 16-byte aligned rows -- the tcgen05 versions
allegro_status_t launch_latent_forward_tc(long E, double rc, const void* rvec, const void* x, const void* s, const void* A, void* z, void* x_new,
                                          cudaStream_t st);
allegro_status_t launch_latent_backward_tc(long E, double rc, const void* rvec, const void* z, const void* g_xnew, const void* A, void* g_x, void* g_s,
                                           void* g_rvec, cudaStream_t st);
static inline bool tc_shape(size_t elem, int n, int dV, std::initializer_list<const void*> ptrs) {
    if (elem != 4 || n != 64 || dV != 1) return false;
    for (const void* p : ptrs)
        if (!aligned16(p)) return false;
    return true;
}

template <typename T>
allegro_status_t launch_latent_forward(long E, int n, int dV, double rc, const void* rvec, const void* x, const void* V, const void* A, void* z,
                                       void* x_new, cudaStream_t st) {
    if (n > 128 || n < 1) { set_error("latent_forward: n = %d unsupported (1 <= n <= 128)", n); return ALLEGRO_EUNSUPPORTED; }
    if (E == 0) return ALLEGRO_OK;
    if (tc_shape(sizeof(T), n, dV, {x, V, A, z, x_new})) return launch_latent_forward_tc(E, rc, rvec, x, V, A, z, x_new, st);
    const int vec = TileVec<T>::N, Kp = tile_kp(2 * n, vec);
    const size_t smem = ((size_t)kTileE * (Kp + vec) + (size_t)Kp * kTileO + kTileE) * sizeof(T);
    ALLEGRO_CUDA(cudaFuncSetAttribute(latent_fwd_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    latent_fwd_kernel<T><<<model_grid(E), 256, smem, st>>>(E, n, dV, (T)rc, (const T*)rvec, (const T*)x, (const T*)V, (const T*)A, (T*)z, (T*)x_new);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
template <typename T>
allegro_status_t launch_latent_backward(long E, int n, int dV, double rc, const void* rvec, const void* z, const void* g_xnew, const void* A,
                                        void* g_x, void* gV, void* g_rvec, cudaStream_t st) {
    if (n > 128 || n < 1) { set_error("latent_backward: n = %d unsupported (1 <= n <= 128)", n); return ALLEGRO_EUNSUPPORTED; }
    if (E == 0) return ALLEGRO_OK;
    if (tc_shape(sizeof(T), n, dV, {z, g_xnew, A, g_x, gV})) return launch_latent_backward_tc(E, rc, rvec, z, g_xnew, A, g_x, gV, g_rvec, st);
    const int vec = TileVec<T>::N, Kp = tile_kp(n, vec);
    const size_t smem = ((size_t)kTileE * (Kp + vec) + (size_t)Kp * kTileO + (size_t)kTileE * (n + 1) + 2 * kTileE) * sizeof(T);
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
