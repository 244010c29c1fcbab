// model.cu -- dtype-only pieces of the two-layer model of BASELINE.json:configs[2] (reading A19) that are not part
// of the tensor-product hot path: the per-edge linear maps (w = W_w x and its transpose), the scalar latent update
// x' = u(r/r_c) SiLU(A [x ; V[:,0e]]) with its VJP, and an in-place add.  Small-K GEMMs ([E x 64] x [64 x 64..128]):
// the weight matrix sits in shared memory (row stride +1: conflict-free), one thread per output element.
#include "common.cuh"
#include "launch.h"

namespace allegro {

// y[e][o] (+)= sum_i x[e][i] Wm[o][i]            (transpose_w == 0, Wm = W [n_out][n_in])
// y[e][o] (+)= sum_i x[e][i] W[i][o]             (transpose_w == 1, W [n_in][n_out]: the VJP of the map above)
template <typename T>
__global__ void __launch_bounds__(256) linear_kernel(long E, int n_out, int n_in, const T* __restrict__ x, const T* __restrict__ W, int transpose_w,
                                                      int accumulate, T* __restrict__ y) {
    extern __shared__ __align__(16) unsigned char lin_raw[];
    T* Ws = reinterpret_cast<T*>(lin_raw);                 // [n_out][n_in + 1]
    const int ld = n_in + 1;
    T* xs = Ws + (size_t)n_out * ld;                       // [epb][n_in]
    const int epb = 256 / n_out;                           // edges per pass
    for (int idx = threadIdx.x; idx < n_out * n_in; idx += 256) {
        const int o = idx / n_in, i = idx - o * n_in;
        Ws[o * ld + i] = transpose_w ? W[(size_t)i * n_out + o] : W[idx];
    }
    const int le = threadIdx.x / n_out, o = threadIdx.x - le * n_out;
    for (long eb = (long)blockIdx.x * epb; eb < E; eb += (long)gridDim.x * epb) {
        __syncthreads();
        const int cnt = (int)min((long)epb, E - eb);
        for (int idx = threadIdx.x; idx < cnt * n_in; idx += 256) xs[idx] = x[(size_t)eb * n_in + idx];
        __syncthreads();
        if (le < cnt) {
            T acc = T(0);
            for (int i = 0; i < n_in; ++i) acc = fma(xs[le * n_in + i], Ws[o * ld + i], acc);
            T* dst = y + (size_t)(eb + le) * n_out + o;
            *dst = accumulate ? *dst + acc : acc;
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
    const int K = 2 * n, ld = K + 1;
    T* As = reinterpret_cast<T*>(lin_raw);  // [n][2n + 1]
    T* in = As + (size_t)n * ld;            // [epb][2n]
    const int epb = 256 / n;
    for (int idx = threadIdx.x; idx < n * K; idx += 256) As[(idx / K) * ld + (idx % K)] = A[idx];
    const int le = threadIdx.x / n, o = threadIdx.x - le * n;
    for (long eb = (long)blockIdx.x * epb; eb < E; eb += (long)gridDim.x * epb) {
        __syncthreads();
        const int cnt = (int)min((long)epb, E - eb);
        for (int idx = threadIdx.x; idx < cnt * n; idx += 256) {
            const int l2 = idx / n, i = idx - l2 * n;
            in[l2 * K + i] = x[(size_t)(eb + l2) * n + i];
            in[l2 * K + n + i] = V[((size_t)(eb + l2) * n + i) * dV];
        }
        __syncthreads();
        if (le < cnt) {
            const size_t e = (size_t)(eb + le);
            T acc = T(0);
            for (int i = 0; i < K; ++i) acc = fma(in[le * K + i], As[o * ld + i], acc);
            const T rx = rvec[3 * e], ry = rvec[3 * e + 1], rz = rvec[3 * e + 2];
            T du;
            const T u = cutoff_u<T>(sqrt(rx * rx + ry * ry + rz * rz) / rc, du);
            const T sg = T(1) / (T(1) + exp(-acc));
            z[e * n + o] = acc;
            x_new[e * n + o] = u * acc * sg;
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
    const int K = 2 * n;
    T* As = reinterpret_cast<T*>(lin_raw);  // [n][2n] (read along o for fixed i: consecutive threads i -> consecutive banks)
    T* gz = As + (size_t)n * K;             // [epb][n]
    T* rs = gz + 256;                       // [epb][n] g_xnew * SiLU(z) for the radial term
    const int epb = 256 / n;
    for (int idx = threadIdx.x; idx < n * K; idx += 256) As[idx] = A[idx];
    const int le = threadIdx.x / n, i = threadIdx.x - le * n;
    for (long eb = (long)blockIdx.x * epb; eb < E; eb += (long)gridDim.x * epb) {
        __syncthreads();
        const int cnt = (int)min((long)epb, E - eb);
        T u = T(0), du = T(0), rx = T(0), ry = T(0), rz = T(0), r = T(1);
        if (le < cnt) {
            const size_t e = (size_t)(eb + le);
            rx = rvec[3 * e]; ry = rvec[3 * e + 1]; rz = rvec[3 * e + 2];
            r = sqrt(rx * rx + ry * ry + rz * rz);
            u = cutoff_u<T>(r / rc, du);
            const T zz = z[e * n + i], g = g_xnew[e * n + i];
            const T sg = T(1) / (T(1) + exp(-zz));
            gz[le * n + i] = g * u * (sg * (T(1) + zz * (T(1) - sg)));
            rs[le * n + i] = g * zz * sg;
        }
        __syncthreads();
        if (le < cnt) {
            const size_t e = (size_t)(eb + le);
            T a0 = T(0), a1 = T(0);
            for (int o = 0; o < n; ++o) {
                const T g = gz[le * n + o];
                a0 = fma(g, As[o * K + i], a0);
                a1 = fma(g, As[o * K + n + i], a1);
            }
            g_x[e * n + i] = a0;
            gV[(e * n + i) * dV] += a1;
            if (i < 3) {
                T s = T(0);
                for (int o = 0; o < n; ++o) s += rs[le * n + o];
                const T comp = i == 0 ? rx : (i == 1 ? ry : rz);
                g_rvec[3 * e + i] += s * du / rc * comp / r;
            }
        }
    }
}

template <typename T>
__global__ void add_inplace_kernel(long count, T* __restrict__ y, const T* __restrict__ x) {
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (long)gridDim.x * blockDim.x) y[i] += x[i];
}

// ------------------------------------------------------------------------------------------------ launchers
static inline unsigned model_grid(long E, int epb) {
    const long want = (E + epb - 1) / epb;
    return (unsigned)(want < 148 * 8 ? (want < 1 ? 1 : want) : 148 * 8);
}

template <typename T>
allegro_status_t launch_linear(long E, int n_out, int n_in, const void* x, const void* W, int transpose_w, int accumulate, void* y, cudaStream_t st) {
    if (n_out > 256 || n_in > 512) { set_error("linear: n_out = %d, n_in = %d unsupported (<= 256, <= 512)", n_out, n_in); return ALLEGRO_EUNSUPPORTED; }
    if (E == 0) return ALLEGRO_OK;
    const int epb = 256 / n_out;
    const size_t smem = ((size_t)n_out * (n_in + 1) + (size_t)epb * n_in) * sizeof(T);
    ALLEGRO_CUDA(cudaFuncSetAttribute(linear_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    linear_kernel<T><<<model_grid(E, epb), 256, smem, st>>>(E, n_out, n_in, (const T*)x, (const T*)W, transpose_w, accumulate, (T*)y);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
template <typename T>
allegro_status_t launch_latent_forward(long E, int n, int dV, double rc, const void* rvec, const void* x, const void* V, const void* A, void* z,
                                       void* x_new, cudaStream_t st) {
    if (n > 128 || n < 3) { set_error("latent_forward: n = %d unsupported (3 <= n <= 128)", n); return ALLEGRO_EUNSUPPORTED; }
    if (E == 0) return ALLEGRO_OK;
    const int epb = 256 / n;
    const size_t smem = ((size_t)n * (2 * n + 1) + (size_t)epb * 2 * n) * sizeof(T);
    ALLEGRO_CUDA(cudaFuncSetAttribute(latent_fwd_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    latent_fwd_kernel<T><<<model_grid(E, epb), 256, smem, st>>>(E, n, dV, (T)rc, (const T*)rvec, (const T*)x, (const T*)V, (const T*)A, (T*)z, (T*)x_new);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
template <typename T>
allegro_status_t launch_latent_backward(long E, int n, int dV, double rc, const void* rvec, const void* z, const void* g_xnew, const void* A,
                                        void* g_x, void* gV, void* g_rvec, cudaStream_t st) {
    if (n > 128 || n < 3) { set_error("latent_backward: n = %d unsupported (3 <= n <= 128)", n); return ALLEGRO_EUNSUPPORTED; }
    if (E == 0) return ALLEGRO_OK;
    const int epb = 256 / n;
    const size_t smem = ((size_t)n * 2 * n + 512) * sizeof(T);
    ALLEGRO_CUDA(cudaFuncSetAttribute(latent_bwd_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    latent_bwd_kernel<T><<<model_grid(E, epb), 256, smem, st>>>(E, n, dV, (T)rc, (const T*)rvec, (const T*)z, (const T*)g_xnew, (const T*)A, (T*)g_x,
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
