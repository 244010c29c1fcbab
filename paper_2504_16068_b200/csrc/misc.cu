// misc.cu -- dtype-only helpers of the hot path: radial weights and their chain rule (A8), force
// assembly (a7), the scalar edge energy of the VJP tests / benchmarks (A12) and the segment sum (A20).
#include <cooperative_groups.h>

#include "common.cuh"
#include "launch.h"
#include "radial.cuh"

namespace allegro {

constexpr int kRadEdges = 128;  // edges per CTA

// w[e][ch] = sum_b W_r[ch][b] B_b(r_e) u(r_e/rc).  Phase 1: one thread per edge evaluates the basis into shared
// memory; phase 2: warp <-> edge, lane <-> channels lane, lane+32, ... (CPL per lane) whose W_r rows sit in
// registers as doubles, so a row w[e][:] is written as whole coalesced lines and the inner loop is LDS + DFMA only.
template <typename T, int CPL, int NB>
__global__ void __launch_bounds__(256) radial_fwd_kernel(int n, int nb, double rc, long E, const T* __restrict__ rvec, const T* __restrict__ W_r,
                                                          T* __restrict__ w) {
    __shared__ double Bs[kRadEdges][NB];
    const long eb = (long)blockIdx.x * kRadEdges;
    const int cnt = (int)min((long)kRadEdges, E - eb);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double Wd[CPL][NB];
#pragma unroll
    for (int q = 0; q < CPL; ++q)
#pragma unroll
        for (int b = 0; b < NB; ++b) Wd[q][b] = (lane + 32 * q < n && b < nb) ? (double)W_r[(lane + 32 * q) * nb + b] : 0.0;
    if ((int)threadIdx.x < cnt) {
        const long e = eb + threadIdx.x;
        const double rx = (double)rvec[3 * e], ry = (double)rvec[3 * e + 1], rz = (double)rvec[3 * e + 2];
        double Bu[kMaxBasis];
        radial_basis<false>(sqrt(rx * rx + ry * ry + rz * rz), rc, nb, Bu, nullptr);
#pragma unroll
        for (int b = 0; b < NB; ++b) Bs[threadIdx.x][b] = b < nb ? Bu[b] : 0.0;
    }
    __syncthreads();
    for (int le = warp; le < cnt; le += 8) {
        double Bv[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) Bv[b] = Bs[le][b];
#pragma unroll
        for (int q = 0; q < CPL; ++q) {
            double s = 0.0;
#pragma unroll
            for (int b = 0; b < NB; ++b) s = fma(Wd[q][b], Bv[b], s);
            if (lane + 32 * q < n) w[(size_t)(eb + le) * n + lane + 32 * q] = (T)s;
        }
    }
}

// g_rvec[e] += (sum_ch g_w[e][ch] dw[e][ch]/dr) rhat_e.  Same mapping; the channel sum is lane-local over the lane's
// channels, then a fixed xor tree.
template <typename T, int CPL, int NB>
__global__ void __launch_bounds__(256) radial_bwd_kernel(int n, int nb, double rc, long E, const T* __restrict__ rvec, const T* __restrict__ W_r,
                                                          const T* __restrict__ g_w, T* __restrict__ g_rvec) {
    __shared__ double dBs[kRadEdges][NB];
    __shared__ double rh[kRadEdges][3];
    const long eb = (long)blockIdx.x * kRadEdges;
    const int cnt = (int)min((long)kRadEdges, E - eb);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double Wd[CPL][NB];
#pragma unroll
    for (int q = 0; q < CPL; ++q)
#pragma unroll
        for (int b = 0; b < NB; ++b) Wd[q][b] = (lane + 32 * q < n && b < nb) ? (double)W_r[(lane + 32 * q) * nb + b] : 0.0;
    if ((int)threadIdx.x < cnt) {
        const long e = eb + threadIdx.x;
        const double rx = (double)rvec[3 * e], ry = (double)rvec[3 * e + 1], rz = (double)rvec[3 * e + 2];
        const double r = sqrt(rx * rx + ry * ry + rz * rz);
        double Bu[kMaxBasis], dBu[kMaxBasis];
        radial_basis<true>(r, rc, nb, Bu, dBu);
#pragma unroll
        for (int b = 0; b < NB; ++b) dBs[threadIdx.x][b] = b < nb ? dBu[b] : 0.0;
        rh[threadIdx.x][0] = rx / r; rh[threadIdx.x][1] = ry / r; rh[threadIdx.x][2] = rz / r;
    }
    __syncthreads();
    for (int le = warp; le < cnt; le += 8) {
        const long e = eb + le;
        double Bv[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) Bv[b] = dBs[le][b];
        double acc = 0.0;
#pragma unroll
        for (int q = 0; q < CPL; ++q) {
            double dw = 0.0;
#pragma unroll
            for (int b = 0; b < NB; ++b) dw = fma(Wd[q][b], Bv[b], dw);
            if (lane + 32 * q < n) acc = fma((double)g_w[(size_t)e * n + lane + 32 * q], dw, acc);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (lane < 3) g_rvec[3 * e + lane] = (T)((double)g_rvec[3 * e + lane] + acc * rh[le][lane]);
    }
}

// F[a] = sum_{e in row a} (g_r[e] - g_r[rev[e]]): one warp per atom, lane-strided partial sums in CSR
// order, fixed xor tree (deterministic; no atomics).
template <typename T>
__global__ void __launch_bounds__(256) force_gather_kernel(int n_atoms, const int* __restrict__ row_ptr, const int* __restrict__ rev,
                                                            const T* __restrict__ g_rvec, T* __restrict__ F) {
    const int a = blockIdx.x * 8 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (a >= n_atoms) return;
    T f0 = T(0), f1 = T(0), f2 = T(0);
    for (int e = row_ptr[a] + lane; e < row_ptr[a + 1]; e += 32) {
        const size_t r = (size_t)rev[e];
        f0 += g_rvec[3 * (size_t)e] - g_rvec[3 * r];
        f1 += g_rvec[3 * (size_t)e + 1] - g_rvec[3 * r + 1];
        f2 += g_rvec[3 * (size_t)e + 2] - g_rvec[3 * r + 2];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        f0 += __shfl_xor_sync(0xffffffffu, f0, o);
        f1 += __shfl_xor_sync(0xffffffffu, f1, o);
        f2 += __shfl_xor_sync(0xffffffffu, f2, o);
    }
    if (lane == 0) { F[3 * (size_t)a] = f0; F[3 * (size_t)a + 1] = f1; F[3 * (size_t)a + 2] = f2; }
}

// e_edge[e] = sum_ch ( q[ch] out[e][ch][0] + kappa/2 sum_k out[e][ch][k]^2 ),  G = q (x) delta_{k,0} + kappa out.
// One warp per edge; lanes stride over the n*dV contiguous elements (coalesced), fixed xor tree.
template <typename T>
__global__ void __launch_bounds__(256) edge_energy_kernel(int n, int dV, long E, const T* __restrict__ out, const T* __restrict__ q, T kappa,
                                                           T* __restrict__ e_edge, T* __restrict__ G) {
    const long e = (long)blockIdx.x * 8 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (e >= E) return;
    const int len = n * dV;
    const T* o = out + (size_t)e * len;
    T* g = G ? G + (size_t)e * len : nullptr;
    T acc = T(0);
    if (kappa == T(0) && g == nullptr) {   // pure linear readout of the scalars: only component 0 of every row is touched
        for (int ch = lane; ch < n; ch += 32) acc = fma(q[ch], o[(size_t)ch * dV], acc);
#pragma unroll
        for (int o2 = 16; o2 > 0; o2 >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o2);
        if (lane == 0 && e_edge) e_edge[e] = acc;
        return;
    }
    for (int idx = lane; idx < len; idx += 32) {
        const T v = o[idx];
        const int ch = idx / dV, k = idx - ch * dV;
        T gv = kappa * v;
        acc = fma(T(0.5) * gv, v, acc);
        if (k == 0) { const T qc = q[ch]; acc = fma(qc, v, acc); gv += qc; }
        if (g) g[idx] = gv;
    }
#pragma unroll
    for (int o2 = 16; o2 > 0; o2 >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o2);
    if (lane == 0 && e_edge) e_edge[e] = acc;
}

// out[s] = sum_{i in [ptr[s], ptr[s+1])} vals[i].  One thread-block CLUSTER of kSegCluster CTAs per segment: every
// thread adds a strided subset in double, each CTA folds its threads with a fixed shared-memory tree, and CTA 0 of
// the cluster adds the CTAs' partials in rank order through distributed shared memory (deterministic, no
// workspace, no atomics).
constexpr int kSegThreads = 512;
constexpr int kSegCluster = 8;
template <typename T>
__global__ void __launch_bounds__(kSegThreads) segment_sum_kernel(const int* __restrict__ ptr, int nseg, const T* __restrict__ vals, T* __restrict__ out) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    __shared__ double sh[kSegThreads];
    const int s = blockIdx.x / kSegCluster;
    const int rank = (int)cluster.block_rank();
    const int i0 = ptr[s], i1 = ptr[s + 1];
    constexpr int STRIDE = kSegThreads * kSegCluster;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    int i = i0 + rank * kSegThreads + threadIdx.x;
    for (; i + 3 * STRIDE < i1; i += 4 * STRIDE) {
        a0 += (double)vals[i]; a1 += (double)vals[i + STRIDE]; a2 += (double)vals[i + 2 * STRIDE]; a3 += (double)vals[i + 3 * STRIDE];
    }
    for (; i < i1; i += STRIDE) a0 += (double)vals[i];
    sh[threadIdx.x] = (a0 + a1) + (a2 + a3);
    __syncthreads();
    for (int o = kSegThreads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    cluster.sync();
    if (rank == 0 && threadIdx.x == 0) {
        double tot = sh[0];
        for (int r = 1; r < kSegCluster; ++r) tot += *cluster.map_shared_rank(&sh[0], r);
        out[s] = (T)tot;
    }
    cluster.sync();  // keep every CTA's shared memory alive until CTA 0 has read it
}

// ------------------------------------------------------------------------------------------------ launchers
// (CPL, NB) instantiations: n <= 32 * CPL channels, nb <= NB basis functions
#define ALLEGRO_RAD_DISPATCH(KERNEL, ...)                                                     \
    do {                                                                                      \
        const unsigned grid = (unsigned)((E + kRadEdges - 1) / kRadEdges);                     \
        if (nb <= 8) {                                                                        \
            if (n <= 32) KERNEL<T, 1, 8><<<grid, 256, 0, st>>>(__VA_ARGS__);                   \
            else if (n <= 64) KERNEL<T, 2, 8><<<grid, 256, 0, st>>>(__VA_ARGS__);              \
            else if (n <= 128) KERNEL<T, 4, 8><<<grid, 256, 0, st>>>(__VA_ARGS__);             \
            else KERNEL<T, 8, 8><<<grid, 256, 0, st>>>(__VA_ARGS__);                           \
        } else {                                                                              \
            if (n <= 32) KERNEL<T, 1, 16><<<grid, 256, 0, st>>>(__VA_ARGS__);                  \
            else if (n <= 64) KERNEL<T, 2, 16><<<grid, 256, 0, st>>>(__VA_ARGS__);             \
            else if (n <= 128) KERNEL<T, 4, 16><<<grid, 256, 0, st>>>(__VA_ARGS__);            \
            else KERNEL<T, 8, 16><<<grid, 256, 0, st>>>(__VA_ARGS__);                          \
        }                                                                                     \
    } while (0)

template <typename T>
allegro_status_t launch_radial_forward(int n, int nb, double rc, long E, const void* rvec, const void* W_r, void* w, cudaStream_t st) {
    if (E == 0) return ALLEGRO_OK;
    if (n > 256) { set_error("radial_forward: n = %d unsupported (n <= 256)", n); return ALLEGRO_EUNSUPPORTED; }
    ALLEGRO_RAD_DISPATCH(radial_fwd_kernel, n, nb, rc, E, (const T*)rvec, (const T*)W_r, (T*)w);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
template <typename T>
allegro_status_t launch_radial_backward(int n, int nb, double rc, long E, const void* rvec, const void* W_r, const void* g_w, void* g_rvec,
                                        cudaStream_t st) {
    if (E == 0) return ALLEGRO_OK;
    if (n > 256) { set_error("radial_backward: n = %d unsupported (n <= 256)", n); return ALLEGRO_EUNSUPPORTED; }
    ALLEGRO_RAD_DISPATCH(radial_bwd_kernel, n, nb, rc, E, (const T*)rvec, (const T*)W_r, (const T*)g_w, (T*)g_rvec);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
template <typename T>
allegro_status_t launch_force_gather(int n_atoms, long E, const int32_t* row_ptr, const int32_t* rev, const void* g_rvec, void* F, cudaStream_t st) {
    (void)E;
    if (n_atoms == 0) return ALLEGRO_OK;
    force_gather_kernel<T><<<(unsigned)((n_atoms + 7) / 8), 256, 0, st>>>(n_atoms, row_ptr, rev, (const T*)g_rvec, (T*)F);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
template <typename T>
allegro_status_t launch_edge_energy(int n, int dV, long E, const void* out, const void* q, double kappa, void* e_edge, void* G, cudaStream_t st) {
    if (E == 0) return ALLEGRO_OK;
    edge_energy_kernel<T><<<(unsigned)((E + 7) / 8), 256, 0, st>>>(n, dV, E, (const T*)out, (const T*)q, (T)kappa, (T*)e_edge, (T*)G);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
// W[a][b] = sum_e g_rvec[e][a] rvec[e][b] (reading A25).  One 8-CTA cluster: every thread adds a strided subset of the edges in
// double, each CTA folds its threads with a fixed shared-memory tree per component, CTA 0 adds the CTAs' partials in rank order
// through distributed shared memory (deterministic, no workspace, no atomics).
template <typename T>
__global__ void __launch_bounds__(kSegThreads) virial_kernel(long E, const T* __restrict__ rvec, const T* __restrict__ g, T* __restrict__ W) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    __shared__ double sh[9][kSegThreads];
    const int rank = (int)cluster.block_rank();
    double acc[9];
#pragma unroll
    for (int i = 0; i < 9; ++i) acc[i] = 0.0;
    for (long e = (long)rank * kSegThreads + threadIdx.x; e < E; e += (long)kSegThreads * kSegCluster) {
        const double r0 = (double)rvec[3 * e], r1 = (double)rvec[3 * e + 1], r2 = (double)rvec[3 * e + 2];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double ga = (double)g[3 * e + a];
            acc[3 * a] = fma(ga, r0, acc[3 * a]);
            acc[3 * a + 1] = fma(ga, r1, acc[3 * a + 1]);
            acc[3 * a + 2] = fma(ga, r2, acc[3 * a + 2]);
        }
    }
#pragma unroll
    for (int i = 0; i < 9; ++i) sh[i][threadIdx.x] = acc[i];
    __syncthreads();
    for (int o = kSegThreads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
#pragma unroll
            for (int i = 0; i < 9; ++i) sh[i][threadIdx.x] += sh[i][threadIdx.x + o];
        }
        __syncthreads();
    }
    cluster.sync();
    if (rank == 0 && threadIdx.x < 9) {
        double tot = sh[threadIdx.x][0];
        for (int r = 1; r < kSegCluster; ++r) tot += *cluster.map_shared_rank(&sh[threadIdx.x][0], r);
        W[threadIdx.x] = (T)tot;
    }
    cluster.sync();  // keep every CTA's shared memory alive until CTA 0 has read it
}

template <typename T>
allegro_status_t launch_virial(long E, const void* rvec, const void* g_rvec, void* W, cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(kSegCluster);
    cfg.blockDim = dim3(kSegThreads);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = kSegCluster;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ALLEGRO_CUDA(cudaLaunchKernelEx(&cfg, virial_kernel<T>, E, (const T*)rvec, (const T*)g_rvec, (T*)W));
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

template <typename T>
allegro_status_t launch_segment_sum(const int32_t* ptr, int nseg, const void* vals, void* out, cudaStream_t st) {
    if (nseg == 0) return ALLEGRO_OK;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)nseg * kSegCluster);
    cfg.blockDim = dim3(kSegThreads);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = kSegCluster;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ALLEGRO_CUDA(cudaLaunchKernelEx(&cfg, segment_sum_kernel<T>, ptr, nseg, (const T*)vals, (T*)out));
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

#define ALLEGRO_INST(T)                                                                                                               \
    template allegro_status_t launch_radial_forward<T>(int, int, double, long, const void*, const void*, void*, cudaStream_t);        \
    template allegro_status_t launch_radial_backward<T>(int, int, double, long, const void*, const void*, const void*, void*, cudaStream_t); \
    template allegro_status_t launch_force_gather<T>(int, long, const int32_t*, const int32_t*, const void*, void*, cudaStream_t);    \
    template allegro_status_t launch_edge_energy<T>(int, int, long, const void*, const void*, double, void*, void*, cudaStream_t);    \
    template allegro_status_t launch_virial<T>(long, const void*, const void*, void*, cudaStream_t);                                   \
    template allegro_status_t launch_segment_sum<T>(const int32_t*, int, const void*, void*, cudaStream_t);
ALLEGRO_INST(float)
ALLEGRO_INST(double)

}  // namespace allegro
