// mix_kernels.cuh -- dense per-path channel mixing (ALLEGRO_W_DENSE; BASELINE.json:configs[2], reading A5):
//   t[e][n][p][M]   = sum_{m1 m2} C^p[m1][m2][M] V[e][n][off1(p)+m1] Eenv[c(e)][n][off2(p)+m2]      (un-weighted paths)
//   out[e][n'][off3(p)+M] = sum_p sum_n W[p][n'][n] t[e][n][p][M]
// and its VJP  gt[e][n][p][M] = sum_n' W[p][n'][n] G[e][n'][off3(p)+M], then the per-path CG VJP with unit weights.
//
// Generic version for any n, fp32 / fp64: the n x n mixes run on the FP32/FP64 FMA pipe with 128-bit shared-memory
// operands (t never leaves the SM: PAPER.md:71).  l_max <= 2 as described next; l_max = 3 with the loops exchanged (mixp_* below).
// One CTA per item; thread <-> (edge slot, channel).  Per tile of `nsl` edges:
//   forward : t (DT values per thread) -> shared tS[slot][col][n]; per path p: W_p -> shared Ws[n'][n] (row stride n+4),
//             acc[off3(p)+M] += <Ws[n'][:], tS[slot][toff(p)+M][:]>; thread (slot, n') stores its out row.
//   backward: G rows -> shared gS[slot][k][n']; per path p: W_p^T -> shared; gt[toff(p)+M] += <WsT[n][:], gS[slot][off3(p)+M][:]>;
//             then the generated per-path VJP (gV row stored, gEenv accumulated in registers over the segment).
// fp32, l_max = 2, n = 64 (configs[2]) is served by the tcgen05 tensor-core version in mix3_kernels.cuh (compiled in inst_mix3.cu).
#pragma once
#include <type_traits>
#include <utility>

#include "common.cuh"
#include "launch.h"

namespace allegro {

template <int I, int N, typename F>
__device__ __forceinline__ void static_for(F&& f) {
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

// dot product of two 16-byte-aligned shared-memory rows of length n (n * sizeof(T) % 16 == 0), 128-bit loads
template <typename T>
__device__ __forceinline__ T dot_rows(const T* __restrict__ a, const T* __restrict__ b, int n, T acc) {
    constexpr int VEC = 16 / (int)sizeof(T);
    const int4* a4 = reinterpret_cast<const int4*>(a);
    const int4* b4 = reinterpret_cast<const int4*>(b);
    for (int i = 0; i < n / VEC; ++i) {
        const int4 av = a4[i], bv = b4[i];
        const T* as = reinterpret_cast<const T*>(&av);
        const T* bs = reinterpret_cast<const T*>(&bv);
#pragma unroll
        for (int k = 0; k < VEC; ++k) acc = fma(as[k], bs[k], acc);
    }
    return acc;
}

template <typename T, int L, int CT>
__global__ void __launch_bounds__(CT) mix_fwd_kernel(int nsl, int n, const int* __restrict__ row_ptr, const int* __restrict__ items,
                                                      const T* __restrict__ V, const T* __restrict__ Eenv, const T* __restrict__ W,
                                                      T* __restrict__ out) {
    using Gen = TPGen<L>;
    constexpr int DV = Gen::DV, DE = Gen::DE, DT = Gen::DT, P = Gen::P;
    constexpr int VEC = 16 / (int)sizeof(T);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    T* tS = reinterpret_cast<T*>(smem_raw);           // [nsl][DT][n]
    T* Ws = tS + (size_t)nsl * DT * n;                // [n][n + VEC]
    const int ldw = n + VEC;
    const int tid = threadIdx.x;
    const int slot = tid / n, ch = tid - slot * n;
    const bool active = slot < nsl;
    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    const int ntiles = (e1 - e0 + nsl - 1) / nsl;
    T E[DE];
#pragma unroll
    for (int j = 0; j < DE; ++j) E[j] = active ? Eenv[((size_t)c * n + ch) * DE + j] : T(0);

    for (int t = 0; t < ntiles; ++t) {
        const int eb = e0 + t * nsl;
        const bool valid = active && eb + slot < e1;
        if (valid) {
            T v[DV], tt[DT];
            row_load<T, DV>(V + ((size_t)(eb + slot) * n + ch) * DV, v);
            Gen::template fwd_paths<T>(v, E, tt);
#pragma unroll
            for (int col = 0; col < DT; ++col) tS[((size_t)slot * DT + col) * n + ch] = tt[col];
        }
        T acc[DV];
#pragma unroll
        for (int k = 0; k < DV; ++k) acc[k] = T(0);
        static_for<0, P>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int toff = Gen::toff(p), off3 = Gen::off3(p), d3 = Gen::d3(p);
            __syncthreads();  // tS complete (p == 0) / previous W_p consumed
            for (int idx = tid; idx < n * n / VEC; idx += CT) {
                const int r = (idx * VEC) / n, cc = (idx * VEC) - r * n;
                *reinterpret_cast<int4*>(Ws + (size_t)r * ldw + cc) = *reinterpret_cast<const int4*>(W + (size_t)p * n * n + (size_t)idx * VEC);
            }
            __syncthreads();
            if (valid) {
#pragma unroll
                for (int M = 0; M < d3; ++M)
                    acc[off3 + M] = dot_rows<T>(Ws + (size_t)ch * ldw, tS + ((size_t)slot * DT + toff + M) * n, n, acc[off3 + M]);
            }
        });
        if (valid) row_store<T, DV>(out + ((size_t)(eb + slot) * n + ch) * DV, acc);
        __syncthreads();  // tS is rewritten by the next tile
    }
}

template <typename T, int L, int CT, bool WANT_GV>
__global__ void __launch_bounds__(CT) mix_bwd_kernel(int n, const int* __restrict__ row_ptr, const int* __restrict__ items,
                                                      const T* __restrict__ G, const T* __restrict__ V, const T* __restrict__ Eenv,
                                                      const T* __restrict__ W, T* __restrict__ gV, T* __restrict__ gE_dst, int gE_by_item) {
    using Gen = TPGen<L>;
    constexpr int DV = Gen::DV, DE = Gen::DE, DT = Gen::DT, P = Gen::P;
    constexpr int VEC = 16 / (int)sizeof(T);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nsl = CT / n;
    T* gS = reinterpret_cast<T*>(smem_raw);           // [nsl][DV][n]
    T* WsT = gS + (size_t)nsl * DV * n;               // [n][n + VEC], WsT[a][b] = W_p[b][a]
    const int ldw = n + VEC;
    const int tid = threadIdx.x;
    const int slot = tid / n, ch = tid - slot * n;
    const bool active = slot < nsl;
    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    const int ntiles = (e1 - e0 + nsl - 1) / nsl;
    T E[DE], gE[DE];
#pragma unroll
    for (int j = 0; j < DE; ++j) { E[j] = active ? Eenv[((size_t)c * n + ch) * DE + j] : T(0); gE[j] = T(0); }

    for (int t = 0; t < ntiles; ++t) {
        const int eb = e0 + t * nsl;
        const bool valid = active && eb + slot < e1;
        if (valid) {
            T g[DV];
            row_load<T, DV>(G + ((size_t)(eb + slot) * n + ch) * DV, g);
#pragma unroll
            for (int k = 0; k < DV; ++k) gS[((size_t)slot * DV + k) * n + ch] = g[k];
        }
        T gt[DT];
#pragma unroll
        for (int col = 0; col < DT; ++col) gt[col] = T(0);
        static_for<0, P>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int toff = Gen::toff(p), off3 = Gen::off3(p), d3 = Gen::d3(p);
            __syncthreads();
            for (int idx = tid; idx < n * n / VEC; idx += CT) {
                const int r = (idx * VEC) / n, cc = (idx * VEC) - r * n;  // W_p[r][cc .. cc+VEC)
                const int4 wv = *reinterpret_cast<const int4*>(W + (size_t)p * n * n + (size_t)idx * VEC);
                const T* ws = reinterpret_cast<const T*>(&wv);
#pragma unroll
                for (int k = 0; k < VEC; ++k) WsT[(size_t)(cc + k) * ldw + r] = ws[k];
            }
            __syncthreads();
            if (valid) {
#pragma unroll
                for (int M = 0; M < d3; ++M)
                    gt[toff + M] = dot_rows<T>(WsT + (size_t)ch * ldw, gS + ((size_t)slot * DV + off3 + M) * n, n, gt[toff + M]);
            }
        });
        if (valid) {
            T v[DV], gv[DV];
            row_load<T, DV>(V + ((size_t)(eb + slot) * n + ch) * DV, v);
            Gen::template bwd_paths<T, WANT_GV>(v, E, gt, gv, gE);
            if constexpr (WANT_GV) row_store<T, DV>(gV + ((size_t)(eb + slot) * n + ch) * DV, gv);
        }
        __syncthreads();  // gS is rewritten by the next tile
    }
    // ---- gEenv: slots summed in slot order
    T* red = reinterpret_cast<T*>(smem_raw);
    __syncthreads();
    if (active) {
#pragma unroll
        for (int j = 0; j < DE; ++j) red[((size_t)slot * n + ch) * DE + j] = gE[j];
    }
    __syncthreads();
    if (slot == 0) {
        T* dst = gE_dst + ((size_t)(gE_by_item ? (long)blockIdx.x : (long)c) * n + ch) * DE;
#pragma unroll
        for (int j = 0; j < DE; ++j) {
            T acc = red[(size_t)ch * DE + j];
            for (int sl = 1; sl < nsl; ++sl) acc += red[((size_t)sl * n + ch) * DE + j];
            dst[j] = acc;
        }
    }
}

// ------------------------------------------------------------------------------------------------------------------
// Gradient with respect to the dense path weights (training; PAPER.md:69 leaves the training kernels to future work):
//   g_W[p][n'][n] = sum_e sum_M G[e][n'][off3(p) + M] * t_p[e][n][M]
// One CTA per (path p, split s of the centres): the n x n accumulator of ONE path lives in registers (4 x 4 blocks per thread),
// so no partial matrix is ever flushed per centre; the CTA walks its centres, recomputes t_p of nsl edges at a time into shared
// memory next to the matching cotangent components, and adds their outer product.  Per centre the sum runs in T, across
// centres in double; the kGwSplits partial matrices are added in split order by gw_dense_final_kernel (no atomics: the
// result is bitwise reproducible).  The CTAs of the 30 paths of a split run side by side and share V / G / Eenv through L2.
constexpr int kGwSplits = 16;
constexpr int kGwMaxBlocks = 4;      // 4 x 4 blocks per thread: n <= 128 with 256 threads

template <typename T, int L, int CT>
__global__ void __launch_bounds__(CT) mix_gw_kernel(int n, int n_centres, const int* __restrict__ row_ptr, const T* __restrict__ G,
                                                     const T* __restrict__ V, const T* __restrict__ Eenv, T* __restrict__ part) {
    using Gen = TPGen<L>;
    constexpr int DV = Gen::DV, DE = Gen::DE, P = Gen::P, D3MAX = 2 * L + 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nsl = CT / n;
    T* ts = reinterpret_cast<T*>(smem_raw);            // [nsl][D3MAX][n]   t_p of the tile
    T* gS = ts + (size_t)nsl * D3MAX * n;             // [nsl][D3MAX][n]   G[e][.][off3 + M]
    const int tid = threadIdx.x;
    const int p = blockIdx.x % P, split = blockIdx.x / P;
    const int c_lo = (int)((long)n_centres * split / kGwSplits), c_hi = (int)((long)n_centres * (split + 1) / kGwSplits);
    const int slot = tid / n, ch = tid - slot * n;
    const bool active = slot < nsl;
    const int nq = n / 4, nblk = nq * nq;              // 4 x 4 blocks of the n x n matrix, block b -> (n' = 4 (b / nq), n = 4 (b % nq))
    double acc[kGwMaxBlocks][16];
#pragma unroll
    for (int k = 0; k < kGwMaxBlocks; ++k)
#pragma unroll
        for (int i = 0; i < 16; ++i) acc[k][i] = 0.0;
    int d3 = 1, off3 = 0;
    static_for<0, P>([&](auto pc) {
        constexpr int pp = decltype(pc)::value;
        if (pp == p) { d3 = Gen::d3(pp); off3 = Gen::off3(pp); }
    });

    for (int c = c_lo; c < c_hi; ++c) {
        const int e0 = row_ptr[c], e1 = row_ptr[c + 1];
        T E[DE];
#pragma unroll
        for (int j = 0; j < DE; ++j) E[j] = active ? Eenv[((size_t)c * n + ch) * DE + j] : T(0);
        T part_c[kGwMaxBlocks][16];
#pragma unroll
        for (int k = 0; k < kGwMaxBlocks; ++k)
#pragma unroll
            for (int i = 0; i < 16; ++i) part_c[k][i] = T(0);
        for (int eb = e0; eb < e1; eb += nsl) {
            __syncthreads();
            if (active) {
                const int e = eb + slot;
                T t[D3MAX], g[D3MAX];
#pragma unroll
                for (int M = 0; M < D3MAX; ++M) { t[M] = T(0); g[M] = T(0); }
                if (e < e1) {
                    const T* vrow = V + ((size_t)e * n + ch) * DV;
                    const T* grow = G + ((size_t)e * n + ch) * DV;
                    static_for<0, P>([&](auto pc) {
                        constexpr int pp = decltype(pc)::value;
                        using Pth = TPPath<L, pp>;
                        if (pp == p) {
                            T tp[Pth::D3];
                            Pth::template fwd<T>(vrow, E, tp);
#pragma unroll
                            for (int M = 0; M < Pth::D3; ++M) { t[M] = tp[M]; g[M] = grow[Pth::OFF3 + M]; }
                        }
                    });
                }
#pragma unroll
                for (int M = 0; M < D3MAX; ++M) {
                    ts[((size_t)slot * D3MAX + M) * n + ch] = t[M];
                    gS[((size_t)slot * D3MAX + M) * n + ch] = g[M];
                }
            }
            __syncthreads();
#pragma unroll
            for (int k = 0; k < kGwMaxBlocks; ++k) {
                const int b = tid + k * CT;
                if (b < nblk) {
                    const int r0 = 4 * (b / nq), c0 = 4 * (b - (b / nq) * nq);
                    for (int sl = 0; sl < nsl; ++sl)
                        for (int M = 0; M < d3; ++M) {
                            const T* gp = gS + ((size_t)sl * D3MAX + M) * n + r0;
                            const T* tp = ts + ((size_t)sl * D3MAX + M) * n + c0;
#pragma unroll
                            for (int i = 0; i < 4; ++i)
#pragma unroll
                                for (int j = 0; j < 4; ++j) part_c[k][4 * i + j] = fma(gp[i], tp[j], part_c[k][4 * i + j]);
                        }
                }
            }
        }
#pragma unroll
        for (int k = 0; k < kGwMaxBlocks; ++k)
#pragma unroll
            for (int i = 0; i < 16; ++i) acc[k][i] += (double)part_c[k][i];
    }
    T* dst = part + ((size_t)split * P + p) * n * n;
#pragma unroll
    for (int k = 0; k < kGwMaxBlocks; ++k) {
        const int b = tid + k * CT;
        if (b < nblk) {
            const int r0 = 4 * (b / nq), c0 = 4 * (b - (b / nq) * nq);
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dst[(size_t)(r0 + i) * n + c0 + j] = (T)acc[k][4 * i + j];
        }
    }
}

// g_W = the split partials added in split order
template <typename T>
__global__ void gw_dense_final_kernel(long count, const T* __restrict__ part, T* __restrict__ g_W) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    double a = 0.0;
    for (int s = 0; s < kGwSplits; ++s) a += (double)part[(size_t)s * count + i];
    g_W[i] = (T)a;
}

static inline bool all_blocks(const allegro_plan* plan) {
    const unsigned full = (1u << (2 * (plan->l_max + 1))) - 1u;
    return (plan->out_blocks & full) == full && (plan->in_blocks & full) == full;
}

// l_max <= 2: all un-weighted path values of an (edge, channel) live in the thread (mix_fwd / mix_bwd); l_max = 3: the
// paths-outer kernels above (312 values do not fit the register file).
#if ALLEGRO_L <= 2
template <typename T>
static allegro_status_t launch_mix_forward(const TpArgs& a) {
    using Gen = TPGen<ALLEGRO_L>;
    constexpr int CT = sizeof(T) == 4 ? 256 : 128;
    constexpr int VEC = 16 / (int)sizeof(T);
    if (a.n % VEC != 0 || a.n > CT) {
        set_error("tp_forward (dense): n = %d unsupported (n %% %d == 0, n <= %d)", a.n, VEC, CT);
        return ALLEGRO_EUNSUPPORTED;
    }
#if ALLEGRO_L == 2
    if constexpr (sizeof(T) == 4) {
        if (a.n == 64) return launch_mix3_forward_f32_l2_n64(a);
    }
#endif
    if (!all_blocks(a.plan)) {
        set_error("tp_forward (dense): block subsets are built for fp32, l_max = 2, n = 64 only");
        return ALLEGRO_EUNSUPPORTED;
    }
    const size_t ws_bytes = (size_t)a.n * (a.n + VEC) * sizeof(T);
    const size_t per_slot = (size_t)Gen::DT * a.n * sizeof(T);
    int nsl = CT / a.n;
    while (nsl > 1 && nsl * per_slot + ws_bytes > 200 * 1024) --nsl;
    const size_t smem = nsl * per_slot + ws_bytes;
    if (smem > 226 * 1024) {
        set_error("tp_forward (dense): n = %d needs %zu bytes of shared memory", a.n, smem);
        return ALLEGRO_EUNSUPPORTED;
    }
    auto k = mix_fwd_kernel<T, ALLEGRO_L, CT>;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k<<<(unsigned)a.n_items, CT, smem, a.st>>>(nsl, a.n, a.row_ptr, a.items, (const T*)a.V, (const T*)a.Eenv, (const T*)a.path_w, (T*)a.out);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

#else
// l_max = 3: the paths-outer kernels of mixp_kernels.cuh, compiled in their own translation units (inst_mixp.cu; the 68 unrolled
// paths make them the slowest files of the build, so they do not sit behind the sparse kernels of this unit)
template <typename T> allegro_status_t launch_mixp_forward(const TpArgs& a);
template <typename T, bool WANT_GV> allegro_status_t launch_mixp_backward(const TpArgs& a, T* gE_dst, int gE_by_item);
template <typename T> allegro_status_t launch_mixp_gw(const TpArgs& a, T* part);

template <typename T>
static allegro_status_t launch_mix_forward(const TpArgs& a) {
    constexpr int CT = sizeof(T) == 4 ? 256 : 128;
    constexpr int VEC = 16 / (int)sizeof(T);
    if (a.n % VEC != 0 || a.n > CT) {
        set_error("tp_forward (dense): n = %d unsupported (n %% %d == 0, n <= %d)", a.n, VEC, CT);
        return ALLEGRO_EUNSUPPORTED;
    }
    if (!all_blocks(a.plan)) {
        set_error("tp_forward (dense): block subsets are built for fp32, l_max = 2, n = 64 only");
        return ALLEGRO_EUNSUPPORTED;
    }
    return launch_mixp_forward<T>(a);
}
#endif

// workspace layout of tp_backward (dense mode): [gE partial rows, one per item (only with items)] [kGwSplits partial g_W (only with g_path_w)]
template <typename T>
static size_t mix_backward_workspace(int n, long n_items, bool have_items, bool want_gw) {
    size_t b = have_items ? align_up((size_t)n_items * n * TPGen<ALLEGRO_L>::DE * sizeof(T), 256) : 0;
    if (want_gw) b += align_up((size_t)kGwSplits * TPGen<ALLEGRO_L>::P * n * n * sizeof(T), 256);
    return b;
}

#if ALLEGRO_L <= 2
template <typename T>
static allegro_status_t launch_mix_backward(const TpArgs& a) {
    using Gen = TPGen<ALLEGRO_L>;
    constexpr int CT = sizeof(T) == 4 ? 256 : 128;
    constexpr int VEC = 16 / (int)sizeof(T);
    if (a.n % VEC != 0 || a.n > CT) {
        set_error("tp_backward (dense): n = %d unsupported (n %% %d == 0, n <= %d)", a.n, VEC, CT);
        return ALLEGRO_EUNSUPPORTED;
    }
    const bool have_items = a.items != nullptr;
    T* gE_dst = have_items ? (T*)a.ws : (T*)a.gEenv;
    if (a.g_path_w != nullptr) {   // training: gradient with respect to W_p (all blocks, explicit cotangent)
        if (!all_blocks(a.plan) || a.q != nullptr || a.n % 4 != 0 || (a.n / 4) * (a.n / 4) > kGwMaxBlocks * CT) {
            set_error("tp_backward (dense): g_path_w needs all blocks, an explicit cotangent and n %% 4 == 0, n <= 128");
            return ALLEGRO_EUNSUPPORTED;
        }
        T* part = (T*)((unsigned char*)a.ws + (have_items ? align_up((size_t)a.n_items * a.n * Gen::DE * sizeof(T), 256) : 0));
        const int nsl = CT / a.n;
        const size_t smem_gw = 2 * (size_t)nsl * (2 * ALLEGRO_L + 1) * a.n * sizeof(T);
        auto kg = mix_gw_kernel<T, ALLEGRO_L, CT>;
        ALLEGRO_CUDA(cudaFuncSetAttribute(kg, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_gw));
        kg<<<(unsigned)(Gen::P * kGwSplits), CT, smem_gw, a.st>>>(a.n, a.n_atoms, a.row_ptr, (const T*)a.G, (const T*)a.V, (const T*)a.Eenv, part);
        ALLEGRO_LAUNCHED();
        const long count = (long)Gen::P * a.n * a.n;
        gw_dense_final_kernel<T><<<(unsigned)((count + 255) / 256), 256, 0, a.st>>>(count, part, (T*)a.g_path_w);
        ALLEGRO_LAUNCHED();
    }
#if ALLEGRO_L == 2
    if constexpr (sizeof(T) == 4) {
        if (a.n == 64) {
            allegro_status_t s2 = launch_mix3_backward_f32_l2_n64(a, (float*)gE_dst, have_items ? 1 : 0);
            if (s2 != ALLEGRO_OK) return s2;
            if (have_items) {
                combine_items_kernel<T><<<(unsigned)a.n_items, 128, 0, a.st>>>(a.items, a.n_items, a.n * Gen::DE, (const T*)a.ws, (T*)a.gEenv);
                ALLEGRO_LAUNCHED();
            }
            return ALLEGRO_OK;
        }
    }
#endif
    if (!all_blocks(a.plan)) {
        set_error("tp_backward (dense): block subsets are built for fp32, l_max = 2, n = 64 only");
        return ALLEGRO_EUNSUPPORTED;
    }
    const int nsl = CT / a.n;
    size_t smem = (size_t)nsl * Gen::DV * a.n * sizeof(T) + (size_t)a.n * (a.n + VEC) * sizeof(T);
    const size_t red = (size_t)CT * Gen::DE * sizeof(T);
    if (smem < red) smem = red;
#define ALLEGRO_MIXB(GV)                                                                                                   \
    {                                                                                                                      \
        auto k = mix_bwd_kernel<T, ALLEGRO_L, CT, GV>;                                                                     \
        ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));                      \
        k<<<(unsigned)a.n_items, CT, smem, a.st>>>(a.n, a.row_ptr, a.items, (const T*)a.G, (const T*)a.V, (const T*)a.Eenv, \
                                                   (const T*)a.path_w, (T*)a.gV, gE_dst, have_items ? 1 : 0);              \
    }
    if (a.gV != nullptr) ALLEGRO_MIXB(true) else ALLEGRO_MIXB(false)
#undef ALLEGRO_MIXB
    ALLEGRO_LAUNCHED();
    if (have_items) {
        combine_items_kernel<T><<<(unsigned)a.n_items, 128, 0, a.st>>>(a.items, a.n_items, a.n * Gen::DE, (const T*)a.ws, (T*)a.gEenv);
        ALLEGRO_LAUNCHED();
    }
    return ALLEGRO_OK;
}
#else
template <typename T>
static allegro_status_t launch_mix_backward(const TpArgs& a) {
    using Gen = TPGen<ALLEGRO_L>;
    constexpr int CT = sizeof(T) == 4 ? 256 : 128;
    constexpr int VEC = 16 / (int)sizeof(T);
    if (a.n % VEC != 0 || a.n > CT) {
        set_error("tp_backward (dense): n = %d unsupported (n %% %d == 0, n <= %d)", a.n, VEC, CT);
        return ALLEGRO_EUNSUPPORTED;
    }
    if (!all_blocks(a.plan) || a.q != nullptr) {
        set_error("tp_backward (dense): block subsets and the on-the-fly cotangent are built for fp32, l_max = 2, n = 64 only");
        return ALLEGRO_EUNSUPPORTED;
    }
    const bool have_items = a.items != nullptr;
    T* gE_dst = have_items ? (T*)a.ws : (T*)a.gEenv;
    if (a.g_path_w != nullptr) {   // training: gradient with respect to W_p
        if (a.n % 4 != 0 || (a.n / 4) * (a.n / 4) > kGwMaxBlocks * CT) {
            set_error("tp_backward (dense): g_path_w needs n %% 4 == 0, n <= 128");
            return ALLEGRO_EUNSUPPORTED;
        }
        T* part = (T*)((unsigned char*)a.ws + (have_items ? align_up((size_t)a.n_items * a.n * Gen::DE * sizeof(T), 256) : 0));
        allegro_status_t sg = launch_mixp_gw<T>(a, part);
        if (sg != ALLEGRO_OK) return sg;
    }
    allegro_status_t sb = a.gV != nullptr ? launch_mixp_backward<T, true>(a, gE_dst, have_items ? 1 : 0)
                                          : launch_mixp_backward<T, false>(a, gE_dst, have_items ? 1 : 0);
    if (sb != ALLEGRO_OK) return sb;
    if (have_items) {
        combine_items_kernel<T><<<(unsigned)a.n_items, 128, 0, a.st>>>(a.items, a.n_items, a.n * Gen::DE, (const T*)a.ws, (T*)a.gEenv);
        ALLEGRO_LAUNCHED();
    }
    return ALLEGRO_OK;
}
#endif

}  // namespace allegro
