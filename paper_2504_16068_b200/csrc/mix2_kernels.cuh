// mix2_kernels.cuh -- second version of the dense per-path channel mix for fp32, l_max = 2, n = 64 (BASELINE.json:configs[2]).
// Compiled by inst_mix2.cu in three parts (forward / VJP with gV / VJP without gV) so that the parts build in parallel.
#pragma once
#include <type_traits>
#include <utility>

#include "common.cuh"
#include "launch.h"

namespace allegro {

template <int I, int N, typename F>
__device__ __forceinline__ void static_for2(F&& f) {
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for2<I + 1, N>(f);
    }
}

// ------------------------------------------------------------------------------------------------
// Version 2 (fp32, n = 32 or 64, l_max <= 2): tiles of TE = 4 * (256 / N) edges, t recomputed PER PATH so that only the
// path's (2 l3 + 1) columns sit in shared memory, and the thread's W_p row (forward: W_p[n'][:], backward: W_p[:][n])
// held in N registers for the whole tile: the inner product reads its other operand with broadcast 128-bit loads and
// every weight element loaded from L2 is used for 4 edges x (2 l3 + 1) columns.
template <int L, int N>
struct Mix2 {
    using Gen = TPGen<L>;
    static constexpr int CT = 256, EG = CT / N, EPT = 4, TE = EG * EPT, DV = Gen::DV, DE = Gen::DE, P = Gen::P;
    static constexpr int D3MAX = 2 * L + 1, LDT = N + 4;
    static constexpr size_t kVt = (size_t)TE * N * DV * sizeof(float);
    static constexpr size_t kFwdSmem = kVt + 2 * (size_t)TE * D3MAX * LDT * sizeof(float);
    static constexpr size_t kBwdSmem = kVt + (size_t)TE * DV * LDT * sizeof(float);
};

template <int N>
__device__ __forceinline__ float dot_reg_smem(const float (&wr)[N], const float* __restrict__ col, float acc) {
    const float4* c4 = reinterpret_cast<const float4*>(col);
#pragma unroll
    for (int k = 0; k < N / 4; ++k) {
        const float4 c = c4[k];
        acc = fmaf(wr[4 * k], c.x, acc);
        acc = fmaf(wr[4 * k + 1], c.y, acc);
        acc = fmaf(wr[4 * k + 2], c.z, acc);
        acc = fmaf(wr[4 * k + 3], c.w, acc);
    }
    return acc;
}

template <int L, int N>
__global__ void __launch_bounds__(256) mix_fwd2_kernel(const int* __restrict__ row_ptr, const int* __restrict__ items, const float* __restrict__ V,
                                                        const float* __restrict__ Eenv, const float* __restrict__ W, float* __restrict__ out) {
    using M2 = Mix2<L, N>;
    constexpr int DV = M2::DV, DE = M2::DE, P = M2::P, EPT = M2::EPT, TE = M2::TE, LDT = M2::LDT, D3MAX = M2::D3MAX;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* Vt = reinterpret_cast<float*>(smem_raw);                 // [TE][N][DV]
    float* tP = reinterpret_cast<float*>(smem_raw + M2::kVt);       // [2][TE * D3MAX][LDT]
    const int tid = threadIdx.x, ch = tid % N, eg = tid / N;
    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    float E[DE];
#pragma unroll
    for (int j = 0; j < DE; ++j) E[j] = Eenv[((size_t)c * N + ch) * DE + j];

    for (int eb = e0; eb < e1; eb += TE) {
        const int cnt = min(TE, e1 - eb);
        {   // V tile: one contiguous byte range, 128-bit coalesced loads
            const int4* src = reinterpret_cast<const int4*>(V + (size_t)eb * N * DV);
            int4* dst = reinterpret_cast<int4*>(Vt);
            for (int idx = tid; idx < cnt * N * DV / 4; idx += 256) dst[idx] = src[idx];
        }
        __syncthreads();
        float acc[EPT][DV];
#pragma unroll
        for (int q = 0; q < EPT; ++q)
#pragma unroll
            for (int k = 0; k < DV; ++k) acc[q][k] = 0.f;
        static_for2<0, P>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            using Pth = TPPath<L, p>;
            constexpr int D3 = Pth::D3, OFF3 = Pth::OFF3;
            float* buf = tP + (size_t)(p & 1) * TE * D3MAX * LDT;
#pragma unroll
            for (int q = 0; q < EPT; ++q) {
                const int el = eg * EPT + q;
                if (el < cnt) {
                    float t[D3];
                    Pth::template fwd<float>(Vt + ((size_t)el * N + ch) * DV, E, t);
#pragma unroll
                    for (int M = 0; M < D3; ++M) buf[(el * D3 + M) * LDT + ch] = t[M];
                }
            }
            float wr[N];
            {
                const float4* w4 = reinterpret_cast<const float4*>(W + ((size_t)p * N + ch) * N);
#pragma unroll
                for (int k = 0; k < N / 4; ++k) {
                    const float4 w = w4[k];
                    wr[4 * k] = w.x; wr[4 * k + 1] = w.y; wr[4 * k + 2] = w.z; wr[4 * k + 3] = w.w;
                }
            }
            __syncthreads();
#pragma unroll
            for (int q = 0; q < EPT; ++q) {
                const int el = eg * EPT + q;
                if (el < cnt) {
#pragma unroll
                    for (int M = 0; M < D3; ++M) acc[q][OFF3 + M] = dot_reg_smem<N>(wr, buf + (el * D3 + M) * LDT, acc[q][OFF3 + M]);
                }
            }
        });
#pragma unroll
        for (int q = 0; q < EPT; ++q) {
            const int el = eg * EPT + q;
            if (el < cnt) row_store<float, DV>(out + ((size_t)(eb + el) * N + ch) * DV, acc[q]);
        }
        __syncthreads();  // Vt and tP are rewritten by the next tile
    }
}

template <int L, int N, bool WANT_GV>
__global__ void __launch_bounds__(256) mix_bwd2_kernel(const int* __restrict__ row_ptr, const int* __restrict__ items, const float* __restrict__ G,
                                                        const float* __restrict__ V, const float* __restrict__ Eenv, const float* __restrict__ W,
                                                        float* __restrict__ gV, float* __restrict__ gE_dst, int gE_by_item) {
    using M2 = Mix2<L, N>;
    constexpr int DV = M2::DV, DE = M2::DE, P = M2::P, EPT = M2::EPT, TE = M2::TE, LDT = M2::LDT, EG = M2::EG;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* Vt = reinterpret_cast<float*>(smem_raw);                 // [TE][N][DV]
    float* gS = reinterpret_cast<float*>(smem_raw + M2::kVt);       // [TE * DV][LDT]: gS[(e, k)][n'] = G[e][n'][k]
    const int tid = threadIdx.x, ch = tid % N, eg = tid / N;
    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    float E[DE], gE[DE];
#pragma unroll
    for (int j = 0; j < DE; ++j) { E[j] = Eenv[((size_t)c * N + ch) * DE + j]; gE[j] = 0.f; }

    for (int eb = e0; eb < e1; eb += TE) {
        const int cnt = min(TE, e1 - eb);
        {
            const int4* src = reinterpret_cast<const int4*>(V + (size_t)eb * N * DV);
            int4* dst = reinterpret_cast<int4*>(Vt);
            for (int idx = tid; idx < cnt * N * DV / 4; idx += 256) dst[idx] = src[idx];
            const float* g = G + (size_t)eb * N * DV;
            for (int idx = tid; idx < cnt * N * DV; idx += 256) {
                const int el = idx / (N * DV), rem = idx - el * (N * DV), np = rem / DV, k = rem - np * DV;
                gS[(el * DV + k) * LDT + np] = g[idx];
            }
        }
        __syncthreads();
        float gv[EPT][DV];
#pragma unroll
        for (int q = 0; q < EPT; ++q)
#pragma unroll
            for (int k = 0; k < DV; ++k) gv[q][k] = 0.f;
        static_for2<0, P>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            using Pth = TPPath<L, p>;
            constexpr int D3 = Pth::D3, OFF3 = Pth::OFF3;
            float wc[N];  // W_p[n'][ch], n' = 0..N-1 (coalesced across ch)
#pragma unroll
            for (int k = 0; k < N; ++k) wc[k] = W[((size_t)p * N + k) * N + ch];
#pragma unroll
            for (int q = 0; q < EPT; ++q) {
                const int el = eg * EPT + q;
                if (el < cnt) {
                    float gt[D3];
#pragma unroll
                    for (int M = 0; M < D3; ++M) gt[M] = dot_reg_smem<N>(wc, gS + (el * DV + OFF3 + M) * LDT, 0.f);
                    Pth::template bwd<float, WANT_GV>(Vt + ((size_t)el * N + ch) * DV, E, gt, gv[q], gE);
                }
            }
        });
        if constexpr (WANT_GV) {
#pragma unroll
            for (int q = 0; q < EPT; ++q) {
                const int el = eg * EPT + q;
                if (el < cnt) row_store<float, DV>(gV + ((size_t)(eb + el) * N + ch) * DV, gv[q]);
            }
        }
        __syncthreads();
    }
    // ---- gEenv: edge groups summed in order
    float* red = reinterpret_cast<float*>(smem_raw);
#pragma unroll
    for (int j = 0; j < DE; ++j) red[((size_t)eg * N + ch) * DE + j] = gE[j];
    __syncthreads();
    if (eg == 0) {
        float* dst = gE_dst + ((size_t)(gE_by_item ? (long)blockIdx.x : (long)c) * N + ch) * DE;
#pragma unroll
        for (int j = 0; j < DE; ++j) {
            float acc = red[(size_t)ch * DE + j];
            for (int g2 = 1; g2 < EG; ++g2) acc += red[((size_t)g2 * N + ch) * DE + j];
            dst[j] = acc;
        }
    }
}

}  // namespace allegro
