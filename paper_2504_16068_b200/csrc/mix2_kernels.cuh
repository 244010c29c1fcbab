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
// Tiles of 2 * (256 / N) edges; t is recomputed PER PATH so that only the path's (2 l3 + 1) columns sit in shared memory; W_p is
// staged once per (tile, path) with coalesced 128-bit loads; the 64 x 64 x columns products run on the tensor cores.
template <int L, int N>
struct Mix2 {
    using Gen = TPGen<L>;
    static constexpr int CT = 256, EG = CT / N, DV = Gen::DV, DE = Gen::DE, P = Gen::P;
    static constexpr int D3MAX = 2 * L + 1, LDT = N + 4;
    static constexpr int EPTF = 2, TEF = EG * EPTF;   // tile: 8 edges (n = 64) so that two CTAs fit one SM
    static constexpr size_t kVtF = (size_t)TEF * N * DV * sizeof(float);
    static constexpr size_t kFwdSmem = 2 * kVtF + ((size_t)TEF * D3MAX + N) * LDT * sizeof(float);
    static constexpr size_t kBwdSmem = kVtF + ((size_t)TEF * DV + (size_t)TEF * D3MAX + N) * LDT * sizeof(float);
};


// 3xTF32 on the tensor cores (legacy mma.sync path; tcgen05 is the next step): x = hi + lo;
// A.B ~= A_lo.B_hi + A_hi.B_lo + A_hi.B_hi keeps ~21 mantissa bits, enough for the 1e-5 fp32 tolerance (plain TF32 is not).
// The split truncates instead of rounding (cvt.rna.tf32 is a ~5-instruction sequence on sm_100a and dominated the kernel:
// profiles/r1_final.md): hi = x with the 13 low mantissa bits cleared, lo = x - hi (exact); the tensor core ignores lo's
// low 13 bits, which leaves a relative error of 2^-20 per product.
__device__ __forceinline__ void split_tf32(float x, uint32_t& hi, uint32_t& lo) {
    hi = __float_as_uint(x) & 0xffffe000u;
    lo = __float_as_uint(x - __uint_as_float(hi));
}
__device__ __forceinline__ void mma_tf32(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// The loop over paths is a RUN-TIME loop: only the small per-path CG code is selected by a compare chain, the
// 64-wide inner products exist once per (2 l3 + 1) in {1, 3, 5}.  (A fully unrolled version is 26k FMAs of straight-line
// code per kernel and stalls on instruction fetch: measured "no_instruction" = 56 % of the warp stall samples.)
template <int L>
struct PathTab {
    using Gen = TPGen<L>;
    int d3[Gen::P], off3[Gen::P];
};
template <int L>
__host__ __device__ constexpr PathTab<L> make_path_tab() {
    PathTab<L> t{};
    for (int p = 0; p < TPGen<L>::P; ++p) { t.d3[p] = TPGen<L>::d3(p); t.off3[p] = TPGen<L>::off3(p); }
    return t;
}

template <int L, int N>
__global__ void __launch_bounds__(256, 2) mix_fwd2_kernel(const int* __restrict__ row_ptr, const int* __restrict__ items, const float* __restrict__ V,
                                                        const float* __restrict__ Eenv, const float* __restrict__ W, float* __restrict__ out) {
    using M2 = Mix2<L, N>;
    constexpr int DV = M2::DV, DE = M2::DE, P = M2::P, EPT = M2::EPTF, TE = M2::TEF, LDT = M2::LDT, D3MAX = M2::D3MAX;
    constexpr PathTab<L> tab = make_path_tab<L>();
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* Vt = reinterpret_cast<float*>(smem_raw);                 // [TE][N][DV]
    float* Os = Vt + (size_t)TE * N * DV;                            // [TE][N][DV] out tile (accumulated over paths)
    float* tP = Os + (size_t)TE * N * DV;                            // [TE * D3MAX][LDT]
    float* Ws = tP + (size_t)TE * D3MAX * LDT;                       // [N][LDT]
    const int tid = threadIdx.x, ch = tid % N, eg = tid / N;
    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    float E[DE];
#pragma unroll
    for (int j = 0; j < DE; ++j) E[j] = Eenv[((size_t)c * N + ch) * DE + j];

    for (int eb = e0; eb < e1; eb += TE) {
        const int cnt = min(TE, e1 - eb);
        {   // V tile: one contiguous byte range, 128-bit coalesced loads; out tile zeroed
            const int4* src = reinterpret_cast<const int4*>(V + (size_t)eb * N * DV);
            int4* dst = reinterpret_cast<int4*>(Vt);
            int4* oz = reinterpret_cast<int4*>(Os);
            for (int idx = tid; idx < cnt * N * DV / 4; idx += 256) { dst[idx] = src[idx]; oz[idx] = make_int4(0, 0, 0, 0); }
        }
        __syncthreads();
        for (int p = 0; p < P; ++p) {
            const int d3 = tab.d3[p], off3 = tab.off3[p];
            float* buf = tP;
            static_for2<0, P>([&](auto pc) {   // t_p of this thread's (edge, channel) pairs: per-path generated code
                constexpr int pp = decltype(pc)::value;
                if (p == pp) {
                    using Pth = TPPath<L, pp>;
#pragma unroll
                    for (int q = 0; q < EPT; ++q) {
                        const int el = eg * EPT + q;
                        if (el < cnt) {
                            float t[Pth::D3];
                            Pth::template fwd<float>(Vt + ((size_t)el * N + ch) * DV, E, t);
#pragma unroll
                            for (int M = 0; M < Pth::D3; ++M) buf[(el * Pth::D3 + M) * LDT + ch] = t[M];
                        }
                    }
                }
            });
            {   // W_p: coalesced 128-bit global reads into shared memory (row stride LDT: conflict-free row reads)
                const float4* w4 = reinterpret_cast<const float4*>(W + (size_t)p * N * N);
#pragma unroll
                for (int it = 0; it < N * N / 4 / 256; ++it) {
                    const int idx = tid + it * 256, r = idx / (N / 4), c4 = idx - r * (N / 4);
                    *reinterpret_cast<float4*>(Ws + r * LDT + 4 * c4) = w4[idx];
                }
            }
            __syncthreads();  // tP[p & 1] and Ws complete
            {   // D[n' (64) x cols (TE * d3)] = W_p . T_p on the tensor cores: warp -> 16 rows (mt) and every other 8-column tile
                const int lane = tid & 31, warp = tid >> 5, g = lane >> 2, t4 = lane & 3;
                const int mt = warp & 3, half = warp >> 2;
                uint32_t ahi[N / 8][4], alo[N / 8][4];
#pragma unroll
                for (int kt = 0; kt < N / 8; ++kt) {
                    const float* w0 = Ws + (mt * 16 + g) * LDT + kt * 8 + t4;
                    split_tf32(w0[0], ahi[kt][0], alo[kt][0]);
                    split_tf32(w0[8 * LDT], ahi[kt][1], alo[kt][1]);
                    split_tf32(w0[4], ahi[kt][2], alo[kt][2]);
                    split_tf32(w0[8 * LDT + 4], ahi[kt][3], alo[kt][3]);
                }
                auto tiles = [&](auto dc) {   // (2 l3 + 1) as a compile-time constant: column -> (edge, M) without integer division
                constexpr int D3 = decltype(dc)::value;
                constexpr int ntiles = TE * D3 / 8;
                for (int nt = half; nt < ntiles; nt += 2) {
                    float dacc[4] = {0.f, 0.f, 0.f, 0.f}, dlo[4] = {0.f, 0.f, 0.f, 0.f}, dmid[4] = {0.f, 0.f, 0.f, 0.f};
                    const float* bcol = buf + (nt * 8 + g) * LDT + t4;
#pragma unroll
                    for (int kt = 0; kt < N / 8; ++kt) {
                        uint32_t bh0, bl0, bh1, bl1;
                        split_tf32(bcol[kt * 8], bh0, bl0);
                        split_tf32(bcol[kt * 8 + 4], bh1, bl1);
                        mma_tf32(dlo, alo[kt], bh0, bh1);   // three independent accumulation chains (the MMA latency, not its
                        mma_tf32(dmid, ahi[kt], bl0, bl1);  // throughput, bounds a single chain of 24 dependent MMAs)
                        mma_tf32(dacc, ahi[kt], bh0, bh1);
                    }
                    // c0: (row g, col 2 t4), c1: (row g, col 2 t4 + 1), c2 / c3: row g + 8; col -> (edge, M) of this path
#pragma unroll
                    for (int i = 0; i < 4; ++i) dacc[i] += dlo[i] + dmid[i];
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int col = nt * 8 + 2 * t4 + (i & 1), row = mt * 16 + g + ((i & 2) ? 8 : 0);
                        const int el = col / D3, M = col - el * D3;
                        Os[((size_t)el * N + row) * DV + off3 + M] += dacc[i];
                    }
                }
                };
                if (d3 == 1) tiles(std::integral_constant<int, 1>{});
                else if (d3 == 3) tiles(std::integral_constant<int, 3>{});
                else tiles(std::integral_constant<int, (L >= 2 ? 5 : 3)>{});
            }
            __syncthreads();  // Ws and tP may be overwritten
        }
        __syncthreads();
        {   // out tile: one contiguous byte range, 128-bit coalesced stores
            int4* dst = reinterpret_cast<int4*>(out + (size_t)eb * N * DV);
            const int4* src = reinterpret_cast<const int4*>(Os);
            for (int idx = tid; idx < cnt * N * DV / 4; idx += 256) dst[idx] = src[idx];
        }
        __syncthreads();  // Vt, Os and tP are rewritten by the next tile
    }
}

template <int L, int N, bool WANT_GV>
__global__ void __launch_bounds__(256, 2) mix_bwd2_kernel(const int* __restrict__ row_ptr, const int* __restrict__ items, const float* __restrict__ G,
                                                           const float* __restrict__ V, const float* __restrict__ Eenv, const float* __restrict__ W,
                                                           float* __restrict__ gV, float* __restrict__ gE_dst, int gE_by_item) {
    using M2 = Mix2<L, N>;
    constexpr int DV = M2::DV, DE = M2::DE, P = M2::P, EPT = M2::EPTF, TE = M2::TEF, LDT = M2::LDT, EG = M2::EG, D3MAX = M2::D3MAX;
    constexpr PathTab<L> tab = make_path_tab<L>();
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* Vt = reinterpret_cast<float*>(smem_raw);                 // [TE][N][DV]
    float* gS = Vt + (size_t)TE * N * DV;                            // [TE * DV][LDT]: gS[(e, k)][n'] = G[e][n'][k]
    float* gtS = gS + (size_t)TE * DV * LDT;                         // [TE * D3MAX][LDT]: gt_p[(e, M)][n]
    float* Ws = gtS + (size_t)TE * D3MAX * LDT;                      // [N][LDT]: W_p[n'][n]
    const int tid = threadIdx.x, ch = tid % N, eg = tid / N;
    const int lane = tid & 31, warp = tid >> 5, g = lane >> 2, t4 = lane & 3, mt = warp & 3, half = warp >> 2;
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
            const float* gp = G + (size_t)eb * N * DV;
            for (int idx = tid; idx < TE * N * DV; idx += 256) {
                const int el = idx / (N * DV), rem = idx - el * (N * DV), np = rem / DV, k = rem - np * DV;
                gS[(el * DV + k) * LDT + np] = el < cnt ? gp[idx] : 0.f;   // zero rows beyond the ragged tail (they feed the MMA)
            }
        }
        __syncthreads();
        float gv[EPT][DV];
#pragma unroll
        for (int q = 0; q < EPT; ++q)
#pragma unroll
            for (int k = 0; k < DV; ++k) gv[q][k] = 0.f;
        for (int p = 0; p < P; ++p) {
            const int d3 = tab.d3[p], off3 = tab.off3[p];
            {   // W_p: coalesced 128-bit global reads into shared memory (every warp finished the previous path's MMA
                // before the "gtS complete" barrier below, so Ws is free)
                const float4* w4 = reinterpret_cast<const float4*>(W + (size_t)p * N * N);
#pragma unroll
                for (int it = 0; it < N * N / 4 / 256; ++it) {
                    const int idx = tid + it * 256, r = idx / (N / 4), c4 = idx - r * (N / 4);
                    *reinterpret_cast<float4*>(Ws + r * LDT + 4 * c4) = w4[idx];
                }
            }
            __syncthreads();  // Ws complete; every thread has consumed the previous path's gtS
            {   // gt_p[n (64) x cols (TE * d3)] = W_p^T . G_p on the tensor cores (3xTF32)
                uint32_t ahi[N / 8][4], alo[N / 8][4];
#pragma unroll
                for (int kt = 0; kt < N / 8; ++kt) {   // A[row = n][k = n'] = W_p[n'][n]
                    const float* w0 = Ws + (kt * 8 + t4) * LDT + mt * 16 + g;
                    split_tf32(w0[0], ahi[kt][0], alo[kt][0]);
                    split_tf32(w0[8], ahi[kt][1], alo[kt][1]);
                    split_tf32(w0[4 * LDT], ahi[kt][2], alo[kt][2]);
                    split_tf32(w0[4 * LDT + 8], ahi[kt][3], alo[kt][3]);
                }
                auto tiles = [&](auto dc) {
                    constexpr int D3 = decltype(dc)::value;
                    constexpr int ntiles = TE * D3 / 8;
                    for (int nt = half; nt < ntiles; nt += 2) {
                        float dacc[4] = {0.f, 0.f, 0.f, 0.f}, dlo[4] = {0.f, 0.f, 0.f, 0.f}, dmid[4] = {0.f, 0.f, 0.f, 0.f};
                        const int colb = nt * 8 + g, elb = colb / D3, Mb = colb - elb * D3;
                        const float* bcol = gS + (elb * DV + off3 + Mb) * LDT + t4;
#pragma unroll
                        for (int kt = 0; kt < N / 8; ++kt) {
                            uint32_t bh0, bl0, bh1, bl1;
                            split_tf32(bcol[kt * 8], bh0, bl0);
                            split_tf32(bcol[kt * 8 + 4], bh1, bl1);
                            mma_tf32(dlo, alo[kt], bh0, bh1);   // three independent accumulation chains
                            mma_tf32(dmid, ahi[kt], bl0, bl1);
                            mma_tf32(dacc, ahi[kt], bh0, bh1);
                        }
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const int col = nt * 8 + 2 * t4 + (i & 1), row = mt * 16 + g + ((i & 2) ? 8 : 0);
                            gtS[col * LDT + row] = dacc[i] + (dlo[i] + dmid[i]);
                        }
                    }
                };
                if (d3 == 1) tiles(std::integral_constant<int, 1>{});
                else if (d3 == 3) tiles(std::integral_constant<int, 3>{});
                else tiles(std::integral_constant<int, (L >= 2 ? 5 : 3)>{});
            }
            __syncthreads();  // gtS complete
            static_for2<0, P>([&](auto pc) {   // per-path CG VJP: generated code selected by a compare chain
                constexpr int pp = decltype(pc)::value;
                if (p == pp) {
                    using Pth = TPPath<L, pp>;
#pragma unroll
                    for (int q = 0; q < EPT; ++q) {
                        const int el = eg * EPT + q;
                        if (el < cnt) {
                            float g3[Pth::D3];
#pragma unroll
                            for (int M = 0; M < Pth::D3; ++M) g3[M] = gtS[(el * Pth::D3 + M) * LDT + ch];
                            Pth::template bwd<float, WANT_GV>(Vt + ((size_t)el * N + ch) * DV, E, g3, gv[q], gE);
                        }
                    }
                }
            });
        }
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
