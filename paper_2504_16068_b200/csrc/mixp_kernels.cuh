// mixp_kernels.cuh -- dense per-path channel mixing at l_max = 3 (ALLEGRO_W_DENSE; Table 1's medium / large models),
// the paths-outer kernels.  Included by inst_mixp.cu only (one translation unit per dtype and kernel).
#pragma once
#include "mix_kernels.cuh"

namespace allegro {

// 68 paths, 312 un-weighted path values per (edge, channel): they do not fit a thread's registers, so the loops are exchanged --
// PATHS OUTER, edges inner.  One CTA per item (a centre's run of at most `tile_edges` edges).  Per path p: W_p (forward) or W_p^T
// (VJP) is staged ONCE per item in shared memory; per tile of nsl x EPT edges thread (slot, n) computes the path's 2 l3 + 1
// un-weighted values of its edges into shared memory and thread (slot, n') adds the mixed values to ITS OWN out rows (a
// read-modify-write of rows that only this thread touches, so program order is the only ordering needed; the first path into a
// block writes).  The item's out / gV rows stay in L2 between paths.  Every sum has a fixed order.
template <typename Gen, int P0>
__host__ __device__ constexpr bool mixp_first_out(int p) {
    for (int q = 0; q < p; ++q)
        if (Gen::off3(q) == Gen::off3(p)) return false;
    return true;
}

// Register tile of a thread: R output rows (channels c0 + r nth, nth = n / R) x EPT edges x (2 l3 + 1) components.  Per group of
// four K columns a thread loads R 128-bit pieces of W rows and EPT x D3 pieces of staged values for 4 R EPT D3 FMAs; the shared-
// memory port (128 B / clk / SM) is what bounds these kernels, so bytes per FMA is the figure of merit.
#ifndef ALLEGRO_MIXP_R
#define ALLEGRO_MIXP_R 2
#endif
#ifndef ALLEGRO_MIXP_EPT
#define ALLEGRO_MIXP_EPT 4
#endif
template <typename T> struct MixpTile {
    static constexpr int R = sizeof(T) == 4 ? ALLEGRO_MIXP_R : 1;     // fp64: one row (the VJP already needs 254 registers)
    static constexpr int EPT = sizeof(T) == 4 ? ALLEGRO_MIXP_EPT : 4;
};

// acc[r][k][M] = <Ws[c0 + r nth][:], tS[slot + nsl k][M][:]>: rows of length n in shared memory, 128-bit loads
template <typename T, int D3, int D3MAX, int R, int EPT>
__device__ __forceinline__ void mixp_dots(const T* __restrict__ Ws, int ldw, int c0, int nth, const T* __restrict__ tS, int slot, int nsl, int n,
                                          T (&acc)[R][EPT][D3]) {
    constexpr int VEC = 16 / (int)sizeof(T);
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int k = 0; k < EPT; ++k)
#pragma unroll
            for (int M = 0; M < D3; ++M) acc[r][k][M] = T(0);
    for (int i = 0; i < n / VEC; ++i) {
        int4 wv[R];
#pragma unroll
        for (int r = 0; r < R; ++r) wv[r] = reinterpret_cast<const int4*>(Ws + (size_t)(c0 + r * nth) * ldw)[i];
#pragma unroll
        for (int k = 0; k < EPT; ++k)
#pragma unroll
            for (int M = 0; M < D3; ++M) {
                const int4 tv = reinterpret_cast<const int4*>(tS + ((size_t)(slot + nsl * k) * D3MAX + M) * n)[i];
                const T* ts = reinterpret_cast<const T*>(&tv);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const T* ws = reinterpret_cast<const T*>(&wv[r]);
#pragma unroll
                    for (int q = 0; q < VEC; ++q) acc[r][k][M] = fma(ws[q], ts[q], acc[r][k][M]);
                }
            }
    }
}

template <typename T, int L, int CT>
__global__ void __launch_bounds__(CT) mixp_fwd_kernel(int n, const int* __restrict__ row_ptr, const int* __restrict__ items,
                                                       const T* __restrict__ V, const T* __restrict__ Eenv, const T* __restrict__ W,
                                                       T* __restrict__ out) {
    using Gen = TPGen<L>;
    constexpr int DV = Gen::DV, DE = Gen::DE, P = Gen::P, D3MAX = 2 * L + 1, R = MixpTile<T>::R, EPT = MixpTile<T>::EPT;
    constexpr int VEC = 16 / (int)sizeof(T);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nth = n / R, nsl = CT / nth, te = nsl * EPT;   // a tile = te edges; thread (slot, c0) owns edges slot + nsl k, rows c0 + r nth
    T* Ws = reinterpret_cast<T*>(smem_raw);            // [n][n + VEC]
    const int ldw = n + VEC;
    T* tS = Ws + (size_t)n * ldw;                      // [te][D3MAX][n]
    const int tid = threadIdx.x;
    const int slot = tid / nth, c0 = tid - slot * nth;
    const bool active = slot < nsl;
    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    const int ntiles = (e1 - e0 + te - 1) / te;
    T E[R][DE];
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int j = 0; j < DE; ++j) E[r][j] = active ? Eenv[((size_t)c * n + c0 + r * nth) * DE + j] : T(0);

    static_for<0, P>([&](auto pc) {
        constexpr int p = decltype(pc)::value;
        using Pth = TPPath<L, p>;
        constexpr bool first = mixp_first_out<Gen, 0>(p);
        __syncthreads();                               // the previous path's Ws / tS are consumed
        for (int idx = tid; idx < n * n / VEC; idx += CT) {
            const int r = (idx * VEC) / n, cc = (idx * VEC) - r * n;
            *reinterpret_cast<int4*>(Ws + (size_t)r * ldw + cc) = *reinterpret_cast<const int4*>(W + (size_t)p * n * n + (size_t)idx * VEC);
        }
        for (int t = 0; t < ntiles; ++t) {
            const int eb = e0 + t * te + slot;
            if (t > 0) __syncthreads();                // tS consumed by the previous tile
            if (active) {
#pragma unroll
                for (int k = 0; k < EPT; ++k) {
                    const int e = eb + nsl * k;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const int ch = c0 + r * nth;
                        T tp[Pth::D3];
                        if (e < e1) {
                            Pth::template fwd<T>(V + ((size_t)e * n + ch) * DV, E[r], tp);
                        } else {
#pragma unroll
                            for (int M = 0; M < Pth::D3; ++M) tp[M] = T(0);
                        }
#pragma unroll
                        for (int M = 0; M < Pth::D3; ++M) tS[((size_t)(slot + nsl * k) * D3MAX + M) * n + ch] = tp[M];
                    }
                }
            }
            __syncthreads();
            if (active) {
                T acc[R][EPT][Pth::D3];
                mixp_dots<T, Pth::D3, D3MAX, R, EPT>(Ws, ldw, c0, nth, tS, slot, nsl, n, acc);
#pragma unroll
                for (int k = 0; k < EPT; ++k) {
                    const int e = eb + nsl * k;
                    if (e < e1) {
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            T* dst = out + ((size_t)e * n + c0 + r * nth) * DV + Pth::OFF3;
#pragma unroll
                            for (int M = 0; M < Pth::D3; ++M) dst[M] = first ? acc[r][k][M] : dst[M] + acc[r][k][M];
                        }
                    }
                }
            }
        }
    });
}

// first path (in path order) that reads input block OFF1 of path p: it writes the gV block, later ones add
template <int L, int Q, int PP>
struct MixpFirstGv {
    static constexpr bool value = (TPPath<L, Q>::OFF1 != TPPath<L, PP>::OFF1) && MixpFirstGv<L, Q + 1, PP>::value;
};
template <int L, int PP>
struct MixpFirstGv<L, PP, PP> {
    static constexpr bool value = true;
};

template <typename T, int L, int CT, bool WANT_GV>
__global__ void __launch_bounds__(CT) mixp_bwd_kernel(int n, const int* __restrict__ row_ptr, const int* __restrict__ items,
                                                       const T* __restrict__ G, const T* __restrict__ V, const T* __restrict__ Eenv,
                                                       const T* __restrict__ W, T* __restrict__ gV, T* __restrict__ gE_dst, int gE_by_item) {
    using Gen = TPGen<L>;
    constexpr int DV = Gen::DV, DE = Gen::DE, P = Gen::P, D3MAX = 2 * L + 1, R = MixpTile<T>::R, EPT = MixpTile<T>::EPT;
    constexpr int VEC = 16 / (int)sizeof(T);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nth = n / R, nsl = CT / nth, te = nsl * EPT;
    T* WsT = reinterpret_cast<T*>(smem_raw);           // [n][n + VEC], WsT[a][b] = W_p[b][a]
    const int ldw = n + VEC;
    T* gS = WsT + (size_t)n * ldw;                     // [te][D3MAX][n]
    const int tid = threadIdx.x;
    const int slot = tid / nth, c0 = tid - slot * nth;
    const bool active = slot < nsl;
    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    const int ntiles = (e1 - e0 + te - 1) / te;
    T E[R][DE], gE[R][DE];
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int j = 0; j < DE; ++j) { E[r][j] = active ? Eenv[((size_t)c * n + c0 + r * nth) * DE + j] : T(0); gE[r][j] = T(0); }

    static_for<0, P>([&](auto pc) {
        constexpr int p = decltype(pc)::value;
        using Pth = TPPath<L, p>;
        constexpr bool first = MixpFirstGv<L, 0, p>::value;
        __syncthreads();
        for (int idx = tid; idx < n * n / VEC; idx += CT) {
            const int r = (idx * VEC) / n, cc = (idx * VEC) - r * n;  // W_p[r][cc .. cc+VEC)
            const int4 wv = *reinterpret_cast<const int4*>(W + (size_t)p * n * n + (size_t)idx * VEC);
            const T* ws = reinterpret_cast<const T*>(&wv);
#pragma unroll
            for (int k = 0; k < VEC; ++k) WsT[(size_t)(cc + k) * ldw + r] = ws[k];
        }
        for (int t = 0; t < ntiles; ++t) {
            const int eb = e0 + t * te + slot;
            if (t > 0) __syncthreads();
            if (active) {
#pragma unroll
                for (int k = 0; k < EPT; ++k) {
                    const int e = eb + nsl * k;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const int ch = c0 + r * nth;
                        const T* grow = G + ((size_t)e * n + ch) * DV + Pth::OFF3;
#pragma unroll
                        for (int M = 0; M < Pth::D3; ++M) gS[((size_t)(slot + nsl * k) * D3MAX + M) * n + ch] = e < e1 ? grow[M] : T(0);
                    }
                }
            }
            __syncthreads();
            if (active) {
                T gt[R][EPT][Pth::D3];
                mixp_dots<T, Pth::D3, D3MAX, R, EPT>(WsT, ldw, c0, nth, gS, slot, nsl, n, gt);
#pragma unroll
                for (int k = 0; k < EPT; ++k) {
                    const int e = eb + nsl * k;
                    if (e < e1) {
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const int ch = c0 + r * nth;
                            T gv[Pth::D1];
                            Pth::template bwd_local<T, WANT_GV>(V + ((size_t)e * n + ch) * DV, E[r], gt[r][k], gv, gE[r]);
                            if constexpr (WANT_GV) {
                                T* dst = gV + ((size_t)e * n + ch) * DV + Pth::OFF1;
#pragma unroll
                                for (int i = 0; i < Pth::D1; ++i) dst[i] = first ? gv[i] : dst[i] + gv[i];
                            }
                        }
                    }
                }
            }
        }
    });
    // ---- gEenv: slots summed in slot order
    T* red = reinterpret_cast<T*>(smem_raw);
    __syncthreads();
    if (active) {
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int j = 0; j < DE; ++j) red[((size_t)slot * n + c0 + r * nth) * DE + j] = gE[r][j];
    }
    __syncthreads();
    if (slot == 0) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int ch = c0 + r * nth;
            T* dst = gE_dst + ((size_t)(gE_by_item ? (long)blockIdx.x : (long)c) * n + ch) * DE;
#pragma unroll
            for (int j = 0; j < DE; ++j) {
                T acc = red[(size_t)ch * DE + j];
                for (int sl = 1; sl < nsl; ++sl) acc += red[((size_t)sl * n + ch) * DE + j];
                dst[j] = acc;
            }
        }
    }
}

// shared memory of the paths-outer kernels: one n x (n + VEC) weight image + nsl x (2 L + 1) x n staged values (and, in the VJP,
// at least the CT x DE reduction rows that reuse the buffer)
template <typename T, int L_>
static size_t mixp_smem(int n, int CT) {
    constexpr int VEC = 16 / (int)sizeof(T);
    const int nsl = CT / (n / MixpTile<T>::R);
    const size_t b = ((size_t)n * (n + VEC) + (size_t)nsl * MixpTile<T>::EPT * (2 * L_ + 1) * n) * sizeof(T);
    const size_t red = (size_t)nsl * n * TPGen<L_>::DE * sizeof(T);
    return b > red ? b : red;
}

}  // namespace allegro
