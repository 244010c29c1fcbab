// tp_kernels.cuh -- the Allegro tensor product and its first derivative, scalar path
// weights.  Included by inst_tp.cu once per (ALLEGRO_T, ALLEGRO_L).
//
// Mapping (sm_100a):
//   * one CTA per segment-plan item = (centre c, edges e0..e1) (A16).  A centre's edges are contiguous
//     (CSR), so its feature rows V[e0..e1) are ONE contiguous byte range.
//   * thread <-> (edge slot, channel): THREADS / n slots of n channels.  The centre's environment row
//     Eenv[c][ch][:] stays in registers for the whole segment (north_star: "staging of each center
//     atom's environment tile, which is reused across its neighbour edges").
//   * V (and G) tiles of `nslots` edges stream through an NST-stage shared-memory ring filled by 1-D
//     bulk async copies (cp.async.bulk + mbarrier complete_tx; SASS UBLKCP).  A thread reads its
//     channel row with 64/128-bit LDS, runs the generated, fully unrolled sparse CG contraction
//     (coefficients = constant-bank FFMA operands), writes the result row back IN PLACE and one thread
//     issues the bulk store of the whole tile (shared -> global).  The outer product V (x) Eenv never
//     exists anywhere.
//   * no float atomics: the per-centre sums of gEenv run over slots in a fixed order.
#pragma once
#include "common.cuh"
#include "launch.h"

namespace allegro {

// NOTE: l_max is a template parameter of every kernel here.  The translation units inst_tp.cu (one per
// l_max) would otherwise instantiate kernels with identical mangled names and different bodies, and the
// linker keeps one of them (ODR): the wrong l_max's code would run.
static_assert(TPGen<ALLEGRO_L>::NNZ <= kCwMax, "coefficient table too small");

// ------------------------------------------------------------------------------------------------
// fold: cw[z] = path_w[path(z)] * C_z  (the "combined tensor"), product in double, rounded once
template <typename T, int L>
__global__ void fold_kernel(const T* __restrict__ path_w, T* __restrict__ cw) {
    using Gen = TPGen<L>;
    const int z = blockIdx.x * blockDim.x + threadIdx.x;
    if (z < Gen::NNZ) cw[z] = (T)((double)path_w[Gen::zpath(z)] * Gen::zcoef(z));
}

// ------------------------------------------------------------------------------------------------
// Energy epilogue (reading A12), fused so that `out` is never re-read from HBM:
//   e_edge[e] = sum_ch ( q[ch] out[e][ch][0] + kappa/2 sum_k out[e][ch][k]^2 ),   G = q (x) delta_{k,0} + kappa out
// WANT_OUT / WANT_G / WANT_E select which of out, G, e_edge are produced (at least one of out, G).
// Shared memory: NST stages of V (each becomes the out tile, or the G tile when !WANT_OUT, in place), then
// 3 G tiles when both out and G are stored, then the mbarriers, then the energy partials.
template <typename T, int L, int THREADS, int NST, bool WANT_OUT, bool WANT_G, bool WANT_E>
__global__ void __launch_bounds__(THREADS) tp_fwd_kernel(int n, const int* __restrict__ row_ptr, const int* __restrict__ items,
                                                          const T* __restrict__ V, const T* __restrict__ Eenv, T* __restrict__ out,
                                                          const T* __restrict__ q, T kappa, T* __restrict__ e_edge, T* __restrict__ G) {
    using Gen = TPGen<L>;
    constexpr int DV = Gen::DV, DE = Gen::DE;
    constexpr bool EPI = WANT_G || WANT_E;
    constexpr bool GBUF = WANT_OUT && WANT_G;  // separate G tiles
    static_assert(WANT_OUT || WANT_G, "nothing to store");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nslots = THREADS / n;
    const int slot = tid / n, ch = tid - slot * n;
    const bool active = slot < nslots;
    const uint32_t row_bytes = (uint32_t)n * DV * sizeof(T);
    const uint32_t stage_bytes = align128((size_t)nslots * row_bytes);
    unsigned char* gbuf = smem_raw + (size_t)NST * stage_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(gbuf + (GBUF ? 3 : 0) * (size_t)stage_bytes);
    T* ered = reinterpret_cast<T*>(reinterpret_cast<unsigned char*>(bars) + 64);  // [2][THREADS / 32] or [2][THREADS]

    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    const int ntiles = (e1 - e0 + nslots - 1) / nslots;
    if (ntiles <= 0) return;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s) mbar_init(&bars[s], 1);
        fence_mbar_init();
    }
    __syncthreads();

    auto issue = [&](int t) {
        const int s = t % NST;
        const int eb = e0 + t * nslots;
        const uint32_t bytes = (uint32_t)min(nslots, e1 - eb) * row_bytes;
        mbar_expect_tx(&bars[s], bytes);
        bulk_load(smem_raw + (size_t)s * stage_bytes, V + (size_t)eb * n * DV, bytes, &bars[s]);
    };
    if (tid == 0) {
        const int pre = ntiles < NST ? ntiles : NST;
        for (int t = 0; t < pre; ++t) issue(t);
    }

    T E[DE];
    T qc = T(0);
    if (active) {
        const T* er = Eenv + ((size_t)c * n + ch) * DE;
#pragma unroll
        for (int j = 0; j < DE; ++j) E[j] = er[j];
        if constexpr (EPI) qc = q[ch];
    } else {
#pragma unroll
        for (int j = 0; j < DE; ++j) E[j] = T(0);
    }
    // how the per-edge energy is summed over the slot's n channels (fixed shape): whole warps -> xor tree + the
    // slot's warps in order; n a power of two below 32 -> xor tree inside the slot's lanes; otherwise channels in order
    const bool warp_tree = (n % 32) == 0;
    const bool sub_tree = n < 32 && (n & (n - 1)) == 0;

    for (int t = 0; t < ntiles; ++t) {
        const int s = t % NST;
        mbar_wait(&bars[s], (uint32_t)(t / NST) & 1u);
        const int eb = e0 + t * nslots;
        const bool valid = active && eb + slot < e1;
        T epart = T(0);
        if (valid) {
            T* row = reinterpret_cast<T*>(smem_raw + (size_t)s * stage_bytes) + ((size_t)slot * n + ch) * DV;
            T v[DV], o[DV];
            row_load<T, DV>(row, v);
            Gen::template fwd<T>(v, E, o);
            if constexpr (WANT_OUT) row_store<T, DV>(row, o);
            if constexpr (EPI) {
                T sq = T(0);
#pragma unroll
                for (int k = 0; k < DV; ++k) sq = fma(o[k], o[k], sq);
                epart = fma(T(0.5) * kappa, sq, qc * o[0]);
                if constexpr (WANT_G) {
#pragma unroll
                    for (int k = 0; k < DV; ++k) o[k] *= kappa;
                    o[0] += qc;
                    T* grow = GBUF ? reinterpret_cast<T*>(gbuf + (size_t)(t % 3) * stage_bytes) + ((size_t)slot * n + ch) * DV : row;
                    row_store<T, DV>(grow, o);
                }
            }
        }
        if constexpr (WANT_E) {
            T* er2 = ered + (size_t)(t & 1) * THREADS;
            if (warp_tree) {
#pragma unroll
                for (int o2 = 16; o2 > 0; o2 >>= 1) epart += __shfl_xor_sync(0xffffffffu, epart, o2);
                if (lane == 0) er2[warp] = epart;
            } else if (sub_tree) {
                for (int o2 = n >> 1; o2 > 0; o2 >>= 1) epart += __shfl_xor_sync(0xffffffffu, epart, o2);
                if (ch == 0 && active) er2[slot] = epart;
            } else {
                er2[tid] = epart;
            }
        }
        fence_proxy_async();
        __syncthreads();
        if constexpr (WANT_E) {
            if (valid && ch == 0) {
                const T* er2 = ered + (size_t)(t & 1) * THREADS;
                T acc;
                if (warp_tree) {
                    const int wps = n >> 5;
                    acc = er2[slot * wps];
                    for (int k = 1; k < wps; ++k) acc += er2[slot * wps + k];
                } else if (sub_tree) {
                    acc = er2[slot];
                } else {
                    acc = er2[slot * n];
                    for (int k = 1; k < n; ++k) acc += er2[slot * n + k];
                }
                e_edge[eb + slot] = acc;
            }
        }
        if (tid == 0) {
            const uint32_t bytes = (uint32_t)min(nslots, e1 - eb) * row_bytes;
            if constexpr (WANT_OUT) bulk_store(out + (size_t)eb * n * DV, smem_raw + (size_t)s * stage_bytes, bytes);
            if constexpr (WANT_G)
                bulk_store(G + (size_t)eb * n * DV, GBUF ? gbuf + (size_t)(t % 3) * stage_bytes : smem_raw + (size_t)s * stage_bytes, bytes);
            bulk_commit();  // one group per tile: the out and G stores of tile t
            if constexpr (NST == 1) {
                if (t + 1 < ntiles) { bulk_wait_read<0>(); issue(t + 1); }  // single stage: store, then refill
            } else if (t >= 1 && t - 1 + NST < ntiles) {
                bulk_wait_read<1>();  // the stores of tile t-1 have finished reading their stage (and G tile (t-1) % 3)
                issue(t - 1 + NST);
            } else if (GBUF && t >= 1) {
                bulk_wait_read<1>();  // G tile (t-1) % 3 is written again by tile t+2
            }
        }
    }
    if (tid == 0) bulk_wait_read<0>();
}

// ------------------------------------------------------------------------------------------------
// First derivative.  Stage = [G tile | V tile]; gV overwrites the G tile in place and is
// bulk-stored; gEenv accumulates in registers over the thread's edges, then over slots in slot order.
// WANT_GW adds the path-weight gradient: per-thread accumulators -> fixed-shape warp tree -> warps in
// order -> one partial row per item (reduced over items by gw_final_kernel).
template <typename T, int L, int THREADS, int NST, bool WANT_GV, bool WANT_GW>
__global__ void __launch_bounds__(THREADS)
    tp_bwd_kernel(int n, const int* __restrict__ row_ptr, const int* __restrict__ items, const T* __restrict__ G, const T* __restrict__ V,
                  const T* __restrict__ Eenv, T* __restrict__ gV, T* __restrict__ gE_dst, int gE_by_item, T* __restrict__ gw_part) {
    using Gen = TPGen<L>;
    constexpr int DV = Gen::DV, DE = Gen::DE, P = Gen::P;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x;
    const int nslots = THREADS / n;
    const int slot = tid / n, ch = tid - slot * n;
    const bool active = slot < nslots;
    const uint32_t row_bytes = (uint32_t)n * DV * sizeof(T);
    const uint32_t tile_bytes = align128((size_t)nslots * row_bytes);
    const uint32_t stage_bytes = 2 * tile_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + (size_t)NST * stage_bytes);
    T* red = reinterpret_cast<T*>(smem_raw + (size_t)NST * stage_bytes + 128);  // [THREADS][DE] or [warps][P]

    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    const int ntiles = (e1 - e0 + nslots - 1) / nslots;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s) mbar_init(&bars[s], 1);
        fence_mbar_init();
    }
    __syncthreads();

    auto issue = [&](int t) {
        const int s = t % NST;
        const int eb = e0 + t * nslots;
        const uint32_t bytes = (uint32_t)min(nslots, e1 - eb) * row_bytes;
        unsigned char* st = smem_raw + (size_t)s * stage_bytes;
        mbar_expect_tx(&bars[s], 2 * bytes);
        bulk_load(st, G + (size_t)eb * n * DV, bytes, &bars[s]);
        bulk_load(st + tile_bytes, V + (size_t)eb * n * DV, bytes, &bars[s]);
    };
    if (tid == 0) {
        const int pre = ntiles < NST ? ntiles : NST;
        for (int t = 0; t < pre; ++t) issue(t);
    }

    T E[DE], gE[DE];
#pragma unroll
    for (int j = 0; j < DE; ++j) { E[j] = T(0); gE[j] = T(0); }
    if (active) {
        const T* er = Eenv + ((size_t)c * n + ch) * DE;
#pragma unroll
        for (int j = 0; j < DE; ++j) E[j] = er[j];
    }
    T gw[WANT_GW ? P : 1];
#pragma unroll
    for (int p = 0; p < (WANT_GW ? P : 1); ++p) gw[p] = T(0);

    for (int t = 0; t < ntiles; ++t) {
        const int s = t % NST;
        mbar_wait(&bars[s], (uint32_t)(t / NST) & 1u);
        const int eb = e0 + t * nslots;
        unsigned char* st = smem_raw + (size_t)s * stage_bytes;
        if (active && eb + slot < e1) {
            T* grow = reinterpret_cast<T*>(st) + ((size_t)slot * n + ch) * DV;
            const T* vrow = reinterpret_cast<const T*>(st + tile_bytes) + ((size_t)slot * n + ch) * DV;
            T v[DV], g[DV], gv[DV];
            row_load<T, DV>(grow, g);
            row_load<T, DV>(vrow, v);
            Gen::template bwd<T, WANT_GV>(v, E, g, gv, gE);
            if constexpr (WANT_GW) Gen::template pathw<T>(v, E, g, gw);
            if constexpr (WANT_GV) row_store<T, DV>(grow, gv);
        }
        if constexpr (WANT_GV) fence_proxy_async();
        __syncthreads();
        if (tid == 0) {
            if constexpr (WANT_GV) {
                const uint32_t bytes = (uint32_t)min(nslots, e1 - eb) * row_bytes;
                bulk_store(gV + (size_t)eb * n * DV, st, bytes);
                bulk_commit();
                if constexpr (NST == 1) {
                    if (t + 1 < ntiles) { bulk_wait_read<0>(); issue(t + 1); }
                } else if (t >= 1 && t - 1 + NST < ntiles) {
                    bulk_wait_read<1>();
                    issue(t - 1 + NST);
                }
            } else {
                if (t + NST < ntiles) issue(t + NST);  // every thread is done with stage s
            }
        }
    }

    // ---- gEenv: slots summed in slot order
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
            for (int sl = 1; sl < nslots; ++sl) acc += red[((size_t)sl * n + ch) * DE + j];
            dst[j] = acc;
        }
    }
    if constexpr (WANT_GW) {
        __syncthreads();
        const int lane = tid & 31, warp = tid >> 5;
#pragma unroll
        for (int p = 0; p < P; ++p) {
            T a = gw[p];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
            if (lane == 0) red[warp * P + p] = a;
        }
        __syncthreads();
        if (tid < P) {
            T acc = red[tid];
            for (int wv = 1; wv < THREADS / 32; ++wv) acc += red[wv * P + tid];
            gw_part[(size_t)blockIdx.x * P + tid] = acc;
        }
    }
    if constexpr (WANT_GV) {
        if (tid == 0) bulk_wait_read<0>();
    }
}

// g_path_w[p] = sum over items of the partial rows: each thread adds a strided subset in order (double),
// then a fixed-shape shared-memory tree.  One CTA per path.
template <typename T>
__global__ void __launch_bounds__(256) gw_final_kernel(const T* __restrict__ gw_part, long n_items, int P, T* __restrict__ g_path_w) {
    __shared__ double sh[256];
    const int p = blockIdx.x;
    double acc = 0.0;
    for (long it = threadIdx.x; it < n_items; it += 256) acc += (double)gw_part[(size_t)it * P + p];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) g_path_w[p] = (T)sh[0];
}

}  // namespace allegro
