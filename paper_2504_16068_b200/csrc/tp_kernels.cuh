// tp_kernels.cuh -- the Allegro tensor product and its first derivative, scalar path
// weights.  Included by inst_tp.cu once per (ALLEGRO_T, ALLEGRO_L).
//
// Mapping (sm_100a):
//   * one CTA per segment-plan item = (centre c, edges e0..e1) (A16).  A centre's edges are contiguous
//     (CSR), so its feature rows V[e0..e1) are ONE contiguous byte range.
//   * warp-specialised: CT compute threads + one producer warp.  The producer's elected lane streams tiles
//     of `nslots` edges through an NST-stage shared-memory ring with 1-D bulk async copies (cp.async.bulk +
//     mbarrier complete_tx; SASS UBLKCP), issues the bulk stores of finished tiles and refills a stage as
//     soon as its store has been read out.  Compute warps only ever wait on a "full" mbarrier and signal
//     "done" with one arrive per warp: there is no block-wide barrier in the steady state, so warps drift
//     apart by up to NST tiles and HBM latency is covered by the ring, not by occupancy.
//   * compute thread <-> (edge slot, channel): CT / n slots of n channels.  The centre's environment row
//     Eenv[c][ch][:] stays in registers for the whole segment (north_star: "staging of each center
//     atom's environment tile, which is reused across its neighbour edges").  A thread reads its channel
//     row with 64/128-bit LDS, runs the generated, fully unrolled sparse CG contraction (coefficients =
//     constant-bank FFMA operands) and writes the result row back IN PLACE.  The outer product V (x) Eenv
//     never exists anywhere.
//   * no float atomics: every reduction has a fixed shape (xor trees, then warps / slots in order).
//
// NOTE: l_max is a template parameter of every kernel here.  The translation units inst_tp.cu (one per
// l_max) would otherwise instantiate kernels with identical mangled names and different bodies, and the
// linker keeps one of them (ODR): the wrong l_max's code would run.
#pragma once
#include "common.cuh"
#include "launch.h"

namespace allegro {

// The folded coefficient table ("combined tensor" Wc = sum_p path_w[p] C^p) travels BY VALUE as a __grid_constant__
// kernel parameter: every coefficient is a constant-bank operand of its FFMA/DFMA (no register, no load instruction), and two
// launches -- different plans, different weights, different streams -- never share state.  Folded on the host when the weights
// are bound (allegro_plan_bind_weights); 1.1 KB (l_max 2, fp32) .. 9.8 KB (l_max 3, fp64) of the 32 KB parameter space.
template <typename T, int NNZ>
struct CwTab {
    T v[NNZ];
};

// Tensor maps of the swizzled variant (SW: feature rows of exactly 128 bytes, i.e. l_max = 3 in fp32): every feature tensor is a
// 2-D array [E n rows][32 floats], box = one edge (n rows), 128-byte swizzle.  a = V, b = the tensor that is stored (out / gV),
// c = the second stored tensor of the forward (G) or the cotangent that the VJP loads (G / out).  Unused (zero) when !SW.
struct alignas(64) TpMaps {
    CUtensorMap a, b, c;
};

// ------------------------------------------------------------------------------------------------
// The tile ring shared by the kernels below.  A stage holds TILES tiles of `tile_bytes` (tile 0 is
// overwritten in place by the result that is stored back).  full[s]: the stage's loads have landed
// (transaction count); done[s]: all compute warps have finished with the stage (one arrive per warp).
struct Ring {
    unsigned char* base;
    uint64_t* full;
    uint64_t* done;
    uint32_t tile_bytes, stage_bytes;
    __device__ __forceinline__ unsigned char* stage(int s) const { return base + (size_t)s * stage_bytes; }
};

__device__ __forceinline__ void ring_init(const Ring& r, int tid, int compute_warps, int NST) {
    if (tid == 0) {
        for (int s = 0; s < NST; ++s) { mbar_init(&r.full[s], 1); mbar_init(&r.done[s], compute_warps); }
        fence_mbar_init();
    }
    __syncthreads();
}

// compute side: every lane has written its rows; make them visible to the async proxy, then one arrive per warp
__device__ __forceinline__ void ring_release(uint64_t* done_bar, int lane) {
    fence_proxy_async();
    __syncwarp();
    if (lane == 0) mbar_arrive(done_bar);
}

// how a per-edge quantity is summed over the n channel threads of a slot (fixed shape -> deterministic)
//   n % 32 == 0             : xor tree inside each warp, then the slot's warps in order (named barrier per slot)
//   n power of two below 32 : xor tree inside the slot's lanes
//   otherwise               : the slot's channels in order (named barrier over all compute threads)
enum { SUM_WARPS = 0, SUM_SUB = 1, SUM_SERIAL = 2 };
__device__ __forceinline__ int slot_sum_mode(int n) { return (n % 32) == 0 ? SUM_WARPS : ((n < 32 && (n & (n - 1)) == 0) ? SUM_SUB : SUM_SERIAL); }

// returns the slot total in the thread with ch == 0 (other threads: unspecified).  `buf` holds 2 * CT values
// (double-buffered by tile parity so that a fast warp cannot overwrite partials that are still being read).
template <typename T, int CT>
__device__ __forceinline__ T slot_sum(T x, int mode, int n, int slot, int ch, int tid, int t, T* buf) {
    T* b = buf + (size_t)(t & 1) * CT;
    const int lane = tid & 31, warp = tid >> 5;
    if (mode == SUM_WARPS) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        const int wps = n >> 5;
        if (wps == 1 || (slot + 1) * n > CT) return x;   // leftover threads (CT % n != 0) own no slot: they must not join a slot's barrier
        if (lane == 0) b[warp] = x;
        named_bar(1 + slot, n);
        if (ch == 0) {
            x = b[slot * wps];
            for (int k = 1; k < wps; ++k) x += b[slot * wps + k];
        }
        return x;
    } else if (mode == SUM_SUB) {
        for (int o = n >> 1; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        return x;
    } else {
        b[tid] = x;
        named_bar(1, CT);
        if (ch == 0 && slot * n + n <= CT) {
            x = b[slot * n];
            for (int k = 1; k < n; ++k) x += b[slot * n + k];
        }
        return x;
    }
}

// ------------------------------------------------------------------------------------------------
// Forward, optionally with the energy epilogue of reading A12 fused so that `out` is never
// re-read from HBM:
//   e_edge[e] = sum_ch ( q[ch] out[e][ch][0] + kappa/2 sum_k out[e][ch][k]^2 ),   G = q (x) delta_{k,0} + kappa out
// WANT_OUT / WANT_G / WANT_E select which of out, G, e_edge are produced (at least one of out, G).
// Stage = [V tile -> out tile (or G tile when !WANT_OUT)] [G tile when both are stored].
template <typename T, int L, int CT, bool WANT_OUT, bool WANT_G, bool WANT_E, bool SW>
__global__ void __launch_bounds__(CT + 32, 2) tp_fwd_kernel(const __grid_constant__ CwTab<T, TPGen<L>::NNZ> cwt, const __grid_constant__ TpMaps tm, int NST, int n, const int* __restrict__ row_ptr, const int* __restrict__ items,
                                                          const T* __restrict__ V, const T* __restrict__ Eenv, T* __restrict__ out,
                                                          const T* __restrict__ q, T kappa, T* __restrict__ e_edge, T* __restrict__ G) {
    using Gen = TPGen<L>;
    constexpr int DV = Gen::DV, DE = Gen::DE;
    constexpr bool EPI = WANT_G || WANT_E;
    constexpr int TILES = (WANT_OUT && WANT_G) ? 2 : 1;
    static_assert(WANT_OUT || WANT_G, "nothing to store");
    extern __shared__ __align__(128) unsigned char smem_dyn[];
    unsigned char* smem_raw = SW ? smem_dyn + ((1024u - (smem_u32(smem_dyn) & 1023u)) & 1023u) : smem_dyn;   // swizzle atoms are 1024-byte aligned
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nslots = CT / n;
    const uint32_t row_bytes = (uint32_t)n * DV * sizeof(T);
    Ring r;
    r.base = smem_raw;
    r.tile_bytes = align128((size_t)nslots * row_bytes);
    r.stage_bytes = TILES * r.tile_bytes;
    r.full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)NST * r.stage_bytes);
    r.done = r.full + NST;
    T* ebuf = reinterpret_cast<T*>(r.done + NST);  // [2][CT]

    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    const int ntiles = (e1 - e0 + nslots - 1) / nslots;
    if (ntiles <= 0) return;
    ring_init(r, tid, CT / 32, NST);

    if (warp == CT / 32) {
        // ---------------------------------------------------------------- producer
        if (lane != 0) return;
        auto issue = [&](int t) {
            const int s = t % NST;
            const int eb = e0 + t * nslots;
            const int ne = min(nslots, e1 - eb);
            const uint32_t bytes = (uint32_t)ne * row_bytes;
            mbar_expect_tx(&r.full[s], bytes);
            if constexpr (SW) {
                for (int i = 0; i < ne; ++i) tma_load_2d(r.stage(s) + (size_t)i * row_bytes, &tm.a, 0, (eb + i) * n, &r.full[s]);
            } else {
                bulk_load(r.stage(s), V + (size_t)eb * n * DV, bytes, &r.full[s]);
            }
        };
        const int pre = ntiles < NST ? ntiles : NST;
        for (int t = 0; t < pre; ++t) issue(t);
        for (int u = 0; u < ntiles; ++u) {
            const int s = u % NST;
            mbar_wait(&r.done[s], (uint32_t)(u / NST) & 1u);
            const int eb = e0 + u * nslots;
            const int ne = min(nslots, e1 - eb);
            const uint32_t bytes = (uint32_t)ne * row_bytes;
            if constexpr (SW) {
                for (int i = 0; i < ne; ++i) {
                    if constexpr (WANT_OUT) tma_store_2d(&tm.b, 0, (eb + i) * n, r.stage(s) + (size_t)i * row_bytes);
                    if constexpr (WANT_G) tma_store_2d(&tm.c, 0, (eb + i) * n, r.stage(s) + (TILES - 1) * r.tile_bytes + (size_t)i * row_bytes);
                }
            } else {
                if constexpr (WANT_OUT) bulk_store(out + (size_t)eb * n * DV, r.stage(s), bytes);
                if constexpr (WANT_G) bulk_store(G + (size_t)eb * n * DV, r.stage(s) + (TILES - 1) * r.tile_bytes, bytes);
            }
            bulk_commit();  // one group per tile
            if (NST == 1) {
                if (u + 1 < ntiles) { bulk_wait_read<0>(); issue(u + 1); }
            } else if (u >= 1 && u - 1 + NST < ntiles) {
                bulk_wait_read<1>();  // the stores of tile u-1 have finished reading their stage
                issue(u - 1 + NST);
            }
        }
        bulk_wait_read<0>();  // shared memory must outlive the last store's read
        return;
    }

    // -------------------------------------------------------------------- compute warps
    const int slot = tid / n, ch = tid - slot * n;
    const bool active = slot < nslots;
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
    const int mode = slot_sum_mode(n);

    for (int t = 0; t < ntiles; ++t) {
        const int s = t % NST;
        mbar_wait(&r.full[s], (uint32_t)(t / NST) & 1u);
        const int eb = e0 + t * nslots;
        const bool valid = active && eb + slot < e1;
        T epart = T(0);
        if (valid) {
            T* row = reinterpret_cast<T*>(r.stage(s)) + ((size_t)slot * n + ch) * DV;
            [[maybe_unused]] const uint32_t sw = ((uint32_t)(slot * n + ch) & 7u) << 4;
            T v[DV], o[DV];
            if constexpr (SW) row_load_sw<T, DV>(reinterpret_cast<const unsigned char*>(row), sw, v);
            else row_load<T, DV>(row, v);
            Gen::template fwd<T>(cwt.v, v, E, o);
            if constexpr (WANT_OUT) {
                if constexpr (SW) row_store_sw<T, DV>(reinterpret_cast<unsigned char*>(row), sw, o);
                else row_store<T, DV>(row, o);
            }
            if constexpr (EPI) {
                T sq = T(0);
#pragma unroll
                for (int k = 0; k < DV; ++k) sq = fma(o[k], o[k], sq);
                epart = fma(T(0.5) * kappa, sq, qc * o[0]);
                if constexpr (WANT_G) {
#pragma unroll
                    for (int k = 0; k < DV; ++k) o[k] *= kappa;
                    o[0] += qc;
                    if constexpr (SW) row_store_sw<T, DV>(reinterpret_cast<unsigned char*>(row) + (TILES - 1) * r.tile_bytes, sw, o);
                    else row_store<T, DV>(reinterpret_cast<T*>(reinterpret_cast<unsigned char*>(row) + (TILES - 1) * r.tile_bytes), o);
                }
            }
        }
        ring_release(&r.done[s], lane);
        if constexpr (WANT_E) {
            const T tot = slot_sum<T, CT>(epart, mode, n, slot, ch, tid, t, ebuf);
            if (valid && ch == 0) e_edge[eb + slot] = tot;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// First derivative.  Stage = [G tile | V tile]; gV overwrites the G tile in place and is
// bulk-stored; gEenv accumulates in registers over the thread's edges, then over slots in slot order.
// COT: tile 0 is loaded from `out` instead of G and the cotangent of the A12 energy, G = q (x) delta_{k,0} +
// kappa out, is formed in registers (G never exists in HBM).
// WANT_GW adds the path-weight gradient: per-thread accumulators -> fixed-shape warp tree -> warps in
// order -> one partial row per item (reduced over items by gw_final_kernel).
template <typename T, int L, int CT, bool WANT_GV, bool WANT_GW, bool COT, bool SW>
__global__ void __launch_bounds__(CT + 32)
    tp_bwd_kernel(const __grid_constant__ CwTab<T, TPGen<L>::NNZ> cwt, const __grid_constant__ TpMaps tm, int NST, int n, const int* __restrict__ row_ptr, const int* __restrict__ items, const T* __restrict__ G, const T* __restrict__ V,
                  const T* __restrict__ Eenv, const T* __restrict__ q, T kappa, T* __restrict__ gV, T* __restrict__ gE_dst, int gE_by_item,
                  T* __restrict__ gw_part) {
    using Gen = TPGen<L>;
    constexpr int DV = Gen::DV, DE = Gen::DE, P = Gen::P;
    extern __shared__ __align__(128) unsigned char smem_dyn[];
    unsigned char* smem_raw = SW ? smem_dyn + ((1024u - (smem_u32(smem_dyn) & 1023u)) & 1023u) : smem_dyn;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nslots = CT / n;
    const uint32_t row_bytes = (uint32_t)n * DV * sizeof(T);
    Ring r;
    r.base = smem_raw;
    r.tile_bytes = align128((size_t)nslots * row_bytes);
    r.stage_bytes = 2 * r.tile_bytes;
    r.full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)NST * r.stage_bytes);
    r.done = r.full + NST;

    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    const int ntiles = (e1 - e0 + nslots - 1) / nslots;
    ring_init(r, tid, CT / 32, NST);

    const bool compute = warp < CT / 32;
    const int slot = tid / n, ch = tid - slot * n;
    const bool active = compute && slot < nslots;
    T gE[DE];
#pragma unroll
    for (int j = 0; j < DE; ++j) gE[j] = T(0);
    T gw[WANT_GW ? P : 1];
#pragma unroll
    for (int p = 0; p < (WANT_GW ? P : 1); ++p) gw[p] = T(0);

    if (!compute) {
        // ---------------------------------------------------------------- producer
        if (lane == 0) {
            auto issue = [&](int t) {
                const int s = t % NST;
                const int eb = e0 + t * nslots;
                const int ne = min(nslots, e1 - eb);
                const uint32_t bytes = (uint32_t)ne * row_bytes;
                mbar_expect_tx(&r.full[s], 2 * bytes);
                if constexpr (SW) {
                    for (int i = 0; i < ne; ++i) {
                        tma_load_2d(r.stage(s) + (size_t)i * row_bytes, &tm.c, 0, (eb + i) * n, &r.full[s]);
                        tma_load_2d(r.stage(s) + r.tile_bytes + (size_t)i * row_bytes, &tm.a, 0, (eb + i) * n, &r.full[s]);
                    }
                } else {
                    bulk_load(r.stage(s), G + (size_t)eb * n * DV, bytes, &r.full[s]);
                    bulk_load(r.stage(s) + r.tile_bytes, V + (size_t)eb * n * DV, bytes, &r.full[s]);
                }
            };
            const int pre = ntiles < NST ? ntiles : NST;
            for (int t = 0; t < pre; ++t) issue(t);
            for (int u = 0; u < ntiles; ++u) {
                const int s = u % NST;
                mbar_wait(&r.done[s], (uint32_t)(u / NST) & 1u);
                if constexpr (WANT_GV) {
                    const int eb = e0 + u * nslots;
                    const int ne = min(nslots, e1 - eb);
                    const uint32_t bytes = (uint32_t)ne * row_bytes;
                    if constexpr (SW) {
                        for (int i = 0; i < ne; ++i) tma_store_2d(&tm.b, 0, (eb + i) * n, r.stage(s) + (size_t)i * row_bytes);
                    } else {
                        bulk_store(gV + (size_t)eb * n * DV, r.stage(s), bytes);
                    }
                    bulk_commit();
                    if (NST == 1) {
                        if (u + 1 < ntiles) { bulk_wait_read<0>(); issue(u + 1); }
                    } else if (u >= 1 && u - 1 + NST < ntiles) {
                        bulk_wait_read<1>();
                        issue(u - 1 + NST);
                    }
                } else {
                    if (u + NST < ntiles) issue(u + NST);  // every warp is done with stage s
                }
            }
            if constexpr (WANT_GV) bulk_wait_read<0>();
        }
    } else {
        // ---------------------------------------------------------------- compute warps
        T E[DE];
        T qc = T(0);
#pragma unroll
        for (int j = 0; j < DE; ++j) E[j] = T(0);
        if (active) {
            const T* er = Eenv + ((size_t)c * n + ch) * DE;
#pragma unroll
            for (int j = 0; j < DE; ++j) E[j] = er[j];
            if constexpr (COT) qc = q[ch];
        }
        for (int t = 0; t < ntiles; ++t) {
            const int s = t % NST;
            mbar_wait(&r.full[s], (uint32_t)(t / NST) & 1u);
            const int eb = e0 + t * nslots;
            if (active && eb + slot < e1) {
                T* grow = reinterpret_cast<T*>(r.stage(s)) + ((size_t)slot * n + ch) * DV;
                const T* vrow = reinterpret_cast<const T*>(r.stage(s) + r.tile_bytes) + ((size_t)slot * n + ch) * DV;
                [[maybe_unused]] const uint32_t sw = ((uint32_t)(slot * n + ch) & 7u) << 4;
                T v[DV], g[DV], gv[DV];
                if constexpr (SW) {
                    row_load_sw<T, DV>(reinterpret_cast<const unsigned char*>(grow), sw, g);
                    row_load_sw<T, DV>(reinterpret_cast<const unsigned char*>(vrow), sw, v);
                } else {
                    row_load<T, DV>(grow, g);
                    row_load<T, DV>(vrow, v);
                }
                if constexpr (COT) {
#pragma unroll
                    for (int k = 0; k < DV; ++k) g[k] *= kappa;
                    g[0] += qc;
                }
                Gen::template bwd<T, WANT_GV>(cwt.v, v, E, g, gv, gE);
                if constexpr (WANT_GW) Gen::template pathw<T>(v, E, g, gw);
                if constexpr (WANT_GV) {
                    if constexpr (SW) row_store_sw<T, DV>(reinterpret_cast<unsigned char*>(grow), sw, gv);
                    else row_store<T, DV>(grow, gv);
                }
            }
            ring_release(&r.done[s], lane);
        }
    }
    __syncthreads();  // all tiles are computed and every store has left shared memory: the ring can be reused

    // ---- gEenv: slots summed in slot order
    T* red = reinterpret_cast<T*>(smem_raw);  // [CT][DE], then [warps][P]
    if (active) {
#pragma unroll
        for (int j = 0; j < DE; ++j) red[((size_t)slot * n + ch) * DE + j] = gE[j];
    }
    __syncthreads();
    if (compute && slot == 0) {
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
        if (compute) {
#pragma unroll
            for (int p = 0; p < P; ++p) {
                T a = gw[p];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
                if (lane == 0) red[warp * P + p] = a;
            }
        }
        __syncthreads();
        if (tid < P) {
            T acc = red[tid];
            for (int wv = 1; wv < CT / 32; ++wv) acc += red[wv * P + tid];
            gw_part[(size_t)blockIdx.x * P + tid] = acc;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Forward + energy + first derivative in ONE pass over V (fusion is the paper's whole argument -- "costly
// intermediate memory reads and writes").  Per (edge, channel) row: out = Wc (V (x) Eenv) stays in registers,
// e_edge and the cotangent G = q (x) delta_{k,0} + kappa out of the A12 energy are formed from it, and the VJP
// gV = Wc^T (G (x) Eenv), gEenv += Wc^T (V (x) G) follows at once: V crosses HBM once, gV once, `out` and G never
// (23.9 KB -> 9.4 KB per edge at C1).  Stage = [V tile -> gV tile in place].  The kernel is then bound by instruction issue
// (1,322 + ~60 FP32 instructions per channel-edge at l_max = 2), not by HBM.
template <typename T, int L, int CT, bool WANT_GV, bool WANT_GW, bool SW>
__global__ void __launch_bounds__(CT + 32, (L >= 3 ? 1 : 2))
    tp_fused_kernel(const __grid_constant__ CwTab<T, TPGen<L>::NNZ> cwt, const __grid_constant__ CwTab<T, TPGen<L>::NNZ> cwt2,
                    const __grid_constant__ TpMaps tm, int NST, int n, const int* __restrict__ row_ptr,
                    const int* __restrict__ items, const T* __restrict__ V, const T* __restrict__ Eenv, const T* __restrict__ q, T kappa,
                    T* __restrict__ e_edge, T* __restrict__ gV, T* __restrict__ gE_dst, int gE_by_item, T* __restrict__ gw_part) {
    using Gen = TPGen<L>;
    constexpr int DV = Gen::DV, DE = Gen::DE, P = Gen::P;
    extern __shared__ __align__(128) unsigned char smem_dyn[];
    unsigned char* smem_raw = SW ? smem_dyn + ((1024u - (smem_u32(smem_dyn) & 1023u)) & 1023u) : smem_dyn;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nslots = CT / n;
    const uint32_t row_bytes = (uint32_t)n * DV * sizeof(T);
    Ring r;
    r.base = smem_raw;
    r.tile_bytes = align128((size_t)nslots * row_bytes);
    r.stage_bytes = r.tile_bytes;
    r.full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)NST * r.stage_bytes);
    r.done = r.full + NST;
    T* ebuf = reinterpret_cast<T*>(r.done + NST);  // [2][CT]

    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    const int ntiles = (e1 - e0 + nslots - 1) / nslots;   // 0 for an empty item: only the zero gEenv row is written
    ring_init(r, tid, CT / 32, NST);

    const bool compute = warp < CT / 32;
    const int slot = tid / n, ch = tid - slot * n;
    const bool active = compute && slot < nslots;
    T gE[DE];
#pragma unroll
    for (int j = 0; j < DE; ++j) gE[j] = T(0);
    T gw[WANT_GW ? P : 1];
#pragma unroll
    for (int p = 0; p < (WANT_GW ? P : 1); ++p) gw[p] = T(0);

    if (!compute) {
        // ---------------------------------------------------------------- producer
        if (lane == 0) {
            auto issue = [&](int t) {
                const int s = t % NST;
                const int eb = e0 + t * nslots;
                const int ne = min(nslots, e1 - eb);
                const uint32_t bytes = (uint32_t)ne * row_bytes;
                mbar_expect_tx(&r.full[s], bytes);
                if constexpr (SW) {
                    for (int i = 0; i < ne; ++i) tma_load_2d(r.stage(s) + (size_t)i * row_bytes, &tm.a, 0, (eb + i) * n, &r.full[s]);
                } else {
                    bulk_load(r.stage(s), V + (size_t)eb * n * DV, bytes, &r.full[s]);
                }
            };
            const int pre = ntiles < NST ? ntiles : NST;
            for (int t = 0; t < pre; ++t) issue(t);
            for (int u = 0; u < ntiles; ++u) {
                const int s = u % NST;
                mbar_wait(&r.done[s], (uint32_t)(u / NST) & 1u);
                if constexpr (WANT_GV) {
                    const int eb = e0 + u * nslots;
                    const int ne = min(nslots, e1 - eb);
                    if constexpr (SW) {
                        for (int i = 0; i < ne; ++i) tma_store_2d(&tm.b, 0, (eb + i) * n, r.stage(s) + (size_t)i * row_bytes);
                    } else {
                        bulk_store(gV + (size_t)eb * n * DV, r.stage(s), (uint32_t)ne * row_bytes);
                    }
                    bulk_commit();
                    if (NST == 1) {
                        if (u + 1 < ntiles) { bulk_wait_read<0>(); issue(u + 1); }
                    } else if (u >= 1 && u - 1 + NST < ntiles) {
                        bulk_wait_read<1>();
                        issue(u - 1 + NST);
                    }
                } else {
                    if (u + NST < ntiles) issue(u + NST);  // every warp is done with stage s
                }
            }
            if constexpr (WANT_GV) bulk_wait_read<0>();
        }
    } else {
        // ---------------------------------------------------------------- compute warps
        T E[DE];
        T qc = T(0);
#pragma unroll
        for (int j = 0; j < DE; ++j) E[j] = T(0);
        if (active) {
            const T* er = Eenv + ((size_t)c * n + ch) * DE;
#pragma unroll
            for (int j = 0; j < DE; ++j) E[j] = er[j];
            qc = q[ch];
        }
        const int mode = slot_sum_mode(n);
        for (int t = 0; t < ntiles; ++t) {
            const int s = t % NST;
            mbar_wait(&r.full[s], (uint32_t)(t / NST) & 1u);
            const int eb = e0 + t * nslots;
            const bool valid = active && eb + slot < e1;
            T epart = T(0);
            if (valid) {
                T* row = reinterpret_cast<T*>(r.stage(s)) + ((size_t)slot * n + ch) * DV;
                [[maybe_unused]] const uint32_t sw = ((uint32_t)(slot * n + ch) & 7u) << 4;
                T v[DV], g[DV], gv[DV];
                if constexpr (SW) row_load_sw<T, DV>(reinterpret_cast<const unsigned char*>(row), sw, v);
                else row_load<T, DV>(row, v);
                Gen::template fwd<T>(cwt.v, v, E, g);                 // g = out
                T sq = T(0);
#pragma unroll
                for (int k = 0; k < DV; ++k) sq = fma(g[k], g[k], sq);
                epart = fma(T(0.5) * kappa, sq, qc * g[0]);
#pragma unroll
                for (int k = 0; k < DV; ++k) g[k] *= kappa;            // g = cotangent of the A12 energy
                g[0] += qc;
                // scheduling fence: the VJP below starts from complete g / v rows (otherwise the two unrolled contractions are
                // interleaved for ILP and their live ranges no longer fit the register file)
#pragma unroll
                for (int k = 0; k < DV; ++k) {
                    if constexpr (sizeof(T) == 4) asm volatile("" : "+f"(g[k]), "+f"(v[k]));
                    else asm volatile("" : "+d"(g[k]), "+d"(v[k]));
                }
                // cwt2 is a second copy of the same table: read through the first one, every coefficient would be kept alive from
                // its forward use to its VJP use (274 .. 1222 values) and spilled
                Gen::template bwd<T, WANT_GV>(cwt2.v, v, E, g, gv, gE);
                if constexpr (WANT_GW) Gen::template pathw<T>(v, E, g, gw);
                if constexpr (WANT_GV) {
                    if constexpr (SW) row_store_sw<T, DV>(reinterpret_cast<unsigned char*>(row), sw, gv);
                    else row_store<T, DV>(row, gv);
                }
            }
            ring_release(&r.done[s], lane);
            const T tot = slot_sum<T, CT>(epart, mode, n, slot, ch, tid, t, ebuf);
            if (valid && ch == 0) e_edge[eb + slot] = tot;
        }
    }
    __syncthreads();  // all tiles are computed and every store has left shared memory: the ring can be reused

    // ---- gEenv: slots summed in slot order
    T* red = reinterpret_cast<T*>(smem_raw);  // [CT][DE], then [warps][P]
    if (active) {
#pragma unroll
        for (int j = 0; j < DE; ++j) red[((size_t)slot * n + ch) * DE + j] = gE[j];
    }
    __syncthreads();
    if (compute && slot == 0) {
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
        if (compute) {
#pragma unroll
            for (int p = 0; p < P; ++p) {
                T a = gw[p];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
                if (lane == 0) red[warp * P + p] = a;
            }
        }
        __syncthreads();
        if (tid < P) {
            T acc = red[tid];
            for (int wv = 1; wv < CT / 32; ++wv) acc += red[wv * P + tid];
            gw_part[(size_t)blockIdx.x * P + tid] = acc;
        }
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
