// mix3_kernels.cuh -- dense per-path channel mix (BASELINE.json:configs[2], row a4 of SURVEY 8) on the sm_100a tensor cores:
// tcgen05.mma (kind::tf32) with fp32 accumulators in tensor memory, W_p staged by bulk async copies (TMA), operands in
// 128-byte-swizzled shared memory.  fp32, l_max = 2, n = 64.
//
//   out[e, n', off3(p) + M] = sum_{p -> block} sum_n W_p[n', n] * t_p[e, n, M],   t_p = channel-wise CG contraction of V_e and Eenv_c
//
// GEMM mapping (per tile of TE = 24 edges of one centre, per path p):   D_b[128 x N_b] += A_p[128 x 64] . B_p[N_b x 64]^T
//   A_p rows  = (channel n', h): h = 0 the raw W_p row (the tensor core truncates fp32 to tf32 = "hi"), h = 1 the exact remainder
//               W - tf32(W) ("lo"); row order 32 q + 16 h + nl with n' = 16 q + nl, so hi and lo of a channel sit in one warp's
//               TMEM lane quarter and are summed with one shuffle.  64 output channels fill the 128-row MMA this way.
//   B_p rows  = column (M, e) of the problem: t_p[e, :, M] over the 64 input channels (K), written by the CUDA cores, once as
//               t (hi by truncation) and once as t - tf32(t) (lo).  Two MMA passes (B hi, B lo) give all four hi/lo products.
//   D_b       = one accumulator per output block b = (l3, p3) in TMEM, columns (M, e); all six blocks of a tile stay resident
//               (480 of 512 columns), so `out` rows leave the SM once, complete, as contiguous 72-byte rows.
#pragma once
#include <type_traits>
#include <utility>

#include "common.cuh"
#include "launch.h"
#include "tc05.cuh"

#ifdef MIX3_DBG
#define MIX3_T0() long long dbg_t0 = clock64()
#define MIX3_ACC(slot, cond) do { const long long dbg_t1 = clock64(); if (cond) mix3_dbg[slot] += dbg_t1 - dbg_t0; dbg_t0 = dbg_t1; } while (0)
#else
#define MIX3_T0() do { } while (0)
#define MIX3_ACC(slot, cond) do { } while (0)
#endif

namespace allegro {

template <int I, int N, typename F>
__device__ __forceinline__ void static_for3(F&& f) {
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for3<I + 1, N>(f);
    }
}

struct Mix3 {
    static constexpr int N = 64, L = 2, DV = 18, DE = 9, P = 30;
    static constexpr int TE = 24, NSLOT = 6, EPS = 4;            // tile edges = 6 slots x 4 consecutive edges
    static constexpr int CT = 384;                                // compute threads (12 warps, 128 registers each); + 1 control warp
    static constexpr int A_BYTES = 2 * 128 * 128;                 // [2 K-atoms][128 rows][128 B]
    static constexpr int BV_BYTES = 2 * 128 * 128;                // one B variant (hi or lo): [2 K-atoms][<=128 rows][128 B]
    static constexpr int B_BYTES = 2 * BV_BYTES;
    static constexpr int NA = 3, NB = 2;                          // ring depths
    static constexpr int IMG_BYTES = 64 * 64 * 4;                 // one path's weight image in global memory (hi rows only)
    static constexpr int OFF_A = 0, OFF_B = NA * A_BYTES, OFF_BAR = OFF_B + NB * B_BYTES;
    static constexpr int SMEM = OFF_BAR + 256 + 1024;             // + barrier block + 1024-byte alignment slack
    // TMEM column base of each output block, indexed by off3 (0e:0, 0o:1, 1e:2, 1o:5, 2e:8, 2o:13); N_b = 32 / 80 / 128
    __host__ __device__ static constexpr int dcol(int off3) {
        return off3 == 0 ? 0 : off3 == 1 ? 32 : off3 == 2 ? 64 : off3 == 5 ? 144 : off3 == 8 ? 224 : 352;
    }
    // is p the first path (in plan order) that mixes into its output block?
    __host__ __device__ static constexpr bool first_of_block(int p) {
        for (int r = 0; r < p; ++r) if (TPGen<2>::off3(r) == TPGen<2>::off3(p)) return false;
        return true;
    }
    __host__ __device__ static constexpr int ncols(int d3) { return d3 == 1 ? 32 : d3 == 3 ? 80 : 128; }
};

// Weight images: img_f[p] feeds the forward (A row = output channel n', K = input channel n), img_b[p] the VJP
// (A row = input channel n, K = output channel n').  Layout [K-atom a][quarter q][row nl][128 B], 16-byte chunk c of a row
// stored at chunk position c ^ (nl & 7): the bytes land in the "hi" rows of the swizzled A tile by plain bulk copies.
__global__ void mix3_prep_kernel(const float* __restrict__ W, float* __restrict__ img_f, float* __restrict__ img_b) {
    const int p = blockIdx.x;
    const float* Wp = W + (size_t)p * 64 * 64;
    for (int idx = threadIdx.x; idx < 64 * 64; idx += blockDim.x) {
        const int row = idx >> 6, k = idx & 63;
        const int a = k >> 5, q = row >> 4, nl = row & 15, c = (k & 31) >> 2;
        const int dst = ((a * 4 + q) * 16 + nl) * 32 + ((c ^ (nl & 7)) << 2) + (k & 3);
        img_f[(size_t)p * 4096 + dst] = Wp[row * 64 + k];   // (n' = row, n = k)
        img_b[(size_t)p * 4096 + dst] = Wp[k * 64 + row];   // (n = row, n' = k)
    }
}

// barrier block in shared memory
struct Mix3Bars {
    uint64_t a_full[Mix3::NA], a_empty[Mix3::NA], b_full[Mix3::NB], b_empty[Mix3::NB], d_full, d_empty;
    uint32_t tmem_slot;
};

__device__ __forceinline__ float tf32_lo(float x) { return x - __uint_as_float(__float_as_uint(x) & 0xffffe000u); }

template <int DUMMY = 0>
__global__ void __launch_bounds__(Mix3::CT + 32, 1) mix3_fwd_kernel(const int* __restrict__ row_ptr, const int* __restrict__ items,
                                                                   const float* __restrict__ V, const float* __restrict__ Eenv,
                                                                   const float* __restrict__ img, float* __restrict__ out) {
    using M3 = Mix3;
    using Gen = TPGen<2>;
    constexpr int DV = M3::DV, DE = M3::DE, P = M3::P, TE = M3::TE;
    extern __shared__ unsigned char smem_raw[];
    unsigned char* sm = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // 1024-byte aligned (128-byte swizzle atoms)
    Mix3Bars* bars = reinterpret_cast<Mix3Bars*>(sm + M3::OFF_BAR);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    if (e1 <= e0) return;
    const int ntiles = (e1 - e0 + TE - 1) / TE;

    if (tid == 0) {
        for (int s = 0; s < M3::NA; ++s) { mbar_init(&bars->a_full[s], 1); mbar_init(&bars->a_empty[s], 1); }
        for (int s = 0; s < M3::NB; ++s) { mbar_init(&bars->b_full[s], M3::CT / 32); mbar_init(&bars->b_empty[s], 1); }
        mbar_init(&bars->d_full, 1);
        mbar_init(&bars->d_empty, M3::CT / 32);
        fence_mbar_init();
    }
    if (warp == M3::CT / 32) { tc05::tmem_alloc(&bars->tmem_slot, 512); tc05::tmem_relinquish(); }
    tc05::fence_before_sync();
    __syncthreads();
    tc05::fence_after_sync();
    const uint32_t tbase = bars->tmem_slot;

    if (warp == M3::CT / 32) {
        // ================= control warp: lane 0 streams the weight images (TMA), lane 1 issues the MMAs
        if (lane == 0) {
            for (int t = 0; t < ntiles; ++t) {
                for (int p = 0; p < P; ++p) {
                    const int sa = p % M3::NA;                                   // 30 paths per tile = 10 ring turns: stage and
                    const uint32_t ph = (uint32_t)(p / M3::NA) & 1u;             // parity depend on p only
                    MIX3_T0();
                    mbar_wait(&bars->a_empty[sa], ph ^ 1u);
                    MIX3_ACC(3, blockIdx.x == 0);
                    mbar_expect_tx(&bars->a_full[sa], M3::IMG_BYTES);
                    unsigned char* dstA = sm + M3::OFF_A + sa * M3::A_BYTES;
                    const unsigned char* src = reinterpret_cast<const unsigned char*>(img) + (size_t)p * M3::IMG_BYTES;
#pragma unroll
                    for (int a = 0; a < 2; ++a)
#pragma unroll
                        for (int q = 0; q < 4; ++q)
                            bulk_load(dstA + a * 16384 + q * 4096, src + (a * 4 + q) * 2048, 2048, &bars->a_full[sa]);
                }
            }
        } else if (lane == 1) {
            constexpr uint32_t id1 = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, 32);
            constexpr uint32_t id3 = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, 80);
            constexpr uint32_t id5 = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, 128);
            // descriptors of K step 0 of every ring stage; K step j adds (j >> 2) * 16384 + (j & 3) * 32 bytes (16-byte units)
            uint64_t adesc[M3::NA], bdesc[M3::NB];
#pragma unroll
            for (int s = 0; s < M3::NA; ++s) adesc[s] = tc05::sdesc_sw128(smem_u32(sm + M3::OFF_A + s * M3::A_BYTES));
#pragma unroll
            for (int s = 0; s < M3::NB; ++s) bdesc[s] = tc05::sdesc_sw128(smem_u32(sm + M3::OFF_B + s * M3::B_BYTES));
            for (int t = 0; t < ntiles; ++t) {
                MIX3_T0();
                if (t > 0) { mbar_wait(&bars->d_empty, (uint32_t)(t - 1) & 1u); tc05::fence_after_sync(); }
                MIX3_ACC(2, blockIdx.x == 0);
                static_for3<0, P>([&](auto pc) {
                    constexpr int p = decltype(pc)::value;
                    constexpr int sa = p % M3::NA, sb = p & 1;
                    constexpr int d3 = Gen::d3(p), off3 = Gen::off3(p);
                    constexpr uint32_t idesc = d3 == 1 ? id1 : d3 == 3 ? id3 : id5;
                    constexpr bool first = M3::first_of_block(p);   // first path of its output block: initialises the accumulator
                    const uint32_t phb = (uint32_t)(t + (p >> 1)) & 1u;          // 15 B-ring turns per tile
                    mbar_wait(&bars->b_full[sb], phb);
                    MIX3_ACC(0, blockIdx.x == 0);
                    tc05::fence_after_sync();
                    const uint32_t dcol = tbase + (uint32_t)M3::dcol(off3);
#pragma unroll
                    for (int v = 0; v < 2; ++v)          // B variant: hi, lo
#pragma unroll
                        for (int j = 0; j < 8; ++j) {    // K step of 8 channels
                            const uint64_t koff = (uint64_t)(((j >> 2) * 16384 + (j & 3) * 32) >> 4);
                            tc05::mma_tf32(dcol, adesc[sa] + koff, bdesc[sb] + (uint64_t)((v * M3::BV_BYTES) >> 4) + koff, idesc,
                                           (first && v == 0 && j == 0) ? 0u : 1u);
                        }
                    tc05::mma_commit(&bars->b_empty[sb]);
                    tc05::mma_commit(&bars->a_empty[sa]);
                    MIX3_ACC(1, blockIdx.x == 0);
                });
                tc05::mma_commit(&bars->d_full);
            }
        }
    } else {
        // ================= compute warps: thread = (edge slot, input channel) for t_p; TMEM lane = (output channel, hi/lo) for the epilogue
        const int ch = tid & 63, slot = tid >> 6;
        float E[DE];
#pragma unroll
        for (int j = 0; j < DE; ++j) E[j] = Eenv[((size_t)c * 64 + ch) * DE + j];
        // B rows are the columns (M, e) = M * 24 + e of the problem; this thread writes element (row, k = ch) for its four edges
        // e = 4 slot + j.  Byte offset inside a B variant for M = 0: row group (e >> 3) * 1024 + (e & 7) * 128, the 16-byte chunk
        // (ch & 31) >> 2 swizzled with (e & 7); M adds 3 row groups (24 rows).
        uint32_t boff[M3::EPS];
#pragma unroll
        for (int j = 0; j < M3::EPS; ++j) {
            const uint32_t e = 4u * slot + j, r = e & 7u;
            boff[j] = (uint32_t)(ch >> 5) * 16384u + (e >> 3) * 1024u + r * 128u + (((((uint32_t)ch & 31u) >> 2) ^ r) << 4) + (((uint32_t)ch & 3u) << 2);
        }
        const int q = warp & 3, wq = warp >> 2, h = lane >> 4, nl = lane & 15;
        for (int t = 0; t < ntiles; ++t) {
            const int eb = e0 + t * TE;
            MIX3_T0();
            float Vr[M3::EPS][DV];
#pragma unroll
            for (int i = 0; i < M3::EPS; ++i) {
                const int e = eb + 4 * slot + i;
                if (e < e1) {
                    row_load<float, DV>(V + ((size_t)e * 64 + ch) * DV, Vr[i]);
                } else {
#pragma unroll
                    for (int k = 0; k < DV; ++k) Vr[i][k] = 0.f;
                }
            }
            static_for3<0, P>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                using Pth = TPPath<2, p>;
                constexpr int sa = p % M3::NA, sb = p & 1;
                constexpr uint32_t pha = (uint32_t)(p / M3::NA) & 1u;
                const uint32_t phb = (uint32_t)(t + (p >> 1)) & 1u;
                unsigned char* As = sm + M3::OFF_A + sa * M3::A_BYTES;
                unsigned char* Bs = sm + M3::OFF_B + sb * M3::B_BYTES;
                // B: t_p of this thread's three edges, hi (raw) and lo
                MIX3_ACC(10, blockIdx.x == 0 && tid == 0 && p == 0);
                mbar_wait(&bars->b_empty[sb], phb ^ 1u);
                if (p == 1 && t > 0) asm volatile("bar.sync 1, %0;" ::"n"(2 * M3::CT) : "memory");
                MIX3_ACC(4, blockIdx.x == 0 && tid == 0);
                // launder E so that V.E products are not kept alive (common subexpressions) from one path to the next
#pragma unroll
                for (int j = 0; j < DE; ++j) asm volatile("" : "+f"(E[j]));
#pragma unroll
                for (int i = 0; i < M3::EPS; ++i) {
                    float tp[Pth::D3];
                    Pth::template fwd<float>(Vr[i], E, tp);
#pragma unroll
                    for (int M = 0; M < Pth::D3; ++M) {
                        unsigned char* dst = Bs + boff[i] + 3 * M * 1024;
                        *reinterpret_cast<float*>(dst) = tp[M];
                        *reinterpret_cast<float*>(dst + M3::BV_BYTES) = tf32_lo(tp[M]);
                    }
                }
                // A lo rows: W - tf32(W) (hi rows arrive by TMA; waited for after the B work so that the copy's latency is covered)
                MIX3_ACC(5, blockIdx.x == 0 && tid == 0);
                mbar_wait(&bars->a_full[sa], pha);
                MIX3_ACC(6, blockIdx.x == 0 && tid == 0);
#pragma unroll
                for (int cid = tid; cid < 1024; cid += M3::CT) {
                    unsigned char* src = As + (cid >> 9) * 16384 + ((cid >> 7) & 3) * 4096 + (cid & 127) * 16;
                    float4 w = *reinterpret_cast<const float4*>(src);
                    w.x = tf32_lo(w.x); w.y = tf32_lo(w.y); w.z = tf32_lo(w.z); w.w = tf32_lo(w.w);
                    *reinterpret_cast<float4*>(src + 2048) = w;
                }
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars->b_full[sb]);
                MIX3_ACC(7, blockIdx.x == 0 && tid == 0);
            });
            // ---- epilogue: TMEM lane (n', h) -> out rows; warp (q, wq) takes edges 8 wq .. 8 wq + 7, lane h its half of them
            mbar_wait(&bars->d_full, (uint32_t)t & 1u);
            MIX3_ACC(8, blockIdx.x == 0 && tid == 0);
            tc05::fence_after_sync();
            // Rows are staged through shared memory (B stage 1 is idle until path 1 of the next tile) so that they leave as
            // fully coalesced 16-byte stores: per warp a private [4 edges][16 channels][18] block, two half-tiles in turn.
            float* stg = reinterpret_cast<float*>(sm + M3::OFF_B + M3::B_BYTES) + warp * (4 * 16 * DV);
            const uint32_t trow = tbase + ((uint32_t)(32 * q) << 16) + (uint32_t)(8 * wq);
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {     // edges 8 wq + 4 hf + {0..3}: lane half h finalises edges 2 h, 2 h + 1 of them
                float o[2][DV];
                static_for3<0, 6>([&](auto bc) {
                    constexpr int b = decltype(bc)::value;
                    constexpr int off3 = b == 0 ? 0 : b == 1 ? 1 : b == 2 ? 2 : b == 3 ? 5 : b == 4 ? 8 : 13;
                    constexpr int d3 = b < 2 ? 1 : b < 4 ? 3 : 5;
                    uint32_t v[d3][4];
#pragma unroll
                    for (int M = 0; M < d3; ++M) tc05::tmem_ld4(trow + (uint32_t)(M3::dcol(off3) + M * TE + 4 * hf), v[M]);
                    tc05::tmem_ld_wait();
#pragma unroll
                    for (int M = 0; M < d3; ++M)
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            const float mine = __uint_as_float(h ? v[M][2 + i] : v[M][i]);
                            const float send = __uint_as_float(h ? v[M][i] : v[M][2 + i]);
                            o[i][off3 + M] = mine + __shfl_xor_sync(0xffffffffu, send, 16);
                        }
                });
                if (hf == 1) {   // all TMEM reads of this warp are done: the accumulators may be overwritten
                    tc05::fence_before_sync();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&bars->d_empty);
                }
#pragma unroll
                for (int i = 0; i < 2; ++i) row_store<float, DV>(stg + ((2 * h + i) * 16 + nl) * DV, o[i]);
                __syncwarp();
                const int ebase = eb + 8 * wq + 4 * hf;
#pragma unroll
                for (int r = 0; r < 9; ++r) {    // 4 edges x 288 floats = 288 float4
                    const int idx = lane + 32 * r, el = idx / 72, w4 = idx - el * 72;
                    if (ebase + el < e1)
                        *reinterpret_cast<float4*>(out + ((size_t)(ebase + el) * 64 + 16 * q) * DV + 4 * w4) = reinterpret_cast<const float4*>(stg)[idx];
                }
                __syncwarp();
            }
            asm volatile("bar.arrive 1, %0;" ::"n"(2 * M3::CT) : "memory");   // staging done; waited for before B stage 1 is rewritten
            MIX3_ACC(9, blockIdx.x == 0 && tid == 0);
        }
    }
    tc05::fence_before_sync();
    __syncthreads();
    if (warp == M3::CT / 32) tc05::tmem_dealloc(tbase, 512);
}

}  // namespace allegro
