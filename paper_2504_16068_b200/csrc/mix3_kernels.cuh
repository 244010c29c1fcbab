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
    static constexpr int CT = 384;                                // compute threads (12 warps, 128 registers each); + 2 control warps
    static constexpr int A_BYTES = 2 * 128 * 128;                 // [2 K-atoms][128 rows][128 B]
    static constexpr int NA = 3, NB = 2;                          // ring depths
    static constexpr int IMG_BYTES = 2 * 128 * 128;               // one path's weight image in global memory (hi and lo rows)
    static constexpr uint32_t ALL = 0x3fffffffu;                  // path mask: every path of the plan
    // TMEM column base of each output block, indexed by off3 (0e:0, 0o:1, 1e:2, 1o:5, 2e:8, 2o:13); N_b = 32 / 80 / 128
    __host__ __device__ static constexpr int dcol(int off3) {
        return off3 == 0 ? 0 : off3 == 1 ? 32 : off3 == 2 ? 64 : off3 == 5 ? 144 : off3 == 8 ? 224 : 352;
    }
    __host__ __device__ static constexpr int ncols(int d3) { return d3 == 1 ? 32 : d3 == 3 ? 80 : 128; }
    // the paths that mix into the output block at component offset off3 (0 = the 0e scalars)
    __host__ __device__ static constexpr uint32_t mask_into(int off3) {
        uint32_t m = 0;
        for (int p = 0; p < P; ++p) if (TPGen<2>::off3(p) == off3) m |= 1u << p;
        return m;
    }
    // (l1, p1) block of V that path p reads: first component (plan order: l1, p1, l2, l3) and width
    __host__ __device__ static constexpr int off1(int p) {
        int idx = 0;
        for (int l1 = 0; l1 <= 2; ++l1)
            for (int p1 = 0; p1 < 2; ++p1)
                for (int l2 = 0; l2 <= 2; ++l2)
                    for (int l3 = (l1 > l2 ? l1 - l2 : l2 - l1); l3 <= (l1 + l2 < 2 ? l1 + l2 : 2); ++l3, ++idx)
                        if (idx == p) return 2 * l1 * l1 + (p1 ? 2 * l1 + 1 : 0);
        return -1;
    }
    __host__ __device__ static constexpr int d1(int p) { return off1(p) < 2 ? 1 : off1(p) < 8 ? 3 : 5; }
    // the paths whose input block has its natural parity (l, (-1)^l): 0e, 1o, 2e -- all that a first layer fed with
    // V0 = v (x) Y(rhat) ever sees non-zero
    __host__ __device__ static constexpr uint32_t mask_natural_in() {
        uint32_t m = 0;
        for (int p = 0; p < P; ++p) if (off1(p) == 0 || off1(p) == 5 || off1(p) == 8) m |= 1u << p;
        return m;
    }
};

// The paths that run (bit p of PMASK), in plan order, as compile-time functions of the sequence index k; shared-memory layout of
// the forward kernel for that set (a B stage holds as many rows as the widest active block needs).
template <uint32_t PMASK>
struct Mix3Seq {
    __host__ __device__ static constexpr bool active(int p) { return ((PMASK >> p) & 1u) != 0; }
    __host__ __device__ static constexpr int count() {
        int n = 0;
        for (int p = 0; p < 30; ++p) n += active(p) ? 1 : 0;
        return n;
    }
    __host__ __device__ static constexpr int path(int k) {
        int n = 0;
        for (int p = 0; p < 30; ++p) if (active(p)) { if (n == k) return p; ++n; }
        return -1;
    }
    // is p the first active path (in plan order) that mixes into its output block?
    __host__ __device__ static constexpr bool first_of_block(int p) {
        for (int r = 0; r < p; ++r) if (active(r) && TPGen<2>::off3(r) == TPGen<2>::off3(p)) return false;
        return true;
    }
    __host__ __device__ static constexpr bool block_active(int off3) {
        for (int p = 0; p < 30; ++p) if (active(p) && TPGen<2>::off3(p) == off3) return true;
        return false;
    }
    __host__ __device__ static constexpr int max_d3() {
        int m = 1;
        for (int p = 0; p < 30; ++p) if (active(p) && TPGen<2>::d3(p) > m) m = TPGen<2>::d3(p);
        return m;
    }
    static constexpr int ATOM = Mix3::ncols(max_d3()) * 128;       // one K-atom of a B variant: [rows][128 B]
    static constexpr int BV_BYTES = 2 * ATOM, B_BYTES = 2 * BV_BYTES;   // B stage: [hi, lo][2 K-atoms][rows][128 B]
    // The epilogue stages `out` rows in B stage 1 when they fit there (the stage is idle from the last MMA of a tile until the
    // first path of the next tile that is written into it); small B stages leave room for a staging area of its own.
    static constexpr int STG_BYTES = (Mix3::CT / 32) * 4 * 16 * Mix3::DV * 4;
    static constexpr bool ALIAS_STG = STG_BYTES <= B_BYTES;
    static constexpr int OFF_A = 0, OFF_B = Mix3::NA * Mix3::A_BYTES, OFF_STG = OFF_B + Mix3::NB * B_BYTES;
    static constexpr int OFF_BAR = OFF_STG + (ALIAS_STG ? 0 : STG_BYTES);
    static constexpr int OFF_RED = OFF_BAR + 256;                 // [2][4 lane quarters][24 edges] partial edge energies
    static constexpr int OFF_YS = OFF_RED + 2 * 4 * Mix3::TE * 4;       // OUTER mode: Y_j(rhat_e) of the tile's edges, [TE][9] floats
    static constexpr int SMEM = OFF_YS + 896 + 1024;             // + barrier block + energy partials + Ys + 1024-byte alignment slack
    static_assert(SMEM <= 232448, "shared memory of the forward kernel");
    static_assert(count() >= 2, "at least two paths");
};

// OUTER mode (layer-1 specialisation): the input features are not read from HBM but generated on chip as the outer product
// V0[e][n][(l, (-1)^l), m] = v0[e][n] Y_lm(rhat_e) of reading A19 (other-parity slots zero).  Y for l <= 2 in the convention of reading
// A1 (real, component-normalised, m = -l..l; Y_1 = sqrt3 (y, z, x)), index j = l^2 + l + m; feature slot of j: 0e -> 0, 1o -> 5..7, 2e -> 8..12.
__device__ __forceinline__ void mix3_sph9(float x, float y, float z, float (&Y)[9]) {
    const float s3 = 1.7320508075688772f, s15 = 3.8729833462074170f, s5h = 1.1180339887498949f;
    Y[0] = 1.f;
    Y[1] = s3 * y; Y[2] = s3 * z; Y[3] = s3 * x;
    Y[4] = s15 * x * y; Y[5] = s15 * y * z; Y[6] = s5h * (3.f * z * z - 1.f); Y[7] = s15 * x * z; Y[8] = 0.5f * s15 * (x * x - y * y);
}
__host__ __device__ constexpr int mix3_nat_slot(int j) { return j == 0 ? 0 : j < 4 ? 4 + j : 4 + j; }   // j 1..3 -> 5..7, j 4..8 -> 8..12
__host__ __device__ constexpr int mix3_nat_j(int slot) { return slot == 0 ? 0 : slot - 4; }             // inverse on the natural slots

// position in a ring of NST stages: stage index and the phase bit of the current turn
template <int NST>
struct RingPos {
    uint32_t s = 0, ph = 0;
    __device__ __forceinline__ void next() { if (++s == NST) { s = 0; ph ^= 1u; } }
};

// Weight images: img_f[p] feeds the forward (A row = output channel n', K = input channel n), img_b[p] the VJP
// (A row = input channel n, K = output channel n').  Each image is the complete swizzled A tile, [K-atom a][row 32 q + 16 h + nl][128 B]
// with the 16-byte chunk c of a row stored at chunk position c ^ (nl & 7): h = 0 rows hold W (the tensor core truncates it to
// tf32), h = 1 rows the exact remainder W - tf32(W).  One 32 KB bulk copy per path puts it into shared memory.
static __global__ void mix3_prep_kernel(const float* __restrict__ W, float* __restrict__ img_f, float* __restrict__ img_b) {
    const int p = blockIdx.x;
    const float* Wp = W + (size_t)p * 64 * 64;
    for (int idx = threadIdx.x; idx < 64 * 64; idx += blockDim.x) {
        const int row = idx >> 6, k = idx & 63;
        const int a = k >> 5, q = row >> 4, nl = row & 15, c = (k & 31) >> 2;
        const int dst = (a * 128 + 32 * q + nl) * 32 + ((c ^ (nl & 7)) << 2) + (k & 3);
        const float wf = Wp[row * 64 + k], wb = Wp[k * 64 + row];   // (n' = row, n = k) ; (n = row, n' = k)
        const float wfh = __uint_as_float(__float_as_uint(wf) & 0xffffe000u), wbh = __uint_as_float(__float_as_uint(wb) & 0xffffe000u);
        img_f[(size_t)p * 8192 + dst] = wf;
        img_f[(size_t)p * 8192 + dst + 16 * 32] = wf - wfh;
        img_b[(size_t)p * 8192 + dst] = wb;
        img_b[(size_t)p * 8192 + dst + 16 * 32] = wb - wbh;
    }
}

// barrier block in shared memory
struct Mix3Bars {
    uint64_t a_full[Mix3::NA], a_empty[Mix3::NA], b_full[Mix3::NB], b_empty[Mix3::NB], d_full, d_empty;
    uint32_t tmem_slot;
};

__device__ __forceinline__ float tf32_lo(float x) { return x - __uint_as_float(__float_as_uint(x) & 0xffffe000u); }

// Energy epilogue (e_edge != NULL): e_edge[e] = sum_n' ( q[n'] out[e][n'][0] + kappa/2 sum_k out[e][n'][k]^2 ) of reading A12, formed
// from the rows while they are in registers; `out` may then be NULL (the rows are never stored: a last layer whose output feeds
// only the readout).  s_out (nullable, [E][64]): compact copy of the 0e scalars out[e][n'][0], what a scalar latent update reads
// (as a 72-byte-strided gather from `out` it costs 8 x the sectors).
// OUTER: V is not read; the rows are generated from rvec [E][3] and v0 [E][64] (see mix3_sph9).
template <uint32_t PMASK, bool OUTER = false>
__global__ void __launch_bounds__(Mix3::CT + 64, 1) mix3_fwd_kernel(const int* __restrict__ row_ptr, const int* __restrict__ items,
                                                                   const float* __restrict__ V, const float* __restrict__ Eenv,
                                                                   const float* __restrict__ img, float* __restrict__ out,
                                                                   const float* __restrict__ qvec, float kappa, float* __restrict__ e_edge,
                                                                   float* __restrict__ s_out, const float* __restrict__ rvec = nullptr,
                                                                   const float* __restrict__ v0 = nullptr) {
    using M3 = Mix3;
    using SQ = Mix3Seq<PMASK>;
    using Gen = TPGen<2>;
    constexpr int DV = M3::DV, DE = M3::DE, NP = SQ::count(), TE = M3::TE;
    extern __shared__ unsigned char smem_raw[];
    unsigned char* sm = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // 1024-byte aligned (128-byte swizzle atoms)
    Mix3Bars* bars = reinterpret_cast<Mix3Bars*>(sm + SQ::OFF_BAR);
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

    if (warp >= M3::CT / 32) {
        // ================= two control warps (one thread each, so that neither spins inside the other's warp): weight images (TMA), MMA issue
        if (warp == M3::CT / 32 && lane == 0) {
            RingPos<M3::NA> ra;
            for (int t = 0; t < ntiles; ++t) {
                static_for3<0, NP>([&](auto kc) {
                    constexpr int p = SQ::path(decltype(kc)::value);
                    MIX3_T0();
                    mbar_wait(&bars->a_empty[ra.s], ra.ph ^ 1u);
                    MIX3_ACC(3, blockIdx.x == 0);
                    mbar_expect_tx(&bars->a_full[ra.s], M3::IMG_BYTES);
                    bulk_load(sm + SQ::OFF_A + ra.s * M3::A_BYTES, reinterpret_cast<const unsigned char*>(img) + (size_t)p * M3::IMG_BYTES,
                              M3::IMG_BYTES, &bars->a_full[ra.s]);
                    ra.next();
                });
            }
        } else if (warp == M3::CT / 32 + 1) {   // the whole warp walks the loop; one elected lane issues
            constexpr uint32_t id1 = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, 32);
            constexpr uint32_t id3 = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, 80);
            constexpr uint32_t id5 = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, 128);
            // descriptors of K step 0 of every ring stage; K step j adds (j >> 2) * 16384 + (j & 3) * 32 bytes (16-byte units)
            const uint32_t adesc0 = tc05::sdesc_lo(smem_u32(sm + SQ::OFF_A)), bdesc0 = tc05::sdesc_lo(smem_u32(sm + SQ::OFF_B));
            RingPos<M3::NA> ra;
            RingPos<M3::NB> rb;
            for (int t = 0; t < ntiles; ++t) {
                MIX3_T0();
                if (t > 0) { mbar_wait(&bars->d_empty, (uint32_t)(t - 1) & 1u); tc05::fence_after_sync(); }
                MIX3_ACC(2, blockIdx.x == 0 && lane == 0);
                static_for3<0, NP>([&](auto kc) {
                    constexpr int k = decltype(kc)::value;
                    constexpr int p = SQ::path(k);
                    constexpr int d3 = Gen::d3(p), off3 = Gen::off3(p);
                    constexpr uint32_t idesc = d3 == 1 ? id1 : d3 == 3 ? id3 : id5;
                    constexpr bool first = SQ::first_of_block(p);   // first path of its output block: initialises the accumulator
                    mbar_wait(&bars->a_full[ra.s], ra.ph);
                    mbar_wait(&bars->b_full[rb.s], rb.ph);
                    MIX3_ACC(0, blockIdx.x == 0 && lane == 0);
                    tc05::fence_after_sync();
                    const uint32_t dcol = tbase + (uint32_t)M3::dcol(off3);
                    if (tc05::elect_one()) {
                    uint32_t ad = adesc0 + ((ra.s * (uint32_t)M3::A_BYTES) >> 4), bd = bdesc0 + ((rb.s * (uint32_t)SQ::B_BYTES) >> 4);
                    asm volatile("" : "+r"(ad), "+r"(bd));   // opaque per path: keeps the descriptor words from being hoisted and spilled
#pragma unroll
                    for (int v = 0; v < 2; ++v)          // B variant: hi, lo
#pragma unroll
                        for (int j = 0; j < 8; ++j) {    // K step of 8 channels
                            const uint32_t aoff = (uint32_t)(((j >> 2) * 16384 + (j & 3) * 32) >> 4);
                            const uint32_t boff = (uint32_t)((v * SQ::BV_BYTES + (j >> 2) * SQ::ATOM + (j & 3) * 32) >> 4);
                            tc05::mma_tf32_lo(dcol, ad + aoff, bd + boff, tc05::kSdescHiSw128, idesc, (first && v == 0 && j == 0) ? 0u : 1u);
                        }
                    tc05::mma_commit(&bars->b_empty[rb.s]);
                    tc05::mma_commit(&bars->a_empty[ra.s]);
                    if (k == NP - 1) tc05::mma_commit(&bars->d_full);
                    }
                    __syncwarp();
                    MIX3_ACC(1, blockIdx.x == 0 && lane == 0);
                    ra.next();
                    rb.next();
                });
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
            boff[j] = (uint32_t)(ch >> 5) * (uint32_t)SQ::ATOM + (e >> 3) * 1024u + r * 128u + (((((uint32_t)ch & 31u) >> 2) ^ r) << 4) + (((uint32_t)ch & 3u) << 2);
        }
        const int q = warp & 3, wq = warp >> 2, h = lane >> 4, nl = lane & 15;
        const float qn = e_edge != nullptr ? qvec[16 * q + nl] : 0.f;
        float* red = reinterpret_cast<float*>(sm + SQ::OFF_RED);
        RingPos<M3::NB> rb;
        for (int t = 0; t < ntiles; ++t) {
            const int eb = e0 + t * TE;
            bool stg_busy = t > 0;
            MIX3_T0();
            if (!OUTER && tid == 0 && eb + TE < e1)     // the next tile's V rows (one contiguous range) are pulled into L2 while this tile computes
                bulk_prefetch_l2(V + (size_t)(eb + TE) * 64 * DV, (uint32_t)min(TE, e1 - eb - TE) * 64 * DV * 4);
            float Vr[M3::EPS][DV];
            if constexpr (OUTER) {      // Y_j of the tile's edges once per tile (shared memory), then the rows v0 (x) Y in registers
                float* Ysw = reinterpret_cast<float*>(sm + SQ::OFF_YS);
                if (tid < TE) {
                    const int e = eb + tid;
                    float Y[9];
                    if (e < e1) {
                        const float rx = rvec[3 * (size_t)e], ry = rvec[3 * (size_t)e + 1], rz = rvec[3 * (size_t)e + 2];
                        const float inv = 1.f / sqrtf(rx * rx + ry * ry + rz * rz);
                        mix3_sph9(rx * inv, ry * inv, rz * inv, Y);
                    } else {
#pragma unroll
                        for (int j = 0; j < 9; ++j) Y[j] = 0.f;
                    }
#pragma unroll
                    for (int j = 0; j < 9; ++j) Ysw[tid * 9 + j] = Y[j];
                }
                float vv[M3::EPS];
#pragma unroll
                for (int i = 0; i < M3::EPS; ++i) {
                    const int e = eb + 4 * slot + i;
                    vv[i] = e < e1 ? v0[(size_t)e * 64 + ch] : 0.f;
                }
                asm volatile("bar.sync 3, %0;" ::"n"(M3::CT) : "memory");
#pragma unroll
                for (int i = 0; i < M3::EPS; ++i) {
#pragma unroll
                    for (int k = 0; k < DV; ++k) Vr[i][k] = 0.f;
#pragma unroll
                    for (int j = 0; j < 9; ++j) Vr[i][mix3_nat_slot(j)] = vv[i] * Ysw[(4 * slot + i) * 9 + j];
                }
            } else {
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
            }
            static_for3<0, NP>([&](auto kc) {
                constexpr int k = decltype(kc)::value;
                constexpr int p = SQ::path(k);
                using Pth = TPPath<2, p>;
                unsigned char* Bs = sm + SQ::OFF_B + rb.s * SQ::B_BYTES;
                // B: t_p of this thread's four edges, hi (raw) and lo
                MIX3_ACC(10, blockIdx.x == 0 && tid == 0 && k == 0);
                mbar_wait(&bars->b_empty[rb.s], rb.ph ^ 1u);
                if constexpr (SQ::ALIAS_STG) {   // first write of this tile into B stage 1, where the epilogue staged the previous tile's rows
                    if (stg_busy && rb.s == 1) { asm volatile("bar.sync 1, %0;" ::"n"(2 * M3::CT) : "memory"); stg_busy = false; }
                }
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
                        *reinterpret_cast<float*>(dst + SQ::BV_BYTES) = tf32_lo(tp[M]);
                    }
                }
                MIX3_ACC(5, blockIdx.x == 0 && tid == 0);
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars->b_full[rb.s]);
                rb.next();
                MIX3_ACC(7, blockIdx.x == 0 && tid == 0);
            });
            // ---- epilogue: TMEM lane (n', h) -> out rows; warp (q, wq) takes edges 8 wq .. 8 wq + 7, lane h its half of them
            mbar_wait(&bars->d_full, (uint32_t)t & 1u);
            MIX3_ACC(8, blockIdx.x == 0 && tid == 0);
            tc05::fence_after_sync();
            // Rows are staged through shared memory (B stage 1 is idle until path 1 of the next tile) so that they leave as
            // fully coalesced 16-byte stores: per warp a private [4 edges][16 channels][18] block, two half-tiles in turn.
            float* stg = reinterpret_cast<float*>(sm + (SQ::ALIAS_STG ? SQ::OFF_B + SQ::B_BYTES : SQ::OFF_STG)) + warp * (4 * 16 * DV);
            const uint32_t trow = tbase + ((uint32_t)(32 * q) << 16) + (uint32_t)(8 * wq);
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {     // edges 8 wq + 4 hf + {0..3}: lane half h finalises edges 2 h, 2 h + 1 of them
                float o[2][DV];
                static_for3<0, 6>([&](auto bc) {
                    constexpr int b = decltype(bc)::value;
                    constexpr int off3 = b == 0 ? 0 : b == 1 ? 1 : b == 2 ? 2 : b == 3 ? 5 : b == 4 ? 8 : 13;
                    constexpr int d3 = b < 2 ? 1 : b < 4 ? 3 : 5;
                    if constexpr (SQ::block_active(off3)) {
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
                    } else {   // no path into this block runs: its components are zeros
#pragma unroll
                        for (int M = 0; M < d3; ++M) { o[0][off3 + M] = 0.f; o[1][off3 + M] = 0.f; }
                    }
                });
                if (hf == 1) {   // all TMEM reads of this warp are done: the accumulators may be overwritten
                    tc05::fence_before_sync();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&bars->d_empty);
                }
                if (e_edge != nullptr) {   // energy partial of this lane quarter's 16 channels, per edge: xor tree inside the half-warp
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        float sq = 0.f;
#pragma unroll
                        for (int k = 0; k < DV; ++k) sq = fmaf(o[i][k], o[i][k], sq);
                        float ep = fmaf(0.5f * kappa, sq, qn * o[i][0]);
#pragma unroll
                        for (int sft = 8; sft > 0; sft >>= 1) ep += __shfl_xor_sync(0xffffffffu, ep, sft);
                        if (nl == 0) red[((t & 1) * 4 + q) * TE + 8 * wq + 4 * hf + 2 * h + i] = ep;
                    }
                }
                if (s_out != nullptr) {
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        const int e = eb + 8 * wq + 4 * hf + 2 * h + i;
                        if (e < e1) s_out[(size_t)e * 64 + 16 * q + nl] = o[i][0];
                    }
                }
                if (out != nullptr) {
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
            }
            if (e_edge != nullptr) {       // the four lane quarters' partials in order (double-buffered by tile parity)
                asm volatile("bar.sync 2, %0;" ::"n"(M3::CT) : "memory");
                if (tid < TE && eb + tid < e1) {
                    const float* rp4 = red + (t & 1) * 4 * TE + tid;
                    e_edge[eb + tid] = ((rp4[0] + rp4[TE]) + rp4[2 * TE]) + rp4[3 * TE];
                }
            }
            if constexpr (SQ::ALIAS_STG) asm volatile("bar.arrive 1, %0;" ::"n"(2 * M3::CT) : "memory");   // staging done; waited for before B stage 1 is rewritten
            MIX3_ACC(9, blockIdx.x == 0 && tid == 0);
        }
    }
    tc05::fence_before_sync();
    __syncthreads();
    if (warp == M3::CT / 32) tc05::tmem_dealloc(tbase, 512);
}


// =====================================================================================================================
// VJP.  gt_p[e, n, M] = sum_n' W_p[n', n] G[e, n', off3(p) + M] on the tensor cores, then the per-path CG VJP on the CUDA cores:
//   D_p[128 x N_b] = A_p[128 x 64] . B_b[N_b x 64]^T,   A_p rows = (input channel n, hi/lo) from the transposed weight image,
//   B_b rows = column (M, e) of block b: G[e, :, off3 + M] over the 64 output channels (K), hi and lo.
// All six blocks' B operands of a tile of TE = 16 edges stay in shared memory (the cotangent tile transposed once), the paths run
// in plan order, every D_p goes TMEM -> registers as soon as it is complete (ring of four accumulators), V rows and the gV rows
// of the thread's four (edge, channel) pairs live in registers for the whole tile.
struct Mix3B {
    static constexpr int DV = 18, DE = 9, P = 30;
    static constexpr int TE = 16, CT = 256;                        // 8 compute warps (<= 168 registers each) + 1 control warp
    static constexpr int ROWS = 288;                                // sum over blocks of d3 * TE
    static constexpr int G_ATOM = ROWS * 128, G_VAR = 2 * G_ATOM, G_BYTES = 2 * G_VAR;   // hi, lo: [2 K-atoms][288 rows][128 B]
    static constexpr int A_BYTES = 2 * 128 * 128, NA = 2, ND = 3;   // 30 paths = 10 turns of the accumulator ring: slot and parity depend on p only
    static constexpr int OFF_G = 0, OFF_A = G_BYTES, OFF_BAR = OFF_A + NA * A_BYTES;
    static constexpr int OFF_YS = OFF_BAR + 256;                    // OUTER mode: Y_j(rhat_e) of the tile's edges, [TE][9] floats
    static constexpr int SMEM = OFF_YS + 640 + 1024;
    // first row of a block's B operand, indexed by off3
    __host__ __device__ static constexpr int rowoff(int off3) {
        return off3 == 0 ? 0 : off3 == 1 ? 16 : off3 == 2 ? 32 : off3 == 5 ? 80 : off3 == 8 ? 128 : 208;
    }
    // TMEM columns: accumulator ring at 0, 80, 160; the V rows of a thread's four pairs (72 columns per warp row wq) at 320 ..
    static constexpr int VCOL = 320;
    __host__ __device__ static constexpr int off1(int p) { return Mix3::off1(p); }
    __host__ __device__ static constexpr int d1(int p) { return Mix3::d1(p); }
    // component k of a feature row -> row of the (M = 0, e = 0) element of its block + 16 M
    __host__ __device__ static constexpr int comprow(int k) {
        return k == 0 ? 0 : k == 1 ? 16 : k < 5 ? 32 + 16 * (k - 2) : k < 8 ? 80 + 16 * (k - 5) : k < 13 ? 128 + 16 * (k - 8) : 208 + 16 * (k - 13);
    }
};
struct Mix3BBars {
    uint64_t a_full[Mix3B::NA], a_empty[Mix3B::NA], d_full[Mix3B::ND], d_empty[Mix3B::ND], g_full;
    uint32_t tmem_slot;
};

// COT: G points at the forward result `out` and the cotangent of the A12 energy, q (x) delta_{k,0} + kappa out, is formed while the
// tile is staged (G never exists in HBM).  g_s (nullable, [E][64]): a compact cotangent of the 0e scalars that is ADDED to
// G[e][n'][0] while the tile is staged (the scalar latent update's VJP writes it; G itself is not modified).
// OUTER (layer-1 specialisation): V = v0 (x) Y(rhat) is generated on chip from rvec [E][3] and v0 [E][64] (see mix3_sph9) and gV is not
// stored: it is contracted at once into g_v0[e][n] = sum_j gV[e][n][slot j] Y_j(rhat_e) ([E][64]) and gYe[e][j] = sum_n gV[e][n][slot j]
// v0[e][n] ([E][9]; lanes by a fixed xor tree, the four lane quarters in order), what the edge embedding's VJP needs.
template <bool WANT_GV, uint32_t PMASK, bool COT, bool OUTER = false>
__global__ void __launch_bounds__(Mix3B::CT + 64, 1) mix3_bwd_kernel(const int* __restrict__ row_ptr, const int* __restrict__ items,
                                                                    const float* __restrict__ G, const float* __restrict__ V,
                                                                    const float* __restrict__ Eenv, const float* __restrict__ img,
                                                                    float* __restrict__ gV, float* __restrict__ gE_dst, int gE_by_item,
                                                                    const float* __restrict__ qvec, float kappa, const float* __restrict__ g_s,
                                                                    const float* __restrict__ rvec = nullptr, const float* __restrict__ v0 = nullptr,
                                                                    float* __restrict__ g_v0 = nullptr, float* __restrict__ gYe = nullptr) {
    static_assert(!OUTER || (WANT_GV && PMASK == Mix3::mask_natural_in()), "OUTER mode: natural-parity input paths, gV accumulated");
    using MB = Mix3B;
    using SQ = Mix3Seq<PMASK>;
    using Gen = TPGen<2>;
    constexpr int DV = MB::DV, DE = MB::DE, NP = SQ::count(), TE = MB::TE;
    extern __shared__ unsigned char smem_raw[];
    unsigned char* sm = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    Mix3BBars* bars = reinterpret_cast<Mix3BBars*>(sm + MB::OFF_BAR);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    int c, e0, e1;
    get_item(items, row_ptr, blockIdx.x, c, e0, e1);
    const int ntiles = (e1 - e0 + TE - 1) / TE;   // 0 for an empty item: only the zero gEenv row is written

    if (tid == 0) {
        for (int s = 0; s < MB::NA; ++s) { mbar_init(&bars->a_full[s], 1); mbar_init(&bars->a_empty[s], 1); }
        for (int s = 0; s < MB::ND; ++s) { mbar_init(&bars->d_full[s], 1); mbar_init(&bars->d_empty[s], MB::CT / 32); }
        mbar_init(&bars->g_full, MB::CT / 32);
        fence_mbar_init();
    }
    if (warp == MB::CT / 32) { tc05::tmem_alloc(&bars->tmem_slot, 512); tc05::tmem_relinquish(); }
    tc05::fence_before_sync();
    __syncthreads();
    tc05::fence_after_sync();
    const uint32_t tbase = bars->tmem_slot;

    if (warp >= MB::CT / 32) {
        if (warp == MB::CT / 32 && lane == 0) {
            // ---- weight images (TMA)
            RingPos<MB::NA> ra;
            for (int t = 0; t < ntiles; ++t)
                static_for3<0, NP>([&](auto kc) {
                    constexpr int p = SQ::path(decltype(kc)::value);
                    mbar_wait(&bars->a_empty[ra.s], ra.ph ^ 1u);
                    mbar_expect_tx(&bars->a_full[ra.s], Mix3::IMG_BYTES);
                    bulk_load(sm + MB::OFF_A + ra.s * MB::A_BYTES, reinterpret_cast<const unsigned char*>(img) + (size_t)p * Mix3::IMG_BYTES,
                              Mix3::IMG_BYTES, &bars->a_full[ra.s]);
                    ra.next();
                });
        } else if (warp == MB::CT / 32 + 1) {
            // ---- MMA issue: the whole warp walks the loop, one elected lane issues
            constexpr uint32_t id1 = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, 16);
            constexpr uint32_t id3 = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, 48);
            constexpr uint32_t id5 = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, 80);
            const uint32_t adesc0 = tc05::sdesc_lo(smem_u32(sm + MB::OFF_A)), gdesc0 = tc05::sdesc_lo(smem_u32(sm + MB::OFF_G));
            RingPos<MB::NA> ra;
            RingPos<MB::ND> rd;
            for (int t = 0; t < ntiles; ++t) {
                mbar_wait(&bars->g_full, (uint32_t)t & 1u);
                static_for3<0, NP>([&](auto kc) {
                    constexpr int p = SQ::path(decltype(kc)::value);
                    constexpr int d3 = Gen::d3(p), off3 = Gen::off3(p);
                    constexpr uint32_t idesc = d3 == 1 ? id1 : d3 == 3 ? id3 : id5;
                    mbar_wait(&bars->a_full[ra.s], ra.ph);
                    mbar_wait(&bars->d_empty[rd.s], rd.ph ^ 1u);
                    tc05::fence_after_sync();
                    const uint32_t dcol = tbase + rd.s * 80u;
                    if (tc05::elect_one()) {
                    uint32_t ad = adesc0 + ((ra.s * (uint32_t)MB::A_BYTES) >> 4), gd = gdesc0;   // opaque per path: otherwise all descriptor words are hoisted out of the loops and spilled
                    asm volatile("" : "+r"(ad), "+r"(gd));
#pragma unroll
                    for (int v = 0; v < 2; ++v)
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const uint32_t koff = (uint32_t)(((j >> 2) * 16384 + (j & 3) * 32) >> 4);
                            const uint32_t goff = (uint32_t)((v * MB::G_VAR + (j >> 2) * MB::G_ATOM + MB::rowoff(off3) * 128 + (j & 3) * 32) >> 4);
                            tc05::mma_tf32_lo(dcol, ad + koff, gd + goff, tc05::kSdescHiSw128, idesc, (v == 0 && j == 0) ? 0u : 1u);
                        }
                    tc05::mma_commit(&bars->d_full[rd.s]);
                    tc05::mma_commit(&bars->a_empty[ra.s]);
                    }
                    __syncwarp();
                    ra.next();
                    rd.next();
                });
            }
        }
    } else {
        // ---- compute warps.  VJP mapping = TMEM lane: channel n = 16 q + nl, hi/lo partner lane ^ 16; warp (q, wq) reads the columns
        // of edges 8 wq .. 8 wq + 7, lane half h finalises edges 8 wq + 4 h + {0..3}.
        const int q = warp & 3, wq = warp >> 2, h = lane >> 4, nl = lane & 15, n = 16 * q + nl;
        float E[DE], gE[DE];
#pragma unroll
        for (int j = 0; j < DE; ++j) { E[j] = Eenv[((size_t)c * 64 + n) * DE + j]; gE[j] = 0.f; }
        // operand mapping: thread = (slot, n'), rows of edges 4 slot + j; byte offset of element (row of e, k = n') for M = 0, block row 0
        const int np = tid & 63, slot = tid >> 6;
        float qn = 0.f;
        if constexpr (COT) qn = qvec[np];
        uint32_t goff[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t e = 4u * slot + j, r = e & 7u;
            goff[j] = (uint32_t)(np >> 5) * MB::G_ATOM + (e >> 3) * 1024u + r * 128u + (((((uint32_t)np & 31u) >> 2) ^ r) << 4) + (((uint32_t)np & 3u) << 2);
        }
        RingPos<MB::ND> rd;
        for (int t = 0; t < ntiles; ++t) {
            const int eb = e0 + t * TE;
            if (tid == 0 && eb + TE < e1) {   // the next tile's cotangent and V rows are pulled into L2 while this tile computes
                const uint32_t nb = (uint32_t)min(TE, e1 - eb - TE) * 64 * DV * 4;
                if (G != nullptr) bulk_prefetch_l2(G + (size_t)(eb + TE) * 64 * DV, nb);
                if (!OUTER) bulk_prefetch_l2(V + (size_t)(eb + TE) * 64 * DV, nb);
            }
            // (a) cotangent tile -> B operands of all six blocks (hi, lo)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int e = eb + 4 * slot + j;
                float g[DV];
                if (e < e1) {
                    if (COT && G == nullptr) {       // kappa == 0: the cotangent is q (x) delta_{k,0}, nothing to read
#pragma unroll
                        for (int k = 0; k < DV; ++k) g[k] = 0.f;
                        g[0] = qn;
                    } else {
                        row_load<float, DV>(G + ((size_t)e * 64 + np) * DV, g);
                        if constexpr (COT) {
#pragma unroll
                            for (int k = 0; k < DV; ++k) g[k] *= kappa;
                            g[0] += qn;
                        }
                    }
                    if (g_s != nullptr) g[0] += g_s[(size_t)e * 64 + np];
                } else {
#pragma unroll
                    for (int k = 0; k < DV; ++k) g[k] = 0.f;
                }
                static_for3<0, DV>([&](auto kc) {   // only the blocks some active path reads
                    constexpr int k = decltype(kc)::value;
                    constexpr int off3k = k == 0 ? 0 : k == 1 ? 1 : k < 5 ? 2 : k < 8 ? 5 : k < 13 ? 8 : 13;
                    if constexpr (SQ::block_active(off3k)) {
                        unsigned char* dst = sm + MB::OFF_G + goff[j] + (MB::comprow(k) / 8) * 1024;
                        *reinterpret_cast<float*>(dst) = g[k];
                        *reinterpret_cast<float*>(dst + MB::G_VAR) = tf32_lo(g[k]);
                    }
                });
            }
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars->g_full);
            // (b) V rows of this thread's four pairs parked in this thread's TMEM lane (columns VCOL + 72 wq + 18 i + k): registers
            // hold the gV accumulators; each path reads back only the (l1, p1) block it contracts
            float gv[4][DV];
            const uint32_t vrow = tbase + ((uint32_t)(32 * q) << 16) + (uint32_t)(MB::VCOL + 72 * wq);
            [[maybe_unused]] float v0r[4];
            [[maybe_unused]] const float* Ys = reinterpret_cast<const float*>(sm + MB::OFF_YS);
            if constexpr (OUTER) {
                if (tid < TE) {      // Y_j of the tile's edges, once per tile
                    float* Yw = reinterpret_cast<float*>(sm + MB::OFF_YS) + tid * 9;
                    const int e = eb + tid;
                    float Y[9];
                    if (e < e1) {
                        const float rx = rvec[3 * (size_t)e], ry = rvec[3 * (size_t)e + 1], rz = rvec[3 * (size_t)e + 2];
                        const float inv = 1.f / sqrtf(rx * rx + ry * ry + rz * rz);
                        mix3_sph9(rx * inv, ry * inv, rz * inv, Y);
                    } else {
#pragma unroll
                        for (int j = 0; j < 9; ++j) Y[j] = 0.f;
                    }
#pragma unroll
                    for (int j = 0; j < 9; ++j) Yw[j] = Y[j];
                }
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int e = eb + 8 * wq + 4 * h + i;
                    v0r[i] = e < e1 ? v0[(size_t)e * 64 + n] : 0.f;
#pragma unroll
                    for (int k = 0; k < DV; ++k) gv[i][k] = 0.f;
                }
                named_bar(1, MB::CT);   // Ys visible to every compute warp
            } else {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int e = eb + 8 * wq + 4 * h + i;
                float vr[DV];
                if (e < e1) {
                    row_load<float, DV>(V + ((size_t)e * 64 + n) * DV, vr);
                } else {
#pragma unroll
                    for (int k = 0; k < DV; ++k) vr[k] = 0.f;
                }
                uint32_t lo16[16], hi2[2];
#pragma unroll
                for (int k = 0; k < 16; ++k) lo16[k] = __float_as_uint(vr[k]);
                hi2[0] = __float_as_uint(vr[16]); hi2[1] = __float_as_uint(vr[17]);
                tc05::tmem_st16(vrow + (uint32_t)(18 * i), lo16);
                tc05::tmem_st2(vrow + (uint32_t)(18 * i + 16), hi2);
#pragma unroll
                for (int k = 0; k < DV; ++k) gv[i][k] = 0.f;
            }
            tc05::tmem_st_wait();
            }
            // (c) paths: consume every accumulator as soon as it is complete
            static_for3<0, NP>([&](auto kc) {
                constexpr int p = SQ::path(decltype(kc)::value);
                using Pth = TPPath<2, p>;
                constexpr int d3 = Pth::D3;
                const uint32_t sd = rd.s;
                mbar_wait(&bars->d_full[sd], rd.ph);
                rd.next();
                tc05::fence_after_sync();
                constexpr int o1 = MB::off1(p), w1 = MB::d1(p);
                uint32_t v[d3][8];
                const uint32_t trow = tbase + ((uint32_t)(32 * q) << 16) + sd * 80u + (uint32_t)(8 * wq);
#pragma unroll
                for (int M = 0; M < d3; ++M) tc05::tmem_ld8(trow + (uint32_t)(M * TE), v[M]);
                float Vb[4][DV];   // only components o1 .. o1 + w1 - 1 are read by this path's code
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    if constexpr (OUTER) {
#pragma unroll
                        for (int k = 0; k < w1; ++k) Vb[i][o1 + k] = v0r[i] * Ys[(8 * wq + 4 * h + i) * 9 + mix3_nat_j(o1 + k)];
                    } else if constexpr (w1 == 1) {
                        uint32_t x[1];
                        tc05::tmem_ld1(vrow + (uint32_t)(18 * i + o1), x);
                        Vb[i][o1] = __uint_as_float(x[0]);
                    } else if constexpr (w1 == 3) {
                        uint32_t x[4];
                        tc05::tmem_ld4(vrow + (uint32_t)(18 * i + o1), x);
#pragma unroll
                        for (int k = 0; k < 3; ++k) Vb[i][o1 + k] = __uint_as_float(x[k]);
                    } else {
                        uint32_t x[4], y[1];
                        tc05::tmem_ld4(vrow + (uint32_t)(18 * i + o1), x);
                        tc05::tmem_ld1(vrow + (uint32_t)(18 * i + o1 + 4), y);
#pragma unroll
                        for (int k = 0; k < 4; ++k) Vb[i][o1 + k] = __uint_as_float(x[k]);
                        Vb[i][o1 + 4] = __uint_as_float(y[0]);
                    }
                }
                tc05::tmem_ld_wait();
                tc05::fence_before_sync();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars->d_empty[sd]);
#pragma unroll
                for (int j = 0; j < DE; ++j) asm volatile("" : "+f"(E[j]));
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    float gt[d3];
#pragma unroll
                    for (int M = 0; M < d3; ++M) {
                        const float mine = __uint_as_float(h ? v[M][4 + i] : v[M][i]);
                        const float send = __uint_as_float(h ? v[M][i] : v[M][4 + i]);
                        gt[M] = mine + __shfl_xor_sync(0xffffffffu, send, 16);
                    }
                    Pth::template bwd<float, WANT_GV>(Vb[i], E, gt, gv[i], gE);
                }
            });
            // (d) OUTER: gV is contracted with Y (-> g_v0) and with v0 over the 64 channels (-> gYe) instead of being stored
            if constexpr (OUTER) {
                float* redY = reinterpret_cast<float*>(sm + MB::OFF_G);   // [4 lane quarters][TE][9] in the (now idle) operand region
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int el = 8 * wq + 4 * h + i, e = eb + el;
                    float sv = 0.f;
#pragma unroll
                    for (int j = 0; j < 9; ++j) sv = fmaf(gv[i][mix3_nat_slot(j)], Ys[el * 9 + j], sv);
                    if (e < e1) g_v0[(size_t)e * 64 + n] = sv;
#pragma unroll
                    for (int j = 0; j < 9; ++j) {
                        float pj = gv[i][mix3_nat_slot(j)] * v0r[i];
#pragma unroll
                        for (int o = 8; o > 0; o >>= 1) pj += __shfl_xor_sync(0xffffffffu, pj, o);
                        if (nl == 0) redY[(q * TE + el) * 9 + j] = pj;
                    }
                }
                named_bar(1, MB::CT);
                if (tid < TE * 9) {
                    const int el = tid / 9, j = tid - el * 9;
                    if (eb + el < e1)
                        gYe[(size_t)(eb + el) * 9 + j] = ((redY[(0 * TE + el) * 9 + j] + redY[(1 * TE + el) * 9 + j]) + redY[(2 * TE + el) * 9 + j]) +
                                                         redY[(3 * TE + el) * 9 + j];
                }
            } else if constexpr (WANT_GV) {
                float* stg = reinterpret_cast<float*>(sm + MB::OFF_G) + warp * (8 * 16 * DV);
#pragma unroll
                for (int i = 0; i < 4; ++i) row_store<float, DV>(stg + ((4 * h + i) * 16 + nl) * DV, gv[i]);
                __syncwarp();
                const int ebase = eb + 8 * wq;
#pragma unroll
                for (int r = 0; r < 18; ++r) {   // 8 edges x 288 floats = 576 float4
                    const int idx = lane + 32 * r, el = idx / 72, w4 = idx - el * 72;
                    if (ebase + el < e1)
                        *reinterpret_cast<float4*>(gV + ((size_t)(ebase + el) * 64 + 16 * q) * DV + 4 * w4) = reinterpret_cast<const float4*>(stg)[idx];
                }
            }
            named_bar(1, MB::CT);   // operand region free for the next tile's cotangent (all MMAs of this tile have completed)
        }
        // ---- gEenv: lane halves by shuffle, the two edge groups (wq) through shared memory, fixed order
#pragma unroll
        for (int j = 0; j < DE; ++j) gE[j] += __shfl_xor_sync(0xffffffffu, gE[j], 16);
        float* red = reinterpret_cast<float*>(sm + MB::OFF_G);
        if (wq == 1 && h == 0) {
#pragma unroll
            for (int j = 0; j < DE; ++j) red[n * DE + j] = gE[j];
        }
        named_bar(1, MB::CT);
        if (wq == 0 && h == 0) {
            float* dst = gE_dst + ((size_t)(gE_by_item ? (long)blockIdx.x : (long)c) * 64 + n) * DE;
#pragma unroll
            for (int j = 0; j < DE; ++j) dst[j] = gE[j] + red[n * DE + j];
        }
    }
    tc05::fence_before_sync();
    __syncthreads();
    if (warp == MB::CT / 32) { __syncwarp(); tc05::tmem_dealloc(tbase, 512); }
}

}  // namespace allegro
