// tclin.cu -- the scalar latent update of the two-layer model (reading A19) on the tensor cores, fp32, n = 64, compact scalars:
//   forward : z[e][o] = sum_i A[o][i] [x ; s][e][i]   (K = 128, N = 64),  x_new = u(|r_e| / r_c) SiLU(z)
//   VJP     : g_z = g_xnew u SiLU'(z);  [g_x ; g_s +=][e][i] = sum_o g_z[e][o] A[o][i]   (K = 64, N = 128);  g_rvec += (sum_o g_xnew SiLU(z)) u' rhat / r_c
// These are dense contractions with 16 flops per byte of HBM traffic: more than the FP32 FMA pipe can feed at the HBM rate
// (model.cu's register-tiled kernels run them at 0.2-0.25 of the HBM roof), so they belong on tcgen05.  fp32 accuracy: both operands
// are split into a tf32 "hi" part (the raw word: the tensor core ignores the low 13 mantissa bits) and the exact remainder "lo";
// D = A_hi B_hi + A_lo B_hi + A_hi B_lo in the fp32 TMEM accumulator (the lo x lo term is below fp32 rounding).
//
// One persistent CTA per SM, tiles of 128 edges = the 128 TMEM lanes.  Per tile: all 8 warps load the rows (lanes along K, fully
// coalesced), split them and store the two A images in the 128-byte-swizzled K-major layout tcgen05 reads; one thread issues the
// MMAs; the warps read the accumulator back (thread = edge row), apply the elementwise part and store whole rows.
#include "common.cuh"
#include "launch.h"
#include "tc05.cuh"

namespace allegro {

namespace {

constexpr int kTcTile = 128, kTcThreads = 256;
constexpr int kAtomA = kTcTile * 128;          // bytes of one 32-float K slab of a 128-row operand
__device__ __forceinline__ float tc_lo(float x) { return x - __uint_as_float(__float_as_uint(x) & 0xffffe000u); }

template <typename T>
__device__ __forceinline__ T tc_cutoff(T xr, T& du) {  // u(x) = 1 - 28x^6 + 48x^7 - 21x^8 and du/dx (reading A8)
    const T x2 = xr * xr, x5 = x2 * x2 * xr, x6 = x5 * xr, x7 = x6 * xr, x8 = x7 * xr;
    du = T(-168) * x5 + T(336) * x6 - T(168) * x7;
    T u = T(1) - T(28) * x6 + T(48) * x7 - T(21) * x8;
    if (xr >= T(1)) { u = T(0); du = T(0); }
    return u;
}

// store four consecutive K values (chunk c of the row: K = 4 c .. 4 c + 3) of operand row r as hi and lo images
__device__ __forceinline__ void tc_store_split(unsigned char* hi, unsigned char* lo, int atom_bytes, int r, int c, float4 v) {
    const uint32_t off = (uint32_t)(c >> 3) * (uint32_t)atom_bytes + tc05::sw128_off((uint32_t)r, (uint32_t)(c & 7));
    *reinterpret_cast<float4*>(hi + off) = v;
    *reinterpret_cast<float4*>(lo + off) = make_float4(tc_lo(v.x), tc_lo(v.y), tc_lo(v.z), tc_lo(v.w));
}

// the three products of the split: nk = K / 8 MMA steps each; A / B: shared-memory addresses of the hi images, lo images follow at +a_lo / +b_lo
__device__ __forceinline__ void tc_issue(uint32_t d_tmem, uint32_t a_hi, uint32_t a_lo, uint32_t b_hi, uint32_t b_lo, int b_atom, int nk, uint32_t idesc) {
    uint32_t acc = 0;
#pragma unroll
    for (int prod = 0; prod < 3; ++prod) {
        const uint32_t a = prod == 1 ? a_lo : a_hi, b = prod == 2 ? b_lo : b_hi;
        for (int j = 0; j < nk; ++j) {
            const uint32_t aoff = (uint32_t)((j >> 2) * kAtomA + (j & 3) * 32), boff = (uint32_t)((j >> 2) * b_atom + (j & 3) * 32);
            tc05::mma_tf32(d_tmem, tc05::sdesc_sw128(a + aoff), tc05::sdesc_sw128(b + boff), idesc, acc);
            acc = 1;
        }
    }
}

struct TcBars {
    uint64_t done;
    uint32_t tmem_slot;
};

// ---------------------------------------------------------------------------------------------------------------- forward
// shared memory (1024-byte aligned): A_hi [4 slabs][128 rows x 128 B] | A_lo | B_hi [4 slabs][64 rows x 128 B] | B_lo | u[128] | barriers
constexpr int kFwdAhi = 0, kFwdAlo = 4 * kAtomA, kFwdBhi = 8 * kAtomA, kFwdBatom = 64 * 128, kFwdBlo = kFwdBhi + 4 * kFwdBatom;
constexpr int kFwdU = kFwdBlo + 4 * kFwdBatom, kFwdBars = kFwdU + kTcTile * 4, kFwdSmem = kFwdBars + 64 + 1024;

__global__ void __launch_bounds__(kTcThreads, 1) tc_latent_fwd_kernel(long E, float rc, const float* __restrict__ rvec, const float* __restrict__ x,
                                                                       const float* __restrict__ s, const float* __restrict__ A,
                                                                       float* __restrict__ z, float* __restrict__ x_new) {
    extern __shared__ unsigned char tc_raw[];
    unsigned char* sm = tc_raw + ((1024u - (smem_u32(tc_raw) & 1023u)) & 1023u);     // 1024-byte aligned, still a shared-window pointer (STS, not ST)
    float* us = reinterpret_cast<float*>(sm + kFwdU);
    TcBars* bars = reinterpret_cast<TcBars*>(sm + kFwdBars);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (warp == 0) {
        tc05::tmem_alloc(&bars->tmem_slot, 64);
        tc05::tmem_relinquish();
    }
    if (tid == 0) {
        mbar_init(&bars->done, 1);
        fence_mbar_init();
    }
    // B = the weights A[o][0..127], row o: 64 rows x 32 chunks, once per CTA
    for (int idx = tid; idx < 64 * 32; idx += kTcThreads) {
        const int o = idx >> 5, c = idx & 31;
        tc_store_split(sm + kFwdBhi, sm + kFwdBlo, kFwdBatom, o, c, *reinterpret_cast<const float4*>(A + (size_t)o * 128 + 4 * c));
    }
    fence_proxy_async();
    tc05::fence_before_sync();
    __syncthreads();
    tc05::fence_after_sync();
    const uint32_t tbase = bars->tmem_slot;
    const uint32_t idesc = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, 64);
    const uint32_t sbase = smem_u32(sm);
    uint32_t phase = 0;
    // rows 16 warp .. + 15: lane l holds chunk l of [x ; s] (K = 4 l .. 4 l + 3): two fully coalesced 256-byte row halves.  The rows of
    // the NEXT tile are loaded into registers right after this tile's MMAs are issued, so that their latency hides behind the MMAs
    // and the epilogue (one CTA per SM: nothing else would cover it)
    const float* src = lane < 16 ? x : s;
    float4 v[16];
    float r3[3] = {1.f, 0.f, 0.f};      // edge vector of row tid (threads 0..127 form the cutoff values)
    auto load_rows = [&](long eb) {
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const long e = eb + 16 * warp + i;
            v[i] = e < E ? *reinterpret_cast<const float4*>(src + (size_t)e * 64 + 4 * (lane & 15)) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
        if (tid < kTcTile && eb + tid < E) {
            r3[0] = rvec[3 * (eb + tid)]; r3[1] = rvec[3 * (eb + tid) + 1]; r3[2] = rvec[3 * (eb + tid) + 2];
        }
    };
    load_rows((long)blockIdx.x * kTcTile);
    for (long eb = (long)blockIdx.x * kTcTile; eb < E; eb += (long)gridDim.x * kTcTile) {
#pragma unroll
        for (int i = 0; i < 16; ++i) tc_store_split(sm + kFwdAhi, sm + kFwdAlo, kAtomA, 16 * warp + i, lane, v[i]);
        if (tid < kTcTile) {
            float du, u = 0.f;
            if (eb + tid < E) u = tc_cutoff<float>(sqrtf(r3[0] * r3[0] + r3[1] * r3[1] + r3[2] * r3[2]) / rc, du);
            us[tid] = u;
        }
        fence_proxy_async();
        __syncthreads();
        if (warp == 0) {
            if (tc05::elect_one()) {
                tc05::fence_after_sync();
                tc_issue(tbase, sbase + kFwdAhi, sbase + kFwdAlo, sbase + kFwdBhi, sbase + kFwdBlo, kFwdBatom, 16, idesc);
                tc05::mma_commit(&bars->done);
            }
            __syncwarp();
        }
        load_rows(eb + (long)gridDim.x * kTcTile);
        mbar_wait(&bars->done, phase);
        phase ^= 1u;
        tc05::fence_after_sync();
        // accumulator row = edge (TMEM lane 32 q + lane), this warp's half of the 64 outputs
        {
            const int q = warp & 3, hc = warp >> 2, r = 32 * q + lane;
            const long e = eb + r;
            const float u = us[r];
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                uint32_t w[16];
                tc05::tmem_ld16(tbase + ((uint32_t)(32 * q) << 16) + (uint32_t)(32 * hc + 16 * g), w);
                tc05::tmem_ld_wait();
                if (e < E) {
                    float zz[16], xn[16];
#pragma unroll
                    for (int k = 0; k < 16; ++k) {
                        zz[k] = __uint_as_float(w[k]);
                        xn[k] = u * zz[k] * (1.f / (1.f + expf(-zz[k])));
                    }
                    float4* zd = reinterpret_cast<float4*>(z + (size_t)e * 64 + 32 * hc + 16 * g);
                    float4* xd = reinterpret_cast<float4*>(x_new + (size_t)e * 64 + 32 * hc + 16 * g);
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        zd[k] = make_float4(zz[4 * k], zz[4 * k + 1], zz[4 * k + 2], zz[4 * k + 3]);
                        xd[k] = make_float4(xn[4 * k], xn[4 * k + 1], xn[4 * k + 2], xn[4 * k + 3]);
                    }
                }
            }
        }
        tc05::fence_before_sync();
        __syncthreads();     // the accumulator and the A images are free for the next tile
    }
    if (warp == 0) tc05::tmem_dealloc(tbase, 64);
}

// -------------------------------------------------------------------------------------------------------------------- VJP
// A operand = g_z [128 edges][K = 64 outputs of the forward map], formed by the loading warps; B = A^T: row i (the 128 inputs), K = o.
// shared memory: A_hi [2 slabs][128 x 128 B] | A_lo | B_hi [2 slabs][128 x 128 B] | B_lo | radial factor per edge [128] | barriers
constexpr int kBwdAhi = 0, kBwdAlo = 2 * kAtomA, kBwdBhi = 4 * kAtomA, kBwdBlo = 6 * kAtomA, kBwdSc = 8 * kAtomA, kBwdBars = kBwdSc + kTcTile * 4,
              kBwdSmem = kBwdBars + 64 + 1024;

__global__ void __launch_bounds__(kTcThreads, 1) tc_latent_bwd_kernel(long E, float rc, const float* __restrict__ rvec, const float* __restrict__ z,
                                                                       const float* __restrict__ g_xnew, const float* __restrict__ A,
                                                                       float* __restrict__ g_x, float* __restrict__ g_s, float* __restrict__ g_rvec) {
    extern __shared__ unsigned char tc_raw[];
    unsigned char* sm = tc_raw + ((1024u - (smem_u32(tc_raw) & 1023u)) & 1023u);     // 1024-byte aligned, still a shared-window pointer (STS, not ST)
    TcBars* bars = reinterpret_cast<TcBars*>(sm + kBwdBars);
    float* scs = reinterpret_cast<float*>(sm + kBwdSc);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (warp == 0) {
        tc05::tmem_alloc(&bars->tmem_slot, 128);
        tc05::tmem_relinquish();
    }
    if (tid == 0) {
        mbar_init(&bars->done, 1);
        fence_mbar_init();
    }
    // B[i][o] = A[o][i]: rows of A read coalesced, scattered into row i, K position o
    for (int idx = tid; idx < 64 * 128; idx += kTcThreads) {
        const int o = idx >> 7, i = idx & 127, c = o >> 2;
        const float a = A[idx];
        const uint32_t off = (uint32_t)(c >> 3) * (uint32_t)kAtomA + tc05::sw128_off((uint32_t)i, (uint32_t)(c & 7)) + (uint32_t)(o & 3) * 4u;
        *reinterpret_cast<float*>(sm + kBwdBhi + off) = a;
        *reinterpret_cast<float*>(sm + kBwdBlo + off) = tc_lo(a);
    }
    fence_proxy_async();
    tc05::fence_before_sync();
    __syncthreads();
    tc05::fence_after_sync();
    const uint32_t tbase = bars->tmem_slot;
    const uint32_t idesc = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, 128);
    const uint32_t sbase = smem_u32(sm);
    uint32_t phase = 0;
    // half-warp per row: rows 16 warp + 2 i + (lane >> 4), chunk c = lane & 15 (outputs 4 c .. 4 c + 3); the next tile's rows are
    // prefetched into registers behind the MMAs and the epilogue, as in the forward kernel
    const int c = lane & 15;
    float4 zv[8], gv[8];
    float rr3[8][3];
    auto load_rows = [&](long eb) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const long e = eb + 16 * warp + 2 * i + (lane >> 4);
            if (e < E) {
                zv[i] = *reinterpret_cast<const float4*>(z + (size_t)e * 64 + 4 * c);
                gv[i] = *reinterpret_cast<const float4*>(g_xnew + (size_t)e * 64 + 4 * c);
                rr3[i][0] = rvec[3 * e]; rr3[i][1] = rvec[3 * e + 1]; rr3[i][2] = rvec[3 * e + 2];
            } else {
                zv[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                gv[i] = zv[i];
                rr3[i][0] = 1.f; rr3[i][1] = 0.f; rr3[i][2] = 0.f;
            }
        }
    };
    load_rows((long)blockIdx.x * kTcTile);
    for (long eb = (long)blockIdx.x * kTcTile; eb < E; eb += (long)gridDim.x * kTcTile) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int r = 16 * warp + 2 * i + (lane >> 4);
            const long e = eb + r;
            float u = 0.f, dus = 0.f;
            if (e < E) {
                const float rr = sqrtf(rr3[i][0] * rr3[i][0] + rr3[i][1] * rr3[i][1] + rr3[i][2] * rr3[i][2]);
                float du;
                u = tc_cutoff<float>(rr / rc, du);
                dus = du / rc / rr;
            }
            const float zz[4] = {zv[i].x, zv[i].y, zv[i].z, zv[i].w}, gg[4] = {gv[i].x, gv[i].y, gv[i].z, gv[i].w};
            float gz[4], sv = 0.f;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float sg = 1.f / (1.f + expf(-zz[k]));
                gz[k] = gg[k] * u * (sg * (1.f + zz[k] * (1.f - sg)));
                sv += gg[k] * zz[k] * sg;
            }
            tc_store_split(sm + kBwdAhi, sm + kBwdAlo, kAtomA, r, c, make_float4(gz[0], gz[1], gz[2], gz[3]));
            // radial term: sum over the 64 outputs = fixed xor tree over the row's 16 lanes
#pragma unroll
            for (int sft = 8; sft > 0; sft >>= 1) sv += __shfl_xor_sync(0xffffffffu, sv, sft);
            if (c == 0) scs[r] = sv * dus;      // the edge's g_rvec update follows below, one thread per edge (independent loads)
        }
        fence_proxy_async();
        __syncthreads();
        if (warp == 0) {
            if (tc05::elect_one()) {
                tc05::fence_after_sync();
                tc_issue(tbase, sbase + kBwdAhi, sbase + kBwdAlo, sbase + kBwdBhi, sbase + kBwdBlo, kAtomA, 8, idesc);
                tc05::mma_commit(&bars->done);
            }
            __syncwarp();
        }
        // while the MMAs run: the radial term of this tile's edges, the old scalar cotangent rows of the warps that add to them,
        // and the next tile's rows
        if (tid < kTcTile && eb + tid < E) {
            const long e = eb + tid;
            const float sc = scs[tid];
            g_rvec[3 * e] += sc * rvec[3 * e];
            g_rvec[3 * e + 1] += sc * rvec[3 * e + 1];
            g_rvec[3 * e + 2] += sc * rvec[3 * e + 2];
        }
        const int q = warp & 3, hc = warp >> 2;
        const long er = eb + 32 * q + lane;
        float* dst = (hc ? g_s : g_x) + (size_t)(er < E ? er : 0) * 64;
        float4 old[16];
        if (hc) {
#pragma unroll
            for (int k = 0; k < 16; ++k) old[k] = er < E ? reinterpret_cast<const float4*>(dst)[k] : make_float4(0.f, 0.f, 0.f, 0.f);
        }
        load_rows(eb + (long)gridDim.x * kTcTile);
        mbar_wait(&bars->done, phase);
        phase ^= 1u;
        tc05::fence_after_sync();
        // columns 0..63 = g_x (overwritten), 64..127 = the compact scalar cotangent (added to)
#pragma unroll
        for (int g = 0; g < 4; ++g) {
            uint32_t w[16];
            tc05::tmem_ld16(tbase + ((uint32_t)(32 * q) << 16) + (uint32_t)(64 * hc + 16 * g), w);
            tc05::tmem_ld_wait();
            if (er < E) {
                float4* d4 = reinterpret_cast<float4*>(dst + 16 * g);
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    float4 o = make_float4(__uint_as_float(w[4 * k]), __uint_as_float(w[4 * k + 1]), __uint_as_float(w[4 * k + 2]), __uint_as_float(w[4 * k + 3]));
                    if (hc) {
                        o.x += old[4 * g + k].x; o.y += old[4 * g + k].y; o.z += old[4 * g + k].z; o.w += old[4 * g + k].w;
                    }
                    d4[k] = o;
                }
            }
        }
        tc05::fence_before_sync();
        __syncthreads();
    }
    if (warp == 0) tc05::tmem_dealloc(tbase, 128);
}

// ------------------------------------------------------------------------------------------------- linear map, K = N = 64
// y[e][o] (+)= sum_i x[e][i] W[o][i] (transpose_w == 0) or sum_i x[e][i] W[i][o] (transpose_w == 1): the per-edge linear of the stacked
// model when the embedding is not factorised (reading A19) and its VJP.  Same scheme as above; 96 KB of images: two CTAs per SM.
constexpr int kLinAhi = 0, kLinAlo = 2 * kAtomA, kLinBhi = 4 * kAtomA, kLinBatom = 64 * 128, kLinBlo = kLinBhi + 2 * kLinBatom,
              kLinBars = kLinBlo + 2 * kLinBatom, kLinSmem = kLinBars + 64 + 1024;

__global__ void __launch_bounds__(kTcThreads, 2) tc_linear64_kernel(long E, const float* __restrict__ x, const float* __restrict__ W, int transpose_w,
                                                                     int accumulate, float* __restrict__ y) {
    extern __shared__ unsigned char tc_raw[];
    unsigned char* sm = tc_raw + ((1024u - (smem_u32(tc_raw) & 1023u)) & 1023u);
    TcBars* bars = reinterpret_cast<TcBars*>(sm + kLinBars);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (warp == 0) {
        tc05::tmem_alloc(&bars->tmem_slot, 64);
        tc05::tmem_relinquish();
    }
    if (tid == 0) {
        mbar_init(&bars->done, 1);
        fence_mbar_init();
    }
    // B row o (an output), K position i (an input)
    for (int idx = tid; idx < 64 * 64; idx += kTcThreads) {
        const int o = transpose_w ? (idx & 63) : (idx >> 6), i = transpose_w ? (idx >> 6) : (idx & 63), c = i >> 2;
        const float a = W[idx];
        const uint32_t off = (uint32_t)(c >> 3) * (uint32_t)kLinBatom + tc05::sw128_off((uint32_t)o, (uint32_t)(c & 7)) + (uint32_t)(i & 3) * 4u;
        *reinterpret_cast<float*>(sm + kLinBhi + off) = a;
        *reinterpret_cast<float*>(sm + kLinBlo + off) = tc_lo(a);
    }
    fence_proxy_async();
    tc05::fence_before_sync();
    __syncthreads();
    tc05::fence_after_sync();
    const uint32_t tbase = bars->tmem_slot;
    const uint32_t idesc = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, 64);
    const uint32_t sbase = smem_u32(sm);
    uint32_t phase = 0;
    const int c = lane & 15;
    float4 xv[8];
    auto load_rows = [&](long eb) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const long e = eb + 16 * warp + 2 * i + (lane >> 4);
            xv[i] = e < E ? *reinterpret_cast<const float4*>(x + (size_t)e * 64 + 4 * c) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
    };
    load_rows((long)blockIdx.x * kTcTile);
    for (long eb = (long)blockIdx.x * kTcTile; eb < E; eb += (long)gridDim.x * kTcTile) {
#pragma unroll
        for (int i = 0; i < 8; ++i) tc_store_split(sm + kLinAhi, sm + kLinAlo, kAtomA, 16 * warp + 2 * i + (lane >> 4), c, xv[i]);
        fence_proxy_async();
        __syncthreads();
        if (warp == 0) {
            if (tc05::elect_one()) {
                tc05::fence_after_sync();
                tc_issue(tbase, sbase + kLinAhi, sbase + kLinAlo, sbase + kLinBhi, sbase + kLinBlo, kLinBatom, 8, idesc);
                tc05::mma_commit(&bars->done);
            }
            __syncwarp();
        }
        load_rows(eb + (long)gridDim.x * kTcTile);
        const int q = warp & 3, hc = warp >> 2;
        const long er = eb + 32 * q + lane;
        float* dst = y + (size_t)(er < E ? er : 0) * 64 + 32 * hc;
        float4 old[8];
        if (accumulate) {
#pragma unroll
            for (int k = 0; k < 8; ++k) old[k] = er < E ? reinterpret_cast<const float4*>(dst)[k] : make_float4(0.f, 0.f, 0.f, 0.f);
        }
        mbar_wait(&bars->done, phase);
        phase ^= 1u;
        tc05::fence_after_sync();
#pragma unroll
        for (int g = 0; g < 2; ++g) {
            uint32_t w[16];
            tc05::tmem_ld16(tbase + ((uint32_t)(32 * q) << 16) + (uint32_t)(32 * hc + 16 * g), w);
            tc05::tmem_ld_wait();
            if (er < E) {
                float4* d4 = reinterpret_cast<float4*>(dst + 16 * g);
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    float4 o = make_float4(__uint_as_float(w[4 * k]), __uint_as_float(w[4 * k + 1]), __uint_as_float(w[4 * k + 2]), __uint_as_float(w[4 * k + 3]));
                    if (accumulate) {
                        o.x += old[4 * g + k].x; o.y += old[4 * g + k].y; o.z += old[4 * g + k].z; o.w += old[4 * g + k].w;
                    }
                    d4[k] = o;
                }
            }
        }
        tc05::fence_before_sync();
        __syncthreads();
    }
    if (warp == 0) tc05::tmem_dealloc(tbase, 64);
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------- launchers
static inline unsigned tc_grid(long E) {
    int dev = 0, n_sm = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    const long tiles = (E + kTcTile - 1) / kTcTile;
    return (unsigned)(tiles < n_sm ? tiles : n_sm);
}

allegro_status_t launch_latent_forward_tc(long E, double rc, const void* rvec, const void* x, const void* s, const void* A, void* z, void* x_new,
                                          cudaStream_t st) {
    ALLEGRO_CUDA(cudaFuncSetAttribute(tc_latent_fwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kFwdSmem));
    tc_latent_fwd_kernel<<<tc_grid(E), kTcThreads, kFwdSmem, st>>>(E, (float)rc, (const float*)rvec, (const float*)x, (const float*)s, (const float*)A,
                                                                   (float*)z, (float*)x_new);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

allegro_status_t launch_latent_backward_tc(long E, double rc, const void* rvec, const void* z, const void* g_xnew, const void* A, void* g_x, void* g_s,
                                           void* g_rvec, cudaStream_t st) {
    ALLEGRO_CUDA(cudaFuncSetAttribute(tc_latent_bwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kBwdSmem));
    tc_latent_bwd_kernel<<<tc_grid(E), kTcThreads, kBwdSmem, st>>>(E, (float)rc, (const float*)rvec, (const float*)z, (const float*)g_xnew,
                                                                   (const float*)A, (float*)g_x, (float*)g_s, (float*)g_rvec);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}


allegro_status_t launch_linear64_tc(long E, const void* x, const void* W, int transpose_w, int accumulate, void* y, cudaStream_t st) {
    ALLEGRO_CUDA(cudaFuncSetAttribute(tc_linear64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kLinSmem));
    const long tiles = (E + kTcTile - 1) / kTcTile;
    const unsigned g1 = tc_grid(E);
    const unsigned grid = (unsigned)(tiles < 2L * g1 ? tiles : 2L * g1);      // two CTAs per SM
    tc_linear64_kernel<<<grid, kTcThreads, kLinSmem, st>>>(E, (const float*)x, (const float*)W, transpose_w, accumulate, (float*)y);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

}  // namespace allegro
