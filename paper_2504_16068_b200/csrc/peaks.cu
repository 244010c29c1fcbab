// peaks.cu -- roofline denominators measured on the device the library runs on ("measure with an FFMA
// micro-benchmark in the same run"; "tensor peak for the C2 mix: measure TF32 the same way").  Diagnostics for bench.py, not part
// of the hot path: both calls synchronise the stream and time their own kernel with CUDA events.
#include "common.cuh"
#include "tc05.cuh"

namespace allegro {

// 8 independent FMA chains per thread, 1024 threads per CTA, 2 CTAs per SM worth of blocks
__global__ void __launch_bounds__(1024) ffma_peak_kernel(int iters, float a, float b, float* __restrict__ sink) {
    float x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = (float)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int i = 0; i < 8; ++i) x[i] = fmaf(x[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    if (s == 123.456f) sink[0] = s;   // never true: keeps the chains alive
}

// one CTA per SM; one thread issues `iters` x 8 tcgen05.mma kind::tf32, M = 128, N = NCOLS, K = 8 each, operands in shared memory
template <int NCOLS>
__global__ void __launch_bounds__(128, 1) tf32_mma_peak_kernel(int iters) {
    extern __shared__ unsigned char peak_smem_raw[];
    unsigned char* sm = peak_smem_raw + ((1024u - (smem_u32(peak_smem_raw) & 1023u)) & 1023u);
    __shared__ uint64_t bar;
    __shared__ uint32_t slot;
    const int tid = threadIdx.x, warp = tid >> 5;
    for (int i = tid; i < 96 * 1024 / 4; i += 128) reinterpret_cast<float*>(sm)[i] = 0.f;
    if (tid == 0) { mbar_init(&bar, 1); fence_mbar_init(); }
    if (warp == 0) { tc05::tmem_alloc(&slot, 256); tc05::tmem_relinquish(); }
    fence_proxy_async();
    tc05::fence_before_sync();
    __syncthreads();
    tc05::fence_after_sync();
    const uint32_t tb = slot;
    if (tid == 0) {
        constexpr uint32_t idesc = tc05::make_idesc(tc05::FMT_TF32, tc05::FMT_TF32, 128, NCOLS);
        const uint32_t a0 = tc05::sdesc_lo(smem_u32(sm)), b0 = tc05::sdesc_lo(smem_u32(sm + 32768));   // A: 128 rows, B: 256 rows, two K-atoms each
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const uint32_t aoff = (uint32_t)(((j >> 2) * 16384 + (j & 3) * 32) >> 4), boff = (uint32_t)(((j >> 2) * 32768 + (j & 3) * 32) >> 4);
                tc05::mma_tf32_lo(tb, a0 + aoff, b0 + boff, tc05::kSdescHiSw128, idesc, 1u);
            }
        }
        tc05::mma_commit(&bar);
        mbar_wait(&bar, 0);
    }
    tc05::fence_before_sync();
    __syncthreads();
    if (warp == 0) tc05::tmem_dealloc(tb, 256);
}

}  // namespace allegro

using namespace allegro;

extern "C" {

allegro_status_t allegro_measure_fp32_fma_peak(void* stream, double* tflops) {
    ALLEGRO_CHECK_ARG(tflops != nullptr, "tflops is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    ALLEGRO_CUDA(cudaGetDevice(&dev));
    ALLEGRO_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float* sink = nullptr;
    ALLEGRO_CUDA(cudaMalloc(&sink, 4));
    cudaEvent_t e0, e1;
    ALLEGRO_CUDA(cudaEventCreate(&e0));
    ALLEGRO_CUDA(cudaEventCreate(&e1));
    const int iters = 4096, blocks = 2 * sms;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {   // rep 0 warms up
        ALLEGRO_CUDA(cudaEventRecord(e0, st));
        ffma_peak_kernel<<<blocks, 1024, 0, st>>>(iters, 1.000001f, 1e-7f, sink);
        ALLEGRO_LAUNCHED();
        ALLEGRO_CUDA(cudaEventRecord(e1, st));
        ALLEGRO_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        ALLEGRO_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        const double tf = 2.0 * 64.0 * iters * 1024.0 * blocks / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    *tflops = best;
    return ALLEGRO_OK;
}

}  // extern "C"

template <int NCOLS>
static allegro_status_t measure_tf32(cudaStream_t st, double* tflops) {
    int dev = 0, sms = 0;
    ALLEGRO_CUDA(cudaGetDevice(&dev));
    ALLEGRO_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int smem = 100 * 1024, iters = 2000;
    ALLEGRO_CUDA(cudaFuncSetAttribute(tf32_mma_peak_kernel<NCOLS>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    cudaEvent_t e0, e1;
    ALLEGRO_CUDA(cudaEventCreate(&e0));
    ALLEGRO_CUDA(cudaEventCreate(&e1));
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        ALLEGRO_CUDA(cudaEventRecord(e0, st));
        tf32_mma_peak_kernel<NCOLS><<<sms, 128, smem, st>>>(iters);
        ALLEGRO_LAUNCHED();
        ALLEGRO_CUDA(cudaEventRecord(e1, st));
        ALLEGRO_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        ALLEGRO_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        const double tf = 2.0 * 128.0 * NCOLS * 8.0 * 8.0 * iters * sms / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *tflops = best;
    return ALLEGRO_OK;
}

extern "C" {

allegro_status_t allegro_measure_tf32_mma_peak(void* stream, double* tflops) {
    ALLEGRO_CHECK_ARG(tflops != nullptr, "tflops is NULL");
    return measure_tf32<256>((cudaStream_t)stream, tflops);
}

allegro_status_t allegro_measure_tf32_mma_rate(int n_cols, void* stream, double* tflops) {
    ALLEGRO_CHECK_ARG(tflops != nullptr, "tflops is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    switch (n_cols) {
        case 16: return measure_tf32<16>(st, tflops);
        case 32: return measure_tf32<32>(st, tflops);
        case 48: return measure_tf32<48>(st, tflops);
        case 80: return measure_tf32<80>(st, tflops);
        case 128: return measure_tf32<128>(st, tflops);
        case 256: return measure_tf32<256>(st, tflops);
    }
    set_error("allegro_measure_tf32_mma_rate: N = %d is not one of 16, 32, 48, 80, 128, 256", n_cols);
    return ALLEGRO_EINVAL;
}

}  // extern "C"
