// inst_mix3.cu -- dense per-path mix on tcgen05 (fp32, l_max = 2, n = 64): one translation unit per part
// (-DALLEGRO_MIX3_PART=0 forward, 1 VJP), built in parallel by build.py.
#ifndef ALLEGRO_MIX3_PART
#error "compile with -DALLEGRO_MIX3_PART=0|1"
#endif
#include "common.cuh"
#define ALLEGRO_CW(z) T(0) /* the folded-coefficient flavour is not used here */
#include "generated/tp_gen.cuh"
#include "mix3_kernels.cuh"

namespace allegro {

// Plan-owned device buffer for the two weight images (forward, VJP); allocated on the first dense call of the plan
// (cudaMalloc: call once before capturing a CUDA graph), rewritten from path_w by every call, freed by allegro_plan_destroy.
static allegro_status_t mix3_images(const TpArgs& a, float** img_f, float** img_b) {
    const allegro_plan* plan = a.plan;
    const size_t bytes = 2 * (size_t)Mix3::P * Mix3::IMG_BYTES;
    if (plan->dense_img == nullptr) {
        void* p = nullptr;
        ALLEGRO_CUDA(cudaMalloc(&p, bytes));
        plan->dense_img = p;
    }
    *img_f = (float*)plan->dense_img;
    *img_b = *img_f + (size_t)Mix3::P * (Mix3::IMG_BYTES / 4);
    mix3_prep_kernel<<<Mix3::P, 256, 0, a.st>>>((const float*)a.path_w, *img_f, *img_b);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

#if ALLEGRO_MIX3_PART == 0
allegro_status_t launch_mix3_forward_f32_l2_n64(const TpArgs& a) {
    float *img_f, *img_b;
    allegro_status_t s = mix3_images(a, &img_f, &img_b);
    if (s != ALLEGRO_OK) return s;
    auto k = mix3_fwd_kernel<0>;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, Mix3::SMEM));
    k<<<(unsigned)a.n_items, Mix3::CT + 64, Mix3::SMEM, a.st>>>(a.row_ptr, a.items, (const float*)a.V, (const float*)a.Eenv, img_f, (float*)a.out);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
#else
allegro_status_t launch_mix3_backward_f32_l2_n64(const TpArgs& a, float* gE_dst, int gE_by_item) {
    float *img_f, *img_b;
    allegro_status_t s = mix3_images(a, &img_f, &img_b);
    if (s != ALLEGRO_OK) return s;
    if (a.gV) {
        auto k = mix3_bwd_kernel<true>;
        ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, Mix3B::SMEM));
        k<<<(unsigned)a.n_items, Mix3B::CT + 64, Mix3B::SMEM, a.st>>>(a.row_ptr, a.items, (const float*)a.G, (const float*)a.V, (const float*)a.Eenv,
                                                                    img_b, (float*)a.gV, gE_dst, gE_by_item);
    } else {
        auto k = mix3_bwd_kernel<false>;
        ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, Mix3B::SMEM));
        k<<<(unsigned)a.n_items, Mix3B::CT + 64, Mix3B::SMEM, a.st>>>(a.row_ptr, a.items, (const float*)a.G, (const float*)a.V, (const float*)a.Eenv,
                                                                    img_b, nullptr, gE_dst, gE_by_item);
    }
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
#endif

}  // namespace allegro
