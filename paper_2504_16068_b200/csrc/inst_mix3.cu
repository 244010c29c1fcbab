// inst_mix3.cu -- dense per-path mix on tcgen05 (fp32, l_max = 2, n = 64): one translation unit per part
// (-DALLEGRO_MIX3_PART=0 forward, 1 VJP), built in parallel by build.py.
#ifndef ALLEGRO_MIX3_PART
#error "compile with -DALLEGRO_MIX3_PART=0|1"
#endif
#include "common.cuh"
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

// which compiled path subset serves the plan's block masks: 0 = all paths, 1 = the paths into the 0e scalars,
// 2 = the paths from the natural-parity input blocks (0e, 1o, 2e), -1 = none
static int mix3_variant(const allegro_plan* plan) {
    const unsigned o = plan->out_blocks & 0x3fu, i = plan->in_blocks & 0x3fu;
    return (i == 0x3fu && o == 0x3fu) ? 0 : (i == 0x3fu && o == 0x1u) ? 1 : (i == 0x19u && o == 0x3fu) ? 2 : -1;
}
static allegro_status_t mix3_unsupported(const allegro_plan* plan) {
    set_error("dense tensor product: block masks in 0x%x / out 0x%x are not built (all / all, all / 0x1, 0x19 / all)", plan->in_blocks & 0x3fu,
              plan->out_blocks & 0x3fu);
    return ALLEGRO_EUNSUPPORTED;
}

#if ALLEGRO_MIX3_PART == 0
static allegro_status_t mix3_fwd_launch_outer(const TpArgs& a, const float* img_f) {
    constexpr uint32_t PMASK = Mix3::mask_natural_in();
    auto k = mix3_fwd_kernel<PMASK, true>;
    constexpr int SMEM = Mix3Seq<PMASK>::SMEM;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM));
    k<<<(unsigned)a.n_items, Mix3::CT + 64, SMEM, a.st>>>(a.row_ptr, a.items, nullptr, (const float*)a.Eenv, img_f, (float*)a.out, (const float*)a.q,
                                                          (float)a.kappa, (float*)a.e_edge, (float*)a.scalars_out, (const float*)a.rvec,
                                                          (const float*)a.v0);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
template <uint32_t PMASK>
static allegro_status_t mix3_fwd_launch(const TpArgs& a, const float* img_f) {
    auto k = mix3_fwd_kernel<PMASK>;
    constexpr int SMEM = Mix3Seq<PMASK>::SMEM;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM));
    k<<<(unsigned)a.n_items, Mix3::CT + 64, SMEM, a.st>>>(a.row_ptr, a.items, (const float*)a.V, (const float*)a.Eenv, img_f, (float*)a.out,
                                                          (const float*)a.q, (float)a.kappa, (float*)a.e_edge, (float*)a.scalars_out, nullptr, nullptr);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
allegro_status_t launch_mix3_forward_f32_l2_n64(const TpArgs& a) {
    const int var = mix3_variant(a.plan);
    if (var < 0) return mix3_unsupported(a.plan);
    float *img_f, *img_b;
    allegro_status_t s = mix3_images(a, &img_f, &img_b);
    if (s != ALLEGRO_OK) return s;
    if (a.v0 != nullptr) {
        if (var != 2) { set_error("tp_forward_outer: the plan must be restricted to the natural-parity input blocks (set_in_blocks(0x19))"); return ALLEGRO_EINVAL; }
        return mix3_fwd_launch_outer(a, img_f);
    }
    return var == 0 ? mix3_fwd_launch<Mix3::ALL>(a, img_f)
           : var == 1 ? mix3_fwd_launch<Mix3::mask_into(0)>(a, img_f)
                      : mix3_fwd_launch<Mix3::mask_natural_in()>(a, img_f);
}
#else
template <bool GV, uint32_t PMASK, bool COT>
static allegro_status_t mix3_bwd_launch(const TpArgs& a, const float* img_b, float* gE_dst, int gE_by_item) {
    auto k = mix3_bwd_kernel<GV, PMASK, COT>;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, Mix3B::SMEM));
    k<<<(unsigned)a.n_items, Mix3B::CT + 64, Mix3B::SMEM, a.st>>>(a.row_ptr, a.items, (const float*)a.G, (const float*)a.V, (const float*)a.Eenv, img_b,
                                                                (float*)a.gV, gE_dst, gE_by_item, (const float*)a.q, (float)a.kappa, (const float*)a.g_scalars, nullptr, nullptr,
                                                                nullptr, nullptr);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
static allegro_status_t mix3_bwd_launch_outer(const TpArgs& a, const float* img_b, float* gE_dst, int gE_by_item) {
    auto k = mix3_bwd_kernel<true, Mix3::mask_natural_in(), false, true>;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, Mix3B::SMEM));
    k<<<(unsigned)a.n_items, Mix3B::CT + 64, Mix3B::SMEM, a.st>>>(a.row_ptr, a.items, (const float*)a.G, nullptr, (const float*)a.Eenv, img_b, nullptr,
                                                                gE_dst, gE_by_item, nullptr, 0.f, (const float*)a.g_scalars, (const float*)a.rvec,
                                                                (const float*)a.v0, (float*)a.g_v0, (float*)a.gYe);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
template <uint32_t PMASK>
static allegro_status_t mix3_bwd_pick(const TpArgs& a, const float* img_b, float* gE_dst, int gE_by_item) {
    if (a.q != nullptr)   // allegro_tp_backward_energy: a.G is the forward result
        return a.gV ? mix3_bwd_launch<true, PMASK, true>(a, img_b, gE_dst, gE_by_item) : mix3_bwd_launch<false, PMASK, true>(a, img_b, gE_dst, gE_by_item);
    return a.gV ? mix3_bwd_launch<true, PMASK, false>(a, img_b, gE_dst, gE_by_item) : mix3_bwd_launch<false, PMASK, false>(a, img_b, gE_dst, gE_by_item);
}
allegro_status_t launch_mix3_backward_f32_l2_n64(const TpArgs& a, float* gE_dst, int gE_by_item) {
    const int var = mix3_variant(a.plan);
    if (var < 0) return mix3_unsupported(a.plan);
    float *img_f, *img_b;
    allegro_status_t s = mix3_images(a, &img_f, &img_b);
    if (s != ALLEGRO_OK) return s;
    if (a.v0 != nullptr) {
        if (var != 2) { set_error("tp_backward_outer: the plan must be restricted to the natural-parity input blocks (set_in_blocks(0x19))"); return ALLEGRO_EINVAL; }
        return mix3_bwd_launch_outer(a, img_b, gE_dst, gE_by_item);
    }
    return var == 0 ? mix3_bwd_pick<Mix3::ALL>(a, img_b, gE_dst, gE_by_item)
           : var == 1 ? mix3_bwd_pick<Mix3::mask_into(0)>(a, img_b, gE_dst, gE_by_item)
                      : mix3_bwd_pick<Mix3::mask_natural_in()>(a, img_b, gE_dst, gE_by_item);
}
#endif

}  // namespace allegro
