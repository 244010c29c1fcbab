// inst_mix2.cu -- dense per-path mix, version 2 (fp32, l_max = 2, n = 64): one translation unit per part
// (-DALLEGRO_MIX2_PART=0 forward, 1 VJP with gV, 2 VJP without gV), built in parallel by build.py.
#ifndef ALLEGRO_MIX2_PART
#error "compile with -DALLEGRO_MIX2_PART=0|1|2"
#endif
#include "common.cuh"
#define ALLEGRO_CW(z) T(0) /* the folded-coefficient flavour is not used here */
#include "generated/tp_gen.cuh"
#include "mix2_kernels.cuh"

namespace allegro {

#if ALLEGRO_MIX2_PART == 0
allegro_status_t launch_mix2_forward_f32_l2_n64(const TpArgs& a) {
    auto k = mix_fwd2_kernel<2, 64>;
    const size_t smem = Mix2<2, 64>::kFwdSmem;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k<<<(unsigned)a.n_items, 256, smem, a.st>>>(a.row_ptr, a.items, (const float*)a.V, (const float*)a.Eenv, (const float*)a.path_w, (float*)a.out);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
#elif ALLEGRO_MIX2_PART == 1
allegro_status_t launch_mix2_backward_gv_f32_l2_n64(const TpArgs& a, float* gE_dst, int gE_by_item) {
    auto k = mix_bwd2_kernel<2, 64, true>;
    const size_t smem = Mix2<2, 64>::kBwdSmem;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k<<<(unsigned)a.n_items, 256, smem, a.st>>>(a.row_ptr, a.items, (const float*)a.G, (const float*)a.V, (const float*)a.Eenv,
                                                (const float*)a.path_w, (float*)a.gV, gE_dst, gE_by_item);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
#else
allegro_status_t launch_mix2_backward_nogv_f32_l2_n64(const TpArgs& a, float* gE_dst, int gE_by_item) {
    auto k = mix_bwd2_kernel<2, 64, false>;
    const size_t smem = Mix2<2, 64>::kBwdSmem;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k<<<(unsigned)a.n_items, 256, smem, a.st>>>(a.row_ptr, a.items, (const float*)a.G, (const float*)a.V, (const float*)a.Eenv,
                                                (const float*)a.path_w, (float*)a.gV, gE_dst, gE_by_item);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
#endif

}  // namespace allegro
