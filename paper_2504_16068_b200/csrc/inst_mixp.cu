// inst_mixp.cu -- the dense per-path mix at l_max = 3 (mixp_kernels.cuh), one translation unit per dtype and kernel:
// -DALLEGRO_T=float|double -DALLEGRO_MIXP_PART=0 (forward) | 1 (VJP with gV) | 2 (VJP without gV) | 3 (gradient of W_p).
// The 68 unrolled paths make each of these a slow file to compile; separate units let build.py run them side by side.
#if !defined(ALLEGRO_T) || !defined(ALLEGRO_MIXP_PART)
#error "compile with -DALLEGRO_T=float|double -DALLEGRO_MIXP_PART=0|1|2|3"
#endif
#define ALLEGRO_L 3
#include "common.cuh"
#include "generated/tp_gen.cuh"
#include "mixp_kernels.cuh"

namespace allegro {

using T = ALLEGRO_T;
constexpr int CT = sizeof(T) == 4 ? 256 : 128;

// one n x (n + VEC) weight image must fit next to the staged tile
static inline allegro_status_t mixp_check_smem(size_t smem, int n) {
    if (smem <= 226 * 1024) return ALLEGRO_OK;
    set_error("dense path weights at l_max = 3: n = %d needs %zu bytes of shared memory (n <= 192 in fp32, n <= 128 in fp64)", n, smem);
    return ALLEGRO_EUNSUPPORTED;
}

#if ALLEGRO_MIXP_PART == 0
template <>
allegro_status_t launch_mixp_forward<T>(const TpArgs& a) {
    const size_t smem = mixp_smem<T, 3>(a.n, CT);
    if (mixp_check_smem(smem, a.n) != ALLEGRO_OK) return ALLEGRO_EUNSUPPORTED;
    auto k = mixp_fwd_kernel<T, 3, CT>;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k<<<(unsigned)a.n_items, CT, smem, a.st>>>(a.n, a.row_ptr, a.items, (const T*)a.V, (const T*)a.Eenv, (const T*)a.path_w, (T*)a.out);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
#elif ALLEGRO_MIXP_PART == 1 || ALLEGRO_MIXP_PART == 2
template <>
allegro_status_t launch_mixp_backward<T, ALLEGRO_MIXP_PART == 1>(const TpArgs& a, T* gE_dst, int gE_by_item) {
    const size_t smem = mixp_smem<T, 3>(a.n, CT);
    if (mixp_check_smem(smem, a.n) != ALLEGRO_OK) return ALLEGRO_EUNSUPPORTED;
    auto k = mixp_bwd_kernel<T, 3, CT, ALLEGRO_MIXP_PART == 1>;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k<<<(unsigned)a.n_items, CT, smem, a.st>>>(a.n, a.row_ptr, a.items, (const T*)a.G, (const T*)a.V, (const T*)a.Eenv, (const T*)a.path_w,
                                               (T*)a.gV, gE_dst, gE_by_item);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
#else
template <>
allegro_status_t launch_mixp_gw<T>(const TpArgs& a, T* part) {
    using Gen = TPGen<3>;
    const int nsl = CT / a.n;
    const size_t smem_gw = 2 * (size_t)nsl * 7 * a.n * sizeof(T);
    auto kg = mix_gw_kernel<T, 3, CT>;
    ALLEGRO_CUDA(cudaFuncSetAttribute(kg, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_gw));
    kg<<<(unsigned)(Gen::P * kGwSplits), CT, smem_gw, a.st>>>(a.n, a.n_atoms, a.row_ptr, (const T*)a.G, (const T*)a.V, (const T*)a.Eenv, part);
    ALLEGRO_LAUNCHED();
    const long count = (long)Gen::P * a.n * a.n;
    gw_dense_final_kernel<T><<<(unsigned)((count + 255) / 256), 256, 0, a.st>>>(count, part, (T*)a.g_path_w);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}
#endif

}  // namespace allegro
