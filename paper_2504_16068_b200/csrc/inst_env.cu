// inst_env.cu -- one translation unit per (ALLEGRO_T, ALLEGRO_L): environment embedding forward / VJP launchers.
#ifndef ALLEGRO_T
#error "compile with -DALLEGRO_T=float|double -DALLEGRO_L=1|2|3"
#endif
#include <cstdlib>

#include "env_kernels.cuh"
#include "envlin_kernels.cuh"

namespace allegro {

constexpr int kEnvThreads = 256;

template <>
allegro_status_t launch_env_embed<ALLEGRO_T, ALLEGRO_L>(const EnvArgs& a) {
    using T = ALLEGRO_T;
    constexpr int DE = (ALLEGRO_L + 1) * (ALLEGRO_L + 1);
    if (a.n > kEnvThreads) {
        set_error("env_embed: n = %d unsupported (n <= %d)", a.n, kEnvThreads);
        return ALLEGRO_EUNSUPPORTED;
    }
    if (a.n_items == 0) return ALLEGRO_OK;
    const bool have_items = a.items != nullptr;
    if (have_items) {
        const size_t need = (size_t)a.n_items * a.n * DE * sizeof(T);
        if (a.ws == nullptr) {
            set_error("env_embed: workspace of %zu bytes required with items", need);
            return ALLEGRO_ENOMEM;
        }
    }
    T* dst = have_items ? (T*)a.ws : (T*)a.Eenv;
    if (a.W_r != nullptr) {
        if (a.n > 128 || a.nb > kMaxBasis) {
            set_error("env_radial_forward: n = %d, n_basis = %d unsupported (n <= 128, n_basis <= %d)", a.n, a.nb, kMaxBasis);
            return ALLEGRO_EUNSUPPORTED;
        }
        if (a.w_out == nullptr) {   // w not requested: factorised form
#define ALLEGRO_GEOFF(NB)                                                                                                  \
    {                                                                                                                      \
        auto k = env_radial_fwd_fact_kernel<T, ALLEGRO_L, NB>;                                                             \
        const size_t smem = sizeof(GeoSmem<T, ALLEGRO_L, NB>) + (size_t)NB * DE * sizeof(double);                          \
        ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));                      \
        k<<<(unsigned)a.n_items, kGeoChunk, smem, a.st>>>(a.n, a.nb, a.rc, (const T*)a.rc_edge, a.row_ptr, a.items, (const T*)a.rvec, (const T*)a.W_r, \
                                                          a.scale, dst, have_items ? 1 : 0);                               \
    }
            if (a.nb <= 8) ALLEGRO_GEOFF(8) else ALLEGRO_GEOFF(16)
#undef ALLEGRO_GEOFF
        } else {
#define ALLEGRO_GEOF(CPL, NB)                                                                                              \
    {                                                                                                                      \
        auto k = env_radial_fwd_kernel<T, ALLEGRO_L, CPL, NB>;                                                             \
        const size_t smem = sizeof(GeoSmem<T, ALLEGRO_L, NB>) + (size_t)32 * CPL * DE * sizeof(T);                         \
        ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));                      \
        k<<<(unsigned)a.n_items, 256, smem, a.st>>>(a.n, a.nb, a.rc, (const T*)a.rc_edge, a.row_ptr, a.items, (const T*)a.rvec, (const T*)a.W_r, \
                                                    (T)a.scale, (T*)a.w_out, dst, have_items ? 1 : 0);                     \
    }
        if (a.nb <= 8) {
            if (a.n <= 32) ALLEGRO_GEOF(1, 8) else if (a.n <= 64) ALLEGRO_GEOF(2, 8) else ALLEGRO_GEOF(4, 8)
        } else {
            if (a.n <= 32) ALLEGRO_GEOF(1, 16) else if (a.n <= 64) ALLEGRO_GEOF(2, 16) else ALLEGRO_GEOF(4, 16)
        }
#undef ALLEGRO_GEOF
        }
        ALLEGRO_LAUNCHED();
    } else {
    env_embed_kernel<T, ALLEGRO_L, kEnvThreads><<<(unsigned)a.n_items, kEnvThreads, 0, a.st>>>(
        a.n, a.row_ptr, a.items, (const T*)a.rvec, (const T*)a.w, (T)a.scale, dst, have_items ? 1 : 0);
    ALLEGRO_LAUNCHED();
    }
    if (have_items) {
        combine_items_kernel<T><<<(unsigned)a.n_items, 128, 0, a.st>>>(a.items, a.n_items, a.n * DE, (const T*)a.ws, (T*)a.Eenv);
        ALLEGRO_LAUNCHED();
    }
    return ALLEGRO_OK;
}

template <>
allegro_status_t launch_env_embed_backward<ALLEGRO_T, ALLEGRO_L>(const EnvBwdArgs& a) {
    using T = ALLEGRO_T;
    if (a.n > kEnvThreads) {
        set_error("env_embed_backward: n = %d unsupported (n <= %d)", a.n, kEnvThreads);
        return ALLEGRO_EUNSUPPORTED;
    }
    if (a.n_atoms == 0) return ALLEGRO_OK;
    if (a.W_r != nullptr) {
        if (a.n > 128 || a.nb > kMaxBasis) {
            set_error("env_radial_backward: n = %d, n_basis = %d unsupported (n <= 128, n_basis <= %d)", a.n, a.nb, kMaxBasis);
            return ALLEGRO_EUNSUPPORTED;
        }
        if (a.g_w == nullptr) {   // g_w not requested: factorised form
            constexpr int DEb = (ALLEGRO_L + 1) * (ALLEGRO_L + 1);
#define ALLEGRO_GEOBF(NB)                                                                                                  \
    env_radial_bwd_fact_kernel<T, ALLEGRO_L, NB><<<(unsigned)a.n_atoms, kGeoChunk, (size_t)a.n * (DEb + a.nb) * sizeof(T), a.st>>>( \
        a.n, a.nb, a.rc, (const T*)a.rc_edge, a.row_ptr, (const T*)a.gEenv, (const T*)a.rvec, (const T*)a.W_r, a.scale, (T*)a.g_rvec);
            if (a.nb <= 8) { ALLEGRO_GEOBF(8) } else { ALLEGRO_GEOBF(16) }
#undef ALLEGRO_GEOBF
            ALLEGRO_LAUNCHED();
            return ALLEGRO_OK;
        }
#define ALLEGRO_GEOB(CPL, NB)                                                                                              \
    {                                                                                                                      \
        auto k = env_radial_bwd_kernel<T, ALLEGRO_L, CPL, NB>;                                                             \
        const size_t smem = sizeof(GeoSmem<T, ALLEGRO_L, NB>);                                                             \
        ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));                      \
        k<<<(unsigned)a.n_atoms, 256, smem, a.st>>>(a.n, a.nb, a.rc, (const T*)a.rc_edge, a.row_ptr, (const T*)a.gEenv, (const T*)a.rvec,       \
                                                    (const T*)a.W_r, (T)a.scale, (T*)a.g_rvec, (T*)a.g_w);                 \
    }
        if (a.nb <= 8) {
            if (a.n <= 32) ALLEGRO_GEOB(1, 8) else if (a.n <= 64) ALLEGRO_GEOB(2, 8) else ALLEGRO_GEOB(4, 8)
        } else {
            if (a.n <= 32) ALLEGRO_GEOB(1, 16) else if (a.n <= 64) ALLEGRO_GEOB(2, 16) else ALLEGRO_GEOB(4, 16)
        }
#undef ALLEGRO_GEOB
        ALLEGRO_LAUNCHED();
        return ALLEGRO_OK;
    }
#define ALLEGRO_ENVB(CPL)                                                                          \
    env_embed_bwd_kernel<T, ALLEGRO_L, CPL><<<(unsigned)a.n_atoms, 256, 0, a.st>>>(                \
        a.n, a.row_ptr, (const T*)a.gEenv, (const T*)a.rvec, (const T*)a.w, (T)a.scale, (T*)a.g_rvec, (T*)a.g_w)
    if (a.n <= 32) ALLEGRO_ENVB(1);
    else if (a.n <= 64) ALLEGRO_ENVB(2);
    else if (a.n <= 128) ALLEGRO_ENVB(4);
    else ALLEGRO_ENVB(8);
#undef ALLEGRO_ENVB
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

template <>
allegro_status_t launch_edge_embed<ALLEGRO_T, ALLEGRO_L>(const EmbedArgs& a) {
    using T = ALLEGRO_T;
    if (a.nb > kMaxBasis || ((size_t)(ALLEGRO_L + 1) * (ALLEGRO_L + 1) * 2 * sizeof(T)) % 8 != 0) {
        set_error("edge_embed: n_basis = %d unsupported (<= %d)", a.nb, kMaxBasis);
        return ALLEGRO_EUNSUPPORTED;
    }
    if (a.n_edges == 0) return ALLEGRO_OK;
    const unsigned grid = (unsigned)((a.n_edges + kGeoChunk - 1) / kGeoChunk);
#define ALLEGRO_EMB(NB)                                                                                                     \
    {                                                                                                                       \
        auto k = edge_embed_kernel<T, ALLEGRO_L, NB>;                                                                       \
        const size_t smem = (sizeof(GeoSmem<T, ALLEGRO_L, NB>) + 15) / 16 * 16 + 8 * 32 * 2 * (ALLEGRO_L + 1) * (ALLEGRO_L + 1) * sizeof(T) + (size_t)2 * a.nb * a.n * sizeof(double); \
        ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));                       \
        k<<<grid, 256, smem, a.st>>>(a.n, a.nb, a.rc, a.n_edges, (const T*)a.rvec, (const T*)a.W_x0, (const T*)a.W_v0, (T*)a.x0, (T*)a.V0, \
                                     (T*)a.v0_out); \
    }
    if (a.nb <= 8) ALLEGRO_EMB(8) else ALLEGRO_EMB(16)
#undef ALLEGRO_EMB
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

template <>
allegro_status_t launch_edge_embed_backward<ALLEGRO_T, ALLEGRO_L>(const EmbedArgs& a) {
    using T = ALLEGRO_T;
    if (a.nb > kMaxBasis) {
        set_error("edge_embed_backward: n_basis = %d unsupported (<= %d)", a.nb, kMaxBasis);
        return ALLEGRO_EUNSUPPORTED;
    }
    if (a.n_edges == 0) return ALLEGRO_OK;
    const unsigned grid = (unsigned)((a.n_edges + kGeoChunk - 1) / kGeoChunk);
    if (a.gV0 == nullptr && a.g_v0 != nullptr) {      // factor form of the cotangent: thread per edge, no reductions
#define ALLEGRO_EMBF(NB)                                                                                                    \
    {                                                                                                                       \
        auto k = edge_embed_factors_bwd_kernel<T, ALLEGRO_L, NB>;                                                           \
        const size_t smem = (size_t)2 * a.n * NB * sizeof(double) + (size_t)2 * kGeoChunk * 33 * sizeof(T);                  \
        ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));                       \
        k<<<grid, kGeoChunk, smem, a.st>>>(a.n, a.nb, a.rc, a.n_edges, (const T*)a.rvec, (const T*)a.W_x0, (const T*)a.W_v0,  \
                                           (const T*)a.g_x0, (const T*)a.g_v0, (const T*)a.gYe, (T*)a.g_rvec);              \
    }
        if (a.nb <= 8) ALLEGRO_EMBF(8) else ALLEGRO_EMBF(16)
#undef ALLEGRO_EMBF
        ALLEGRO_LAUNCHED();
        return ALLEGRO_OK;
    }
#define ALLEGRO_EMBB(NB)                                                                                                    \
    {                                                                                                                       \
        auto k = edge_embed_bwd_kernel<T, ALLEGRO_L, NB>;                                                                   \
        const size_t smem = (sizeof(GeoSmem<T, ALLEGRO_L, NB>) + 15) / 16 * 16 + 8 * 32 * 2 * (ALLEGRO_L + 1) * (ALLEGRO_L + 1) * sizeof(T) + (size_t)2 * a.nb * a.n * sizeof(double); \
        ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));                       \
        k<<<grid, 256, smem, a.st>>>(a.n, a.nb, a.rc, a.n_edges, (const T*)a.rvec, (const T*)a.W_x0, (const T*)a.W_v0,     \
                                     (const T*)a.g_x0, (const T*)a.gV0, (T*)a.g_rvec, (const T*)a.g_v0, (const T*)a.gYe);   \
    }
    if (a.nb <= 8) ALLEGRO_EMBB(8) else ALLEGRO_EMBB(16)
#undef ALLEGRO_EMBB
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

template <>
allegro_status_t launch_env_linear<ALLEGRO_T, ALLEGRO_L>(const EnvLinArgs& a) {
    using T = ALLEGRO_T;
    constexpr int DE = (ALLEGRO_L + 1) * (ALLEGRO_L + 1);
    if (a.n_in < 1 || a.n_in > kEnvLinThreads || a.n_out > 256) {
        set_error("env_linear_forward: n_in = %d, n = %d unsupported (n_in <= %d, n <= 256)", a.n_in, a.n_out, kEnvLinThreads);
        return ALLEGRO_EUNSUPPORTED;
    }
    if (a.n_atoms == 0) return ALLEGRO_OK;
    const size_t smem = ((size_t)kEnvLinChunk * DE + 2 * (size_t)kEnvLinThreads * DE + (size_t)a.n_in * (a.n_out + 1)) * sizeof(T);
    auto k = env_linear_fwd_kernel<T, ALLEGRO_L>;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    // persistent: W^T is staged once per CTA; one wave of as many CTAs as are resident at this shared-memory size
    int per_sm = 1, n_sm = 148, dev = 0;
    ALLEGRO_CUDA(cudaGetDevice(&dev));
    ALLEGRO_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    ALLEGRO_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, kEnvLinThreads, smem));
    if (per_sm < 1) per_sm = 1;
    const unsigned grid = (unsigned)(a.n_atoms < n_sm * per_sm ? a.n_atoms : n_sm * per_sm);
    k<<<grid, kEnvLinThreads, smem, a.st>>>(a.n_atoms, a.n_out, a.n_in, a.row_ptr, (const T*)a.rvec, (const T*)a.x, (const T*)a.W, (T)a.scale,
                                                           (T*)a.Eenv);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

template <>
allegro_status_t launch_env_linear_backward<ALLEGRO_T, ALLEGRO_L>(const EnvLinArgs& a) {
    using T = ALLEGRO_T;
    constexpr int DE = (ALLEGRO_L + 1) * (ALLEGRO_L + 1);
    if (a.n_in < 1 || a.n_in > kEnvLinThreads || a.n_out > 256) {
        set_error("env_linear_backward: n_in = %d, n = %d unsupported (n_in <= %d, n <= 256)", a.n_in, a.n_out, kEnvLinThreads);
        return ALLEGRO_EUNSUPPORTED;
    }
    if (a.n_atoms == 0) return ALLEGRO_OK;
    size_t smem = ((size_t)kEnvLinChunk * (2 * DE + 4) + (size_t)a.n_out * DE + (size_t)a.n_in * DE + (size_t)kEnvLinThreads * DE) * sizeof(T);
    // the chunk's x rows are staged in shared memory when that still leaves two CTAs per SM
    const size_t xs_bytes = (size_t)kEnvLinChunk * (a.n_in + 1) * sizeof(T);
    const int stage_x = smem + xs_bytes <= 100 * 1024 ? 1 : 0;
    if (stage_x) smem += xs_bytes;
    auto k = env_linear_bwd_kernel<T, ALLEGRO_L>;
    ALLEGRO_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k<<<(unsigned)a.n_atoms, kEnvLinThreads, smem, a.st>>>(a.n_out, a.n_in, a.row_ptr, (const T*)a.gEenv, (const T*)a.rvec, (const T*)a.x, (const T*)a.W,
                                                           (T)a.scale, (T*)a.g_rvec, a.acc_g_rvec, (T*)a.g_x, a.acc_g_x, stage_x);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

}  // namespace allegro
