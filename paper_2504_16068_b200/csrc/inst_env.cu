// inst_env.cu -- one translation unit per (ALLEGRO_T, ALLEGRO_L): environment embedding forward / VJP launchers.
#ifndef ALLEGRO_T
#error "compile with -DALLEGRO_T=float|double -DALLEGRO_L=1|2|3"
#endif
#include "env_kernels.cuh"

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
    env_embed_kernel<T, ALLEGRO_L, kEnvThreads><<<(unsigned)a.n_items, kEnvThreads, 0, a.st>>>(
        a.n, a.row_ptr, a.items, (const T*)a.rvec, (const T*)a.w, (T)a.scale, dst, have_items ? 1 : 0);
    ALLEGRO_LAUNCHED();
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

}  // namespace allegro
