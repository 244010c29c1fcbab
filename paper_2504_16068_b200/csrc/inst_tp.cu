// inst_tp.cu -- one translation unit per (ALLEGRO_T, ALLEGRO_L): instantiates the tensor-product kernels for
// that dtype and l_max and defines their launchers.  Compiled six times by build.py
// (-DALLEGRO_T=float|double -DALLEGRO_L=1|2|3).
#ifndef ALLEGRO_T
#error "compile with -DALLEGRO_T=float|double -DALLEGRO_L=1|2|3"
#endif
#include "common.cuh"

namespace allegro {
constexpr int kCwMax = 1222;  // nnz of the l_max = 3 plan
// Folded coefficient table Wc[z] = path_w[path(z)] * C_z of the call in flight.  Constant memory, so every
// coefficient is a constant-bank operand of its FFMA/DFMA (no register, no load instruction).
__constant__ ALLEGRO_T c_cw[kCwMax];
__device__ ALLEGRO_T g_cw_stage[kCwMax];  // fold_kernel writes here; copied device-to-device into c_cw on the stream
}  // namespace allegro
#define ALLEGRO_CW(z) ::allegro::c_cw[z]
#include "generated/tp_gen.cuh"
#include "tp_kernels.cuh"
#include "mix_kernels.cuh"

namespace allegro {

using Gen = TPGen<ALLEGRO_L>;

template <typename T> struct Cfg {
    static constexpr int THREADS = sizeof(T) == 4 ? 256 : 128;
};

static inline int pick_stages(size_t stage_bytes, size_t extra) {
    // as many stages (<= 3) as fit next to `extra` in the 227 KB a CTA may use; the wrapper decides the
    // occupancy through the total (several CTAs per SM when the stage is small)
    const size_t cap2 = 110 * 1024;  // two CTAs per SM
    const size_t cap1 = 220 * 1024;  // one CTA per SM
    if (3 * stage_bytes + extra <= cap2) return 3;
    if (2 * stage_bytes + extra <= cap2) return 2;
    if (3 * stage_bytes + extra <= cap1) return 3;
    if (2 * stage_bytes + extra <= cap1) return 2;
    return 1;
}

template <typename T>
static allegro_status_t fold_weights(const TpArgs& a) {
    T* stage = nullptr;
    ALLEGRO_CUDA(cudaGetSymbolAddress((void**)&stage, g_cw_stage));
    fold_kernel<T, ALLEGRO_L><<<(Gen::NNZ + 127) / 128, 128, 0, a.st>>>((const T*)a.path_w, stage);
    ALLEGRO_LAUNCHED();
    ALLEGRO_CUDA(cudaMemcpyToSymbolAsync(c_cw, stage, sizeof(T) * Gen::NNZ, 0, cudaMemcpyDeviceToDevice, a.st));
    return ALLEGRO_OK;
}

template <typename K>
static allegro_status_t set_smem(K kernel, size_t bytes) {
    ALLEGRO_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return ALLEGRO_OK;
}

template <>
allegro_status_t launch_tp_forward<ALLEGRO_T, ALLEGRO_L>(const TpArgs& a) {
    using T = ALLEGRO_T;
    constexpr int TH = Cfg<T>::THREADS;
    if (a.n > TH || ((size_t)a.n * Gen::DV * sizeof(T)) % 16 != 0) {
        set_error("tp_forward: n = %d unsupported (need n <= %d and n*dV*sizeof(T) %% 16 == 0)", a.n, TH);
        return ALLEGRO_EUNSUPPORTED;
    }
    if (a.n_items == 0) return ALLEGRO_OK;
    if (a.plan->wmode == ALLEGRO_W_DENSE) return launch_mix_forward<T>(a);
    allegro_status_t s = fold_weights<T>(a);
    if (s != ALLEGRO_OK) return s;
    const int nslots = TH / a.n;
    const size_t stage = align128((size_t)nslots * a.n * Gen::DV * sizeof(T));
    const bool w_out = a.out != nullptr, w_g = a.Gout != nullptr, w_e = a.e_edge != nullptr;
    const size_t extra = ((w_out && w_g) ? 3 * stage : 0) + 64 + 2 * TH * sizeof(T);
    const int nst = pick_stages(stage, extra + 128);
    const size_t smem = nst * stage + extra;
#define ALLEGRO_FWD(NST, WO, WG, WE)                                                                               \
    {                                                                                                              \
        auto k = tp_fwd_kernel<T, ALLEGRO_L, TH, NST, WO, WG, WE>;                                                 \
        if ((s = set_smem(k, smem)) != ALLEGRO_OK) return s;                                                       \
        k<<<(unsigned)a.n_items, TH, smem, a.st>>>(a.n, a.row_ptr, a.items, (const T*)a.V, (const T*)a.Eenv, (T*)a.out, \
                                                   (const T*)a.q, (T)a.kappa, (T*)a.e_edge, (T*)a.Gout);           \
    }
#define ALLEGRO_FWD_N(WO, WG, WE) \
    if (nst == 3) ALLEGRO_FWD(3, WO, WG, WE) else if (nst == 2) ALLEGRO_FWD(2, WO, WG, WE) else ALLEGRO_FWD(1, WO, WG, WE)
    if (w_out && !w_g && !w_e) { ALLEGRO_FWD_N(true, false, false) }
    else if (w_out && w_g && w_e) { ALLEGRO_FWD_N(true, true, true) }
    else if (w_out && w_g) { ALLEGRO_FWD_N(true, true, false) }
    else if (w_out && w_e) { ALLEGRO_FWD_N(true, false, true) }
    else if (w_g && w_e) { ALLEGRO_FWD_N(false, true, true) }
    else if (w_g) { ALLEGRO_FWD_N(false, true, false) }
    else {
        set_error("tp_forward: nothing to store (out and G are both NULL)");
        return ALLEGRO_EINVAL;
    }
#undef ALLEGRO_FWD_N
#undef ALLEGRO_FWD
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

// workspace layout of tp_backward (scalar mode): [gE partial rows, one per item (only with items)] [gw partial rows, one per item]
template <>
size_t tp_backward_workspace<ALLEGRO_T, ALLEGRO_L>(int n, int n_atoms, long n_items, bool have_items, int wmode, bool want_gw) {
    using T = ALLEGRO_T;
    (void)n_atoms;
    if (wmode == ALLEGRO_W_DENSE) return mix_backward_workspace<T>(n, n_items, have_items, want_gw);
    size_t b = 0;
    if (have_items) b += align_up((size_t)n_items * n * Gen::DE * sizeof(T), 256);
    if (want_gw) b += align_up((size_t)n_items * Gen::P * sizeof(T), 256);
    return b;
}

template <>
allegro_status_t launch_tp_backward<ALLEGRO_T, ALLEGRO_L>(const TpArgs& a) {
    using T = ALLEGRO_T;
    constexpr int TH = Cfg<T>::THREADS;
    if (a.n > TH || ((size_t)a.n * Gen::DV * sizeof(T)) % 16 != 0) {
        set_error("tp_backward: n = %d unsupported (need n <= %d and n*dV*sizeof(T) %% 16 == 0)", a.n, TH);
        return ALLEGRO_EUNSUPPORTED;
    }
    const bool have_items = a.items != nullptr;
    const bool want_gw = a.g_path_w != nullptr;
    const size_t need = tp_backward_workspace<T, ALLEGRO_L>(a.n, a.n_atoms, a.n_items, have_items, a.plan->wmode, want_gw);
    if (need > a.ws_bytes || (need > 0 && a.ws == nullptr)) {
        set_error("tp_backward: workspace too small (%zu < %zu bytes)", a.ws_bytes, need);
        return ALLEGRO_ENOMEM;
    }
    if (a.n_items == 0) {
        if (want_gw) ALLEGRO_CUDA(cudaMemsetAsync(a.g_path_w, 0, sizeof(T) * Gen::P, a.st));
        return ALLEGRO_OK;
    }
    if (a.plan->wmode == ALLEGRO_W_DENSE) return launch_mix_backward<T>(a);
    allegro_status_t s = fold_weights<T>(a);
    if (s != ALLEGRO_OK) return s;
    unsigned char* ws = (unsigned char*)a.ws;
    T* gE_part = nullptr;
    if (have_items) { gE_part = (T*)ws; ws += align_up((size_t)a.n_items * a.n * Gen::DE * sizeof(T), 256); }
    T* gw_part = want_gw ? (T*)ws : nullptr;
    T* gE_dst = have_items ? gE_part : (T*)a.gEenv;

    const int nslots = TH / a.n;
    const size_t stage = 2 * (size_t)align128((size_t)nslots * a.n * Gen::DV * sizeof(T));
    const size_t red = 128 + (size_t)TH * Gen::DE * sizeof(T);
    const int nst = pick_stages(stage, red + 256);
    const size_t smem = nst * stage + red;
#define ALLEGRO_BWD(NST, GV, GW)                                                                                          \
    {                                                                                                                     \
        auto k = tp_bwd_kernel<T, ALLEGRO_L, TH, NST, GV, GW>;                                                                       \
        if ((s = set_smem(k, smem)) != ALLEGRO_OK) return s;                                                              \
        k<<<(unsigned)a.n_items, TH, smem, a.st>>>(a.n, a.row_ptr, a.items, (const T*)a.G, (const T*)a.V, (const T*)a.Eenv, \
                                                   (T*)a.gV, gE_dst, have_items ? 1 : 0, gw_part);                        \
    }
#define ALLEGRO_BWD_N(GV, GW) \
    if (nst == 3) ALLEGRO_BWD(3, GV, GW) else if (nst == 2) ALLEGRO_BWD(2, GV, GW) else ALLEGRO_BWD(1, GV, GW)
    const bool want_gv = a.gV != nullptr;
    if (want_gv && want_gw) { ALLEGRO_BWD_N(true, true) }
    else if (want_gv) { ALLEGRO_BWD_N(true, false) }
    else if (want_gw) { ALLEGRO_BWD_N(false, true) }
    else { ALLEGRO_BWD_N(false, false) }
#undef ALLEGRO_BWD_N
#undef ALLEGRO_BWD
    ALLEGRO_LAUNCHED();
    if (have_items) {
        combine_items_kernel<T><<<(unsigned)a.n_items, 128, 0, a.st>>>(a.items, a.n_items, a.n * Gen::DE, gE_part, (T*)a.gEenv);
        ALLEGRO_LAUNCHED();
    }
    if (want_gw) {
        gw_final_kernel<T><<<Gen::P, 256, 0, a.st>>>(gw_part, a.n_items, Gen::P, (T*)a.g_path_w);
        ALLEGRO_LAUNCHED();
    }
    return ALLEGRO_OK;
}

}  // namespace allegro
