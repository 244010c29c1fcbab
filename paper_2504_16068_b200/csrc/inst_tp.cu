// inst_tp.cu -- one translation unit per (ALLEGRO_T, ALLEGRO_L): instantiates the tensor-product kernels for
// that dtype and l_max and defines their launchers.  Compiled six times by build.py
// (-DALLEGRO_T=float|double -DALLEGRO_L=1|2|3).
#ifndef ALLEGRO_T
#error "compile with -DALLEGRO_T=float|double -DALLEGRO_L=1|2|3"
#endif
#include "common.cuh"
#include "generated/tp_gen.cuh"
#include "tp_kernels.cuh"
#include "mix_kernels.cuh"

namespace allegro {

using Gen = TPGen<ALLEGRO_L>;

template <typename T> struct Cfg {
    static constexpr int THREADS = sizeof(T) == 4 ? 256 : 128;  // compute threads; one producer warp is added at launch
    // VJP at l_max = 3, fp32: 168 registers per thread allow one CTA per SM only, so that CTA gets 12 compute warps instead of 8
    static constexpr int THREADS_BWD = (sizeof(T) == 4 && ALLEGRO_L == 3) ? 384 : THREADS;
};

// Ring depth: as many stages as fit (<= 4) with two CTAs per SM; if that leaves fewer than 3, one CTA per SM
// with up to 6 stages.  `extra` = barriers + reduction scratch.
static inline int pick_stages(size_t stage_bytes, size_t extra) {
    const size_t cap2 = 113 * 1024, cap1 = 226 * 1024;
    int nst = 1;
    for (int k : {4, 3}) if (k * stage_bytes + extra <= cap2) { nst = k; break; }
    if (nst == 1) {
        for (int k : {6, 4, 3, 2}) if (k * stage_bytes + extra <= cap1) { nst = k; break; }
    }
    return nst;
}

// Swizzled 2-D TMA variant: feature rows of exactly 128 bytes (l_max = 3 in fp32), box = one edge = n rows (n % 8 == 0, n <= 256)
template <typename T>
static bool use_swizzle(int n) { return sizeof(T) * Gen::DV == 128 && n % 8 == 0 && n <= 256; }

// the plan's folded coefficient table as a kernel parameter (bound by allegro_plan_bind_weights or by the call itself)
template <typename T>
static allegro_status_t folded_table(const TpArgs& a, CwTab<T, Gen::NNZ>& tab) {
    if (a.path_w != nullptr) {
        allegro_status_t s = bind_scalar_weights(a.plan, a.path_w, a.st);
        if (s != ALLEGRO_OK) return s;
    } else if (!a.plan->cw_bound) {
        set_error("tensor product (scalar weights): path_w is NULL and no weights are bound to the plan (allegro_plan_bind_weights)");
        return ALLEGRO_EINVAL;
    }
    for (int z = 0; z < Gen::NNZ; ++z) tab.v[z] = (T)a.plan->cw[z];
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
    CwTab<T, Gen::NNZ> cwt;
    allegro_status_t s = folded_table<T>(a, cwt);
    if (s != ALLEGRO_OK) return s;
    const int nslots = TH / a.n;
    const size_t tile = align128((size_t)nslots * a.n * Gen::DV * sizeof(T));
    const bool w_out = a.out != nullptr, w_g = a.Gout != nullptr, w_e = a.e_edge != nullptr;
    const size_t stage = ((w_out && w_g) ? 2 : 1) * tile;
    const bool sw = use_swizzle<T>(a.n);
    const size_t extra = 2 * 6 * 8 + 2 * TH * sizeof(T) + 64 + (sw ? 1024 : 0);
    const int nst = pick_stages(stage, extra);
    const size_t smem = nst * stage + extra;
    TpMaps tm{};
    if (sw) {
        const unsigned long long rows = (unsigned long long)a.n_edges * a.n;
        if ((s = make_row128_map(&tm.a, a.V, rows, a.n)) != ALLEGRO_OK) return s;
        if (w_out && (s = make_row128_map(&tm.b, a.out, rows, a.n)) != ALLEGRO_OK) return s;
        if (w_g && (s = make_row128_map(&tm.c, a.Gout, rows, a.n)) != ALLEGRO_OK) return s;
    }
#define ALLEGRO_FWD_SW(WO, WG, WE, SW)                                                                             \
    {                                                                                                              \
        auto k = tp_fwd_kernel<T, ALLEGRO_L, TH, WO, WG, WE, SW>;                                                  \
        if ((s = set_smem(k, smem)) != ALLEGRO_OK) return s;                                                       \
        k<<<(unsigned)a.n_items, TH + 32, smem, a.st>>>(cwt, tm, nst, a.n, a.row_ptr, a.items, (const T*)a.V, (const T*)a.Eenv, (T*)a.out, \
                                                        (const T*)a.q, (T)a.kappa, (T*)a.e_edge, (T*)a.Gout);      \
    }
#define ALLEGRO_FWD(WO, WG, WE)                                                                                    \
    {                                                                                                              \
        if constexpr (sizeof(T) * Gen::DV == 128) {                                                                \
            if (sw) ALLEGRO_FWD_SW(WO, WG, WE, true) else ALLEGRO_FWD_SW(WO, WG, WE, false)                        \
        } else ALLEGRO_FWD_SW(WO, WG, WE, false)                                                                   \
    }
    if (w_out && !w_g && !w_e) { ALLEGRO_FWD(true, false, false) }
    else if (w_out && w_g && w_e) { ALLEGRO_FWD(true, true, true) }
    else if (w_out && w_e) { ALLEGRO_FWD(true, false, true) }
    else if (w_g && w_e && !w_out) { ALLEGRO_FWD(false, true, true) }
    else {
        set_error("tp_forward_energy: unsupported output combination (G needs e_edge)");
        return ALLEGRO_EUNSUPPORTED;
    }
#undef ALLEGRO_FWD
#undef ALLEGRO_FWD_SW
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
    constexpr int TH = Cfg<T>::THREADS_BWD;
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
    CwTab<T, Gen::NNZ> cwt;
    allegro_status_t s = folded_table<T>(a, cwt);
    if (s != ALLEGRO_OK) return s;
    unsigned char* ws = (unsigned char*)a.ws;
    T* gE_part = nullptr;
    if (have_items) { gE_part = (T*)ws; ws += align_up((size_t)a.n_items * a.n * Gen::DE * sizeof(T), 256); }
    T* gw_part = want_gw ? (T*)ws : nullptr;
    T* gE_dst = have_items ? gE_part : (T*)a.gEenv;

    const int nslots = TH / a.n;
    const size_t stage = 2 * (size_t)align128((size_t)nslots * a.n * Gen::DV * sizeof(T));
    const bool sw = use_swizzle<T>(a.n);
    const size_t extra = 2 * 6 * 8 + 64 + (sw ? 1024 : 0);
    const int nst = pick_stages(stage, extra);
    const size_t smem = nst * stage + extra;
    const bool cot = a.q != nullptr;  // tile 0 is `out`; the A12 cotangent is formed in registers
    const bool want_gv = a.gV != nullptr;
    TpMaps tm{};
    if (sw) {
        const unsigned long long rows = (unsigned long long)a.n_edges * a.n;
        if ((s = make_row128_map(&tm.a, a.V, rows, a.n)) != ALLEGRO_OK) return s;
        if ((s = make_row128_map(&tm.c, a.G, rows, a.n)) != ALLEGRO_OK) return s;
        if (want_gv && (s = make_row128_map(&tm.b, a.gV, rows, a.n)) != ALLEGRO_OK) return s;
    }
#define ALLEGRO_BWD_SW(GV, GW, COT, SW)                                                                                   \
    {                                                                                                                     \
        auto k = tp_bwd_kernel<T, ALLEGRO_L, TH, GV, GW, COT, SW>;                                                        \
        if ((s = set_smem(k, smem)) != ALLEGRO_OK) return s;                                                              \
        k<<<(unsigned)a.n_items, TH + 32, smem, a.st>>>(cwt, tm, nst, a.n, a.row_ptr, a.items, (const T*)a.G, (const T*)a.V, (const T*)a.Eenv, \
                                                        (const T*)a.q, (T)a.kappa, (T*)a.gV, gE_dst, have_items ? 1 : 0, gw_part); \
    }
#define ALLEGRO_BWD(GV, GW, COT)                                                                                          \
    {                                                                                                                     \
        if constexpr (sizeof(T) * Gen::DV == 128) {                                                                       \
            if (sw) ALLEGRO_BWD_SW(GV, GW, COT, true) else ALLEGRO_BWD_SW(GV, GW, COT, false)                             \
        } else ALLEGRO_BWD_SW(GV, GW, COT, false)                                                                         \
    }
    if (cot) {
        if (want_gv && want_gw) { ALLEGRO_BWD(true, true, true) }
        else if (want_gv) { ALLEGRO_BWD(true, false, true) }
        else if (want_gw) { ALLEGRO_BWD(false, true, true) }
        else { ALLEGRO_BWD(false, false, true) }
    } else {
        if (want_gv && want_gw) { ALLEGRO_BWD(true, true, false) }
        else if (want_gv) { ALLEGRO_BWD(true, false, false) }
        else if (want_gw) { ALLEGRO_BWD(false, true, false) }
        else { ALLEGRO_BWD(false, false, false) }
    }
#undef ALLEGRO_BWD
#undef ALLEGRO_BWD_SW
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

// forward + energy + VJP in one pass (scalar weights); workspace as for tp_backward
template <>
allegro_status_t launch_tp_fused<ALLEGRO_T, ALLEGRO_L>(const TpArgs& a) {
    using T = ALLEGRO_T;
    constexpr int TH = Cfg<T>::THREADS;
    if (a.n > TH || ((size_t)a.n * Gen::DV * sizeof(T)) % 16 != 0) {
        set_error("tp_fused: n = %d unsupported (need n <= %d and n*dV*sizeof(T) %% 16 == 0)", a.n, TH);
        return ALLEGRO_EUNSUPPORTED;
    }
    const bool have_items = a.items != nullptr;
    const bool want_gw = a.g_path_w != nullptr;
    const size_t need = tp_backward_workspace<T, ALLEGRO_L>(a.n, a.n_atoms, a.n_items, have_items, a.plan->wmode, want_gw);
    if (need > a.ws_bytes || (need > 0 && a.ws == nullptr)) {
        set_error("tp_fused: workspace too small (%zu < %zu bytes)", a.ws_bytes, need);
        return ALLEGRO_ENOMEM;
    }
    if (a.n_items == 0) {
        if (want_gw) ALLEGRO_CUDA(cudaMemsetAsync(a.g_path_w, 0, sizeof(T) * Gen::P, a.st));
        return ALLEGRO_OK;
    }
    CwTab<T, Gen::NNZ> cwt;
    allegro_status_t s = folded_table<T>(a, cwt);
    if (s != ALLEGRO_OK) return s;
    unsigned char* ws = (unsigned char*)a.ws;
    T* gE_part = nullptr;
    if (have_items) { gE_part = (T*)ws; ws += align_up((size_t)a.n_items * a.n * Gen::DE * sizeof(T), 256); }
    T* gw_part = want_gw ? (T*)ws : nullptr;
    T* gE_dst = have_items ? gE_part : (T*)a.gEenv;

    const int nslots = TH / a.n;
    const size_t stage = (size_t)align128((size_t)nslots * a.n * Gen::DV * sizeof(T));
    const bool sw = use_swizzle<T>(a.n);
    const size_t extra = 2 * 6 * 8 + 2 * TH * sizeof(T) + 64 + (sw ? 1024 : 0);
    size_t red = (size_t)TH * Gen::DE * sizeof(T);          // the gEenv / g_path_w reductions reuse the ring
    if (want_gw && (size_t)(TH / 32) * Gen::P * sizeof(T) > red) red = (size_t)(TH / 32) * Gen::P * sizeof(T);
    int nst = pick_stages(stage, extra);
    while (nst * stage < red) ++nst;
    const size_t smem = nst * stage + extra;
    const bool want_gv = a.gV != nullptr;
    TpMaps tm{};
    if (sw) {
        const unsigned long long rows = (unsigned long long)a.n_edges * a.n;
        if ((s = make_row128_map(&tm.a, a.V, rows, a.n)) != ALLEGRO_OK) return s;
        if (want_gv && (s = make_row128_map(&tm.b, a.gV, rows, a.n)) != ALLEGRO_OK) return s;
    }
#define ALLEGRO_FUSED_SW(GV, GW, SW)                                                                                       \
    {                                                                                                                     \
        auto k = tp_fused_kernel<T, ALLEGRO_L, TH, GV, GW, SW>;                                                           \
        if ((s = set_smem(k, smem)) != ALLEGRO_OK) return s;                                                              \
        k<<<(unsigned)a.n_items, TH + 32, smem, a.st>>>(cwt, cwt, tm, nst, a.n, a.row_ptr, a.items, (const T*)a.V, (const T*)a.Eenv, (const T*)a.q, \
                                                        (T)a.kappa, (T*)a.e_edge, (T*)a.gV, gE_dst, have_items ? 1 : 0, gw_part); \
    }
#define ALLEGRO_FUSED(GV, GW)                                                                                             \
    {                                                                                                                     \
        if constexpr (sizeof(T) * Gen::DV == 128) {                                                                       \
            if (sw) ALLEGRO_FUSED_SW(GV, GW, true) else ALLEGRO_FUSED_SW(GV, GW, false)                                   \
        } else ALLEGRO_FUSED_SW(GV, GW, false)                                                                            \
    }
    if (want_gv && want_gw) { ALLEGRO_FUSED(true, true) }
    else if (want_gv) { ALLEGRO_FUSED(true, false) }
    else if (want_gw) { ALLEGRO_FUSED(false, true) }
    else { ALLEGRO_FUSED(false, false) }
#undef ALLEGRO_FUSED
#undef ALLEGRO_FUSED_SW
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
