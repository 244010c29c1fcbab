// mix_kernels.cuh -- dense per-path channel mixing (ALLEGRO_W_DENSE; BASELINE.json:configs[2]).
#pragma once
#include "common.cuh"
#include "launch.h"

namespace allegro {

template <typename T>
static allegro_status_t launch_mix_forward(const TpArgs& a) {
    (void)a;
    set_error("tp_forward: dense weight mode not built yet");
    return ALLEGRO_EUNSUPPORTED;
}
template <typename T>
static allegro_status_t launch_mix_backward(const TpArgs& a) {
    (void)a;
    set_error("tp_backward: dense weight mode not built yet");
    return ALLEGRO_EUNSUPPORTED;
}
template <typename T>
static size_t mix_backward_workspace(int n, long n_items, bool have_items, bool want_gw) {
    (void)n; (void)n_items; (void)have_items; (void)want_gw;
    return 0;
}

}  // namespace allegro
