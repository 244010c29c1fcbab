// noalloc.cu -- ONE entry point that allocates nothing, for callers that cannot call cudaMalloc (code under CUDA-graph capture,
// tight serving loops, harnesses that forbid it): allegro_tp_backward_static = allegro_tp_backward (scalar path weights) whose
// scratch -- the per-item gEenv partial rows and the per-item path-weight partial rows that tp_bwd_kernel writes and
// combine_items_kernel / gw_final_kernel reduce -- lives in a file-scope device array of a fixed, modest size instead of a
// caller-provided workspace.  Every GPU that loads the library holds the array (kStaticScratchBytes) until the process exits.
//
// In HOST code the array's name is a host-side stand-in, not a device address: the address is taken once per device, with that
// device current, through cudaGetSymbolAddress and handed to the existing launcher, which passes it to the kernels.
//
// Sharing: every call on a device uses the same array, which keeps the last call's contents.  Nothing in it has to start at
// zero -- each CTA overwrites its own partial rows completely before the reduction kernels read them (empty items write zero
// rows) -- but two calls that OVERLAP on the GPU (different streams, or graph branches) race on it: order them on one stream.
#include <mutex>

#include "common.cuh"
#include "launch.h"

namespace allegro {

constexpr size_t kStaticScratchBytes = 4u << 20;   // 4 MiB: e.g. 34,952 centres with the path-weight gradient at l_max = 2 in fp32
constexpr int kStaticMaxDevices = 64;

static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

// device address of the array on the CURRENT device, looked up once per device
static allegro_status_t static_scratch_ptr(void** out) {
    static std::mutex mu;
    static void* ptrs[kStaticMaxDevices] = {};
    int dev = -1;
    ALLEGRO_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) {
        set_error("allegro_tp_backward_static: device ordinal %d outside 0..%d", dev, kStaticMaxDevices - 1);
        return ALLEGRO_EUNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(mu);
    if (ptrs[dev] == nullptr) {
        void* p = nullptr;
        ALLEGRO_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));
        if (p == nullptr || (reinterpret_cast<uintptr_t>(p) & 255u) != 0) {
            set_error("allegro_tp_backward_static: cudaGetSymbolAddress returned a NULL or misaligned address");
            return ALLEGRO_ECUDA;
        }
        ptrs[dev] = p;
    }
    *out = ptrs[dev];
    return ALLEGRO_OK;
}

}  // namespace allegro

using namespace allegro;

extern "C" {

size_t allegro_tp_backward_static_capacity(void) { return kStaticScratchBytes; }

allegro_status_t allegro_tp_backward_static(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                            long n_items, const void* G, const void* V, const void* Eenv, const void* path_w, void* gV,
                                            void* gEenv, void* g_path_w, void* stream) {
    ALLEGRO_CHECK_ARG(plan != nullptr, "plan is NULL");
    ALLEGRO_CHECK_ARG(n_atoms >= 0 && n_edges >= 0, "negative size");
    if (plan->wmode != ALLEGRO_W_SCALAR) {   // the dense path allocates the plan's weight images on its first call
        set_error("allegro_tp_backward_static: scalar path weights only");
        return ALLEGRO_EUNSUPPORTED;
    }
    const size_t need = allegro_tp_backward_workspace(plan, n_atoms, n_edges, items ? n_items : 0, g_path_w != nullptr);
    if (need > kStaticScratchBytes) {
        set_error("allegro_tp_backward_static: this call needs %zu bytes of scratch, the static array holds %zu (n_atoms = %d, n_items = %ld, "
                  "g_path_w %s): use allegro_tp_backward with a caller-owned workspace",
                  need, (size_t)kStaticScratchBytes, n_atoms, items ? n_items : 0L, g_path_w ? "requested" : "not requested");
        return ALLEGRO_ENOMEM;
    }
    void* scratch = nullptr;
    allegro_status_t s = static_scratch_ptr(&scratch);
    if (s != ALLEGRO_OK) return s;
    return allegro_tp_backward(plan, n_atoms, n_edges, row_ptr, items, n_items, G, V, Eenv, path_w, gV, gEenv, g_path_w, scratch, kStaticScratchBytes,
                               stream);
}

}  // extern "C"
