// api.cu -- the C ABI of include/allegro_b200.h: argument checks and dispatch to the per-(dtype, l_max)
// launchers.  No arithmetic of the method lives here.
#include <cstdarg>
#include <cstring>
#include <new>

#include "common.cuh"
#include "launch.h"

namespace allegro {

std::atomic<long> g_launches{0};
static thread_local char t_err[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof t_err, fmt, ap);
    va_end(ap);
}

// explicit specialisations live in inst_tp.cu / inst_env.cu (one object per dtype and l_max)
#define ALLEGRO_DECL(T, L)                                                                     \
    template <> allegro_status_t launch_env_embed<T, L>(const EnvArgs&);                       \
    template <> allegro_status_t launch_edge_embed<T, L>(const EmbedArgs&);                    \
    template <> allegro_status_t launch_edge_embed_backward<T, L>(const EmbedArgs&);           \
    template <> allegro_status_t launch_env_embed_backward<T, L>(const EnvBwdArgs&);           \
    template <> allegro_status_t launch_env_linear<T, L>(const EnvLinArgs&);                   \
    template <> allegro_status_t launch_env_linear_backward<T, L>(const EnvLinArgs&);          \
    template <> allegro_status_t launch_tp_forward<T, L>(const TpArgs&);                       \
    template <> allegro_status_t launch_tp_backward<T, L>(const TpArgs&);                      \
    template <> allegro_status_t launch_tp_fused<T, L>(const TpArgs&);                         \
    template <> size_t tp_backward_workspace<T, L>(int, int, long, bool, int, bool);
ALLEGRO_DECL(float, 1) ALLEGRO_DECL(float, 2) ALLEGRO_DECL(float, 3)
ALLEGRO_DECL(double, 1) ALLEGRO_DECL(double, 2) ALLEGRO_DECL(double, 3)
#undef ALLEGRO_DECL

// call F<T, L>(args...) for the plan's dtype and l_max
#define ALLEGRO_DISPATCH(plan, F, ...)                                   \
    ((plan)->dtype == ALLEGRO_F32                                        \
         ? ((plan)->l_max == 1 ? F<float, 1>(__VA_ARGS__)                \
            : (plan)->l_max == 2 ? F<float, 2>(__VA_ARGS__)              \
                                 : F<float, 3>(__VA_ARGS__))             \
         : ((plan)->l_max == 1 ? F<double, 1>(__VA_ARGS__)               \
            : (plan)->l_max == 2 ? F<double, 2>(__VA_ARGS__)             \
                                 : F<double, 3>(__VA_ARGS__)))

// cw[z] = path_w[path(z)] * C_z (0 for paths into a masked-out output block), product in double, rounded once to the plan's dtype
static void fold_host(const allegro_plan* plan, const void* path_w_host) {
    const size_t nnz = plan->tab.nnz.size();
    plan->cw.resize(nnz);
    for (size_t z = 0; z < nnz; ++z) {
        const NonZero& q = plan->tab.nnz[z];
        double w = plan->dtype == ALLEGRO_F32 ? (double)((const float*)path_w_host)[q.path] : ((const double*)path_w_host)[q.path];
        if (!plan->path_active(q.path)) w = 0.0;
        const double c = w * q.c;
        plan->cw[z] = plan->dtype == ALLEGRO_F32 ? (double)(float)c : c;
    }
    plan->cw_bound = true;
}

allegro_status_t bind_scalar_weights(const allegro_plan* plan, const void* path_w_dev, cudaStream_t st) {
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    ALLEGRO_CUDA(cudaStreamIsCapturing(st, &cs));
    if (cs != cudaStreamCaptureStatusNone) {
        set_error("scalar path weights cannot be read back while the stream is capturing: call allegro_plan_bind_weights first and pass path_w = NULL");
        return ALLEGRO_EINVAL;
    }
    double host[128];   // P <= 68 values of at most 8 bytes
    const size_t bytes = plan->tab.paths.size() * (plan->dtype == ALLEGRO_F32 ? 4 : 8);
    ALLEGRO_CUDA(cudaMemcpyAsync(host, path_w_dev, bytes, cudaMemcpyDeviceToHost, st));
    ALLEGRO_CUDA(cudaStreamSynchronize(st));
    fold_host(plan, host);
    return ALLEGRO_OK;
}

allegro_status_t make_row128_map(CUtensorMap* map, const void* base, unsigned long long rows, unsigned box_rows) {
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    if (encode == nullptr) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        ALLEGRO_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
        if (fn == nullptr || qres != cudaDriverEntryPointSuccess) {
            set_error("cuTensorMapEncodeTiled is not available from this driver");
            return ALLEGRO_ECUDA;
        }
        encode = (encode_fn)fn;
    }
    const cuuint64_t dims[2] = {32, rows};
    const cuuint64_t strides[1] = {128};           // bytes between rows
    const cuuint32_t box[2] = {32, box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                              CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_error("cuTensorMapEncodeTiled failed (%d) for %llu rows, box of %u rows", (int)r, rows, box_rows);
        return ALLEGRO_ECUDA;
    }
    return ALLEGRO_OK;
}

}  // namespace allegro

using namespace allegro;

extern "C" {

allegro_status_t allegro_plan_create(int l_max, allegro_parity_t parity, int n_channels, allegro_dtype_t dtype, allegro_wmode_t wmode,
                                     allegro_plan_t** out) {
    ALLEGRO_CHECK_ARG(out != nullptr, "out is NULL");
    *out = nullptr;
    ALLEGRO_CHECK_ARG(dtype == ALLEGRO_F32 || dtype == ALLEGRO_F64, "bad dtype");
    ALLEGRO_CHECK_ARG(wmode == ALLEGRO_W_SCALAR || wmode == ALLEGRO_W_DENSE, "bad weight mode");
    ALLEGRO_CHECK_ARG(n_channels >= 1, "n_channels < 1");
    if (l_max < 1 || l_max > 3 || parity != ALLEGRO_PARITY_FULL || n_channels > 256) {
        set_error("allegro_plan_create: unsupported (l_max = %d, parity = %d, n = %d); l_max 1..3, full parity, n <= 256", l_max, (int)parity,
                  n_channels);
        return ALLEGRO_EUNSUPPORTED;
    }
    allegro_plan* p = new (std::nothrow) allegro_plan();
    if (!p) { set_error("allegro_plan_create: out of host memory"); return ALLEGRO_ENOMEM; }
    p->l_max = l_max; p->n = n_channels; p->dtype = (int)dtype; p->wmode = (int)wmode;
    build_tables(l_max, p->tab);
    *out = p;
    return ALLEGRO_OK;
}
void allegro_plan_destroy(allegro_plan_t* plan) {
    if (plan && plan->dense_img) cudaFree(plan->dense_img);
    delete plan;
}
allegro_status_t allegro_plan_set_out_blocks(allegro_plan_t* plan, unsigned block_mask) {
    ALLEGRO_CHECK_ARG(plan != nullptr, "plan is NULL");
    const unsigned full = (1u << (2 * (plan->l_max + 1))) - 1u;
    ALLEGRO_CHECK_ARG((block_mask & full) != 0, "empty block mask");
    plan->out_blocks = block_mask & full;
    plan->cw_bound = false;   // a bound table was folded for the previous mask
    return ALLEGRO_OK;
}
allegro_status_t allegro_plan_set_in_blocks(allegro_plan_t* plan, unsigned block_mask) {
    ALLEGRO_CHECK_ARG(plan != nullptr, "plan is NULL");
    const unsigned full = (1u << (2 * (plan->l_max + 1))) - 1u;
    ALLEGRO_CHECK_ARG((block_mask & full) != 0, "empty block mask");
    plan->in_blocks = block_mask & full;
    plan->cw_bound = false;
    return ALLEGRO_OK;
}
allegro_status_t allegro_plan_bind_weights(allegro_plan_t* plan, const void* path_w, void* stream) {
    ALLEGRO_CHECK_ARG(plan != nullptr && path_w != nullptr, "plan / path_w is NULL");
    ALLEGRO_CHECK_ARG(plan->wmode == ALLEGRO_W_SCALAR, "scalar path weights only (dense weights are read by every call)");
    return bind_scalar_weights(plan, path_w, (cudaStream_t)stream);
}
int allegro_plan_num_paths(const allegro_plan_t* plan) { return plan ? (int)plan->tab.paths.size() : -1; }
int allegro_plan_dim_v(const allegro_plan_t* plan) { return plan ? plan->tab.dV : -1; }
int allegro_plan_dim_e(const allegro_plan_t* plan) { return plan ? plan->tab.dE : -1; }
long allegro_plan_nnz(const allegro_plan_t* plan) { return plan ? (long)plan->tab.nnz.size() : -1; }

allegro_status_t allegro_plan_paths(const allegro_plan_t* plan, int32_t* l1, int32_t* p1, int32_t* l2, int32_t* l3, int32_t* p3, int32_t* off1,
                                    int32_t* off2, int32_t* off3) {
    ALLEGRO_CHECK_ARG(plan && l1 && p1 && l2 && l3 && p3 && off1 && off2 && off3, "NULL argument");
    for (size_t p = 0; p < plan->tab.paths.size(); ++p) {
        const PathInfo& q = plan->tab.paths[p];
        l1[p] = q.l1; p1[p] = q.p1; l2[p] = q.l2; l3[p] = q.l3; p3[p] = q.p3; off1[p] = q.off1; off2[p] = q.off2; off3[p] = q.off3;
    }
    return ALLEGRO_OK;
}
allegro_status_t allegro_plan_cg(const allegro_plan_t* plan, int32_t* path, int32_t* i, int32_t* j, int32_t* k, double* coef) {
    ALLEGRO_CHECK_ARG(plan && path && i && j && k && coef, "NULL argument");
    for (size_t z = 0; z < plan->tab.nnz.size(); ++z) {
        const NonZero& q = plan->tab.nnz[z];
        path[z] = q.path; i[z] = q.i; j[z] = q.j; k[z] = q.k; coef[z] = q.c;
    }
    return ALLEGRO_OK;
}
allegro_status_t allegro_cg_real_block(int l1, int l2, int l3, double* C) {
    ALLEGRO_CHECK_ARG(C != nullptr, "C is NULL");
    ALLEGRO_CHECK_ARG(l1 >= 0 && l2 >= 0 && l3 >= 0 && l1 <= 8 && l2 <= 8 && l3 <= 8, "l out of range 0..8");
    std::vector<double> c;
    cg_real_block(l1, l2, l3, c);
    std::memcpy(C, c.data(), c.size() * sizeof(double));
    return ALLEGRO_OK;
}
allegro_status_t allegro_segments_build(const int32_t* row_ptr_host, int n_atoms, int tile_edges, int32_t* items, long cap, long* n_items) {
    ALLEGRO_CHECK_ARG(row_ptr_host && n_items, "NULL argument");
    ALLEGRO_CHECK_ARG(n_atoms >= 0 && tile_edges >= 1 && cap >= 0, "negative size");
    for (int i = 0; i < n_atoms; ++i) ALLEGRO_CHECK_ARG(row_ptr_host[i + 1] >= row_ptr_host[i], "row_ptr not monotone");
    *n_items = build_segments(row_ptr_host, n_atoms, tile_edges, items, cap);
    return ALLEGRO_OK;
}

#define ALLEGRO_CHECK_GRAPH()                                                                     \
    ALLEGRO_CHECK_ARG(plan != nullptr, "plan is NULL");                                           \
    ALLEGRO_CHECK_ARG(n_atoms >= 0 && n_edges >= 0 && n_edges < 2147483647L, "bad n_atoms / n_edges"); \
    ALLEGRO_CHECK_ARG(row_ptr != nullptr || n_atoms == 0, "row_ptr is NULL")

allegro_status_t allegro_env_embed(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                   long n_items, const void* rvec, const void* w, double scale, void* Eenv, void* workspace,
                                   size_t workspace_bytes, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((rvec && w) || n_edges == 0, "rvec / w is NULL");
    ALLEGRO_CHECK_ARG(Eenv || n_atoms == 0, "Eenv is NULL");
    ALLEGRO_CHECK_ARG(aligned16(Eenv) && aligned16(w), "Eenv / w not 16-byte aligned");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    const size_t need = allegro_env_workspace(plan, n_atoms, items ? n_items : 0);
    if (items && (workspace == nullptr || workspace_bytes < need)) {
        set_error("allegro_env_embed: workspace too small (%zu < %zu bytes)", workspace_bytes, need);
        return ALLEGRO_ENOMEM;
    }
    EnvArgs a{plan->n, n_atoms, n_edges, row_ptr, items, items ? n_items : (long)n_atoms, rvec, w, scale, Eenv, workspace, (cudaStream_t)stream};
    return ALLEGRO_DISPATCH(plan, launch_env_embed, a);
}

allegro_status_t allegro_env_radial_forward(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                            long n_items, const void* rvec, const void* W_r, int n_basis, double r_cut, double scale, void* w,
                                            void* Eenv, void* workspace, size_t workspace_bytes, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG(rvec || n_edges == 0, "rvec is NULL");
    ALLEGRO_CHECK_ARG(W_r != nullptr && n_basis >= 1 && r_cut > 0, "W_r is NULL or bad n_basis / r_cut");
    ALLEGRO_CHECK_ARG(Eenv || n_atoms == 0, "Eenv is NULL");
    ALLEGRO_CHECK_ARG(aligned16(Eenv) && aligned16(w), "Eenv / w not 16-byte aligned");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    const size_t need = allegro_env_workspace(plan, n_atoms, items ? n_items : 0);
    if (items && (workspace == nullptr || workspace_bytes < need)) {
        set_error("allegro_env_radial_forward: workspace too small (%zu < %zu bytes)", workspace_bytes, need);
        return ALLEGRO_ENOMEM;
    }
    EnvArgs a{plan->n, n_atoms, n_edges, row_ptr, items, items ? n_items : (long)n_atoms, rvec, nullptr, scale, Eenv, workspace,
              (cudaStream_t)stream, W_r, n_basis, r_cut, w};
    return ALLEGRO_DISPATCH(plan, launch_env_embed, a);
}

allegro_status_t allegro_env_radial_backward(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const void* gEenv,
                                             const void* rvec, const void* W_r, int n_basis, double r_cut, double scale, void* g_rvec,
                                             void* g_w, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((rvec && g_rvec) || n_edges == 0, "rvec / g_rvec is NULL");
    ALLEGRO_CHECK_ARG(W_r != nullptr && n_basis >= 1 && r_cut > 0, "W_r is NULL or bad n_basis / r_cut");
    ALLEGRO_CHECK_ARG(gEenv || n_atoms == 0, "gEenv is NULL");
    EnvBwdArgs a{plan->n, n_atoms, n_edges, row_ptr, gEenv, rvec, nullptr, scale, g_rvec, g_w, (cudaStream_t)stream, W_r, n_basis, r_cut};
    return ALLEGRO_DISPATCH(plan, launch_env_embed_backward, a);
}

allegro_status_t allegro_env_linear_forward(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const void* rvec,
                                            const void* x, const void* W, int n_in, double scale, void* Eenv, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((rvec && x) || n_edges == 0, "rvec / x is NULL");
    ALLEGRO_CHECK_ARG(W != nullptr && n_in >= 1, "W is NULL or bad n_in");
    ALLEGRO_CHECK_ARG(Eenv || n_atoms == 0, "Eenv is NULL");
    EnvLinArgs a{};
    a.n_out = plan->n; a.n_in = n_in; a.n_atoms = n_atoms; a.n_edges = n_edges; a.row_ptr = row_ptr; a.rvec = rvec; a.x = x; a.W = W;
    a.scale = scale; a.Eenv = Eenv; a.st = (cudaStream_t)stream;
    return ALLEGRO_DISPATCH(plan, launch_env_linear, a);
}

allegro_status_t allegro_env_linear_backward(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const void* gEenv,
                                             const void* rvec, const void* x, const void* W, int n_in, double scale, void* g_rvec,
                                             int accumulate_g_rvec, void* g_x, int accumulate_g_x, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((rvec && x && g_rvec && g_x) || n_edges == 0, "rvec / x / g_rvec / g_x is NULL");
    ALLEGRO_CHECK_ARG(W != nullptr && n_in >= 1, "W is NULL or bad n_in");
    ALLEGRO_CHECK_ARG(gEenv || n_atoms == 0, "gEenv is NULL");
    EnvLinArgs a{};
    a.n_out = plan->n; a.n_in = n_in; a.n_atoms = n_atoms; a.n_edges = n_edges; a.row_ptr = row_ptr; a.rvec = rvec; a.x = x; a.W = W;
    a.scale = scale; a.gEenv = gEenv; a.g_rvec = g_rvec; a.acc_g_rvec = accumulate_g_rvec; a.g_x = g_x; a.acc_g_x = accumulate_g_x;
    a.st = (cudaStream_t)stream;
    return ALLEGRO_DISPATCH(plan, launch_env_linear_backward, a);
}

allegro_status_t allegro_env_radial_forward_typed(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                                  long n_items, const void* rvec, const void* W_r, int n_basis, const void* rc_edge, double scale,
                                                  void* w, void* Eenv, void* workspace, size_t workspace_bytes, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((rvec && rc_edge) || n_edges == 0, "rvec / rc_edge is NULL");
    ALLEGRO_CHECK_ARG(W_r != nullptr && n_basis >= 1, "W_r is NULL or bad n_basis");
    ALLEGRO_CHECK_ARG(Eenv || n_atoms == 0, "Eenv is NULL");
    ALLEGRO_CHECK_ARG(aligned16(Eenv) && aligned16(w), "Eenv / w not 16-byte aligned");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    const size_t need = allegro_env_workspace(plan, n_atoms, items ? n_items : 0);
    if (items && (workspace == nullptr || workspace_bytes < need)) {
        set_error("allegro_env_radial_forward_typed: workspace too small (%zu < %zu bytes)", workspace_bytes, need);
        return ALLEGRO_ENOMEM;
    }
    EnvArgs a{plan->n, n_atoms, n_edges, row_ptr, items, items ? n_items : (long)n_atoms, rvec, nullptr, scale, Eenv, workspace,
              (cudaStream_t)stream, W_r, n_basis, 1.0, w, rc_edge};
    return ALLEGRO_DISPATCH(plan, launch_env_embed, a);
}

allegro_status_t allegro_env_radial_backward_typed(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const void* gEenv,
                                                   const void* rvec, const void* W_r, int n_basis, const void* rc_edge, double scale, void* g_rvec,
                                                   void* g_w, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((rvec && g_rvec && rc_edge) || n_edges == 0, "rvec / g_rvec / rc_edge is NULL");
    ALLEGRO_CHECK_ARG(W_r != nullptr && n_basis >= 1, "W_r is NULL or bad n_basis");
    ALLEGRO_CHECK_ARG(gEenv || n_atoms == 0, "gEenv is NULL");
    EnvBwdArgs a{plan->n, n_atoms, n_edges, row_ptr, gEenv, rvec, nullptr, scale, g_rvec, g_w, (cudaStream_t)stream, W_r, n_basis, 1.0, rc_edge};
    return ALLEGRO_DISPATCH(plan, launch_env_embed_backward, a);
}

allegro_status_t allegro_tp_forward(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                    long n_items, const void* V, const void* Eenv, const void* path_w, void* out, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((V && out) || n_edges == 0, "V / out is NULL");
    ALLEGRO_CHECK_ARG(Eenv || n_atoms == 0, "Eenv is NULL");
    ALLEGRO_CHECK_ARG(path_w != nullptr || plan->wmode == ALLEGRO_W_SCALAR, "path_w is NULL (dense mode)");
    ALLEGRO_CHECK_ARG(plan->wmode != ALLEGRO_W_DENSE || aligned16(path_w), "dense path_w not 16-byte aligned");
    ALLEGRO_CHECK_ARG(V != out || n_edges == 0, "out aliases V");
    ALLEGRO_CHECK_ARG(aligned16(V) && aligned16(out) && aligned16(Eenv), "feature tensor not 16-byte aligned");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    TpArgs a{};
    a.plan = plan; a.n = plan->n; a.n_atoms = n_atoms; a.n_edges = n_edges; a.row_ptr = row_ptr; a.items = items;
    a.n_items = items ? n_items : (long)n_atoms;
    a.V = V; a.Eenv = Eenv; a.path_w = path_w; a.out = out; a.st = (cudaStream_t)stream;
    return ALLEGRO_DISPATCH(plan, launch_tp_forward, a);
}

// tensor-core dense kernels exist for this shape only (inst_mix3.cu)
static bool dense_tc_shape(const allegro_plan_t* plan) {
    return plan->wmode == ALLEGRO_W_DENSE && plan->dtype == ALLEGRO_F32 && plan->l_max == 2 && plan->n == 64;
}

allegro_status_t allegro_tp_forward_aux(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                        long n_items, const void* V, const void* Eenv, const void* path_w, void* out, void* out_scalars,
                                        void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((V && out) || n_edges == 0, "V / out is NULL");
    ALLEGRO_CHECK_ARG(Eenv || n_atoms == 0, "Eenv is NULL");
    ALLEGRO_CHECK_ARG(path_w != nullptr && aligned16(path_w), "path_w is NULL or not 16-byte aligned");
    ALLEGRO_CHECK_ARG(V != out || n_edges == 0, "out aliases V");
    ALLEGRO_CHECK_ARG(aligned16(V) && aligned16(out) && aligned16(Eenv), "feature tensor not 16-byte aligned");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    if (!dense_tc_shape(plan)) {
        set_error("allegro_tp_forward_aux: dense weights with fp32, l_max = 2, n = 64 only");
        return ALLEGRO_EUNSUPPORTED;
    }
    TpArgs a{};
    a.plan = plan; a.n = plan->n; a.n_atoms = n_atoms; a.n_edges = n_edges; a.row_ptr = row_ptr; a.items = items;
    a.n_items = items ? n_items : (long)n_atoms;
    a.V = V; a.Eenv = Eenv; a.path_w = path_w; a.out = out; a.scalars_out = out_scalars; a.st = (cudaStream_t)stream;
    return ALLEGRO_DISPATCH(plan, launch_tp_forward, a);
}

allegro_status_t allegro_tp_backward_aux(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                         long n_items, const void* G, const void* g_scalars, const void* V, const void* Eenv, const void* path_w,
                                         void* gV, void* gEenv, void* workspace, size_t workspace_bytes, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((G && V) || n_edges == 0, "G / V is NULL");
    ALLEGRO_CHECK_ARG((Eenv && gEenv) || n_atoms == 0, "Eenv / gEenv is NULL");
    ALLEGRO_CHECK_ARG(path_w != nullptr && aligned16(path_w), "path_w is NULL or not 16-byte aligned");
    ALLEGRO_CHECK_ARG(gV == nullptr || (gV != G && gV != V), "gV aliases an input");
    ALLEGRO_CHECK_ARG(aligned16(G) && aligned16(V) && aligned16(gV) && aligned16(Eenv) && aligned16(gEenv) && aligned16(workspace),
                      "tensor not 16-byte aligned");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    if (!dense_tc_shape(plan)) {
        set_error("allegro_tp_backward_aux: dense weights with fp32, l_max = 2, n = 64 only");
        return ALLEGRO_EUNSUPPORTED;
    }
    TpArgs a{};
    a.plan = plan; a.n = plan->n; a.n_atoms = n_atoms; a.n_edges = n_edges; a.row_ptr = row_ptr; a.items = items;
    a.n_items = items ? n_items : (long)n_atoms;
    a.G = G; a.g_scalars = g_scalars; a.V = V; a.Eenv = Eenv; a.path_w = path_w; a.gV = gV; a.gEenv = gEenv;
    a.ws = workspace; a.ws_bytes = workspace_bytes; a.st = (cudaStream_t)stream;
    return ALLEGRO_DISPATCH(plan, launch_tp_backward, a);
}

allegro_status_t allegro_tp_forward_outer(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                          long n_items, const void* rvec, const void* v0, const void* Eenv, const void* path_w, void* out,
                                          void* out_scalars, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((rvec && v0 && out) || n_edges == 0, "rvec / v0 / out is NULL");
    ALLEGRO_CHECK_ARG(Eenv || n_atoms == 0, "Eenv is NULL");
    ALLEGRO_CHECK_ARG(path_w != nullptr && aligned16(path_w), "path_w is NULL or not 16-byte aligned");
    ALLEGRO_CHECK_ARG(aligned16(out) && aligned16(Eenv), "feature tensor not 16-byte aligned");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    if (!dense_tc_shape(plan)) {
        set_error("allegro_tp_forward_outer: dense weights with fp32, l_max = 2, n = 64 only");
        return ALLEGRO_EUNSUPPORTED;
    }
    TpArgs a{};
    a.plan = plan; a.n = plan->n; a.n_atoms = n_atoms; a.n_edges = n_edges; a.row_ptr = row_ptr; a.items = items;
    a.n_items = items ? n_items : (long)n_atoms;
    a.rvec = rvec; a.v0 = v0; a.Eenv = Eenv; a.path_w = path_w; a.out = out; a.scalars_out = out_scalars; a.st = (cudaStream_t)stream;
    return ALLEGRO_DISPATCH(plan, launch_tp_forward, a);
}

allegro_status_t allegro_tp_backward_outer(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                           long n_items, const void* G, const void* g_scalars, const void* rvec, const void* v0, const void* Eenv,
                                           const void* path_w, void* g_v0, void* gY, void* gEenv, void* workspace, size_t workspace_bytes,
                                           void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((G && rvec && v0 && g_v0 && gY) || n_edges == 0, "G / rvec / v0 / g_v0 / gY is NULL");
    ALLEGRO_CHECK_ARG((Eenv && gEenv) || n_atoms == 0, "Eenv / gEenv is NULL");
    ALLEGRO_CHECK_ARG(path_w != nullptr && aligned16(path_w), "path_w is NULL or not 16-byte aligned");
    ALLEGRO_CHECK_ARG(aligned16(G) && aligned16(Eenv) && aligned16(gEenv) && aligned16(workspace), "tensor not 16-byte aligned");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    if (!dense_tc_shape(plan)) {
        set_error("allegro_tp_backward_outer: dense weights with fp32, l_max = 2, n = 64 only");
        return ALLEGRO_EUNSUPPORTED;
    }
    TpArgs a{};
    a.plan = plan; a.n = plan->n; a.n_atoms = n_atoms; a.n_edges = n_edges; a.row_ptr = row_ptr; a.items = items;
    a.n_items = items ? n_items : (long)n_atoms;
    a.G = G; a.g_scalars = g_scalars; a.rvec = rvec; a.v0 = v0; a.Eenv = Eenv; a.path_w = path_w; a.g_v0 = g_v0; a.gYe = gY; a.gEenv = gEenv;
    a.ws = workspace; a.ws_bytes = workspace_bytes; a.st = (cudaStream_t)stream;
    return ALLEGRO_DISPATCH(plan, launch_tp_backward, a);
}

allegro_status_t allegro_tp_forward_energy(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                           long n_items, const void* V, const void* Eenv, const void* path_w, const void* q, double kappa,
                                           void* out, void* e_edge, void* G, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG(V || n_edges == 0, "V is NULL");
    ALLEGRO_CHECK_ARG(out || G || (plan->wmode == ALLEGRO_W_DENSE && e_edge), "out and G are both NULL");
    ALLEGRO_CHECK_ARG(Eenv || n_atoms == 0, "Eenv is NULL");
    ALLEGRO_CHECK_ARG(q != nullptr, "q is NULL");
    ALLEGRO_CHECK_ARG((V != out && V != G && (out != G || !out)) || n_edges == 0, "out / G alias V or each other");
    ALLEGRO_CHECK_ARG(aligned16(V) && aligned16(out) && aligned16(G) && aligned16(Eenv), "feature tensor not 16-byte aligned");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    if (plan->wmode != ALLEGRO_W_SCALAR && !(plan->dtype == ALLEGRO_F32 && plan->l_max == 2 && plan->n == 64 && path_w != nullptr && G == nullptr && e_edge != nullptr)) {
        set_error("allegro_tp_forward_energy: scalar path weights, or dense weights with fp32, l_max = 2, n = 64, e_edge and no G");
        return ALLEGRO_EUNSUPPORTED;
    }
    TpArgs a{};
    a.plan = plan; a.n = plan->n; a.n_atoms = n_atoms; a.n_edges = n_edges; a.row_ptr = row_ptr; a.items = items;
    a.n_items = items ? n_items : (long)n_atoms;
    a.V = V; a.Eenv = Eenv; a.path_w = path_w; a.out = out; a.q = q; a.kappa = kappa; a.e_edge = e_edge; a.Gout = G;
    a.st = (cudaStream_t)stream;
    return ALLEGRO_DISPATCH(plan, launch_tp_forward, a);
}

allegro_status_t allegro_tp_backward(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                     long n_items, const void* G, const void* V, const void* Eenv, const void* path_w, void* gV, void* gEenv,
                                     void* g_path_w, void* workspace, size_t workspace_bytes, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((G && V) || n_edges == 0, "G / V is NULL");
    ALLEGRO_CHECK_ARG((Eenv && gEenv) || n_atoms == 0, "Eenv / gEenv is NULL");
    ALLEGRO_CHECK_ARG(path_w != nullptr || plan->wmode == ALLEGRO_W_SCALAR, "path_w is NULL (dense mode)");
    ALLEGRO_CHECK_ARG(plan->wmode != ALLEGRO_W_DENSE || aligned16(path_w), "dense path_w not 16-byte aligned");
    ALLEGRO_CHECK_ARG(gV == nullptr || (gV != G && gV != V), "gV aliases an input");
    ALLEGRO_CHECK_ARG(aligned16(G) && aligned16(V) && aligned16(gV) && aligned16(Eenv) && aligned16(gEenv) && aligned16(workspace),
                      "tensor not 16-byte aligned");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    TpArgs a{};
    a.plan = plan; a.n = plan->n; a.n_atoms = n_atoms; a.n_edges = n_edges; a.row_ptr = row_ptr; a.items = items;
    a.n_items = items ? n_items : (long)n_atoms;
    a.G = G; a.V = V; a.Eenv = Eenv; a.path_w = path_w; a.gV = gV; a.gEenv = gEenv; a.g_path_w = g_path_w;
    a.ws = workspace; a.ws_bytes = workspace_bytes; a.st = (cudaStream_t)stream;
    return ALLEGRO_DISPATCH(plan, launch_tp_backward, a);
}

allegro_status_t allegro_tp_backward_energy(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                            long n_items, const void* out, const void* V, const void* Eenv, const void* path_w, const void* q,
                                            double kappa, void* gV, void* gEenv, void* g_path_w, void* workspace, size_t workspace_bytes,
                                            void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG(V || n_edges == 0, "V is NULL");
    ALLEGRO_CHECK_ARG(out || n_edges == 0 || (plan->wmode == ALLEGRO_W_DENSE && kappa == 0.0), "out is NULL (allowed in dense mode with kappa == 0 only)");
    ALLEGRO_CHECK_ARG((Eenv && gEenv) || n_atoms == 0, "Eenv / gEenv is NULL");
    ALLEGRO_CHECK_ARG(q != nullptr, "q is NULL");
    ALLEGRO_CHECK_ARG(gV == nullptr || (gV != out && gV != V), "gV aliases an input");
    ALLEGRO_CHECK_ARG(aligned16(out) && aligned16(V) && aligned16(gV) && aligned16(Eenv) && aligned16(gEenv) && aligned16(workspace),
                      "tensor not 16-byte aligned");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    if (plan->wmode != ALLEGRO_W_SCALAR && !(plan->dtype == ALLEGRO_F32 && plan->l_max == 2 && plan->n == 64 && path_w != nullptr && g_path_w == nullptr)) {
        set_error("allegro_tp_backward_energy: scalar path weights, or dense weights with fp32, l_max = 2, n = 64");
        return ALLEGRO_EUNSUPPORTED;
    }
    TpArgs a{};
    a.plan = plan; a.n = plan->n; a.n_atoms = n_atoms; a.n_edges = n_edges; a.row_ptr = row_ptr; a.items = items;
    a.n_items = items ? n_items : (long)n_atoms;
    a.G = out; a.V = V; a.Eenv = Eenv; a.path_w = path_w; a.q = q; a.kappa = kappa; a.gV = gV; a.gEenv = gEenv; a.g_path_w = g_path_w;
    a.ws = workspace; a.ws_bytes = workspace_bytes; a.st = (cudaStream_t)stream;
    return ALLEGRO_DISPATCH(plan, launch_tp_backward, a);
}

allegro_status_t allegro_tp_fused_energy(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items,
                                         long n_items, const void* V, const void* Eenv, const void* path_w, const void* q, double kappa, void* e_edge,
                                         void* gV, void* gEenv, void* g_path_w, void* workspace, size_t workspace_bytes, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((V && e_edge) || n_edges == 0, "V / e_edge is NULL");
    ALLEGRO_CHECK_ARG((Eenv && gEenv) || n_atoms == 0, "Eenv / gEenv is NULL");
    ALLEGRO_CHECK_ARG(q != nullptr, "q is NULL");
    ALLEGRO_CHECK_ARG(gV == nullptr || gV != V, "gV aliases V");
    ALLEGRO_CHECK_ARG(aligned16(V) && aligned16(gV) && aligned16(Eenv) && aligned16(gEenv) && aligned16(workspace), "tensor not 16-byte aligned");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    if (plan->wmode != ALLEGRO_W_SCALAR) {
        set_error("allegro_tp_fused_energy: scalar path weights only");
        return ALLEGRO_EUNSUPPORTED;
    }
    TpArgs a{};
    a.plan = plan; a.n = plan->n; a.n_atoms = n_atoms; a.n_edges = n_edges; a.row_ptr = row_ptr; a.items = items;
    a.n_items = items ? n_items : (long)n_atoms;
    a.V = V; a.Eenv = Eenv; a.path_w = path_w; a.q = q; a.kappa = kappa; a.e_edge = e_edge; a.gV = gV; a.gEenv = gEenv; a.g_path_w = g_path_w;
    a.ws = workspace; a.ws_bytes = workspace_bytes; a.st = (cudaStream_t)stream;
    return ALLEGRO_DISPATCH(plan, launch_tp_fused, a);
}

// ---- second derivative (training): a composition of the first-derivative and forward kernels, see the header
namespace {
struct Dbw { size_t tmp_feat, tmp_env, gw2, bwd, bwd_bytes, total; };
Dbw dbw_layout(const allegro_plan_t* plan, int N, long E) {
    const size_t s = plan->dtype == ALLEGRO_F32 ? 4 : 8;
    const size_t n = plan->n, dV = plan->tab.dV, dE = plan->tab.dE, P = plan->tab.paths.size();
    Dbw L{};
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off += allegro::align_up(bytes ? bytes : 1, 256); return o; };
    L.tmp_feat = take((size_t)E * n * dV * s); L.tmp_env = take((size_t)N * n * dE * s); L.gw2 = take(P * s);
    L.bwd_bytes = allegro_tp_backward_workspace(plan, N, E, 0, 1);
    L.bwd = take(L.bwd_bytes);
    L.total = off;
    return L;
}
}  // namespace

size_t allegro_tp_double_backward_workspace(const allegro_plan_t* plan, int n_atoms, long n_edges) {
    if (!plan || n_atoms < 0 || n_edges < 0) return 0;
    return dbw_layout(plan, n_atoms, n_edges).total;
}

allegro_status_t allegro_tp_double_backward(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const void* G, const void* V,
                                            const void* Eenv, const void* path_w, const void* aV, const void* bE, void* dG, void* dV, void* dEenv,
                                            void* d_path_w, void* workspace, size_t workspace_bytes, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((G && V && aV && dG && dV) || n_edges == 0, "NULL edge tensor");
    ALLEGRO_CHECK_ARG((Eenv && bE && dEenv) || n_atoms == 0, "NULL centre tensor");
    if (plan->wmode != ALLEGRO_W_SCALAR) {
        set_error("allegro_tp_double_backward: scalar path weights only");
        return ALLEGRO_EUNSUPPORTED;
    }
    const Dbw L = dbw_layout(plan, n_atoms, n_edges);
    if (workspace == nullptr || workspace_bytes < L.total || !aligned16(workspace)) {
        set_error("allegro_tp_double_backward: workspace too small or misaligned (%zu < %zu bytes)", workspace_bytes, L.total);
        return ALLEGRO_ENOMEM;
    }
    if (path_w != nullptr) {       // bind once; the four launches below use the bound table
        allegro_status_t b = bind_scalar_weights(plan, path_w, (cudaStream_t)stream);
        if (b != ALLEGRO_OK) return b;
    }
    unsigned char* ws = (unsigned char*)workspace;
    const allegro_dtype_t dt = (allegro_dtype_t)plan->dtype;
    const long feat = n_edges * plan->n * plan->tab.dV;
    allegro_status_t r;
    // dG = fwd(aV, Eenv) + fwd(V, bE)
    if ((r = allegro_tp_forward(plan, n_atoms, n_edges, row_ptr, nullptr, 0, aV, Eenv, nullptr, dG, stream)) != ALLEGRO_OK) return r;
    if ((r = allegro_tp_forward(plan, n_atoms, n_edges, row_ptr, nullptr, 0, V, bE, nullptr, ws + L.tmp_feat, stream)) != ALLEGRO_OK) return r;
    if ((r = allegro_add_inplace(feat, dt, dG, ws + L.tmp_feat, stream)) != ALLEGRO_OK) return r;
    // dEenv = the gEenv output of the first derivative with aV in V's place; its path-weight output is sum C aV Eenv G
    if ((r = allegro_tp_backward(plan, n_atoms, n_edges, row_ptr, nullptr, 0, G, aV, Eenv, nullptr, nullptr, dEenv, d_path_w, ws + L.bwd, L.bwd_bytes,
                                 stream)) != ALLEGRO_OK) return r;
    // dV = the gV output of the first derivative with bE in Eenv's place; its path-weight output is sum C V bE G
    if ((r = allegro_tp_backward(plan, n_atoms, n_edges, row_ptr, nullptr, 0, G, V, bE, nullptr, dV, ws + L.tmp_env, d_path_w ? ws + L.gw2 : nullptr,
                                 ws + L.bwd, L.bwd_bytes, stream)) != ALLEGRO_OK) return r;
    if (d_path_w) return allegro_add_inplace((long)plan->tab.paths.size(), dt, d_path_w, ws + L.gw2, stream);
    return ALLEGRO_OK;
}

size_t allegro_tp_backward_workspace(const allegro_plan_t* plan, int n_atoms, long n_edges, long n_items, int want_g_path_w) {
    (void)n_edges;
    if (!plan) return 0;
    const bool have_items = n_items > 0;
    const long ni = have_items ? n_items : (long)n_atoms;
    return ALLEGRO_DISPATCH(plan, tp_backward_workspace, plan->n, n_atoms, ni, have_items, plan->wmode, want_g_path_w != 0);
}
size_t allegro_env_workspace(const allegro_plan_t* plan, int n_atoms, long n_items) {
    (void)n_atoms;
    if (!plan || n_items <= 0) return 0;
    return (size_t)n_items * plan->n * plan->tab.dE * (plan->dtype == ALLEGRO_F32 ? 4 : 8);
}

allegro_status_t allegro_env_embed_backward(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const void* gEenv,
                                            const void* rvec, const void* w, double scale, void* g_rvec, void* g_w, void* stream) {
    ALLEGRO_CHECK_GRAPH();
    ALLEGRO_CHECK_ARG((rvec && w && g_rvec) || n_edges == 0, "rvec / w / g_rvec is NULL");
    ALLEGRO_CHECK_ARG(gEenv || n_atoms == 0, "gEenv is NULL");
    EnvBwdArgs a{plan->n, n_atoms, n_edges, row_ptr, gEenv, rvec, w, scale, g_rvec, g_w, (cudaStream_t)stream};
    return ALLEGRO_DISPATCH(plan, launch_env_embed_backward, a);
}

allegro_status_t allegro_force_gather(int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* rev, const void* g_rvec,
                                      allegro_dtype_t dtype, void* F, void* stream) {
    ALLEGRO_CHECK_ARG(n_atoms >= 0 && n_edges >= 0, "negative size");
    ALLEGRO_CHECK_ARG((row_ptr && F) || n_atoms == 0, "row_ptr / F is NULL");
    ALLEGRO_CHECK_ARG((rev && g_rvec) || n_edges == 0, "rev / g_rvec is NULL");
    ALLEGRO_CHECK_ARG(dtype == ALLEGRO_F32 || dtype == ALLEGRO_F64, "bad dtype");
    return dtype == ALLEGRO_F32 ? launch_force_gather<float>(n_atoms, n_edges, row_ptr, rev, g_rvec, F, (cudaStream_t)stream)
                                : launch_force_gather<double>(n_atoms, n_edges, row_ptr, rev, g_rvec, F, (cudaStream_t)stream);
}

allegro_status_t allegro_radial_forward(int n_channels, int n_basis, double r_cut, allegro_dtype_t dtype, long n_edges, const void* rvec,
                                        const void* W_r, void* w, void* stream) {
    ALLEGRO_CHECK_ARG(n_channels >= 1 && n_basis >= 1 && n_basis <= 16 && r_cut > 0 && n_edges >= 0, "bad size");
    ALLEGRO_CHECK_ARG(W_r && ((rvec && w) || n_edges == 0), "NULL argument");
    ALLEGRO_CHECK_ARG(dtype == ALLEGRO_F32 || dtype == ALLEGRO_F64, "bad dtype");
    return dtype == ALLEGRO_F32 ? launch_radial_forward<float>(n_channels, n_basis, r_cut, n_edges, rvec, W_r, w, (cudaStream_t)stream)
                                : launch_radial_forward<double>(n_channels, n_basis, r_cut, n_edges, rvec, W_r, w, (cudaStream_t)stream);
}
allegro_status_t allegro_radial_backward(int n_channels, int n_basis, double r_cut, allegro_dtype_t dtype, long n_edges, const void* rvec,
                                         const void* W_r, const void* g_w, void* g_rvec, void* stream) {
    ALLEGRO_CHECK_ARG(n_channels >= 1 && n_basis >= 1 && n_basis <= 16 && r_cut > 0 && n_edges >= 0, "bad size");
    ALLEGRO_CHECK_ARG(W_r && ((rvec && g_w && g_rvec) || n_edges == 0), "NULL argument");
    ALLEGRO_CHECK_ARG(dtype == ALLEGRO_F32 || dtype == ALLEGRO_F64, "bad dtype");
    return dtype == ALLEGRO_F32
               ? launch_radial_backward<float>(n_channels, n_basis, r_cut, n_edges, rvec, W_r, g_w, g_rvec, (cudaStream_t)stream)
               : launch_radial_backward<double>(n_channels, n_basis, r_cut, n_edges, rvec, W_r, g_w, g_rvec, (cudaStream_t)stream);
}

allegro_status_t allegro_edge_energy(const allegro_plan_t* plan, long n_edges, const void* out, const void* q, double kappa, void* e_edge,
                                     void* G, void* stream) {
    ALLEGRO_CHECK_ARG(plan != nullptr && n_edges >= 0, "bad argument");
    ALLEGRO_CHECK_ARG(q && (out || n_edges == 0), "NULL argument");
    return plan->dtype == ALLEGRO_F32
               ? launch_edge_energy<float>(plan->n, plan->tab.dV, n_edges, out, q, kappa, e_edge, G, (cudaStream_t)stream)
               : launch_edge_energy<double>(plan->n, plan->tab.dV, n_edges, out, q, kappa, e_edge, G, (cudaStream_t)stream);
}

allegro_status_t allegro_virial(long n_edges, const void* rvec, const void* g_rvec, allegro_dtype_t dtype, void* W, void* stream) {
    ALLEGRO_CHECK_ARG(n_edges >= 0 && W != nullptr && ((rvec && g_rvec) || n_edges == 0), "bad argument");
    ALLEGRO_CHECK_ARG(dtype == ALLEGRO_F32 || dtype == ALLEGRO_F64, "bad dtype");
    return dtype == ALLEGRO_F32 ? launch_virial<float>(n_edges, rvec, g_rvec, W, (cudaStream_t)stream)
                                : launch_virial<double>(n_edges, rvec, g_rvec, W, (cudaStream_t)stream);
}

allegro_status_t allegro_segment_sum(const int32_t* ptr, int n_segments, const void* vals, allegro_dtype_t dtype, void* out, void* stream) {
    ALLEGRO_CHECK_ARG(n_segments >= 0 && ((ptr && out) || n_segments == 0), "bad argument");
    ALLEGRO_CHECK_ARG(dtype == ALLEGRO_F32 || dtype == ALLEGRO_F64, "bad dtype");
    return dtype == ALLEGRO_F32 ? launch_segment_sum<float>(ptr, n_segments, vals, out, (cudaStream_t)stream)
                                : launch_segment_sum<double>(ptr, n_segments, vals, out, (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------------------------- one-call MD step from HOST buffers
namespace {
struct StepLayout {
    size_t row_ptr, rev, e_ptr, rvec, V, W_r, path_w, q, Eenv, gEenv, out, gV, e_edge, g_r, F, e_tot, total;
};
StepLayout step_layout(const allegro_plan_t* plan, int N, long E, int nb, int want_gV) {
    const size_t s = plan->dtype == ALLEGRO_F32 ? 4 : 8;
    const size_t n = plan->n, dV = plan->tab.dV, dE = plan->tab.dE, P = plan->tab.paths.size();
    StepLayout L{};
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off += allegro::align_up(bytes ? bytes : 1, 256); return o; };
    L.row_ptr = take((size_t)(N + 1) * 4); L.rev = take((size_t)E * 4); L.e_ptr = take(8);
    L.rvec = take((size_t)E * 3 * s); L.V = take((size_t)E * n * dV * s); L.W_r = take(n * nb * s); L.path_w = take(P * s); L.q = take(n * s);
    L.Eenv = take((size_t)N * n * dE * s); L.gEenv = take((size_t)N * n * dE * s); L.out = take((size_t)E * n * dV * s);
    L.gV = want_gV ? take((size_t)E * n * dV * s) : 0;
    L.e_edge = take((size_t)E * s); L.g_r = take((size_t)E * 3 * s); L.F = take((size_t)N * 3 * s); L.e_tot = take(s);
    L.total = off;
    return L;
}
}  // namespace

size_t allegro_layer_step_host_workspace(const allegro_plan_t* plan, int n_atoms, long n_edges, int n_basis, int want_gV) {
    if (!plan || n_atoms < 0 || n_edges < 0 || n_basis < 1) return 0;
    return step_layout(plan, n_atoms, n_edges, n_basis, want_gV).total;
}

allegro_status_t allegro_layer_step_host(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr_host,
                                         const int32_t* rev_host, const void* rvec_host, const void* V_host, const void* W_r_host, int n_basis,
                                         double r_cut, const void* path_w_host, const void* q_host, double kappa, double scale, int want_gV,
                                         void* F_host, void* e_tot_host, void* workspace, size_t workspace_bytes, void* stream) {
    ALLEGRO_CHECK_ARG(plan != nullptr && n_atoms >= 0 && n_edges >= 0 && n_edges < 2147483647L, "bad plan / sizes");
    ALLEGRO_CHECK_ARG(row_ptr_host && W_r_host && path_w_host && q_host && F_host && e_tot_host, "NULL host argument");
    ALLEGRO_CHECK_ARG((rev_host && rvec_host && V_host) || n_edges == 0, "NULL host tensor");
    ALLEGRO_CHECK_ARG(plan->wmode == ALLEGRO_W_SCALAR, "scalar path weights only");
    const StepLayout L = step_layout(plan, n_atoms, n_edges, n_basis, want_gV);
    if (workspace == nullptr || workspace_bytes < L.total || !aligned16(workspace)) {
        set_error("allegro_layer_step_host: workspace too small or misaligned (%zu < %zu bytes)", workspace_bytes, L.total);
        return ALLEGRO_ENOMEM;
    }
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char* ws = (unsigned char*)workspace;
    const size_t s = plan->dtype == ALLEGRO_F32 ? 4 : 8;
    const size_t n = plan->n, dV = plan->tab.dV;
    const int32_t e_ptr[2] = {0, (int32_t)n_edges};
    ALLEGRO_CUDA(cudaMemcpyAsync(ws + L.row_ptr, row_ptr_host, (size_t)(n_atoms + 1) * 4, cudaMemcpyHostToDevice, st));
    ALLEGRO_CUDA(cudaMemcpyAsync(ws + L.e_ptr, e_ptr, 8, cudaMemcpyHostToDevice, st));
    if (n_edges > 0) {
        ALLEGRO_CUDA(cudaMemcpyAsync(ws + L.rev, rev_host, (size_t)n_edges * 4, cudaMemcpyHostToDevice, st));
        ALLEGRO_CUDA(cudaMemcpyAsync(ws + L.rvec, rvec_host, (size_t)n_edges * 3 * s, cudaMemcpyHostToDevice, st));
        ALLEGRO_CUDA(cudaMemcpyAsync(ws + L.V, V_host, (size_t)n_edges * n * dV * s, cudaMemcpyHostToDevice, st));
    }
    ALLEGRO_CUDA(cudaMemcpyAsync(ws + L.W_r, W_r_host, n * n_basis * s, cudaMemcpyHostToDevice, st));
    fold_host(plan, path_w_host);   // the combined tensor travels as a kernel parameter: nothing to copy
    ALLEGRO_CUDA(cudaMemcpyAsync(ws + L.q, q_host, n * s, cudaMemcpyHostToDevice, st));
    const int32_t* rp = (const int32_t*)(ws + L.row_ptr);
    allegro_status_t r;
    if ((r = allegro_env_radial_forward(plan, n_atoms, n_edges, rp, nullptr, 0, ws + L.rvec, ws + L.W_r, n_basis, r_cut, scale, nullptr,
                                        ws + L.Eenv, nullptr, 0, stream)) != ALLEGRO_OK) return r;
    if ((r = allegro_tp_forward_energy(plan, n_atoms, n_edges, rp, nullptr, 0, ws + L.V, ws + L.Eenv, nullptr, ws + L.q, kappa, ws + L.out,
                                       ws + L.e_edge, nullptr, stream)) != ALLEGRO_OK) return r;
    if ((r = allegro_tp_backward_energy(plan, n_atoms, n_edges, rp, nullptr, 0, ws + L.out, ws + L.V, ws + L.Eenv, nullptr, ws + L.q, kappa,
                                        want_gV ? ws + L.gV : nullptr, ws + L.gEenv, nullptr, nullptr, 0, stream)) != ALLEGRO_OK) return r;
    if ((r = allegro_env_radial_backward(plan, n_atoms, n_edges, rp, ws + L.gEenv, ws + L.rvec, ws + L.W_r, n_basis, r_cut, scale, ws + L.g_r,
                                         nullptr, stream)) != ALLEGRO_OK) return r;
    if ((r = allegro_force_gather(n_atoms, n_edges, rp, (const int32_t*)(ws + L.rev), ws + L.g_r, (allegro_dtype_t)plan->dtype, ws + L.F,
                                  stream)) != ALLEGRO_OK) return r;
    if ((r = allegro_segment_sum((const int32_t*)(ws + L.e_ptr), 1, ws + L.e_edge, (allegro_dtype_t)plan->dtype, ws + L.e_tot, stream)) != ALLEGRO_OK)
        return r;
    ALLEGRO_CUDA(cudaMemcpyAsync(F_host, ws + L.F, (size_t)n_atoms * 3 * s, cudaMemcpyDeviceToHost, st));
    ALLEGRO_CUDA(cudaMemcpyAsync(e_tot_host, ws + L.e_tot, s, cudaMemcpyDeviceToHost, st));
    ALLEGRO_CUDA(cudaStreamSynchronize(st));
    return ALLEGRO_OK;
}

// ---------------------------------------------------------------------------------------------- one-launch MD step (CUDA graph inside the library)
struct allegro_step {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    unsigned char* ws = nullptr;
    size_t off_Eenv = 0, off_gEenv = 0, off_out = 0, off_gV = 0, off_e_edge = 0, off_g_r = 0, off_e_ptr = 0, total = 0;
    bool fused = true;   // l_max <= 2: forward + energy + VJP in one kernel (no `out`); l_max = 3: two kernels (the fused one is slower there)
    bool have_gV = false;
    int kernels = 0;
};
namespace {
void graph_step_layout(const allegro_plan_t* plan, int N, long E, int want_gV, allegro_step& L) {
    const size_t s = plan->dtype == ALLEGRO_F32 ? 4 : 8;
    const size_t n = plan->n, dV = plan->tab.dV, dE = plan->tab.dE;
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off += allegro::align_up(bytes ? bytes : 1, 256); return o; };
    L.off_e_ptr = take(8);
    L.fused = plan->l_max <= 2;
    L.off_Eenv = take((size_t)N * n * dE * s); L.off_gEenv = take((size_t)N * n * dE * s);
    L.off_out = L.fused ? 0 : take((size_t)E * n * dV * s);
    L.off_gV = want_gV ? take((size_t)E * n * dV * s) : 0;
    L.off_e_edge = take((size_t)E * s); L.off_g_r = take((size_t)E * 3 * s);
    L.total = off;
    L.have_gV = want_gV != 0;
}
}  // namespace

size_t allegro_layer_step_workspace(const allegro_plan_t* plan, int n_atoms, long n_edges, int want_gV) {
    if (!plan || n_atoms < 0 || n_edges < 0) return 0;
    allegro_step L;
    graph_step_layout(plan, n_atoms, n_edges, want_gV, L);
    return L.total;
}

allegro_status_t allegro_layer_step_create(const allegro_plan_t* plan, int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* rev,
                                           const void* rvec, const void* V, const void* W_r, int n_basis, double r_cut, const void* q, double kappa,
                                           double scale, int want_gV, void* F, void* e_tot, void* workspace, size_t workspace_bytes,
                                           allegro_step_t** out) {
    ALLEGRO_CHECK_ARG(out != nullptr, "out is NULL");
    *out = nullptr;
    ALLEGRO_CHECK_ARG(plan != nullptr && n_atoms >= 0 && n_edges >= 0 && n_edges < 2147483647L, "bad plan / sizes");
    ALLEGRO_CHECK_ARG(plan->wmode == ALLEGRO_W_SCALAR, "scalar path weights only");
    ALLEGRO_CHECK_ARG(plan->cw_bound, "bind the path weights first (allegro_plan_bind_weights)");
    ALLEGRO_CHECK_ARG(row_ptr && W_r && q && F && e_tot, "NULL argument");
    ALLEGRO_CHECK_ARG((rev && rvec && V) || n_edges == 0, "NULL tensor");
    allegro_step* st = new (std::nothrow) allegro_step();
    if (!st) { set_error("allegro_layer_step_create: out of host memory"); return ALLEGRO_ENOMEM; }
    graph_step_layout(plan, n_atoms, n_edges, want_gV, *st);
    if (workspace == nullptr || workspace_bytes < st->total || !aligned16(workspace)) {
        set_error("allegro_layer_step_create: workspace too small or misaligned (%zu < %zu bytes)", workspace_bytes, st->total);
        delete st;
        return ALLEGRO_ENOMEM;
    }
    st->ws = (unsigned char*)workspace;
    unsigned char* ws = st->ws;
    cudaStream_t cs = nullptr;
    allegro_status_t r = ALLEGRO_OK;
    auto fail = [&](allegro_status_t code) {
        if (cs) cudaStreamDestroy(cs);
        allegro_layer_step_destroy(st);
        return code;
    };
    if (cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking) != cudaSuccess) { set_error("allegro_layer_step_create: cudaStreamCreate failed"); return fail(ALLEGRO_ECUDA); }
    const int32_t e_ptr[2] = {0, (int32_t)n_edges};
    if (cudaMemcpyAsync(ws + st->off_e_ptr, e_ptr, 8, cudaMemcpyHostToDevice, cs) != cudaSuccess || cudaStreamSynchronize(cs) != cudaSuccess) {
        set_error("allegro_layer_step_create: workspace is not device memory?");
        return fail(ALLEGRO_ECUDA);
    }
    auto sequence = [&](void* stream) -> allegro_status_t {
        allegro_status_t s;
        if ((s = allegro_env_radial_forward(plan, n_atoms, n_edges, row_ptr, nullptr, 0, rvec, W_r, n_basis, r_cut, scale, nullptr, ws + st->off_Eenv,
                                            nullptr, 0, stream)) != ALLEGRO_OK) return s;
        if (st->fused) {
            if ((s = allegro_tp_fused_energy(plan, n_atoms, n_edges, row_ptr, nullptr, 0, V, ws + st->off_Eenv, nullptr, q, kappa, ws + st->off_e_edge,
                                             want_gV ? ws + st->off_gV : nullptr, ws + st->off_gEenv, nullptr, nullptr, 0, stream)) != ALLEGRO_OK) return s;
        } else {
            if ((s = allegro_tp_forward_energy(plan, n_atoms, n_edges, row_ptr, nullptr, 0, V, ws + st->off_Eenv, nullptr, q, kappa, ws + st->off_out,
                                               ws + st->off_e_edge, nullptr, stream)) != ALLEGRO_OK) return s;
            if ((s = allegro_tp_backward_energy(plan, n_atoms, n_edges, row_ptr, nullptr, 0, ws + st->off_out, V, ws + st->off_Eenv, nullptr, q, kappa,
                                                want_gV ? ws + st->off_gV : nullptr, ws + st->off_gEenv, nullptr, nullptr, 0, stream)) != ALLEGRO_OK) return s;
        }
        if ((s = allegro_env_radial_backward(plan, n_atoms, n_edges, row_ptr, ws + st->off_gEenv, rvec, W_r, n_basis, r_cut, scale, ws + st->off_g_r,
                                             nullptr, stream)) != ALLEGRO_OK) return s;
        if ((s = allegro_force_gather(n_atoms, n_edges, row_ptr, rev, ws + st->off_g_r, (allegro_dtype_t)plan->dtype, F, stream)) != ALLEGRO_OK) return s;
        return allegro_segment_sum((const int32_t*)(ws + st->off_e_ptr), 1, ws + st->off_e_edge, (allegro_dtype_t)plan->dtype, e_tot, stream);
    };
    // one eager pass first: it sets every kernel's attributes outside the capture and proves the arguments
    if ((r = sequence(cs)) != ALLEGRO_OK) return fail(r);
    if (cudaStreamSynchronize(cs) != cudaSuccess) { set_error("allegro_layer_step_create: the eager pass failed: %s", cudaGetErrorString(cudaGetLastError())); return fail(ALLEGRO_ECUDA); }
    const long k0 = g_launches.load();
    if (cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { set_error("allegro_layer_step_create: cudaStreamBeginCapture failed"); return fail(ALLEGRO_ECUDA); }
    r = sequence(cs);
    const cudaError_t ce = cudaStreamEndCapture(cs, &st->graph);
    st->kernels = (int)(g_launches.load() - k0);
    if (r != ALLEGRO_OK) return fail(r);
    if (ce != cudaSuccess || st->graph == nullptr) { set_error("allegro_layer_step_create: capture failed: %s", cudaGetErrorString(ce)); return fail(ALLEGRO_ECUDA); }
    if (cudaGraphInstantiate(&st->exec, st->graph, 0) != cudaSuccess) { set_error("allegro_layer_step_create: cudaGraphInstantiate failed"); return fail(ALLEGRO_ECUDA); }
    cudaStreamDestroy(cs);
    *out = st;
    return ALLEGRO_OK;
}

allegro_status_t allegro_layer_step_launch(allegro_step_t* step, void* stream) {
    ALLEGRO_CHECK_ARG(step != nullptr && step->exec != nullptr, "step is NULL");
    ALLEGRO_CUDA(cudaGraphLaunch(step->exec, (cudaStream_t)stream));
    g_launches.fetch_add(step->kernels);
    return ALLEGRO_OK;
}
void* allegro_layer_step_buffer(const allegro_step_t* step, const char* name) {
    if (!step || !name) return nullptr;
    if (!strcmp(name, "Eenv")) return step->ws + step->off_Eenv;
    if (!strcmp(name, "gEenv")) return step->ws + step->off_gEenv;
    if (!strcmp(name, "out")) return step->fused ? nullptr : step->ws + step->off_out;
    if (!strcmp(name, "gV")) return step->have_gV ? step->ws + step->off_gV : nullptr;
    if (!strcmp(name, "e_edge")) return step->ws + step->off_e_edge;
    if (!strcmp(name, "g_rvec")) return step->ws + step->off_g_r;
    return nullptr;
}
int allegro_layer_step_num_kernels(const allegro_step_t* step) { return step ? step->kernels : -1; }
void allegro_layer_step_destroy(allegro_step_t* step) {
    if (!step) return;
    if (step->exec) cudaGraphExecDestroy(step->exec);
    if (step->graph) cudaGraphDestroy(step->graph);
    delete step;
}

// ---------------------------------------------------------------------------------------------- two-layer model helpers
allegro_status_t allegro_edge_embed(const allegro_plan_t* plan, long n_edges, const void* rvec, const void* W_x0, const void* W_v0, int n_basis,
                                    double r_cut, void* x0, void* V0, void* stream) {
    ALLEGRO_CHECK_ARG(plan != nullptr && n_edges >= 0, "plan is NULL or n_edges < 0");
    ALLEGRO_CHECK_ARG((rvec && x0 && V0) || n_edges == 0, "NULL tensor");
    ALLEGRO_CHECK_ARG(W_x0 && W_v0 && n_basis >= 1 && r_cut > 0, "bad weights / n_basis / r_cut");
    ALLEGRO_CHECK_ARG(aligned16(V0), "V0 not 16-byte aligned");
    EmbedArgs a{plan->n, n_basis, r_cut, n_edges, rvec, W_x0, W_v0, x0, V0, nullptr, nullptr, nullptr, (cudaStream_t)stream};
    return ALLEGRO_DISPATCH(plan, launch_edge_embed, a);
}
allegro_status_t allegro_edge_embed_backward(const allegro_plan_t* plan, long n_edges, const void* rvec, const void* W_x0, const void* W_v0,
                                             int n_basis, double r_cut, const void* g_x0, const void* gV0, void* g_rvec, void* stream) {
    ALLEGRO_CHECK_ARG(plan != nullptr && n_edges >= 0, "plan is NULL or n_edges < 0");
    ALLEGRO_CHECK_ARG((rvec && g_x0 && gV0 && g_rvec) || n_edges == 0, "NULL tensor");
    ALLEGRO_CHECK_ARG(W_x0 && W_v0 && n_basis >= 1 && r_cut > 0, "bad weights / n_basis / r_cut");
    ALLEGRO_CHECK_ARG(aligned16(gV0), "gV0 not 16-byte aligned");
    EmbedArgs a{plan->n, n_basis, r_cut, n_edges, rvec, W_x0, W_v0, nullptr, nullptr, g_x0, gV0, g_rvec, (cudaStream_t)stream};
    return ALLEGRO_DISPATCH(plan, launch_edge_embed_backward, a);
}
allegro_status_t allegro_edge_embed_factors(const allegro_plan_t* plan, long n_edges, const void* rvec, const void* W_x0, const void* W_v0, int n_basis,
                                            double r_cut, void* x0, void* v0, void* stream) {
    ALLEGRO_CHECK_ARG(plan != nullptr && n_edges >= 0, "plan is NULL or n_edges < 0");
    ALLEGRO_CHECK_ARG((rvec && x0 && v0) || n_edges == 0, "NULL tensor");
    ALLEGRO_CHECK_ARG(W_x0 && W_v0 && n_basis >= 1 && r_cut > 0, "bad weights / n_basis / r_cut");
    EmbedArgs a{plan->n, n_basis, r_cut, n_edges, rvec, W_x0, W_v0, x0, nullptr, nullptr, nullptr, nullptr, (cudaStream_t)stream};
    a.v0_out = v0;
    return ALLEGRO_DISPATCH(plan, launch_edge_embed, a);
}
allegro_status_t allegro_edge_embed_factors_backward(const allegro_plan_t* plan, long n_edges, const void* rvec, const void* W_x0, const void* W_v0,
                                                     int n_basis, double r_cut, const void* g_x0, const void* g_v0, const void* gY, void* g_rvec,
                                                     void* stream) {
    ALLEGRO_CHECK_ARG(plan != nullptr && n_edges >= 0, "plan is NULL or n_edges < 0");
    ALLEGRO_CHECK_ARG((rvec && g_x0 && g_v0 && gY && g_rvec) || n_edges == 0, "NULL tensor");
    ALLEGRO_CHECK_ARG(W_x0 && W_v0 && n_basis >= 1 && r_cut > 0, "bad weights / n_basis / r_cut");
    EmbedArgs a{plan->n, n_basis, r_cut, n_edges, rvec, W_x0, W_v0, nullptr, nullptr, g_x0, nullptr, g_rvec, (cudaStream_t)stream};
    a.g_v0 = g_v0; a.gYe = gY;
    return ALLEGRO_DISPATCH(plan, launch_edge_embed_backward, a);
}
allegro_status_t allegro_linear(long n_rows, int n_out, int n_in, allegro_dtype_t dtype, const void* x, const void* W, int transpose_w,
                                int accumulate, void* y, void* stream) {
    ALLEGRO_CHECK_ARG(n_rows >= 0 && n_out >= 1 && n_in >= 1, "bad size");
    ALLEGRO_CHECK_ARG((x && y) || n_rows == 0, "x / y is NULL");
    ALLEGRO_CHECK_ARG(W != nullptr && x != y, "W is NULL or y aliases x");
    return dtype == ALLEGRO_F32 ? launch_linear<float>(n_rows, n_out, n_in, x, W, transpose_w, accumulate, y, (cudaStream_t)stream)
                                : launch_linear<double>(n_rows, n_out, n_in, x, W, transpose_w, accumulate, y, (cudaStream_t)stream);
}
allegro_status_t allegro_latent_forward(long n_edges, int n_channels, int dim_v, double r_cut, allegro_dtype_t dtype, const void* rvec,
                                        const void* x, const void* V, const void* A, void* z, void* x_new, void* stream) {
    ALLEGRO_CHECK_ARG(n_edges >= 0 && n_channels >= 1 && dim_v >= 1 && r_cut > 0, "bad size");
    ALLEGRO_CHECK_ARG((rvec && x && V && z && x_new) || n_edges == 0, "NULL tensor");
    ALLEGRO_CHECK_ARG(A != nullptr, "A is NULL");
    return dtype == ALLEGRO_F32 ? launch_latent_forward<float>(n_edges, n_channels, dim_v, r_cut, rvec, x, V, A, z, x_new, (cudaStream_t)stream)
                                : launch_latent_forward<double>(n_edges, n_channels, dim_v, r_cut, rvec, x, V, A, z, x_new, (cudaStream_t)stream);
}
allegro_status_t allegro_latent_backward(long n_edges, int n_channels, int dim_v, double r_cut, allegro_dtype_t dtype, const void* rvec,
                                         const void* z, const void* g_xnew, const void* A, void* g_x, void* gV, void* g_rvec, void* stream) {
    ALLEGRO_CHECK_ARG(n_edges >= 0 && n_channels >= 1 && dim_v >= 1 && r_cut > 0, "bad size");
    ALLEGRO_CHECK_ARG((rvec && z && g_xnew && g_x && gV && g_rvec) || n_edges == 0, "NULL tensor");
    ALLEGRO_CHECK_ARG(A != nullptr, "A is NULL");
    return dtype == ALLEGRO_F32
               ? launch_latent_backward<float>(n_edges, n_channels, dim_v, r_cut, rvec, z, g_xnew, A, g_x, gV, g_rvec, (cudaStream_t)stream)
               : launch_latent_backward<double>(n_edges, n_channels, dim_v, r_cut, rvec, z, g_xnew, A, g_x, gV, g_rvec, (cudaStream_t)stream);
}
allegro_status_t allegro_add_inplace(long count, allegro_dtype_t dtype, void* y, const void* x, void* stream) {
    ALLEGRO_CHECK_ARG(count >= 0 && ((x && y) || count == 0), "bad argument");
    return dtype == ALLEGRO_F32 ? launch_add_inplace<float>(count, y, x, (cudaStream_t)stream)
                                : launch_add_inplace<double>(count, y, x, (cudaStream_t)stream);
}

const char* allegro_status_str(allegro_status_t s) {
    switch (s) {
        case ALLEGRO_OK: return "ALLEGRO_OK";
        case ALLEGRO_EINVAL: return "ALLEGRO_EINVAL";
        case ALLEGRO_EUNSUPPORTED: return "ALLEGRO_EUNSUPPORTED";
        case ALLEGRO_ECUDA: return "ALLEGRO_ECUDA";
        case ALLEGRO_ENOMEM: return "ALLEGRO_ENOMEM";
    }
    return "ALLEGRO_?";
}
const char* allegro_last_error(void) { return t_err; }
long allegro_launch_count(void) { return g_launches.load(); }

}  // extern "C"
