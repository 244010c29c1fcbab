// launch.h -- argument packs and launcher declarations shared by api.cu (dispatch) and the
// per-(dtype, l_max) instantiation units inst_tp.cu / inst_env.cu.  Internal, not part of the ABI.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

#include "allegro_b200.h"
#include "plan.h"

namespace allegro {

struct EnvArgs {
    int n, n_atoms;
    long n_edges;
    const int32_t* row_ptr;
    const int32_t* items;  // nullable
    long n_items;          // number of CTAs' worth of work (== n_atoms when items == nullptr)
    const void* rvec;
    const void* w;
    double scale;
    void* Eenv;
    void* ws;
    cudaStream_t st;
    // fused radial variant (allegro_env_radial_forward): W_r != nullptr; w is then an optional OUTPUT (w_out)
    const void* W_r;
    int nb;
    double rc;
    void* w_out;
    const void* rc_edge;  // nullable: per-edge cutoff radii T[E] (per-edge-type cutoffs, reading A27); overrides rc
};
struct EnvBwdArgs {
    int n, n_atoms;
    long n_edges;
    const int32_t* row_ptr;
    const void* gEenv;
    const void* rvec;
    const void* w;
    double scale;
    void* g_rvec;
    void* g_w;  // nullable
    cudaStream_t st;
    // fused radial variant (allegro_env_radial_backward): W_r != nullptr; w is not read
    const void* W_r;
    int nb;
    double rc;
    const void* rc_edge;  // nullable: per-edge cutoff radii T[E]
};
struct EnvLinArgs {
    int n_out, n_in, n_atoms;
    long n_edges;
    const int32_t* row_ptr;
    const void* rvec;
    const void* x;
    const void* W;        // [n_out][n_in]
    double scale;
    void* Eenv;           // forward output
    const void* gEenv;    // backward input
    void* g_rvec;
    int acc_g_rvec;
    void* g_x;
    int acc_g_x;
    cudaStream_t st;
};
struct TpArgs {
    const allegro_plan* plan;
    int n, n_atoms;
    long n_edges;
    const int32_t* row_ptr;
    const int32_t* items;  // nullable
    long n_items;
    const void* V;
    const void* Eenv;
    const void* path_w;
    void* out;  // forward (nullable in the energy variant)
    // forward energy epilogue (allegro_tp_forward_energy): all nullable
    const void* q;
    double kappa;
    void* e_edge;
    void* Gout;
    // backward
    const void* G;
    void* gV;        // nullable
    void* gEenv;     // required
    void* g_path_w;  // nullable
    void* ws;
    size_t ws_bytes;
    cudaStream_t st;
    // dense mode, fp32 / l_max 2 / n 64 only (allegro_tp_forward_aux / _backward_aux): compact side channel of the 0e scalars
    void* scalars_out;      // forward: T[E][n] copy of out[:, :, 0e]
    const void* g_scalars;  // backward: T[E][n] added to G[:, :, 0e]
    // layer-1 specialisation (allegro_tp_forward_outer / _backward_outer): V = v0 (x) Y(rhat) generated on chip, V == NULL
    const void* rvec;       // T[E][3]
    const void* v0;         // T[E][n]
    void* g_v0;             // backward: T[E][n]
    void* gYe;              // backward: T[E][dE]
};

struct EmbedArgs {
    int n, nb;
    double rc;
    long n_edges;
    const void* rvec;
    const void* W_x0;
    const void* W_v0;
    void* x0;          // forward outputs
    void* V0;
    const void* g_x0;  // backward inputs
    const void* gV0;
    void* g_rvec;      // backward: accumulated into
    cudaStream_t st;
    void* v0_out;      // forward, nullable: the factor v0[e][n] of V0 = v0 (x) Y (V0 itself is then optional)
    const void* g_v0;  // backward, with gV0 == NULL: <gV0[e][n], Y(e)>            (allegro_tp_backward_outer)
    const void* gYe;   // backward, with gV0 == NULL: sum_n gV0[e][n][slot j] v0[e][n]
};
template <typename T, int L> allegro_status_t launch_edge_embed(const EmbedArgs& a);
template <typename T, int L> allegro_status_t launch_edge_embed_backward(const EmbedArgs& a);
template <typename T, int L> allegro_status_t launch_env_embed(const EnvArgs& a);
template <typename T, int L> allegro_status_t launch_env_embed_backward(const EnvBwdArgs& a);
template <typename T, int L> allegro_status_t launch_env_linear(const EnvLinArgs& a);
template <typename T, int L> allegro_status_t launch_env_linear_backward(const EnvLinArgs& a);
template <typename T, int L> allegro_status_t launch_tp_forward(const TpArgs& a);
template <typename T, int L> allegro_status_t launch_tp_backward(const TpArgs& a);
template <typename T, int L> allegro_status_t launch_tp_fused(const TpArgs& a);
template <typename T, int L> size_t tp_backward_workspace(int n, int n_atoms, long n_items, bool have_items, int wmode, bool want_gw);

// dtype-only helpers (misc.cu)
template <typename T>
allegro_status_t launch_radial_forward(int n, int nb, double rc, long E, const void* rvec, const void* W_r, void* w, cudaStream_t st);
template <typename T>
allegro_status_t launch_radial_backward(int n, int nb, double rc, long E, const void* rvec, const void* W_r, const void* g_w, void* g_rvec,
                                        cudaStream_t st);
template <typename T>
allegro_status_t launch_force_gather(int n_atoms, long E, const int32_t* row_ptr, const int32_t* rev, const void* g_rvec, void* F, cudaStream_t st);
template <typename T>
allegro_status_t launch_edge_energy(int n, int dV, long E, const void* out, const void* q, double kappa, void* e_edge, void* G, cudaStream_t st);
template <typename T>
allegro_status_t launch_virial(long E, const void* rvec, const void* g_rvec, void* W, cudaStream_t st);
template <typename T>
allegro_status_t launch_segment_sum(const int32_t* ptr, int nseg, const void* vals, void* out, cudaStream_t st);

// 2-D tensor map over a feature tensor whose rows are exactly 128 bytes: [rows][32 x 4 B], box = box_rows rows, 128-byte swizzle
// (api.cu; cuTensorMapEncodeTiled through cudaGetDriverEntryPoint, no link-time dependency on libcuda)
allegro_status_t make_row128_map(CUtensorMap* map, const void* base, unsigned long long rows, unsigned box_rows);

// scalar path weights: fold path_w (DEVICE, [P]) with the CG table into plan->cw on the host (api.cu); synchronises the stream
allegro_status_t bind_scalar_weights(const allegro_plan* plan, const void* path_w_dev, cudaStream_t st);

// dense per-path mix on tcgen05 (inst_mix3.cu)
allegro_status_t launch_mix3_forward_f32_l2_n64(const TpArgs& a);
allegro_status_t launch_mix3_backward_f32_l2_n64(const TpArgs& a, float* gE_dst, int gE_by_item);

// dtype-only pieces of the two-layer model (model.cu)
template <typename T>
allegro_status_t launch_linear(long E, int n_out, int n_in, const void* x, const void* W, int transpose_w, int accumulate, void* y, cudaStream_t st);
template <typename T>
allegro_status_t launch_latent_forward(long E, int n, int dV, double rc, const void* rvec, const void* x, const void* V, const void* A, void* z,
                                       void* x_new, cudaStream_t st);
template <typename T>
allegro_status_t launch_latent_backward(long E, int n, int dV, double rc, const void* rvec, const void* z, const void* g_xnew, const void* A,
                                        void* g_x, void* gV, void* g_rvec, cudaStream_t st);
template <typename T>
allegro_status_t launch_add_inplace(long count, void* y, const void* x, cudaStream_t st);

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace allegro
