// plan.h -- internal host-side plan tables of the product library (not part of the ABI).
// Shares nothing with oracle/: the complex CG coefficients here come from the ladder-operator
// recursion, not from the Racah sum.
#pragma once
#include <cstdint>
#include <vector>

namespace allegro {

struct PathInfo {
    int l1, p1, l2, l3, p3, off1, off2, off3;
};
struct NonZero {
    int path, i, j, k;
    double c;
};

struct PlanTables {
    int l_max = 0;
    int dV = 0, dE = 0;
    std::vector<PathInfo> paths;
    std::vector<NonZero> nnz;  // sorted (path, i, j, k)
};

// <j1 m1 j2 m2 | J M>, Condon-Shortley, all (m1, m2) for one (j1, j2, J): table[(m1+j1)*(2j2+1) + (m2+j2)][M+J]
void cg_complex_ladder(int j1, int j2, int J, std::vector<double>& table);
// real-basis block C[m1][m2][M] (reading A2: C = Re T + Im T)
void cg_real_block(int l1, int l2, int l3, std::vector<double>& C);
void build_tables(int l_max, PlanTables& t);
long build_segments(const int32_t* row_ptr, int n_atoms, int tile_edges, int32_t* items, long cap);

}  // namespace allegro

struct allegro_plan {
    int l_max, n, dtype, wmode;
    allegro::PlanTables tab;
    mutable void* dense_img = nullptr;  // device: weight images of the tcgen05 dense mix (inst_mix3.cu), plan-owned
    // output blocks (l3, p3) that are computed: bit b = block b in component order (0e, 0o, 1e, 1o, ...); the others are written as
    // zeros by the forward and ignored in the cotangent by the VJP (allegro_plan_set_out_blocks)
    unsigned out_blocks = ~0u;
    // input blocks (l1, p1) of V that are present: the others are taken as identically zero (not read; their gV is written as
    // zeros) -- a first layer fed with V0 = v (x) Y(rhat) only has the natural-parity blocks (allegro_plan_set_in_blocks)
    unsigned in_blocks = ~0u;
    // scalar mode: the folded coefficient table cw[z] = path_w[path(z)] * C_z of the weights bound last (allegro_plan_bind_weights),
    // in tab.nnz order, already rounded to the plan's dtype; passed to the kernels BY VALUE as a kernel parameter
    mutable std::vector<double> cw;
    mutable bool cw_bound = false;
    bool path_active(int p) const {
        const allegro::PathInfo& q = tab.paths[p];
        return ((out_blocks >> (2 * q.l3 + q.p3)) & 1u) != 0 && ((in_blocks >> (2 * q.l1 + q.p1)) & 1u) != 0;   // parity: 0 even, 1 odd
    }
};
