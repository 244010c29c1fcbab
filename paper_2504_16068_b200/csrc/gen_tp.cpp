// gen_tp.cpp -- build-time code generator: unrolls the compressed sparse CG tensor of plan.cpp into
// straight-line CUDA device functions, one set per l_max (north_star: "the sparse CG table unrolled at
// compile time per (l_max, parity) plan").
//
// usage: gen_tp <out_dir>   -> writes <out_dir>/tp_gen.cuh
//
// Two flavours are emitted per l_max:
//   folded : coefficient z is read as cw[z] (= path_w[path(z)] * C_z, the "combined tensor"); cw is the first argument, a
//            reference to a __grid_constant__ kernel parameter -> a constant-bank FFMA operand; output index = out component k.
//   paths  : coefficient is a compile-time literal, output index = toff(path) + M (one slot per
//            (path, M): the un-weighted t[e][n][p][M] that feeds the dense per-path channel mix and
//            the path-weight gradient).
#include <cstdio>
#include <cstdlib>
#include <map>
#include <string>
#include <vector>

#include "plan.h"

using namespace allegro;

struct Term { int k; int z; double c; };
struct Pair { int i, j; std::vector<Term> terms; };

static std::vector<Pair> group_pairs(const PlanTables& t, bool paths_flavour, const std::vector<int>& toff) {
    std::map<std::pair<int, int>, int> idx;
    std::vector<Pair> pairs;
    for (size_t z = 0; z < t.nnz.size(); ++z) {
        const NonZero& q = t.nnz[z];
        auto key = std::make_pair(q.i, q.j);
        auto it = idx.find(key);
        if (it == idx.end()) {
            idx[key] = (int)pairs.size();
            pairs.push_back(Pair{q.i, q.j, {}});
            it = idx.find(key);
        }
        int k = paths_flavour ? toff[q.path] + (q.k - t.paths[q.path].off3) : q.k;
        pairs[it->second].terms.push_back(Term{k, (int)z, q.c});
    }
    return pairs;
}

static std::string coef(bool paths_flavour, const Term& tm) {
    char buf[64];
    if (paths_flavour) snprintf(buf, sizeof buf, "T(%.17g)", tm.c);
    else snprintf(buf, sizeof buf, "cw[%d]", tm.z);
    return buf;
}

static void emit(FILE* f, int L) {
    PlanTables t;
    build_tables(L, t);
    const int P = (int)t.paths.size();
    std::vector<int> toff(P + 1, 0);
    for (int p = 0; p < P; ++p) toff[p + 1] = toff[p] + 2 * t.paths[p].l3 + 1;
    const int DT = toff[P];
    fprintf(f, "\n// ======================= l_max = %d: P = %d, nnz = %zu, dV = %d, dE = %d, dT = %d\n", L, P, t.nnz.size(), t.dV,
            t.dE, DT);
    fprintf(f, "template <> struct TPGen<%d> {\n", L);
    fprintf(f, "    static constexpr int LMAX = %d, DV = %d, DE = %d, P = %d, NNZ = %zu, DT = %d;\n", L, t.dV, t.dE, P, t.nnz.size(), DT);
    for (int flavour = 0; flavour < 2; ++flavour) {
        const bool pf = flavour == 1;
        std::vector<Pair> pairs = group_pairs(t, pf, toff);
        const int DO = pf ? DT : t.dV;
        const char* sfx = pf ? "_paths" : "";
        // ---------------- forward
        fprintf(f, "    // %s forward: %zu products + %zu FMA\n", pf ? "per-path (un-weighted)" : "folded", pairs.size(), t.nnz.size());
        char cwarg[64] = "";
        if (!pf) snprintf(cwarg, sizeof cwarg, "const T (&cw)[%zu], ", t.nnz.size());
        fprintf(f, "    template <typename T> static __device__ __forceinline__ void fwd%s(%sconst T (&V)[%d], const T (&E)[%d], T (&O)[%d]) {\n",
                sfx, cwarg, t.dV, t.dE, DO);
        std::vector<char> touched(DO, 0);
        for (const Pair& pr : pairs) {
            fprintf(f, "        { const T p = V[%d] * E[%d];", pr.i, pr.j);
            for (const Term& tm : pr.terms) {
                if (!touched[tm.k]) { fprintf(f, " O[%d] = %s * p;", tm.k, coef(pf, tm).c_str()); touched[tm.k] = 1; }
                else fprintf(f, " O[%d] = fma(%s, p, O[%d]);", tm.k, coef(pf, tm).c_str(), tm.k);
            }
            fprintf(f, " }\n");
        }
        for (int k = 0; k < DO; ++k) if (!touched[k]) fprintf(f, "        O[%d] = T(0);\n", k);
        fprintf(f, "    }\n");
        // ---------------- backward: gV assigned, gE accumulated
        fprintf(f, "    // %s VJP: cotangent G -> gV (assigned, if WANT_GV) and gE (accumulated)\n", pf ? "per-path" : "folded");
        fprintf(f, "    template <typename T, bool WANT_GV> static __device__ __forceinline__ void bwd%s(%sconst T (&V)[%d], const T (&E)[%d], const T (&G)[%d], T (&gV)[%d], T (&gE)[%d]) {\n",
                sfx, cwarg, t.dV, t.dE, DO, t.dV, t.dE);
        std::vector<char> tv(t.dV, 0);
        for (const Pair& pr : pairs) {
            fprintf(f, "        { T s = %s * G[%d];", coef(pf, pr.terms[0]).c_str(), pr.terms[0].k);
            for (size_t q = 1; q < pr.terms.size(); ++q) fprintf(f, " s = fma(%s, G[%d], s);", coef(pf, pr.terms[q]).c_str(), pr.terms[q].k);
            fprintf(f, " gE[%d] = fma(s, V[%d], gE[%d]);", pr.j, pr.i, pr.j);
            if (!tv[pr.i]) { fprintf(f, " if (WANT_GV) gV[%d] = s * E[%d];", pr.i, pr.j); tv[pr.i] = 1; }
            else fprintf(f, " if (WANT_GV) gV[%d] = fma(s, E[%d], gV[%d]);", pr.i, pr.j, pr.i);
            fprintf(f, " }\n");
        }
        for (int i = 0; i < t.dV; ++i) if (!tv[i]) fprintf(f, "        if (WANT_GV) gV[%d] = T(0);\n", i);
        fprintf(f, "    }\n");
    }
    // ---------------- path-weight gradient: gw[p] += sum_{(i,j,k) in p} C V[i] E[j] G[k]
    {
        fprintf(f, "    // path-weight gradient, accumulated: gw[p] += sum_{nnz of p} C V E G(out comp)\n");
        fprintf(f, "    template <typename T> static __device__ __forceinline__ void pathw(const T (&V)[%d], const T (&E)[%d], const T (&G)[%d], T (&gw)[%d]) {\n",
                t.dV, t.dE, t.dV, P);
        size_t z = 0;
        for (int p = 0; p < P; ++p) {
            fprintf(f, "        { T a = T(0);\n");
            while (z < t.nnz.size() && t.nnz[z].path == p) {
                // group by (i,j) inside the path (list is sorted (path,i,j,k))
                int i = t.nnz[z].i, j = t.nnz[z].j;
                fprintf(f, "          { T s = T(%.17g) * G[%d];", t.nnz[z].c, t.nnz[z].k);
                ++z;
                while (z < t.nnz.size() && t.nnz[z].path == p && t.nnz[z].i == i && t.nnz[z].j == j) {
                    fprintf(f, " s = fma(T(%.17g), G[%d], s);", t.nnz[z].c, t.nnz[z].k);
                    ++z;
                }
                fprintf(f, " a = fma(V[%d] * E[%d], s, a); }\n", i, j);
            }
            fprintf(f, "          gw[%d] += a; }\n", p);
        }
        fprintf(f, "    }\n");
    }
    // ---------------- small integer tables for the dense mix
    fprintf(f, "    // t-slot offset of each path, and the out block it mixes into\n");
    fprintf(f, "    static __host__ __device__ constexpr int toff(int p) { constexpr int v[%d] = {", P + 1);
    for (int p = 0; p <= P; ++p) fprintf(f, "%d%s", toff[p], p == P ? "" : ",");
    fprintf(f, "}; return v[p]; }\n");
    fprintf(f, "    static __host__ __device__ constexpr int off3(int p) { constexpr int v[%d] = {", P);
    for (int p = 0; p < P; ++p) fprintf(f, "%d%s", t.paths[p].off3, p == P - 1 ? "" : ",");
    fprintf(f, "}; return v[p]; }\n");
    fprintf(f, "    static __host__ __device__ constexpr int d3(int p) { constexpr int v[%d] = {", P);
    for (int p = 0; p < P; ++p) fprintf(f, "%d%s", 2 * t.paths[p].l3 + 1, p == P - 1 ? "" : ",");
    fprintf(f, "}; return v[p]; }\n");
    fprintf(f, "};\n");
}

// Per-path device functions for the dense per-path channel mix: un-weighted t_p = C^p (V (x) E) of ONE path and
// its VJP, with the feature row read through a pointer (shared memory) so that only the path's V block is touched.
static void emit_paths(FILE* f, int L) {
    PlanTables t;
    build_tables(L, t);
    const int P = (int)t.paths.size();
    int toff = 0;
    size_t z = 0;
    for (int p = 0; p < P; ++p) {
        const int d3 = 2 * t.paths[p].l3 + 1, off3 = t.paths[p].off3;
        const int d1 = 2 * t.paths[p].l1 + 1, off1 = t.paths[p].off1;
        fprintf(f, "template <> struct TPPath<%d, %d> {\n    static constexpr int D3 = %d, TOFF = %d, OFF3 = %d, D1 = %d, OFF1 = %d;\n", L, p, d3, toff, off3, d1, off1);
        std::vector<Pair> pairs;
        std::map<std::pair<int, int>, int> idx;
        for (; z < t.nnz.size() && t.nnz[z].path == p; ++z) {
            const NonZero& q = t.nnz[z];
            auto key = std::make_pair(q.i, q.j);
            if (!idx.count(key)) { idx[key] = (int)pairs.size(); pairs.push_back(Pair{q.i, q.j, {}}); }
            pairs[idx[key]].terms.push_back(Term{q.k - off3, (int)z, q.c});
        }
        fprintf(f, "    template <typename T> static __device__ __forceinline__ void fwd(const T* __restrict__ V, const T (&E)[%d], T (&t)[%d]) {\n", t.dE, d3);
        std::vector<char> touched(d3, 0);
        for (const Pair& pr : pairs) {
            fprintf(f, "        { const T p = V[%d] * E[%d];", pr.i, pr.j);
            for (const Term& tm : pr.terms) {
                if (!touched[tm.k]) { fprintf(f, " t[%d] = T(%.17g) * p;", tm.k, tm.c); touched[tm.k] = 1; }
                else fprintf(f, " t[%d] = fma(T(%.17g), p, t[%d]);", tm.k, tm.c, tm.k);
            }
            fprintf(f, " }\n");
        }
        for (int k = 0; k < d3; ++k) if (!touched[k]) fprintf(f, "        t[%d] = T(0);\n", k);
        fprintf(f, "    }\n");
        fprintf(f, "    template <typename T, bool WANT_GV> static __device__ __forceinline__ void bwd(const T* __restrict__ V, const T (&E)[%d], const T (&gt)[%d], T (&gV)[%d], T (&gE)[%d]) {\n",
                t.dE, d3, t.dV, t.dE);
        for (const Pair& pr : pairs) {
            fprintf(f, "        { T s = T(%.17g) * gt[%d];", pr.terms[0].c, pr.terms[0].k);
            for (size_t q = 1; q < pr.terms.size(); ++q) fprintf(f, " s = fma(T(%.17g), gt[%d], s);", pr.terms[q].c, pr.terms[q].k);
            fprintf(f, " gE[%d] = fma(s, V[%d], gE[%d]); if (WANT_GV) gV[%d] = fma(s, E[%d], gV[%d]); }\n", pr.j, pr.i, pr.j, pr.i, pr.j, pr.i);
        }
        fprintf(f, "    }\n");
        // the same VJP with the feature cotangent of the path's OWN input block only (gv[i - OFF1], overwritten): the paths-outer kernels
        fprintf(f, "    template <typename T, bool WANT_GV> static __device__ __forceinline__ void bwd_local(const T* __restrict__ V, const T (&E)[%d], const T (&gt)[%d], T (&gv)[%d], T (&gE)[%d]) {\n",
                t.dE, d3, d1, t.dE);
        fprintf(f, "        if (WANT_GV) {");
        for (int i = 0; i < d1; ++i) fprintf(f, " gv[%d] = T(0);", i);
        fprintf(f, " }\n");
        for (const Pair& pr : pairs) {
            fprintf(f, "        { T s = T(%.17g) * gt[%d];", pr.terms[0].c, pr.terms[0].k);
            for (size_t q = 1; q < pr.terms.size(); ++q) fprintf(f, " s = fma(T(%.17g), gt[%d], s);", pr.terms[q].c, pr.terms[q].k);
            fprintf(f, " gE[%d] = fma(s, V[%d], gE[%d]); if (WANT_GV) gv[%d] = fma(s, E[%d], gv[%d]); }\n", pr.j, pr.i, pr.j, pr.i - off1, pr.j, pr.i - off1);
        }
        fprintf(f, "    }\n};\n");
        toff += d3;
    }
}

int main(int argc, char** argv) {
    if (argc < 2) { fprintf(stderr, "usage: gen_tp <out_dir>\n"); return 2; }
    std::string path = std::string(argv[1]) + "/tp_gen.cuh";
    FILE* f = fopen(path.c_str(), "w");
    if (!f) { perror("fopen"); return 1; }
    fprintf(f, "// GENERATED by gen_tp.cpp from the plan tables of plan.cpp -- do not edit, not committed.\n");
    fprintf(f, "#pragma once\n");
    fprintf(f, "template <int L> struct TPGen;\n");
    for (int L = 1; L <= 3; ++L) emit(f, L);
    fprintf(f, "\n// per-path functions (dense mix)\ntemplate <int L, int PTH> struct TPPath;\n");
    for (int L = 1; L <= 3; ++L) emit_paths(f, L);
    fclose(f);
    return 0;
}
