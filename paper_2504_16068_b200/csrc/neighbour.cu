// neighbour.cu -- cell-list neighbour builder on the GPU (the MD plugin keeps the neighbour list on the
// device): positions -> the CSR edge list the hot path takes (reading A7: directed edges, both directions, CSR by centre, neighbour
// index ascending inside a row, r_e = x_j - x_i + shift, 0 < |r_e| < r_c strict, minimum image) plus the reverse-edge permutation
// (A17).  Integer results are bit-exact against the host builder of the workloads: the keep / drop decision is taken in double
// with the same operation order (explicit round-to-nearest intrinsics: no FMA contraction), for the pair (min(i,j), max(i,j)) as
// the host does, and the edge vector of the second direction is the exact negation of the first.
//
//   count : cell index per atom -> histogram -> scan -> atoms scattered into cell order -> thread per atom counts its neighbours in the
//           27 surrounding cells (all atoms when a box direction holds fewer than three cells) -> scan -> row_ptr; E returned to the host
//   fill  : thread per atom writes its neighbours, sorts its row by index (rows are ~100 long), writes rvec; thread per edge finds
//           the reverse edge by binary search in the neighbour's row
// Integer atomics only order atoms inside a cell, and rows are sorted afterwards: the output does not depend on scheduling.
#include "common.cuh"
#include "launch.h"

namespace allegro {

struct NbrGrid {
    double box, rc, cell[3], lo[3];
    int nc[3];
    int periodic, brute;
    const int* species;        // nullable: per-edge-type cutoffs (reading A27)
    const double* rc_table;    // [n_species][n_species]
    int n_species;
};

__device__ __forceinline__ int nbr_cell_of(const NbrGrid& g, const double* __restrict__ p, int d) {
    int c = (int)floor((p[d] - g.lo[d]) / g.cell[d]);
    return c < 0 ? 0 : (c >= g.nc[d] ? g.nc[d] - 1 : c);
}

__device__ __forceinline__ double nbr_rc(const NbrGrid& g, int a, int b) {
    return g.species ? g.rc_table[g.species[a] * g.n_species + g.species[b]] : g.rc;
}

// edge vector of the ordered pair (a < b) as the host computes it; returns true when 0 < |d| < rc (the pair's own cutoff)
__device__ __forceinline__ bool nbr_pair(const NbrGrid& g, const double* __restrict__ pos, int a, int b, double (&d)[3]) {
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        double x = __dsub_rn(pos[3 * (size_t)b + k], pos[3 * (size_t)a + k]);
        if (g.periodic) x = __dsub_rn(x, __dmul_rn(g.box, rint(__ddiv_rn(x, g.box))));
        d[k] = x;
    }
    const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
    const double r = __dsqrt_rn(r2);
    return r > 0.0 && r < nbr_rc(g, a, b);
}

__global__ void nbr_cell_kernel(NbrGrid g, int N, const double* __restrict__ pos, int* __restrict__ cell_id, int* __restrict__ cell_cnt) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int c = (nbr_cell_of(g, pos + 3 * (size_t)i, 2) * g.nc[1] + nbr_cell_of(g, pos + 3 * (size_t)i, 1)) * g.nc[0] + nbr_cell_of(g, pos + 3 * (size_t)i, 0);
    cell_id[i] = c;
    atomicAdd(&cell_cnt[c], 1);
}

// exclusive scan of in[0..n) into out[0..n], out[n] = total; one CTA walks the array in chunks of its size
__global__ void __launch_bounds__(1024) nbr_scan_kernel(int n, const int* __restrict__ in, int* __restrict__ out) {
    __shared__ int sh[1024];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        const int i = base + threadIdx.x;
        const int v = i < n ? in[i] : 0;
        sh[threadIdx.x] = v;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) {
            const int t = (int)threadIdx.x >= o ? sh[threadIdx.x - o] : 0;
            __syncthreads();
            sh[threadIdx.x] += t;
            __syncthreads();
        }
        if (i < n) out[i] = carry + sh[threadIdx.x] - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry += sh[1023];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[n] = carry;
}

__global__ void nbr_scatter_kernel(int N, const int* __restrict__ cell_id, const int* __restrict__ cell_start, int* __restrict__ cursor,
                                   int* __restrict__ sorted) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int c = cell_id[i];
    sorted[cell_start[c] + atomicAdd(&cursor[c], 1)] = i;
}

// visit every candidate neighbour j != i of atom i exactly once
template <typename F>
__device__ __forceinline__ void nbr_visit(const NbrGrid& g, int N, int i, const double* __restrict__ pos, const int* __restrict__ cell_start,
                                          const int* __restrict__ sorted, F&& f) {
    if (g.brute) {
        for (int j = 0; j < N; ++j) if (j != i) f(j);
        return;
    }
    int c[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) c[d] = nbr_cell_of(g, pos + 3 * (size_t)i, d);
    for (int dz = -1; dz <= 1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
            for (int dx = -1; dx <= 1; ++dx) {
                int x = c[0] + dx, y = c[1] + dy, z = c[2] + dz;
                if (g.periodic) {
                    x = (x + g.nc[0]) % g.nc[0]; y = (y + g.nc[1]) % g.nc[1]; z = (z + g.nc[2]) % g.nc[2];
                } else if (x < 0 || y < 0 || z < 0 || x >= g.nc[0] || y >= g.nc[1] || z >= g.nc[2]) {
                    continue;
                }
                const int cc = (z * g.nc[1] + y) * g.nc[0] + x;
                for (int s = cell_start[cc]; s < cell_start[cc + 1]; ++s) {
                    const int j = sorted[s];
                    if (j != i) f(j);
                }
            }
}

__global__ void nbr_count_kernel(NbrGrid g, int N, const double* __restrict__ pos, const int* __restrict__ mol_id, const int* __restrict__ cell_start,
                                 const int* __restrict__ sorted, int* __restrict__ deg) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int cnt = 0;
    nbr_visit(g, N, i, pos, cell_start, sorted, [&](int j) {
        if (mol_id && mol_id[i] != mol_id[j]) return;
        double d[3];
        if (nbr_pair(g, pos, i < j ? i : j, i < j ? j : i, d)) ++cnt;
    });
    deg[i] = cnt;
}

template <typename T>
__global__ void nbr_fill_kernel(NbrGrid g, int N, const double* __restrict__ pos, const int* __restrict__ mol_id, const int* __restrict__ cell_start,
                                const int* __restrict__ sorted, const int* __restrict__ row_ptr, int* __restrict__ col, T* __restrict__ rvec,
                                T* __restrict__ rc_edge) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int r0 = row_ptr[i], r1 = row_ptr[i + 1];
    int w = r0;
    nbr_visit(g, N, i, pos, cell_start, sorted, [&](int j) {
        if (mol_id && mol_id[i] != mol_id[j]) return;
        double d[3];
        if (nbr_pair(g, pos, i < j ? i : j, i < j ? j : i, d) && w < r1) col[w++] = j;
    });
    for (int a = r0 + 1; a < r1; ++a) {        // insertion sort of the row by neighbour index
        const int v = col[a];
        int b = a - 1;
        while (b >= r0 && col[b] > v) { col[b + 1] = col[b]; --b; }
        col[b + 1] = v;
    }
    for (int e = r0; e < r1; ++e) {
        const int j = col[e];
        double d[3];
        nbr_pair(g, pos, i < j ? i : j, i < j ? j : i, d);
        const double sgn = i < j ? 1.0 : -1.0;
#pragma unroll
        for (int k = 0; k < 3; ++k) rvec[3 * (size_t)e + k] = (T)(sgn * d[k]);
        if (rc_edge) rc_edge[e] = (T)nbr_rc(g, i, j);
    }
}

__global__ void nbr_rev_kernel(int N, const int* __restrict__ row_ptr, const int* __restrict__ col, int* __restrict__ rev) {
    const int i = blockIdx.x;      // one CTA per centre
    for (int e = row_ptr[i] + threadIdx.x; e < row_ptr[i + 1]; e += blockDim.x) {
        const int j = col[e];
        int lo = row_ptr[j], hi = row_ptr[j + 1] - 1, found = -1;
        while (lo <= hi) {
            const int mid = (lo + hi) >> 1, v = col[mid];
            if (v == i) { found = mid; break; }
            if (v < i) lo = mid + 1; else hi = mid - 1;
        }
        rev[e] = found;
    }
}

struct NbrWs {
    int *cell_id, *sorted, *deg, *cell_cnt, *cell_start, *cursor;
    size_t total;
};
static NbrWs nbr_layout(void* ws, int N, long ncells) {
    NbrWs L{};
    size_t off = 0;
    auto take = [&](size_t count) { int* p = ws ? (int*)((unsigned char*)ws + off) : nullptr; off += align_up(count * 4, 256); return p; };
    L.cell_id = take(N); L.sorted = take(N); L.deg = take(N); L.cell_cnt = take(ncells + 1); L.cell_start = take(ncells + 1); L.cursor = take(ncells + 1);
    L.total = off;
    return L;
}
static const long kNbrMaxCells = 1L << 21;

// grid geometry from the box (periodic) or from a caller-given bounding box (open)
static allegro_status_t nbr_grid(int N, double box, double rc, const double* lo, const double* hi, const int32_t* species, int n_species,
                                 const double* rc_table, NbrGrid& g) {
    g.box = box; g.rc = rc; g.periodic = box > 0.0 ? 1 : 0; g.brute = 0;
    g.species = (species && rc_table && n_species > 0) ? species : nullptr;
    g.rc_table = rc_table; g.n_species = n_species;
    long cells = 1;
    for (int d = 0; d < 3; ++d) {
        const double ext = g.periodic ? box : (hi[d] - lo[d]);
        g.lo[d] = g.periodic ? 0.0 : lo[d];
        long nc = (long)floor(ext / rc);
        if (nc < 1) nc = 1;
        while (cells * nc > kNbrMaxCells && nc > 1) nc = (nc + 1) / 2;      // coarser cells are still correct (cell edge >= rc)
        g.nc[d] = (int)nc;
        g.cell[d] = ext / (double)nc;
        if (g.cell[d] <= 0.0) g.cell[d] = 1.0;
        cells *= nc;
        if (g.periodic && nc < 3) g.brute = 1;      // the 27 surrounding cells would not be distinct
    }
    if (g.periodic && !(rc < box / 2)) {
        set_error("neighbour list: minimum image needs r_cut < box / 2 (r_cut = %g, box = %g)", rc, box);
        return ALLEGRO_EINVAL;
    }
    (void)N;
    return ALLEGRO_OK;
}

}  // namespace allegro

using namespace allegro;

extern "C" {

size_t allegro_neighbour_workspace(int n_atoms) {
    if (n_atoms < 0) return 0;
    return nbr_layout(nullptr, n_atoms, kNbrMaxCells).total;
}

allegro_status_t allegro_neighbour_count(int n_atoms, const double* pos, double box, const double* bbox_lo_host, const double* bbox_hi_host, double r_cut,
                                         const int32_t* mol_id, const int32_t* species, int n_species, const double* rc_table, int32_t* row_ptr,
                                         void* workspace, size_t workspace_bytes, void* stream, long* n_edges_host) {
    ALLEGRO_CHECK_ARG(n_atoms >= 0 && r_cut > 0 && row_ptr != nullptr && n_edges_host != nullptr, "bad argument");
    ALLEGRO_CHECK_ARG(pos != nullptr || n_atoms == 0, "pos is NULL");
    ALLEGRO_CHECK_ARG(box > 0.0 || (bbox_lo_host && bbox_hi_host), "open systems need a bounding box");
    cudaStream_t st = (cudaStream_t)stream;
    NbrGrid g;
    allegro_status_t s = nbr_grid(n_atoms, box, r_cut, bbox_lo_host, bbox_hi_host, species, n_species, rc_table, g);
    if (s != ALLEGRO_OK) return s;
    const long ncells = (long)g.nc[0] * g.nc[1] * g.nc[2];
    const NbrWs L = nbr_layout(workspace, n_atoms, kNbrMaxCells);
    if (workspace == nullptr || workspace_bytes < L.total) {
        set_error("allegro_neighbour_count: workspace too small (%zu < %zu bytes)", workspace_bytes, L.total);
        return ALLEGRO_ENOMEM;
    }
    *n_edges_host = 0;
    if (n_atoms == 0) { ALLEGRO_CUDA(cudaMemsetAsync(row_ptr, 0, 4, st)); return ALLEGRO_OK; }
    const unsigned nb = (unsigned)((n_atoms + 127) / 128);
    ALLEGRO_CUDA(cudaMemsetAsync(L.cell_cnt, 0, (size_t)(ncells + 1) * 4, st));
    ALLEGRO_CUDA(cudaMemsetAsync(L.cursor, 0, (size_t)(ncells + 1) * 4, st));
    nbr_cell_kernel<<<nb, 128, 0, st>>>(g, n_atoms, pos, L.cell_id, L.cell_cnt);
    ALLEGRO_LAUNCHED();
    nbr_scan_kernel<<<1, 1024, 0, st>>>((int)ncells, L.cell_cnt, L.cell_start);
    ALLEGRO_LAUNCHED();
    nbr_scatter_kernel<<<nb, 128, 0, st>>>(n_atoms, L.cell_id, L.cell_start, L.cursor, L.sorted);
    ALLEGRO_LAUNCHED();
    nbr_count_kernel<<<nb, 128, 0, st>>>(g, n_atoms, pos, mol_id, L.cell_start, L.sorted, L.deg);
    ALLEGRO_LAUNCHED();
    nbr_scan_kernel<<<1, 1024, 0, st>>>(n_atoms, L.deg, row_ptr);
    ALLEGRO_LAUNCHED();
    int32_t total = 0;
    ALLEGRO_CUDA(cudaMemcpyAsync(&total, row_ptr + n_atoms, 4, cudaMemcpyDeviceToHost, st));
    ALLEGRO_CUDA(cudaStreamSynchronize(st));
    *n_edges_host = total;
    return ALLEGRO_OK;
}

allegro_status_t allegro_neighbour_fill(int n_atoms, const double* pos, double box, const double* bbox_lo_host, const double* bbox_hi_host, double r_cut,
                                        const int32_t* mol_id, const int32_t* species, int n_species, const double* rc_table, const int32_t* row_ptr,
                                        long n_edges, int32_t* col, int32_t* rev, void* rvec, void* rc_edge, allegro_dtype_t dtype, void* workspace,
                                        size_t workspace_bytes, void* stream) {
    ALLEGRO_CHECK_ARG(n_atoms >= 0 && r_cut > 0 && row_ptr != nullptr && n_edges >= 0, "bad argument");
    ALLEGRO_CHECK_ARG((col && rev && rvec) || n_edges == 0, "NULL output");
    ALLEGRO_CHECK_ARG(box > 0.0 || (bbox_lo_host && bbox_hi_host), "open systems need a bounding box");
    ALLEGRO_CHECK_ARG(dtype == ALLEGRO_F32 || dtype == ALLEGRO_F64, "bad dtype");
    cudaStream_t st = (cudaStream_t)stream;
    NbrGrid g;
    allegro_status_t s = nbr_grid(n_atoms, box, r_cut, bbox_lo_host, bbox_hi_host, species, n_species, rc_table, g);
    if (s != ALLEGRO_OK) return s;
    const NbrWs L = nbr_layout(workspace, n_atoms, kNbrMaxCells);
    if (workspace == nullptr || workspace_bytes < L.total) {
        set_error("allegro_neighbour_fill: workspace too small (%zu < %zu bytes)", workspace_bytes, L.total);
        return ALLEGRO_ENOMEM;
    }
    if (n_atoms == 0 || n_edges == 0) return ALLEGRO_OK;
    const unsigned nb = (unsigned)((n_atoms + 127) / 128);
    if (dtype == ALLEGRO_F32) nbr_fill_kernel<float><<<nb, 128, 0, st>>>(g, n_atoms, pos, mol_id, L.cell_start, L.sorted, row_ptr, col, (float*)rvec, (float*)rc_edge);
    else nbr_fill_kernel<double><<<nb, 128, 0, st>>>(g, n_atoms, pos, mol_id, L.cell_start, L.sorted, row_ptr, col, (double*)rvec, (double*)rc_edge);
    ALLEGRO_LAUNCHED();
    nbr_rev_kernel<<<(unsigned)n_atoms, 64, 0, st>>>(n_atoms, row_ptr, col, rev);
    ALLEGRO_LAUNCHED();
    return ALLEGRO_OK;
}

}  // extern "C"
