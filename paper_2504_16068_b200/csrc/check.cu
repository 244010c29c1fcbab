// check.cu -- allegro_check_graph: a debugging aid, not part of the hot path.  The kernels index with row_ptr / items / rev
// UNCHECKED (a check per access would cost the hot loops their bandwidth), and compute-sanitizer is not available on every GPU
// pool, so a wrong index list shows up as a sticky fault or as silently wrong forces.  This call validates the integer inputs of
// a step on the device, before the step: one pass, a few reads per edge, one device -> host copy of the verdict.
//
// The verdict lives in a file-scope device array (no allocation); concurrent calls of allegro_check_graph on one device must be
// ordered by the caller.  The call synchronises `stream`.
#include "common.cuh"
#include "launch.h"

namespace allegro {

// violation classes; g_check[2 * k] = count, g_check[2 * k + 1] = smallest offending index (atom, item or edge)
enum { kBadRowPtr = 0, kBadItem = 1, kBadRev = 2, kBadVec = 3, kNumChecks = 4 };

static __device__ unsigned long long g_check[2 * kNumChecks];

__device__ __forceinline__ void check_fail(int k, long idx) {
    atomicAdd(&g_check[2 * k], 1ull);
    atomicMin(&g_check[2 * k + 1], (unsigned long long)idx);
}

__global__ void check_reset_kernel() {
    if (threadIdx.x < kNumChecks) {
        g_check[2 * threadIdx.x] = 0ull;
        g_check[2 * threadIdx.x + 1] = ~0ull;
    }
}

// row_ptr[0] == 0, row_ptr[i] <= row_ptr[i + 1], row_ptr[N] == E
__global__ void check_row_ptr_kernel(int n_atoms, long n_edges, const int* __restrict__ row_ptr) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n_atoms) return;
    const int a = row_ptr[i];
    if (i == 0 && a != 0) check_fail(kBadRowPtr, 0);
    if (i == n_atoms) {
        if ((long)a != n_edges) check_fail(kBadRowPtr, i);
        return;
    }
    if (a < 0 || row_ptr[i + 1] < a) check_fail(kBadRowPtr, i);
}

// items (c, e0, e1): centres ascending without gaps, every centre's items tile its row in order (an empty row has one empty item).
// Only read when row_ptr passed its own test on the centre concerned: c is range-checked first.
__global__ void check_items_kernel(int n_atoms, long n_items, const int* __restrict__ row_ptr, const int* __restrict__ items) {
    const long it = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (it >= n_items) return;
    const int c = items[3 * it], e0 = items[3 * it + 1], e1 = items[3 * it + 2];
    if (c < 0 || c >= n_atoms) { check_fail(kBadItem, it); return; }
    const int r0 = row_ptr[c], r1 = row_ptr[c + 1];
    bool ok = r0 <= e0 && e0 <= e1 && e1 <= r1;
    if (it == 0) {
        ok = ok && c == 0 && e0 == r0;
    } else {
        const int pc = items[3 * (it - 1)], pe1 = items[3 * (it - 1) + 2];
        if (pc == c) ok = ok && e0 == pe1 && e1 > e0;     // a continuation item is never empty
        else ok = ok && c == pc + 1 && e0 == r0;
    }
    if (it == n_items - 1) {
        ok = ok && c == n_atoms - 1 && e1 == r1;
    } else if (items[3 * (it + 1)] != c) {
        ok = ok && e1 == r1;
    }
    if (!ok) check_fail(kBadItem, it);
}

// rev: an involution of [0, E) without fixed points; with col (optional, the far end of every edge) the reverse of (i -> j) is (j -> i)
__global__ void check_rev_kernel(int n_atoms, long n_edges, const int* __restrict__ row_ptr, const int* __restrict__ rev,
                                 const int* __restrict__ col) {
    const int c = blockIdx.x;
    for (long e = row_ptr[c] + threadIdx.x; e < row_ptr[c + 1]; e += blockDim.x) {
        const int r = rev[e];
        bool ok = r >= 0 && (long)r < n_edges && (long)r != e;
        if (ok) ok = (long)rev[r] == e;
        if (ok && col != nullptr) {
            const int j = col[e];
            ok = j >= 0 && j < n_atoms;
            if (ok) ok = (long)r >= row_ptr[j] && (long)r < row_ptr[j + 1] && col[r] == c;
        }
        if (!ok) check_fail(kBadRev, e);
    }
}

// edge vectors: finite and of non-zero length (the kernels divide by |r_e|)
template <typename T>
__global__ void check_rvec_kernel(long n_edges, const T* __restrict__ rvec) {
    const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_edges) return;
    const T x = rvec[3 * e], y = rvec[3 * e + 1], z = rvec[3 * e + 2];
    const T r2 = x * x + y * y + z * z;
    if (!(r2 > T(0)) || !isfinite(r2)) check_fail(kBadVec, e);
}

}  // namespace allegro

using namespace allegro;

extern "C" {

allegro_status_t allegro_check_graph(int n_atoms, long n_edges, const int32_t* row_ptr, const int32_t* items, long n_items, const int32_t* rev,
                                     const int32_t* col, const void* rvec, allegro_dtype_t dtype, long* n_bad, void* stream) {
    ALLEGRO_CHECK_ARG(n_atoms >= 0 && n_edges >= 0 && n_edges < 2147483647L, "bad n_atoms / n_edges");
    ALLEGRO_CHECK_ARG(row_ptr != nullptr, "row_ptr is NULL");
    ALLEGRO_CHECK_ARG(items == nullptr || n_items >= n_atoms, "n_items < n_atoms");
    ALLEGRO_CHECK_ARG(col == nullptr || rev != nullptr, "col without rev");
    ALLEGRO_CHECK_ARG(dtype == ALLEGRO_F32 || dtype == ALLEGRO_F64, "bad dtype");
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long h[2 * kNumChecks];
    check_reset_kernel<<<1, 32, 0, st>>>();
    ALLEGRO_LAUNCHED();
    check_row_ptr_kernel<<<(unsigned)(n_atoms / 256 + 1), 256, 0, st>>>(n_atoms, n_edges, row_ptr);
    ALLEGRO_LAUNCHED();
    ALLEGRO_CUDA(cudaMemcpyFromSymbolAsync(h, g_check, sizeof(h), 0, cudaMemcpyDeviceToHost, st));
    ALLEGRO_CUDA(cudaStreamSynchronize(st));
    // the other lists are indexed THROUGH row_ptr: they are only looked at once row_ptr itself is sound
    if (h[2 * kBadRowPtr] == 0) {
        if (items != nullptr && n_items > 0) {
            check_items_kernel<<<(unsigned)((n_items + 255) / 256), 256, 0, st>>>(n_atoms, n_items, row_ptr, items);
            ALLEGRO_LAUNCHED();
        }
        if (rev != nullptr && n_atoms > 0) {
            check_rev_kernel<<<(unsigned)n_atoms, 128, 0, st>>>(n_atoms, n_edges, row_ptr, rev, col);
            ALLEGRO_LAUNCHED();
        }
        if (rvec != nullptr && n_edges > 0) {
            if (dtype == ALLEGRO_F32) check_rvec_kernel<float><<<(unsigned)((n_edges + 255) / 256), 256, 0, st>>>(n_edges, (const float*)rvec);
            else check_rvec_kernel<double><<<(unsigned)((n_edges + 255) / 256), 256, 0, st>>>(n_edges, (const double*)rvec);
            ALLEGRO_LAUNCHED();
        }
        ALLEGRO_CUDA(cudaMemcpyFromSymbolAsync(h, g_check, sizeof(h), 0, cudaMemcpyDeviceToHost, st));
        ALLEGRO_CUDA(cudaStreamSynchronize(st));
    }
    long total = 0;
    for (int k = 0; k < kNumChecks; ++k) total += (long)h[2 * k];
    if (n_bad != nullptr) *n_bad = total;
    if (total == 0) return ALLEGRO_OK;
    static const char* const what[kNumChecks] = {"row_ptr (first bad atom index", "items (first bad item", "rev / col (first bad edge", "rvec (first bad edge"};
    for (int k = 0; k < kNumChecks; ++k)
        if (h[2 * k] != 0) {
            set_error("allegro_check_graph: %ld violation(s) in all; %llu in %s %llu)", total, h[2 * k], what[k], h[2 * k + 1]);
            break;
        }
    return ALLEGRO_EINVAL;
}

}  // extern "C"
