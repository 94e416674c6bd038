// omni_noalloc.cuh -- the source-vector step (a1 + a2: S of Eq. 9; ||S||^2) as ONE kernel that needs no
// workspace from an allocator: for callers that cannot call cudaMalloc (stream capture, serving loops, harnesses that
// forbid it).  A variant of source_kernel (omni_kernels.cuh): same arithmetic per cell, in the same order, but
//   * validity (Eq. 13 :176) of the cell and of its 2 * naxes neighbours is evaluated on the fly from mask / NaN instead
//     of being read from the link bytes the solver's set-up kernels build in an allocated workspace, and S goes straight
//     to the caller's (unpadded) array;
//   * the only scratch left is the deterministic grid reduction of ||S||^2 -- one fp64 partial per CTA, a ticket, the
//     last CTA adding the partials in slot order -- and it lives in a fixed static __device__ array owned by the library
//     (omni_api.cu: g_noalloc_scratch), whose size bounds the problem: one CTA per NOALLOC_CELLS_PER_CTA cells, one slot
//     per CTA.
#pragma once
#include "omni_kernels.cuh"

namespace omni {

constexpr int NOALLOC_SCRATCH_BYTES = 256 * 1024;                      // per GPU that loads the library, until exit
constexpr int NOALLOC_HEADER_DOUBLES = 8;                              // [0]: ticket (as unsigned), [1]: ||S||^2 of the last call
constexpr int NOALLOC_SLOTS = NOALLOC_SCRATCH_BYTES / 8 - NOALLOC_HEADER_DOUBLES;      // 32 760 CTA partials
constexpr int NOALLOC_THREADS = 256, NOALLOC_ITEMS = 16;
constexpr int NOALLOC_CELLS_PER_CTA = NOALLOC_THREADS * NOALLOC_ITEMS;                 // 4096
constexpr long long NOALLOC_MAX_CELLS = (long long)NOALLOC_SLOTS * NOALLOC_CELLS_PER_CTA;   // 134 184 960 (500^3 fits)

template <typename T>
__global__ void __launch_bounds__(NOALLOC_THREADS)
source_noalloc_kernel(int nx, int ny, int nz, int naxes, const T* __restrict__ gx, const T* __restrict__ gy,
                      const T* __restrict__ gz, const uint8_t* __restrict__ mask, T hs0, T hs1, T hs2,
                      T* __restrict__ S, double* __restrict__ scratch, double* __restrict__ norm_out)
{
    __shared__ double red[NOALLOC_THREADS / 32];
    __shared__ int is_last;
    const long long n = (long long)nx * ny * nz;
    const long long sy = nx, sz = (long long)nx * ny;
    auto valid = [&](long long q) {
        if (mask != nullptr && mask[q] == 0) return false;
        if (isnan(gx[q]) || isnan(gy[q])) return false;
        return !(naxes == 3 && isnan(gz[q]));
    };
    double sq = 0.0;
    const long long base = (long long)blockIdx.x * NOALLOC_CELLS_PER_CTA + threadIdx.x;
#pragma unroll 4
    for (int it = 0; it < NOALLOC_ITEMS; ++it) {
        const long long u = base + (long long)it * NOALLOC_THREADS;
        if (u >= n) break;
        // n <= NOALLOC_MAX_CELLS < 2^31: 32-bit index arithmetic
        const unsigned int u32 = (unsigned int)u, row = u32 / (unsigned int)nx;
        const int i = (int)(u32 - row * (unsigned int)nx);
        const int k = (int)(row / (unsigned int)ny), j = (int)(row - (unsigned int)k * (unsigned int)ny);
        T s = T(0);
        if (valid(u)) {
            // same terms, same order as source_kernel: E W N S (F B); faces to missing cells contribute nothing (Eq. 49 :656)
            const T cx = gx[u], cy = gy[u];
            if (i + 1 < nx && valid(u + 1)) s -= hs0 * (gx[u + 1] + cx);
            if (i > 0 && valid(u - 1)) s += hs0 * (gx[u - 1] + cx);
            if (j + 1 < ny && valid(u + sy)) s -= hs1 * (gy[u + sy] + cy);
            if (j > 0 && valid(u - sy)) s += hs1 * (gy[u - sy] + cy);
            if (naxes == 3) {
                const bool f = (k + 1 < nz) && valid(u + sz), b = (k > 0) && valid(u - sz);
                if (f || b) {
                    const T cz = gz[u];
                    if (f) s -= hs2 * (gz[u + sz] + cz);
                    if (b) s += hs2 * (gz[u - sz] + cz);
                }
            }
        }
        S[u] = s;
        sq += (double)s * (double)s;
    }
    // deterministic reduction: thread -> warp -> CTA slot; the last CTA (ticket) adds the slots in slot order
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
    double* partial = scratch + NOALLOC_HEADER_DOUBLES;
    sq = warp_sum(sq);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sq;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < NOALLOC_THREADS / 32; ++w) t += red[w];
        partial[blockIdx.x] = t;
        __threadfence();
        is_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        double t = 0.0;
        for (unsigned int b = threadIdx.x; b < gridDim.x; b += NOALLOC_THREADS) t += __ldcg(&partial[b]);
        t = warp_sum(t);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = t;
        __syncthreads();
        if (threadIdx.x == 0) {
            double n2 = 0.0;
            for (int w = 0; w < NOALLOC_THREADS / 32; ++w) n2 += red[w];
            *ticket = 0u;
            scratch[1] = n2;
            if (norm_out != nullptr) *norm_out = sqrt(n2);
        }
    }
}

}  // namespace omni
