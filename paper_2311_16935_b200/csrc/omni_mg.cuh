// omni_mg.cuh -- geometric-multigrid V-cycle used as the preconditioner of CG on the fixed-point system L P = S
// (omni_solve_pcg_*, SURVEY.md 8(f) NEXT-2 ii; reading R-P1 of DESIGN.md).  Not the paper's iteration: the paper names
// only "CG"; this accelerates the separately named fixed-point solve of omni_solve_direct_*.
//
//   levels    level 0 = the grid (padded layout of the solver, its link bytes); level l+1 halves (ceil) every axis of
//             level l with >= 8 cells; a coarse cell is valid iff one of its children is
//   operator  (L_l x)_C = sum_d v_l(C+d) w_l[a] (x_C - x_{C+d}); w_0[a] = t_a = F_a / A_tot (Eq. 10 :109),
//             w_{l+1}[a] = w_l[a] 2^m (1/4 if axis a was halved else 1), m = number of halved axes
//   transfer  restriction = sum over the children, prolongation = the parent's value (transposes of each other)
//   smoother  damped Jacobi x <- x + omega D^-1 (b - L x), omega = 0.8; 2 sweeps before and after the coarse-grid
//             correction (the first from x = 0), 8 on the coarsest level
// One thread per cell (per coarse cell in the restriction, which gathers its children in a fixed order: deterministic).
// Bandwidth-bound elementwise / 7-point kernels on plain coalesced loads; neighbours come from L1 / L2.
#pragma once
#include "omni_kernels.cuh"

namespace omni {

constexpr int MG_MAX_LEVELS = 16;
constexpr int MG_MIN_COARSEN = 8;
constexpr int MG_NU = 2, MG_NU_COARSEST = 8;
constexpr double MG_OMEGA = 0.8;

template <typename T>
struct MgLevel {
    int nx, ny, nz, px;          // logical size and row pitch in cells (level 0: the solver's padded pitch)
    long long pplane, n;         // px * ny, px * ny * nz
    int hx, hy, hz;              // 1: this axis is halved to make the next level
    T w[3];                      // link weights of this level
    const uint8_t* link;         // bits 0..5 = v(C+d) for d = E W N S F B, bit 6 = cell valid
    T *x, *xt, *b;               // iterate, second Jacobi buffer, right-hand side
};

template <typename T>
__device__ __forceinline__ bool mg_cell(const MgLevel<T>& L, long long c, int& i, int& j, int& k)
{
    if (c >= L.n) return false;
    i = (int)(c % L.px);
    const long long row = c / L.px;
    j = (int)(row % L.ny);
    k = (int)(row / L.ny);
    return i < L.nx;
}

// (D, L x) at cell c from its link byte
template <typename T>
__device__ __forceinline__ void mg_stencil(const MgLevel<T>& L, const T* __restrict__ x, long long c, uint32_t l, T& D, T& Lx)
{
    const T xc = x[c];
    D = T(0); Lx = T(0);
    if (l & 1u) { D += L.w[0]; Lx += L.w[0] * (xc - x[c + 1]); }
    if (l & 2u) { D += L.w[0]; Lx += L.w[0] * (xc - x[c - 1]); }
    if (l & 4u) { D += L.w[1]; Lx += L.w[1] * (xc - x[c + L.px]); }
    if (l & 8u) { D += L.w[1]; Lx += L.w[1] * (xc - x[c - L.px]); }
    if (l & 16u) { D += L.w[2]; Lx += L.w[2] * (xc - x[c + L.pplane]); }
    if (l & 32u) { D += L.w[2]; Lx += L.w[2] * (xc - x[c - L.pplane]); }
}

template <typename T>
__device__ __forceinline__ T mg_diag(const MgLevel<T>& L, uint32_t l)
{
    T D = T(0);
    if (l & 1u) D += L.w[0];
    if (l & 2u) D += L.w[0];
    if (l & 4u) D += L.w[1];
    if (l & 8u) D += L.w[1];
    if (l & 16u) D += L.w[2];
    if (l & 32u) D += L.w[2];
    return D;
}

// FIRST: xout = omega D^-1 b (a sweep from x = 0); else xout = xin + omega D^-1 (b - L xin).  0 at missing cells.
template <typename T, bool FIRST>
__global__ void __launch_bounds__(256)
mg_jacobi_kernel(const MgLevel<T> L, const T* __restrict__ xin, T* __restrict__ xout)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int i, j, k;
    if (c >= L.n) return;
    if (!mg_cell(L, c, i, j, k)) { xout[c] = T(0); return; }
    const uint32_t l = L.link[c];
    T v = T(0);
    if (l & LINK_VALID) {
        if (FIRST) {
            const T D = mg_diag(L, l);
            if (D > T(0)) v = (T)MG_OMEGA * (L.b[c] / D);
        } else {
            T D, Lx;
            mg_stencil(L, xin, c, l, D, Lx);
            v = xin[c];
            if (D > T(0)) v += (T)MG_OMEGA * ((L.b[c] - Lx) / D);
        }
    }
    xout[c] = v;
}

// coarse right-hand side: b_c[I] = sum over the valid children C of I of (b - L x)_C, children in a fixed order
template <typename T>
__global__ void __launch_bounds__(256)
mg_residual_restrict_kernel(const MgLevel<T> F, const MgLevel<T> C, const T* __restrict__ x)
{
    const long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int ci, cj, ck;
    if (I >= C.n) return;
    if (!mg_cell(C, I, ci, cj, ck)) { C.b[I] = T(0); return; }
    T s = T(0);
    for (int dk = 0; dk <= F.hz; ++dk)
        for (int dj = 0; dj <= F.hy; ++dj)
            for (int di = 0; di <= F.hx; ++di) {
                const int i = (F.hx ? 2 * ci : ci) + di, j = (F.hy ? 2 * cj : cj) + dj, k = (F.hz ? 2 * ck : ck) + dk;
                if (i >= F.nx || j >= F.ny || k >= F.nz) continue;
                const long long c = i + (long long)F.px * (j + (long long)F.ny * k);
                const uint32_t l = F.link[c];
                if (!(l & LINK_VALID)) continue;
                T D, Lx;
                mg_stencil(F, x, c, l, D, Lx);
                s += F.b[c] - Lx;
            }
    C.b[I] = s;
}

// x += prolong(e): every valid fine cell receives its parent's value
template <typename T>
__global__ void __launch_bounds__(256)
mg_prolong_add_kernel(const MgLevel<T> F, const MgLevel<T> C, T* __restrict__ x, const T* __restrict__ e)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int i, j, k;
    if (!mg_cell(F, c, i, j, k)) return;
    if (!(F.link[c] & LINK_VALID)) return;
    const long long I = (F.hx ? i >> 1 : i) + (long long)C.px * ((F.hy ? j >> 1 : j) + (long long)C.ny * (F.hz ? k >> 1 : k));
    x[c] += e[I];
}

// validity of the next level: a coarse cell is valid iff one of its children is
template <typename T>
__global__ void __launch_bounds__(256)
mg_coarse_valid_kernel(const MgLevel<T> F, const MgLevel<T> C, uint8_t* __restrict__ vc)
{
    const long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int ci, cj, ck;
    if (I >= C.n) return;
    uint8_t any = 0;
    if (mg_cell(C, I, ci, cj, ck))
        for (int dk = 0; dk <= F.hz; ++dk)
            for (int dj = 0; dj <= F.hy; ++dj)
                for (int di = 0; di <= F.hx; ++di) {
                    const int i = (F.hx ? 2 * ci : ci) + di, j = (F.hy ? 2 * cj : cj) + dj, k = (F.hz ? 2 * ck : ck) + dk;
                    if (i >= F.nx || j >= F.ny || k >= F.nz) continue;
                    if (F.link[i + (long long)F.px * (j + (long long)F.ny * k)] & LINK_VALID) any = 1;
                }
    vc[I] = any;
}

// link bytes of a level from its validity bytes (naxes = 2: no F / B links)
template <typename T>
__global__ void __launch_bounds__(256)
mg_link_kernel(const MgLevel<T> C, const uint8_t* __restrict__ vc, uint8_t* __restrict__ link, int naxes)
{
    const long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int i, j, k;
    if (I >= C.n) return;
    uint32_t l = 0;
    if (mg_cell(C, I, i, j, k) && vc[I]) {
        l = LINK_VALID;
        if (i + 1 < C.nx && vc[I + 1]) l |= 1u;
        if (i > 0 && vc[I - 1]) l |= 2u;
        if (j + 1 < C.ny && vc[I + C.px]) l |= 4u;
        if (j > 0 && vc[I - C.px]) l |= 8u;
        if (naxes == 3) {
            if (k + 1 < C.nz && vc[I + C.pplane]) l |= 16u;
            if (k > 0 && vc[I - C.pplane]) l |= 32u;
        }
    }
    link[I] = (uint8_t)l;
}

// rho = r . z of the preconditioned recurrence (deterministic: per-block partials, last block adds them in order);
// then beta = rho / rho_old (0 at the first iteration of an inner solve), rho_old <- rho.  r and z are 0 at missing cells.
template <typename T>
__global__ void __launch_bounds__(256)
mg_dot_kernel(long long n, const T* __restrict__ r, const T* __restrict__ z, Scalars* sc, double* partial, CondHandles cond)
{
    __shared__ double red[8];
    __shared__ int is_last;
    double s = 0.0;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += (long long)gridDim.x * blockDim.x)
        s += (double)r[c] * (double)z[c];
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += red[w];
        partial[blockIdx.x] = t;
        __threadfence();
        is_last = (atomicAdd(&sc->ticket[3], 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        double t = 0.0;
        for (unsigned int b = threadIdx.x; b < gridDim.x; b += 256) t += __ldcg(&partial[b]);
        t = warp_sum(t);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = t;
        __syncthreads();
        if (threadIdx.x == 0) {
            double rho = 0.0;
            for (int w = 0; w < 8; ++w) rho += red[w];
            sc->ticket[3] = 0;
            if (!(rho > 0.0) || !isfinite(rho)) {          // B is positive on the range of L: r.Br <= 0 is a breakdown
                sc->status = ST_BREAKDOWN; sc->inner_go = 0; sc->outer_go = 0;
                if (cond.use & 1) cudaGraphSetConditional((cudaGraphConditionalHandle)cond.h_outer, 0u);
                if (cond.use & 2) cudaGraphSetConditional((cudaGraphConditionalHandle)cond.h_inner, 0u);
            } else {
                sc->beta = (sc->k > 0) ? rho / sc->rho : 0.0;
                sc->rho = rho;
            }
        }
    }
}

}  // namespace omni
