// omni_mg.cuh -- geometric-multigrid V-cycle used as the preconditioner of CG on the fixed-point system L P = S
// (omni_solve_pcg_*, SURVEY.md 8(f) NEXT-2 ii; reading R-P1 of DESIGN.md).  Not the paper's iteration: the paper names
// only "CG"; this accelerates the separately named fixed-point solve of omni_solve_direct_*.
//
//   levels    level 0 = the grid (padded layout of the solver, its link bytes); level l+1 halves (ceil) every axis of
//             level l with >= 8 cells whose weight is >= 0.7 of the largest such weight (semi-coarsening: point smoothing
//             only works along strongly coupled axes; t_a ~ 1 / Delta_a, so the axis with the larger spacing waits until
//             the halvings of the others have made it strong); a coarse cell is valid iff one of its children is
//   operator  (L_l x)_C = sum_d v_l(C+d) w_l[a] (x_C - x_{C+d}); w_0[a] = t_a = F_a / A_tot (Eq. 10 :109),
//             w_{l+1}[a] = w_l[a] 2^m (1/4 if axis a was halved else 1), m = number of halved axes
//   transfer  restriction = sum over the children, prolongation = the parent's value (transposes of each other)
//   smoother  damped Jacobi x <- x + omega D^-1 (b - L x), omega = 0.8; 2 sweeps before and after the coarse-grid
//             correction (the first from x = 0), 8 on the coarsest level
// One thread per cell (per coarse cell in the restriction, which gathers its children in a fixed order: deterministic),
// cell indices from a 3D launch (no integer division).
// Bandwidth-bound elementwise / 7-point kernels on plain coalesced loads; neighbours come from L1 / L2.
#pragma once
#include "omni_kernels.cuh"

namespace omni {

constexpr int MG_MAX_LEVELS = 24;
constexpr int MG_MIN_COARSEN = 8;
constexpr double MG_THETA = 0.7;          // an axis is halved only while its weight is >= MG_THETA x the largest (semi-coarsening)
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

// Launch shape of every level kernel: blocks of MG_BX x MG_BY threads over (x, y), one plane per blockIdx.z -- a
// thread's cell comes from its indices, with no integer division (a linear index split by 64-bit / and % costs more than
// the 7-point stencil itself and kept these kernels at a third of the memory roofline).
constexpr int MG_BX = 64, MG_BY = 4;
template <typename T>
inline dim3 mg_grid(const MgLevel<T>& L) { return dim3((unsigned)((L.px + MG_BX - 1) / MG_BX), (unsigned)((L.ny + MG_BY - 1) / MG_BY), (unsigned)L.nz); }
inline dim3 mg_block() { return dim3(MG_BX, MG_BY, 1); }

// the thread's cell (i, j, k) and linear index c in level L; false outside the array (i >= px or j >= ny);
// cells with nx <= i < px are the pad cells of level 0
template <typename T>
__device__ __forceinline__ bool mg_cell(const MgLevel<T>& L, int& i, int& j, int& k, long long& c)
{
    i = blockIdx.x * MG_BX + threadIdx.x;
    j = blockIdx.y * MG_BY + threadIdx.y;
    k = blockIdx.z;
    if (i >= L.px || j >= L.ny) return false;
    c = i + (long long)L.px * (j + (long long)L.ny * k);
    return true;
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
__global__ void __launch_bounds__(MG_BX * MG_BY)
mg_jacobi_kernel(const MgLevel<T> L, const T* __restrict__ xin, T* __restrict__ xout)
{
    long long c;
    int i, j, k;
    if (!mg_cell(L, i, j, k, c)) return;
    if (i >= L.nx) { xout[c] = T(0); return; }
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

// ---- the same sweep, four cells of a row per thread (rows are padded to a multiple of 4 cells on every level): 16 /
// 32-byte loads, every neighbour load issued unconditionally (by position, not by link bit) so that a thread has ~10
// independent loads in flight instead of a link -> neighbour chain; one cell per thread leaves the memory system at a
// third of its bandwidth.  Link bits select the weights: a missing link contributes w = 0.
template <typename T, bool FIRST>
__global__ void __launch_bounds__(MG_BX * MG_BY)
mg_jacobi4_kernel(const MgLevel<T> L, const T* __restrict__ xin, T* __restrict__ xout)
{
    const int i0 = (blockIdx.x * MG_BX + threadIdx.x) * 4, j = blockIdx.y * MG_BY + threadIdx.y, k = blockIdx.z;
    if (i0 >= L.px || j >= L.ny) return;
    const long long c = i0 + (long long)L.px * (j + (long long)L.ny * k);
    const uint32_t lw = *reinterpret_cast<const uint32_t*>(L.link + c);
    T b[4], v[4];
    ld_chunk<T, 4>(L.b + c, b);
    if (FIRST) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const uint32_t l = (lw >> (8 * q)) & 0xffu;
            const T D = mg_diag(L, l);
            v[q] = ((l & LINK_VALID) && D > T(0)) ? (T)MG_OMEGA * (b[q] / D) : T(0);
        }
    } else {
        T xc[4], xn[4], xs[4], xf[4], xb[4];
        ld_chunk<T, 4>(xin + c, xc);
        zero_chunk<T, 4>(xn); zero_chunk<T, 4>(xs); zero_chunk<T, 4>(xf); zero_chunk<T, 4>(xb);
        if (j + 1 < L.ny) ld_chunk<T, 4>(xin + c + L.px, xn);
        if (j > 0) ld_chunk<T, 4>(xin + c - L.px, xs);
        if (k + 1 < L.nz) ld_chunk<T, 4>(xin + c + L.pplane, xf);
        if (k > 0) ld_chunk<T, 4>(xin + c - L.pplane, xb);
        const T xl = (i0 > 0) ? xin[c - 1] : T(0), xr = (i0 + 4 < L.px) ? xin[c + 4] : T(0);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const uint32_t l = (lw >> (8 * q)) & 0xffu;
            const T e = (q == 3) ? xr : xc[q < 3 ? q + 1 : 3], w = (q == 0) ? xl : xc[q > 0 ? q - 1 : 0];
            // same terms in the same order as mg_stencil; an absent link has weight 0
            const T w0 = (l & 1u) ? L.w[0] : T(0), w1 = (l & 2u) ? L.w[0] : T(0), w2 = (l & 4u) ? L.w[1] : T(0);
            const T w3 = (l & 8u) ? L.w[1] : T(0), w4 = (l & 16u) ? L.w[2] : T(0), w5 = (l & 32u) ? L.w[2] : T(0);
            T D = T(0), Lx = T(0);
            D += w0; Lx += w0 * (xc[q] - e);
            D += w1; Lx += w1 * (xc[q] - w);
            D += w2; Lx += w2 * (xc[q] - xn[q]);
            D += w3; Lx += w3 * (xc[q] - xs[q]);
            D += w4; Lx += w4 * (xc[q] - xf[q]);
            D += w5; Lx += w5 * (xc[q] - xb[q]);
            T r = T(0);
            if (l & LINK_VALID) {
                r = xc[q];
                if (D > T(0)) r += (T)MG_OMEGA * ((b[q] - Lx) / D);
            }
            v[q] = r;
        }
    }
    st_chunk<T, 4>(xout + c, v);
}

// coarse right-hand side with the x axis halved, two coarse cells = one 4-cell fine chunk per child row and thread;
// children are added in the same (plane, row, cell) order as in mg_residual_restrict_kernel
template <typename T>
__global__ void __launch_bounds__(MG_BX * MG_BY)
mg_residual_restrict4_kernel(const MgLevel<T> F, const MgLevel<T> C, const T* __restrict__ x)
{
    const int ci0 = (blockIdx.x * MG_BX + threadIdx.x) * 2, cj = blockIdx.y * MG_BY + threadIdx.y, ck = blockIdx.z;
    if (ci0 >= C.px || cj >= C.ny) return;
    const long long I = ci0 + (long long)C.px * (cj + (long long)C.ny * ck);
    const int i0 = 2 * ci0;
    T s[2] = { T(0), T(0) };
    if (i0 < F.px) {
        for (int dk = 0; dk <= F.hz; ++dk)
            for (int dj = 0; dj <= F.hy; ++dj) {
                const int j = (F.hy ? 2 * cj : cj) + dj, k = (F.hz ? 2 * ck : ck) + dk;
                if (j >= F.ny || k >= F.nz) continue;
                const long long c = i0 + (long long)F.px * (j + (long long)F.ny * k);
                const uint32_t lw = *reinterpret_cast<const uint32_t*>(F.link + c);
                if (!(lw & 0x40404040u)) continue;
                T b[4], xc[4], xn[4], xs[4], xf[4], xb[4];
                ld_chunk<T, 4>(F.b + c, b);
                ld_chunk<T, 4>(x + c, xc);
                zero_chunk<T, 4>(xn); zero_chunk<T, 4>(xs); zero_chunk<T, 4>(xf); zero_chunk<T, 4>(xb);
                if (j + 1 < F.ny) ld_chunk<T, 4>(x + c + F.px, xn);
                if (j > 0) ld_chunk<T, 4>(x + c - F.px, xs);
                if (k + 1 < F.nz) ld_chunk<T, 4>(x + c + F.pplane, xf);
                if (k > 0) ld_chunk<T, 4>(x + c - F.pplane, xb);
                const T xl = (i0 > 0) ? x[c - 1] : T(0), xr = (i0 + 4 < F.px) ? x[c + 4] : T(0);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const uint32_t l = (lw >> (8 * q)) & 0xffu;
                    if (!(l & LINK_VALID)) continue;
                    const T e = (q == 3) ? xr : xc[q < 3 ? q + 1 : 3], w = (q == 0) ? xl : xc[q > 0 ? q - 1 : 0];
                    T Lx = T(0);
                    if (l & 1u) Lx += F.w[0] * (xc[q] - e);
                    if (l & 2u) Lx += F.w[0] * (xc[q] - w);
                    if (l & 4u) Lx += F.w[1] * (xc[q] - xn[q]);
                    if (l & 8u) Lx += F.w[1] * (xc[q] - xs[q]);
                    if (l & 16u) Lx += F.w[2] * (xc[q] - xf[q]);
                    if (l & 32u) Lx += F.w[2] * (xc[q] - xb[q]);
                    s[q >> 1] += b[q] - Lx;
                }
            }
    }
    C.b[I] = (ci0 < C.nx) ? s[0] : T(0);
    C.b[I + 1] = (ci0 + 1 < C.nx) ? s[1] : T(0);
}

// x += prolong(e), four fine cells per thread
template <typename T>
__global__ void __launch_bounds__(MG_BX * MG_BY)
mg_prolong_add4_kernel(const MgLevel<T> F, const MgLevel<T> C, T* __restrict__ x, const T* __restrict__ e)
{
    const int i0 = (blockIdx.x * MG_BX + threadIdx.x) * 4, j = blockIdx.y * MG_BY + threadIdx.y, k = blockIdx.z;
    if (i0 >= F.px || j >= F.ny) return;
    const long long c = i0 + (long long)F.px * (j + (long long)F.ny * k);
    const uint32_t lw = *reinterpret_cast<const uint32_t*>(F.link + c);
    if (!(lw & 0x40404040u)) return;                              // no valid cell in the chunk
    const long long I = (F.hx ? i0 >> 1 : i0) + (long long)C.px * ((F.hy ? j >> 1 : j) + (long long)C.ny * (F.hz ? k >> 1 : k));
    T v[4];
    ld_chunk<T, 4>(x + c, v);
#pragma unroll
    for (int q = 0; q < 4; ++q)
        if ((lw >> (8 * q)) & LINK_VALID) {
            const int ci = F.hx ? (q >> 1) : q;                   // parent of fine cell i0 + q relative to I
            if ((F.hx ? ((i0 + q) >> 1) : (i0 + q)) < C.nx) v[q] += e[I + ci];
        }
    st_chunk<T, 4>(x + c, v);
}

// coarse right-hand side: b_c[I] = sum over the valid children C of I of (b - L x)_C, children in a fixed order
template <typename T>
__global__ void __launch_bounds__(MG_BX * MG_BY)
mg_residual_restrict_kernel(const MgLevel<T> F, const MgLevel<T> C, const T* __restrict__ x)
{
    long long I;
    int ci, cj, ck;
    if (!mg_cell(C, ci, cj, ck, I)) return;
    if (ci >= C.nx) { C.b[I] = T(0); return; }
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
__global__ void __launch_bounds__(MG_BX * MG_BY)
mg_prolong_add_kernel(const MgLevel<T> F, const MgLevel<T> C, T* __restrict__ x, const T* __restrict__ e)
{
    long long c;
    int i, j, k;
    if (!mg_cell(F, i, j, k, c) || i >= F.nx) return;
    if (!(F.link[c] & LINK_VALID)) return;
    const long long I = (F.hx ? i >> 1 : i) + (long long)C.px * ((F.hy ? j >> 1 : j) + (long long)C.ny * (F.hz ? k >> 1 : k));
    x[c] += e[I];
}

// validity of the next level: a coarse cell is valid iff one of its children is
template <typename T>
__global__ void __launch_bounds__(MG_BX * MG_BY)
mg_coarse_valid_kernel(const MgLevel<T> F, const MgLevel<T> C, uint8_t* __restrict__ vc)
{
    long long I;
    int ci, cj, ck;
    if (!mg_cell(C, ci, cj, ck, I)) return;
    uint8_t any = 0;
    if (ci < C.nx)
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
__global__ void __launch_bounds__(MG_BX * MG_BY)
mg_link_kernel(const MgLevel<T> C, const uint8_t* __restrict__ vc, uint8_t* __restrict__ link, int naxes)
{
    long long I;
    int i, j, k;
    if (!mg_cell(C, i, j, k, I)) return;
    uint32_t l = 0;
    if (i < C.nx && vc[I]) {
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
