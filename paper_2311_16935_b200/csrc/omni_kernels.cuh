// omni_kernels.cuh -- sm_100a kernels of the matrix-based omnidirectional pressure integration hot path.
// Zigunov & Charonko, arXiv 2311.16935 (citations: PAPER.md:<line>); notation of DESIGN.md section 2.
//
//   K0a validity, K0b stencil codes + interior flags        (Eq. 13 :176; Eq. 16/18/19/20 :202-227; Eq. 25 :266)
//   K1  source vector S + ||S||^2                              (last sum of Eq. 9 :100; Eq. 49-50 :656)
//   K2  outer boundary update: P += delta, r = S - L P, eps_R  (Eq. 12 :119; Eq. 41 :442; Alg. 1 :141-148)
//   K3  p = r + beta p (fused), gamma = p . M p                (CG, :124)
//   K4  q = M p recomputed, delta += alpha p, r -= alpha q, rho' = r.r
//   K7  P_out with NaN at missing cells                        (:158)
// K2/K3/K4 run on the TMA + mbarrier tile pipeline of omni_tma.cuh; this header holds the shared device helpers
// (geometry, coefficient tables, operator evaluation, face corrections) and the one-off kernels K0, K1, K7.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

namespace omni {

struct Geom {
    int nx, ny, nz;      // logical grid (batch mode: nz = number of stacked 2D snapshots)
    int naxes;           // 2: 2D scheme (nz == 1, or nz stacked 2D snapshots with no coupling across planes); 3: 3D
    int batch;           // 1: stacked 2D snapshots; the mask, if any, is one plane shared by all snapshots
    int px;              // padded row pitch in cells (multiple of 8); cells nx..px-1 are permanently missing
    long long pplane;    // px * ny
    long long npad;      // px * ny * nz
    // Box faces never flag a group: a cell whose code equals the code it would have in a mask-free box is handled by the
    // fast path plus additive per-axis corrections (x: per lane, y: per row, z: per plane; face_fix / xedge_fix).  A
    // group is flagged only if a mask / NaN cell changes some code.  fix[a] = 1 iff axis a is long enough (n_a >= 4)
    // for its four face classes (cells 0, 1, n-2, n-1) to be distinct cells; otherwise that axis' faces do flag.
    uint32_t icode;
    int fix[3];
    int xfix;            // = fix[0]
    // tile-plane flags for the K3/K4 tiles (tbx x tby cells): bit (k & 31) of tflags[(ty*ntx + tx)*twords + (k >> 5)]
    // is set iff some group of tile (tx, ty) is flagged in plane k; unset bits let a warp skip the per-row flag word
    int tbx, tby, ntx, nty, twords;
    // z-slab sharding (omni_slab.cuh): the local grid is a window of the global one with up to two halo planes per
    // side; the tile kernels emit, and the reductions count, only the planes [kz0, kz1) this rank owns (0, nz otherwise)
    int kz0, kz1;
};

// stencil coefficients, already divided by A_tot (Eq. 10 :109), in the arithmetic type T
template <typename T>
struct Coef {
    T t[3];    // F_a / A_tot: weight of a fully interior link (Eq. 5 :75 / Eq. 23 :258); also the L-operator weight
    T caa[3];  // c_aa / A_tot         far-face constant       (Eq. 17 :207 / Eq. 32 :314)
    T cab[3];  // c_{a,(a+1)%3} / A_tot  side-face constants   (Eq. 17 / Eq. 33 :317)
    T cac[3];  // c_{a,(a+2)%3} / A_tot
    T hs[3];   // Delta_a * t_a / 2: face-average factor of the source term (Eq. 9 :100)
    T lut[3][32];      // lut[a][far | nb<<1 | nc<<3] = far*caa + nb*cab + nc*cac: weight of a coded link
    T fc[3][4][6];     // fc[axis][class][d] = t_a(d) - w_d(face-class code): what the fast path over-subtracts there
    uint32_t icode;    // wcode of a fully interior cell of this geometry (2D: no z links)
};

// which x-edge cells a thread's chunk holds (thread constants)
struct XEdge {
    bool L, A, B;      // holds cells {0,1} / cell nx-2 / cell nx-1
    bool any;          // L || A || B
    int posA, posB;    // their positions inside the chunk
};
template <int V>
__device__ __forceinline__ XEdge make_xedge(const Geom& g, int x)
{
    XEdge e;
    const bool on = g.xfix != 0;
    e.L = on && (x == 0);
    e.posA = (g.nx - 2) % V; e.posB = (g.nx - 1) % V;
    e.A = on && (x == g.nx - 2 - e.posA);
    e.B = on && (x == g.nx - 1 - e.posB);
    e.any = e.L || e.A || e.B;
    return e;
}

// device-resident loop state: no scalar ever visits the host inside the iteration
struct Scalars {
    double rho, gamma, alpha, beta;
    double alpha_prev; // alpha of the CG iteration whose delta update is pending (lazy delta, omni_tma.cuh K4)
    double normS2;     // ||S||^2
    double thresh2;    // (0.1 * tol)^2 * ||S||^2   inner stop (A3)
    double inner_rel2; // omni_solve_pcg fp32 only (0 elsewhere): an inner solve also stops at ||r||^2 <= inner_rel2 ||r0||^2
    double thresh2_in; // the inner threshold of the current outer iteration: max(thresh2, inner_rel2 ||r0||^2), set by K2
    double tol2S;      // tol^2 * ||S||^2           outer stop (Eq. 41)
    double epsR2;      // ||r0||^2 of the last outer check
    double tol;
    long long cg_total;
    int k;             // CG iteration index inside the current outer iteration
    int n;             // outer iterations done
    int inner_go, outer_go;
    int pend;          // 1: delta still lacks alpha_prev * p of the last (even) CG iteration
    int dzero;         // 1: delta counts as zero in the next K2 (no CG iteration has run since the last fold: the first
                       //    outer check, or an outer iteration whose inner loop did not start) -- K2 must not fold a stale delta
    int status;        // omni_status
    int max_cg, max_outer;
    unsigned int ticket[4];
    unsigned int bar_count;  // use count of the loop kernel's grid barrier, carried from one launch to the next (omni_loop.cuh)
    // optional residual history (omni_set_history): eps_R (Eq. 41) of every outer residual check, entry i = check i
    // and, optionally, the CG iterations the outer iteration before the check took (0 for the first check)
    // and the pressure-update metric eps_P (Eq. 40 :438) of the update that led to the check (0 for the first check)
    double* hist;
    int* hist_k;
    double* hist_p;
    int hist_cap, hist_n;
    int* status_out;   // optional device word that receives the final status (omni_options::d_status)
    // sharded solves: defer = 1 makes the reducing kernels leave their grid totals in red_out instead of acting on them;
    // the totals are summed over the ranks and a one-thread kernel then runs the same finalize code on every rank
    int defer;
    double red_out[4];
};

// dP2 = ||P^n - P^(n-1)||^2, P2 = ||P^n||^2 (Eq. 40); either 0 when nothing was folded
__device__ __forceinline__ void record_history(Scalars* s, double epsR2, int k_prev, double dP2 = 0.0, double P2 = 0.0)
{
    if (s->hist_n < s->hist_cap) {
        if (s->hist != nullptr) s->hist[s->hist_n] = (s->normS2 > 0.0) ? sqrt(epsR2 / s->normS2) : 0.0;
        if (s->hist_k != nullptr) s->hist_k[s->hist_n] = k_prev;
        if (s->hist_p != nullptr) s->hist_p[s->hist_n] = (P2 > 0.0) ? sqrt(dP2 / P2) : 0.0;
    }
    s->hist_n += 1;
}

struct CondHandles {
    unsigned long long h_outer, h_inner;   // cudaGraphConditionalHandle
    int use;                               // bit 0: h_outer is live (inside the conditional-node graph), bit 1: h_inner is
};

enum { ST_OK = 0, ST_NOT_CONVERGED = 1, ST_BREAKDOWN = -4 };

// per-cell code layout.  wcode: for direction d (0..5 = E W N S F B, axis a = d/2) bits [5d, 5d+5) hold
// far (1 bit: v(Q+d)), nb (2 bits: v(Q+e_b)+v(Q-e_b), b=(a+1)%3), nc (2 bits, c=(a+2)%3), all zero when the link is
// absent; bit 30 = cell valid.  link: bits 0..5 = v(C+d), bit 6 = cell valid.
constexpr uint32_t WCODE_VALID = 1u << 30;
constexpr uint8_t LINK_VALID = 1u << 6;

// ------------------------------------------------------------------------------------------------ small helpers

template <typename T, int V>
__device__ __forceinline__ void ld_chunk(const T* __restrict__ p, T (&v)[V])
{
    constexpr int BYTES = V * (int)sizeof(T);
    static_assert(BYTES == 8 || BYTES % 16 == 0, "chunk must be 8 bytes or a multiple of 16");
    if constexpr (BYTES == 8) {
        uint2 u = *reinterpret_cast<const uint2*>(p);
        memcpy(v, &u, 8);
    } else {
        constexpr int NV = BYTES / 16;
        uint4 u[NV];
#pragma unroll
        for (int i = 0; i < NV; ++i) u[i] = reinterpret_cast<const uint4*>(p)[i];
        memcpy(v, u, sizeof(u));
    }
}

template <typename T, int V>
__device__ __forceinline__ void st_chunk(T* __restrict__ p, const T (&v)[V])
{
    constexpr int BYTES = V * (int)sizeof(T);
    if constexpr (BYTES == 8) {
        uint2 u;
        memcpy(&u, v, 8);
        *reinterpret_cast<uint2*>(p) = u;
    } else {
        constexpr int NV = BYTES / 16;
        uint4 u[NV];
        memcpy(u, v, sizeof(u));
#pragma unroll
        for (int i = 0; i < NV; ++i) reinterpret_cast<uint4*>(p)[i] = u[i];
    }
}

template <typename T, int V>
__device__ __forceinline__ void zero_chunk(T (&v)[V])
{
#pragma unroll
    for (int i = 0; i < V; ++i) v[i] = T(0);
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// weight of one link from its 5 code bits (Eq. 16/19 :202/:223, Eq. 25 :266, divided by A_tot): table in the
// kernel-parameter constant bank
template <typename T>
__device__ __forceinline__ T link_weight(uint32_t bits, const Coef<T>& K, int a)
{
    return K.lut[a][bits & 31u];
}

// (M p)_C = p_C - sum_d w1_d p_{C+d}   (Eq. 9 rearranged, A1); general (coded) cell
template <typename T>
__device__ __forceinline__ T apply_M_coded(uint32_t code, T c, T e, T w, T n, T s, T f, T b, const Coef<T>& K)
{
    if (!(code & WCODE_VALID)) return T(0);
    T acc = c;
    acc -= link_weight(code, K, 0) * e;
    acc -= link_weight(code >> 5, K, 0) * w;
    acc -= link_weight(code >> 10, K, 1) * n;
    acc -= link_weight(code >> 15, K, 1) * s;
    acc -= link_weight(code >> 20, K, 2) * f;
    acc -= link_weight(code >> 25, K, 2) * b;
    return acc;
}

// interior cell: every link carries its full face share t_a (Eq. 5 :75: A^{n+1} = F_a, A^n = 0)
template <typename T>
__device__ __forceinline__ T apply_M_interior(T c, T e, T w, T n, T s, T f, T b, const Coef<T>& K)
{
    return c - K.t[0] * (e + w) - K.t[1] * (n + s) - K.t[2] * (f + b);
}

// q[I] += sum_d xc[cls][d] * neighbour_d: turns the interior formula into the exact one at an x-edge cell
template <int I, typename T, int V>
__device__ __forceinline__ void xfix_cell(T (&q)[V], const T (&vm)[V], const T (&vc)[V], const T (&vp)[V],
                                          const T (&vn)[V], const T (&vs)[V], T xl, T xr, const T (&c)[6])
{
    const T w = (I == 0) ? xl : vc[I > 0 ? I - 1 : 0];
    const T e = (I == V - 1) ? xr : vc[I < V - 1 ? I + 1 : V - 1];
    q[I] += c[0] * e + c[1] * w + c[2] * vn[I] + c[3] * vs[I] + c[4] * vp[I] + c[5] * vm[I];
}
template <int I, typename T, int V>
__device__ __forceinline__ void xfix_zero_after(T (&q)[V])
{
#pragma unroll
    for (int i = I + 1; i < V; ++i) q[i] = T(0);      // pad cells nx..px-1
}

// face class of position i on an axis of length n: 0, 1 (cells 0, 1), 2, 3 (cells n-2, n-1), -1 otherwise / axis off
__device__ __forceinline__ int face_class(int i, int n, int on)
{
    // selects, not branches: evaluated per emitted plane in the tile kernels
    int c = -1;
    c = (i == n - 1) ? 3 : c;
    c = (i == n - 2) ? 2 : c;
    c = (i == 1) ? 1 : c;
    c = (i == 0) ? 0 : c;
    return on ? c : -1;
}

// whole-chunk correction for a row (y class) or plane (z class) next to a box face: uniform over the warp
template <typename T, int V>
__device__ __forceinline__ void face_fix(T (&q)[V], const T (&vm)[V], const T (&vc)[V], const T (&vp)[V],
                                         const T (&vn)[V], const T (&vs)[V], T xl, T xr, const T (&c)[6])
{
#pragma unroll
    for (int i = 0; i < V; ++i) {
        const T w = (i == 0) ? xl : vc[i > 0 ? i - 1 : 0];
        const T e = (i == V - 1) ? xr : vc[i < V - 1 ? i + 1 : V - 1];
        q[i] += c[0] * e + c[1] * w + c[2] * vn[i] + c[3] * vs[i] + c[4] * vp[i] + c[5] * vm[i];
    }
}

template <typename T, int V>
__device__ __forceinline__ void xedge_fix(T (&q)[V], const T (&vm)[V], const T (&vc)[V], const T (&vp)[V],
                                          const T (&vn)[V], const T (&vs)[V], T xl, T xr, const XEdge& xe,
                                          const Coef<T>& K)
{
    if (xe.L) {
        xfix_cell<0, T, V>(q, vm, vc, vp, vn, vs, xl, xr, K.fc[0][0]);
        xfix_cell<1, T, V>(q, vm, vc, vp, vn, vs, xl, xr, K.fc[0][1]);
    }
    if (xe.A) {
        switch (xe.posA) {
#define OMNI_CASE(I) case I: if (I < V) xfix_cell<(I < V ? I : 0), T, V>(q, vm, vc, vp, vn, vs, xl, xr, K.fc[0][2]); break;
            OMNI_CASE(0) OMNI_CASE(1) OMNI_CASE(2) OMNI_CASE(3) OMNI_CASE(4) OMNI_CASE(5) OMNI_CASE(6) OMNI_CASE(7)
#undef OMNI_CASE
        }
    }
    if (xe.B) {
        switch (xe.posB) {
#define OMNI_CASE(I) case I: if (I < V) { xfix_cell<(I < V ? I : 0), T, V>(q, vm, vc, vp, vn, vs, xl, xr, K.fc[0][3]); \
                                          xfix_zero_after<(I < V ? I : 0), T, V>(q); } break;
            OMNI_CASE(0) OMNI_CASE(1) OMNI_CASE(2) OMNI_CASE(3) OMNI_CASE(4) OMNI_CASE(5) OMNI_CASE(6) OMNI_CASE(7)
#undef OMNI_CASE
        }
    }
}

// q = M p for the V cells of one thread; fb = flag bit of the thread's 4-cell group (0 = interior or box face: fast
// path + face corrections; else `code` holds the chunk's codes -- fetched a plane ahead by the caller -- and the
// cells that need it take the coded path)
template <typename T, int V>
__device__ __forceinline__ void apply_M_chunk(T (&q)[V], const T (&vm)[V], const T (&vc)[V], const T (&vp)[V],
                                              const T (&vn)[V], const T (&vs)[V], T xl, T xr, uint32_t fb,
                                              const uint32_t (&code)[V], const Coef<T>& K,
                                              const XEdge& xe, int ycls, int zcls)
{
#pragma unroll
    for (int i = 0; i < V; ++i) {
        T w = (i == 0) ? xl : vc[i - 1];
        T e = (i == V - 1) ? xr : vc[i + 1];
        q[i] = apply_M_interior(vc[i], e, w, vn[i], vs[i], vp[i], vm[i], K);
    }
    if (fb == 0) {
        if (ycls >= 0) face_fix<T, V>(q, vm, vc, vp, vn, vs, xl, xr, K.fc[1][ycls]);      // warp-uniform
        if (zcls >= 0) face_fix<T, V>(q, vm, vc, vp, vn, vs, xl, xr, K.fc[2][zcls]);      // CTA-uniform
        if (xe.any) xedge_fix<T, V>(q, vm, vc, vp, vn, vs, xl, xr, xe, K);               // last: zeroes the pad cells
    } else {
#pragma unroll
        for (int i = 0; i < V; ++i) {
            T w = (i == 0) ? xl : vc[i - 1];
            T e = (i == V - 1) ? xr : vc[i + 1];
            if (code[i] != K.icode) q[i] = apply_M_coded(code[i], vc[i], e, w, vn[i], vs[i], vp[i], vm[i], K);
        }
    }
}

// q = L p for the V cells of one thread, (L p)_C = sum_d v(C+d) t_a (p_C - p_{C+d}): the operator of the fixed-point
// system L P = S (M - W^n of Eq. 12 :119 at P^{n+1} = P^n), used by omni_solve_direct.  Unflagged chunks have the
// links of the mask-free box: the interior formula already sees zeros beyond the faces (TMA zero fill, pad cells), so
// only the diagonal loses t_a per missing face link.  Flagged chunks: lk[i] = link byte of cell i.
template <typename T, int V>
__device__ __forceinline__ void apply_L_chunk(T (&q)[V], const T (&vm)[V], const T (&vc)[V], const T (&vp)[V],
                                              const T (&vn)[V], const T (&vs)[V], T xl, T xr, uint32_t fb,
                                              const uint32_t (&lk)[V], const Coef<T>& K,
                                              const XEdge& xe, int ycls, int zcls)
{
    if (fb == 0) {
        T dg = T(0);
        if (ycls == 0 || ycls == 3) dg += K.t[1];
        if (zcls == 0 || zcls == 3) dg += K.t[2];
#pragma unroll
        for (int i = 0; i < V; ++i) {
            T w = (i == 0) ? xl : vc[i - 1];
            T e = (i == V - 1) ? xr : vc[i + 1];
            q[i] = apply_M_interior(vc[i], e, w, vn[i], vs[i], vp[i], vm[i], K) - dg * vc[i];
        }
        if (xe.any) {
            if (xe.L) q[0] -= K.t[0] * vc[0];
            if (xe.B) {
#pragma unroll
                for (int i = 0; i < V; ++i) {
                    if (i == xe.posB) q[i] -= K.t[0] * vc[i];
                    if (i > xe.posB) q[i] = T(0);                 // pad cells nx..px-1
                }
            }
        }
    } else {
#pragma unroll
        for (int i = 0; i < V; ++i) {
            T w = (i == 0) ? xl : vc[i - 1];
            T e = (i == V - 1) ? xr : vc[i + 1];
            const uint32_t l = lk[i];
            T acc = T(0);
            if (l & 1u) acc += K.t[0] * (vc[i] - e);
            if (l & 2u) acc += K.t[0] * (vc[i] - w);
            if (l & 4u) acc += K.t[1] * (vc[i] - vn[i]);
            if (l & 8u) acc += K.t[1] * (vc[i] - vs[i]);
            if (l & 16u) acc += K.t[2] * (vc[i] - vp[i]);
            if (l & 32u) acc += K.t[2] * (vc[i] - vm[i]);
            q[i] = (l & LINK_VALID) ? acc : T(0);
        }
    }
}

// the operator a CG kernel applies: M (Alg. 1) or L (fixed-point solve); `code` holds stencil codes resp. link bytes
template <bool LOP, typename T, int V>
__device__ __forceinline__ void apply_op_chunk(T (&q)[V], const T (&vm)[V], const T (&vc)[V], const T (&vp)[V],
                                               const T (&vn)[V], const T (&vs)[V], T xl, T xr, uint32_t fb,
                                               const uint32_t (&code)[V], const Coef<T>& K,
                                               const XEdge& xe, int ycls, int zcls)
{
    if constexpr (LOP) apply_L_chunk<T, V>(q, vm, vc, vp, vn, vs, xl, xr, fb, code, K, xe, ycls, zcls);
    else apply_M_chunk<T, V>(q, vm, vc, vp, vn, vs, xl, xr, fb, code, K, xe, ycls, zcls);
}

// per-cell data of a flagged chunk: the V stencil codes (M) or the V link bytes (L), one per array element
template <bool LOP, int V>
__device__ __forceinline__ void load_cell_codes(const uint32_t* __restrict__ wcode, const uint8_t* __restrict__ link,
                                                long long cell, uint32_t (&code)[V])
{
    if constexpr (!LOP) {
        ld_chunk<uint32_t, V>(wcode + cell, code);
    } else if constexpr (V == 4) {
        const uint32_t w = *reinterpret_cast<const uint32_t*>(link + cell);
#pragma unroll
        for (int i = 0; i < 4; ++i) code[i] = (w >> (8 * i)) & 0xffu;
    } else {
        static_assert(V == 2, "chunks hold 4 fp32 or 2 fp64 cells");
        const uint32_t w = *reinterpret_cast<const unsigned short*>(link + cell);
        code[0] = w & 0xffu; code[1] = w >> 8;
    }
}

// interior-flag bits of the V/4 groups starting at padded cell idx (one bit per 4 cells, global linear bit index)
template <int V>
__device__ __forceinline__ uint32_t flag_bits(const uint32_t* __restrict__ flags, long long idx)
{
    long long g = idx >> 2;
    return (flags[g >> 5] >> (unsigned)(g & 31)) & ((1u << (V >= 4 ? V / 4 : 1)) - 1u);
}

// padded linear index -> (i, row = j + ny*k); 32-bit arithmetic wherever the grid allows it
__device__ __forceinline__ void split_pid(const Geom& g, long long pid, int& i, long long& row)
{
    if (g.npad < (1LL << 31)) {
        const unsigned int r = (unsigned int)pid / (unsigned int)g.px;
        i = (int)((unsigned int)pid - r * (unsigned int)g.px);
        row = r;
    } else {
        i = (int)(pid % g.px);
        row = pid / g.px;
    }
}

// ------------------------------------------------------------------------------------------------ K0a validity
template <typename T>
__global__ void validity_kernel(Geom g, const T* __restrict__ gx, const T* __restrict__ gy, const T* __restrict__ gz,
                                const uint8_t* __restrict__ mask, uint8_t* __restrict__ vbyte)
{
    long long pid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (pid >= g.npad) return;
    int i;
    long long row;                                // j + ny*k
    split_pid(g, pid, i, row);
    uint8_t ok = 0;
    if (i < g.nx) {
        long long u = row * g.nx + i;             // user-layout index
        ok = (mask == nullptr) || (mask[g.batch ? (u % ((long long)g.nx * g.ny)) : u] != 0);
        if (gx != nullptr) {
            if (isnan(gx[u]) || isnan(gy[u])) ok = 0;
            if (g.naxes == 3 && isnan(gz[u])) ok = 0;
        }
    }
    vbyte[pid] = ok;
}

// ------------------------------------------------------------------------------------------------ K0b codes
__device__ __forceinline__ int vget(const Geom& g, const uint8_t* __restrict__ v, int i, int j, int k)
{
    if (i < 0 || j < 0 || k < 0 || i >= g.nx || j >= g.ny || k >= g.nz) return 0;
    return v[i + (long long)g.px * (j + (long long)g.ny * k)];
}

// validity in the mask-free box, seen by the face corrections: axes whose faces are corrected (fix[a]) end at the box,
// the others are treated as unbounded (their face cells then differ from this code and get flagged); an inactive z axis
// (2D) has no neighbours at all
__device__ __forceinline__ uint32_t vbox(const Geom& g, int i, int j, int k)
{
    if (g.fix[0] && (i < 0 || i >= g.nx)) return 0u;
    if (g.fix[1] && (j < 0 || j >= g.ny)) return 0u;
    if (g.naxes == 2) return 1u;              // planes are independent 2D problems: k is never offset (see box_code)
    if (g.fix[2] && (k < 0 || k >= g.nz)) return 0u;
    return 1u;
}
__device__ __forceinline__ uint32_t box_code(const Geom& g, int i, int j, int k)
{
    if (i >= g.nx) return g.fix[0] ? 0u : g.icode;      // pad cells: expected only where xedge_fix zeroes them
    if (!vbox(g, i, j, k)) return 0u;
    const int naxes = g.naxes;
    uint32_t code = WCODE_VALID;
    for (int d = 0; d < 2 * naxes; ++d) {
        const int a = d >> 1, sg = (d & 1) ? -1 : 1;
        int e[3] = { 0, 0, 0 };
        e[a] = sg;
        const int qi = i + e[0], qj = j + e[1], qk = k + e[2];
        if (!vbox(g, qi, qj, qk)) continue;
        const int b = (a + 1) % 3, cc = (a + 2) % 3;
        int eb[3] = { 0, 0, 0 }, ec[3] = { 0, 0, 0 };
        eb[b] = 1; ec[cc] = 1;
        const uint32_t far = vbox(g, qi + e[0], qj + e[1], qk + e[2]);
        const uint32_t nb = (b < naxes) ? vbox(g, qi + eb[0], qj + eb[1], qk + eb[2]) + vbox(g, qi - eb[0], qj - eb[1], qk - eb[2]) : 0u;
        const uint32_t nc = (cc < naxes) ? vbox(g, qi + ec[0], qj + ec[1], qk + ec[2]) + vbox(g, qi - ec[0], qj - ec[1], qk - ec[2]) : 0u;
        code |= (far | (nb << 1) | (nc << 3)) << (5 * d);
    }
    return code;
}

// decode one 4-cell group cell by cell (any position: faces, corners, mask surface); returns its flag
__device__ __forceinline__ bool decode_group(const Geom& g, const uint8_t* __restrict__ vbyte, uint8_t* __restrict__ link,
                                             uint32_t* __restrict__ wcode, long long base, int i0, int j, int k)
{
    const int naxes = g.naxes;
    uint32_t codes[4];
    uint32_t links = 0;
    bool flagged = false;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const int i = i0 + c;
        uint32_t code = 0, lk = 0;
        if (vget(g, vbyte, i, j, k)) {
            code = WCODE_VALID; lk = LINK_VALID;
            for (int d = 0; d < 6; ++d) {
                const int a = d >> 1, sg = (d & 1) ? -1 : 1;
                int e[3] = { 0, 0, 0 };
                e[a] = sg;
                const int qi = i + e[0], qj = j + e[1], qk = k + e[2];
                if (a >= naxes) continue;                       // 2D scheme: no F/B links at all
                if (!vget(g, vbyte, qi, qj, qk)) continue;
                lk |= 1u << d;
                const int b = (a + 1) % 3, cc = (a + 2) % 3;
                int eb[3] = { 0, 0, 0 }, ec[3] = { 0, 0, 0 };
                eb[b] = 1; ec[cc] = 1;
                uint32_t far = vget(g, vbyte, qi + e[0], qj + e[1], qk + e[2]);
                uint32_t nb = (b < naxes) ? vget(g, vbyte, qi + eb[0], qj + eb[1], qk + eb[2]) +
                                            vget(g, vbyte, qi - eb[0], qj - eb[1], qk - eb[2]) : 0u;
                uint32_t nc = (cc < naxes) ? vget(g, vbyte, qi + ec[0], qj + ec[1], qk + ec[2]) +
                                             vget(g, vbyte, qi - ec[0], qj - ec[1], qk - ec[2]) : 0u;
                code |= (far | (nb << 1) | (nc << 3)) << (5 * d);
            }
        }
        codes[c] = code;
        links |= lk << (8 * c);
        // two or more cells away from every face the mask-free box code is the interior code
        const bool deep = (i >= 2 && i < g.nx - 2) && (j >= 2 && j < g.ny - 2) && (g.naxes == 2 || (k >= 2 && k < g.nz - 2));
        const uint32_t expect = deep ? g.icode : box_code(g, i, j, k);
        flagged |= (code != expect);
    }
    *reinterpret_cast<uint4*>(wcode + base) = make_uint4(codes[0], codes[1], codes[2], codes[3]);
    *reinterpret_cast<uint32_t*>(link + base) = links;
    return flagged;
}

// K0b pass 1: one thread per 4-cell group.  A group at least two cells away from every face whose 25-cell
// neighbourhoods are all valid (23 aligned word loads instead of ~150 byte loads) is interior: nothing to decode,
// nothing flagged.  Every other group (box faces, the neighbourhood of masked cells: a few per cent, but at least one
// lane of half the warps of a 500-cell row) is appended to a work list with a warp-aggregated atomic and decoded by
// pass 2 with all lanes busy, instead of stalling its whole warp on the cell-by-cell path here.
__global__ void codes_kernel(Geom g, const uint8_t* __restrict__ vbyte, uint8_t* __restrict__ link,
                             uint32_t* __restrict__ wcode, uint32_t* __restrict__ flags, uint32_t* __restrict__ worklist,
                             unsigned int* __restrict__ work_count)
{
    const long long grp = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long ngrp = g.npad >> 2;
    bool defer = false;
    if (grp < ngrp) {
        const long long base = grp << 2;
        int i0, j, k;
        if (g.npad < (1LL << 31)) {                  // 32-bit index arithmetic wherever it fits
            const unsigned int b32 = (unsigned int)base, row = b32 / (unsigned int)g.px;
            i0 = (int)(b32 - row * (unsigned int)g.px);
            k = (int)(row / (unsigned int)g.ny);
            j = (int)(row - (unsigned int)k * (unsigned int)g.ny);
        } else {
            i0 = (int)(base % g.px);
            const long long row = base / g.px;
            j = (int)(row % g.ny); k = (int)(row / g.ny);
        }
        const bool deep_grp = (i0 >= 4) && (i0 + 8 <= g.nx) && (j >= 2) && (j < g.ny - 2) &&
                              (g.naxes == 2 || (k >= 2 && k < g.nz - 2));
        bool all_valid = false;
        if (deep_grp) {
            const long long sy = g.px, sz = g.pplane;
            const uint8_t* c0 = vbyte + base;
            auto w = [&](long long off) { return *reinterpret_cast<const uint32_t*>(c0 + off); };
            uint32_t m = w(-4) & w(0) & w(4);
            m &= w(-sy - 4) & w(-sy) & w(-sy + 4) & w(sy - 4) & w(sy) & w(sy + 4) & w(-2 * sy) & w(2 * sy);
            if (g.naxes == 3)
                m &= w(-sz - 4) & w(-sz) & w(-sz + 4) & w(sz - 4) & w(sz) & w(sz + 4) & w(-2 * sz) & w(2 * sz) &
                     w(-sz - sy) & w(-sz + sy) & w(sz - sy) & w(sz + sy);
            all_valid = (m == 0x01010101u);
        }
        if (all_valid) {
            *reinterpret_cast<uint4*>(wcode + base) = make_uint4(g.icode, g.icode, g.icode, g.icode);
            *reinterpret_cast<uint32_t*>(link + base) = (g.naxes == 3) ? 0x7f7f7f7fu : 0x4f4f4f4fu;
        } else {
            defer = true;
        }
    }
    const unsigned int lane = threadIdx.x & 31u;
    const uint32_t m = __ballot_sync(0xffffffffu, defer);
    if (m) {
        unsigned int at = 0;
        const int leader = __ffs(m) - 1;
        if ((int)lane == leader) at = atomicAdd(work_count, (unsigned int)__popc(m));
        at = __shfl_sync(0xffffffffu, at, leader);
        if (defer) worklist[at + __popc(m & ((1u << lane) - 1u))] = (uint32_t)grp;
    }
    if (lane == 0 && grp < ngrp) flags[grp >> 5] = 0u;       // pass 2 sets the bits of the flagged groups
}

// K0b pass 2: the deferred groups, one per thread (grid-stride over the work list)
__global__ void codes_worklist_kernel(Geom g, const uint8_t* __restrict__ vbyte, uint8_t* __restrict__ link,
                                      uint32_t* __restrict__ wcode, uint32_t* __restrict__ flags,
                                      uint32_t* __restrict__ tflags, const uint32_t* __restrict__ worklist,
                                      const unsigned int* __restrict__ work_count)
{
    const unsigned int n = *work_count;
    for (unsigned int w = blockIdx.x * blockDim.x + threadIdx.x; w < n; w += gridDim.x * blockDim.x) {
        const long long grp = worklist[w];
        const long long base = grp << 2;
        const int i0 = (int)(base % g.px);
        const long long row = base / g.px;
        const int j = (int)(row % g.ny), k = (int)(row / g.ny);
        if (decode_group(g, vbyte, link, wcode, base, i0, j, k)) {
            atomicOr(&flags[grp >> 5], 1u << (unsigned)(grp & 31));
            const int tile = (j / g.tby) * g.ntx + (i0 / g.tbx);
            atomicOr(&tflags[(size_t)tile * g.twords + (k >> 5)], 1u << (k & 31));
        }
    }
}

__device__ __forceinline__ void source_finalize(Scalars* sc, double n2)
{
    sc->normS2 = n2;
    sc->thresh2 = (0.1 * sc->tol) * (0.1 * sc->tol) * n2;
    sc->tol2S = sc->tol * sc->tol * n2;
    if (!(n2 > 0.0)) {                 // zero (or NaN) source: P = 0, no iterations (A4)
        sc->outer_go = 0; sc->inner_go = 0;
        if (!isfinite(n2)) sc->status = ST_BREAKDOWN;
    }
}

// ------------------------------------------------------------------------------------------------ K1 source
// S_C = - sum_d v(C+d) sgn(d) (Delta_a t_a / 2) (g_a(C+d) + g_a(C))     (Eq. 9 :100, w^{n+1}+w^n = t_a)
template <typename T>
__global__ void __launch_bounds__(256)
source_kernel(Geom g, const T* __restrict__ gx, const T* __restrict__ gy, const T* __restrict__ gz,
              const uint8_t* __restrict__ link, Coef<T> K, T* __restrict__ S, Scalars* sc, double* partial)
{
    __shared__ double red[8];
    __shared__ int is_last;
    // grid-stride: a few thousand CTAs (one ticket atomic each), every thread walks cells a whole grid apart
    double sq = 0.0;
    for (long long pid = (long long)blockIdx.x * blockDim.x + threadIdx.x; pid < g.npad;
         pid += (long long)gridDim.x * blockDim.x) {
        int i;
        long long row;
        split_pid(g, pid, i, row);
        T s = T(0);
        const uint32_t l = link[pid];
        if (l & LINK_VALID) {
            const long long u = row * g.nx + i;
            const long long sy = g.nx, sz = (long long)g.nx * g.ny;
            const T cx = gx[u], cy = gy[u];
            if (l & 1u) s -= K.hs[0] * (gx[u + 1] + cx);
            if (l & 2u) s += K.hs[0] * (gx[u - 1] + cx);
            if (l & 4u) s -= K.hs[1] * (gy[u + sy] + cy);
            if (l & 8u) s += K.hs[1] * (gy[u - sy] + cy);
            if (l & 48u) {
                const T cz = gz[u];
                if (l & 16u) s -= K.hs[2] * (gz[u + sz] + cz);
                if (l & 32u) s += K.hs[2] * (gz[u - sz] + cz);
            }
        }
        S[pid] = s;
        if (g.kz0 > 0 || g.kz1 < g.nz) {                 // a slab counts the planes it owns
            const int k = (int)(row / g.ny);
            if (k < g.kz0 || k >= g.kz1) s = T(0);
        }
        sq += (double)s * (double)s;
    }
    sq = warp_sum(sq);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sq;
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
            double n2 = 0.0;
            for (int w = 0; w < 8; ++w) n2 += red[w];
            sc->ticket[3] = 0;
            if (sc->defer) sc->red_out[0] = n2; else source_finalize(sc, n2);
        }
    }
}

// ------------------------------------------------------------------------------------------------ K7 finalize
template <typename T>
__global__ void finalize_kernel(Geom g, const double* P0, const double* P1, const Scalars* sc,
                                const uint8_t* __restrict__ link, T* __restrict__ out, double* __restrict__ out64)
{
    const double* __restrict__ P = (sc->n & 1) ? P0 : P1;      // the last K2 wrote Pbuf[(n & 1) ^ 1]
    long long u = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    long long nuser = (long long)g.nx * g.ny * g.nz;
    if (u == 0 && sc->status_out != nullptr) *sc->status_out = sc->status;
    if (u >= nuser) return;
    int i;
    long long row;
    if (nuser < (1LL << 31)) {
        const unsigned int r = (unsigned int)u / (unsigned int)g.nx;
        i = (int)((unsigned int)u - r * (unsigned int)g.nx);
        row = r;
    } else {
        i = (int)(u % g.nx);
        row = u / g.nx;
    }
    const long long pid = row * g.px + i;
    const bool ok = (link[pid] & LINK_VALID) != 0;
    out[u] = ok ? (T)P[pid] : (T)nan("");
    if (out64 != nullptr) out64[u] = ok ? P[pid] : nan("");      // the fp64 master pressure itself (omni_options::d_P64_out)
}

// ------------------------------------------------------------------------------------------------ K0a / K1 / K7, four cells per thread
// The one-cell-per-thread kernels above leave the memory system at 30-40 % of its bandwidth (few bytes in flight per
// thread, an index division per cell, neighbour loads that wait for the link byte).  When the caller's rows are whole
// 16-byte chunks (nx % 4 == 0, 16-byte aligned arrays) these variants take one 4-cell chunk per thread: vector loads,
// (x, y, plane) from the launch indices, neighbour chunks loaded by POSITION before the link bits select the terms.
// Same arithmetic per cell, same order.
constexpr int SETUP_BX = 64, SETUP_BY = 4;

template <typename T>
__global__ void __launch_bounds__(SETUP_BX * SETUP_BY)
validity4_kernel(Geom g, const T* __restrict__ gx, const T* __restrict__ gy, const T* __restrict__ gz,
                 const uint8_t* __restrict__ mask, uint8_t* __restrict__ vbyte)
{
    const int i0 = (blockIdx.x * SETUP_BX + threadIdx.x) * 4, j = blockIdx.y * SETUP_BY + threadIdx.y, k = blockIdx.z;
    if (i0 >= g.px || j >= g.ny) return;
    const long long pid = i0 + (long long)g.px * (j + (long long)g.ny * k);
    uint32_t ok = 0;
    if (i0 < g.nx) {
        const long long u = i0 + (long long)g.nx * (j + (long long)g.ny * k);
        uint32_t m = 0x01010101u;
        if (mask != nullptr) m = *reinterpret_cast<const uint32_t*>(mask + (g.batch ? i0 + (long long)g.nx * j : u));
        T a[4], b[4], c[4];
        zero_chunk<T, 4>(a); zero_chunk<T, 4>(b); zero_chunk<T, 4>(c);
        if (gx != nullptr) {
            ld_chunk<T, 4>(gx + u, a);
            ld_chunk<T, 4>(gy + u, b);
            if (g.naxes == 3) ld_chunk<T, 4>(gz + u, c);
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            uint32_t v = ((m >> (8 * q)) & 0xffu) != 0;
            if (isnan(a[q]) || isnan(b[q]) || isnan(c[q])) v = 0;
            ok |= v << (8 * q);
        }
    }
    *reinterpret_cast<uint32_t*>(vbyte + pid) = ok;
}

// K1: blocks stride over (4-row group, plane) items, threads over the chunks of a row; one partial per block as in
// source_kernel (same ticket, same finalize)
template <typename T>
__global__ void __launch_bounds__(SETUP_BX * SETUP_BY)
source4_kernel(Geom g, const T* __restrict__ gx, const T* __restrict__ gy, const T* __restrict__ gz,
               const uint8_t* __restrict__ link, Coef<T> K, T* __restrict__ S, Scalars* sc, double* partial)
{
    __shared__ double red[SETUP_BX * SETUP_BY / 32];
    __shared__ int is_last;
    const int nyb = (g.ny + SETUP_BY - 1) / SETUP_BY;
    const long long items = (long long)nyb * g.nz;
    const long long sy = g.nx, sz = (long long)g.nx * g.ny;
    double sq = 0.0;
    for (long long w = blockIdx.x; w < items; w += gridDim.x) {
        const int k = (int)(w / nyb), j = (int)(w - (long long)k * nyb) * SETUP_BY + threadIdx.y;
        if (j >= g.ny) continue;
        const bool own = (k >= g.kz0 && k < g.kz1);                 // a slab counts the planes it owns
        for (int i0 = threadIdx.x * 4; i0 < g.px; i0 += SETUP_BX * 4) {
            const long long pid = i0 + (long long)g.px * (j + (long long)g.ny * k);
            T s[4];
            zero_chunk<T, 4>(s);
            const uint32_t lw = *reinterpret_cast<const uint32_t*>(link + pid);
            if (lw & 0x40404040u) {                                  // (implies i0 < nx)
                const long long u = i0 + (long long)g.nx * (j + (long long)g.ny * k);
                T xc[4], yc[4], yn[4], ys[4], zc[4], zf[4], zb[4];
                ld_chunk<T, 4>(gx + u, xc);
                ld_chunk<T, 4>(gy + u, yc);
                zero_chunk<T, 4>(yn); zero_chunk<T, 4>(ys); zero_chunk<T, 4>(zc); zero_chunk<T, 4>(zf); zero_chunk<T, 4>(zb);
                if (j + 1 < g.ny) ld_chunk<T, 4>(gy + u + sy, yn);
                if (j > 0) ld_chunk<T, 4>(gy + u - sy, ys);
                if (g.naxes == 3) {
                    ld_chunk<T, 4>(gz + u, zc);
                    if (k + 1 < g.nz) ld_chunk<T, 4>(gz + u + sz, zf);
                    if (k > 0) ld_chunk<T, 4>(gz + u - sz, zb);
                }
                const T xl = (i0 > 0) ? gx[u - 1] : T(0), xr = (i0 + 4 < g.nx) ? gx[u + 4] : T(0);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const uint32_t l = (lw >> (8 * q)) & 0xffu;
                    if (!(l & LINK_VALID)) continue;
                    const T e = (q == 3) ? xr : xc[q < 3 ? q + 1 : 3], wv = (q == 0) ? xl : xc[q > 0 ? q - 1 : 0];
                    T v = T(0);
                    if (l & 1u) v -= K.hs[0] * (e + xc[q]);
                    if (l & 2u) v += K.hs[0] * (wv + xc[q]);
                    if (l & 4u) v -= K.hs[1] * (yn[q] + yc[q]);
                    if (l & 8u) v += K.hs[1] * (ys[q] + yc[q]);
                    if (l & 16u) v -= K.hs[2] * (zf[q] + zc[q]);
                    if (l & 32u) v += K.hs[2] * (zb[q] + zc[q]);
                    s[q] = v;
                }
            }
            st_chunk<T, 4>(S + pid, s);
            if (own) {
#pragma unroll
                for (int q = 0; q < 4; ++q) sq += (double)s[q] * (double)s[q];
            }
        }
    }
    const int tid = threadIdx.y * SETUP_BX + threadIdx.x;
    sq = warp_sum(sq);
    if ((tid & 31) == 0) red[tid >> 5] = sq;
    __syncthreads();
    if (tid == 0) {
        double t = 0.0;
        for (int w = 0; w < SETUP_BX * SETUP_BY / 32; ++w) t += red[w];
        partial[blockIdx.x] = t;
        __threadfence();
        is_last = (atomicAdd(&sc->ticket[3], 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        double t = 0.0;
        for (unsigned int b = tid; b < gridDim.x; b += SETUP_BX * SETUP_BY) t += __ldcg(&partial[b]);
        t = warp_sum(t);
        __syncthreads();
        if ((tid & 31) == 0) red[tid >> 5] = t;
        __syncthreads();
        if (tid == 0) {
            double n2 = 0.0;
            for (int w = 0; w < SETUP_BX * SETUP_BY / 32; ++w) n2 += red[w];
            sc->ticket[3] = 0;
            if (sc->defer) sc->red_out[0] = n2; else source_finalize(sc, n2);
        }
    }
}

template <typename T>
__global__ void __launch_bounds__(SETUP_BX * SETUP_BY)
finalize4_kernel(Geom g, const double* P0, const double* P1, const Scalars* sc, const uint8_t* __restrict__ link,
                 T* __restrict__ out, double* __restrict__ out64)
{
    const double* __restrict__ P = (sc->n & 1) ? P0 : P1;      // the last K2 wrote Pbuf[(n & 1) ^ 1]
    const int i0 = (blockIdx.x * SETUP_BX + threadIdx.x) * 4, j = blockIdx.y * SETUP_BY + threadIdx.y, k = blockIdx.z;
    if (i0 == 0 && j == 0 && k == 0 && sc->status_out != nullptr) *sc->status_out = sc->status;
    if (i0 >= g.nx || j >= g.ny) return;
    const long long pid = i0 + (long long)g.px * (j + (long long)g.ny * k);
    const long long u = i0 + (long long)g.nx * (j + (long long)g.ny * k);
    const uint32_t lw = *reinterpret_cast<const uint32_t*>(link + pid);
    double p[4], o64[4];
    ld_chunk<double, 4>(P + pid, p);
    T o[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const bool ok = ((lw >> (8 * q)) & LINK_VALID) != 0;
        o[q] = ok ? (T)p[q] : (T)nan("");
        o64[q] = ok ? p[q] : nan("");
    }
    st_chunk<T, 4>(out + u, o);
    if (out64 != nullptr) st_chunk<double, 4>(out64 + u, o64);
}

// copies between the caller's unpadded layout and the padded internal layout (step entry points only)
template <typename TI, typename TO>
__global__ void pad_copy_kernel(Geom g, const TI* __restrict__ in, TO* __restrict__ out, int to_padded,
                                const uint8_t* __restrict__ link)
{
    long long pid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (pid >= g.npad) return;
    int i;
    long long row;
    split_pid(g, pid, i, row);
    long long u = row * g.nx + i;
    if (to_padded) out[pid] = (i < g.nx && (link[pid] & LINK_VALID)) ? (TO)in[u] : TO(0);
    else if (i < g.nx) out[u] = (TO)in[pid];
}

// ------------------------------------------------------------------------------------------------ cascade (first guess)
// omni_solve_cascade: grids coarsened by 2 along every axis longer than one cell.  A coarse cell is valid iff one of
// its children is (in the box, mask != 0, no NaN component); its gradient is the mean over the valid children.
// Caller layout (unpadded) on both sides; one thread per coarse cell.
template <typename T>
__global__ void restrict_kernel(int nx, int ny, int nz, int fx, int fy, int fz, int cx, int cy, int cz, int ncomp,
                                const T* __restrict__ gx, const T* __restrict__ gy, const T* __restrict__ gz,
                                const uint8_t* __restrict__ mask, T* __restrict__ ox, T* __restrict__ oy,
                                T* __restrict__ oz, uint8_t* __restrict__ omask)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long nc = (long long)cx * cy * cz;
    if (c >= nc) return;
    const int ci = (int)(c % cx), cj = (int)((c / cx) % cy), ck = (int)(c / ((long long)cx * cy));
    T sx = T(0), sy = T(0), sz = T(0);
    int cnt = 0;
    for (int dk = 0; dk < fz; ++dk)
        for (int dj = 0; dj < fy; ++dj)
            for (int di = 0; di < fx; ++di) {
                const int i = ci * fx + di, j = cj * fy + dj, k = ck * fz + dk;
                if (i >= nx || j >= ny || k >= nz) continue;
                const long long u = i + (long long)nx * (j + (long long)ny * k);
                if (mask != nullptr && mask[u] == 0) continue;
                const T a = gx[u], b = gy[u], e = (ncomp == 3) ? gz[u] : T(0);
                if (isnan(a) || isnan(b) || isnan(e)) continue;
                sx += a; sy += b; sz += e; ++cnt;
            }
    const T inv = cnt ? T(1) / T(cnt) : T(0);
    ox[c] = sx * inv; oy[c] = sy * inv;
    if (ncomp == 3) oz[c] = sz * inv;
    omask[c] = cnt ? 1 : 0;
}

// first guess of a level: the parent's pressure (0 where the parent is missing); one thread per fine cell
template <typename T>
__global__ void prolong_kernel(int nx, int ny, int nz, int fx, int fy, int fz, int cx, int cy,
                               const T* __restrict__ Pc, T* __restrict__ Pf)
{
    const long long u = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long n = (long long)nx * ny * nz;
    if (u >= n) return;
    const int i = (int)(u % nx), j = (int)((u / nx) % ny), k = (int)(u / ((long long)nx * ny));
    const T v = Pc[(i / fx) + (long long)cx * ((j / fy) + (long long)cy * (k / fz))];
    Pf[u] = isnan(v) ? T(0) : v;
}

// ------------------------------------------------------------------------------------------------ NEXT-4: f(u), Eq. 1
// g = -rho (du/dt + (u . grad) u) + mu lap u with second-order central differences; a cell whose
// 2*naxes-neighbour stencil touches a missing cell (outside the box, mask == 0, NaN velocity) gets NaN in every
// component (reading R-V1), which the solver treats as missing (Eq. 13 :176).  Caller layout
// (unpadded, x fastest); one thread per cell; at* = optional local accelerations (nullptr = steady).
template <typename T>
__global__ void velocity_source_kernel(int nx, int ny, int nz, int ncomp, T idx2, T idy2, T idz2, T ihx, T ihy, T ihz,
                                       T rho, T mu, const T* __restrict__ u, const T* __restrict__ v,
                                       const T* __restrict__ w, const T* __restrict__ atx, const T* __restrict__ aty,
                                       const T* __restrict__ atz, const uint8_t* __restrict__ mask,
                                       T* __restrict__ gx, T* __restrict__ gy, T* __restrict__ gz)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long n = (long long)nx * ny * nz;
    if (c >= n) return;
    const int i = (int)(c % nx), j = (int)((c / nx) % ny), k = (int)(c / ((long long)nx * ny));
    const long long sy = nx, sz = (long long)nx * ny;
    auto ok = [&](long long q) {
        if (mask != nullptr && mask[q] == 0) return false;
        if (isnan(u[q]) || isnan(v[q])) return false;
        return !(ncomp == 3 && isnan(w[q]));
    };
    bool good = ok(c) && i > 0 && i < nx - 1 && j > 0 && j < ny - 1 && (ncomp == 2 || (k > 0 && k < nz - 1));
    if (good) good = ok(c - 1) && ok(c + 1) && ok(c - sy) && ok(c + sy) && (ncomp == 2 || (ok(c - sz) && ok(c + sz)));
    const T qnan = (T)nan("");
    if (!good) {
        gx[c] = qnan; gy[c] = qnan;
        if (ncomp == 3) gz[c] = qnan;
        return;
    }
    const T uc = u[c], vc = v[c], wc = (ncomp == 3) ? w[c] : T(0);
    auto term = [&](const T* __restrict__ f, const T* __restrict__ at) {
        const T fc = f[c];
        T conv = uc * ((f[c + 1] - f[c - 1]) * ihx) + vc * ((f[c + sy] - f[c - sy]) * ihy);
        T lap = (f[c + 1] - T(2) * fc + f[c - 1]) * idx2 + (f[c + sy] - T(2) * fc + f[c - sy]) * idy2;
        if (ncomp == 3) {
            conv += wc * ((f[c + sz] - f[c - sz]) * ihz);
            lap += (f[c + sz] - T(2) * fc + f[c - sz]) * idz2;
        }
        return -rho * ((at != nullptr ? at[c] : T(0)) + conv) + mu * lap;
    };
    gx[c] = term(u, atx);
    gy[c] = term(v, aty);
    if (ncomp == 3) gz[c] = term(w, atz);
}

// ------------------------------------------------------------------------------------------------ RANS source fields
// Eq. 42: f_i = -rho (ubar_j d_j ubar_i + d_j R_ij)                                  (COMPRESSIBLE = false)
// Eq. 43-44 (:540-545):  theta = T/T_inf = 1 + (gamma-1)/2 M_inf^2 (1 - V^2/V_inf^2), uu_ij = ubar_i ubar_j + R_ij,
//                        (delta_ij + uu_ij/(R T)) g_j = -(1/(R T)) (d_j uu_ij - uu_ij/T d_j T)       (COMPRESSIBLE = true)
// solved cell by cell for g = grad ln(P/P_inf) (Gaussian elimination with partial pivoting, 2x2 / 3x3).
// Second-order central differences, caller layout, one thread per cell; a cell whose stencil touches a missing cell
// (outside the box, mask == 0, NaN in any input) gets NaN in every component (reading R-V1).
template <typename T>
struct RansArgs {
    const T* u[3];            // mean velocity (u[2] null in 2D)
    const T* R[6];            // Reynolds stresses: 2D xx, yy, xy; 3D xx, yy, zz, xy, xz, yz (all null: none)
    const uint8_t* mask;
    T* g[3];
    T ih[3];                  // 1 / (2 h_a)
    T rho;                    // Eq. 42
    T cth, inv_v2, rt_inf;    // Eq. 43-44: (gamma-1)/2 M_inf^2, 1 / V_inf^2, R T_inf
    int has_R;
};

__host__ __device__ __forceinline__ int stress_slot(int nd, int i, int j)
{
    if (i == j) return i;
    if (nd == 2) return 2;
    return i + j + 2;         // (0,1) -> 3, (0,2) -> 4, (1,2) -> 5
}

template <typename T, bool COMPRESSIBLE>
__global__ void rans_source_kernel(int nx, int ny, int nz, int nd, const RansArgs<T> a)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long n = (long long)nx * ny * nz;
    if (c >= n) return;
    const int i = (int)(c % nx), j = (int)((c / nx) % ny), k = (int)(c / ((long long)nx * ny));
    const long long st[3] = { 1, nx, (long long)nx * ny };
    const int nR = (nd == 2) ? 3 : 6;
    auto ok = [&](long long q) {
        if (a.mask != nullptr && a.mask[q] == 0) return false;
        for (int m = 0; m < nd; ++m)
            if (isnan(a.u[m][q])) return false;
        if (a.has_R)
            for (int m = 0; m < nR; ++m)
                if (isnan(a.R[m][q])) return false;
        return true;
    };
    bool good = ok(c) && i > 0 && i < nx - 1 && j > 0 && j < ny - 1 && (nd == 2 || (k > 0 && k < nz - 1));
    if (good)
        for (int m = 0; m < nd; ++m) good = good && ok(c - st[m]) && ok(c + st[m]);
    if (!good) {
        const T qnan = (T)nan("");
        for (int m = 0; m < nd; ++m) a.g[m][c] = qnan;
        return;
    }
    T uc[3] = { T(0), T(0), T(0) };
    for (int m = 0; m < nd; ++m) uc[m] = a.u[m][c];
    if constexpr (!COMPRESSIBLE) {
        for (int p = 0; p < nd; ++p) {
            T conv = T(0), div = T(0);
            for (int q = 0; q < nd; ++q) {
                conv += uc[q] * ((a.u[p][c + st[q]] - a.u[p][c - st[q]]) * a.ih[q]);
                if (a.has_R) {
                    const T* __restrict__ Rpq = a.R[stress_slot(nd, p < q ? p : q, p < q ? q : p)];
                    div += (Rpq[c + st[q]] - Rpq[c - st[q]]) * a.ih[q];
                }
            }
            a.g[p][c] = -a.rho * (conv + div);
        }
    } else {
        auto theta_at = [&](long long q) {
            T v2 = T(0);
            for (int m = 0; m < nd; ++m) v2 += a.u[m][q] * a.u[m][q];
            return T(1) + a.cth * (T(1) - v2 * a.inv_v2);
        };
        auto uu_at = [&](int p, int q, long long cell) {
            T v = a.u[p][cell] * a.u[q][cell];
            if (a.has_R) v += a.R[stress_slot(nd, p < q ? p : q, p < q ? q : p)][cell];
            return v;
        };
        const T th = theta_at(c);
        const T rt = a.rt_inf * th;
        T dth[3] = { T(0), T(0), T(0) };
        for (int q = 0; q < nd; ++q) dth[q] = (theta_at(c + st[q]) - theta_at(c - st[q])) * a.ih[q];
        T A[3][4];
        for (int p = 0; p < 3; ++p)
            for (int q = 0; q < 4; ++q) A[p][q] = (p == q) ? T(1) : T(0);
        for (int p = 0; p < nd; ++p) {
            T b = T(0);
            for (int q = 0; q < nd; ++q) {
                const T uu = uu_at(p, q, c);
                A[p][q] = ((p == q) ? T(1) : T(0)) + uu / rt;
                const T duu = (uu_at(p, q, c + st[q]) - uu_at(p, q, c - st[q])) * a.ih[q];
                b += -(T(1) / rt) * (duu - uu / th * dth[q]);
            }
            A[p][3] = b;
        }
        // Gaussian elimination with partial pivoting on the nd x nd system (rows beyond nd are identity)
#pragma unroll
        for (int col = 0; col < 3; ++col) {
            int piv = col;
            for (int r = col + 1; r < 3; ++r)
                if (fabs(A[r][col]) > fabs(A[piv][col])) piv = r;
            for (int q = 0; q < 4; ++q) { const T t = A[col][q]; A[col][q] = A[piv][q]; A[piv][q] = t; }
            for (int r = col + 1; r < 3; ++r) {
                const T f = A[r][col] / A[col][col];
                for (int q = col; q < 4; ++q) A[r][q] -= f * A[col][q];
            }
        }
        T x[3];
        for (int r = 2; r >= 0; --r) {
            T s = A[r][3];
            for (int q = r + 1; q < 3; ++q) s -= A[r][q] * x[q];
            x[r] = s / A[r][r];
        }
        for (int m = 0; m < nd; ++m) a.g[m][c] = x[m];
    }
}

}  // namespace omni
