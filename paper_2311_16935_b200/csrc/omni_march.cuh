// omni_march.cuh -- the cp.async z-marching tile engine and the K2 operator (outer boundary update).
// (K3 / K4, the CG inner loop, run on the TMA + mbarrier pipeline of omni_tma.cuh.)
//
// A CTA owns a column of the grid: W = 32*V cells wide (1 KB of the widest streamed array), TYR-2 output rows (+2 halo
// rows), zlen planes (+1 halo plane on each side).  Every thread owns one 32-byte chunk per streamed array and plane.
//   * global -> shared: each thread copies ITS chunks of the planes ahead with cp.async (LDGSTS, zero-fill outside the
//     box) into a D-deep ring of private shared-memory slots, so (D-1) planes x all streamed arrays are in flight per
//     SM without holding registers; nobody else reads those slots, so the ring needs no barrier.
//   * registers: stencil input of planes k-1, k, k+1 for the own chunk (z neighbours).
//   * y neighbours: the current plane is published to a double-buffered exchange tile (one __syncthreads per plane);
//     x neighbours: warp shuffles, plus two scalar halo cells per row copied with the ring.
//   * reduction: fp64 per-thread partials -> warp shuffle -> CTA -> fixed slot; the last-arriving CTA (atomic ticket)
//     adds the slots in slot order and updates the device-resident loop scalars (deterministic; no host sync).
#pragma once
#include "omni_kernels.cuh"

namespace omni {

__device__ __forceinline__ void set_cond(const CondHandles& h, int outer, int inner)
{
#if defined(__CUDA_ARCH__)
    if (h.use) {
        if (outer >= 0) cudaGraphSetConditional((cudaGraphConditionalHandle)h.h_outer, (unsigned)outer);
        if (inner >= 0) cudaGraphSetConditional((cudaGraphConditionalHandle)h.h_inner, (unsigned)inner);
    }
#endif
}

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, bool ok)
{
    const int sz = ok ? 16 : 0;      // src-size 0: nothing is read, the 16 destination bytes are zero-filled
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
template <int B>
__device__ __forceinline__ void cp_async_small(uint32_t dst, const void* src, bool ok)
{
    const int sz = ok ? B : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2, %3;" ::"r"(dst), "l"(src), "n"(B), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// one ring stage seen by one thread: PIECES 16-byte pieces (piece q of thread t at (q*NTHR + t)*16: conflict-free
// LDS.128), then 4 halo slots of 8 bytes per row
template <int NTHR, int PIECES>
struct StageW {
    uint32_t base, halo;     // shared-space addresses
    int tid;
    template <typename T, int NP>
    __device__ __forceinline__ void put(int q0, const T* src, long long idx, bool ok) const
    {
        constexpr int EPP = 16 / (int)sizeof(T);     // elements per piece
#pragma unroll
        for (int i = 0; i < NP; ++i)
            cp_async16(base + (uint32_t)(((q0 + i) * NTHR + tid) * 16), ok ? (const void*)(src + idx + i * EPP) : (const void*)src, ok);
    }
    template <typename T>
    __device__ __forceinline__ void put_halo(int slot, const T* src, long long idx, bool ok) const
    {
        cp_async_small<(int)sizeof(T)>(halo + (uint32_t)(slot * 8), ok ? (const void*)(src + idx) : (const void*)src, ok);
    }
};
template <int NTHR, int PIECES>
struct StageR {
    const char* base;
    const char* halo;
    int tid;
    template <typename T, int V>
    __device__ __forceinline__ void get(int q0, T (&v)[V]) const
    {
        constexpr int NP = V * (int)sizeof(T) / 16;
        uint4 u[NP];
#pragma unroll
        for (int i = 0; i < NP; ++i) u[i] = *reinterpret_cast<const uint4*>(base + ((q0 + i) * NTHR + tid) * 16);
        memcpy(v, u, sizeof(u));
    }
    template <typename T>
    __device__ __forceinline__ T get_halo(int slot) const { return *reinterpret_cast<const T*>(halo + slot * 8); }
};

template <class Op>
struct MarchSmem {
    static constexpr int NTHR = 32 * Op::TYR;
    static constexpr int STAGE_BYTES = Op::PIECES * NTHR * 16 + Op::TYR * 4 * 8;
    static constexpr int XCH_BYTES = 2 * Op::TYR * 32 * Op::V * (int)sizeof(typename Op::VT);
    static constexpr int TOTAL = Op::D * STAGE_BYTES + XCH_BYTES;
};

template <class Op>
__global__ void __launch_bounds__(32 * Op::TYR, Op::MINB)
march_kernel(const Geom g, const int zlen, const typename Op::Args a)
{
    using VT = typename Op::VT;
    constexpr int V = Op::V, TYR = Op::TYR, TYO = TYR - 2, W = 32 * V, NACC = Op::NACC, D = Op::D;
    constexpr int NTHR = 32 * TYR, PIECES = Op::PIECES;
    using SM = MarchSmem<Op>;
    extern __shared__ __align__(16) char smem[];
    __shared__ double red[NACC][TYR];
    __shared__ int is_last;

    if (!Op::active(a)) {       // uniform: the device-side loop state says this launch has nothing to do
        if (threadIdx.x == 0 && threadIdx.y == 0 && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) Op::idle(a);
        return;
    }

    const int lane = threadIdx.x, ty = threadIdx.y, tid = ty * 32 + lane;
    const int x = blockIdx.x * W + lane * V;
    const int j = blockIdx.y * TYO + ty - 1;
    const int k0 = blockIdx.z * zlen;
    const int k1 = min(g.nz, k0 + zlen);
    const bool ldok = (x < g.px) && (j >= 0) && (j < g.ny);
    const bool outrow = ldok && (ty >= 1) && (ty <= TYO);
    const bool lok = ldok && (lane == 0) && (x > 0);
    const bool rok = ldok && (lane == 31) && (x + V < g.px);
    const long long rowbase = (long long)j * g.px + x;

    VT(*xch)[TYR][W] = reinterpret_cast<VT(*)[TYR][W]>(smem + D * SM::STAGE_BYTES);
    const uint32_t smem_s = (uint32_t)__cvta_generic_to_shared(smem);

    const typename Op::Ctx ctx(a);
    const typename Op::TC tc = Op::thread_init(g, x, j);

    // event c consumes the main arrays of plane c and the extra arrays of plane c-1; its data sits in ring slot
    // (c - k0 + 1) % D.  Planes outside [0, nz) and the far side of the segment's halo planes are zero-filled.
    auto issue = [&](int c, int slot, long long off) {      // off = rowbase + c * pplane
        StageW<NTHR, PIECES> st{ smem_s + (uint32_t)(slot * SM::STAGE_BYTES),
                                 smem_s + (uint32_t)(slot * SM::STAGE_BYTES + PIECES * NTHR * 16 + ty * 32), tid };
        const bool pin = (c >= 0) && (c < g.nz) && (c <= k1);
        const bool ein = (c - 1 >= k0) && (c - 1 < k1);
        Op::issue(a, ctx, st, off, ldok && pin, lok && pin, rok && pin, off - g.pplane, outrow && ein);
        cp_async_commit();
    };

    VT vm[V], vc[V], vn_[V], hlc = VT(0), hrc = VT(0), hln, hrn;
    typename Op::Extra ex;
    double acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = 0.0;
    zero_chunk<VT, V>(vm);
    zero_chunk<VT, V>(vc);

    long long off = rowbase + (long long)(k0 - 1) * g.pplane;     // offset of plane c
#pragma unroll
    for (int s = 0; s < D; ++s) issue(k0 - 1 + s, s, off + s * g.pplane);
    const long long doff = (long long)D * g.pplane;

    // flag word of the plane emitted at the NEXT event, fetched one event early so that its latency is hidden
    uint32_t fw_next = 0, fw_cur = 0;
    int slot = 0, buf = 0;
    for (int c = k0 - 1; c <= k1; ++c) {
        cp_async_wait<D - 1>();
        {
            StageR<NTHR, PIECES> sr{ smem + slot * SM::STAGE_BYTES,
                                     smem + slot * SM::STAGE_BYTES + PIECES * NTHR * 16 + ty * 32, tid };
            Op::consume(a, ctx, sr, vn_, hln, hrn, ex);
        }
        issue(c + D, slot, off + doff);
        fw_cur = fw_next;
        if (outrow && c >= k0 && c < k1) fw_next = a.flags[(off >> 2) >> 5];     // plane c is emitted at event c+1
        if (c >= k0 + 1) {           // emit plane c-1: vm = plane c-2, vc = plane c-1, vn_ = plane c
            const long long idx = off - g.pplane;
            st_chunk<VT, V>(&xch[buf][ty][lane * V], vc);
            __syncthreads();
            VT xl = __shfl_up_sync(0xffffffffu, vc[V - 1], 1);
            VT xr = __shfl_down_sync(0xffffffffu, vc[0], 1);
            if (lane == 0) xl = hlc;
            if (lane == 31) xr = hrc;
            if (outrow) {
                VT vN[V], vS[V];
                ld_chunk<VT, V>(&xch[buf][ty + 1][lane * V], vN);
                ld_chunk<VT, V>(&xch[buf][ty - 1][lane * V], vS);
                const uint32_t fb = (fw_cur >> (unsigned)((idx >> 2) & 31)) & ((1u << (V / 4)) - 1u);
                Op::emit(a, ctx, idx, c - 1, vm, vc, vn_, vN, vS, xl, xr, ex, fb, tc, acc);
            }
            buf ^= 1;
        }
#pragma unroll
        for (int i = 0; i < V; ++i) { vm[i] = vc[i]; vc[i] = vn_[i]; }
        hlc = hln; hrc = hrn;
        off += g.pplane;
        slot = (slot + 1 == D) ? 0 : slot + 1;
    }
    cp_async_wait<0>();

    // deterministic grid reduction: CTA partial -> fixed slot -> last-arriving CTA sums all slots in slot order
    const unsigned int nblk = gridDim.x * gridDim.y * gridDim.z;
    const unsigned int bid = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
#pragma unroll
    for (int i = 0; i < NACC; ++i) {
        double s = warp_sum(acc[i]);
        if (lane == 0) red[i][ty] = s;
    }
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < NACC; ++i) {
            double s = 0.0;
            for (int w = 0; w < TYR; ++w) s += red[i][w];
            a.partial[(size_t)i * nblk + bid] = s;
        }
        __threadfence();
        unsigned int t = atomicAdd(&a.sc->ticket[Op::TICKET], 1u);
        is_last = (t == nblk - 1);
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        double tot[NACC];
#pragma unroll
        for (int i = 0; i < NACC; ++i) {
            double s = 0.0;
            for (unsigned int b = tid; b < nblk; b += NTHR) s += __ldcg(&a.partial[(size_t)i * nblk + b]);
            s = warp_sum(s);
            __syncthreads();
            if (lane == 0) red[i][ty] = s;
            __syncthreads();
            s = 0.0;
            for (int w = 0; w < TYR; ++w) s += red[i][w];
            tot[i] = s;
        }
        if (tid == 0) {
            a.sc->ticket[Op::TICKET] = 0;
            Op::finalize(a, tot);
        }
    }
}

// ------------------------------------------------------------------------------------------------ K2
// outer boundary update (Eq. 12 collapsed): P <- P + delta; r0 = S - L P with
// (L P)_C = sum_d v(C+d) t_a (P_C - P_{C+d}) = ([W^{n+1}] - [W^n]) P; eps_R^2 ||S||^2 = ||r0||^2 (Eq. 41).
// P is always fp64 (master pressure, A9); delta, S, r are T.  P is double-buffered: neighbouring CTAs read
// P + delta in their halos, so the folded field goes to the other buffer (read Pbuf[n&1], write Pbuf[(n&1)^1]).
template <typename T, int TYR_, int D_, int MINB_>
struct OpK2 {
    using VT = double;
    enum { V = 4, TYR = TYR_, D = D_, MINB = MINB_, NACC = 2, TICKET = 2, NPT = 4 * sizeof(T) / 16, PIECES = 2 + 2 * NPT };
    struct Args {
        double* Pbuf[2]; const T* delta; const T* S; T* r; const uint8_t* link; const uint32_t* flags;
        double t[3]; Scalars* sc; double* partial; CondHandles cond;
        int fold_delta;   // 0: residual of P as given (omni_residual); 1: inside the solve
        int nz, fixz;     // box faces normal to z are not flagged either: their links are cleared per plane
    };
    struct Ctx {
        const double* Pin; double* Pout;
        __device__ Ctx(const Args& a) { int par = a.sc->n & 1; Pin = a.Pbuf[par]; Pout = a.Pbuf[par ^ 1]; }
    };
    struct Extra { T S[V]; };
    // thread constant: link bytes of an unflagged chunk (all six links, minus the box faces normal to x, pads invalid)
    using TC = uint32_t;
    __device__ static TC thread_init(const Geom& g, int x, int j)
    {
        uint32_t lk = 0;
#pragma unroll
        for (int i = 0; i < V; ++i) {
            const int gi = x + i;
            uint32_t l = 0x7fu;
            if (g.nz == 1) l &= ~48u;
            if (g.fix[0]) {
                if (gi == 0) l &= ~2u;
                if (gi == g.nx - 1) l &= ~1u;
                if (gi >= g.nx) l = 0;
            }
            if (g.fix[1]) {                      // box faces normal to y (rows are not flagged for them)
                if (j == 0) l &= ~8u;
                if (j == g.ny - 1) l &= ~4u;
            }
            lk |= l << (8 * i);
        }
        return lk;
    }
    __device__ static bool active(const Args& a) { return a.sc->outer_go != 0; }
    __device__ static void idle(const Args& a) { set_cond(a.cond, 0, 0); }
    template <class SW>
    __device__ static void issue(const Args& a, const Ctx& c, const SW& st, long long idx, bool ok, bool lok, bool rok,
                                 long long eidx, bool eok)
    {
        st.template put<double, 2>(0, c.Pin, idx, ok);
        st.template put<T, NPT>(2, a.delta, idx, ok);
        if (threadIdx.x == 0) { st.put_halo(0, c.Pin, idx - 1, lok); st.put_halo(1, a.delta, idx - 1, lok); }
        if (threadIdx.x == 31) { st.put_halo(2, c.Pin, idx + V, rok); st.put_halo(3, a.delta, idx + V, rok); }
        st.template put<T, NPT>(2 + NPT, a.S, eidx, eok);
    }
    template <class SR>
    __device__ static void consume(const Args&, const Ctx&, const SR& sr, double (&v)[V], double& hl, double& hr, Extra& e)
    {
        double P[V]; T d[V];
        sr.template get<double, V>(0, P);
        sr.template get<T, V>(2, d);
#pragma unroll
        for (int i = 0; i < V; ++i) v[i] = P[i] + (double)d[i];
        hl = hr = 0.0;
        if (threadIdx.x == 0) hl = sr.template get_halo<double>(0) + (double)sr.template get_halo<T>(1);
        if (threadIdx.x == 31) hr = sr.template get_halo<double>(2) + (double)sr.template get_halo<T>(3);
        sr.template get<T, V>(2 + NPT, e.S);
    }
    __device__ static void emit(const Args& a, const Ctx& c, long long idx, int kp, const double (&vm)[V], const double (&vc)[V],
                                const double (&vp)[V], const double (&vn)[V], const double (&vs)[V], double xl,
                                double xr, const Extra& e, uint32_t fb, const TC& lk_const, double (&acc)[2])
    {
        if (a.fold_delta) st_chunk<double, V>(c.Pout + idx, vc);
        uint32_t lk = lk_const;
        if (a.fixz) {
            if (kp == 0) lk &= ~0x20202020u;
            if (kp == a.nz - 1) lk &= ~0x10101010u;
        }
        if (fb) lk = *reinterpret_cast<const uint32_t*>(a.link + idx);
        T rn[V];
#pragma unroll
        for (int i = 0; i < V; ++i) {
            double w = (i == 0) ? xl : vc[i - 1];
            double ee = (i == V - 1) ? xr : vc[i + 1];
            uint32_t l = (lk >> (8 * i)) & 0xffu;
            double LP = 0.0;
            if (l & 1u) LP += a.t[0] * (vc[i] - ee);
            if (l & 2u) LP += a.t[0] * (vc[i] - w);
            if (l & 4u) LP += a.t[1] * (vc[i] - vn[i]);
            if (l & 8u) LP += a.t[1] * (vc[i] - vs[i]);
            if (l & 16u) LP += a.t[2] * (vc[i] - vp[i]);
            if (l & 32u) LP += a.t[2] * (vc[i] - vm[i]);
            double rr = (l & LINK_VALID) ? ((double)e.S[i] - LP) : 0.0;
            rn[i] = (T)rr;
            acc[0] += rr * rr;
            acc[1] += (double)rn[i] * (double)rn[i];
        }
        st_chunk<T, V>(a.r + idx, rn);
    }
    __device__ static void finalize(const Args& a, const double (&tot)[2])
    {
        Scalars* s = a.sc;
        s->epsR2 = tot[0];
        if (!a.fold_delta) return;
        if (!isfinite(tot[0])) {
            s->status = ST_BREAKDOWN; s->inner_go = 0; s->outer_go = 0;
            set_cond(a.cond, 0, 0);
            return;
        }
        if (tot[0] <= s->tol2S || s->n >= s->max_outer) {
            s->status = (tot[0] <= s->tol2S) ? ST_OK : ST_NOT_CONVERGED;
            s->inner_go = 0; s->outer_go = 0;
            set_cond(a.cond, 0, 0);
            return;
        }
        s->n += 1;
        s->k = 0;
        s->beta = 0.0;
        s->rho = tot[1];
        int go = (tot[1] > s->thresh2) && (tot[1] != 0.0) && (s->max_cg > 0);
        s->inner_go = go;
        set_cond(a.cond, 1, go);
    }
};

}  // namespace omni
