// omni_tma.cuh -- K3 / K4 on a TMA + mbarrier producer/consumer pipeline (sm_100a).
//
// A CTA owns a column of the grid: BX = 32*V cells (512 bytes) x BY rows x zlen planes.  One producer warp issues,
// per plane, a few cp.async.bulk.tensor (TMA) box loads -- the tile of every streamed array, the stencil input with
// its one-cell halo in x and y -- into a D-deep ring of shared-memory stages; out-of-box coordinates (box faces, the
// planes before/after the grid) are zero-filled by the TMA unit, so the kernels carry no bounds logic.  BY consumer
// warps (one row each, V cells per lane) wait on the stage's "full" mbarrier, read the centre / N / S chunks of plane
// c-1 and the own chunk of planes c-2 and c from the three resident stages (x neighbours by shuffle), evaluate the
// operator, store, and release the oldest stage through its "empty" mbarrier.  Warps only ever wait for data, never
// for each other: there is no CTA-wide barrier in the loop and no state carried in registers across planes.
// The grid reduction at the end is the deterministic fixed-slot + last-CTA scheme of omni_march.cuh.
#pragma once
#include <cuda.h>
#include <type_traits>
#include "omni_march.cuh"

namespace omni {

// ------------------------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    // labels are local to the PTX block scope, so the loop can be inlined any number of times
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_LOOP:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                 "@p bra WAIT_DONE;\n\tbra WAIT_LOOP;\n\tWAIT_DONE:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(dst), "l"((unsigned long long)map), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

// tensor maps of one solve (host-encoded, passed as a __grid_constant__ kernel parameter)
struct alignas(64) TmaSet {
    CUtensorMap r_h, p_h[2];     // boxes with halo: (BX + 2 HX) x (BY + 2) x 1
    CUtensorMap r_c, d_c;        // plain boxes: BX x BY x 1
};

template <typename T, int BY_>
struct TileGeom {
    static constexpr int V = 16 / (int)sizeof(T);          // cells per lane (one 16-byte piece)
    static constexpr int BX = 32 * V;                      // 512 bytes per row
    static constexpr int BY = BY_;
    static constexpr int HX = 16 / (int)sizeof(T);         // x halo in cells (16 bytes: TMA box rows are 16 B multiples)
    static constexpr int PITCH_H = (BX + 2 * HX) * (int)sizeof(T);       // 544 bytes
    static constexpr int TILE_H = ((BY + 2) * PITCH_H + 127) / 128 * 128;
    static constexpr int TILE_C = BY * BX * (int)sizeof(T);              // multiple of 512
    static constexpr int NTHR = 32 * (BY + 1);             // BY consumer warps + 1 producer warp
};

// explicit shared-space loads (generic LD through a computed pointer costs an address-space check and a longer
// scoreboard): addresses are 32-bit shared-window offsets
template <typename T, int V>
__device__ __forceinline__ void lds_chunk(uint32_t addr, T (&v)[V])
{
    static_assert(V * sizeof(T) == 16, "one 16-byte piece per lane");
    uint4 u;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(u.x), "=r"(u.y), "=r"(u.z), "=r"(u.w) : "r"(addr));
    memcpy(v, &u, 16);
}
__device__ __forceinline__ float lds_scalar(uint32_t addr, float)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ double lds_scalar(uint32_t addr, double)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}

template <class Op>
__global__ void __launch_bounds__(Op::TG::NTHR, Op::MINB)
tma_kernel(const Geom g, const int zlen, const typename Op::Args a, const __grid_constant__ TmaSet maps)
{
    using TG = typename Op::TG;
    using T = typename Op::VT;
    constexpr int V = TG::V, BX = TG::BX, BY = TG::BY, D = Op::D, NACC = 1;
    extern __shared__ __align__(128) char smem_raw[];
    __shared__ double red[BY + 1];
    __shared__ int is_last;
    __shared__ __align__(8) unsigned long long bars[2 * D];

    if (!Op::active(a)) {
        if (threadIdx.x == 0 && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) Op::idle(a);
        return;
    }
    // dynamic shared memory is only guaranteed 16-byte aligned: round up to 128 for the TMA destinations
    char* smem = reinterpret_cast<char*>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~uintptr_t(127));
    const uint32_t smem_s = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t bar_s = (uint32_t)__cvta_generic_to_shared(bars);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int x0 = blockIdx.x * BX, y0 = blockIdx.y * BY;
    const int k0 = blockIdx.z * zlen, k1 = min(g.nz, k0 + zlen);
    const int E = k1 - k0 + 2;                       // events: planes k0-1 .. k1
    const typename Op::Ctx ctx(a);

    if (threadIdx.x == 0) {
        for (int s = 0; s < D; ++s) { mbar_init(bar_s + 8 * s, 1); mbar_init(bar_s + 8 * (D + s), BY); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    double acc = 0.0;
    if (warp == BY) {
        // ---------------------------------------------------------------- producer warp (one elected lane)
        if (lane == 0) {
            int s = 0;
            uint32_t phase = 1;                     // parity of the previous use of slot s (first pass: no wait)
            for (int e = 0; e < E; ++e) {
                if (e >= D) mbar_wait(bar_s + 8 * (D + s), phase);
                const int c = k0 - 1 + e;
                Op::produce(a, ctx, maps, smem_s + (uint32_t)(s * Op::STAGE_BYTES), bar_s + 8 * s, x0, y0, c,
                            (c >= k0) && (c < k1));
                s = (s + 1 == D) ? 0 : s + 1;
                phase ^= (s == 0);
            }
        }
    } else {
        // ---------------------------------------------------------------- consumer warps: row = y0 + warp
        const int x = x0 + lane * V, j = y0 + warp;
        const bool out = (x < g.nx) && (j < g.ny);      // chunks made only of pad cells (x >= nx) stay zero
        const typename Op::TC tc = Op::thread_init(g, x);
        const int ycls = face_class(j, g.ny, g.fix[1]);  // rows next to the box faces normal to y (uniform per warp)
        const long long rowbase = (long long)j * g.px + x;
        // tile-plane flag bits (a group of this tile is flagged in plane k): a CTA whose planes are all clear -- every
        // CTA of a mask-free box -- runs the CLEAN loop, compiled without the coded path, the flag words and their
        // branches; only CTAs next to masked cells run the general loop
        const uint32_t* tf = a.tflags + (size_t)(blockIdx.y * gridDim.x + blockIdx.x) * g.twords;
        uint32_t anyf = 0;
        for (int w = k0 >> 5; w <= (k1 - 1) >> 5; ++w) {
            uint32_t m = tf[w];
            if (w == (k0 >> 5)) m &= ~0u << (k0 & 31);
            if (w == ((k1 - 1) >> 5)) m &= (2u << ((k1 - 1) & 31)) - 1u;
            anyf |= m;
        }
        auto run = [&](auto clean_tag) {
            constexpr bool CLEAN = decltype(clean_tag)::value;
            // running state instead of per-event div/mod: slot of event e, its phase bit, the shared addresses of
            // the stages of events e-2 / e-1 / e, the cell offset of plane c
            int s = 0, sB = 0;
            uint32_t phase = 0;
            uint32_t aB = smem_s, aC = smem_s, aF = smem_s;
            long long off = rowbase + (long long)(k0 - 1) * g.pplane;
            typename Op::State st;
            // general loop only: the row's flag words of the planes kp, kp+1 (and kp+2, fetched now) and the chunk's
            // stencil codes of planes kp and kp+1 -- every global load is issued at least one plane before its use
            uint32_t fwA = 0, fwB = 0, codeA[V], codeB[V];
#pragma unroll
            for (int i = 0; i < V; ++i) codeA[i] = codeB[i] = 0u;
            auto flag_word = [&](long long cell) { return a.flags[(cell >> 2) >> 5]; };
            auto flag_bit = [&](uint32_t w, long long cell) { return (w >> (unsigned)((cell >> 2) & 31)) & 1u; };
            if (!CLEAN && out) {
                const long long c0 = rowbase + (long long)k0 * g.pplane;
                fwA = flag_word(c0);
                if (k0 + 1 < k1) fwB = flag_word(c0 + g.pplane);
                if (flag_bit(fwA, c0)) ld_chunk<uint32_t, V>(a.wcode + c0, codeA);
            }
            for (int e = 0; e < E; ++e) {
                mbar_wait(bar_s + 8 * s, phase);
                Op::advance(st, ctx, aF, warp, lane);
                if (e >= 2) {                        // emit plane c-1 from stages e-2 (B), e-1 (centre), e (F)
                    const int kp = k0 + e - 2;       // the plane being emitted
                    const int zcls = face_class(kp, g.nz, g.fix[2]);
                    const long long idx = off - g.pplane;
                    uint32_t fb = 0, fwC = 0;
                    if (!CLEAN && out) {
                        fb = flag_bit(fwA, idx);
                        if (kp + 2 < k1) fwC = flag_word(idx + 2 * g.pplane);
                        if (kp + 1 < k1 && flag_bit(fwB, off)) ld_chunk<uint32_t, V>(a.wcode + off, codeB);
                    }
                    Op::template emit<CLEAN>(a, ctx, st, idx, aB, aC, aF, warp, lane, out, fb, codeA, tc, ycls, zcls, acc);
                    if (!CLEAN) {
                        fwA = fwB; fwB = fwC;
#pragma unroll
                        for (int i = 0; i < V; ++i) codeA[i] = codeB[i];
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar_s + 8 * (D + sB));
                    sB = (sB + 1 == D) ? 0 : sB + 1;
                }
                off += g.pplane;
                aB = aC; aC = aF;
                s = (s + 1 == D) ? 0 : s + 1;
                phase ^= (s == 0);
                aF = smem_s + (uint32_t)(s * Op::STAGE_BYTES);
            }
        };
        if (anyf) run(std::false_type{}); else run(std::true_type{});
    }

    // deterministic grid reduction (all warps, the producer contributes 0)
    const unsigned int nblk = gridDim.x * gridDim.y * gridDim.z;
    const unsigned int bid = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
    {
        double sacc = warp_sum(acc);
        if (lane == 0) red[warp] = sacc;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < BY; ++w) s += red[w];
        a.partial[bid] = s;
        __threadfence();
        unsigned int t = atomicAdd(&a.sc->ticket[Op::TICKET], 1u);
        is_last = (t == nblk - 1);
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        double s = 0.0;
        for (unsigned int b = threadIdx.x; b < nblk; b += TG::NTHR) s += __ldcg(&a.partial[b]);
        s = warp_sum(s);
        __syncthreads();
        if (lane == 0) red[warp] = s;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot[NACC] = { 0.0 };
            for (int w = 0; w <= BY; ++w) tot[0] += red[w];
            a.sc->ticket[Op::TICKET] = 0;
            Op::finalize(a, tot);
        }
    }
}

// ------------------------------------------------------------------------------------------------ K3 (TMA)
// p_new = r + beta p_old evaluated from the raw r / p_old tiles wherever the stencil needs it (centre, N, S, F, B
// chunks and the two x-halo cells); store p_new; gamma = p_new . M p_new; last CTA: alpha = rho / gamma.
template <typename T, int BY_, int D_, int MINB_>
struct OpT3 {
    using VT = T;
    using TG = TileGeom<T, BY_>;
    enum { V = TG::V, D = D_, MINB = MINB_, TICKET = 0, STAGE_BYTES = 2 * TG::TILE_H,
           BOX_H = (BY_ + 2) * TG::PITCH_H };
    struct Args {
        T* pbuf[2]; const uint32_t* wcode; const uint32_t* flags; const uint32_t* tflags;
        Coef<T> K; Scalars* sc; double* partial; CondHandles cond;
    };
    struct Ctx {
        T beta; int par; T* pnew;
        __device__ Ctx(const Args& a) { beta = (T)a.sc->beta; par = a.sc->k & 1; pnew = a.pbuf[par ^ 1]; }
    };
    using TC = XEdge;
    __device__ static TC thread_init(const Geom& g, int x) { return make_xedge<V>(g, x); }
    __device__ static bool active(const Args& a) { return a.sc->inner_go != 0; }
    __device__ static void idle(const Args& a) { set_cond(a.cond, -1, 0); }
    __device__ static void produce(const Args&, const Ctx& c, const TmaSet& m, uint32_t stage, uint32_t bar, int x0, int y0,
                                   int plane, bool)
    {
        mbar_expect_tx(bar, 2 * BOX_H);
        tma_load_3d(stage, &m.r_h, bar, x0 - TG::HX, y0 - 1, plane);
        tma_load_3d(stage + TG::TILE_H, &m.p_h[c.par], bar, x0 - TG::HX, y0 - 1, plane);
    }
    __device__ static void pnew_chunk(uint32_t st, int off, T beta, T (&v)[V])
    {
        T r[V], p[V];
        lds_chunk<T, V>(st + off, r);
        lds_chunk<T, V>(st + TG::TILE_H + off, p);
#pragma unroll
        for (int i = 0; i < V; ++i) v[i] = r[i] + beta * p[i];
    }
    // own-chunk p_new of the last three planes: each plane's chunk is formed once (when its stage arrives) and reused
    // as F, centre and B neighbour of three consecutive emissions
    struct State {
        T m[V], c[V], f[V];
        __device__ State() { zero_chunk<T, V>(m); zero_chunk<T, V>(c); zero_chunk<T, V>(f); }
    };
    __device__ static void advance(State& st, const Ctx& c, uint32_t sF, int warp, int lane)
    {
        const int off = (warp + 1) * TG::PITCH_H + (TG::HX + lane * V) * (int)sizeof(T);
#pragma unroll
        for (int i = 0; i < V; ++i) { st.m[i] = st.c[i]; st.c[i] = st.f[i]; }
        pnew_chunk(sF, off, c.beta, st.f);
    }
    template <bool CLEAN>
    __device__ static void emit(const Args& a, const Ctx& c, const State& st, long long idx, uint32_t, uint32_t sC, uint32_t,
                                int warp, int lane, bool out, uint32_t fb, const uint32_t (&code)[V], const TC& xe, int ycls, int zcls,
                                double& acc)
    {
        const int row = (warp + 1) * TG::PITCH_H;
        const int off = row + (TG::HX + lane * V) * (int)sizeof(T);
        T vn[V], vs[V];
        const T (&vm)[V] = st.m;
        const T (&vc)[V] = st.c;
        const T (&vp)[V] = st.f;
        pnew_chunk(sC, off + TG::PITCH_H, c.beta, vn);
        pnew_chunk(sC, off - TG::PITCH_H, c.beta, vs);
        // x neighbours: shuffles inside the warp, the row's two halo cells (same address for all lanes) at its ends
        const int hl_off = row + (TG::HX - 1) * (int)sizeof(T), hr_off = row + (TG::HX + TG::BX) * (int)sizeof(T);
        const T hl = lds_scalar(sC + hl_off, T()) + c.beta * lds_scalar(sC + TG::TILE_H + hl_off, T());
        const T hr = lds_scalar(sC + hr_off, T()) + c.beta * lds_scalar(sC + TG::TILE_H + hr_off, T());
        T xl = __shfl_up_sync(0xffffffffu, vc[V - 1], 1);
        T xr = __shfl_down_sync(0xffffffffu, vc[0], 1);
        if (lane == 0) xl = hl;
        if (lane == 31) xr = hr;
        if (!out) return;
        st_chunk<T, V>(c.pnew + idx, vc);
        T q[V];
        apply_M_chunk<T, V>(q, vm, vc, vp, vn, vs, xl, xr, CLEAN ? 0u : fb, code, a.K, xe, ycls, zcls);
#pragma unroll
        for (int i = 0; i < V; ++i) acc += (double)vc[i] * (double)q[i];
    }
    __device__ static void finalize(const Args& a, const double (&tot)[1])
    {
        Scalars* s = a.sc;
        const double gamma = tot[0];
        s->gamma = gamma;
        if (!(gamma > 0.0) || !isfinite(gamma)) {
            s->status = ST_BREAKDOWN; s->inner_go = 0; s->outer_go = 0;
            set_cond(a.cond, 0, 0);
        } else {
            s->alpha = s->rho / gamma;
        }
    }
};

// ------------------------------------------------------------------------------------------------ K4 (TMA)
// q = M p recomputed from the haloed p tile; delta += alpha p; r -= alpha q; rho' = r.r; beta, loop test.
template <typename T, int BY_, int D_, int MINB_>
struct OpT4 {
    using VT = T;
    using TG = TileGeom<T, BY_>;
    enum { V = TG::V, D = D_, MINB = MINB_, TICKET = 1, STAGE_BYTES = TG::TILE_H + 2 * TG::TILE_C,
           BOX_H = (BY_ + 2) * TG::PITCH_H };
    struct Args {
        T* r; T* delta; int p_fixed;      // p_fixed >= 0: read p from pbuf[p_fixed] (omni_apply_M), else by parity
        const uint32_t* wcode; const uint32_t* flags; const uint32_t* tflags;
        Coef<T> K; Scalars* sc; double* partial; CondHandles cond;
        T* q_out;                         // only for omni_apply_M: store q, leave r / delta untouched
    };
    struct Ctx {
        T alpha; int pidx; bool first;
        __device__ Ctx(const Args& a)
        {
            alpha = (T)a.sc->alpha;
            first = (a.sc->k == 0);
            pidx = (a.p_fixed >= 0) ? a.p_fixed : ((a.sc->k & 1) ^ 1);
        }
    };
    using TC = XEdge;
    __device__ static TC thread_init(const Geom& g, int x) { return make_xedge<V>(g, x); }
    __device__ static bool active(const Args& a) { return a.sc->inner_go != 0; }
    __device__ static void idle(const Args& a) { set_cond(a.cond, -1, 0); }
    __device__ static void produce(const Args& a, const Ctx& c, const TmaSet& m, uint32_t stage, uint32_t bar, int x0,
                                   int y0, int plane, bool inner)
    {
        const bool ext = inner && (a.q_out == nullptr);
        const bool dl = ext && !c.first;           // first CG iteration: delta counts as zero, never read
        mbar_expect_tx(bar, BOX_H + (ext ? TG::TILE_C : 0) + (dl ? TG::TILE_C : 0));
        tma_load_3d(stage, &m.p_h[c.pidx], bar, x0 - TG::HX, y0 - 1, plane);
        if (ext) tma_load_3d(stage + TG::TILE_H, &m.r_c, bar, x0, y0, plane);
        if (dl) tma_load_3d(stage + TG::TILE_H + TG::TILE_C, &m.d_c, bar, x0, y0, plane);
    }
    struct State {};
    __device__ static void advance(State&, const Ctx&, uint32_t, int, int) {}
    template <bool CLEAN>
    __device__ static void emit(const Args& a, const Ctx& c, const State&, long long idx, uint32_t sB, uint32_t sC, uint32_t sF,
                                int warp, int lane, bool out, uint32_t fb, const uint32_t (&code)[V], const TC& xe, int ycls, int zcls,
                                double& acc)
    {
        const int row = (warp + 1) * TG::PITCH_H;
        const int off = row + (TG::HX + lane * V) * (int)sizeof(T);
        T vm[V], vc[V], vp[V], vn[V], vs[V];
        lds_chunk<T, V>(sC + off, vc);
        lds_chunk<T, V>(sC + off + TG::PITCH_H, vn);
        lds_chunk<T, V>(sC + off - TG::PITCH_H, vs);
        lds_chunk<T, V>(sF + off, vp);
        lds_chunk<T, V>(sB + off, vm);
        const T hl = lds_scalar(sC + row + (TG::HX - 1) * (int)sizeof(T), T());
        const T hr = lds_scalar(sC + row + (TG::HX + TG::BX) * (int)sizeof(T), T());
        T xl = __shfl_up_sync(0xffffffffu, vc[V - 1], 1);
        T xr = __shfl_down_sync(0xffffffffu, vc[0], 1);
        if (lane == 0) xl = hl;
        if (lane == 31) xr = hr;
        if (!out) return;
        T q[V];
        apply_M_chunk<T, V>(q, vm, vc, vp, vn, vs, xl, xr, CLEAN ? 0u : fb, code, a.K, xe, ycls, zcls);
        if (a.q_out != nullptr) {
            st_chunk<T, V>(a.q_out + idx, q);
#pragma unroll
            for (int i = 0; i < V; ++i) acc += (double)vc[i] * (double)q[i];
            return;
        }
        const int eoff = TG::TILE_H + (warp * TG::BX + lane * V) * (int)sizeof(T);
        T er[V], ed[V], rn[V], dn[V];
        lds_chunk<T, V>(sC + eoff, er);
        if (c.first) zero_chunk<T, V>(ed); else lds_chunk<T, V>(sC + eoff + TG::TILE_C, ed);
#pragma unroll
        for (int i = 0; i < V; ++i) {
            rn[i] = er[i] - c.alpha * q[i];
            dn[i] = ed[i] + c.alpha * vc[i];
            acc += (double)rn[i] * (double)rn[i];
        }
        st_chunk<T, V>(a.r + idx, rn);
        st_chunk<T, V>(a.delta + idx, dn);
    }
    __device__ static void finalize(const Args& a, const double (&tot)[1])
    {
        Scalars* s = a.sc;
        if (a.q_out != nullptr) { s->gamma = tot[0]; return; }
        const double rho1 = tot[0];
        if (!isfinite(rho1)) {
            s->status = ST_BREAKDOWN; s->inner_go = 0; s->outer_go = 0;
            set_cond(a.cond, 0, 0);
            return;
        }
        s->beta = rho1 / s->rho;
        s->rho = rho1;
        s->k += 1;
        s->cg_total += 1;
        const int go = (rho1 > s->thresh2) && (rho1 != 0.0) && (s->k < s->max_cg);
        s->inner_go = go;
        set_cond(a.cond, -1, go);
    }
};

}  // namespace omni
