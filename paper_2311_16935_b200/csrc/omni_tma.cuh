// omni_tma.cuh -- K2 / K3 / K4 on a TMA + mbarrier producer/consumer pipeline (sm_100a).
//
// A CTA owns a column of the grid: BX = 32*V cells (512 bytes) x BY rows x zlen planes.  One producer warp issues,
// per plane, a few cp.async.bulk.tensor (TMA) box loads -- the tile of every streamed array, the stencil input with
// its one-cell halo in x and y -- into a D-deep ring of shared-memory stages; out-of-box coordinates (box faces, the
// planes before/after the grid) are zero-filled by the TMA unit, so the kernels carry no bounds logic.  BY consumer
// warps (one row each, V cells per lane) wait on the stage's "full" mbarrier, read the centre / N / S chunks of plane
// c-1 and the own chunk of planes c-2 and c from the three resident stages (x neighbours by shuffle), evaluate the
// operator, store, and release the oldest stage through its "empty" mbarrier.  Warps only ever wait for data, never
// for each other: there is no CTA-wide barrier in the loop and no state carried in registers across planes.
// The grid reduction at the end is deterministic: fp64 per-thread partials -> warp shuffle -> CTA -> fixed slot; the
// last-arriving CTA (atomic ticket) adds the slots in slot order and updates the device-resident loop scalars.
#pragma once
#include <cuda.h>
#include <type_traits>
#include "omni_kernels.cuh"

#ifndef OMNI_ZIGZAG
#define OMNI_ZIGZAG 0      // 1: K4 marches z downwards (+3 % at 256^3 fp32, -4 % at 500^3: profiles/r2_loop_and_rows.md); 0: every kernel upwards
#endif

namespace omni {

// loop conditions of the CUDA-graph WHILE nodes, written by a kernel's last CTA (no-op outside the graph)
__device__ __forceinline__ void set_cond(const CondHandles& h, int outer, int inner)
{
#if defined(__CUDA_ARCH__)
    if ((h.use & 1) && outer >= 0) cudaGraphSetConditional((cudaGraphConditionalHandle)h.h_outer, (unsigned)outer);
    if ((h.use & 2) && inner >= 0) cudaGraphSetConditional((cudaGraphConditionalHandle)h.h_inner, (unsigned)inner);
#endif
}

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
    // K2 (64-cell tiles: the fp64 master pressure sets the 16-byte lane chunk)
    CUtensorMap p_c[2];          // plain: both p buffers (K4's lazy delta update reads p_{k-1} without halo)
    CUtensorMap P_h[2], d2_h;    // haloed: P (fp64, both buffers), delta (T)
    CUtensorMap S_c;             // plain: S (T)
};

// z segments of a launch: uniform (n == 0: segment b covers planes [b zlen, (b+1) zlen)) or a table of boundaries
// (segment b covers [k[b], k[b+1]); tapered schedules, tma_config)
struct ZSeg {
    enum { MAXSEG = 48 };
    int n, zlen;
    int k[MAXSEG + 1];
};

template <typename T, int BY_, int R_>
struct TileGeom {
    static_assert(BY_ % R_ == 0, "a tile's rows are shared out evenly among its consumer warps");
    static constexpr int V = 16 / (int)sizeof(T);          // cells per lane (one 16-byte piece)
    static constexpr int BX = 32 * V;                      // 512 bytes per row
    static constexpr int BY = BY_;
    static constexpr int R = R_;                           // rows per consumer warp (neighbouring rows: N / S values are shared in registers)
    static constexpr int NCW = BY_ / R_;                   // consumer warps
    static constexpr int HX = 16 / (int)sizeof(T);         // x halo in cells (16 bytes: TMA box rows are 16 B multiples)
    static constexpr int PITCH_H = (BX + 2 * HX) * (int)sizeof(T);       // 544 bytes
    static constexpr int TILE_H = ((BY + 2) * PITCH_H + 127) / 128 * 128;
    static constexpr int TILE_C = BY * BX * (int)sizeof(T);              // multiple of 512
    static constexpr int NTHR = 32 * (NCW + 1);            // NCW consumer warps + 1 producer warp
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

// a thread's contribution to a dot product: fp64 products for fp64 data; for fp32 data the V products of one 16-byte
// chunk are summed in fp32 (fused multiply-adds) and enter the fp64 accumulator as one term -- one conversion per
// chunk instead of two per cell, the fp32 sum of 4 terms adding 1e-7 relative to a term, like the data's own rounding
template <typename T, int V>
__device__ __forceinline__ double chunk_dot(const T (&a)[V], const T (&b)[V])
{
    if constexpr (sizeof(T) == 8) {
        double s = 0.0;
#pragma unroll
        for (int i = 0; i < V; ++i) s += (double)a[i] * (double)b[i];
        return s;
    } else {
        float s = 0.f;
#pragma unroll
        for (int i = 0; i < V; ++i) s = fmaf((float)a[i], (float)b[i], s);
        return (double)s;
    }
}

#ifdef OMNI_TUNING   // tuning builds only: per-CTA timeline (start, end, SM) of the last launch of each operator
__device__ unsigned long long g_cta_trace[3][3 * 8192];
__device__ __forceinline__ unsigned long long dbg_timer()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
#endif

// (re)initialise the ring of a pass: D "full" barriers (one arrival: the producer's expect_tx) and D "empty" barriers
// (BY arrivals: one per consumer warp).  again = the same words held the ring of an earlier pass (loop kernel); every
// thread of the CTA has left that pass (the caller synchronises before and after).
__device__ __forceinline__ void ring_init(uint32_t bar_s, int D, int nmax, int consumers, bool again)
{
    if (again)
        for (int s = 0; s < 2 * nmax; ++s) asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(bar_s + 8 * s) : "memory");
    for (int s = 0; s < D; ++s) { mbar_init(bar_s + 8 * s, 1); mbar_init(bar_s + 8 * (D + s), consumers); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// One pass of a column -- planes [k0, k1) of tile (x0, y0) -- through the TMA ring.  Event e = 0 .. k1-k0+1 loads one
// plane; the march runs up (plane k0-1+e) or, for Op::REV, down (plane k1-e), so that a kernel that follows another can
// start where the other ended and find those planes still in L2 ("zig-zag").  At event e >= 2 the
// plane of event e-1 is emitted from the three resident stages.  Called by every thread of the CTA after ring_init +
// __syncthreads; warps only wait for data, never for each other.  acc: per-thread fp64 partials (producer warp: 0).
template <class Op>
__device__ __forceinline__ void run_column(const Geom& g, const typename Op::Args& a, const typename Op::Ctx& ctx,
                                           const TmaSet& maps, uint32_t smem_s, uint32_t bar_s, int tx, int ty,
                                           int k0, int k1, double (&acc)[Op::NACC])
{
    using TG = typename Op::TG;
    constexpr int V = TG::V, BX = TG::BX, BY = TG::BY, R = TG::R, NCW = TG::NCW;
    constexpr bool REV = Op::REV;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int x0 = tx * BX, y0 = ty * BY;
    const int n = k1 - k0, E = n + 2;                 // emitted planes; events
    const int pl0 = REV ? k1 : k0 - 1;                // plane of event 0
    // ring depth and stage size may depend on what this launch streams (K4: DESIGN.md section 6, lazy delta)
    const int D = Op::stages(ctx);
    const uint32_t SB = (uint32_t)Op::stage_bytes(ctx);

    if (warp == NCW) {
        // ---------------------------------------------------------------- producer warp (one elected lane)
        if (lane == 0) {
            int s = 0;
            uint32_t phase = 1;                     // parity of the previous use of slot s (first pass: no wait)
            for (int e = 0; e < E; ++e) {
                if (e >= D) mbar_wait(bar_s + 8 * (D + s), phase);
                const int c = REV ? pl0 - e : pl0 + e;
                Op::produce(a, ctx, maps, smem_s + (uint32_t)s * SB, bar_s + 8 * s, x0, y0, c,
                            (c >= k0) && (c < k1));
                s = (s + 1 == D) ? 0 : s + 1;
                phase ^= (s == 0);
            }
        }
        return;
    }
    // ---------------------------------------------------------------- consumer warps: rows y0 + warp R .. + R - 1
    const int x = x0 + lane * V, j0 = y0 + warp * R;
    bool out[R];                                    // chunks made only of pad cells (x >= nx) stay zero
    int ycls[R];                                    // rows next to the box faces normal to y (uniform per warp)
#pragma unroll
    for (int r = 0; r < R; ++r) {
        out[r] = (x < g.nx) && (j0 + r < g.ny);
        ycls[r] = face_class(j0 + r, g.ny, g.fix[1]);
    }
    const typename Op::TC tc = Op::thread_init(g, x);
    const long long rowbase = (long long)j0 * g.px + x;
    const long long step = REV ? -g.pplane : g.pplane;
    // tile-plane flag bits (a group of this tile is flagged in plane k): a CTA whose planes are all clear -- every
    // CTA of a mask-free box -- runs the CLEAN loop, compiled without the coded path, the flag words and their
    // branches; only CTAs next to masked cells run the general loop
    const uint32_t* tf = a.tflags + (size_t)(ty * g.ntx + x0 / g.tbx) * g.twords;
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
        // the stages of events e-2 / e-1 / e, the cell offset of the plane of event e
        int s = 0, sB = 0;
        uint32_t phase = 0;
        uint32_t a2 = smem_s, a1 = smem_s, a0 = smem_s;
        long long off = rowbase + (long long)pl0 * g.pplane;
        typename Op::State st;
        // general loop only, per row: the flag words of the emitted plane, the next one (and the one after, fetched
        // now) and the chunk's stencil codes of the emitted and the next plane -- every global load is issued at least
        // one plane before its use
        uint32_t fwA[R], fwB[R], fb[R], codeA[R][V], codeB[R][V];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            fwA[r] = fwB[r] = fb[r] = 0u;
#pragma unroll
            for (int i = 0; i < V; ++i) codeA[r][i] = codeB[r][i] = 0u;
        }
        auto flag_word = [&](long long cell) { return a.flags[(cell >> 2) >> 5]; };
        auto flag_bit = [&](uint32_t w, long long cell) { return (w >> (unsigned)((cell >> 2) & 31)) & 1u; };
        if (!CLEAN) {
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (out[r]) {
                    const long long c0 = off + step + (long long)r * g.px;          // first emitted plane
                    fwA[r] = flag_word(c0);
                    if (n > 1) fwB[r] = flag_word(c0 + step);
                    if (flag_bit(fwA[r], c0)) Op::load_codes(a, c0, codeA[r]);
                }
        }
        // two events per trip: half of the ring / window rotation becomes register renaming (+2 % on the fp64
        // kernels at 256^3, +0.5 % at 500^3 fp32; three per trip is slower: profiles/r1_tile_variants.md)
#pragma unroll 2
        for (int e = 0; e < E; ++e) {
            mbar_wait(bar_s + 8 * s, phase);
            Op::advance(st, ctx, a0, warp, lane);
            if (e >= 2) {                        // emit the plane of event e-1 from the stages of events e-2, e-1, e
                const int i = e - 2;             // index of the emitted plane in march order
                const int kp = REV ? k1 - 1 - i : k0 + i;
                const int zcls = face_class(kp, g.nz, g.fix[2]);
                const long long idx = off - step;
                if (!CLEAN) {
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        uint32_t fwC = 0;
                        fb[r] = 0;
                        if (out[r]) {
                            const long long cr = idx + (long long)r * g.px;
                            fb[r] = flag_bit(fwA[r], cr);
                            if (i + 2 < n) fwC = flag_word(cr + 2 * step);
                            if (i + 1 < n && flag_bit(fwB[r], cr + step)) Op::load_codes(a, cr + step, codeB[r]);
                        }
                        fwA[r] = fwB[r]; fwB[r] = fwC;
                    }
                }
                // stage of plane kp-1 (B), of plane kp, of plane kp+1 (F)
                Op::template emit<CLEAN>(a, ctx, st, idx, g.px, REV ? a0 : a2, a1, REV ? a2 : a0, warp, lane, out, fb, codeA,
                                         tc, ycls, zcls, acc);
                if (!CLEAN) {
#pragma unroll
                    for (int r = 0; r < R; ++r)
#pragma unroll
                        for (int q = 0; q < V; ++q) codeA[r][q] = codeB[r][q];
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_s + 8 * (D + sB));
                sB = (sB + 1 == D) ? 0 : sB + 1;
            }
            off += step;
            a2 = a1; a1 = a0;
            s = (s + 1 == D) ? 0 : s + 1;
            phase ^= (s == 0);
            a0 = smem_s + (uint32_t)s * SB;
        }
    };
    if (anyf) run(std::false_type{}); else run(std::true_type{});
}

// tile and z segment of a CTA; Op::REV kernels take their CTAs in the opposite order (high z first, z table mirrored:
// the long segments of a tapered schedule still come first)
template <bool REV>
__device__ __forceinline__ void cta_column(const Geom& g, const ZSeg& zs, int& tx, int& ty, int& k0, int& k1)
{
    const int bz = blockIdx.z;
    const int nzr = g.kz1 - g.kz0;                   // planes to emit: all of them, or the ones a slab owns
    int lo = zs.n ? zs.k[bz] : bz * zs.zlen;
    int hi = zs.n ? zs.k[bz + 1] : min(nzr, lo + zs.zlen);
    if (REV) {
        tx = gridDim.x - 1 - blockIdx.x; ty = gridDim.y - 1 - blockIdx.y;
        k0 = g.kz0 + nzr - hi; k1 = g.kz0 + nzr - lo;
    } else {
        tx = blockIdx.x; ty = blockIdx.y;
        k0 = g.kz0 + lo; k1 = g.kz0 + hi;
    }
}

template <class Op>
__global__ void __launch_bounds__(Op::TG::NTHR, Op::MINB)
tma_kernel(const Geom g, const ZSeg zs, const typename Op::Args a, const __grid_constant__ TmaSet maps)
{
    using TG = typename Op::TG;
    constexpr int NCW = TG::NCW, NACC = Op::NACC;
    extern __shared__ __align__(128) char smem_raw[];
    __shared__ double red[NACC][NCW + 1];
    __shared__ int is_last;
    __shared__ __align__(8) unsigned long long bars[2 * Op::DMAX];

    if (!Op::active(a)) {
        if (threadIdx.x == 0 && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) Op::idle(a);
        return;
    }
#ifdef OMNI_TUNING
    const unsigned long long dbg_t0 = dbg_timer();
#endif
    // dynamic shared memory is only guaranteed 16-byte aligned: round up to 128 for the TMA destinations
    char* smem = reinterpret_cast<char*>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~uintptr_t(127));
    const uint32_t smem_s = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t bar_s = (uint32_t)__cvta_generic_to_shared(bars);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int tx, ty, k0, k1;
    cta_column<Op::REV>(g, zs, tx, ty, k0, k1);
    const typename Op::Ctx ctx(a);
    if (threadIdx.x == 0) ring_init(bar_s, Op::stages(ctx), Op::DMAX, NCW, false);
    __syncthreads();

    double acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = 0.0;
    run_column<Op>(g, a, ctx, maps, smem_s, bar_s, tx, ty, k0, k1, acc);

    // deterministic grid reduction (all warps, the producer contributes 0)
    const unsigned int nblk = gridDim.x * gridDim.y * gridDim.z;
    const unsigned int bid = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
#pragma unroll
    for (int i = 0; i < NACC; ++i) {
        double sacc = warp_sum(acc[i]);
        if (lane == 0) red[i][warp] = sacc;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < NACC; ++i) {
            double s = 0.0;
            for (int w = 0; w < NCW; ++w) s += red[i][w];
            a.partial[(size_t)i * nblk + bid] = s;
        }
        __threadfence();
        unsigned int t = atomicAdd(&a.sc->ticket[Op::TICKET], 1u);
        is_last = (t == nblk - 1);
    }
    __syncthreads();
#ifdef OMNI_TUNING
    if (threadIdx.x == 0 && bid < 8192) {
        unsigned int smid;
        asm volatile("mov.u32 %0, %smid;" : "=r"(smid));
        g_cta_trace[Op::TICKET][3 * bid] = dbg_t0;
        g_cta_trace[Op::TICKET][3 * bid + 1] = dbg_timer();
        g_cta_trace[Op::TICKET][3 * bid + 2] = smid | ((unsigned long long)nblk << 32);
    }
#endif
    if (is_last) {
        __threadfence();
        double tot[NACC];
#pragma unroll
        for (int i = 0; i < NACC; ++i) {
            double s = 0.0;
            for (unsigned int b = threadIdx.x; b < nblk; b += TG::NTHR) s += __ldcg(&a.partial[(size_t)i * nblk + b]);
            s = warp_sum(s);
            __syncthreads();
            if (lane == 0) red[i][warp] = s;
            __syncthreads();
            s = 0.0;
            for (int w = 0; w <= NCW; ++w) s += red[i][w];
            tot[i] = s;
        }
        if (threadIdx.x == 0) {
            a.sc->ticket[Op::TICKET] = 0;
            if (a.sc->defer) {
#pragma unroll
                for (int i = 0; i < NACC; ++i) a.sc->red_out[i] = tot[i];      // summed over the ranks first (omni_slab.cuh)
            } else {
                Op::finalize(a, tot);
            }
        }
    }
}

// sharded solves: the finalize step of Op on the rank-summed totals (one thread; every rank runs it on identical numbers)
template <class Op>
__global__ void op_finalize_kernel(const typename Op::Args a)
{
    if (!Op::active(a)) return;
    double tot[Op::NACC];
#pragma unroll
    for (int i = 0; i < Op::NACC; ++i) tot[i] = a.sc->red_out[i];
    Op::finalize(a, tot);
}

// ------------------------------------------------------------------------------------------------ K3 (TMA)
// p_new = r + beta p_old evaluated from the raw r / p_old tiles wherever the stencil needs it (centre, N, S, F, B
// chunks and the two x-halo cells); store p_new; gamma = p_new . M p_new; last CTA: alpha = rho / gamma.
template <typename T, int BY_, int R_, int D_, int MINB_, bool LOP_ = false>
struct OpT3 {
    using VT = T;
    using TG = TileGeom<T, BY_, R_>;
    enum { V = TG::V, R = R_, D = D_, DMAX = D_, MINB = MINB_, NACC = 1, TICKET = 0, STAGE_BYTES = 2 * TG::TILE_H,
           SMEM_BYTES = D_ * STAGE_BYTES, BOX_H = (BY_ + 2) * TG::PITCH_H };
    static constexpr bool REV = false;       // marches z upwards
    struct Args {
        T* pbuf[2]; const uint32_t* wcode; const uint8_t* link; const uint32_t* flags; const uint32_t* tflags;
        Coef<T> K; Scalars* sc; double* partial; CondHandles cond;
    };
    struct Ctx {
        T beta; int par; T* pnew;
        __device__ Ctx(const Args& a) : Ctx(a, a.sc->beta, a.sc->k) {}
        __device__ Ctx(const Args& a, double beta_, int k) { beta = (T)beta_; par = k & 1; pnew = a.pbuf[par ^ 1]; }
    };
    using TC = XEdge;
    __device__ static int stages(const Ctx&) { return D; }
    __device__ static int stage_bytes(const Ctx&) { return STAGE_BYTES; }
    __device__ static TC thread_init(const Geom& g, int x) { return make_xedge<V>(g, x); }
    __device__ static bool active(const Args& a) { return a.sc->inner_go != 0; }
    __device__ static void idle(const Args& a) { set_cond(a.cond, -1, 0); }
    __device__ static void load_codes(const Args& a, long long cell, uint32_t (&code)[V]) { load_cell_codes<LOP_, V>(a.wcode, a.link, cell, code); }
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
    // own-chunk p_new of the last three planes, for each of the warp's R rows: a plane's chunks are formed once (when its
    // stage arrives) and reused as F, centre and B neighbour of three consecutive emissions -- and, within a plane, as
    // N / S neighbour of the rows next to them
    struct State {
        T m[R][V], c[R][V], f[R][V];
        __device__ State()
        {
#pragma unroll
            for (int r = 0; r < R; ++r) { zero_chunk<T, V>(m[r]); zero_chunk<T, V>(c[r]); zero_chunk<T, V>(f[r]); }
        }
    };
    __device__ static void advance(State& st, const Ctx& c, uint32_t sNew, int warp, int lane)
    {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int off = (warp * R + r + 1) * TG::PITCH_H + (TG::HX + lane * V) * (int)sizeof(T);
#pragma unroll
            for (int i = 0; i < V; ++i) { st.m[r][i] = st.c[r][i]; st.c[r][i] = st.f[r][i]; }
            pnew_chunk(sNew, off, c.beta, st.f[r]);
        }
    }
    template <bool CLEAN>
    __device__ static void emit(const Args& a, const Ctx& c, const State& st, long long idx, int px, uint32_t, uint32_t sC, uint32_t,
                                int warp, int lane, const bool (&out)[R], const uint32_t (&fb)[R], const uint32_t (&code)[R][V],
                                const TC& xe, const int (&ycls)[R], int zcls, double (&accs)[1])
    {
        double& acc = accs[0];
        const int row0 = (warp * R + 1) * TG::PITCH_H;                     // shared-memory row of the warp's first row
        const int xoff = (TG::HX + lane * V) * (int)sizeof(T);
        // rows j0-1 .. j0+R of the emitted plane: the two outer ones from the stage, the warp's own from the window
        T rows[R + 2][V];
        pnew_chunk(sC, row0 - TG::PITCH_H + xoff, c.beta, rows[0]);
        pnew_chunk(sC, row0 + R * TG::PITCH_H + xoff, c.beta, rows[R + 1]);
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int i = 0; i < V; ++i) rows[r + 1][i] = st.c[r][i];
        const int hl_off = (TG::HX - 1) * (int)sizeof(T), hr_off = (TG::HX + TG::BX) * (int)sizeof(T);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const T (&vc)[V] = rows[r + 1];
            // x neighbours: shuffles inside the warp, the row's two halo cells (same address for all lanes) at its ends
            const int row = row0 + r * TG::PITCH_H;
            const T hl = lds_scalar(sC + row + hl_off, T()) + c.beta * lds_scalar(sC + TG::TILE_H + row + hl_off, T());
            const T hr = lds_scalar(sC + row + hr_off, T()) + c.beta * lds_scalar(sC + TG::TILE_H + row + hr_off, T());
            T xl = __shfl_up_sync(0xffffffffu, vc[V - 1], 1);
            T xr = __shfl_down_sync(0xffffffffu, vc[0], 1);
            if (lane == 0) xl = hl;
            if (lane == 31) xr = hr;
            if (out[r]) {
                st_chunk<T, V>(c.pnew + idx + (long long)r * px, vc);
                T q[V];
                apply_op_chunk<LOP_, T, V>(q, REV ? st.f[r] : st.m[r], vc, REV ? st.m[r] : st.f[r], rows[r + 2], rows[r], xl, xr,
                                           CLEAN ? 0u : fb[r], code[r], a.K, xe, ycls[r], zcls);
                acc += chunk_dot<T, V>(vc, q);
            }
        }
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
// q = A p recomputed from the haloed p tile; r -= alpha q; rho' = r.r; beta, loop test.
// Lazy delta: delta does not have to exist between CG iterations, only when K2 folds it into P.  Both p buffers are
// alive in K4 -- p_k (haloed, for the stencil) and p_{k-1} (K3 overwrites it only in the next iteration) -- so delta
// is touched every SECOND iteration: even k stream {p, r} and leave alpha_k p_k pending; odd k stream {p, p_old, r,
// delta} and apply delta += alpha_{k-1} p_{k-1} + alpha_k p_k.  7.5 instead of 8 passes per CG iteration on average
// (K4: 3 / 6 instead of 5 / 5).  A pending update at loop exit is applied by flush_delta_kernel before K2.
// The ring is sized per parity: DO_ stages of {p_h, r, p_old, delta} or as many {p_h, r} stages as fit the same bytes.
template <typename T, int BY_, int R_, int DO_, int MINB_, bool LOP_ = false>
struct OpT4 {
    using VT = T;
    using TG = TileGeom<T, BY_, R_>;
    enum { V = TG::V, R = R_, MINB = MINB_, NACC = 1, TICKET = 1,
           STAGE_ODD = TG::TILE_H + 3 * TG::TILE_C, STAGE_EVEN = TG::TILE_H + TG::TILE_C,
           D_ODD = DO_, D_EVEN = (DO_ * STAGE_ODD) / STAGE_EVEN, DMAX = D_EVEN, SMEM_BYTES = DO_ * STAGE_ODD,
           BOX_H = (BY_ + 2) * TG::PITCH_H };
    // marches z downwards, CTAs in the opposite order: K4 starts on the planes K3 has just written (p_new) and read (r),
    // the next K3 on the planes K4 has just written (r) -- what the L2 still holds of them is not fetched from DRAM
    static constexpr bool REV = OMNI_ZIGZAG != 0;
    struct Args {
        T* r; T* delta; int p_fixed;      // p_fixed >= 0: read p from pbuf[p_fixed] (omni_apply_M), else by parity
        const uint32_t* wcode; const uint8_t* link; const uint32_t* flags; const uint32_t* tflags;
        Coef<T> K; Scalars* sc; double* partial; CondHandles cond;
        T* q_out;                         // only for omni_apply_M: store q, leave r / delta untouched
        int pcg;                          // 1: preconditioned recurrence (omni_solve_pcg): rho = r.z and beta come from
                                          //    mg_dot_kernel after the V-cycle; this kernel only tests ||r||
    };
    struct Ctx {
        T alpha, alpha_prev; int pidx, pold; bool odd, first, step;
        __device__ Ctx(const Args& a) : Ctx(a, a.sc->alpha, a.sc->alpha_prev, a.sc->k) {}
        __device__ Ctx(const Args& a, double alpha_, double alpha_prev_, int k)
        {
            alpha = (T)alpha_;
            alpha_prev = (T)alpha_prev_;
            step = (a.q_out != nullptr);
            odd = (k & 1) != 0;
            first = (k == 1);                        // first delta write of this inner solve: delta counts as zero
            pidx = (a.p_fixed >= 0) ? a.p_fixed : ((k & 1) ^ 1);
            pold = k & 1;
        }
    };
    using TC = XEdge;
    __device__ static int stages(const Ctx& c) { return (c.odd || c.step) ? D_ODD : D_EVEN; }
    __device__ static int stage_bytes(const Ctx& c) { return (c.odd || c.step) ? STAGE_ODD : STAGE_EVEN; }
    __device__ static TC thread_init(const Geom& g, int x) { return make_xedge<V>(g, x); }
    __device__ static bool active(const Args& a) { return a.sc->inner_go != 0; }
    __device__ static void idle(const Args& a) { set_cond(a.cond, -1, 0); }
    __device__ static void load_codes(const Args& a, long long cell, uint32_t (&code)[V]) { load_cell_codes<LOP_, V>(a.wcode, a.link, cell, code); }
    __device__ static void produce(const Args&, const Ctx& c, const TmaSet& m, uint32_t stage, uint32_t bar, int x0,
                                   int y0, int plane, bool inner)
    {
        const bool ext = inner && !c.step;
        const bool upd = ext && c.odd;
        const bool dl = upd && !c.first;
        mbar_expect_tx(bar, BOX_H + (ext ? TG::TILE_C : 0) + (upd ? TG::TILE_C : 0) + (dl ? TG::TILE_C : 0));
        tma_load_3d(stage, &m.p_h[c.pidx], bar, x0 - TG::HX, y0 - 1, plane);
        if (ext) tma_load_3d(stage + TG::TILE_H, &m.r_c, bar, x0, y0, plane);
        if (upd) tma_load_3d(stage + TG::TILE_H + TG::TILE_C, &m.p_c[c.pold], bar, x0, y0, plane);
        if (dl) tma_load_3d(stage + TG::TILE_H + 2 * TG::TILE_C, &m.d_c, bar, x0, y0, plane);
    }
    struct State {};
    __device__ static void advance(State&, const Ctx&, uint32_t, int, int) {}
    template <bool CLEAN>
    __device__ static void emit(const Args& a, const Ctx& c, const State&, long long idx, int px, uint32_t sB, uint32_t sC, uint32_t sF,
                                int warp, int lane, const bool (&out)[R], const uint32_t (&fb)[R], const uint32_t (&code)[R][V],
                                const TC& xe, const int (&ycls)[R], int zcls, double (&accs)[1])
    {
        double& acc = accs[0];
        const int row0 = (warp * R + 1) * TG::PITCH_H;
        const int xoff = (TG::HX + lane * V) * (int)sizeof(T);
        // rows j0-1 .. j0+R of the emitted plane: each is the N / S neighbour of the rows next to it
        T rows[R + 2][V];
#pragma unroll
        for (int q = 0; q < R + 2; ++q) lds_chunk<T, V>(sC + row0 + (q - 1) * TG::PITCH_H + xoff, rows[q]);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const T (&vc)[V] = rows[r + 1];
            const int row = row0 + r * TG::PITCH_H;
            T vp[V], vm[V];
            lds_chunk<T, V>(sF + row + xoff, vp);
            lds_chunk<T, V>(sB + row + xoff, vm);
            const T hl = lds_scalar(sC + row + (TG::HX - 1) * (int)sizeof(T), T());
            const T hr = lds_scalar(sC + row + (TG::HX + TG::BX) * (int)sizeof(T), T());
            T xl = __shfl_up_sync(0xffffffffu, vc[V - 1], 1);
            T xr = __shfl_down_sync(0xffffffffu, vc[0], 1);
            if (lane == 0) xl = hl;
            if (lane == 31) xr = hr;
            if (!out[r]) continue;
            const long long cell = idx + (long long)r * px;
            T q[V];
            apply_op_chunk<LOP_, T, V>(q, vm, vc, vp, rows[r + 2], rows[r], xl, xr, CLEAN ? 0u : fb[r], code[r], a.K, xe, ycls[r], zcls);
            if (c.step) {
                st_chunk<T, V>(a.q_out + cell, q);
                acc += chunk_dot<T, V>(vc, q);
                continue;
            }
            const int eoff = TG::TILE_H + ((warp * R + r) * TG::BX + lane * V) * (int)sizeof(T);
            T er[V], rn[V];
            lds_chunk<T, V>(sC + eoff, er);
#pragma unroll
            for (int i = 0; i < V; ++i) rn[i] = er[i] - c.alpha * q[i];
            acc += chunk_dot<T, V>(rn, rn);
            st_chunk<T, V>(a.r + cell, rn);
            if (c.odd) {
                T ep[V], ed[V], dn[V];
                lds_chunk<T, V>(sC + eoff + TG::TILE_C, ep);
                if (c.first) zero_chunk<T, V>(ed); else lds_chunk<T, V>(sC + eoff + 2 * TG::TILE_C, ed);
#pragma unroll
                for (int i = 0; i < V; ++i) dn[i] = (ed[i] + c.alpha_prev * ep[i]) + c.alpha * vc[i];
                st_chunk<T, V>(a.delta + cell, dn);
            }
        }
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
        if (s->k & 1) { s->pend = 0; } else { s->pend = 1; s->alpha_prev = s->alpha; }
        if (!a.pcg) {
            s->beta = rho1 / s->rho;
            s->rho = rho1;
        }
        s->k += 1;
        s->cg_total += 1;
        const int go = (rho1 > s->thresh2_in) && (rho1 != 0.0) && (s->k < s->max_cg);
        s->inner_go = go;
        set_cond(a.cond, -1, go);
    }
};

// delta += alpha_prev * p_last for the update an even last CG iteration left pending (no-op otherwise); K2, which runs
// next, clears the flag.  One 16-byte chunk per thread step, grid-stride.
template <typename T>
__global__ void flush_delta_kernel(long long npad, T* __restrict__ delta, const T* p0, const T* p1, const Scalars* sc)
{
    if (!sc->pend) return;
    constexpr int V = 16 / (int)sizeof(T);
    const int k = sc->k;                             // iterations done; the pending one is k - 1 (even)
    const T* __restrict__ p = ((k - 1) & 1) ? p0 : p1;        // p_{k-1} lives in pbuf[((k-1) & 1) ^ 1]
    const T al = (T)sc->alpha_prev;
    const bool first = (k == 1);
    for (long long c = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * V; c < npad;
         c += (long long)gridDim.x * blockDim.x * V) {
        T pv[V], dv[V];
        ld_chunk<T, V>(p + c, pv);
        if (first) zero_chunk<T, V>(dv); else ld_chunk<T, V>(delta + c, dv);
#pragma unroll
        for (int i = 0; i < V; ++i) dv[i] += al * pv[i];
        st_chunk<T, V>(delta + c, dv);
    }
}

// ------------------------------------------------------------------------------------------------ K2 (TMA)
// outer boundary update (Eq. 12 collapsed): P <- P + delta (into the other P buffer);
// r0 = S - L P with (L P)_C = sum_d v(C+d) t_a (P_C - P_{C+d}) = ([W^{n+1}] - [W^n]) P; eps_R^2 ||S||^2 = ||r0||^2 (Eq. 41).
// P is always fp64 (master pressure, A9), so a lane's 16-byte chunk is 2 cells and the tile is 64 cells wide;
// delta, S, r are T.  Links of unflagged chunks come from the position (box faces); flagged chunks read their link bytes.
__device__ __forceinline__ void lds_pair(uint32_t addr, float (&v)[2])
{
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v[0]), "=f"(v[1]) : "r"(addr));
}
__device__ __forceinline__ void lds_pair(uint32_t addr, double (&v)[2])
{
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v[0]), "=d"(v[1]) : "r"(addr));
}

template <typename T, int BY_, int R_, int D_, int MINB_>
struct OpT2 {
    using VT = double;
    struct TG {
        static constexpr int V = 2, BX = 64, BY = BY_, R = R_, NCW = BY_ / R_, NTHR = 32 * (NCW + 1);
        static constexpr int HXP = 2, PITCH_P = (BX + 2 * HXP) * 8;                      // 544 bytes
        static constexpr int HXD = 16 / (int)sizeof(T), PITCH_D = (BX + 2 * HXD) * (int)sizeof(T);
        static constexpr int BOX_P = (BY_ + 2) * PITCH_P, BOX_D = (BY_ + 2) * PITCH_D;
        static constexpr int TILE_P = (BOX_P + 127) / 128 * 128, TILE_D = (BOX_D + 127) / 128 * 128;
        static constexpr int TILE_S = BY_ * BX * (int)sizeof(T);
    };
    // accumulators: ||r0||^2 in fp64, ||r0 rounded to T||^2 (= rho of the CG), ||delta||^2 and ||P + delta||^2 (Eq. 40)
    enum { V = 2, R = R_, D = D_, DMAX = D_, MINB = MINB_, NACC = 4, TICKET = 2, STAGE_BYTES = TG::TILE_P + TG::TILE_D + TG::TILE_S,
           SMEM_BYTES = D_ * STAGE_BYTES };
    static constexpr bool REV = false;
    struct Args {
        double* Pbuf[2]; T* r; const uint8_t* link; const uint32_t* flags; const uint32_t* tflags;
        double t[3]; Scalars* sc; double* partial; CondHandles cond;
        int fold_delta;   // 0: residual of P as given (omni_residual); 1: inside the solve
    };
    struct Ctx {
        int par; double* Pout; bool dz, want_p;
        __device__ Ctx(const Args& a) : Ctx(a, a.sc->n, a.sc->dzero) {}
        __device__ Ctx(const Args& a, int n, int dzero)
        {
            par = a.fold_delta ? (n & 1) : 0; Pout = a.Pbuf[par ^ 1];
            dz = !a.fold_delta || dzero != 0;             // delta counts as zero: neither loaded nor added
            want_p = a.sc->hist_p != nullptr;             // Eq. 40 history asked for: two more sums
        }
    };
    // thread constant: link bytes of an unflagged chunk as far as x decides (box faces normal to x, pad cells)
    using TC = uint32_t;
    __device__ static TC thread_init(const Geom& g, int x)
    {
        uint32_t lk = 0;
#pragma unroll
        for (int i = 0; i < V; ++i) {
            const int gi = x + i;
            uint32_t l = 0x7fu;
            if (g.naxes == 2) l &= ~48u;
            if (g.fix[0]) {
                if (gi == 0) l &= ~2u;
                if (gi == g.nx - 1) l &= ~1u;
                if (gi >= g.nx) l = 0;
            }
            lk |= l << (8 * i);
        }
        return lk;
    }
    __device__ static int stages(const Ctx&) { return D; }
    __device__ static int stage_bytes(const Ctx&) { return STAGE_BYTES; }
    __device__ static bool active(const Args& a) { return a.sc->outer_go != 0; }
    __device__ static void idle(const Args& a) { set_cond(a.cond, 0, 0); }
    __device__ static void load_codes(const Args& a, long long cell, uint32_t (&code)[V])
    {
        code[0] = *reinterpret_cast<const unsigned short*>(a.link + cell);
        code[1] = 0u;
    }
    __device__ static void produce(const Args&, const Ctx& c, const TmaSet& m, uint32_t stage, uint32_t bar, int x0, int y0,
                                   int plane, bool inner)
    {
        mbar_expect_tx(bar, TG::BOX_P + (c.dz ? 0 : TG::BOX_D) + (inner ? TG::TILE_S : 0));
        tma_load_3d(stage, &m.P_h[c.par], bar, x0 - TG::HXP, y0 - 1, plane);
        if (!c.dz) tma_load_3d(stage + TG::TILE_P, &m.d2_h, bar, x0 - TG::HXD, y0 - 1, plane);
        if (inner) tma_load_3d(stage + TG::TILE_P + TG::TILE_D, &m.S_c, bar, x0, y0, plane);
    }
    struct State {};
    __device__ static void advance(State&, const Ctx&, uint32_t, int, int) {}
    __device__ static void value(uint32_t st, int offP, int offD, bool dz, double (&v)[V])
    {
        double P[2]; T d[2] = { T(0), T(0) };
        lds_pair(st + offP, P);
        if (!dz) lds_pair(st + TG::TILE_P + offD, d);
        v[0] = P[0] + (double)d[0];
        v[1] = P[1] + (double)d[1];
    }
    __device__ static void delta_of(uint32_t st, int offD, bool dz, double (&dd)[V])
    {
        T d[2] = { T(0), T(0) };
        if (!dz) lds_pair(st + TG::TILE_P + offD, d);
        dd[0] = (double)d[0]; dd[1] = (double)d[1];
    }
    template <bool CLEAN>
    __device__ static void emit(const Args& a, const Ctx& c, const State&, long long idx, int px, uint32_t sB, uint32_t sC, uint32_t sF,
                                int warp, int lane, const bool (&out)[R], const uint32_t (&fb)[R], const uint32_t (&code)[R][V],
                                const TC& lk_x, const int (&ycls)[R], int zcls, double (&acc)[4])
    {
        const int rowP0 = (warp * R + 1) * TG::PITCH_P, rowD0 = (warp * R + 1) * TG::PITCH_D;
        const int xP = (TG::HXP + lane * V) * 8, xD = (TG::HXD + lane * V) * (int)sizeof(T);
        // P + delta of rows j0-1 .. j0+R of the emitted plane
        double rows[R + 2][V];
#pragma unroll
        for (int q = 0; q < R + 2; ++q) value(sC, rowP0 + (q - 1) * TG::PITCH_P + xP, rowD0 + (q - 1) * TG::PITCH_D + xD, c.dz, rows[q]);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const double (&vc)[V] = rows[r + 1];
            const double (&vn)[V] = rows[r + 2];
            const double (&vs)[V] = rows[r];
            const int rowP = rowP0 + r * TG::PITCH_P, rowD = rowD0 + r * TG::PITCH_D;
            double vm[V], vp[V];
            value(sF, rowP + xP, rowD + xD, c.dz, vp);
            value(sB, rowP + xP, rowD + xD, c.dz, vm);
            double hl = lds_scalar(sC + rowP + (TG::HXP - 1) * 8, double());
            double hr = lds_scalar(sC + rowP + (TG::HXP + TG::BX) * 8, double());
            if (!c.dz) {
                hl += (double)lds_scalar(sC + TG::TILE_P + rowD + (TG::HXD - 1) * (int)sizeof(T), T());
                hr += (double)lds_scalar(sC + TG::TILE_P + rowD + (TG::HXD + TG::BX) * (int)sizeof(T), T());
            }
            double xl = __shfl_up_sync(0xffffffffu, vc[V - 1], 1);
            double xr = __shfl_down_sync(0xffffffffu, vc[0], 1);
            if (lane == 0) xl = hl;
            if (lane == 31) xr = hr;
            if (!out[r]) continue;
            const long long cell = idx + (long long)r * px;
            if (a.fold_delta) st_chunk<double, V>(c.Pout + cell, vc);
            uint32_t lk = lk_x;
            if (ycls[r] == 0) lk &= ~0x0808u;       // row 0: no S link; last row: no N link (faces normal to y)
            if (ycls[r] == 3) lk &= ~0x0404u;
            if (zcls == 0) lk &= ~0x2020u;          // first plane: no B link; last plane: no F link
            if (zcls == 3) lk &= ~0x1010u;
            if (!CLEAN && fb[r]) lk = code[r][0];
            T S[2];
            lds_pair(sC + TG::TILE_P + TG::TILE_D + ((warp * R + r) * TG::BX + lane * V) * (int)sizeof(T), S);
            double dd[V] = { 0.0, 0.0 };
            if (c.want_p) delta_of(sC, rowD + xD, c.dz, dd);
            T rn[V];
#pragma unroll
            for (int i = 0; i < V; ++i) {
                const double w = (i == 0) ? xl : vc[0];
                const double ee = (i == V - 1) ? xr : vc[1];
                const uint32_t l = (lk >> (8 * i)) & 0xffu;
                double LP = 0.0;
                if (l & 1u) LP += a.t[0] * (vc[i] - ee);
                if (l & 2u) LP += a.t[0] * (vc[i] - w);
                if (l & 4u) LP += a.t[1] * (vc[i] - vn[i]);
                if (l & 8u) LP += a.t[1] * (vc[i] - vs[i]);
                if (l & 16u) LP += a.t[2] * (vc[i] - vp[i]);
                if (l & 32u) LP += a.t[2] * (vc[i] - vm[i]);
                const double rr = (l & LINK_VALID) ? ((double)S[i] - LP) : 0.0;
                rn[i] = (T)rr;
                acc[0] += rr * rr;
                acc[1] += (double)rn[i] * (double)rn[i];
                if (c.want_p && (l & LINK_VALID)) { acc[2] += dd[i] * dd[i]; acc[3] += vc[i] * vc[i]; }
            }
            st_chunk<T, V>(a.r + cell, rn);
        }
    }
    __device__ static void finalize(const Args& a, const double (&tot)[4])
    {
        Scalars* s = a.sc;
        s->epsR2 = tot[0];
        if (!a.fold_delta) return;
        record_history(s, tot[0], s->k, tot[2], tot[3]);
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
        s->pend = 0;
        s->beta = 0.0;
        s->rho = tot[1];
        s->thresh2_in = fmax(s->thresh2, s->inner_rel2 * tot[1]);
        const int go = (tot[1] > s->thresh2_in) && (tot[1] != 0.0) && (s->max_cg > 0);
        s->inner_go = go;
        s->dzero = !go;      // an inner loop that does not start leaves the old delta behind: the next K2 must not fold it again
        set_cond(a.cond, 1, go);
    }
};

}  // namespace omni
