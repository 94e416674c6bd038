// omni_loop.cuh -- the whole two-level iteration (Alg. 1) as ONE cooperative launch of the TMA tile
// pipeline, for grids between the L2-resident ones (persist_kernel, omni_persist.cuh: plain loads) and the multi-wave
// ones (one launch per kernel under the conditional graph, omni_tma.cuh).
//
// At 128^3 - 256^3 a K3 or K4 launch lasts 17 - 120 us, of which 10 - 18 us are launch latency, pipeline fill, the
// drain of the last wave and the last-CTA reduction.  Here every CTA keeps ONE column (tile x
// z segment) for the whole solve: the grid is one wave by construction (cooperative launch: tiles x segments <=
// resident CTA slots), every reduction is the tagged-slot grid barrier + all-reduce of omni_persist.cuh (all CTAs end up
// with bit-identical alpha, beta, eps_R and loop decisions in registers), and K4 marches its column downwards, starting
// on the planes K3 has just left in L2, K3 upwards again from where K4 ended.
// The phases run the same Op code as the stand-alone kernels (run_column<K2 / K3 / K4>): same arithmetic per cell; the
// reductions add the per-CTA partials in another (fixed) order, like persist_kernel.
//
// Memory ordering between phases: a phase's global stores (generic proxy) are read by other CTAs' TMA loads (async
// proxy) in the next phase.  Writers: stores -> fence.proxy.async -> CTA barrier -> st.release.gpu of the slot;
// readers: ld.acquire.gpu of all slots -> CTA barrier -> fence.proxy.async -> TMA issue.
#pragma once
#include "omni_tma.cuh"
#include "omni_persist.cuh"

namespace omni {

template <class K2, class K3, class K4>
struct LoopArgs {
    typename K2::Args a2;
    typename K3::Args a3;
    typename K4::Args a4;
    double* slots;                       // grid-barrier slots (PERSIST_SLOT_BYTES, zeroed at launch)
    unsigned long long timeout_ns;
};

#ifdef OMNI_TUNING   // tuning builds only: per-CTA timeline of the first phases (phase start, end of the column pass, end of the barrier)
__device__ unsigned long long g_loop_trace[64][1024][3];
__device__ int g_loop_trace_n;
#define LOOP_TRACE_BEGIN() const unsigned long long tr0__ = dbg_timer();
#define LOOP_TRACE_MID() const unsigned long long tr1__ = dbg_timer();
#define LOOP_TRACE_END(ph) do { if (threadIdx.x == 0 && (ph) < 64 && blockIdx.x < 1024) { g_loop_trace[ph][blockIdx.x][0] = tr0__; \
    g_loop_trace[ph][blockIdx.x][1] = tr1__; g_loop_trace[ph][blockIdx.x][2] = dbg_timer(); if (blockIdx.x == 0) g_loop_trace_n = (ph) + 1; } (ph)++; } while (0)
#else
#define LOOP_TRACE_BEGIN()
#define LOOP_TRACE_MID()
#define LOOP_TRACE_END(ph)
#endif

__device__ __forceinline__ void fence_proxy_async_global()
{
    asm volatile("fence.proxy.async.global;" ::: "memory");
}

template <class K2, class K3, class K4, int MINB>
__global__ void __launch_bounds__(K3::TG::NTHR, MINB)
tma_loop_kernel(const Geom g, const ZSeg zs, const LoopArgs<K2, K3, K4> a, const __grid_constant__ TmaSet maps)
{
    using TG = typename K3::TG;
    using T = typename K3::VT;
    static_assert(TG::NTHR == K4::TG::NTHR && TG::BX == K4::TG::BX && TG::BY == K4::TG::BY, "K3 and K4 share the tile");
    static_assert(K2::TG::NTHR == TG::NTHR && K2::TG::BY == TG::BY && K2::TG::R == TG::R && TG::BX % K2::TG::BX == 0, "K2 tiles subdivide it in x");
    constexpr int NT = TG::NTHR, BY = TG::BY, NCW = TG::NCW, R = TG::R, NW = NT / 32, V = TG::V;
    constexpr int XR = TG::BX / K2::TG::BX;          // K2 columns per K3 column (fp32: 2, the fp64 master pressure halves the tile)
    constexpr int NB34 = (K3::DMAX > K4::DMAX) ? K3::DMAX : K4::DMAX;
    constexpr int NBAR = (NB34 > K2::DMAX) ? NB34 : K2::DMAX;
    extern __shared__ __align__(128) char smem_raw[];
    __shared__ double red[2 * (NW + 1)];
    __shared__ int flag;
    __shared__ __align__(8) unsigned long long bars[2 * NBAR];

    Scalars* sc = a.a3.sc;
    if (!sc->outer_go) return;                      // zero source: nothing to iterate (A4)

    char* smem = reinterpret_cast<char*>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~uintptr_t(127));
    const uint32_t smem_s = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t bar_s = (uint32_t)__cvta_generic_to_shared(bars);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // one column per CTA for the whole solve, marched up by K2 and K3, down by K4; 1D grid (the barrier indexes its
    // slots by blockIdx.x)
    const int ntx = (g.px + TG::BX - 1) / TG::BX, nty = (g.ny + BY - 1) / BY;
    const int ntx2 = (g.px + K2::TG::BX - 1) / K2::TG::BX;
    const int tx = blockIdx.x % ntx, ty = (blockIdx.x / ntx) % nty, seg = blockIdx.x / (ntx * nty);
    const int k0 = zs.n ? zs.k[seg] : seg * zs.zlen;
    const int k1 = zs.n ? zs.k[seg + 1] : min(g.nz, k0 + zs.zlen);      // (never used on a slab: kz0 = 0, kz1 = nz)

    GridSync gs{ { 2u, 2u }, red, &flag, a.timeout_ns };

    // loop state, identical in every thread of the grid
    const double thresh2 = sc->thresh2, tol2S = sc->tol2S;
    const int max_cg = sc->max_cg, max_outer = sc->max_outer;
    double rho = 0.0, beta = 0.0, alpha = 0.0, alpha_prev = 0.0, gamma = 0.0, epsR2 = 0.0;
    int n = sc->n, k = 0, pend = 0, dzero = sc->dzero, status = ST_OK;
    long long cg_total = 0;
    bool again = false;
#ifdef OMNI_TUNING
    int trace_ph = 0;
#endif

    for (;;) {
        // ------------------------------------------------------------------ K2: P += delta, r = S - L P, eps_R (Eq. 41)
        {
            const typename K2::Ctx c2(a.a2, n, dzero);
            double acc[4] = { 0.0, 0.0, 0.0, 0.0 }, tot[2];
            LOOP_TRACE_BEGIN()
#pragma unroll 1
            for (int h = 0; h < XR; ++h) {
                const int tx2 = tx * XR + h;
                if (tx2 >= ntx2) break;                                    // CTA-uniform
                if (threadIdx.x == 0) ring_init(bar_s, K2::stages(c2), NBAR, NCW, again);
                again = true;
                fence_proxy_async_global();          // the producer's TMA loads follow the acquire of the last barrier
                __syncthreads();
                run_column<K2>(g, a.a2, c2, maps, smem_s, bar_s, tx2, ty, k0, k1, acc);
                __syncthreads();                     // every warp has left the ring before it is torn down
            }
            fence_proxy_async_global();              // this phase's stores, before the release in the barrier
            LOOP_TRACE_MID()
            const double acc01[2] = { acc[0], acc[1] }, acc23[2] = { acc[2], acc[3] };
            double totp[2] = { 0.0, 0.0 };
            if (!grid_allreduce<2, NT>(gs, a.slots, acc01, tot)) { status = ST_BARRIER_TIMEOUT; break; }
            // Eq. 40 only when its history was asked for (grid-uniform): a second exchange
            if (sc->hist_p != nullptr && !grid_allreduce<2, NT>(gs, a.slots, acc23, totp)) { status = ST_BARRIER_TIMEOUT; break; }
            LOOP_TRACE_END(trace_ph);
            epsR2 = tot[0];
            if (blockIdx.x == 0 && threadIdx.x == 0) record_history(sc, tot[0], k, totp[0], totp[1]);
            if (!isfinite(tot[0])) { status = ST_BREAKDOWN; break; }
            if (tot[0] <= tol2S || n >= max_outer) { status = (tot[0] <= tol2S) ? ST_OK : ST_NOT_CONVERGED; break; }
            n += 1;
            k = 0;
            pend = 0;
            beta = 0.0;
            rho = tot[1];
            // an inner loop that does not start leaves the old delta behind: the next K2 must not fold it again
            dzero = !((tot[1] > thresh2) && (tot[1] != 0.0) && (max_cg > 0));
            if (dzero) continue;
        }
        // ------------------------------------------------------------------ inner CG
        bool stop_all = false;
        for (;;) {
            // ---- K3: p_new = r + beta p_old, gamma = p_new . A p_new
            {
                const typename K3::Ctx c3(a.a3, beta, k);
                LOOP_TRACE_BEGIN()
                if (threadIdx.x == 0) ring_init(bar_s, K3::stages(c3), NBAR, NCW, true);
                fence_proxy_async_global();
                __syncthreads();
                double acc[1] = { 0.0 }, tot[1];
                run_column<K3>(g, a.a3, c3, maps, smem_s, bar_s, tx, ty, k0, k1, acc);
                fence_proxy_async_global();
                LOOP_TRACE_MID()
                if (!grid_allreduce<1, NT>(gs, a.slots, acc, tot)) { status = ST_BARRIER_TIMEOUT; stop_all = true; break; }
                LOOP_TRACE_END(trace_ph);
                gamma = tot[0];
                if (!(gamma > 0.0) || !isfinite(gamma)) { status = ST_BREAKDOWN; stop_all = true; break; }
                alpha = rho / gamma;
            }
            // ---- K4: q = A p_new recomputed, r -= alpha q, rho' = r . r, lazy delta
            {
                const typename K4::Ctx c4(a.a4, alpha, alpha_prev, k);
                LOOP_TRACE_BEGIN()
                if (threadIdx.x == 0) ring_init(bar_s, K4::stages(c4), NBAR, NCW, true);
                fence_proxy_async_global();
                __syncthreads();
                double acc[1] = { 0.0 }, tot[1];
                run_column<K4>(g, a.a4, c4, maps, smem_s, bar_s, tx, ty, k0, k1, acc);
                fence_proxy_async_global();
                LOOP_TRACE_MID()
                if (!grid_allreduce<1, NT>(gs, a.slots, acc, tot)) { status = ST_BARRIER_TIMEOUT; stop_all = true; break; }
                LOOP_TRACE_END(trace_ph);
                const double rho1 = tot[0];
                if (!isfinite(rho1)) { status = ST_BREAKDOWN; stop_all = true; break; }
                if (k & 1) { pend = 0; } else { pend = 1; alpha_prev = alpha; }
                beta = rho1 / rho;
                rho = rho1;
                k += 1;
                cg_total += 1;
                if (!((rho1 > thresh2) && (rho1 != 0.0) && (k < max_cg))) break;
            }
        }
        if (stop_all) break;
        // ------------------------------------------------------------------ pending half of the lazy delta update
        // (an even last CG iteration): delta += alpha_prev p_{k-1} on the own column -- every thread touches the chunks
        // it wrote itself in K3 / K4 -- then a barrier, because K2 reads delta with its halo through TMA
        if (pend) {
            if (warp < NCW) {
                const int x = tx * TG::BX + lane * V;
                const T* __restrict__ p = a.a3.pbuf[((k - 1) & 1) ^ 1];
                const T al = (T)alpha_prev;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int j = ty * BY + warp * R + r;
                    if (x < g.nx && j < g.ny) {
                        long long c = (long long)j * g.px + x + (long long)k0 * g.pplane;
                        for (int kk = k0; kk < k1; ++kk, c += g.pplane) {
                            T pv[V], dv[V];
                            ld_chunk<T, V>(p + c, pv);
                            if (k == 1) zero_chunk<T, V>(dv); else ld_chunk<T, V>(a.a4.delta + c, dv);
#pragma unroll
                            for (int i = 0; i < V; ++i) dv[i] += al * pv[i];
                            st_chunk<T, V>(a.a4.delta + c, dv);
                        }
                    }
                }
            }
            pend = 0;
            fence_proxy_async_global();
            double acc[1] = { 0.0 }, tot[1];
            if (!grid_allreduce<1, NT>(gs, a.slots, acc, tot)) { status = ST_BARRIER_TIMEOUT; break; }
        }
    }

    if (blockIdx.x == 0 && threadIdx.x == 0) {
        sc->n = n; sc->k = k; sc->cg_total = cg_total; sc->status = status; sc->pend = 0; sc->dzero = dzero;
        sc->rho = rho; sc->beta = beta; sc->alpha = alpha; sc->alpha_prev = alpha_prev; sc->gamma = gamma; sc->epsR2 = epsR2;
        sc->inner_go = 0; sc->outer_go = 0;
    }
}

}  // namespace omni
