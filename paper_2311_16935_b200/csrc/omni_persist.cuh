// omni_persist.cuh -- the whole two-level iteration (Alg. 1) as ONE persistent cooperative kernel,
// for grids whose state is L2-resident and whose K2/K3/K4 launches are latency-, not bandwidth-bound.
//
// Same per-cell arithmetic as the tile kernels of omni_tma.cuh (the operator helpers of omni_kernels.cuh are shared),
// same phase order (K2 ; { K3 ; K4 }*), same stopping rules; the phases are separated by a grid barrier that doubles
// as the deterministic reduction point: every CTA leaves its fp64 partial in a slot, crosses the barrier, and sums all
// slots in the same fixed order, so all CTAs hold bit-identical scalars (alpha, beta, the loop tests) in registers and
// take the same control decisions with no further communication.  Two barriers per CG iteration, one per outer check.
// Vectors written by other CTAs are read with ld.global.cg (L2), never through a possibly stale L1 line.
#pragma once
#include "omni_kernels.cuh"

namespace omni {

template <typename T>
struct PersistArgs {
    T* r; T* pbuf[2]; T* delta; const T* S; double* Pbuf[2];
    const uint8_t* link; const uint32_t* wcode; const uint32_t* flags;
    Coef<T> K; double t[3];
    Scalars* sc; double* slots;             // slots[2][2][2][gridDim.x]: [region][set][accumulator][CTA], tagged values; zero at launch
    unsigned long long timeout_ns;          // longest wait at a grid barrier before the kernel gives up (status OMNI_ERR_CUDA)
};


constexpr int PERSIST_MAX_CTAS = 1024;
constexpr size_t PERSIST_SLOT_BYTES = (size_t)2 * 2 * 2 * PERSIST_MAX_CTAS * 8;
constexpr int ST_BARRIER_TIMEOUT = -2;      // = OMNI_ERR_CUDA: a CTA waited longer than PersistArgs::timeout_ns at a grid barrier

#ifndef OMNI_PERSIST_LDCG
#define OMNI_PERSIST_LDCG 0
#endif
template <typename T> __device__ __forceinline__ T ldd(const T* p) { return OMNI_PERSIST_LDCG ? __ldcg(p) : *reinterpret_cast<const volatile T*>(p); }
template <typename T, int V>
__device__ __forceinline__ void ldcg_chunk(const T* p, T (&v)[V])
{
    constexpr int BYTES = V * (int)sizeof(T);
    static_assert(BYTES == 8 || BYTES == 16, "persistent path moves 8- or 16-byte chunks");
    // plain (coherent) loads: never the non-coherent path, these arrays are rewritten by other CTAs between phases
    // (plain L1-cached loads behind the barrier's acquire were measured: 3-7 % faster, not worth leaving the coherent path)
    if constexpr (BYTES == 8) {
        uint2 u;
        if (OMNI_PERSIST_LDCG) u = __ldcg(reinterpret_cast<const uint2*>(p));
        else asm volatile("ld.global.v2.u32 {%0, %1}, [%2];" : "=r"(u.x), "=r"(u.y) : "l"(p) : "memory");
        memcpy(v, &u, 8);
    } else {
        uint4 u;
        if (OMNI_PERSIST_LDCG) u = __ldcg(reinterpret_cast<const uint4*>(p));
        else asm volatile("ld.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(u.x), "=r"(u.y), "=r"(u.z), "=r"(u.w) : "l"(p) : "memory");
        memcpy(v, &u, 16);
    }
}

__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ unsigned long long global_timer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}

// Grid barrier + all-reduce of NACC fp64 accumulators in one exchange.  Each CTA publishes its partial in its own
// 8-byte slot with st.release.gpu; the mantissa's last bit carries the use count's parity (the partial loses that bit:
// 1e-16 relative, below the rounding of the sum itself), so one single-copy-atomic word is both the value and its
// arrival flag: no counter, no second round trip.  Warp 0 of every CTA polls all slots with ld.acquire.gpu and sums
// them in the same fixed order, so every CTA gets the same bits.  Slots alternate between two sets by barrier parity
// (a CTA can be at most one barrier ahead of the slowest reader), each set flips its tag on every use.
// Release: the publishing lane's st.release follows the CTA-wide barrier that follows the phase's stores (cumulative);
// acquire: warp 0's ld.acquire precede the CTA-wide barrier that releases the other warps to their loads.
// Returns false if a slot did not arrive within gs.timeout_ns (a CTA is not resident or died): every CTA then leaves
// the kernel.
struct GridSync {
    // Two slot regions with their own use counts: [0] the CG barriers (K3, K4: one accumulator), [1] the outer barrier
    // (K2: two accumulators) -- a slot's tag must flip on each of ITS uses, so barriers that publish different numbers
    // of accumulators cannot share a region.  Counts start at 2: set = count & 1, tag = (count >> 1) & 1; between two
    // uses of the same set of a region lies one full barrier of that region, which every reader of the first has left.
    unsigned int count[2];
    double* red;                     // shared: [2][NW + 1]
    int* flag;                       // shared
    unsigned long long timeout_ns;
};

template <bool RELAXED = false>
__device__ __forceinline__ void slot_publish(double* slot, double v, unsigned int tag)
{
    const unsigned long long b = ((unsigned long long)__double_as_longlong(v) & ~1ULL) | tag;
    if (RELAXED) asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" :: "l"(slot), "l"(b) : "memory");
    else asm volatile("st.release.gpu.global.u64 [%0], %1;" :: "l"(slot), "l"(b) : "memory");
}
// RELAXED (omni_resident.cuh): no data other than the slot itself crosses the barrier, so neither side needs a fence
template <bool RELAXED = false>
__device__ __forceinline__ bool slot_poll(const double* slot, unsigned int tag, double& v)
{
    unsigned long long b;
    if (RELAXED) asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(b) : "l"(slot) : "memory");
    else asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(b) : "l"(slot) : "memory");
    v = __longlong_as_double((long long)(b & ~1ULL));
    return (unsigned int)(b & 1ULL) == tag;
}

template <int NACC, int NT, bool RELAXED = false>
__device__ __forceinline__ bool grid_allreduce(GridSync& gs, double* slots, const double (&acc)[NACC], double (&tot)[NACC])
{
    constexpr int R = NACC - 1;                                    // region: 0 for one accumulator, 1 for two
    static_assert(NACC == 1 || NACC == 2, "regions are keyed by the accumulator count");
    constexpr int NW = NT / 32, PB = 5;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned int G = gridDim.x, tag = (gs.count[R] >> 1) & 1u;
    double* my = slots + ((size_t)R * 2 + (gs.count[R] & 1u)) * 2 * G;   // [region][set][accumulator][CTA]
#pragma unroll
    for (int i = 0; i < NACC; ++i) {
        const double s = warp_sum(acc[i]);
        if (lane == 0) gs.red[i * (NW + 1) + warp] = s;
    }
    __syncthreads();                                               // every store of the phase is issued
    if (warp == 0) {
        int ok = 1;
#pragma unroll
        for (int i = 0; i < NACC; ++i) {
            const double s = warp_sum(lane < NW ? gs.red[i * (NW + 1) + lane] : 0.0);
            if (lane == 0) slot_publish<RELAXED>(my + (size_t)i * G + blockIdx.x, s, tag);
        }
#pragma unroll
        for (int i = 0; i < NACC; ++i) {
            // a lane's slots are fetched PB at a time with independent loads; the late ones are polled again
            double s = 0.0;
            for (unsigned int b0 = lane; b0 < G; b0 += 32 * PB) {
                double v[PB];
                bool got[PB];
#pragma unroll
                for (int u = 0; u < PB; ++u) {
                    const unsigned int b = b0 + 32 * u;
                    v[u] = 0.0;
                    got[u] = (b >= G) || slot_poll<RELAXED>(my + (size_t)i * G + b, tag, v[u]);
                }
#pragma unroll
                for (int u = 0; u < PB; ++u) {
                    if (!got[u]) {
                        const double* sl = my + (size_t)i * G + b0 + 32 * u;
                        const unsigned long long t0 = global_timer_ns();
                        while (!slot_poll<RELAXED>(sl, tag, v[u])) {
                            if (global_timer_ns() - t0 > gs.timeout_ns) { ok = 0; break; }
                        }
                    }
                    s += v[u];                                     // fixed order: b0, b0 + 32, ...
                }
            }
            s = warp_sum(s);                                       // xor butterfly: the same bits in every lane and CTA
            if (lane == 0) gs.red[i * (NW + 1) + NW] = s;
        }
        ok = __all_sync(0xffffffffu, ok);
        if (lane == 0) *gs.flag = ok;
    }
    __syncthreads();
    if (!*gs.flag) return false;
#pragma unroll
    for (int i = 0; i < NACC; ++i) tot[i] = gs.red[i * (NW + 1) + NW];
    __syncthreads();                                               // red / flag are reused by the next reduction
    gs.count[R] += 1u;
    return true;
}

// one warp task = 32 consecutive chunks of one grid row; a warp walks its tasks t0, t0 + NW, ... without divisions
template <int V>
struct RowTask {
    int seg, j, k, nsx, dseg, drow;
    int x;
    long long idx;
    bool inb, out;
    __device__ __forceinline__ RowTask(const Geom& g, int t0, int nsx_, int step, int lane)   // task counts < 2^31 (host)
    {
        nsx = nsx_;
        seg = t0 % nsx;
        const int row = t0 / nsx;
        j = row % g.ny;
        k = row / g.ny;
        dseg = step % nsx;
        drow = step / nsx;
        place(g, lane);
    }
    __device__ __forceinline__ void place(const Geom& g, int lane)
    {
        x = (seg * 32 + lane) * V;
        inb = x < g.px;
        out = x < g.nx;
        idx = (long long)x + (long long)g.px * (j + (long long)g.ny * k);
    }
    __device__ __forceinline__ void next(const Geom& g, int lane)
    {
        seg += dseg;
        j += drow;
        if (seg >= nsx) { seg -= nsx; j += 1; }
        while (j >= g.ny) { j -= g.ny; k += 1; }
        place(g, lane);
    }
};

// K2 phase of the persistent kernels on the row tasks [lo2, hi2) of this CTA: Pout = Pin + delta (unless dzero),
// r = S - L Pout written to rout; acc = { ||r||^2 in fp64, ||r rounded to T||^2 }, accp = { ||delta||^2, ||Pout||^2 } if want_p
template <typename T>
__device__ __forceinline__ void persist_k2_rows(const Geom& g, const PersistArgs<T>& a, T* __restrict__ rout, const double* Pin,
                                                double* Pout, bool dzero, bool want_p, int lo2, int hi2, int wfirst, int wstep,
                                                int nsx2, int lane, double (&acc)[2], double (&accp)[2])
{
    const bool three = g.naxes == 3;
    const long long pp = g.pplane;
    RowTask<2> tk(g, lo2 + wfirst, nsx2, wstep, lane);
    for (int t = lo2 + wfirst; t < hi2; t += wstep, tk.next(g, lane)) {
        auto val = [&](long long i, bool ok, double (&v)[2]) {
            v[0] = v[1] = 0.0;
            if (ok) {
                double P[2]; T d[2] = { T(0), T(0) };
                ldcg_chunk<double, 2>(Pin + i, P);
                if (!dzero) ldcg_chunk<T, 2>(a.delta + i, d);
                v[0] = P[0] + (double)d[0];
                v[1] = P[1] + (double)d[1];
            }
        };
        auto val1 = [&](long long i) { return ldd(Pin + i) + (dzero ? 0.0 : (double)ldd(a.delta + i)); };
        // every load of the task is issued before the first use
        uint32_t fw = 0, lkb = 0;
        T S[2] = { T(0), T(0) };
        if (tk.out) {
            fw = flag_bits<2>(a.flags, tk.idx);
            lkb = *reinterpret_cast<const unsigned short*>(a.link + tk.idx);
            ld_chunk<T, 2>(a.S + tk.idx, S);
        }
        double vm[2], vc[2], vp[2], vn[2], vs[2];
        val(tk.idx, tk.inb, vc);
        val(tk.idx + g.px, tk.inb && tk.j + 1 < g.ny, vn);
        val(tk.idx - g.px, tk.inb && tk.j > 0, vs);
        val(tk.idx + pp, tk.inb && three && tk.k + 1 < g.nz, vp);
        val(tk.idx - pp, tk.inb && three && tk.k > 0, vm);
        double xl = __shfl_up_sync(0xffffffffu, vc[1], 1);
        double xr = __shfl_down_sync(0xffffffffu, vc[0], 1);
        if (lane == 0) xl = (tk.x > 0) ? val1(tk.idx - 1) : 0.0;
        if (lane == 31) xr = (tk.x + 2 < g.px) ? val1(tk.idx + 2) : 0.0;
        if (!tk.out) continue;
        st_chunk<double, 2>(Pout + tk.idx, vc);
        uint32_t lk = 0;
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int gi = tk.x + i;
            uint32_t l = 0x7fu;
            if (!three) l &= ~48u;
            if (g.fix[0]) {
                if (gi == 0) l &= ~2u;
                if (gi == g.nx - 1) l &= ~1u;
                if (gi >= g.nx) l = 0;
            }
            lk |= l << (8 * i);
        }
        const int ycls = face_class(tk.j, g.ny, g.fix[1]), zcls = face_class(tk.k, g.nz, g.fix[2]);
        if (ycls == 0) lk &= ~0x0808u;
        if (ycls == 3) lk &= ~0x0404u;
        if (zcls == 0) lk &= ~0x2020u;
        if (zcls == 3) lk &= ~0x1010u;
        if (fw) lk = lkb;
        T rn[2];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const double w = (i == 0) ? xl : vc[0];
            const double ee = (i == 1) ? xr : vc[1];
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
            if (want_p && (l & LINK_VALID)) accp[1] += vc[i] * vc[i];
        }
        if (want_p && !dzero) {
            T d[2];
            ldcg_chunk<T, 2>(a.delta + tk.idx, d);
#pragma unroll
            for (int i = 0; i < 2; ++i)
                if ((lk >> (8 * i)) & LINK_VALID) accp[0] += (double)d[i] * (double)d[i];
        }
        st_chunk<T, 2>(rout + tk.idx, rn);
    }
}

template <typename T, int NT, bool LOP>
__global__ void __launch_bounds__(NT, 1)
persist_kernel(const Geom g, const PersistArgs<T> a)
{
    constexpr int V = 16 / (int)sizeof(T);
    constexpr int NW = NT / 32;
    __shared__ double red[2 * (NW + 1)];
    __shared__ int flag;
    Scalars* sc = a.sc;
    if (!sc->outer_go) return;                             // zero source: nothing to iterate (A4)

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nsx = (g.nx + 32 * V - 1) / (32 * V), nsx2 = (g.nx + 63) / 64;
    const long long rows = (long long)g.ny * g.nz;
    const long long ntask = rows * nsx, ntask2 = rows * nsx2;
    // each CTA owns a contiguous run of row segments (neighbouring rows share the CTA, hence L1 / L2 sectors)
    const int lo1 = (int)(ntask * blockIdx.x / gridDim.x), hi1 = (int)(ntask * (blockIdx.x + 1) / gridDim.x);
    const int lo2 = (int)(ntask2 * blockIdx.x / gridDim.x), hi2 = (int)(ntask2 * (blockIdx.x + 1) / gridDim.x);
    const int wfirst = warp, wstep = NW;
    const bool three = g.naxes == 3;
    const long long pp = g.pplane;

    GridSync gs{ { 2u, 2u }, red, &flag, a.timeout_ns };

    // loop state, identical in every thread of the grid
    const double thresh2 = sc->thresh2, tol2S = sc->tol2S;
    const int max_cg = sc->max_cg, max_outer = sc->max_outer;
    int n = sc->n, k = 0, status = ST_OK;
    long long cg_total = 0;
    double rho = 0.0, beta = 0.0, alpha = 0.0, gamma = 0.0, epsR2 = 0.0;
    bool dzero = sc->dzero != 0;                 // delta counts as zero in the next K2 (Scalars::dzero)

    for (;;) {
        // ------------------------------------------------------------------------------ K2: P += delta, r = S - L P
        {
            const int par = n & 1;
            const double* Pin = a.Pbuf[par];
            double* Pout = a.Pbuf[par ^ 1];
            double acc[2] = { 0.0, 0.0 }, accp[2] = { 0.0, 0.0 };
            const bool want_p = sc->hist_p != nullptr;             // Eq. 40 history asked for (grid-uniform)
            persist_k2_rows<T>(g, a, a.r, Pin, Pout, dzero, want_p, lo2, hi2, wfirst, wstep, nsx2, lane, acc, accp);
            double tot[2], totp[2] = { 0.0, 0.0 };
            if (!grid_allreduce<2, NT>(gs, a.slots, acc, tot)) { status = ST_BARRIER_TIMEOUT; break; }
            if (want_p && !grid_allreduce<2, NT>(gs, a.slots, accp, totp)) { status = ST_BARRIER_TIMEOUT; break; }
            epsR2 = tot[0];
            if (blockIdx.x == 0 && threadIdx.x == 0) record_history(sc, tot[0], k, totp[0], totp[1]);
            if (!isfinite(tot[0])) { status = ST_BREAKDOWN; break; }
            if (tot[0] <= tol2S || n >= max_outer) { status = (tot[0] <= tol2S) ? ST_OK : ST_NOT_CONVERGED; break; }
            n += 1;
            k = 0;
            beta = 0.0;
            rho = tot[1];
            // an inner loop that does not start leaves the old delta behind: the next K2 must not fold it again
            dzero = !((tot[1] > thresh2) && (tot[1] != 0.0) && (max_cg > 0));
            if (dzero) continue;
        }
        // ------------------------------------------------------------------------------ inner CG on M delta = r0
        bool stop_all = false;
        for (;;) {
            const int par = k & 1;
            const T* pold = a.pbuf[par];
            T* pnew = a.pbuf[par ^ 1];
            // ---- K3: p_new = r + beta p_old (recomputed at the stencil's neighbours), gamma = p_new . M p_new
            {
                const T b = (T)beta;
                double acc[1] = { 0.0 };
                RowTask<V> tk(g, lo1 + wfirst, nsx, wstep, lane);
                for (int t = lo1 + wfirst; t < hi1; t += wstep, tk.next(g, lane)) {
                    auto pn = [&](long long i, bool ok, T (&v)[V]) {
                        zero_chunk<T, V>(v);
                        if (ok) {
                            T r[V], p[V];
                            ldcg_chunk<T, V>(a.r + i, r);
                            ldcg_chunk<T, V>(pold + i, p);
#pragma unroll
                            for (int c = 0; c < V; ++c) v[c] = r[c] + b * p[c];
                        }
                    };
                    auto pn1 = [&](long long i) { return ldd(a.r + i) + b * ldd(pold + i); };
                    uint32_t fb = 0, code[V];
#pragma unroll
                    for (int c = 0; c < V; ++c) code[c] = 0u;
                    if (tk.out) {
                        fb = flag_bits<V>(a.flags, tk.idx);
                        if (fb) load_cell_codes<LOP, V>(a.wcode, a.link, tk.idx, code);
                    }
                    T vm[V], vc[V], vp[V], vn[V], vs[V];
                    pn(tk.idx, tk.inb, vc);
                    pn(tk.idx + g.px, tk.inb && tk.j + 1 < g.ny, vn);
                    pn(tk.idx - g.px, tk.inb && tk.j > 0, vs);
                    pn(tk.idx + pp, tk.inb && three && tk.k + 1 < g.nz, vp);
                    pn(tk.idx - pp, tk.inb && three && tk.k > 0, vm);
                    T xl = __shfl_up_sync(0xffffffffu, vc[V - 1], 1);
                    T xr = __shfl_down_sync(0xffffffffu, vc[0], 1);
                    if (lane == 0) xl = (tk.x > 0) ? pn1(tk.idx - 1) : T(0);
                    if (lane == 31) xr = (tk.x + V < g.px) ? pn1(tk.idx + V) : T(0);
                    if (!tk.out) continue;
                    st_chunk<T, V>(pnew + tk.idx, vc);
                    const XEdge xe = make_xedge<V>(g, tk.x);
                    T q[V];
                    apply_op_chunk<LOP, T, V>(q, vm, vc, vp, vn, vs, xl, xr, fb, code, a.K, xe, face_class(tk.j, g.ny, g.fix[1]),
                                        face_class(tk.k, g.nz, g.fix[2]));
#pragma unroll
                    for (int c = 0; c < V; ++c) acc[0] += (double)vc[c] * (double)q[c];
                }
                double tot[1];
                if (!grid_allreduce<1, NT>(gs, a.slots, acc, tot)) { status = ST_BARRIER_TIMEOUT; stop_all = true; break; }
                gamma = tot[0];
                if (!(gamma > 0.0) || !isfinite(gamma)) { status = ST_BREAKDOWN; stop_all = true; break; }
                alpha = rho / gamma;
            }
            // ---- K4: q = M p recomputed; delta += alpha p; r -= alpha q; rho' = r . r
            {
                const T al = (T)alpha;
                const bool first = (k == 0);
                double acc[1] = { 0.0 };
                RowTask<V> tk(g, lo1 + wfirst, nsx, wstep, lane);
                for (int t = lo1 + wfirst; t < hi1; t += wstep, tk.next(g, lane)) {
                    auto ld = [&](long long i, bool ok, T (&v)[V]) {
                        zero_chunk<T, V>(v);
                        if (ok) ldcg_chunk<T, V>(pnew + i, v);
                    };
                    uint32_t fb = 0, code[V];
                    T er[V], ed[V];
#pragma unroll
                    for (int c = 0; c < V; ++c) code[c] = 0u;
                    zero_chunk<T, V>(er); zero_chunk<T, V>(ed);
                    if (tk.out) {
                        fb = flag_bits<V>(a.flags, tk.idx);
                        if (fb) load_cell_codes<LOP, V>(a.wcode, a.link, tk.idx, code);
                        ldcg_chunk<T, V>(a.r + tk.idx, er);
                        if (!first) ldcg_chunk<T, V>(a.delta + tk.idx, ed);
                    }
                    T vm[V], vc[V], vp[V], vn[V], vs[V];
                    ld(tk.idx, tk.inb, vc);
                    ld(tk.idx + g.px, tk.inb && tk.j + 1 < g.ny, vn);
                    ld(tk.idx - g.px, tk.inb && tk.j > 0, vs);
                    ld(tk.idx + pp, tk.inb && three && tk.k + 1 < g.nz, vp);
                    ld(tk.idx - pp, tk.inb && three && tk.k > 0, vm);
                    T xl = __shfl_up_sync(0xffffffffu, vc[V - 1], 1);
                    T xr = __shfl_down_sync(0xffffffffu, vc[0], 1);
                    if (lane == 0) xl = (tk.x > 0) ? ldd(pnew + tk.idx - 1) : T(0);
                    if (lane == 31) xr = (tk.x + V < g.px) ? ldd(pnew + tk.idx + V) : T(0);
                    if (!tk.out) continue;
                    const XEdge xe = make_xedge<V>(g, tk.x);
                    T q[V];
                    apply_op_chunk<LOP, T, V>(q, vm, vc, vp, vn, vs, xl, xr, fb, code, a.K, xe, face_class(tk.j, g.ny, g.fix[1]),
                                        face_class(tk.k, g.nz, g.fix[2]));
                    T rn[V], dn[V];
#pragma unroll
                    for (int c = 0; c < V; ++c) {
                        rn[c] = er[c] - al * q[c];
                        dn[c] = ed[c] + al * vc[c];
                        acc[0] += (double)rn[c] * (double)rn[c];
                    }
                    st_chunk<T, V>(a.r + tk.idx, rn);
                    st_chunk<T, V>(a.delta + tk.idx, dn);
                }
                double tot[1];
                if (!grid_allreduce<1, NT>(gs, a.slots, acc, tot)) { status = ST_BARRIER_TIMEOUT; stop_all = true; break; }
                const double rho1 = tot[0];
                if (!isfinite(rho1)) { status = ST_BREAKDOWN; stop_all = true; break; }
                beta = rho1 / rho;
                rho = rho1;
                k += 1;
                cg_total += 1;
                if (!((rho1 > thresh2) && (rho1 != 0.0) && (k < max_cg))) break;
            }
        }
        if (stop_all) break;
    }

    if (blockIdx.x == 0 && threadIdx.x == 0) {
        sc->n = n; sc->k = k; sc->cg_total = cg_total; sc->status = status;
        sc->rho = rho; sc->beta = beta; sc->alpha = alpha; sc->gamma = gamma; sc->epsR2 = epsR2;
        sc->inner_go = 0; sc->outer_go = 0;
    }
}

}  // namespace omni
