// omni_persist1.cuh -- the fixed-point solve L P = S (omni_solve_direct_*) with SINGLE-REDUCTION conjugate gradients
// (Chronopoulos & Gear; SURVEY.md 8(d) V5, 8(f) NEXT-2 i) as one persistent cooperative kernel.
//
// persist_kernel (omni_persist.cuh) crosses two grid barriers per CG iteration -- one for gamma = p.Ap, one for
// rho' = r.r -- and on L2-resident grids those barriers ARE the iteration time (2 x ~2.5 us + skew of 6.5 us at 64^2,
// 17 us at 1024^2).  With s = A p carried by the recurrence s = w + beta s (w = A r) both inner products of an iteration,
// gamma' = r.r and delta' = w.r, are taken at the same point: ONE barrier per iteration.  The identity that replaces p.Ap,
// alpha = gamma / (delta - beta gamma / alpha_prev), needs A = A^T: valid for L, NOT for the paper's nonsymmetric M
// (reading A2), so this kernel exists for the fixed-point solve only.
//
// One phase per iteration; a thread forms, for its own chunk AND on the fly for the six neighbouring chunks,
//     s' = w + beta s,  r' = r - alpha s'          (r, w, s of the previous iteration: complete after the last barrier)
// then w' = L r' from those seven r', p' = r + beta p and delta += alpha p' on its own chunk, and the two partial sums.
// r, w, s are double-buffered (neighbours still read the old ones); p and delta are touched at the own chunk only.
// Same stopping rules, same outer (fp64 refinement) phase as persist_kernel: persist_k2_rows.
#pragma once
#include "omni_persist.cuh"

namespace omni {

template <typename T>
struct Persist1Args {
    PersistArgs<T> base;         // S, Pbuf, delta, link, flags, K, t, sc, slots, timeout (r / pbuf unused)
    T* rb[2]; T* wb[2]; T* sb[2]; T* p;
};

template <typename T, int NT>
__global__ void __launch_bounds__(NT, 1)
persist_cg1_kernel(const Geom g, const Persist1Args<T> A)
{
    constexpr int V = 16 / (int)sizeof(T);
    constexpr int NW = NT / 32;
    __shared__ double red[2 * (NW + 1)];
    __shared__ int flag;
    const PersistArgs<T>& a = A.base;
    Scalars* sc = a.sc;
    if (!sc->outer_go) return;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nsx = (g.nx + 32 * V - 1) / (32 * V), nsx2 = (g.nx + 63) / 64;
    const long long rows = (long long)g.ny * g.nz;
    const long long ntask = rows * nsx, ntask2 = rows * nsx2;
    const int lo1 = (int)(ntask * blockIdx.x / gridDim.x), hi1 = (int)(ntask * (blockIdx.x + 1) / gridDim.x);
    const int lo2 = (int)(ntask2 * blockIdx.x / gridDim.x), hi2 = (int)(ntask2 * (blockIdx.x + 1) / gridDim.x);
    const int wfirst = warp, wstep = NW;
    const bool three = g.naxes == 3;
    const long long pp = g.pplane;

    GridSync gs{ { 2u, 2u }, red, &flag, a.timeout_ns };
    const double thresh2 = sc->thresh2, tol2S = sc->tol2S;
    const int max_cg = sc->max_cg, max_outer = sc->max_outer;
    const bool want_p = sc->hist_p != nullptr;
    int n = sc->n, k = 0, status = ST_OK, cur = 0;
    long long cg_total = 0;
    double gamma = 0.0, delta = 0.0, beta = 0.0, alpha = 0.0, epsR2 = 0.0;
    bool dzero = sc->dzero != 0;

    // (L x)_C of one chunk from its seven chunks and its link bytes (apply_L_chunk of omni_kernels.cuh)
    auto applyL = [&](T (&q)[V], const T (&vm)[V], const T (&vc)[V], const T (&vp)[V], const T (&vn)[V], const T (&vs)[V], T xl,
                      T xr, uint32_t fb, const uint32_t (&code)[V], const RowTask<V>& tk) {
        const XEdge xe = make_xedge<V>(g, tk.x);
        apply_L_chunk<T, V>(q, vm, vc, vp, vn, vs, xl, xr, fb, code, a.K, xe, face_class(tk.j, g.ny, g.fix[1]),
                            face_class(tk.k, g.nz, g.fix[2]));
    };

    for (;;) {
        // ------------------------------------------------------------------ outer check: P += delta, r = S - L P
        T* rc = A.rb[cur];
        {
            const int par = n & 1;
            double acc[2] = { 0.0, 0.0 }, accp[2] = { 0.0, 0.0 }, tot[2], totp[2] = { 0.0, 0.0 };
            persist_k2_rows<T>(g, a, rc, a.Pbuf[par], a.Pbuf[par ^ 1], dzero, want_p, lo2, hi2, wfirst, wstep, nsx2, lane, acc, accp);
            if (!grid_allreduce<2, NT>(gs, a.slots, acc, tot)) { status = ST_BARRIER_TIMEOUT; break; }
            if (want_p && !grid_allreduce<2, NT>(gs, a.slots, accp, totp)) { status = ST_BARRIER_TIMEOUT; break; }
            epsR2 = tot[0];
            if (blockIdx.x == 0 && threadIdx.x == 0) record_history(sc, tot[0], k, totp[0], totp[1]);
            if (!isfinite(tot[0])) { status = ST_BREAKDOWN; break; }
            if (tot[0] <= tol2S || n >= max_outer) { status = (tot[0] <= tol2S) ? ST_OK : ST_NOT_CONVERGED; break; }
            n += 1;
            k = 0;
            gamma = tot[1];
            dzero = !((tot[1] > thresh2) && (tot[1] != 0.0) && (max_cg > 0));
            if (dzero) continue;
        }
        // ------------------------------------------------------------------ start: w = L r, delta = w . r
        {
            T* wc = A.wb[cur];
            double acc[1] = { 0.0 }, tot[1];
            RowTask<V> tk(g, lo1 + wfirst, nsx, wstep, lane);
            for (int t = lo1 + wfirst; t < hi1; t += wstep, tk.next(g, lane)) {
                auto ld = [&](long long i, bool ok, T (&v)[V]) {
                    zero_chunk<T, V>(v);
                    if (ok) ldcg_chunk<T, V>(rc + i, v);
                };
                uint32_t fb = 0, code[V];
#pragma unroll
                for (int c = 0; c < V; ++c) code[c] = 0u;
                if (tk.out) {
                    fb = flag_bits<V>(a.flags, tk.idx);
                    if (fb) load_cell_codes<true, V>(a.wcode, a.link, tk.idx, code);
                }
                T vm[V], vc[V], vp[V], vn[V], vs[V];
                ld(tk.idx, tk.inb, vc);
                ld(tk.idx + g.px, tk.inb && tk.j + 1 < g.ny, vn);
                ld(tk.idx - g.px, tk.inb && tk.j > 0, vs);
                ld(tk.idx + pp, tk.inb && three && tk.k + 1 < g.nz, vp);
                ld(tk.idx - pp, tk.inb && three && tk.k > 0, vm);
                T xl = __shfl_up_sync(0xffffffffu, vc[V - 1], 1);
                T xr = __shfl_down_sync(0xffffffffu, vc[0], 1);
                if (lane == 0) xl = (tk.x > 0) ? ldd(rc + tk.idx - 1) : T(0);
                if (lane == 31) xr = (tk.x + V < g.px) ? ldd(rc + tk.idx + V) : T(0);
                if (!tk.out) continue;
                T q[V];
                applyL(q, vm, vc, vp, vn, vs, xl, xr, fb, code, tk);
#pragma unroll
                for (int c = 0; c < V; ++c) acc[0] += (double)q[c] * (double)vc[c];
                st_chunk<T, V>(wc + tk.idx, q);
            }
            if (!grid_allreduce<1, NT>(gs, a.slots, acc, tot)) { status = ST_BARRIER_TIMEOUT; break; }
            delta = tot[0];
            if (!(delta > 0.0) || !isfinite(delta)) { status = ST_BREAKDOWN; break; }
            alpha = gamma / delta;
            beta = 0.0;
        }
        // ------------------------------------------------------------------ iterations: one phase, one barrier each
        bool stop_all = false;
        for (;;) {
            const T* ro = A.rb[cur]; const T* wo = A.wb[cur]; const T* so = A.sb[cur];
            T* rn_ = A.rb[cur ^ 1]; T* wn_ = A.wb[cur ^ 1]; T* sn_ = A.sb[cur ^ 1];
            const T al = (T)alpha, be = (T)beta;
            const bool first = (k == 0);
            double acc[2] = { 0.0, 0.0 }, tot[2];
            RowTask<V> tk(g, lo1 + wfirst, nsx, wstep, lane);
            for (int t = lo1 + wfirst; t < hi1; t += wstep, tk.next(g, lane)) {
                // r' = r - alpha (w + beta s) of a chunk (0 outside the box)
                auto rnew = [&](long long i, bool ok, T (&v)[V]) {
                    zero_chunk<T, V>(v);
                    if (ok) {
                        T r[V], w[V], s[V];
                        ldcg_chunk<T, V>(ro + i, r);
                        ldcg_chunk<T, V>(wo + i, w);
                        ldcg_chunk<T, V>(so + i, s);
#pragma unroll
                        for (int c = 0; c < V; ++c) v[c] = r[c] - al * (w[c] + be * s[c]);
                    }
                };
                auto rnew1 = [&](long long i) { return ldd(ro + i) - al * (ldd(wo + i) + be * ldd(so + i)); };
                uint32_t fb = 0, code[V];
#pragma unroll
                for (int c = 0; c < V; ++c) code[c] = 0u;
                T r0[V], w0[V], s0[V], p0[V], d0[V];
                zero_chunk<T, V>(r0); zero_chunk<T, V>(w0); zero_chunk<T, V>(s0); zero_chunk<T, V>(p0); zero_chunk<T, V>(d0);
                if (tk.out) {
                    fb = flag_bits<V>(a.flags, tk.idx);
                    if (fb) load_cell_codes<true, V>(a.wcode, a.link, tk.idx, code);
                    ldcg_chunk<T, V>(ro + tk.idx, r0);
                    ldcg_chunk<T, V>(wo + tk.idx, w0);
                    ldcg_chunk<T, V>(so + tk.idx, s0);
                    ldcg_chunk<T, V>(A.p + tk.idx, p0);
                    if (!first) ldcg_chunk<T, V>(a.delta + tk.idx, d0);
                }
                T vm[V], vc[V], vp[V], vn[V], vs[V], sc_[V];
#pragma unroll
                for (int c = 0; c < V; ++c) { sc_[c] = w0[c] + be * s0[c]; vc[c] = r0[c] - al * sc_[c]; }
                rnew(tk.idx + g.px, tk.inb && tk.j + 1 < g.ny, vn);
                rnew(tk.idx - g.px, tk.inb && tk.j > 0, vs);
                rnew(tk.idx + pp, tk.inb && three && tk.k + 1 < g.nz, vp);
                rnew(tk.idx - pp, tk.inb && three && tk.k > 0, vm);
                T xl = __shfl_up_sync(0xffffffffu, vc[V - 1], 1);
                T xr = __shfl_down_sync(0xffffffffu, vc[0], 1);
                if (lane == 0) xl = (tk.x > 0) ? rnew1(tk.idx - 1) : T(0);
                if (lane == 31) xr = (tk.x + V < g.px) ? rnew1(tk.idx + V) : T(0);
                if (!tk.out) continue;
                T q[V], pn[V], dn[V];
                applyL(q, vm, vc, vp, vn, vs, xl, xr, fb, code, tk);
#pragma unroll
                for (int c = 0; c < V; ++c) {
                    pn[c] = r0[c] + be * p0[c];
                    dn[c] = d0[c] + al * pn[c];
                    acc[0] += (double)vc[c] * (double)vc[c];
                    acc[1] += (double)q[c] * (double)vc[c];
                }
                st_chunk<T, V>(rn_ + tk.idx, vc);
                st_chunk<T, V>(sn_ + tk.idx, sc_);
                st_chunk<T, V>(wn_ + tk.idx, q);
                st_chunk<T, V>(A.p + tk.idx, pn);
                st_chunk<T, V>(a.delta + tk.idx, dn);
            }
            if (!grid_allreduce<2, NT>(gs, a.slots, acc, tot)) { status = ST_BARRIER_TIMEOUT; stop_all = true; break; }
            const double gamma1 = tot[0], delta1 = tot[1];
            if (!isfinite(gamma1) || !isfinite(delta1)) { status = ST_BREAKDOWN; stop_all = true; break; }
            cur ^= 1;
            k += 1;
            cg_total += 1;
            if (!((gamma1 > thresh2) && (gamma1 != 0.0) && (k < max_cg))) { gamma = gamma1; break; }
            beta = gamma1 / gamma;
            const double den = delta1 - beta * gamma1 / alpha;
            // delta - beta gamma / alpha stands for p.Ap > 0; when rounding (fp32, hundreds of iterations) has eaten it,
            // the recurred s = A p is no longer usable: end this inner solve -- the outer check re-evaluates the true
            // residual from the fp64 pressure and the recurrences restart from it (residual replacement)
            if (!isfinite(den)) { status = ST_BREAKDOWN; stop_all = true; break; }
            if (!(den > 0.0)) { gamma = gamma1; break; }
            alpha = gamma1 / den;
            gamma = gamma1;
        }
        if (stop_all) break;
    }

    if (blockIdx.x == 0 && threadIdx.x == 0) {
        sc->n = n; sc->k = k; sc->cg_total = cg_total; sc->status = status;
        sc->rho = gamma; sc->beta = beta; sc->alpha = alpha; sc->gamma = delta; sc->epsR2 = epsR2;
        sc->inner_go = 0; sc->outer_go = 0;
    }
}

}  // namespace omni
