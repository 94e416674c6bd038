// omni_resident.cuh -- the persistent loop of omni_persist.cuh with the CG vectors kept ON THE SM between iterations,
// for grids small enough that the direction vector p fits the shared memory of the whole GPU (148 x 227 KB): up to
// 1024 x 1024 (2D) and 128^3 (3D) in both precisions.
//
// omni_persist.cuh streams every vector through L2 in every phase and crosses two fenced grid barriers per CG
// iteration; at these sizes an iteration is bound by those round trips (a fenced barrier of 148 CTAs costs 3.9 us),
// not by bandwidth.  Here each CTA owns a BOX of grid rows, [j0, j1) x [k0, k1) with the whole x extent, for the
// entire inner solve; a thread owns one 16-byte x chunk of consecutive rows of the box:
//   * p of the box and of the one-row / one-plane halo around it lives in shared memory (the stencil M p, Eq. 12 :119,
//     reads neighbours from there);
//   * r and delta (the CG solution, Alg. 1 :146) are touched cell by cell by their thread only.  They live in the SM's
//     TENSOR MEMORY, used as a thread-private scratchpad through tcgen05.ld / st (RM 3, at most RES_NI rows per thread), which
//     leaves the shared memory to p and to q = Op p.  Otherwise (more rows per thread): r in shared memory beside p (RM 0), behind L2 where p alone fills
//     the shared memory (RM 2), or in registers (RM 1, on request); delta in shared memory when it fits, else in global
//     memory and touched every second iteration (lazy, as in the tile kernel K4: delta += alpha_{k-1} p_{k-1} + alpha_k p_k
//     with p_{k-1} = (p_k - r_k) / beta_k recovered from what is on chip);
//   * per CG iteration the only global traffic is the halo of r: K4 sends r of the box's boundary rows to the
//     neighbours, which form p_new = r + beta p_old on their halo themselves (p_old of the halo is in their shared
//     memory), so no p ever travels.  The rows travel as self-validating 8-byte messages { 32 payload bits, 32-bit
//     epoch = number of the CG iteration that wrote them } (the scheme of NCCL's low-latency protocol): a reader polls
//     until the epoch is the one it expects, so the exchange needs no fence, and the two grid barriers of an iteration
//     -- which remain, as the deterministic all-reduce of gamma and rho' -- carry nothing but their own slot and are
//     relaxed (grid_allreduce_relaxed below: 1.6 us).  The fenced barriers remain around K2, once per outer iteration.
// Phase order, arithmetic per cell (apply_op_chunk of omni_kernels.cuh), stopping rules and the K2 phase (outer update
// through L2, persist_k2_rows) are those of persist_kernel; the reductions differ from it only in the order in which
// cells are added (fp32: a chunk's four products are added in fp32 first, as in the tile kernels, A9).
//
// Race notes.  Messages of a boundary row: written in K4 of iteration c (epoch c + 1), polled by the neighbour in K3 (i)
// of iteration c + 1 (which it enters only after the rho' barrier of iteration c), overwritten in K4 of iteration c + 1,
// i.e. after the gamma barrier of iteration c + 1, which the neighbour joins only after its polls have returned.
// Shared p: written in K3 (i), __syncthreads, read in K3 (ii) and K4; the next write is behind the rho' barrier's
// __syncthreads.  The first K3 (i) of an inner solve reads its halo of r from the global r array K2 wrote (fenced barrier).
#pragma once
#include "omni_persist.cuh"

namespace omni {

#ifdef OMNI_RES_TRACE
__device__ unsigned long long g_res_trace[16];
#define RES_T(i) do { if (blockIdx.x == (unsigned)g_res_trace[15] && threadIdx.x == 0) { const unsigned long long t_ = global_timer_ns(); g_res_trace[i] += t_ - tr_last; tr_last = t_; } } while (0)
#else
#define RES_T(i) do { } while (0)
#endif

constexpr int RES_NT = 512;        // threads per CTA: up to 128 registers each
constexpr int RES_NI = 16;         // rows per thread whose r and delta fit the thread's share of tensor memory (and, RM 1, 64 registers)
constexpr int RES_SMEM_MAX = (227 - 5) * 1024;    // dynamic shared memory the plan may use (static: 4.4 KB of barrier scratch)

// Start of part i when an axis of n cells is cut into `parts` boxes.  wface = 0: equal counts.  wface > 0 (operator M on an
// axis with face classes): a cell costs 4, a cell of a face class (0, 1, n-2, n-1; they run the face correction of
// DESIGN.md section 6 on top of the interior formula) 4 + wface, and the cuts equalise the cost, so that the boxes on the
// faces of the grid -- for which every barrier would otherwise wait -- get fewer rows.  Only where every part keeps at
// least four cells.
__host__ __device__ inline int res_split(int n, int parts, int i, int wface)
{
    if (i <= 0) return 0;
    if (i >= parts) return n;
    if (wface <= 0 || n < 8 * parts) return (int)((long long)n * i / parts);
    const long long total = 4LL * n + 4LL * wface;
    const long long target = (total * i + parts - 1) / parts;          // smallest x with cost(x) >= target
    auto cost = [&](long long x) { return 4 * x + (long long)wface * ((x < 2 ? x : 2) + (x > n - 2 ? x - (n - 2) : 0)); };
    int lo = 0, hi = n;                                                 // cost(lo) < target <= cost(hi)
    while (hi - lo > 1) {
        const int mid = (lo + hi) / 2;
        if (cost(mid) >= target) hi = mid; else lo = mid;
    }
    return hi;
}

template <typename T>
struct ResidentArgs {
    PersistArgs<T> a;
    unsigned long long* xchg;   // halo messages: sizeof(T) / 4 words per cell, indexed like the padded grid; zero at launch
    int gy, gz;        // CTA b owns rows j in [res_split(ny, gy, by), res_split(ny, gy, by + 1)) of the planes k cut likewise by bz; by = b % gy, bz = b / gy
    int ly, lz;        // largest box (rows, planes): the extents of the shared p array
    int zpad;          // 1: 3D operator, the p array has a halo plane below and above
    int pxs;           // row pitch of the p array in cells: px + 2 chunks (a zero chunk left and right of every row)
    int dres;          // 1: delta lives in shared memory
    int qres;          // 1: q = Op p of K3 is kept in shared memory for K4 (no second stencil pass)
    int rpt;           // rows per thread the shared r / delta arrays are laid out for
    int wy, wz;        // res_split weights of the y and z cuts
};

// one chunk (16 bytes of T) as four messages { payload, epoch }
template <typename T, int V>
__device__ __forceinline__ void msg_send(unsigned long long* m, const T (&v)[V], uint32_t epoch)
{
    uint32_t w[4];
    memcpy(w, v, 16);
    const unsigned long long e = (unsigned long long)epoch << 32;
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" :: "l"(m), "l"(e | w[0]), "l"(e | w[1]) : "memory");
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" :: "l"(m + 2), "l"(e | w[2]), "l"(e | w[3]) : "memory");
}
// the loads (in flight until msg_decode looks at them) ...
__device__ __forceinline__ void msg_load(const unsigned long long* m, unsigned long long (&b)[4])
{
    // strong L2 loads (weak ones may be hoisted out of a polling loop or served from L1); every 8-byte word validates itself
    // through its epoch
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(b[0]), "=l"(b[1]) : "l"(m) : "memory");
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(b[2]), "=l"(b[3]) : "l"(m + 2) : "memory");
}
// ... and their check: true iff all four words carry the expected epoch
template <typename T, int V>
__device__ __forceinline__ bool msg_decode(const unsigned long long (&b)[4], T (&v)[V], uint32_t epoch)
{
    uint32_t w[4];
    bool ok = true;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        w[i] = (uint32_t)b[i];
        ok = ok && (uint32_t)(b[i] >> 32) == epoch;
    }
    memcpy(v, w, 16);
    return ok;
}
template <typename T, int V>
__device__ __forceinline__ bool msg_try(const unsigned long long* m, T (&v)[V], uint32_t epoch)
{
    unsigned long long b[4];
    msg_load(m, b);
    return msg_decode<T, V>(b, v, epoch);
}

// Relaxed grid barrier + all-reduce of one fp64 accumulator, for barriers that carry nothing but their own slot: no
// fence on either side.  Its own slots (one 128-byte line per CTA and set, behind the fenced barrier's regions) and its
// own use count; tags as in grid_allreduce.  Thread b of every CTA polls slot b, so the G polls of a CTA are in flight
// at once, and every warp then adds the G values from shared memory in slot order.  Measured on B200 with 148 CTAs
// (strong loads are served one by one per SM, and per L2 line): 4.9 us per barrier when warp 0 polls packed slots,
// 3.0 us when every thread polls one packed slot, 1.6 us with a line per slot; the fenced barrier costs 3.9 us.
constexpr int RES_SLOT_STRIDE = 16;                  // doubles: one slot per 128-byte line
constexpr size_t RES_SLOT_OFFSET = 2048;             // doubles: behind the 8 * G <= 1184 doubles of the fenced regions
static_assert((RES_SLOT_OFFSET + 2 * 148 * RES_SLOT_STRIDE) * 8 <= PERSIST_SLOT_BYTES, "relaxed slots fit the slot buffer");

template <int NT>
__device__ __forceinline__ bool grid_allreduce_relaxed(GridSync& gs, unsigned int& count, double* slots, double* sv, int* late,
                                                       double acc, double& tot)
{
    constexpr int NW = NT / 32;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned int G = gridDim.x, tag = (count >> 1) & 1u;
    double* my = slots + RES_SLOT_OFFSET + (size_t)(count & 1u) * G * RES_SLOT_STRIDE;
    double s = warp_sum(acc);
    if (lane == 0) gs.red[warp] = s;
    __syncthreads();
    if (warp == 0) {
        s = warp_sum(lane < NW ? gs.red[lane] : 0.0);
        if (lane == 0) slot_publish<true>(my + (size_t)blockIdx.x * RES_SLOT_STRIDE, s, tag);
    }
    if (threadIdx.x < G) {
        double v;
        unsigned int spins = 0;
        unsigned long long t0 = 0;
        while (!slot_poll<true>(my + (size_t)threadIdx.x * RES_SLOT_STRIDE, tag, v)) {
            if ((++spins & 255u) == 0u) {
                const unsigned long long t = global_timer_ns();
                if (t0 == 0) t0 = t;
                if (t - t0 > gs.timeout_ns) { *late = 1; break; }      // shared; zero until a wait times out
            }
        }
        sv[threadIdx.x] = v;
    }
    __syncthreads();
    double t = 0.0;
    for (unsigned int b = lane; b < G; b += 32) t += sv[b];           // fixed order, the same in every warp and CTA
    tot = warp_sum(t);
    count += 1u;
    return *late == 0;
}

// ---- Tensor memory as a per-thread scratchpad.  The 256 KB of TMEM of an SM (512 columns x 128 lanes x 32 bit) are the
// accumulator store of tcgen05.mma; nothing here multiplies matrices, but tcgen05.ld / tcgen05.st move registers to and
// from it with the 32x32b shape in which lane i of a warp owns TMEM lane 32 (warp % 4) + i: thread-private storage with
// a 12-cycle load, exactly what r and delta need (CG touches them cell by cell).  The four warps that share a lane
// quarter take 128 columns each: 32 chunks of 16 bytes per thread, RES_NI for r and RES_NI for delta.
__device__ __forceinline__ void tmem_alloc512(uint32_t* smem_slot)        // one whole warp
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                 :: "r"((uint32_t)__cvta_generic_to_shared(smem_slot)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc512(uint32_t base)            // one whole warp
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(base), "r"(512u) : "memory");
}
// whole warp; the registers are valid after tmem_wait_ld (one wait covers every load issued before it)
__device__ __forceinline__ void tmem_ld_raw(uint32_t taddr, uint32_t (&w)[4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
template <typename T, int V>
__device__ __forceinline__ void tmem_ld_chunk(uint32_t taddr, T (&v)[V])
{
    uint32_t w[4];
    tmem_ld_raw(taddr, w);
    tmem_wait_ld();
    memcpy(v, w, 16);
}
template <typename T, int V>
__device__ __forceinline__ void tmem_st_chunk(uint32_t taddr, const T (&v)[V])   // whole warp
{
    uint32_t w[4];
    memcpy(w, v, 16);
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};"
                 :: "r"(taddr), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// loop over the rows of a thread: unrolled when r lives in registers (static register indices), rolled otherwise
template <bool UNROLL, typename F>
__device__ __forceinline__ void res_for_rows(int nrt, F&& f)
{
    if constexpr (UNROLL) {
#pragma unroll
        for (int it = 0; it < RES_NI; ++it) {
            if (it >= nrt) break;
            f(it);
        }
    } else {
#pragma unroll 1
        for (int it = 0; it < nrt; ++it) f(it);
    }
}

// where r of the box lives -- RM 0: shared memory, beside p; 1: registers (p alone fills the shared memory: 128^3 fp64);
// 2: the global r array (through L2; same grids as 1).  With RM 2 a thread's loads of r are one L2 round trip per row;
// issuing them four rows ahead (16 + 16 more registers for r and the lazy delta) was tried and is slower (128^3 fp64:
// 29.8 -> 36.3 us per iteration): with 190 KB of shared memory the L1 is 28 KB and the 230 B per thread it spills miss it.
//   3: r AND delta in tensor memory (tmem_* above): shared memory holds p and, where it fits, q.
// UNI (RM 3 only; true otherwise): the host has checked that in every box all lanes of a warp own the same number of rows
// (resident_uniform), so the warp-wide tcgen05 instructions need no per-lane mask.  Without it the row loops that touch
// tensor memory run to the warp's longest lane under a `live` predicate.
template <typename T, bool LOP, int RM, bool UNI = true>
__global__ void __launch_bounds__(RES_NT, 1)
resident_kernel(const Geom g, const ResidentArgs<T> ra)
{
    static_assert(RM == 3 || UNI, "only the tensor-memory variant has a masked form");
    constexpr int V = 16 / (int)sizeof(T), NT = RES_NT, NW = NT / 32, MW = (int)sizeof(T) / 4;
    constexpr bool RREG = RM == 1, RTM = RM == 3;
    __shared__ uint32_t tmem_base_slot;
    extern __shared__ __align__(16) unsigned char res_smem[];
    __shared__ double red[2 * (NW + 1)];
    __shared__ double sv[PERSIST_MAX_CTAS > NT ? NT : PERSIST_MAX_CTAS];
    __shared__ int flag;
    __shared__ int halo_late;
    const PersistArgs<T>& a = ra.a;
    Scalars* sc = a.sc;
    if (!sc->outer_go) return;                             // zero source: nothing to iterate (A4)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const bool three = g.naxes == 3;
    // ---- the K2 phase's share: row segments in linear order, as in persist_kernel
    const int nsx2 = (g.nx + 63) / 64;
    const long long ntask2 = (long long)g.ny * g.nz * nsx2;
    const int lo2 = (int)(ntask2 * blockIdx.x / gridDim.x), hi2 = (int)(ntask2 * (blockIdx.x + 1) / gridDim.x);
    // ---- the CG phases' share: this CTA's box
    const int by = (int)blockIdx.x % ra.gy, bz = (int)blockIdx.x / ra.gy;
    const int j0 = res_split(g.ny, ra.gy, by, ra.wy), j1 = res_split(g.ny, ra.gy, by + 1, ra.wy);
    const int k0 = res_split(g.nz, ra.gz, bz, ra.wz), k1 = res_split(g.nz, ra.gz, bz + 1, ra.wz);
    const int lyb = j1 - j0, lzb = k1 - k0, nrows = lyb * lzb;
    const int cpr = g.px / V;                              // chunks per row
    const int rs = ra.pxs, pls = (ra.ly + 2) * ra.pxs, zpad = ra.zpad;
    T* const ps = reinterpret_cast<T*>(res_smem);
    const int p_elems = (ra.lz + 2 * zpad) * pls;
    // r (unless RREG) and delta (dres only) of this thread's row `it` at [(it * NT + tid) * V]
    T* const rsm = ps + p_elems;
    T* const ds = rsm + (RM != 0 ? 0 : ra.rpt * NT * V);
    T* const qs = RTM ? rsm : ds + ra.rpt * NT * V;        // qres only (RM 0: implies dres)
    // a thread owns x chunk xc of the rows [r_lo, r_lo + nrt) of the box (rows numbered y-fastest): NT / cpr row groups
    const int nrg = NT / cpr, grp = tid / cpr, xc = tid - grp * cpr, x = xc * V;
    const int rpg = (nrows + nrg - 1) / nrg;
    const int r_lo = min(grp * rpg, nrows);
    const int nrt = (grp < nrg && x < g.nx) ? min(rpg, nrows - r_lo) : 0;      // a chunk of pad cells only is never touched
    const int jl0 = r_lo % lyb, kl0 = r_lo / lyb;
    const int off0 = (kl0 + zpad) * pls + (jl0 + 1) * rs + V + x, wrap = pls - lyb * rs;
    const XEdge xe = make_xedge<V>(g, x);
    auto cell_idx = [&](int jl, int kl) { return (long long)x + (long long)g.px * ((j0 + jl) + (long long)g.ny * (k0 + kl)); };
    // halo rows of the box that exist in the grid: y-, y+ (one per plane), z-, z+ (one per row)
    const int nA = (j0 > 0) ? lzb : 0, nB = (j1 < g.ny) ? lzb : 0;
    const int nC = (three && k0 > 0) ? lyb : 0, nD = (three && k1 < g.nz) ? lyb : 0;
    const int nhc = (nA + nB + nC + nD) * cpr;

    // tcgen05.ld / st are warp-wide: with r in tensor memory every lane of a warp walks the same number of rows (the
    // largest of the warp); `live` tells a lane whether row `it` is one of its own
    int nloop = nrt;
    if constexpr (!UNI) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nloop = max(nloop, __shfl_xor_sync(0xffffffffu, nloop, o));
    }
    // tensor-memory address of chunk `slot` (0 .. 31) of this thread: lane quarter of the warp, 128 columns per warp
    uint32_t tm_base = 0;
    auto tm_addr = [&](int slot) { return tm_base + (uint32_t)(slot * 4); };
#define RES_ROWS_BEGIN                                                                                   \
    {                                                                                                    \
        int jl = jl0, kl = kl0, off = off0;                                                              \
        res_for_rows<RREG>(nloop, [&](const int it) {                                                    \
            const bool live = UNI || it < nrt;
#define RES_ROWS_END                                                                                     \
            jl += 1; off += rs;                                                                          \
            if (jl == lyb) { jl = 0; kl += 1; off += wrap; }                                             \
        });                                                                                              \
    }
    // the same walk for loops without warp-wide instructions: every lane stops after its own rows, no mask
#define RES_ROWS_BEGIN_LANE                                                                              \
    {                                                                                                    \
        int jl = jl0, kl = kl0, off = off0;                                                              \
        res_for_rows<RREG>(nrt, [&](const int it) {                                                      \
            constexpr bool live = true;

    // per row of this thread, one bit each (the codes and the box never change during a solve):
    //   slow: the chunk is flagged (mask / NaN changed a code) or the row lies in a face class of the grid -- everything
    //         else is the interior formula (plus the x-edge correction in the two or three threads that hold such cells)
    //   bnd:  the row is on the box boundary: its r travels to a neighbour
    uint32_t fbm = 0, slowm = 0, bndm = 0;
    RES_ROWS_BEGIN_LANE
        if (live) {
            if (flag_bits<V>(a.flags, cell_idx(jl, kl))) fbm |= 1u << it;
            if (face_class(j0 + jl, g.ny, g.fix[1]) >= 0 || face_class(k0 + kl, g.nz, g.fix[2]) >= 0) slowm |= 1u << it;
            if ((jl == 0 && j0 > 0) || (jl == lyb - 1 && j1 < g.ny) || (three && ((kl == 0 && k0 > 0) || (kl == lzb - 1 && k1 < g.nz))))
                bndm |= 1u << it;
        }
        (void)off;
    RES_ROWS_END
    slowm |= fbm;

    if constexpr (RTM) {
        // all 512 columns of this SM's tensor memory (one CTA per SM); released at the kernel's single exit below
        if (warp == 0) tmem_alloc512(&tmem_base_slot);
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        tm_base = tmem_base_slot + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(128 * (warp >> 2));
    }

    GridSync gs{ { 2u, 2u }, red, &flag, a.timeout_ns };
    unsigned int rcount = 2u;                              // use count of the relaxed barrier (set = count & 1, tag = (count >> 1) & 1)
    if (tid == 0) halo_late = 0;

    // loop state, identical in every thread of the grid
    const double thresh2 = sc->thresh2, tol2S = sc->tol2S;
    const int max_cg = sc->max_cg, max_outer = sc->max_outer;
    int n = sc->n, k = 0, status = ST_OK;
    long long cg_total = 0;
    double rho = 0.0, beta = 0.0, alpha = 0.0, gamma = 0.0, epsR2 = 0.0, alpha_prev = 0.0;
    bool dzero = sc->dzero != 0;
    T rr[RREG ? RES_NI : 1][V];
    // r of row `it` (slots 0 .. RES_NI-1 of the thread's tensor memory with RM 3) and, RM 3 only, delta (slots RES_NI ..)
    auto r_ld = [&](int it, int jl, int kl, bool live, T (&v)[V]) {
        if constexpr (RM == 3) {
            __syncwarp();
            tmem_ld_chunk<T, V>(tm_addr(it), v);
        } else if (live) {
            if constexpr (RM == 1) {
#pragma unroll
                for (int c = 0; c < V; ++c) v[c] = rr[it][c];
            } else if constexpr (RM == 0) {
                ld_chunk<T, V>(rsm + (size_t)(it * NT + tid) * V, v);
            } else {
                ld_chunk<T, V>(a.r + cell_idx(jl, kl), v);         // this thread's own store (or K2's, behind a fenced barrier)
            }
        }
    };
    auto r_st = [&](int it, int jl, int kl, bool live, const T (&v)[V]) {
        if constexpr (RM == 3) {
            __syncwarp();
            tmem_st_chunk<T, V>(tm_addr(it), v);
        } else if (live) {
            if constexpr (RM == 1) {
#pragma unroll
                for (int c = 0; c < V; ++c) rr[it][c] = v[c];
            } else if constexpr (RM == 0) {
                st_chunk<T, V>(rsm + (size_t)(it * NT + tid) * V, v);
            } else {
                st_chunk<T, V>(a.r + cell_idx(jl, kl), v);
            }
        }
    };
#ifdef OMNI_RES_TRACE
    unsigned long long tr_last = global_timer_ns();
#endif

    // q = Op p for the chunk at shared offset off; vs / vc / vn (the rows below, at and above it) are carried from one
    // row of the thread to the next while the rows stay in one plane (carry)
    T vs[V], vc[V], vn[V];
    bool carry = false;
    auto stencil = [&](int off, int it, int jl, int kl, T (&q)[V]) {
        const T* c = ps + off;
        if (!carry) { ld_chunk<T, V>(c - rs, vs); ld_chunk<T, V>(c, vc); }
        ld_chunk<T, V>(c + rs, vn);
        T vm[V], vp[V];
        if (three) { ld_chunk<T, V>(c + pls, vp); ld_chunk<T, V>(c - pls, vm); }
        else { zero_chunk<T, V>(vp); zero_chunk<T, V>(vm); }
        const T xl = c[-1], xr = c[V];
        uint32_t code[V];
#pragma unroll
        for (int i = 0; i < V; ++i) code[i] = 0u;
        if (!((slowm >> it) & 1u)) {
            apply_op_chunk<LOP, T, V>(q, vm, vc, vp, vn, vs, xl, xr, 0u, code, a.K, xe, -1, -1);     // interior formula (+ x-edge cells)
        } else {
            const uint32_t fb = (fbm >> it) & 1u;
            if (fb) load_cell_codes<LOP, V>(a.wcode, a.link, cell_idx(jl, kl), code);
            apply_op_chunk<LOP, T, V>(q, vm, vc, vp, vn, vs, xl, xr, fb, code, a.K, xe,
                                      face_class(j0 + jl, g.ny, g.fix[1]), face_class(k0 + kl, g.nz, g.fix[2]));
        }
    };
    // after the row's work: the next row of the thread is the one above (carry) unless the plane ends
#define RES_CARRY_NEXT                                                                                   \
        carry = (jl + 1 != lyb);                                                                         \
        if (carry) {                                                                                     \
            _Pragma("unroll") for (int c_ = 0; c_ < V; ++c_) { vs[c_] = vc[c_]; vc[c_] = vn[c_]; }       \
        }
    auto dot_chunk = [&](const T (&u)[V], const T (&w)[V]) -> double {
        if constexpr (sizeof(T) == 4) {
            T s = T(0);
#pragma unroll
            for (int c = 0; c < V; ++c) s += u[c] * w[c];
            return (double)s;
        } else {
            double s = 0.0;
#pragma unroll
            for (int c = 0; c < V; ++c) s += (double)u[c] * (double)w[c];
            return s;
        }
    };

    for (;;) {
        // ------------------------------------------------------------------------------ K2: P += delta, r = S - L P
        {
            const int par = n & 1;
            const double* Pin = a.Pbuf[par];
            double* Pout = a.Pbuf[par ^ 1];
            double acc[2] = { 0.0, 0.0 }, accp[2] = { 0.0, 0.0 };
            const bool want_p = sc->hist_p != nullptr;
            persist_k2_rows<T>(g, a, a.r, Pin, Pout, dzero, want_p, lo2, hi2, warp, NW, nsx2, lane, acc, accp);
            double tot[2], totp[2] = { 0.0, 0.0 };
            if (!grid_allreduce<2, NT>(gs, a.slots, acc, tot)) { status = ST_BARRIER_TIMEOUT; break; }
            if (want_p && !grid_allreduce<2, NT>(gs, a.slots, accp, totp)) { status = ST_BARRIER_TIMEOUT; break; }
            epsR2 = tot[0];
            if (blockIdx.x == 0 && tid == 0) record_history(sc, tot[0], k, totp[0], totp[1]);
            if (!isfinite(tot[0])) { status = ST_BREAKDOWN; break; }
            if (tot[0] <= tol2S || n >= max_outer) { status = (tot[0] <= tol2S) ? ST_OK : ST_NOT_CONVERGED; break; }
            n += 1;
            k = 0;
            beta = 0.0;
            rho = tot[1];
            dzero = !((tot[1] > thresh2) && (tot[1] != 0.0) && (max_cg > 0));
            if (dzero) continue;
        }
        // ------------------------------------------------------------------------------ r into registers, p = 0
        for (int i = tid * V; i < p_elems; i += NT * V) {
            T z[V];
            zero_chunk<T, V>(z);
            st_chunk<T, V>(ps + i, z);
        }
        RES_ROWS_BEGIN
            if constexpr (RM != 2) {
                T v[V];
                zero_chunk<T, V>(v);
                if (live) ldcg_chunk<T, V>(a.r + cell_idx(jl, kl), v);
                r_st(it, jl, kl, live, v);
            }
            (void)off;
        RES_ROWS_END
        if constexpr (RTM) tmem_wait_st();
        __syncthreads();
        RES_T(0);
        // ------------------------------------------------------------------------------ inner CG on Op delta = r0
        bool stop_all = false;
        for (;;) {
            // ---- K3 (i): p = r + beta p on the box (r in registers) and on its halo (r from the neighbours' K4 / from K2)
            {
                const T b = (T)beta;
                const uint32_t epoch = (uint32_t)cg_total;          // what the neighbours' last K4 stamped
                // the halo, four chunks per thread in flight (updating the box's rows under these loads was tried: the
                // registers it takes spill elsewhere and cost more than the latency it hides)
                for (int h0 = tid; h0 < nhc; h0 += 4 * NT) {
                    T hr[4][V];
                    int hoff[4];
                    long long hidx[4];
                    bool got[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int h = h0 + u * NT;
                        hoff[u] = -1;
                        hidx[u] = 0;
                        got[u] = true;
                        if (h < nhc) {
                            int row = h / cpr;
                            const int hx = h - row * cpr;
                            int jl, kl;
                            if (row < nA) { jl = -1; kl = row; }
                            else if ((row -= nA) < nB) { jl = lyb; kl = row; }
                            else if ((row -= nB) < nC) { jl = row; kl = -1; }
                            else { jl = row - nC; kl = lzb; }
                            if (hx * V >= g.nx) continue;              // a chunk of pad cells only: p stays 0, nobody sends it
                            hoff[u] = (kl + zpad) * pls + (jl + 1) * rs + V + hx * V;
                            hidx[u] = (long long)hx * V + (long long)g.px * ((j0 + jl) + (long long)g.ny * (k0 + kl));
                            if (k == 0) ldcg_chunk<T, V>(a.r + hidx[u], hr[u]);
                            else got[u] = msg_try<T, V>(ra.xchg + hidx[u] * MW, hr[u], epoch);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        if (hoff[u] >= 0) {
                            if (!got[u]) {
                                const unsigned long long t0 = global_timer_ns();
                                while (!msg_try<T, V>(ra.xchg + hidx[u] * MW, hr[u], epoch)) {
                                    if (global_timer_ns() - t0 > a.timeout_ns) {
                                        halo_late = 1;
#ifdef OMNI_RES_TRACE
                                        g_res_trace[10] = 1000000ULL * (blockIdx.x + 1) + tid; g_res_trace[11] = (unsigned long long)hidx[u]; g_res_trace[12] = epoch;
#endif
                                        break;
                                    }
                                }
                            }
                            T p[V];
                            ld_chunk<T, V>(ps + hoff[u], p);
#pragma unroll
                            for (int c = 0; c < V; ++c) p[c] = hr[u][c] + b * p[c];
                            st_chunk<T, V>(ps + hoff[u], p);
                        }
                    }
                }
                RES_ROWS_BEGIN
                    T p[V], r[V];
                    r_ld(it, jl, kl, live, r);
                    if (live) {
                        ld_chunk<T, V>(ps + off, p);
#pragma unroll
                        for (int c = 0; c < V; ++c) p[c] = r[c] + b * p[c];
                        st_chunk<T, V>(ps + off, p);
                    }
                RES_ROWS_END
            }
            __syncthreads();
            if (halo_late) { status = ST_BARRIER_TIMEOUT; stop_all = true; break; }
            RES_T(1);
            // ---- K3 (ii): gamma = p . Op p
            {
                double acc[1] = { 0.0 };
                carry = false;
                RES_ROWS_BEGIN_LANE
                    if (live) {
                        T q[V];
                        stencil(off, it, jl, kl, q);
                        acc[0] += dot_chunk(vc, q);
                        if (ra.qres) st_chunk<T, V>(qs + (size_t)(it * NT + tid) * V, q);
                        RES_CARRY_NEXT
                    }
                RES_ROWS_END
                double tot[1];
                RES_T(2);
                if (!grid_allreduce_relaxed<NT>(gs, rcount, a.slots, sv, &halo_late, acc[0], tot[0])) { status = ST_BARRIER_TIMEOUT; stop_all = true; break; }
                RES_T(3);
                gamma = tot[0];
                if (!(gamma > 0.0) || !isfinite(gamma)) { status = ST_BREAKDOWN; stop_all = true; break; }
                alpha = rho / gamma;
            }
            // ---- K4: q = Op p again; r -= alpha q; delta += alpha p; rho' = r . r; boundary rows of r to the neighbours
            {
                const T al = (T)alpha;
                const bool odd = (k & 1) != 0;
                // lazy delta (global): at odd k, delta += alpha_{k-1} p_{k-1} + alpha_k p_k = c1 p_k - c2 r_k
                const T c2 = odd ? (T)(alpha_prev / beta) : T(0), c1 = (T)((odd ? alpha_prev / beta : 0.0) + alpha);
                const uint32_t epoch = (uint32_t)(cg_total + 1);
                double acc[1] = { 0.0 };
                carry = false;
                RES_ROWS_BEGIN
                    T q[V], r[V];
                    zero_chunk<T, V>(q);
                    if (live) {
                        if (ra.qres) {
                            ld_chunk<T, V>(qs + (size_t)(it * NT + tid) * V, q);
                            ld_chunk<T, V>(ps + off, vc);
                        } else {
                            stencil(off, it, jl, kl, q);
                        }
                    }
                    if constexpr (RTM) {
                        // r and delta of the row: two loads, one wait
                        uint32_t wr[4], wd[4] = { 0u, 0u, 0u, 0u };
                        __syncwarp();
                        tmem_ld_raw(tm_addr(it), wr);
                        if (k != 0) tmem_ld_raw(tm_addr(RES_NI + it), wd);
                        tmem_wait_ld();
                        T d[V];
                        memcpy(r, wr, 16);
                        memcpy(d, wd, 16);
                        if (live) {
#pragma unroll
                            for (int c = 0; c < V; ++c) d[c] += al * vc[c];
                        }
                        tmem_st_chunk<T, V>(tm_addr(RES_NI + it), d);
                    } else {
                        r_ld(it, jl, kl, live, r);
                    }
                    if (live) {
                        if constexpr (RTM) {
                        } else if (ra.dres) {
                            T d[V];
                            T* dp = ds + (size_t)(it * NT + tid) * V;
                            if (k == 0) zero_chunk<T, V>(d);
                            else ld_chunk<T, V>(dp, d);
#pragma unroll
                            for (int c = 0; c < V; ++c) d[c] += al * vc[c];
                            st_chunk<T, V>(dp, d);
                        } else if (odd) {
                            T d[V];
                            T* dp = a.delta + cell_idx(jl, kl);
                            if (k == 1) zero_chunk<T, V>(d);
                            else ld_chunk<T, V>(dp, d);             // this thread's own store of two iterations ago
#pragma unroll
                            for (int c = 0; c < V; ++c) d[c] += c1 * vc[c] - c2 * r[c];
                            st_chunk<T, V>(dp, d);
                        }
#pragma unroll
                        for (int c = 0; c < V; ++c) r[c] -= al * q[c];
                        acc[0] += dot_chunk(r, r);
                        if ((bndm >> it) & 1u) msg_send<T, V>(ra.xchg + cell_idx(jl, kl) * MW, r, epoch);
                        if (!ra.qres) { RES_CARRY_NEXT }
                    }
                    r_st(it, jl, kl, live, r);
                RES_ROWS_END
                if constexpr (RTM) tmem_wait_st();
                double tot[1];
                RES_T(4);
                if (!grid_allreduce_relaxed<NT>(gs, rcount, a.slots, sv, &halo_late, acc[0], tot[0])) { status = ST_BARRIER_TIMEOUT; stop_all = true; break; }
                RES_T(5);
                const double rho1 = tot[0];
                if (!isfinite(rho1)) { status = ST_BREAKDOWN; stop_all = true; break; }
                beta = rho1 / rho;
                rho = rho1;
                alpha_prev = alpha;
                k += 1;
                cg_total += 1;
                if (!((rho1 > thresh2) && (rho1 != 0.0) && (k < max_cg))) break;
            }
        }
        if (stop_all) break;
        // ------------------------------------------------------------------------------ delta to global for K2
        {
            const bool pend = (k & 1) != 0;        // k iterations done; the last one (index k - 1) was even: its update is pending
            const T al = (T)alpha;
            if (RTM || ra.dres || pend) {
                RES_ROWS_BEGIN
                    T d[V];
                    if constexpr (RTM) { __syncwarp(); tmem_ld_chunk<T, V>(tm_addr(RES_NI + it), d); }
                    if (live) {
                        T* dp = a.delta + cell_idx(jl, kl);
                        if constexpr (RTM) {
                        } else if (ra.dres) {
                            ld_chunk<T, V>(ds + (size_t)(it * NT + tid) * V, d);
                        } else {
                            T p[V];
                            ld_chunk<T, V>(ps + off, p);
                            if (k == 1) zero_chunk<T, V>(d);
                            else ld_chunk<T, V>(dp, d);
#pragma unroll
                            for (int c = 0; c < V; ++c) d[c] += al * p[c];
                        }
                        st_chunk<T, V>(dp, d);
                    }
                RES_ROWS_END
            }
            // K2 reads delta of other CTAs' cells: a fenced barrier
            double z[1] = { 0.0 }, zt[1];
            if (!grid_allreduce<1, NT>(gs, a.slots, z, zt)) { status = ST_BARRIER_TIMEOUT; break; }
        }
    }
#undef RES_ROWS_BEGIN
#undef RES_ROWS_BEGIN_LANE
#undef RES_ROWS_END
#undef RES_CARRY_NEXT

    if constexpr (RTM) {
        tmem_wait_st();
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (warp == 0) tmem_dealloc512(tmem_base_slot);
    }
    if (blockIdx.x == 0 && tid == 0) {
        sc->n = n; sc->k = k; sc->cg_total = cg_total; sc->status = status;
        sc->rho = rho; sc->beta = beta; sc->alpha = alpha; sc->gamma = gamma; sc->epsR2 = epsR2;
        sc->inner_go = 0; sc->outer_go = 0;
    }
}

// ---- host side: does every warp of every box own the same number of rows in all its lanes?  (the thread -> rows map of the kernel)
inline bool resident_uniform(const Geom& g, int elem_size, int gy, int gz, int wy, int wz)
{
    const int V = 16 / elem_size, cpr = g.px / V, nrg = RES_NT / cpr;
    for (int bz = 0; bz < gz; ++bz)
        for (int by = 0; by < gy; ++by) {
            const int nrows = (res_split(g.ny, gy, by + 1, wy) - res_split(g.ny, gy, by, wy)) *
                              (res_split(g.nz, gz, bz + 1, wz) - res_split(g.nz, gz, bz, wz));
            const int rpg = (nrows + nrg - 1) / nrg;
            for (int w = 0; w < RES_NT / 32; ++w) {
                int first = -1;
                for (int l = 0; l < 32; ++l) {
                    const int tid = 32 * w + l, grp = tid / cpr, x = (tid - grp * cpr) * V;
                    const int r_lo = std::min(grp * rpg, nrows);
                    const int nrt = (grp < nrg && x < g.nx) ? std::min(rpg, nrows - r_lo) : 0;
                    if (l == 0) first = nrt;
                    else if (nrt != first) return false;
                }
            }
        }
    return true;
}

// ---- host side: the box decomposition.  Returns false if the grid does not fit the SMs' memory.
struct ResidentPlan {
    int gy, gz, ly, lz, zpad, pxs, dres, qres, rpt, rreg, wy, wz, rtm, uni;   // rtm: r and delta in tensor memory; uni: resident_uniform    // rreg: r does not fit the shared memory beside p
    unsigned smem_bytes;
};

inline bool resident_plan(const Geom& g, int elem_size, int nsm, bool lop, bool allow_tm, ResidentPlan& best)
{
    const int V = 16 / elem_size;
    const long long cpr = g.px / V;
    if (cpr > RES_NT) return false;                       // a row is one chunk per thread at most
    const long long nrg = RES_NT / cpr;
    const bool three = g.naxes == 3;
    const int zpad = three ? 1 : 0;
    const long long pxs = (long long)g.px + 2 * V;
    // a row of a face class costs 1.75 x an interior row under M (measured per-CTA phase times);
    // under L the two differ by one multiply
    const bool fy = !lop && g.fix[1], fz = !lop && three && g.fix[2];
    auto faces = [](int n, int a, int b) {                // cells of a face class in [a, b)
        int c = 0;
        for (int x : { 0, 1, n - 2, n - 1 }) c += (x >= a && x < b) ? 1 : 0;
        return c;
    };
    double best_cost = -1.0;
    for (int gy = 1; gy <= nsm && gy <= g.ny; ++gy) {
        int gz = nsm / gy;
        if (gz > g.nz) gz = g.nz;
        if (gz < 1) break;
        for (int weighted = 0; weighted < 2; ++weighted) {
            // (under L the weighted cut costs nothing and only matters where it makes the largest box small enough to fit)
            const int wy = (weighted && g.fix[1]) ? 3 : 0, wz = (weighted && three && g.fix[2]) ? 3 : 0;
            if (weighted && !wy && !wz) continue;
            long long ly = 0, lz = 0;                               // largest box
            double worst = 0.0;                                     // rows per thread of the slowest box, in interior-row units
            for (int bz = 0; bz < gz; ++bz) {
                const int k0 = res_split(g.nz, gz, bz, wz), k1 = res_split(g.nz, gz, bz + 1, wz);
                lz = std::max<long long>(lz, k1 - k0);
                for (int by = 0; by < gy; ++by) {
                    const int j0 = res_split(g.ny, gy, by, wy), j1 = res_split(g.ny, gy, by + 1, wy);
                    ly = std::max<long long>(ly, j1 - j0);
                    const double rows = (double)(((long long)(j1 - j0) * (k1 - k0) + nrg - 1) / nrg);
                    const double f = 1.0 + (fy ? 0.75 * faces(g.ny, j0, j1) / (j1 - j0) : 0.0) + (fz ? 0.75 * faces(g.nz, k0, k1) / (k1 - k0) : 0.0);
                    worst = std::max(worst, rows * f);
                }
            }
            const long long rpt = (ly * lz + nrg - 1) / nrg;           // rows per thread of the largest box
            const long long p_bytes = (lz + 2 * zpad) * (ly + 2) * pxs * elem_size;
            const long long v_bytes = rpt * RES_NT * 16;               // one more box vector (r, delta, q) in shared memory
            if (p_bytes > RES_SMEM_MAX || rpt > 32) continue;       // (one mask bit per row of a thread)
            const bool rtm = allow_tm && rpt <= RES_NI;              // r and delta fit the thread's share of tensor memory
            const bool rreg = rtm || p_bytes + v_bytes > RES_SMEM_MAX;
            const long long halo_rows = (gy > 1 ? 2 * lz : 0) + ((three && gz > 1) ? 2 * ly : 0);
            // time of an iteration ~ what the slowest thread walks three times (update, two stencils) + the halo rows a CTA updates
            const double cost = 3.0 * worst * (double)nrg + (double)halo_rows;
            if (best_cost < 0.0 || cost < best_cost) {
                best_cost = cost;
                best.gy = gy; best.gz = gz; best.ly = (int)ly; best.lz = (int)lz; best.zpad = zpad; best.pxs = (int)pxs;
                best.rpt = (int)rpt; best.rreg = rreg ? 1 : 0; best.wy = wy; best.wz = wz; best.rtm = rtm ? 1 : 0;
                best.dres = (!rreg && p_bytes + 2 * v_bytes <= RES_SMEM_MAX) ? 1 : 0;
                best.qres = rtm ? (p_bytes + v_bytes <= RES_SMEM_MAX ? 1 : 0) : (!rreg && p_bytes + 3 * v_bytes <= RES_SMEM_MAX) ? 1 : 0;
                best.smem_bytes = (unsigned)(p_bytes + (rreg ? 0 : v_bytes) + (best.dres ? v_bytes : 0) + (best.qres ? v_bytes : 0));
            }
        }
    }
    if (best_cost >= 0.0) best.uni = resident_uniform(g, elem_size, best.gy, best.gz, best.wy, best.wz) ? 1 : 0;
    return best_cost >= 0.0;
}

}  // namespace omni
