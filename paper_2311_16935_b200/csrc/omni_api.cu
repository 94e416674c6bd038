// omni_api.cu -- C ABI (include/omni.h) over the kernels of omni_kernels.cuh and omni_tma.cuh.
// Host logic only: argument validation, geometry constants (a0), workspace carving, launch configuration and the
// loop driver (CUDA graph with device-side conditional WHILE nodes, or a host-driven debug loop).
#include "omni_tma.cuh"
#include "omni_persist.cuh"
#include "omni_persist1.cuh"
#include "omni_resident.cuh"
#include "omni_loop.cuh"
#include "omni_mg.cuh"
#include "omni_slab.cuh"
#include "omni_noalloc.cuh"
#include "../../include/omni.h"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <mutex>
#include <vector>
#include <type_traits>

using namespace omni;

// Scratch of omni_source_noalloc_* (omni_noalloc.cuh): a fixed array in every GPU that loads the library, held until the
// process exits.  In HOST code this name is only a stand-in for the symbol, never a device address: the address is
// fetched per device with cudaGetSymbolAddress (noalloc_scratch_ptr below) and passed to the kernel.
static __device__ __align__(256) unsigned char g_noalloc_scratch[omni::NOALLOC_SCRATCH_BYTES];

// tile shape and pipeline depths of K2 / K3 / K4 (each can be overridden at build time for sweeps)
#ifndef OMNI_BY
#define OMNI_BY 8          // rows of a tile
#endif
#ifndef OMNI_R
#define OMNI_R 1           // rows of a tile per consumer warp (2 and 4 share N / S values in registers and halve the control overhead, but the halved warp count costs more: profiles/r2_loop_and_rows.md)
#endif
#ifndef OMNI_D3
#define OMNI_D3 6          // K3 ring depth
#endif
#ifndef OMNI_D4
#define OMNI_D4 4          // K4 ring depth in its 4-array iterations ({p_h, r, p_old, delta}); more in the 2-array ones
#endif
#ifndef OMNI_MINB
#define OMNI_MINB 3        // CTAs per SM the kernels are compiled for
#endif
#ifndef OMNI_D4_F64
#define OMNI_D4_F64 6      // fp64 K4 runs fewer CTAs per SM (registers): deeper ring from the same shared memory
#endif
#ifndef OMNI_TAPER_F
#define OMNI_TAPER_F 0.5     // tapered z segments (tma_config): fraction of the remaining planes per slot; 0 = uniform segments
#define OMNI_TAPER_MIN 24    // and the shortest segment
#endif
#define OMNI_PCG_INNER_REL_F32 1e-2         // omni_solve_pcg_f32: relative reduction after which an inner solve returns to the fp64 refinement
#define OMNI_PERSIST_MAX_CELLS 1500000LL   // automatic mode: grids up to this many padded cells take the persistent loop
#ifndef OMNI_LOOPK_MAX_CELLS
#define OMNI_LOOPK_MAX_CELLS 0LL           // ... and up to this many the cooperative tile-loop kernel (omni_loop.cuh, loop mode 4), if its grid fits one wave; 0: only on request
#endif
#define OMNI_PERSIST_SMALL_CELLS 65536LL   // persistent loop: 512-thread CTAs up to here, 1024-thread CTAs above

namespace {

std::atomic<long long> g_launches{0};
std::atomic<int> g_loop_mode{0};
std::atomic<double*> g_hist{nullptr};     // omni_set_history: device buffer for the eps_R history of the next solves
std::atomic<int> g_hist_cap{0};
std::atomic<int*> g_hist_k{nullptr};

// Per-call options (omni_options of include/omni.h).  omni_solve_ex_* installs its caller's struct for the duration of
// the call on the calling thread; every other entry point runs with the process-wide defaults the omni_set_* setters
// maintain.  Nothing a call reads can be changed by another thread's call.
struct CallOpts {
    int loop_mode;
    double* hist; int* hist_k; double* hist_p; int hist_cap;
    double* P64;
    int* status;
    int single_reduction;
};
thread_local const CallOpts* tl_opts = nullptr;
CallOpts current_opts()
{
    if (tl_opts) return *tl_opts;
    CallOpts o;
    o.loop_mode = g_loop_mode.load();
    o.hist = g_hist.load(); o.hist_k = g_hist_k.load(); o.hist_p = nullptr; o.hist_cap = g_hist_cap.load();
    o.P64 = nullptr; o.status = nullptr; o.single_reduction = 0;
    return o;
}

// optional per-kernel timing of the host-driven loop (omni_profile_*): CUDA events around every K2/K3/K4 launch
std::atomic<int> g_profile{0};
std::mutex g_prof_mu;
double g_prof_ms[3] = { 0, 0, 0 };
long long g_prof_n[3] = { 0, 0, 0 };
struct ProfRec { int which; cudaEvent_t e0, e1; };

#define CK(call)                                       \
    do {                                               \
        cudaError_t e__ = (call);                      \
        if (e__ != cudaSuccess) return OMNI_ERR_CUDA;  \
    } while (0)

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Workspace comes from a library-owned stream-ordered pool per device whose release threshold is unbounded: freed
// blocks stay mapped between calls (re-mapping ~5 GB costs ~10 ms per call with the default pool, measured on B200).
// omni_release_memory() trims it.
std::mutex g_pool_mu;
cudaMemPool_t g_pools[64] = {};

// Executable graphs in flight: cudaGraphExecDestroy on a running conditional graph blocks the host until it has
// finished (measured: the whole solve), so a launched graph is parked here with an event and destroyed by a later call
// (or by omni_release_memory) once the event has completed -- omni_solve_* with info == NULL stays asynchronous.
struct PendingGraph { cudaGraphExec_t exec; cudaEvent_t done; };
std::mutex g_pend_mu;
std::vector<PendingGraph> g_pending;

void reap_graphs(bool wait)
{
    std::lock_guard<std::mutex> lk(g_pend_mu);
    size_t keep = 0;
    for (size_t i = 0; i < g_pending.size(); ++i) {
        PendingGraph& pg = g_pending[i];
        if (wait) cudaEventSynchronize(pg.done);
        if (cudaEventQuery(pg.done) == cudaSuccess) {
            cudaGraphExecDestroy(pg.exec);
            cudaEventDestroy(pg.done);
        } else {
            g_pending[keep++] = pg;
        }
    }
    g_pending.resize(keep);
    cudaGetLastError();        // cudaErrorNotReady from the queries is not an error
}

void park_graph(cudaGraphExec_t exec, cudaStream_t st)
{
    cudaEvent_t ev = nullptr;
    if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess || cudaEventRecord(ev, st) != cudaSuccess) {
        if (ev) cudaEventDestroy(ev);
        cudaGetLastError();
        cudaGraphExecDestroy(exec);            // falls back to the blocking destroy
        return;
    }
    std::lock_guard<std::mutex> lk(g_pend_mu);
    g_pending.push_back(PendingGraph{ exec, ev });
}

cudaMemPool_t device_pool()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return nullptr; }
    std::lock_guard<std::mutex> lk(g_pool_mu);
    if (!g_pools[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        unsigned long long thr = ~0ULL;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
        g_pools[dev] = pool;
    }
    return g_pools[dev];
}

template <typename P>
cudaError_t pool_alloc(P** ptr, size_t bytes, cudaStream_t st)
{
    cudaMemPool_t pool = device_pool();
    if (!pool) return cudaMallocAsync((void**)ptr, bytes, st);
    return cudaMallocFromPoolAsync((void**)ptr, bytes, pool, st);
}

// Per-device facts, looked up once per device (the library serves any device of the process: pools, occupancy and
// kernel attributes are all per device).
constexpr int MAX_DEVICES = 64;
struct DevInfo { int dev, sms, coop; };
DevInfo device_info()
{
    static std::mutex mu;
    static DevInfo cache[MAX_DEVICES];
    static bool have[MAX_DEVICES] = {};
    DevInfo d{ 0, 148, 0 };
    if (cudaGetDevice(&d.dev) != cudaSuccess) { cudaGetLastError(); d.dev = 0; return d; }
    const bool cached = d.dev >= 0 && d.dev < MAX_DEVICES;
    std::lock_guard<std::mutex> lk(mu);
    if (cached && have[d.dev]) return cache[d.dev];
    if (cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, d.dev) != cudaSuccess || d.sms < 1) d.sms = 148;
    if (cudaDeviceGetAttribute(&d.coop, cudaDevAttrCooperativeLaunch, d.dev) != cudaSuccess) d.coop = 0;
    cudaGetLastError();
    if (cached) { cache[d.dev] = d; have[d.dev] = true; }
    return d;
}

// ------------------------------------------------------------------------------------------------ a0 constants

// c_aa for general spacing: measure of the rays that cross two directly opposed, parallel db x dc rectangles a
// distance da apart (A7; the geometry of PAPER.md:273 / Fig. 5b), written with the closed form of the
// classical radiative configuration factor between aligned parallel rectangles, X = db/da, Y = dc/da:
//   c_aa = 2 da^2 { ln sqrt[(1+X^2)(1+Y^2)/(1+X^2+Y^2)] + X sqrt(1+Y^2) atan(X/sqrt(1+Y^2))
//                   + Y sqrt(1+X^2) atan(Y/sqrt(1+X^2)) - X atan X - Y atan Y }.
double far_face_measure(double da, double db, double dc)
{
    const double X = db / da, Y = dc / da;
    const double X2 = 1.0 + X * X, Y2 = 1.0 + Y * Y;
    const double sx = std::sqrt(X2), sy = std::sqrt(Y2);
    const double v = 0.5 * std::log(X2 * Y2 / (X2 + Y2 - 1.0)) + X * sy * std::atan(X / sy) + Y * sx * std::atan(Y / sx)
                     - X * std::atan(X) - Y * std::atan(Y);
    return 2.0 * da * da * v;
}

struct HostConst {
    double F[3], Atot, c[3][3];
};

void host_constants(int naxes, double dx, double dy, double dz, HostConst& H)
{
    const double PI = 3.14159265358979323846;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) H.c[a][b] = 0.0;
    if (naxes == 2) {                                          // 2D scheme
        const double dd = std::hypot(dx, dy);
        H.F[0] = 2.0 * dy; H.F[1] = 2.0 * dx; H.F[2] = 0.0;     // Eq. 5 :75
        H.Atot = 4.0 * (dx + dy);                              // Eq. 8 :94
        H.c[0][0] = 2.0 * (dd - dx);                           // Eq. 17 :207-212
        H.c[1][1] = 2.0 * (dd - dy);
        H.c[0][1] = H.c[1][0] = dx + dy - dd;
        return;
    }
    const double d[3] = { dx, dy, dz };
    H.F[0] = PI * dy * dz; H.F[1] = PI * dx * dz; H.F[2] = PI * dx * dy;      // Eq. 23 :258
    H.Atot = 2.0 * PI * (dx * dy + dx * dz + dy * dz);                       // Eq. 24 :262
    double s[3];
    for (int a = 0; a < 3; ++a) {
        H.c[a][a] = far_face_measure(d[a], d[(a + 1) % 3], d[(a + 2) % 3]);
        s[a] = 0.5 * (H.F[a] - H.c[a][a]);      // c_ab + c_ac: the pieces of face a add up to F_a (Eq. 25 :266)
    }
    H.c[0][1] = H.c[1][0] = 0.5 * (s[0] + s[1] - s[2]);                      // c_jk = c_kj (:304)
    H.c[0][2] = H.c[2][0] = 0.5 * (s[0] + s[2] - s[1]);
    H.c[1][2] = H.c[2][1] = 0.5 * (s[1] + s[2] - s[0]);
}

uint32_t std_axis_code(int ax, int pos, int n, int naxes);

template <typename T>
Coef<T> make_coef(const HostConst& H, double dx, double dy, double dz, const Geom& g)
{
    Coef<T> K;
    const double d[3] = { dx, dy, dz };
    for (int a = 0; a < 3; ++a) {
        K.t[a] = (T)(H.F[a] / H.Atot);
        K.caa[a] = (T)(H.c[a][a] / H.Atot);
        K.cab[a] = (T)(H.c[a][(a + 1) % 3] / H.Atot);
        K.cac[a] = (T)(H.c[a][(a + 2) % 3] / H.Atot);
        K.hs[a] = (T)(d[a] * (H.F[a] / H.Atot) * 0.5);
        for (int bits = 0; bits < 32; ++bits) {
            const int far = bits & 1, nb = (bits >> 1) & 3, nc = (bits >> 3) & 3;
            K.lut[a][bits] = (T)((far * H.c[a][a] + nb * H.c[a][(a + 1) % 3] + nc * H.c[a][(a + 2) % 3]) / H.Atot);
        }
    }
    K.icode = g.icode;
    const int naxes = g.naxes;
    const int n3[3] = { g.nx, g.ny, g.nz };
    for (int ax = 0; ax < 3; ++ax)
        for (int cls = 0; cls < 4; ++cls) {
            const int pos = (cls < 2) ? cls : n3[ax] - 4 + cls;          // cells 0, 1, n-2, n-1
            const uint32_t code = (ax < naxes && n3[ax] >= 4) ? std_axis_code(ax, pos, n3[ax], naxes) : g.icode;
            for (int d = 0; d < 6; ++d) {
                const int a = d >> 1;
                const uint32_t bits = (code >> (5 * d)) & 31u;
                const int far = bits & 1, nb = (bits >> 1) & 3, nc = (bits >> 3) & 3;
                const double w = (far * H.c[a][a] + nb * H.c[a][(a + 1) % 3] + nc * H.c[a][(a + 2) % 3]) / H.Atot;
                K.fc[ax][cls][d] = (T)(H.F[a] / H.Atot - w);
            }
        }
    return K;
}

// ------------------------------------------------------------------------------------------------ geometry / workspace

// wcode of the cell at position pos of axis ax (length n) when only that axis is bounded (mirrors codes_kernel)
uint32_t std_axis_code(int ax, int pos, int n, int naxes)
{
    auto vx = [&](int ii) { return (ii >= 0 && ii < n) ? 1u : 0u; };
    uint32_t code = WCODE_VALID;
    for (int d = 0; d < 2 * naxes; ++d) {
        const int a = d >> 1, sg = (d & 1) ? -1 : 1;
        const int q = pos + (a == ax ? sg : 0);
        if (!vx(q)) continue;
        const int b = (a + 1) % 3, c = (a + 2) % 3;
        const uint32_t far = vx(q + (a == ax ? sg : 0));
        auto side = [&](int s_ax) -> uint32_t {
            if (s_ax >= naxes) return 0u;
            if (s_ax == ax) return vx(q + 1) + vx(q - 1);
            return 2u;
        };
        code |= (far | (side(b) << 1) | (side(c) << 3)) << (5 * d);
    }
    return code;
}

bool make_geom(int nx, int ny, int nz, int elem_size, Geom& g, int batch = 0)
{
    if (nx < 1 || ny < 1 || nz < 1) return false;
    const long long pad = (elem_size == 4) ? 8 : 4;        // one thread chunk = 32 bytes
    const long long px = ((long long)nx + pad - 1) / pad * pad;
    const long long npad = px * (long long)ny * (long long)nz;
    if (npad > (1LL << 40) || px > 0x7fffffff) return false;
    g.nx = nx; g.ny = ny; g.nz = nz; g.px = (int)px;
    g.kz0 = 0; g.kz1 = nz;
    g.pplane = px * ny;
    g.npad = npad;
    const int naxes = (nz > 1 && !batch) ? 3 : 2;
    g.naxes = naxes; g.batch = batch ? 1 : 0;
    const int n3[3] = { nx, ny, nz };
    for (int a = 0; a < 3; ++a) g.fix[a] = (a < naxes && n3[a] >= 4) ? 1 : 0;
    g.xfix = g.fix[0];
    g.icode = std_axis_code(0, 2, 5, naxes);
    g.tbx = 512 / elem_size; g.tby = OMNI_BY;                 // the K3/K4 tile (omni_tma.cuh TileGeom)
    g.ntx = (g.px + g.tbx - 1) / g.tbx; g.nty = (ny + g.tby - 1) / g.tby;
    g.twords = (nz + 31) / 32;
    return true;
}

template <typename T>
struct Workspace {
    uint8_t* link; uint32_t* wcode; uint32_t* flags; uint32_t* tflags;
    T *S, *r, *p0, *p1, *delta;
    double* P; double* P1; double* partial; Scalars* sc;
    double* slots;                // exchange slots of the persistent loop's grid barrier
};

size_t partial_slots(const Geom& g)
{
    // one fp64 slot per CTA and accumulator.  1D kernels: at most ceil(npad / 256) blocks.  Tile kernels: NACC x
    // (x tiles) x (y tiles) x (z segments) with at most nz segments; the finest tiling is K2's (64 cells x 8 rows,
    // NACC = 4).  A thin cross-section with a long z axis has far more tile CTAs than npad / 256 (launch_tma checks).
    const size_t lin = (size_t)((g.npad + 255) / 256) * 2 + 64;
    const size_t tile = (size_t)4 * (size_t)((g.px + 63) / 64) * (size_t)((g.ny + OMNI_BY - 1) / OMNI_BY) * (size_t)g.nz + 64;
    return std::max(lin, tile);
}

template <typename T>
size_t carve(const Geom& g, char* base, Workspace<T>* w)
{
    size_t off = 0;
    auto take = [&](size_t bytes) {
        char* p = base ? base + off : nullptr;
        off += align_up(bytes, 256);
        return p;
    };
    const size_t n = (size_t)g.npad;
    char* link = take(n);
    char* wcode = take(n * 4);
    char* flags = take(((n / 4 + 31) / 32 + 1) * 4);
    char* tflags = take((size_t)g.ntx * g.nty * g.twords * 4);
    char* S = take(n * sizeof(T));
    char* r = take(n * sizeof(T));
    char* p0 = take(n * sizeof(T));
    char* p1 = take(n * sizeof(T));
    char* delta = take(n * sizeof(T));
    char* P = take(n * sizeof(double));
    char* P1 = take(n * sizeof(double));
    char* partial = take(partial_slots(g) * sizeof(double));
    char* sc = take(sizeof(Scalars));
    char* slots = take(PERSIST_SLOT_BYTES);
    if (w) {
        w->slots = (double*)slots;
        w->link = (uint8_t*)link; w->wcode = (uint32_t*)wcode; w->flags = (uint32_t*)flags; w->tflags = (uint32_t*)tflags;
        w->S = (T*)S; w->r = (T*)r; w->p0 = (T*)p0; w->p1 = (T*)p1; w->delta = (T*)delta;
        w->P = (double*)P; w->P1 = (double*)P1; w->partial = (double*)partial; w->sc = (Scalars*)sc;
    }
    return off;
}

__global__ void init_scalars_kernel(Scalars* sc, double tol, int max_outer, int max_cg, double* hist = nullptr, int hist_cap = 0,
                                    int* hist_k = nullptr, double inner_rel = 0.0, double* hist_p = nullptr, int* status_out = nullptr,
                                    int defer = 0)
{
    Scalars s;
    memset(&s, 0, sizeof(s));
    s.tol = tol; s.max_outer = max_outer; s.max_cg = max_cg;
    s.inner_rel2 = inner_rel * inner_rel;
    s.hist = hist; s.hist_k = hist_k; s.hist_p = hist_p; s.hist_cap = hist_cap; s.hist_n = 0;
    s.status_out = status_out;
    s.defer = defer;
    s.inner_go = 0; s.outer_go = 1; s.status = ST_OK;
    s.dzero = 1;                     // no CG iteration has run yet: the first K2 takes delta as zero
    s.bar_count = 2;                 // grid barrier of the loop kernel: set 0, tag 1 against zeroed slots (omni_persist.cuh)
    *sc = s;
}

// ------------------------------------------------------------------------------------------------ launch configuration

struct MarchCfg { dim3 grid, block; ZSeg zs; };

// K2 / K3 / K4: TMA + mbarrier pipeline (omni_tma.cuh): 512-byte x 8-row tiles, 8 consumer warps + 1 producer warp,
// several CTAs per SM (shared memory: K3 6 stages x 10.8 KB, K4 4 x 17.4 KB or 7 x 9.4 KB by iteration parity,
// K2 5 x 10.3 KB fp32 / 4 x 14.8 KB fp64).
#ifndef OMNI_MINB_F64
#define OMNI_MINB_F64 2    // CTAs per SM the fp64 K4 is compiled for (registers)
#endif
template <typename T, bool LOP = false> using K3 = OpT3<T, OMNI_BY, OMNI_R, OMNI_D3, OMNI_MINB, LOP>;
template <typename T, bool LOP = false> using K4 = OpT4<T, OMNI_BY, OMNI_R, (sizeof(T) == 8 ? OMNI_D4_F64 : OMNI_D4), (sizeof(T) == 8 ? OMNI_MINB_F64 : OMNI_MINB), LOP>;
template <typename T> using K2 = OpT2<T, OMNI_BY, OMNI_R, (sizeof(T) == 8 ? 4 : 5), OMNI_MINB>;


template <class Op>
MarchCfg tma_config(const Geom& g)
{
    using TG = typename Op::TG;
    constexpr int SMEM = Op::SMEM_BYTES + 128;
    // CTA slots of the current device (SMs x resident CTAs); the shared-memory opt-in is a per-device attribute too
    static std::mutex mu;
    static int slots_cache[MAX_DEVICES] = {};
    const DevInfo di = device_info();
    int slots = 0;
    {
        std::lock_guard<std::mutex> lk(mu);
        const bool cached = di.dev >= 0 && di.dev < MAX_DEVICES;
        if (cached) slots = slots_cache[di.dev];
        if (slots == 0) {
            int occ = 1;
            cudaFuncSetAttribute(tma_kernel<Op>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, tma_kernel<Op>, TG::NTHR, SMEM);
            if (occ < 1) occ = 1;
            slots = di.sms * occ;
            if (cached) slots_cache[di.dev] = slots;
        }
    }
    const int nzr = g.kz1 - g.kz0;                 // planes to emit (a slab: the planes it owns)
    const int ntx = (g.px + TG::BX - 1) / TG::BX, nty = (g.ny + TG::BY - 1) / TG::BY;
    const long long tiles = (long long)ntx * nty;
    int best = 1;
    double best_cost = 1e300;
    for (int ns = 1; ns <= nzr; ns = (ns < 16 ? ns + 1 : ns + ns / 8)) {
        const int zlen = (nzr + ns - 1) / ns;
        const int nseg = (nzr + zlen - 1) / zlen;
        const long long ctas = tiles * nseg;
        const long long waves = (ctas + slots - 1) / slots;
        // CTAs next to masked cells run the slower general loop: with fewer than three waves a few of them become
        // the tail of the launch, so shallow schedules are penalised (measured on the masked 256^3 case)
        const double cost = (double)waves * (zlen + (nseg > 1 ? 2 : 0) + 3) * (waves < 3 ? 1.25 : 1.0);
        if (cost < best_cost) { best_cost = cost; best = nseg; }
        if (zlen <= 4) break;
    }
#ifdef OMNI_TUNING   // tuning builds only: force the number of z segments from the environment
    if (const char* ev = getenv("OMNI_NSEG")) { const int v = atoi(ev); if (v >= 1) best = v < nzr ? v : nzr; }
#endif
    MarchCfg c;
    c.zs.n = 0;
    c.zs.zlen = (nzr + best - 1) / best;
    int nseg = (nzr + c.zs.zlen - 1) / c.zs.zlen;
    // Tapered z segments: CTAs are dispatched in blockIdx order, z slowest, so the segments of
    // later z indices start later.  Long segments first (few halo planes, few pipeline fills), short ones last: the
    // launch then drains in the time of a short CTA instead of about half a long one.  Each segment takes the
    // fraction taper_f of the planes still to be assigned per CTA slot, but at least taper_min planes.
    double taper_f = OMNI_TAPER_F;
    int taper_min = OMNI_TAPER_MIN;
#ifdef OMNI_TUNING
    if (const char* ev = getenv("OMNI_TAPER_F")) taper_f = atof(ev);
    if (const char* ev = getenv("OMNI_TAPER_MIN")) taper_min = atoi(ev) > 1 ? atoi(ev) : 1;
#endif
    if (taper_f > 0.0 && (double)tiles * nzr / slots >= 2.0 * taper_min) {
        int k = 0, n = 0;
        bool ok = true;
        c.zs.k[0] = 0;
        while (k < nzr) {
            const double rem = (double)(nzr - k) * (double)tiles / slots;     // planes left per CTA slot
            int len = (int)(rem * taper_f + 0.5);
            if (len < taper_min) len = taper_min;
            if (nzr - k - len < (taper_min + 1) / 2) len = nzr - k;
            if (n == ZSeg::MAXSEG) { ok = false; break; }
            k += len;
            c.zs.k[++n] = k;
        }
        if (ok) { c.zs.n = n; nseg = n; }
    }
    c.grid = dim3(ntx, nty, nseg);
    c.block = dim3(TG::NTHR, 1, 1);
    return c;
}

template <class Op>
cudaError_t launch_tma(const Geom& g, const typename Op::Args& a, const TmaSet& maps, cudaStream_t st)
{
    const MarchCfg c = tma_config<Op>(g);
    // every CTA owns Op::NACC slots of the partial buffer (carve / partial_slots)
    if ((size_t)Op::NACC * c.grid.x * c.grid.y * c.grid.z > partial_slots(g)) return cudaErrorInvalidConfiguration;
    tma_kernel<Op><<<c.grid, c.block, Op::SMEM_BYTES + 128, st>>>(g, c.zs, a, maps);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return cudaGetLastError();
}

// host-side tensor maps (driver entry point fetched through the runtime: no link-time dependency on libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

template <typename T>
bool encode_map(CUtensorMap* m, const Geom& g, const T* base, int bx, int by)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t dims[3] = { (cuuint64_t)g.px, (cuuint64_t)g.ny, (cuuint64_t)g.nz };
    const cuuint64_t strides[2] = { (cuuint64_t)g.px * sizeof(T), (cuuint64_t)g.pplane * sizeof(T) };
    const cuuint32_t box[3] = { (cuuint32_t)bx, (cuuint32_t)by, 1u };
    const cuuint32_t estr[3] = { 1u, 1u, 1u };
    const CUtensorMapDataType dt = (sizeof(T) == 4) ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
    return fn(m, dt, 3, (void*)base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

inline unsigned blocks_for(long long n, int bs) { return (unsigned)((n + bs - 1) / bs); }

// ------------------------------------------------------------------------------------------------ setup shared by all entry points

// the caller's rows are whole 16-byte chunks of 4 cells: nx % 4 == 0, every given array 16-byte aligned (mask: 4-byte)
template <typename A, typename B, typename Cc>
bool rows_are_chunks(const Geom& g, const A* a, const B* b, const Cc* c, const unsigned char* mask)
{
    if (g.nx % 4 != 0 || g.nz > 65535 || (g.ny + SETUP_BY - 1) / SETUP_BY > 65535) return false;
    const uintptr_t bits = (uintptr_t)a | (uintptr_t)b | (uintptr_t)c;
    return (bits & 15) == 0 && ((uintptr_t)mask & 3) == 0;
}
inline dim3 setup_grid(const Geom& g)
{
    return dim3((unsigned)((g.px / 4 + SETUP_BX - 1) / SETUP_BX), (unsigned)((g.ny + SETUP_BY - 1) / SETUP_BY), (unsigned)g.nz);
}

template <typename T>
int setup_codes(const Geom& g, const Workspace<T>& w, const T* gx, const T* gy, const T* gz, const uint8_t* mask,
                cudaStream_t st)
{
    uint8_t* vbyte = reinterpret_cast<uint8_t*>(w.p0);       // scratch: p0 is cleared afterwards
    if (rows_are_chunks(g, gx, gy, gz, mask))
        validity4_kernel<T><<<setup_grid(g), dim3(SETUP_BX, SETUP_BY), 0, st>>>(g, gx, gy, gz, mask, vbyte);
    else
        validity_kernel<T><<<blocks_for(g.npad, 256), 256, 0, st>>>(g, gx, gy, gz, mask, vbyte);
    CK(cudaGetLastError());
    CK(cudaMemsetAsync(w.tflags, 0, (size_t)g.ntx * g.nty * g.twords * 4, st));
    // work list of the groups that need the cell-by-cell decode: scratch in p1 (4 bytes per 4-cell group at most),
    // its counter in the first word of the barrier slots (both are cleared again below / before their own use)
    uint32_t* worklist = reinterpret_cast<uint32_t*>(w.p1);
    unsigned int* work_count = reinterpret_cast<unsigned int*>(w.slots);
    CK(cudaMemsetAsync(work_count, 0, sizeof(unsigned int), st));
    codes_kernel<<<blocks_for(g.npad / 4, 256), 256, 0, st>>>(g, vbyte, w.link, w.wcode, w.flags, worklist, work_count);
    CK(cudaGetLastError());
    {
        const int nsm = device_info().sms;
        long long nb = (g.npad / 4 + 127) / 128;
        if (nb > 16LL * nsm) nb = 16LL * nsm;
        if (nb < 1) nb = 1;
        codes_worklist_kernel<<<(unsigned)nb, 128, 0, st>>>(g, vbyte, w.link, w.wcode, w.flags, w.tflags, worklist, work_count);
        CK(cudaGetLastError());
    }
    g_launches.fetch_add(3, std::memory_order_relaxed);
    const size_t n = (size_t)g.npad;
    CK(cudaMemsetAsync(w.p0, 0, n * sizeof(T), st));
    CK(cudaMemsetAsync(w.p1, 0, n * sizeof(T), st));
    CK(cudaMemsetAsync(w.delta, 0, n * sizeof(T), st));
    CK(cudaMemsetAsync(w.r, 0, n * sizeof(T), st));          // pad cells of r are never written afterwards
    CK(cudaMemsetAsync(w.P, 0, n * sizeof(double), st));
    CK(cudaMemsetAsync(w.P1, 0, n * sizeof(double), st));
    return OMNI_OK;
}

template <typename T>
int launch_source(const Geom& g, const Workspace<T>& w, const Coef<T>& K, const T* gx, const T* gy, const T* gz,
                  cudaStream_t st)
{
    unsigned nb = blocks_for(g.npad, 256);
    if (nb > 4736u) nb = 4736u;                 // 148 SMs x 8 CTAs x 4: the kernel is grid-stride
    if (rows_are_chunks(g, gx, gy, gz, (const unsigned char*)nullptr)) {
        const long long items = (long long)((g.ny + SETUP_BY - 1) / SETUP_BY) * g.nz;
        if (items < (long long)nb) nb = (unsigned)items;
        source4_kernel<T><<<nb, dim3(SETUP_BX, SETUP_BY), 0, st>>>(g, gx, gy, gz, w.link, K, w.S, w.sc, w.partial);
    } else {
        source_kernel<T><<<nb, 256, 0, st>>>(g, gx, gy, gz, w.link, K, w.S, w.sc, w.partial);
    }
    g_launches.fetch_add(1, std::memory_order_relaxed);
    CK(cudaGetLastError());
    return OMNI_OK;
}

template <typename T>
typename K2<T>::Args k2_args(const Geom& g, const Workspace<T>& w, const HostConst& H, CondHandles ch, int fold)
{
    (void)g;
    typename K2<T>::Args a;
    a.Pbuf[0] = w.P; a.Pbuf[1] = fold ? w.P1 : w.P; a.r = w.r; a.link = w.link; a.flags = w.flags; a.tflags = w.tflags;
    for (int i = 0; i < 3; ++i) a.t[i] = H.F[i] / H.Atot;
    a.sc = w.sc; a.partial = w.partial; a.cond = ch; a.fold_delta = fold;
    return a;
}
template <typename T, bool LOP = false>
typename K3<T, LOP>::Args k3_args(const Workspace<T>& w, const Coef<T>& K, CondHandles ch)
{
    typename K3<T, LOP>::Args a;
    a.pbuf[0] = w.p0; a.pbuf[1] = w.p1; a.wcode = w.wcode; a.link = w.link; a.flags = w.flags; a.tflags = w.tflags;
    a.K = K; a.sc = w.sc; a.partial = w.partial; a.cond = ch;
    return a;
}
template <typename T, bool LOP = false>
typename K4<T, LOP>::Args k4_args(const Workspace<T>& w, const Coef<T>& K, CondHandles ch)
{
    typename K4<T, LOP>::Args a;
    a.r = w.r; a.delta = w.delta; a.p_fixed = -1; a.wcode = w.wcode; a.link = w.link; a.flags = w.flags; a.tflags = w.tflags;
    a.K = K; a.sc = w.sc; a.partial = w.partial; a.cond = ch; a.q_out = nullptr; a.pcg = 0;
    return a;
}
template <typename T>
bool make_tma_set(const Geom& g, const Workspace<T>& w, TmaSet& m)
{
    using TG = typename K3<T>::TG;
    const int hx = TG::BX + 2 * TG::HX, hy = TG::BY + 2;
    return encode_map<T>(&m.r_h, g, w.r, hx, hy) && encode_map<T>(&m.p_h[0], g, w.p0, hx, hy) &&
           encode_map<T>(&m.p_h[1], g, w.p1, hx, hy) && encode_map<T>(&m.r_c, g, w.r, TG::BX, TG::BY) &&
           encode_map<T>(&m.d_c, g, w.delta, TG::BX, TG::BY) &&
           encode_map<T>(&m.p_c[0], g, w.p0, TG::BX, TG::BY) && encode_map<T>(&m.p_c[1], g, w.p1, TG::BX, TG::BY) &&
           encode_map<double>(&m.P_h[0], g, w.P, 64 + 4, TG::BY + 2) && encode_map<double>(&m.P_h[1], g, w.P1, 64 + 4, TG::BY + 2) &&
           encode_map<T>(&m.d2_h, g, w.delta, 64 + 2 * (16 / (int)sizeof(T)), TG::BY + 2) &&
           encode_map<T>(&m.S_c, g, w.S, 64, TG::BY);
}

// ------------------------------------------------------------------------------------------------ loop drivers

// delta += alpha p of a CG iteration K4 left pending (lazy delta); no-op kernel when nothing is pending
template <typename T>
cudaError_t launch_flush(const Geom& g, const Workspace<T>& w, cudaStream_t st)
{
    const int nsm = device_info().sms;
    constexpr int V = 16 / (int)sizeof(T);
    long long nb = (g.npad / V + 255) / 256;
    if (nb > 8LL * nsm) nb = 8LL * nsm;
    if (nb < 1) nb = 1;
    flush_delta_kernel<T><<<(unsigned)nb, 256, 0, st>>>(g.npad, w.delta, w.p0, w.p1, w.sc);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return cudaGetLastError();
}

// longest wait at a grid barrier of the persistent loop: 30 s by default (a healthy grid that is merely descheduled
// on a time-shared GPU must not be reported as an error), OMNI_BARRIER_TIMEOUT_S overrides
unsigned long long barrier_timeout_ns()
{
    static unsigned long long v = 0;
    if (v == 0) {
        const char* e = getenv("OMNI_BARRIER_TIMEOUT_S");
        const double s = e ? atof(e) : 30.0;
        v = (unsigned long long)((s > 0.001 ? s : 30.0) * 1e9);
    }
    return v;
}

// ---- cooperative tile-loop kernel (omni_loop.cuh): the whole of Alg. 1 in one launch of the TMA pipeline
template <typename T, bool LOP> struct LoopK {
    using A2 = K2<T>;
    using A = K3<T, LOP>;
    using B = K4<T, LOP>;
    static constexpr int MINB = (sizeof(T) == 8) ? OMNI_MINB_F64 : OMNI_MINB;
    static constexpr int S34 = ((int)A::SMEM_BYTES > (int)B::SMEM_BYTES ? (int)A::SMEM_BYTES : (int)B::SMEM_BYTES);
    static constexpr int SMEM = (S34 > (int)A2::SMEM_BYTES ? S34 : (int)A2::SMEM_BYTES) + 128;
    static auto kernel() { return tma_loop_kernel<A2, A, B, MINB>; }
};

// one column (tile x z segment) per CTA, all CTAs resident at once: segments = resident slots / tiles, at least
// OMNI_LOOPK_MINZ planes each.  Returns false if the tiles alone exceed the slots (the caller takes the graph loop).
#ifndef OMNI_LOOPK_MINZ
#define OMNI_LOOPK_MINZ 6
#endif
template <typename T, bool LOP>
bool loop_config(const Geom& g, MarchCfg& c)
{
    using L = LoopK<T, LOP>;
    using TG = typename L::A::TG;
    static std::mutex mu;
    static int slots_cache[MAX_DEVICES] = {};
    const DevInfo di = device_info();
    if (!di.coop) return false;
    int slots = 0;
    {
        std::lock_guard<std::mutex> lk(mu);
        const bool cached = di.dev >= 0 && di.dev < MAX_DEVICES;
        if (cached) slots = slots_cache[di.dev];
        if (slots == 0) {
            int occ = 0;
            cudaFuncSetAttribute(L::kernel(), cudaFuncAttributeMaxDynamicSharedMemorySize, L::SMEM);
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, L::kernel(), TG::NTHR, L::SMEM);
            cudaGetLastError();
            slots = occ < 1 ? -1 : di.sms * occ;
            if (cached) slots_cache[di.dev] = slots;
        }
    }
    const int ntx = (g.px + TG::BX - 1) / TG::BX, nty = (g.ny + TG::BY - 1) / TG::BY;
    const long long tiles = (long long)ntx * nty;
    if (slots < 1 || tiles > slots || tiles > PERSIST_MAX_CTAS) return false;
    int nseg = (int)(slots / tiles);
#ifdef OMNI_TUNING
    if (const char* ev = getenv("OMNI_LOOPK_NSEG")) { const int v = atoi(ev); if (v >= 1 && v < nseg) nseg = v; }
#endif
    if (nseg > g.nz / OMNI_LOOPK_MINZ) nseg = g.nz / OMNI_LOOPK_MINZ;
    if (nseg < 1) nseg = 1;
    if (tiles * nseg > PERSIST_MAX_CTAS) nseg = (int)(PERSIST_MAX_CTAS / tiles);
    c.zs.n = 0;
    c.zs.zlen = (g.nz + nseg - 1) / nseg;
    nseg = (g.nz + c.zs.zlen - 1) / c.zs.zlen;
    c.grid = dim3((unsigned)(tiles * nseg), 1, 1);
    c.block = dim3(TG::NTHR, 1, 1);
    return true;
}

// Returns -100 if the grid does not fit one wave on this device or cannot be launched cooperatively (the caller then
// takes the graph loop).
template <typename T, bool LOP>
int run_loop_loopk(const Geom& g, const Workspace<T>& w, const HostConst& H, const Coef<T>& K, cudaStream_t st)
{
    using L = LoopK<T, LOP>;
    MarchCfg c;
    if (!loop_config<T, LOP>(g, c)) return -100;
    TmaSet maps;
    if (!make_tma_set<T>(g, w, maps)) return OMNI_ERR_CUDA;
    CondHandles ch{ 0, 0, 0 };
    LoopArgs<typename L::A2, typename L::A, typename L::B> a;
    a.a2 = k2_args<T>(g, w, H, ch, 1);
    a.a3 = k3_args<T, LOP>(w, K, ch);
    a.a4 = k4_args<T, LOP>(w, K, ch);
    a.slots = w.slots;
    a.timeout_ns = barrier_timeout_ns();
    CK(cudaMemsetAsync(w.slots, 0, (size_t)8 * c.grid.x * sizeof(double), st));
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = c.grid; cfg.blockDim = c.block; cfg.dynamicSmemBytes = L::SMEM; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, L::kernel(), g, c.zs, a, maps) != cudaSuccess) {
        cudaGetLastError();
        return -100;
    }
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return OMNI_OK;
}

// Host-driven loop (debug / profiling): one synchronisation per outer iteration (plus one per 16 CG iterations).
template <typename T, bool LOP>
int run_loop_host(const Geom& g, const Workspace<T>& w, const HostConst& H, const Coef<T>& K, int max_outer, int max_cg,
                  cudaStream_t st)
{
    CondHandles ch{ 0, 0, 0 };
    const auto a2 = k2_args<T>(g, w, H, ch, 1);
    const auto a3 = k3_args<T, LOP>(w, K, ch);
    const auto a4 = k4_args<T, LOP>(w, K, ch);
    TmaSet maps;
    if (!make_tma_set<T>(g, w, maps)) return OMNI_ERR_CUDA;
    const bool prof = g_profile.load() != 0;
    std::vector<ProfRec> recs;
    auto timed = [&](int which, auto&& launch) -> cudaError_t {
        if (!prof) return launch();
        ProfRec r{ which, nullptr, nullptr };
        cudaEventCreate(&r.e0); cudaEventCreate(&r.e1);
        cudaEventRecord(r.e0, st);
        cudaError_t e = launch();
        cudaEventRecord(r.e1, st);
        recs.push_back(r);
        return e;
    };
    Scalars h;
    memset(&h, 0, sizeof(h));
    int rc = OMNI_OK;
    for (long long it = 0; it <= (long long)max_outer && rc == OMNI_OK; ++it) {
        if (timed(0, [&] { return launch_tma<K2<T>>(g, a2, maps, st); }) != cudaSuccess) { rc = OMNI_ERR_CUDA; break; }
        int done = 0;
        bool synced = false;
        while (done < max_cg) {
            const int batch = (max_cg - done < 16) ? (max_cg - done) : 16;
            for (int c = 0; c < batch; ++c) {
                if (timed(1, [&] { return launch_tma<K3<T, LOP>>(g, a3, maps, st); }) != cudaSuccess) rc = OMNI_ERR_CUDA;
                if (timed(2, [&] { return launch_tma<K4<T, LOP>>(g, a4, maps, st); }) != cudaSuccess) rc = OMNI_ERR_CUDA;
            }
            done += batch;
            if (rc != OMNI_OK) break;
            if (cudaMemcpyAsync(&h, w.sc, sizeof(Scalars), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
                cudaStreamSynchronize(st) != cudaSuccess) { rc = OMNI_ERR_CUDA; break; }
            synced = true;
            if (!h.inner_go) break;
        }
        if (rc == OMNI_OK && launch_flush<T>(g, w, st) != cudaSuccess) rc = OMNI_ERR_CUDA;
        if (rc == OMNI_OK && !synced) {
            if (cudaMemcpyAsync(&h, w.sc, sizeof(Scalars), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
                cudaStreamSynchronize(st) != cudaSuccess) rc = OMNI_ERR_CUDA;
        }
        if (!h.outer_go) break;
    }
    if (prof) {
        cudaStreamSynchronize(st);
        // launches that found the loop flag cleared return at once; keep only those that did the work:
        // a kernel that ran is >= 10x longer than an idle one, so split at 1/4 of the per-kind median
        std::vector<float> ms(recs.size(), 0.f);
        for (size_t i = 0; i < recs.size(); ++i) cudaEventElapsedTime(&ms[i], recs[i].e0, recs[i].e1);
        std::lock_guard<std::mutex> lk(g_prof_mu);
        for (int kind = 0; kind < 3; ++kind) {
            std::vector<float> v;
            for (size_t i = 0; i < recs.size(); ++i) if (recs[i].which == kind) v.push_back(ms[i]);
            if (v.empty()) continue;
            std::vector<float> sorted = v;
            std::sort(sorted.begin(), sorted.end());
            const float cut = 0.25f * sorted[sorted.size() / 2];
            for (float x : v) if (x >= cut) { g_prof_ms[kind] += x; g_prof_n[kind] += 1; }
        }
        for (auto& r : recs) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
    }
    return rc;
}

// ------------------------------------------------------------------------------------------------ multigrid preconditioner (omni_mg.cuh)
template <typename T>
struct MgHier {
    int nlev;
    MgLevel<T> L[MG_MAX_LEVELS];
    void* mem;                       // one pool block: level-0 iterates, coarse links / iterates / right-hand sides
    long long launches_per_cycle;    // kernels one V-cycle enqueues (launch accounting)
};

// Level sizes and weights (reading R-P1), one pool block for all levels, link bytes of the coarse levels.
// Level 0 aliases the solver's arrays: link bytes and right-hand side r in the padded layout.
template <typename T>
int mg_build(const Geom& g, const Workspace<T>& w, const HostConst& H, MgHier<T>& M, cudaStream_t st)
{
    M.nlev = 0; M.mem = nullptr; M.launches_per_cycle = 0;
    MgLevel<T> L0 = {};
    L0.nx = g.nx; L0.ny = g.ny; L0.nz = g.nz; L0.px = g.px; L0.pplane = g.pplane; L0.n = g.npad;
    for (int a = 0; a < 3; ++a) L0.w[a] = (T)(a < g.naxes ? H.F[a] / H.Atot : 0.0);
    double wd[3] = { H.F[0] / H.Atot, H.F[1] / H.Atot, g.naxes == 3 ? H.F[2] / H.Atot : 0.0 };
    L0.link = w.link; L0.b = w.r;
    M.L[M.nlev++] = L0;
    while (M.nlev < MG_MAX_LEVELS) {
        MgLevel<T>& F = M.L[M.nlev - 1];
        const bool ok[3] = { F.nx >= MG_MIN_COARSEN, F.ny >= MG_MIN_COARSEN, g.naxes == 3 && F.nz >= MG_MIN_COARSEN };
        double wmax = 0.0;
        for (int a = 0; a < 3; ++a)
            if (ok[a] && wd[a] > wmax) wmax = wd[a];
        F.hx = ok[0] && wd[0] >= MG_THETA * wmax;                    // strongly coupled axes only (reading R-P1)
        F.hy = ok[1] && wd[1] >= MG_THETA * wmax;
        F.hz = ok[2] && wd[2] >= MG_THETA * wmax;
        const int m = F.hx + F.hy + F.hz;
        if (m == 0) break;
        MgLevel<T> C = {};
        C.nx = F.hx ? (F.nx + 1) / 2 : F.nx; C.ny = F.hy ? (F.ny + 1) / 2 : F.ny; C.nz = F.hz ? (F.nz + 1) / 2 : F.nz;
        C.px = (C.nx + 3) / 4 * 4;            // rows padded to whole 4-cell chunks (pad cells: link 0, values 0)
        C.pplane = (long long)C.px * C.ny; C.n = C.pplane * C.nz;
        const int h[3] = { F.hx, F.hy, F.hz };
        for (int a = 0; a < 3; ++a) {
            wd[a] = wd[a] * (double)(1 << m) * (h[a] ? 0.25 : 1.0);
            C.w[a] = (T)wd[a];
        }
        M.L[M.nlev++] = C;
    }
    M.L[M.nlev - 1].hx = M.L[M.nlev - 1].hy = M.L[M.nlev - 1].hz = 0;
    // carve
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off += align_up(bytes, 256); return o; };
    size_t o_x[MG_MAX_LEVELS], o_xt[MG_MAX_LEVELS], o_b[MG_MAX_LEVELS], o_link[MG_MAX_LEVELS];
    for (int l = 0; l < M.nlev; ++l) {
        const size_t n = (size_t)M.L[l].n;
        o_x[l] = take(n * sizeof(T)); o_xt[l] = take(n * sizeof(T));
        o_b[l] = l ? take(n * sizeof(T)) : 0; o_link[l] = l ? take(n) : 0;
    }
    const size_t o_vc = take(M.nlev > 1 ? (size_t)M.L[1].n : 1);
    if (pool_alloc(&M.mem, off, st) != cudaSuccess) { cudaGetLastError(); M.mem = nullptr; return OMNI_ERR_ALLOC; }
    char* base = (char*)M.mem;
    for (int l = 0; l < M.nlev; ++l) {
        M.L[l].x = (T*)(base + o_x[l]); M.L[l].xt = (T*)(base + o_xt[l]);
        if (l) { M.L[l].b = (T*)(base + o_b[l]); M.L[l].link = (const uint8_t*)(base + o_link[l]); }
    }
    uint8_t* vc = (uint8_t*)(base + o_vc);
    for (int l = 1; l < M.nlev; ++l) {
        mg_coarse_valid_kernel<T><<<mg_grid(M.L[l]), mg_block(), 0, st>>>(M.L[l - 1], M.L[l], vc);
        mg_link_kernel<T><<<mg_grid(M.L[l]), mg_block(), 0, st>>>(M.L[l], vc, (uint8_t*)(base + o_link[l]), g.naxes);
        g_launches.fetch_add(2, std::memory_order_relaxed);
    }
    CK(cudaGetLastError());
    return OMNI_OK;
}

// enqueue B_l(b_l) (V-cycle from level l down and up again); returns the array that holds the result
template <typename T>
T* mg_vcycle(MgHier<T>& M, int l, cudaStream_t st)
{
    const MgLevel<T>& L = M.L[l];
    const bool last = (l + 1 == M.nlev);
    const dim3 nt = mg_block();
    dim3 nb = mg_grid(L);
    nb.x = (unsigned)((L.px / 4 + MG_BX - 1) / MG_BX);               // four cells of a row per thread
    T *cur = L.x, *oth = L.xt;
    mg_jacobi4_kernel<T, true><<<nb, nt, 0, st>>>(L, nullptr, cur);
    M.launches_per_cycle += 1;
    for (int sw = 1; sw < (last ? MG_NU_COARSEST : MG_NU); ++sw) {
        mg_jacobi4_kernel<T, false><<<nb, nt, 0, st>>>(L, cur, oth);
        std::swap(cur, oth);
        M.launches_per_cycle += 1;
    }
    if (last) return cur;
    const MgLevel<T>& C = M.L[l + 1];
    if (L.hx) {                                                      // x halved: two coarse cells (one fine chunk) per thread
        dim3 nc = mg_grid(C);
        nc.x = (unsigned)((C.px / 2 + MG_BX - 1) / MG_BX);
        mg_residual_restrict4_kernel<T><<<nc, nt, 0, st>>>(L, C, cur);
    } else {
        mg_residual_restrict_kernel<T><<<mg_grid(C), nt, 0, st>>>(L, C, cur);
    }
    T* e = mg_vcycle<T>(M, l + 1, st);
    mg_prolong_add4_kernel<T><<<nb, nt, 0, st>>>(L, C, cur, e);
    M.launches_per_cycle += 2;
    for (int sw = 0; sw < MG_NU; ++sw) {
        mg_jacobi4_kernel<T, false><<<nb, nt, 0, st>>>(L, cur, oth);
        std::swap(cur, oth);
        M.launches_per_cycle += 1;
    }
    return cur;
}

// CUDA-graph loop: outer WHILE { K2 ; inner WHILE { K3 ; K4 } }, conditions written by the kernels' last CTAs.
// mg != nullptr (omni_solve_pcg): the inner body is one PRECONDITIONED CG iteration -- V-cycle z = B r, rho = r.z and
// beta (mg_dot_kernel), K3 with z in the place of r (p = z + beta p), K4 testing ||r|| only.
template <typename T, bool LOP>
int run_loop_graph(const Geom& g, const Workspace<T>& w, const HostConst& H, const Coef<T>& K, cudaStream_t st,
                   MgHier<T>* mg = nullptr)
{
    cudaGraph_t G = nullptr;
    cudaGraphExec_t exec = nullptr;
    cudaStream_t cap = nullptr;
    int rc = OMNI_ERR_CUDA;
    reap_graphs(false);
    // occupancy queries happen here, outside any stream capture (results are cached per kernel)
    (void)tma_config<K2<T>>(g); (void)tma_config<K3<T, LOP>>(g); (void)tma_config<K4<T, LOP>>(g);
    TmaSet maps;
    if (!make_tma_set<T>(g, w, maps)) return OMNI_ERR_CUDA;
    do {
        if (cudaGraphCreate(&G, 0) != cudaSuccess) break;
        cudaGraphConditionalHandle hOuter, hInner;
        if (cudaGraphConditionalHandleCreate(&hOuter, G, 1, cudaGraphCondAssignDefault) != cudaSuccess) break;
        if (cudaGraphConditionalHandleCreate(&hInner, G, 0, cudaGraphCondAssignDefault) != cudaSuccess) break;
        CondHandles ch{ (unsigned long long)hOuter, (unsigned long long)hInner, 3 };

        cudaGraphNodeParams po = {};
        po.type = cudaGraphNodeTypeConditional;
        po.conditional.handle = hOuter;
        po.conditional.type = cudaGraphCondTypeWhile;
        po.conditional.size = 1;
        cudaGraphNode_t nOuter;
        if (cudaGraphAddNode(&nOuter, G, nullptr, 0, &po) != cudaSuccess) break;
        cudaGraph_t bodyOuter = po.conditional.phGraph_out[0];

        if (cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking) != cudaSuccess) break;
        // K2 into the outer body
        if (cudaStreamBeginCaptureToGraph(cap, bodyOuter, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) != cudaSuccess) break;
        cudaError_t e = launch_tma<K2<T>>(g, k2_args<T>(g, w, H, ch, 1), maps, cap);
        cudaGraph_t tmp = nullptr;
        if (cudaStreamEndCapture(cap, &tmp) != cudaSuccess || e != cudaSuccess) break;
        cudaGraphNode_t k2node;
        size_t nn = 1;
        if (cudaGraphGetNodes(bodyOuter, &k2node, &nn) != cudaSuccess || nn != 1) break;

        cudaGraphNodeParams pi = {};
        pi.type = cudaGraphNodeTypeConditional;
        pi.conditional.handle = hInner;
        pi.conditional.type = cudaGraphCondTypeWhile;
        pi.conditional.size = 1;
        cudaGraphNode_t nInner;
        if (cudaGraphAddNode(&nInner, bodyOuter, &k2node, 1, &pi) != cudaSuccess) break;
        cudaGraph_t bodyInner = pi.conditional.phGraph_out[0];

        if (cudaStreamBeginCaptureToGraph(cap, bodyInner, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) != cudaSuccess) break;
        auto a4 = k4_args<T, LOP>(w, K, ch);
        TmaSet maps3 = maps;
        bool okm = true;
        if (mg) {
            mg->launches_per_cycle = 0;
            T* z = mg_vcycle<T>(*mg, 0, cap);
            unsigned nbd = blocks_for(g.npad, 256);
            if (nbd > 4736u) nbd = 4736u;
            mg_dot_kernel<T><<<nbd, 256, 0, cap>>>(g.npad, w.r, z, w.sc, w.partial, ch);
            mg->launches_per_cycle += 1;
            using TG = typename K3<T>::TG;
            okm = encode_map<T>(&maps3.r_h, g, z, TG::BX + 2 * TG::HX, TG::BY + 2);     // K3 forms p = z + beta p
            a4.pcg = 1;
        }
        cudaError_t e3 = launch_tma<K3<T, LOP>>(g, k3_args<T, LOP>(w, K, ch), maps3, cap);
        cudaError_t e4 = launch_tma<K4<T, LOP>>(g, a4, maps, cap);
        if (cudaStreamEndCapture(cap, &tmp) != cudaSuccess || e3 != cudaSuccess || e4 != cudaSuccess || !okm || cudaGetLastError() != cudaSuccess) break;
        // after the inner loop: the delta update an even last iteration left pending
        if (cudaStreamBeginCaptureToGraph(cap, bodyOuter, &nInner, nullptr, 1, cudaStreamCaptureModeThreadLocal) != cudaSuccess) break;
        cudaError_t ef = launch_flush<T>(g, w, cap);
        if (cudaStreamEndCapture(cap, &tmp) != cudaSuccess || ef != cudaSuccess) break;
        g_launches.fetch_sub(4, std::memory_order_relaxed);     // captured, not launched; counted from the device state

        if (cudaGraphInstantiate(&exec, G, 0) != cudaSuccess) break;
        if (cudaGraphLaunch(exec, st) != cudaSuccess) break;
        rc = OMNI_OK;
    } while (0);
    if (rc != OMNI_OK) cudaGetLastError();
    if (exec) {
        if (rc == OMNI_OK) park_graph(exec, st); else cudaGraphExecDestroy(exec);
    }
    if (G) cudaGraphDestroy(G);
    if (cap) cudaStreamDestroy(cap);
    return rc;
}

// Persistent loop: the whole iteration in one cooperative launch (omni_persist.cuh).  Returns -100 if the device cannot
// co-schedule the grid (the caller then falls back to the graph loop).  NT = threads per CTA: 512 (up to 128 registers)
// for the smallest grids, where one row segment per warp is all there is; 1024 where a warp has several segments and
// twice the warps in flight hide more of the L2 latency.
template <typename T, int NT, bool LOP>
int launch_persist(const Geom& g, const Workspace<T>& w, const HostConst& H, const Coef<T>& K, int nsm, cudaStream_t st)
{
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, persist_kernel<T, NT, LOP>, NT, 0) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        return -100;
    }
    PersistArgs<T> a;
    a.r = w.r; a.pbuf[0] = w.p0; a.pbuf[1] = w.p1; a.delta = w.delta; a.S = w.S; a.Pbuf[0] = w.P; a.Pbuf[1] = w.P1;
    a.link = w.link; a.wcode = w.wcode; a.flags = w.flags; a.K = K;
    for (int i = 0; i < 3; ++i) a.t[i] = H.F[i] / H.Atot;
    a.sc = w.sc; a.slots = w.slots;
    a.timeout_ns = barrier_timeout_ns();
    // one warp per 64-cell row segment of K2 (the finest phase), at most one CTA per SM, at most PERSIST_MAX_CTAS slots
    const long long tasks = (long long)g.ny * g.nz * ((g.nx + 63) / 64);
    const int nw = NT / 32;
    long long G = (tasks + nw - 1) / nw;
    if (G > nsm) G = nsm;
    if (G > PERSIST_MAX_CTAS) G = PERSIST_MAX_CTAS;
    if (G < 1) G = 1;
    CK(cudaMemsetAsync(w.slots, 0, (size_t)8 * G * sizeof(double), st));
    Geom gg = g;
    void* params[2] = { (void*)&gg, (void*)&a };
    // a grid the context cannot co-schedule (fewer usable SMs than the device reports: MPS, green contexts) is not an
    // error of the solve: report "cannot" and let the caller take the graph loop
    if (cudaLaunchCooperativeKernel((const void*)persist_kernel<T, NT, LOP>, dim3((unsigned)G), dim3(NT), params, 0, st) != cudaSuccess) {
        cudaGetLastError();
        return -100;
    }
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return OMNI_OK;
}

template <typename T, bool LOP>
int run_loop_persist(const Geom& g, const Workspace<T>& w, const HostConst& H, const Coef<T>& K, cudaStream_t st)
{
    const DevInfo di = device_info();
    const int nsm = di.sms, coop = di.coop;
    if (!coop || nsm < 1) return -100;
    if ((long long)g.ny * g.nz * ((g.nx + 63) / 64) >= (1LL << 31)) return -100;      // 32-bit task indices
    return (g.npad <= OMNI_PERSIST_SMALL_CELLS) ? launch_persist<T, 512, LOP>(g, w, H, K, nsm, st)
                                                : launch_persist<T, 1024, LOP>(g, w, H, K, nsm, st);
}

// SM-resident loop (omni_resident.cuh): the persistent loop with p in shared memory and r in registers for the whole
// inner solve.  Returns -100 if the grid does not fit the SMs or the device cannot co-schedule it.
// OMNI_RESIDENT_TMEM=0 keeps r and delta of the resident loop out of tensor memory (A / B measurements).
int resident_tmem_policy()
{
    static int v = -1;
    if (v < 0) {
        const char* e = getenv("OMNI_RESIDENT_TMEM");
        v = e ? atoi(e) : 1;                                  // 0: never, else wherever a thread has at most RES_NI rows
    }
    return v;
}


// The search walks every box of every candidate grid (1 - 2 ms of host time at 1024^2 or 128^3): its results are kept, keyed
// by what they depend on; the last few geometries of a process cover the solves it repeats.
bool resident_plan_auto(const Geom& g, int elem_size, int nsm, bool lop, ResidentPlan& pl)
{
    struct Entry { int nx, ny, nz, naxes, fix1, fix2, esz, nsm, lop, ok; ResidentPlan pl; };
    static std::mutex mu;
    static std::vector<Entry> cache;
    const Entry key = { g.nx, g.ny, g.nz, g.naxes, g.fix[1], g.fix[2], elem_size, nsm, lop ? 1 : 0, 0, ResidentPlan() };
    {
        std::lock_guard<std::mutex> lk(mu);
        for (const Entry& e : cache)
            if (e.nx == key.nx && e.ny == key.ny && e.nz == key.nz && e.naxes == key.naxes && e.fix1 == key.fix1 && e.fix2 == key.fix2 &&
                e.esz == key.esz && e.nsm == key.nsm && e.lop == key.lop) {
                pl = e.pl;
                return e.ok != 0;
            }
    }
    Entry e = key;
    e.ok = resident_plan(g, elem_size, nsm, lop, resident_tmem_policy() != 0, e.pl) ? 1 : 0;
    pl = e.pl;
    std::lock_guard<std::mutex> lk(mu);
    if (cache.size() >= 32) cache.erase(cache.begin());
    cache.push_back(e);
    return e.ok != 0;
}

template <typename T, bool LOP, int RM, bool UNI = true>
int launch_resident(const Geom& g, const Workspace<T>& w, const HostConst& H, const Coef<T>& K, const ResidentPlan& pl, cudaStream_t st)
{
    const int G = pl.gy * pl.gz;
    if (cudaFuncSetAttribute(resident_kernel<T, LOP, RM, UNI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem_bytes) != cudaSuccess) {
        cudaGetLastError();
        return -100;
    }
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, resident_kernel<T, LOP, RM, UNI>, RES_NT, pl.smem_bytes) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        return -100;
    }
    ResidentArgs<T> ra;
    PersistArgs<T>& a = ra.a;
    a.r = w.r; a.pbuf[0] = w.p0; a.pbuf[1] = w.p1; a.delta = w.delta; a.S = w.S; a.Pbuf[0] = w.P; a.Pbuf[1] = w.P1;
    a.link = w.link; a.wcode = w.wcode; a.flags = w.flags; a.K = K;
    for (int i = 0; i < 3; ++i) a.t[i] = H.F[i] / H.Atot;
    a.sc = w.sc; a.slots = w.slots;
    a.timeout_ns = barrier_timeout_ns();
    ra.gy = pl.gy; ra.gz = pl.gz; ra.ly = pl.ly; ra.lz = pl.lz; ra.zpad = pl.zpad; ra.pxs = pl.pxs; ra.dres = pl.dres; ra.qres = pl.qres; ra.rpt = pl.rpt; ra.wy = pl.wy; ra.wz = pl.wz;
    // the halo messages take the place of the two p buffers, which this loop does not use (carve: p1 follows p0); no
    // message of an earlier solve may carry a live epoch
    ra.xchg = (unsigned long long*)w.p0;
    CK(cudaMemsetAsync(w.p0, 0, (size_t)2 * (size_t)g.npad * sizeof(T), st));
    CK(cudaMemsetAsync(w.slots, 0, PERSIST_SLOT_BYTES, st));
    Geom gg = g;
    void* params[2] = { (void*)&gg, (void*)&ra };
    if (cudaLaunchCooperativeKernel((const void*)resident_kernel<T, LOP, RM, UNI>, dim3((unsigned)G), dim3(RES_NT), params, pl.smem_bytes, st) != cudaSuccess) {
        cudaGetLastError();
        return -100;
    }
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return OMNI_OK;
}

template <typename T, bool LOP>
int run_loop_resident(const Geom& g, const Workspace<T>& w, const HostConst& H, const Coef<T>& K, cudaStream_t st)
{
    const DevInfo di = device_info();
    if (!di.coop || di.sms < 1) return -100;
    if (g.npad >= (1LL << 31) || (long long)g.ny * g.nz * ((g.nx + 63) / 64) >= (1LL << 31)) return -100;
    ResidentPlan pl;
    if (!resident_plan_auto(g, (int)sizeof(T), di.sms < 148 ? di.sms : 148, LOP, pl)) return -100;     // relaxed slots: room for 148 CTAs
    if (pl.gy * pl.gz > 148 || pl.gy * pl.gz > RES_NT) return -100;          // relaxed slots: RES_SLOT_OFFSET
    if (pl.rtm) return pl.uni ? launch_resident<T, LOP, 3, true>(g, w, H, K, pl, st) : launch_resident<T, LOP, 3, false>(g, w, H, K, pl, st);
    if (!pl.rreg) return launch_resident<T, LOP, 0>(g, w, H, K, pl, st);
    static const int rmode = getenv("OMNI_RESIDENT_R") ? atoi(getenv("OMNI_RESIDENT_R")) : 2;
    if (rmode == 1 && pl.rpt <= RES_NI) return launch_resident<T, LOP, 1>(g, w, H, K, pl, st);
    return launch_resident<T, LOP, 2>(g, w, H, K, pl, st);
}

// Single-reduction CG for the fixed-point solve (omni_persist1.cuh): the persistent kernel with one grid barrier per
// iteration.  Four more vectors (double-buffered r, w, s and p) come from the pool.  -100: cannot be co-scheduled.
template <typename T, int NT>
int launch_persist1(const Geom& g, const Workspace<T>& w, const HostConst& H, const Coef<T>& K, int nsm, cudaStream_t st)
{
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, persist_cg1_kernel<T, NT>, NT, 0) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        return -100;
    }
    const size_t nb = align_up((size_t)g.npad * sizeof(T), 256);
    char* extra = nullptr;
    if (pool_alloc(&extra, 4 * nb, st) != cudaSuccess) { cudaGetLastError(); return OMNI_ERR_ALLOC; }
    CK(cudaMemsetAsync(extra, 0, 4 * nb, st));
    Persist1Args<T> A;
    PersistArgs<T>& a = A.base;
    a.r = w.r; a.pbuf[0] = w.p0; a.pbuf[1] = w.p1; a.delta = w.delta; a.S = w.S; a.Pbuf[0] = w.P; a.Pbuf[1] = w.P1;
    a.link = w.link; a.wcode = w.wcode; a.flags = w.flags; a.K = K;
    for (int i = 0; i < 3; ++i) a.t[i] = H.F[i] / H.Atot;
    a.sc = w.sc; a.slots = w.slots;
    a.timeout_ns = barrier_timeout_ns();
    A.rb[0] = w.r; A.rb[1] = (T*)extra;
    A.wb[0] = w.p0; A.wb[1] = w.p1;
    A.sb[0] = (T*)(extra + nb); A.sb[1] = (T*)(extra + 2 * nb);
    A.p = (T*)(extra + 3 * nb);
    const long long tasks = (long long)g.ny * g.nz * ((g.nx + 63) / 64);
    const int nw = NT / 32;
    long long G = (tasks + nw - 1) / nw;
    if (G > nsm) G = nsm;
    if (G > PERSIST_MAX_CTAS) G = PERSIST_MAX_CTAS;
    if (G < 1) G = 1;
    CK(cudaMemsetAsync(w.slots, 0, (size_t)8 * G * sizeof(double), st));
    Geom gg = g;
    void* params[2] = { (void*)&gg, (void*)&A };
    int rc = OMNI_OK;
    if (cudaLaunchCooperativeKernel((const void*)persist_cg1_kernel<T, NT>, dim3((unsigned)G), dim3(NT), params, 0, st) != cudaSuccess) {
        cudaGetLastError();
        rc = -100;
    } else {
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    cudaFreeAsync(extra, st);
    return rc;
}

template <typename T>
int run_loop_persist1(const Geom& g, const Workspace<T>& w, const HostConst& H, const Coef<T>& K, cudaStream_t st)
{
    const DevInfo di = device_info();
    if (!di.coop || di.sms < 1) return -100;
    if ((long long)g.ny * g.nz * ((g.nx + 63) / 64) >= (1LL << 31)) return -100;
    return (g.npad <= OMNI_PERSIST_SMALL_CELLS) ? launch_persist1<T, 512>(g, w, H, K, di.sms, st)
                                                : launch_persist1<T, 1024>(g, w, H, K, di.sms, st);
}

// loop selection: g_loop_mode 0 = automatic (SM-resident kernel where the grid fits the SMs, else the persistent kernel for grids up
// to OMNI_PERSIST_MAX_CELLS padded cells, CUDA graph above), 1 = host-driven, 2 = CUDA graph, 3 = persistent kernel,
// 4 = whole-solve tile loop kernel, 5 = SM-resident kernel
long long persist_max_cells()
{
    static long long v = -1;
    if (v < 0) {
        const char* e = getenv("OMNI_PERSIST_MAX_CELLS");
        v = e ? atoll(e) : OMNI_PERSIST_MAX_CELLS;
        if (v < 0) v = 0;
    }
    return v;
}

bool resident_enabled()
{
    static int v = -1;
    if (v < 0) {
        const char* e = getenv("OMNI_RESIDENT");
        v = (e && atoi(e) == 0) ? 0 : 1;
    }
    return v != 0;
}

long long loopk_max_cells()
{
    static long long v = -1;
    if (v < 0) {
        const char* e = getenv("OMNI_LOOPK_MAX_CELLS");
        v = e ? atoll(e) : OMNI_LOOPK_MAX_CELLS;
        if (v < 0) v = 0;
    }
    return v;
}

bool valid_common(int nx, int ny, int nz, double dx, double dy, double dz, double tol, int max_outer, int max_cg)
{
    if (nx < 1 || ny < 1 || nz < 1) return false;
    if (!(dx > 0.0) || !(dy > 0.0) || !std::isfinite(dx) || !std::isfinite(dy)) return false;
    if (nz > 1 && (!(dz > 0.0) || !std::isfinite(dz))) return false;
    if (!(tol >= 0.0) || !std::isfinite(tol) || max_outer < 0 || max_cg < 0) return false;
    return true;
}

template <typename T>
int solve_ws(int nx, int ny, int nz, double dx, double dy, double dz, const T* gx, const T* gy, const T* gz,
             const unsigned char* mask, T* P_out, double tol, int max_outer, int max_cg, void* ws, size_t ws_bytes,
             void* stream, omni_info* info, int batch = 0, const T* P_init = nullptr, int lop = 0, int pcg = 0)
{
    Geom g;
    if (!valid_common(nx, ny, batch ? 1 : nz, dx, dy, dz, tol, max_outer, max_cg) || !make_geom(nx, ny, nz, (int)sizeof(T), g, batch)) return OMNI_ERR_INVALID_ARG;
    if (!gx || !gy || (g.naxes == 3 && !gz) || !P_out || !ws) return OMNI_ERR_INVALID_ARG;
    if (((uintptr_t)ws & 255) != 0) return OMNI_ERR_INVALID_ARG;
    if (ws_bytes < carve<T>(g, nullptr, nullptr)) return OMNI_ERR_ALLOC;
    cudaStream_t st = (cudaStream_t)stream;
    Workspace<T> w;
    carve<T>(g, (char*)ws, &w);
    HostConst H;
    host_constants(g.naxes, dx, dy, dz, H);
    const Coef<T> K = make_coef<T>(H, dx, dy, dz, g);

    // omni_solve_pcg in fp32: an inner solve cannot resolve more than a few digits of its correction (the fp32 vectors
    // floor the recursive residual at ~1e-4 ||r0|| on 1000-cell-wide grids), so it hands back to the fp64 refinement
    // after two digits (reading R-P1)
    const double inner_rel = (pcg && sizeof(T) == 4) ? OMNI_PCG_INNER_REL_F32 : 0.0;
    const CallOpts opt = current_opts();
    init_scalars_kernel<<<1, 1, 0, st>>>(w.sc, tol, max_outer, max_cg, opt.hist, opt.hist_cap, opt.hist_k, inner_rel, opt.hist_p, opt.status);
    CK(cudaGetLastError());
    g_launches.fetch_add(1, std::memory_order_relaxed);
    int rc = setup_codes<T>(g, w, gx, gy, gz, mask, st);
    if (rc != OMNI_OK) return rc;
    rc = launch_source<T>(g, w, K, gx, gy, gz, st);
    if (rc != OMNI_OK) return rc;
    if (P_init) {       // first guess P^0 ("zero ... or any other arbitrary value"); 0 at missing cells
        const unsigned nbk = blocks_for(g.npad, 256);
        pad_copy_kernel<T, double><<<nbk, 256, 0, st>>>(g, P_init, w.P, 1, w.link);
        pad_copy_kernel<T, double><<<nbk, 256, 0, st>>>(g, P_init, w.P1, 1, w.link);
        CK(cudaGetLastError());
        g_launches.fetch_add(2, std::memory_order_relaxed);
    }

    int mode = opt.loop_mode;
    if (mode == 0) {
        // automatic: the SM-resident loop wherever p fits the SMs' shared memory (measured 1.1 - 2.2 x the persistent or
        // graph loop where r fits beside it, 1.2 - 1.35 x at 128^3 fp64 where r stays in L2), else by size as before
        ResidentPlan pl;
        const DevInfo di = device_info();
        const bool one_red = lop && opt.single_reduction;          // that option is the persistent loop's
        if (!one_red && !pcg && resident_enabled() && di.coop && resident_plan_auto(g, (int)sizeof(T), di.sms < 148 ? di.sms : 148, lop != 0, pl))
            mode = 5;
        else
            mode = (g.npad <= persist_max_cells()) ? 3 : (g.npad <= loopk_max_cells()) ? 4 : 2;
    }
    MgHier<T> mg;
    mg.mem = nullptr; mg.launches_per_cycle = 0;
    if (pcg) {
        // multigrid-preconditioned CG on L P = S: always the graph loop (its body holds the V-cycle's kernels)
        rc = mg_build<T>(g, w, H, mg, st);
        if (rc != OMNI_OK) return rc;
        rc = run_loop_graph<T, true>(g, w, H, K, st, &mg);
        cudaFreeAsync(mg.mem, st);                        // stream-ordered: after the graph has run
        if (rc != OMNI_OK) return rc;
        mode = -2;
    }
    // lop: the CG kernels apply L instead of M (omni_solve_direct); everything else -- K2, scalars, loop control -- is shared
    if (mode == 5) {
        rc = lop ? run_loop_resident<T, true>(g, w, H, K, st) : run_loop_resident<T, false>(g, w, H, K, st);
        if (rc == -100) mode = 3;
    }
    if (mode == 3) {
        // fixed-point solve with omni_options::single_reduction: the one-barrier-per-iteration kernel (L = L^T only)
        if (lop && opt.single_reduction) rc = run_loop_persist1<T>(g, w, H, K, st);
        else rc = lop ? run_loop_persist<T, true>(g, w, H, K, st) : run_loop_persist<T, false>(g, w, H, K, st);
        if (rc == -100) mode = 2;
    }
    if (mode == 4) {
        rc = lop ? run_loop_loopk<T, true>(g, w, H, K, st) : run_loop_loopk<T, false>(g, w, H, K, st);
        if (rc == -100) mode = 2;
    }
    if (mode == 1) rc = lop ? run_loop_host<T, true>(g, w, H, K, max_outer, max_cg, st) : run_loop_host<T, false>(g, w, H, K, max_outer, max_cg, st);
    else if (mode == 2) rc = lop ? run_loop_graph<T, true>(g, w, H, K, st) : run_loop_graph<T, false>(g, w, H, K, st);
    if (rc != OMNI_OK) return rc;

    if (rows_are_chunks(g, P_out, opt.P64, (const T*)nullptr, (const unsigned char*)nullptr))
        finalize4_kernel<T><<<setup_grid(g), dim3(SETUP_BX, SETUP_BY), 0, st>>>(g, w.P, w.P1, w.sc, w.link, P_out, opt.P64);
    else
        finalize_kernel<T><<<blocks_for((long long)nx * ny * nz, 256), 256, 0, st>>>(g, w.P, w.P1, w.sc, w.link, P_out, opt.P64);
    CK(cudaGetLastError());
    g_launches.fetch_add(1, std::memory_order_relaxed);

    if (info) {
        Scalars h;
        CK(cudaMemcpyAsync(&h, w.sc, sizeof(Scalars), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        info->outer_iters = h.n;
        info->cg_iters_total = h.cg_total;
        info->norm_S = std::sqrt(h.normS2);
        info->eps_R_final = (h.normS2 > 0.0) ? std::sqrt(h.epsR2 / h.normS2) : 0.0;
        info->status = h.status;
        // kernels launched by the device-side loop of the graph, from its own counters: K2 + flush per outer check,
        // K3 + K4 per CG iteration
        if (mode == 2) g_launches.fetch_add((long long)(h.normS2 > 0.0 ? 2 * h.n + 1 : 0) + 2 * h.cg_total, std::memory_order_relaxed);
        if (mode == -2) g_launches.fetch_add((long long)(h.normS2 > 0.0 ? 2 * h.n + 1 : 0) + (2 + mg.launches_per_cycle) * h.cg_total, std::memory_order_relaxed);
        return h.status;
    }
    return OMNI_OK;
}

template <typename T>
int solve_alloc(int nx, int ny, int nz, double dx, double dy, double dz, const T* gx, const T* gy, const T* gz,
                const unsigned char* mask, T* P_out, double tol, int max_outer, int max_cg, void* stream, omni_info* info,
                int batch = 0, const T* P_init = nullptr, int lop = 0, int pcg = 0)
{
    Geom g;
    if (!valid_common(nx, ny, batch ? 1 : nz, dx, dy, dz, tol, max_outer, max_cg) || !make_geom(nx, ny, nz, (int)sizeof(T), g, batch)) return OMNI_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = carve<T>(g, nullptr, nullptr);
    void* ws = nullptr;
    if (pool_alloc(&ws, bytes, st) != cudaSuccess) { cudaGetLastError(); return OMNI_ERR_ALLOC; }
    int rc = solve_ws<T>(nx, ny, nz, dx, dy, dz, gx, gy, gz, mask, P_out, tol, max_outer, max_cg, ws, bytes, stream, info,
                         batch, P_init, lop, pcg);
    cudaFreeAsync(ws, st);
    return rc;
}

// Cascadic first guess for the fixed-point solve: solve L P = S on grids coarsened by 2 (restrict_kernel), coarsest
// first, and hand each level's pressure to the next finer one as its first guess (prolong_kernel).  The coarse levels
// only produce guesses: their status is not examined, and the answer is whatever the finest-level solve, with the
// caller's tol and caps, converges to.
template <typename T>
int solve_cascade(int nx, int ny, int nz, double dx, double dy, double dz, const T* gx, const T* gy, const T* gz,
                  const unsigned char* mask, T* P_out, double tol, int max_outer, int max_cg, int levels, void* stream,
                  omni_info* info)
{
    Geom g0;
    if (!valid_common(nx, ny, nz, dx, dy, dz, tol, max_outer, max_cg) || levels < 0 || !make_geom(nx, ny, nz, (int)sizeof(T), g0))
        return OMNI_ERR_INVALID_ARG;
    if (!gx || !gy || (nz > 1 && !gz) || !P_out) return OMNI_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    struct Level { int nx, ny, nz, fx, fy, fz; double dx, dy, dz; const T *gx, *gy, *gz; const unsigned char* mask; T* P; void* own; };
    std::vector<Level> lv;
    lv.push_back(Level{ nx, ny, nz, 1, 1, 1, dx, dy, dz, gx, gy, gz, mask, P_out, nullptr });
    const int ncomp = (nz > 1) ? 3 : 2;
    int rc = OMNI_OK;
    for (int l = 1; l <= levels && rc == OMNI_OK; ++l) {
        const Level f = lv.back();
        const int fx = f.nx > 1 ? 2 : 1, fy = f.ny > 1 ? 2 : 1, fz = f.nz > 1 ? 2 : 1;
        const int cx = (f.nx + fx - 1) / fx, cy = (f.ny + fy - 1) / fy, cz = (f.nz + fz - 1) / fz;
        // stop where a coarser grid is too small to be worth a solve (or would lose an axis of a 3D problem)
        if ((fx == 2 && cx < 8) || (fy == 2 && cy < 8) || (fz == 2 && cz < 8)) break;
        const size_t n = (size_t)cx * cy * cz;
        const size_t bytes = align_up((ncomp + 1) * n * sizeof(T), 256) + align_up(n, 256);
        void* own = nullptr;
        if (pool_alloc(&own, bytes, st) != cudaSuccess) { cudaGetLastError(); rc = OMNI_ERR_ALLOC; break; }
        T* b = (T*)own;
        unsigned char* cm = (unsigned char*)own + align_up((ncomp + 1) * n * sizeof(T), 256);
        Level c{ cx, cy, cz, fx, fy, fz, f.dx * fx, f.dy * fy, f.dz * fz, b, b + n, ncomp == 3 ? b + 2 * n : nullptr, cm,
                 b + (size_t)ncomp * n, own };
        restrict_kernel<T><<<blocks_for((long long)n, 256), 256, 0, st>>>(f.nx, f.ny, f.nz, fx, fy, fz, cx, cy, cz, ncomp, f.gx, f.gy,
                                                                         f.gz, f.mask, b, b + n, ncomp == 3 ? b + 2 * n : nullptr, cm);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        lv.push_back(c);
        if (cudaGetLastError() != cudaSuccess) rc = OMNI_ERR_CUDA;
    }
    for (int l = (int)lv.size() - 1; l >= 0 && rc >= 0; --l) {
        const Level& L = lv[l];
        T* pinit = nullptr;
        if (l + 1 < (int)lv.size()) {
            const Level& C = lv[l + 1];
            const size_t n = (size_t)L.nx * L.ny * L.nz;
            if (pool_alloc((void**)&pinit, n * sizeof(T), st) != cudaSuccess) { cudaGetLastError(); rc = OMNI_ERR_ALLOC; break; }
            prolong_kernel<T><<<blocks_for((long long)n, 256), 256, 0, st>>>(L.nx, L.ny, L.nz, C.fx, C.fy, C.fz, C.nx, C.ny, C.P, pinit);
            g_launches.fetch_add(1, std::memory_order_relaxed);
            if (cudaGetLastError() != cudaSuccess) { cudaFreeAsync(pinit, st); rc = OMNI_ERR_CUDA; break; }
        }
        const int r = solve_alloc<T>(L.nx, L.ny, L.nz, L.dx, L.dy, L.dz, L.gx, L.gy, L.gz, L.mask, L.P, tol, max_outer, max_cg, stream,
                                     l == 0 ? info : nullptr, 0, pinit, 1);
        if (pinit) cudaFreeAsync(pinit, st);
        if (l == 0 || r < 0) rc = r;
    }
    for (auto& L : lv)
        if (L.own) cudaFreeAsync(L.own, st);
    return rc;
}

// NEXT-4: the upstream step g = f(u) (Eq. 1 :23) on device arrays in the caller's layout
template <typename T>
int velocity_source(int nx, int ny, int nz, double dx, double dy, double dz, const T* u, const T* v, const T* w,
                    const T* atx, const T* aty, const T* atz, const unsigned char* mask, double rho, double mu,
                    T* gx, T* gy, T* gz, void* stream)
{
    if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0.0) || !(dy > 0.0) || (nz > 1 && !(dz > 0.0))) return OMNI_ERR_INVALID_ARG;
    if (!std::isfinite(rho) || !std::isfinite(mu)) return OMNI_ERR_INVALID_ARG;
    const int ncomp = (nz > 1) ? 3 : 2;
    if (!u || !v || !gx || !gy || (ncomp == 3 && (!w || !gz))) return OMNI_ERR_INVALID_ARG;
    if ((atx == nullptr) != (aty == nullptr) || (ncomp == 3 && (atx == nullptr) != (atz == nullptr))) return OMNI_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const long long n = (long long)nx * ny * nz;
    velocity_source_kernel<T><<<blocks_for(n, 256), 256, 0, st>>>(
        nx, ny, nz, ncomp, (T)(1.0 / (dx * dx)), (T)(1.0 / (dy * dy)), (T)(ncomp == 3 ? 1.0 / (dz * dz) : 0.0),
        (T)(0.5 / dx), (T)(0.5 / dy), (T)(ncomp == 3 ? 0.5 / dz : 0.0), (T)rho, (T)mu, u, v, w, atx, aty, atz, mask, gx, gy, gz);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    CK(cudaGetLastError());
    return OMNI_OK;
}

// NEXT-4: RANS source fields (Eq. 42 :507; Eq. 43-44 :540-545) on device arrays in the caller's layout
template <typename T>
int rans_source(bool compressible, int nx, int ny, int nz, double dx, double dy, double dz, const T* u, const T* v, const T* w,
                const T* const* stress, const unsigned char* mask, double rho, double gamma, double mach_inf, double v_inf,
                double rgas_t_inf, T* gx, T* gy, T* gz, void* stream)
{
    if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0.0) || !(dy > 0.0) || (nz > 1 && !(dz > 0.0))) return OMNI_ERR_INVALID_ARG;
    const int nd = (nz > 1) ? 3 : 2, nR = (nd == 2) ? 3 : 6;
    if (!u || !v || !gx || !gy || (nd == 3 && (!w || !gz))) return OMNI_ERR_INVALID_ARG;
    int given = 0;
    if (stress)
        for (int m = 0; m < nR; ++m) given += (stress[m] != nullptr);
    if (given != 0 && given != nR) return OMNI_ERR_INVALID_ARG;
    if (compressible) {
        if (!(gamma > 1.0) || !std::isfinite(gamma) || !std::isfinite(mach_inf) || !(v_inf > 0.0) || !std::isfinite(v_inf) ||
            !(rgas_t_inf > 0.0) || !std::isfinite(rgas_t_inf))
            return OMNI_ERR_INVALID_ARG;
    } else if (!std::isfinite(rho)) {
        return OMNI_ERR_INVALID_ARG;
    }
    RansArgs<T> a;
    a.u[0] = u; a.u[1] = v; a.u[2] = (nd == 3) ? w : nullptr;
    for (int m = 0; m < 6; ++m) a.R[m] = (given && m < nR) ? stress[m] : nullptr;
    a.mask = mask;
    a.g[0] = gx; a.g[1] = gy; a.g[2] = (nd == 3) ? gz : nullptr;
    a.ih[0] = (T)(0.5 / dx); a.ih[1] = (T)(0.5 / dy); a.ih[2] = (T)(nd == 3 ? 0.5 / dz : 0.0);
    a.rho = (T)rho;
    a.cth = (T)(compressible ? 0.5 * (gamma - 1.0) * mach_inf * mach_inf : 0.0);
    a.inv_v2 = (T)(compressible ? 1.0 / (v_inf * v_inf) : 0.0);
    a.rt_inf = (T)rgas_t_inf;
    a.has_R = given ? 1 : 0;
    cudaStream_t st = (cudaStream_t)stream;
    const long long n = (long long)nx * ny * nz;
    if (compressible) rans_source_kernel<T, true><<<blocks_for(n, 256), 256, 0, st>>>(nx, ny, nz, nd, a);
    else rans_source_kernel<T, false><<<blocks_for(n, 256), 256, 0, st>>>(nx, ny, nz, nd, a);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    CK(cudaGetLastError());
    return OMNI_OK;
}

// ------------------------------------------------------------------------------------------------ z-slab sharding (omni_slab.cuh)
template <typename T>
struct SlabRank {
    int rank, z0, z1, zlo, zhi;
    Geom g; Workspace<T> w; void* ws; TmaSet maps;
    const T *gx, *gy, *gz; const uint8_t* mask; T* P_out;
};

// Halo exchange of one array: every rank's planes just outside its owned range receive the neighbour's outermost owned
// plane.  comm == nullptr: all ranks are local (plane copies on the stream); else one local rank and NCCL.
template <typename T, typename U, typename F>
int slab_exchange(std::vector<SlabRank<T>>& R, int nranks, void* comm, F&& base, cudaStream_t st)
{
    if (!comm) {
        for (int s = 0; s + 1 < (int)R.size(); ++s) {
            SlabRank<T>&lo = R[s], &hi = R[s + 1];
            U* a = base(lo); U* b = base(hi);
            const size_t bytes = (size_t)lo.g.pplane * sizeof(U);
            // lo's first plane above its range <- hi's first owned plane; hi's last plane below its range <- lo's last owned one
            CK(cudaMemcpyAsync(a + (size_t)lo.g.kz1 * lo.g.pplane, b + (size_t)hi.g.kz0 * hi.g.pplane, bytes, cudaMemcpyDeviceToDevice, st));
            CK(cudaMemcpyAsync(b + (size_t)(hi.g.kz0 - 1) * hi.g.pplane, a + (size_t)(lo.g.kz1 - 1) * lo.g.pplane, bytes, cudaMemcpyDeviceToDevice, st));
        }
        return OMNI_OK;
    }
    const NcclApi& N = nccl_api();
    SlabRank<T>& r = R[0];
    U* a = base(r);
    const size_t bytes = (size_t)r.g.pplane * sizeof(U);
    if (N.GroupStart() != 0) return OMNI_ERR_CUDA;
    int bad = 0;
    if (r.rank > 0) {
        bad |= N.Send(a + (size_t)r.g.kz0 * r.g.pplane, bytes, NcclApi::Int8, r.rank - 1, comm, st);
        bad |= N.Recv(a + (size_t)(r.g.kz0 - 1) * r.g.pplane, bytes, NcclApi::Int8, r.rank - 1, comm, st);
    }
    if (r.rank + 1 < nranks) {
        bad |= N.Send(a + (size_t)(r.g.kz1 - 1) * r.g.pplane, bytes, NcclApi::Int8, r.rank + 1, comm, st);
        bad |= N.Recv(a + (size_t)r.g.kz1 * r.g.pplane, bytes, NcclApi::Int8, r.rank + 1, comm, st);
    }
    bad |= N.GroupEnd();
    return bad ? OMNI_ERR_CUDA : OMNI_OK;
}

// sum of Scalars::red_out[0..n) over all ranks, left in every rank's red_out
template <typename T>
int slab_allreduce(std::vector<SlabRank<T>>& R, void* comm, Scalars* const* d_scs, int n, cudaStream_t st)
{
    if (!comm) {
        if (R.size() > 1) {
            slab_sum_kernel<<<1, 32, 0, st>>>(d_scs, (int)R.size(), n);
            g_launches.fetch_add(1, std::memory_order_relaxed);
            CK(cudaGetLastError());
        }
        return OMNI_OK;
    }
    double* p = R[0].w.sc->red_out;            // device address of the member
    return nccl_api().AllReduce(p, p, (size_t)n, NcclApi::Float64, NcclApi::Sum, comm, st) == 0 ? OMNI_OK : OMNI_ERR_CUDA;
}

// Alg. 1 (lop = 0) or CG on L P = S (lop = 1) on z-slabs; host-driven loop (one synchronisation per outer iteration and
// per 16 CG iterations, like loop mode 1).  Local windows: d_g*, d_mask, d_P_out hold the planes [zlo, zhi) of each
// local rank (omni_slab_plan); P_out is written on the whole window, the owned planes are the result.
template <typename T>
int solve_slab(int nx, int ny, int nz, double dx, double dy, double dz, int nlocal, const int* ranks, const T* const* gx,
               const T* const* gy, const T* const* gz, const unsigned char* const* mask, T* const* P_out, double tol,
               int max_outer, int max_cg, int lop, int nranks, void* comm, void* stream, omni_info* info)
{
    if (!valid_common(nx, ny, nz, dx, dy, dz, tol, max_outer, max_cg) || nz < 2 || nranks < 1 || nlocal < 1 || !ranks || !gx || !gy ||
        !gz || !P_out)
        return OMNI_ERR_INVALID_ARG;
    if (comm ? (nlocal != 1 || !nccl_api().ok) : (nlocal != nranks)) return OMNI_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<SlabRank<T>> R((size_t)nlocal);
    HostConst H;
    host_constants(3, dx, dy, dz, H);
    int rc = OMNI_OK;
    Scalars** d_scs = nullptr;
    auto cleanup = [&]() {
        for (auto& r : R)
            if (r.ws) cudaFreeAsync(r.ws, st);
        if (d_scs) cudaFreeAsync(d_scs, st);
    };
    for (auto& r : R) r.ws = nullptr;
    for (int i = 0; i < nlocal && rc == OMNI_OK; ++i) {
        SlabRank<T>& r = R[(size_t)i];
        r.rank = ranks[i];
        if ((!comm && r.rank != i) || !slab_plan(nz, nranks, r.rank, r.z0, r.z1, r.zlo, r.zhi) || !gx[i] || !gy[i] || !gz[i] || !P_out[i] ||
            !make_geom(nx, ny, r.zhi - r.zlo, (int)sizeof(T), r.g)) { rc = OMNI_ERR_INVALID_ARG; break; }
        r.g.kz0 = r.z0 - r.zlo; r.g.kz1 = r.z1 - r.zlo;
        r.gx = gx[i]; r.gy = gy[i]; r.gz = gz[i]; r.mask = mask ? mask[i] : nullptr; r.P_out = P_out[i];
        const size_t bytes = carve<T>(r.g, nullptr, nullptr);
        if (pool_alloc(&r.ws, bytes, st) != cudaSuccess) { cudaGetLastError(); r.ws = nullptr; rc = OMNI_ERR_ALLOC; break; }
        carve<T>(r.g, (char*)r.ws, &r.w);
    }
    if (rc != OMNI_OK) { cleanup(); return rc; }
    std::vector<Scalars*> h_scs;
    for (auto& r : R) h_scs.push_back(r.w.sc);
    if (pool_alloc((void**)&d_scs, sizeof(Scalars*) * R.size(), st) != cudaSuccess) { cudaGetLastError(); d_scs = nullptr; cleanup(); return OMNI_ERR_ALLOC; }
    cudaMemcpyAsync(d_scs, h_scs.data(), sizeof(Scalars*) * R.size(), cudaMemcpyHostToDevice, st);
    cudaStreamSynchronize(st);            // h_scs is a host temporary

    CondHandles ch{ 0, 0, 0 };
    auto each = [&](auto&& fn) { for (auto& r : R) { if (rc == OMNI_OK) { const int e = fn(r); if (e != OMNI_OK) rc = e; } } };
    // setup per rank: scalars (deferred finalize), validity / codes / source on the window, tensor maps
    each([&](SlabRank<T>& r) {
        const Coef<T> K = make_coef<T>(H, dx, dy, dz, r.g);
        init_scalars_kernel<<<1, 1, 0, st>>>(r.w.sc, tol, max_outer, max_cg, nullptr, 0, nullptr, 0.0, nullptr, nullptr, 1);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        int e = setup_codes<T>(r.g, r.w, r.gx, r.gy, r.gz, r.mask, st);
        if (e == OMNI_OK) e = launch_source<T>(r.g, r.w, K, r.gx, r.gy, r.gz, st);
        if (e == OMNI_OK && !make_tma_set<T>(r.g, r.w, r.maps)) e = OMNI_ERR_CUDA;
        return e;
    });
    if (rc == OMNI_OK) rc = slab_allreduce<T>(R, comm, d_scs, 1, st);
    each([&](SlabRank<T>& r) { source_finalize_kernel<<<1, 1, 0, st>>>(r.w.sc); g_launches.fetch_add(1, std::memory_order_relaxed); return OMNI_OK; });

    auto launch_fin = [&](auto op_tag, SlabRank<T>& r, const auto& args) {
        using Op = typename decltype(op_tag)::type;
        op_finalize_kernel<Op><<<1, 1, 0, st>>>(args);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        return cudaGetLastError() == cudaSuccess ? OMNI_OK : OMNI_ERR_CUDA;
    };
    Scalars h;
    memset(&h, 0, sizeof(h));
    h.outer_go = 1;
    auto read_scalars = [&]() {
        if (cudaMemcpyAsync(&h, R[0].w.sc, sizeof(Scalars), cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess)
            rc = OMNI_ERR_CUDA;
    };
    if (rc == OMNI_OK) read_scalars();
    for (long long it = 0; it <= (long long)max_outer && rc == OMNI_OK && h.outer_go; ++it) {
        const int par = h.n & 1;                   // K2 reads Pbuf[par], writes Pbuf[par ^ 1]
        // K2: halo planes of delta first (the correction of the last inner solve), then the fold + residual
        if (it > 0) rc = slab_exchange<T, T>(R, nranks, comm, [](SlabRank<T>& r) { return r.w.delta; }, st);
        each([&](SlabRank<T>& r) { return launch_tma<K2<T>>(r.g, k2_args<T>(r.g, r.w, H, ch, 1), r.maps, st) == cudaSuccess ? OMNI_OK : OMNI_ERR_CUDA; });
        if (rc == OMNI_OK) rc = slab_allreduce<T>(R, comm, d_scs, 4, st);
        each([&](SlabRank<T>& r) { return launch_fin(std::common_type<K2<T>>{}, r, k2_args<T>(r.g, r.w, H, ch, 1)); });
        if (rc == OMNI_OK) rc = slab_exchange<T, double>(R, nranks, comm, [par](SlabRank<T>& r) { return par ? r.w.P : r.w.P1; }, st);
        if (rc == OMNI_OK) rc = slab_exchange<T, T>(R, nranks, comm, [](SlabRank<T>& r) { return r.w.r; }, st);
        if (rc == OMNI_OK) read_scalars();
        if (rc != OMNI_OK || !h.outer_go) break;
        // inner CG; the device decides when it ends (kernels of a finished loop return at once)
        int k = 0;
        while (k < max_cg && rc == OMNI_OK && h.inner_go) {
            const int batch = (max_cg - k < 16) ? (max_cg - k) : 16;
            for (int c = 0; c < batch && rc == OMNI_OK; ++c, ++k) {
                const int pn = (k & 1) ^ 1;                 // K3 writes pbuf[pn]
                each([&](SlabRank<T>& r) {
                    const Coef<T> K = make_coef<T>(H, dx, dy, dz, r.g);
                    cudaError_t e = lop ? launch_tma<K3<T, true>>(r.g, k3_args<T, true>(r.w, K, ch), r.maps, st)
                                        : launch_tma<K3<T, false>>(r.g, k3_args<T, false>(r.w, K, ch), r.maps, st);
                    return e == cudaSuccess ? OMNI_OK : OMNI_ERR_CUDA;
                });
                if (rc == OMNI_OK) rc = slab_allreduce<T>(R, comm, d_scs, 1, st);
                each([&](SlabRank<T>& r) {
                    const Coef<T> K = make_coef<T>(H, dx, dy, dz, r.g);
                    return lop ? launch_fin(std::common_type<K3<T, true>>{}, r, k3_args<T, true>(r.w, K, ch))
                               : launch_fin(std::common_type<K3<T, false>>{}, r, k3_args<T, false>(r.w, K, ch));
                });
                if (rc == OMNI_OK) rc = slab_exchange<T, T>(R, nranks, comm, [pn](SlabRank<T>& r) { return pn ? r.w.p1 : r.w.p0; }, st);
                each([&](SlabRank<T>& r) {
                    const Coef<T> K = make_coef<T>(H, dx, dy, dz, r.g);
                    cudaError_t e = lop ? launch_tma<K4<T, true>>(r.g, k4_args<T, true>(r.w, K, ch), r.maps, st)
                                        : launch_tma<K4<T, false>>(r.g, k4_args<T, false>(r.w, K, ch), r.maps, st);
                    return e == cudaSuccess ? OMNI_OK : OMNI_ERR_CUDA;
                });
                if (rc == OMNI_OK) rc = slab_allreduce<T>(R, comm, d_scs, 1, st);
                each([&](SlabRank<T>& r) {
                    const Coef<T> K = make_coef<T>(H, dx, dy, dz, r.g);
                    return lop ? launch_fin(std::common_type<K4<T, true>>{}, r, k4_args<T, true>(r.w, K, ch))
                               : launch_fin(std::common_type<K4<T, false>>{}, r, k4_args<T, false>(r.w, K, ch));
                });
                if (rc == OMNI_OK) rc = slab_exchange<T, T>(R, nranks, comm, [](SlabRank<T>& r) { return r.w.r; }, st);
            }
            if (rc == OMNI_OK) read_scalars();
        }
        each([&](SlabRank<T>& r) { return launch_flush<T>(r.g, r.w, st) == cudaSuccess ? OMNI_OK : OMNI_ERR_CUDA; });
    }
    each([&](SlabRank<T>& r) {
        finalize_kernel<T><<<blocks_for((long long)nx * ny * r.g.nz, 256), 256, 0, st>>>(r.g, r.w.P, r.w.P1, r.w.sc, r.w.link, r.P_out, nullptr);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        return cudaGetLastError() == cudaSuccess ? OMNI_OK : OMNI_ERR_CUDA;
    });
    if (rc == OMNI_OK) read_scalars();
    if (rc == OMNI_OK && info) {
        info->outer_iters = h.n; info->cg_iters_total = h.cg_total; info->norm_S = std::sqrt(h.normS2);
        info->eps_R_final = (h.normS2 > 0.0) ? std::sqrt(h.epsR2 / h.normS2) : 0.0;
        info->status = h.status;
    }
    const int status = h.status;
    cleanup();
    if (rc == OMNI_ERR_CUDA) cudaGetLastError();
    return rc == OMNI_OK ? status : rc;
}

template <typename T>
int solve_host(int nx, int ny, int nz, double dx, double dy, double dz, const T* gx, const T* gy, const T* gz,
               const unsigned char* mask, T* P_out, double tol, int max_outer, int max_cg, void* stream, omni_info* info)
{
    Geom g;
    if (!valid_common(nx, ny, nz, dx, dy, dz, tol, max_outer, max_cg) || !make_geom(nx, ny, nz, (int)sizeof(T), g)) return OMNI_ERR_INVALID_ARG;
    if (!gx || !gy || (nz > 1 && !gz) || !P_out) return OMNI_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)nx * ny * nz;
    const int ncomp = (nz > 1) ? 3 : 2;
    T* dbuf = nullptr;
    uint8_t* dmask = nullptr;
    if (pool_alloc((void**)&dbuf, (ncomp + 1) * n * sizeof(T), st) != cudaSuccess) { cudaGetLastError(); return OMNI_ERR_ALLOC; }
    if (mask && pool_alloc((void**)&dmask, n, st) != cudaSuccess) { cudaGetLastError(); cudaFreeAsync(dbuf, st); return OMNI_ERR_ALLOC; }
    int rc = OMNI_ERR_CUDA;
    omni_info local;
    do {
        if (cudaMemcpyAsync(dbuf, gx, n * sizeof(T), cudaMemcpyHostToDevice, st) != cudaSuccess) break;
        if (cudaMemcpyAsync(dbuf + n, gy, n * sizeof(T), cudaMemcpyHostToDevice, st) != cudaSuccess) break;
        if (ncomp == 3 && cudaMemcpyAsync(dbuf + 2 * n, gz, n * sizeof(T), cudaMemcpyHostToDevice, st) != cudaSuccess) break;
        if (mask && cudaMemcpyAsync(dmask, mask, n, cudaMemcpyHostToDevice, st) != cudaSuccess) break;
        T* dP = dbuf + (size_t)ncomp * n;
        rc = solve_alloc<T>(nx, ny, nz, dx, dy, dz, dbuf, dbuf + n, ncomp == 3 ? dbuf + 2 * n : nullptr, dmask, dP, tol,
                            max_outer, max_cg, stream, &local);
        if (rc < 0) break;
        if (cudaMemcpyAsync(P_out, dP, n * sizeof(T), cudaMemcpyDeviceToHost, st) != cudaSuccess) { rc = OMNI_ERR_CUDA; break; }
        if (cudaStreamSynchronize(st) != cudaSuccess) { rc = OMNI_ERR_CUDA; break; }
        if (info) *info = local;
    } while (0);
    cudaFreeAsync(dbuf, st);
    if (dmask) cudaFreeAsync(dmask, st);
    if (rc == OMNI_ERR_CUDA) cudaGetLastError();
    return rc;
}

// ------------------------------------------------------------------------------------------------ step entry points

template <typename T>
struct StepCtx {
    Geom g; Workspace<T> w; HostConst H; Coef<T> K; void* ws; cudaStream_t st;
};

template <typename T>
int step_begin(StepCtx<T>& c, int nx, int ny, int nz, double dx, double dy, double dz, const T* gx, const T* gy,
               const T* gz, const unsigned char* mask, void* stream)
{
    if (!valid_common(nx, ny, nz, dx, dy, dz, 0.0, 0, 0) || !make_geom(nx, ny, nz, (int)sizeof(T), c.g)) return OMNI_ERR_INVALID_ARG;
    c.st = (cudaStream_t)stream;
    const size_t bytes = carve<T>(c.g, nullptr, nullptr);
    c.ws = nullptr;
    if (pool_alloc(&c.ws, bytes, c.st) != cudaSuccess) { cudaGetLastError(); return OMNI_ERR_ALLOC; }
    carve<T>(c.g, (char*)c.ws, &c.w);
    host_constants(c.g.naxes, dx, dy, dz, c.H);
    c.K = make_coef<T>(c.H, dx, dy, dz, c.g);
    init_scalars_kernel<<<1, 1, 0, c.st>>>(c.w.sc, 0.0, 0, 0);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    int rc = setup_codes<T>(c.g, c.w, gx, gy, gz, mask, c.st);
    return rc;
}

template <typename T>
int step_end(StepCtx<T>& c, int rc, Scalars* h)
{
    if (rc == OMNI_OK && h) {
        if (cudaMemcpyAsync(h, c.w.sc, sizeof(Scalars), cudaMemcpyDeviceToHost, c.st) != cudaSuccess) rc = OMNI_ERR_CUDA;
    }
    if (cudaStreamSynchronize(c.st) != cudaSuccess) rc = OMNI_ERR_CUDA;
    if (c.ws) cudaFreeAsync(c.ws, c.st);
    if (rc == OMNI_ERR_CUDA) cudaGetLastError();
    return rc;
}

template <typename T>
int source_step(int nx, int ny, int nz, double dx, double dy, double dz, const T* gx, const T* gy, const T* gz,
                const unsigned char* mask, T* S_out, double* norm_S, void* stream)
{
    if (!gx || !gy || (nz > 1 && !gz) || !S_out) return OMNI_ERR_INVALID_ARG;
    StepCtx<T> c;
    int rc = step_begin<T>(c, nx, ny, nz, dx, dy, dz, gx, gy, gz, mask, stream);
    if (rc == OMNI_ERR_INVALID_ARG || rc == OMNI_ERR_ALLOC) return rc;
    Scalars h;
    if (rc == OMNI_OK) rc = launch_source<T>(c.g, c.w, c.K, gx, gy, gz, c.st);
    if (rc == OMNI_OK) {
        pad_copy_kernel<T, T><<<blocks_for(c.g.npad, 256), 256, 0, c.st>>>(c.g, c.w.S, S_out, 0, c.w.link);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        if (cudaGetLastError() != cudaSuccess) rc = OMNI_ERR_CUDA;
    }
    rc = step_end<T>(c, rc, &h);
    if (rc == OMNI_OK && norm_S) *norm_S = std::sqrt(h.normS2);
    return rc;
}

__global__ void force_go_kernel(Scalars* sc, double alpha)
{
    sc->inner_go = 1; sc->outer_go = 1; sc->k = 0; sc->alpha = alpha; sc->beta = 0.0;
}

template <typename T>
int apply_M_step(int nx, int ny, int nz, double dx, double dy, double dz, const unsigned char* mask, const T* p, T* q,
                 double* pq, void* stream)
{
    if (!p || !q) return OMNI_ERR_INVALID_ARG;
    StepCtx<T> c;
    int rc = step_begin<T>(c, nx, ny, nz, dx, dy, dz, (const T*)nullptr, (const T*)nullptr, (const T*)nullptr, mask, stream);
    if (rc == OMNI_ERR_INVALID_ARG || rc == OMNI_ERR_ALLOC) return rc;
    Scalars h;
    if (rc == OMNI_OK) {
        const unsigned nb = blocks_for(c.g.npad, 256);
        pad_copy_kernel<T, T><<<nb, 256, 0, c.st>>>(c.g, p, c.w.p0, 1, c.w.link);
        force_go_kernel<<<1, 1, 0, c.st>>>(c.w.sc, 0.0);
        CondHandles ch{ 0, 0, 0 };
        auto a4 = k4_args<T>(c.w, c.K, ch);
        a4.p_fixed = 0;
        a4.q_out = c.w.r;
        TmaSet maps;
        cudaError_t e = make_tma_set<T>(c.g, c.w, maps) ? launch_tma<K4<T>>(c.g, a4, maps, c.st) : cudaErrorUnknown;
        pad_copy_kernel<T, T><<<nb, 256, 0, c.st>>>(c.g, c.w.r, q, 0, c.w.link);
        g_launches.fetch_add(3, std::memory_order_relaxed);
        if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = OMNI_ERR_CUDA;
    }
    rc = step_end<T>(c, rc, &h);
    if (rc == OMNI_OK && pq) *pq = h.gamma;
    return rc;
}

template <typename T>
int residual_step(int nx, int ny, int nz, double dx, double dy, double dz, const T* gx, const T* gy, const T* gz,
                  const unsigned char* mask, const double* P, T* r_out, double* eps_R, void* stream)
{
    if (!gx || !gy || (nz > 1 && !gz) || !P || !r_out) return OMNI_ERR_INVALID_ARG;
    StepCtx<T> c;
    int rc = step_begin<T>(c, nx, ny, nz, dx, dy, dz, gx, gy, gz, mask, stream);
    if (rc == OMNI_ERR_INVALID_ARG || rc == OMNI_ERR_ALLOC) return rc;
    Scalars h;
    if (rc == OMNI_OK) rc = launch_source<T>(c.g, c.w, c.K, gx, gy, gz, c.st);
    if (rc == OMNI_OK) {
        const unsigned nb = blocks_for(c.g.npad, 256);
        pad_copy_kernel<double, double><<<nb, 256, 0, c.st>>>(c.g, P, c.w.P, 1, c.w.link);
        force_go_kernel<<<1, 1, 0, c.st>>>(c.w.sc, 0.0);
        CondHandles ch{ 0, 0, 0 };
        TmaSet maps;
        cudaError_t e = make_tma_set<T>(c.g, c.w, maps) ? launch_tma<K2<T>>(c.g, k2_args<T>(c.g, c.w, c.H, ch, 0), maps, c.st) : cudaErrorUnknown;
        pad_copy_kernel<T, T><<<nb, 256, 0, c.st>>>(c.g, c.w.r, r_out, 0, c.w.link);
        g_launches.fetch_add(3, std::memory_order_relaxed);
        if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = OMNI_ERR_CUDA;
    }
    rc = step_end<T>(c, rc, &h);
    if (rc == OMNI_OK && eps_R) *eps_R = (h.normS2 > 0.0) ? std::sqrt(h.epsR2 / h.normS2) : 0.0;
    return rc;
}

}  // namespace

// ================================================================================================ C ABI

extern "C" {

int omni_solve_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_gx, const double* d_gy,
                   const double* d_gz, const unsigned char* d_mask, double* d_P_out, double tol, int max_outer,
                   int max_cg, void* stream, omni_info* info)
{
    if (!d_gx || !d_gy || (nz > 1 && !d_gz) || !d_P_out) return OMNI_ERR_INVALID_ARG;
    return solve_alloc<double>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_out, tol, max_outer, max_cg, stream, info);
}

int omni_solve_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_gx, const float* d_gy,
                   const float* d_gz, const unsigned char* d_mask, float* d_P_out, double tol, int max_outer,
                   int max_cg, void* stream, omni_info* info)
{
    if (!d_gx || !d_gy || (nz > 1 && !d_gz) || !d_P_out) return OMNI_ERR_INVALID_ARG;
    return solve_alloc<float>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_out, tol, max_outer, max_cg, stream, info);
}

size_t omni_workspace_bytes(int nx, int ny, int nz, int dtype)
{
    Geom g;
    if (dtype != OMNI_F32 && dtype != OMNI_F64) return 0;
    if (!make_geom(nx, ny, nz, dtype == OMNI_F32 ? 4 : 8, g)) return 0;
    return dtype == OMNI_F32 ? carve<float>(g, nullptr, nullptr) : carve<double>(g, nullptr, nullptr);
}

int omni_solve_f64_ws(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_gx, const double* d_gy,
                      const double* d_gz, const unsigned char* d_mask, double* d_P_out, double tol, int max_outer,
                      int max_cg, void* d_workspace, size_t workspace_bytes, void* stream, omni_info* info)
{
    return solve_ws<double>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_out, tol, max_outer, max_cg, d_workspace,
                            workspace_bytes, stream, info);
}

int omni_solve_f32_ws(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_gx, const float* d_gy,
                      const float* d_gz, const unsigned char* d_mask, float* d_P_out, double tol, int max_outer,
                      int max_cg, void* d_workspace, size_t workspace_bytes, void* stream, omni_info* info)
{
    return solve_ws<float>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_out, tol, max_outer, max_cg, d_workspace,
                           workspace_bytes, stream, info);
}

int omni_solve_host_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* h_gx, const double* h_gy,
                        const double* h_gz, const unsigned char* h_mask, double* h_P_out, double tol, int max_outer,
                        int max_cg, void* stream, omni_info* info)
{
    return solve_host<double>(nx, ny, nz, dx, dy, dz, h_gx, h_gy, h_gz, h_mask, h_P_out, tol, max_outer, max_cg, stream, info);
}

int omni_solve_host_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* h_gx, const float* h_gy,
                        const float* h_gz, const unsigned char* h_mask, float* h_P_out, double tol, int max_outer,
                        int max_cg, void* stream, omni_info* info)
{
    return solve_host<float>(nx, ny, nz, dx, dy, dz, h_gx, h_gy, h_gz, h_mask, h_P_out, tol, max_outer, max_cg, stream, info);
}

int omni_solve_batch2d_f64(int nx, int ny, int nb, double dx, double dy, const double* d_gx, const double* d_gy,
                           const unsigned char* d_mask2d, const double* d_P_init, double* d_P_out, double tol,
                           int max_outer, int max_cg, void* stream, omni_info* info)
{
    if (!d_gx || !d_gy || !d_P_out || nb < 1) return OMNI_ERR_INVALID_ARG;
    return solve_alloc<double>(nx, ny, nb, dx, dy, 1.0, d_gx, d_gy, nullptr, d_mask2d, d_P_out, tol, max_outer, max_cg, stream,
                               info, 1, d_P_init);
}

int omni_solve_batch2d_f32(int nx, int ny, int nb, double dx, double dy, const float* d_gx, const float* d_gy,
                           const unsigned char* d_mask2d, const float* d_P_init, float* d_P_out, double tol,
                           int max_outer, int max_cg, void* stream, omni_info* info)
{
    if (!d_gx || !d_gy || !d_P_out || nb < 1) return OMNI_ERR_INVALID_ARG;
    return solve_alloc<float>(nx, ny, nb, dx, dy, 1.0, d_gx, d_gy, nullptr, d_mask2d, d_P_out, tol, max_outer, max_cg, stream,
                              info, 1, d_P_init);
}

int omni_solve_pcg_batch2d_f64(int nx, int ny, int nb, double dx, double dy, const double* d_gx, const double* d_gy,
                               const unsigned char* d_mask2d, const double* d_P_init, double* d_P_out, double tol,
                               int max_outer, int max_cg, void* stream, omni_info* info)
{
    if (!d_gx || !d_gy || !d_P_out || nb < 1) return OMNI_ERR_INVALID_ARG;
    return solve_alloc<double>(nx, ny, nb, dx, dy, 1.0, d_gx, d_gy, nullptr, d_mask2d, d_P_out, tol, max_outer, max_cg, stream,
                               info, 1, d_P_init, 1, 1);
}

int omni_solve_pcg_batch2d_f32(int nx, int ny, int nb, double dx, double dy, const float* d_gx, const float* d_gy,
                               const unsigned char* d_mask2d, const float* d_P_init, float* d_P_out, double tol,
                               int max_outer, int max_cg, void* stream, omni_info* info)
{
    if (!d_gx || !d_gy || !d_P_out || nb < 1) return OMNI_ERR_INVALID_ARG;
    return solve_alloc<float>(nx, ny, nb, dx, dy, 1.0, d_gx, d_gy, nullptr, d_mask2d, d_P_out, tol, max_outer, max_cg, stream,
                              info, 1, d_P_init, 1, 1);
}

int omni_solve_direct_batch2d_f64(int nx, int ny, int nb, double dx, double dy, const double* d_gx, const double* d_gy,
                                  const unsigned char* d_mask2d, const double* d_P_init, double* d_P_out, double tol,
                                  int max_outer, int max_cg, void* stream, omni_info* info)
{
    if (!d_gx || !d_gy || !d_P_out || nb < 1) return OMNI_ERR_INVALID_ARG;
    return solve_alloc<double>(nx, ny, nb, dx, dy, 1.0, d_gx, d_gy, nullptr, d_mask2d, d_P_out, tol, max_outer, max_cg, stream,
                               info, 1, d_P_init, 1);
}

int omni_solve_direct_batch2d_f32(int nx, int ny, int nb, double dx, double dy, const float* d_gx, const float* d_gy,
                                  const unsigned char* d_mask2d, const float* d_P_init, float* d_P_out, double tol,
                                  int max_outer, int max_cg, void* stream, omni_info* info)
{
    if (!d_gx || !d_gy || !d_P_out || nb < 1) return OMNI_ERR_INVALID_ARG;
    return solve_alloc<float>(nx, ny, nb, dx, dy, 1.0, d_gx, d_gy, nullptr, d_mask2d, d_P_out, tol, max_outer, max_cg, stream,
                              info, 1, d_P_init, 1);
}

int omni_solve_guess_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_gx, const double* d_gy,
                         const double* d_gz, const unsigned char* d_mask, const double* d_P_init, double* d_P_out,
                         double tol, int max_outer, int max_cg, void* stream, omni_info* info)
{
    return solve_alloc<double>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_out, tol, max_outer, max_cg, stream, info,
                               0, d_P_init, 0);
}

int omni_solve_guess_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_gx, const float* d_gy,
                         const float* d_gz, const unsigned char* d_mask, const float* d_P_init, float* d_P_out,
                         double tol, int max_outer, int max_cg, void* stream, omni_info* info)
{
    return solve_alloc<float>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_out, tol, max_outer, max_cg, stream, info,
                              0, d_P_init, 0);
}

int omni_solve_direct_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_gx, const double* d_gy,
                          const double* d_gz, const unsigned char* d_mask, const double* d_P_init, double* d_P_out,
                          double tol, int max_outer, int max_cg, void* stream, omni_info* info)
{
    return solve_alloc<double>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_out, tol, max_outer, max_cg, stream, info,
                               0, d_P_init, 1);
}

int omni_solve_direct_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_gx, const float* d_gy,
                          const float* d_gz, const unsigned char* d_mask, const float* d_P_init, float* d_P_out,
                          double tol, int max_outer, int max_cg, void* stream, omni_info* info)
{
    return solve_alloc<float>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_out, tol, max_outer, max_cg, stream, info,
                              0, d_P_init, 1);
}

int omni_solve_pcg_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_gx, const double* d_gy,
                       const double* d_gz, const unsigned char* d_mask, const double* d_P_init, double* d_P_out,
                       double tol, int max_outer, int max_cg, void* stream, omni_info* info)
{
    return solve_alloc<double>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_out, tol, max_outer, max_cg, stream, info,
                               0, d_P_init, 1, 1);
}

int omni_solve_pcg_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_gx, const float* d_gy,
                       const float* d_gz, const unsigned char* d_mask, const float* d_P_init, float* d_P_out,
                       double tol, int max_outer, int max_cg, void* stream, omni_info* info)
{
    return solve_alloc<float>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_out, tol, max_outer, max_cg, stream, info,
                              0, d_P_init, 1, 1);
}

void omni_options_init(omni_options* o)
{
    if (!o) return;
    memset(o, 0, sizeof(*o));
    o->struct_size = sizeof(omni_options);
    o->loop_mode = -1;
}

extern "C++" {
namespace {
template <typename T>
int solve_ex(int nx, int ny, int nz, double dx, double dy, double dz, const T* gx, const T* gy, const T* gz,
             const unsigned char* mask, const T* P_init, T* P_out, double tol, int max_outer, int max_cg, int method,
             const omni_options* o, void* stream, omni_info* info)
{
    if (method != OMNI_METHOD_ALG1 && method != OMNI_METHOD_DIRECT && method != OMNI_METHOD_PCG) return OMNI_ERR_INVALID_ARG;
    CallOpts c = current_opts();
    if (o) {
        if (o->struct_size != sizeof(omni_options)) return OMNI_ERR_INVALID_ARG;
        if (o->loop_mode > 5 || o->loop_mode < -1 || o->hist_capacity < 0) return OMNI_ERR_INVALID_ARG;
        if (o->hist_capacity == 0 && (o->d_hist_eps_R || o->d_hist_cg_iters || o->d_hist_eps_P)) return OMNI_ERR_INVALID_ARG;
        if (o->loop_mode >= 0) c.loop_mode = o->loop_mode;
        c.hist = o->d_hist_eps_R; c.hist_k = o->d_hist_cg_iters; c.hist_p = o->d_hist_eps_P; c.hist_cap = o->hist_capacity;
        c.P64 = o->d_P64_out; c.status = o->d_status; c.single_reduction = o->single_reduction != 0;
    }
    tl_opts = &c;
    const int rc = solve_alloc<T>(nx, ny, nz, dx, dy, dz, gx, gy, gz, mask, P_out, tol, max_outer, max_cg, stream, info, 0, P_init,
                                  method != OMNI_METHOD_ALG1, method == OMNI_METHOD_PCG);
    tl_opts = nullptr;
    return rc;
}
}  // namespace
}  // extern "C++"

int omni_solve_ex_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_gx, const double* d_gy,
                      const double* d_gz, const unsigned char* d_mask, const double* d_P_init, double* d_P_out, double tol,
                      int max_outer, int max_cg, int method, const omni_options* options, void* stream, omni_info* info)
{
    return solve_ex<double>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_init, d_P_out, tol, max_outer, max_cg, method,
                            options, stream, info);
}

int omni_solve_ex_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_gx, const float* d_gy,
                      const float* d_gz, const unsigned char* d_mask, const float* d_P_init, float* d_P_out, double tol,
                      int max_outer, int max_cg, int method, const omni_options* options, void* stream, omni_info* info)
{
    return solve_ex<float>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_init, d_P_out, tol, max_outer, max_cg, method,
                           options, stream, info);
}

int omni_solve_cascade_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_gx, const double* d_gy,
                           const double* d_gz, const unsigned char* d_mask, double* d_P_out, double tol, int max_outer,
                           int max_cg, int levels, void* stream, omni_info* info)
{
    return solve_cascade<double>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_out, tol, max_outer, max_cg, levels, stream, info);
}

int omni_solve_cascade_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_gx, const float* d_gy,
                           const float* d_gz, const unsigned char* d_mask, float* d_P_out, double tol, int max_outer,
                           int max_cg, int levels, void* stream, omni_info* info)
{
    return solve_cascade<float>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P_out, tol, max_outer, max_cg, levels, stream, info);
}

int omni_velocity_source_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_u, const double* d_v,
                             const double* d_w, const double* d_dudt, const double* d_dvdt, const double* d_dwdt,
                             const unsigned char* d_mask, double rho, double mu, double* d_gx, double* d_gy, double* d_gz,
                             void* stream)
{
    return velocity_source<double>(nx, ny, nz, dx, dy, dz, d_u, d_v, d_w, d_dudt, d_dvdt, d_dwdt, d_mask, rho, mu, d_gx, d_gy, d_gz, stream);
}

int omni_velocity_source_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_u, const float* d_v,
                             const float* d_w, const float* d_dudt, const float* d_dvdt, const float* d_dwdt,
                             const unsigned char* d_mask, double rho, double mu, float* d_gx, float* d_gy, float* d_gz,
                             void* stream)
{
    return velocity_source<float>(nx, ny, nz, dx, dy, dz, d_u, d_v, d_w, d_dudt, d_dvdt, d_dwdt, d_mask, rho, mu, d_gx, d_gy, d_gz, stream);
}

int omni_rans_source_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_u, const double* d_v,
                         const double* d_w, const double* const* d_stress, const unsigned char* d_mask, double rho,
                         double* d_fx, double* d_fy, double* d_fz, void* stream)
{
    return rans_source<double>(false, nx, ny, nz, dx, dy, dz, d_u, d_v, d_w, d_stress, d_mask, rho, 0, 0, 0, 0, d_fx, d_fy, d_fz, stream);
}

int omni_rans_source_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_u, const float* d_v,
                         const float* d_w, const float* const* d_stress, const unsigned char* d_mask, double rho,
                         float* d_fx, float* d_fy, float* d_fz, void* stream)
{
    return rans_source<float>(false, nx, ny, nz, dx, dy, dz, d_u, d_v, d_w, d_stress, d_mask, rho, 0, 0, 0, 0, d_fx, d_fy, d_fz, stream);
}

int omni_compressible_rans_source_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_u,
                                      const double* d_v, const double* d_w, const double* const* d_stress,
                                      const unsigned char* d_mask, double gamma, double mach_inf, double v_inf,
                                      double rgas_t_inf, double* d_gx, double* d_gy, double* d_gz, void* stream)
{
    return rans_source<double>(true, nx, ny, nz, dx, dy, dz, d_u, d_v, d_w, d_stress, d_mask, 0, gamma, mach_inf, v_inf, rgas_t_inf,
                               d_gx, d_gy, d_gz, stream);
}

int omni_compressible_rans_source_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_u,
                                      const float* d_v, const float* d_w, const float* const* d_stress,
                                      const unsigned char* d_mask, double gamma, double mach_inf, double v_inf,
                                      double rgas_t_inf, float* d_gx, float* d_gy, float* d_gz, void* stream)
{
    return rans_source<float>(true, nx, ny, nz, dx, dy, dz, d_u, d_v, d_w, d_stress, d_mask, 0, gamma, mach_inf, v_inf, rgas_t_inf,
                              d_gx, d_gy, d_gz, stream);
}

int omni_slab_plan(int nz, int nranks, int rank, int* z0, int* z1, int* zlo, int* zhi)
{
    int a, b, c, d;
    if (!slab_plan(nz, nranks, rank, a, b, c, d)) return OMNI_ERR_INVALID_ARG;
    if (z0) *z0 = a;
    if (z1) *z1 = b;
    if (zlo) *zlo = c;
    if (zhi) *zhi = d;
    return OMNI_OK;
}

int omni_slab_unique_id(char* h_id128)
{
    if (!h_id128 || !nccl_api().ok) return OMNI_ERR_CUDA;
    NcclApi::UniqueId id;
    if (nccl_api().GetUniqueId(&id) != 0) return OMNI_ERR_CUDA;
    memcpy(h_id128, id.internal, 128);
    return OMNI_OK;
}

int omni_slab_comm_create(int rank, int nranks, const char* h_id128, void** comm)
{
    if (!h_id128 || !comm || nranks < 1 || rank < 0 || rank >= nranks) return OMNI_ERR_INVALID_ARG;
    if (!nccl_api().ok) return OMNI_ERR_CUDA;
    NcclApi::UniqueId id;
    memcpy(id.internal, h_id128, 128);
    return nccl_api().CommInitRank(comm, nranks, id, rank) == 0 ? OMNI_OK : OMNI_ERR_CUDA;
}

void omni_slab_comm_destroy(void* comm)
{
    if (comm && nccl_api().ok) nccl_api().CommDestroy(comm);
}

int omni_solve_slab_f64(int nx, int ny, int nz, double dx, double dy, double dz, int nlocal, const int* h_ranks,
                        const double* const* h_gx, const double* const* h_gy, const double* const* h_gz,
                        const unsigned char* const* h_mask, double* const* h_P_out, double tol, int max_outer, int max_cg,
                        int method, int nranks, void* comm, void* stream, omni_info* info)
{
    if (method != OMNI_METHOD_ALG1 && method != OMNI_METHOD_DIRECT) return OMNI_ERR_INVALID_ARG;
    return solve_slab<double>(nx, ny, nz, dx, dy, dz, nlocal, h_ranks, h_gx, h_gy, h_gz, h_mask, h_P_out, tol, max_outer, max_cg,
                              method == OMNI_METHOD_DIRECT, nranks, comm, stream, info);
}

int omni_solve_slab_f32(int nx, int ny, int nz, double dx, double dy, double dz, int nlocal, const int* h_ranks,
                        const float* const* h_gx, const float* const* h_gy, const float* const* h_gz,
                        const unsigned char* const* h_mask, float* const* h_P_out, double tol, int max_outer, int max_cg,
                        int method, int nranks, void* comm, void* stream, omni_info* info)
{
    if (method != OMNI_METHOD_ALG1 && method != OMNI_METHOD_DIRECT) return OMNI_ERR_INVALID_ARG;
    return solve_slab<float>(nx, ny, nz, dx, dy, dz, nlocal, h_ranks, h_gx, h_gy, h_gz, h_mask, h_P_out, tol, max_outer, max_cg,
                             method == OMNI_METHOD_DIRECT, nranks, comm, stream, info);
}

extern "C++" {
namespace {
// device address of g_noalloc_scratch on the CURRENT device, looked up once per device with that device current
int noalloc_scratch_ptr(double** out)
{
    static std::mutex mu;
    static double* cache[MAX_DEVICES] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return OMNI_ERR_CUDA; }
    std::lock_guard<std::mutex> lk(mu);
    if (dev >= 0 && dev < MAX_DEVICES && cache[dev]) { *out = cache[dev]; return OMNI_OK; }
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || p == nullptr) { cudaGetLastError(); return OMNI_ERR_CUDA; }
    if (dev >= 0 && dev < MAX_DEVICES) cache[dev] = (double*)p;
    *out = (double*)p;
    return OMNI_OK;
}

template <typename T>
int source_noalloc(int nx, int ny, int nz, double dx, double dy, double dz, const T* gx, const T* gy, const T* gz,
                   const unsigned char* mask, T* S_out, double* d_norm_S, void* stream)
{
    if (!valid_common(nx, ny, nz, dx, dy, dz, 0.0, 0, 0)) return OMNI_ERR_INVALID_ARG;
    if (!gx || !gy || (nz > 1 && !gz) || !S_out) return OMNI_ERR_INVALID_ARG;
    const long long n = (long long)nx * ny * nz;
    if (n > NOALLOC_MAX_CELLS) return OMNI_ERR_TOO_LARGE;          // one reduction slot per 4096 cells, 32 760 slots
    const int naxes = nz > 1 ? 3 : 2;
    HostConst H;
    host_constants(naxes, dx, dy, dz, H);
    const double d[3] = { dx, dy, dz };
    T hs[3];
    for (int a = 0; a < 3; ++a) hs[a] = (T)(a < naxes ? d[a] * (H.F[a] / H.Atot) * 0.5 : 0.0);      // as make_coef: Coef::hs
    double* scratch = nullptr;
    const int rc = noalloc_scratch_ptr(&scratch);
    if (rc != OMNI_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // the array keeps the last call's contents: the ticket must start at zero (an aborted call may have left it set)
    CK(cudaMemsetAsync(scratch, 0, NOALLOC_HEADER_DOUBLES * sizeof(double), st));
    const unsigned nb = (unsigned)((n + NOALLOC_CELLS_PER_CTA - 1) / NOALLOC_CELLS_PER_CTA);
    source_noalloc_kernel<T><<<nb, NOALLOC_THREADS, 0, st>>>(nx, ny, nz, naxes, gx, gy, gz, mask, hs[0], hs[1], hs[2], S_out, scratch,
                                                             d_norm_S);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    CK(cudaGetLastError());
    return OMNI_OK;
}
}  // namespace
}  // extern "C++"

int omni_source_noalloc_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_gx, const double* d_gy,
                            const double* d_gz, const unsigned char* d_mask, double* d_S_out, double* d_norm_S, void* stream)
{
    return source_noalloc<double>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_S_out, d_norm_S, stream);
}

int omni_source_noalloc_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_gx, const float* d_gy,
                            const float* d_gz, const unsigned char* d_mask, float* d_S_out, double* d_norm_S, void* stream)
{
    return source_noalloc<float>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_S_out, d_norm_S, stream);
}

long long omni_source_noalloc_max_cells(void) { return NOALLOC_MAX_CELLS; }

int omni_constants(int nx, int ny, int nz, double dx, double dy, double dz, double* h_out13)
{
    if (!h_out13 || !valid_common(nx, ny, nz, dx, dy, dz, 0.0, 0, 0)) return OMNI_ERR_INVALID_ARG;
    HostConst H;
    host_constants(nz > 1 ? 3 : 2, dx, dy, dz, H);
    h_out13[0] = H.F[0]; h_out13[1] = H.F[1]; h_out13[2] = H.F[2]; h_out13[3] = H.Atot;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) h_out13[4 + 3 * a + b] = H.c[a][b];
    return OMNI_OK;
}

int omni_source_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_gx, const double* d_gy,
                    const double* d_gz, const unsigned char* d_mask, double* d_S_out, double* h_norm_S, void* stream)
{
    return source_step<double>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_S_out, h_norm_S, stream);
}
int omni_source_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_gx, const float* d_gy,
                    const float* d_gz, const unsigned char* d_mask, float* d_S_out, double* h_norm_S, void* stream)
{
    return source_step<float>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_S_out, h_norm_S, stream);
}

int omni_apply_M_f64(int nx, int ny, int nz, double dx, double dy, double dz, const unsigned char* d_mask,
                     const double* d_p, double* d_q, double* h_pq, void* stream)
{
    return apply_M_step<double>(nx, ny, nz, dx, dy, dz, d_mask, d_p, d_q, h_pq, stream);
}
int omni_apply_M_f32(int nx, int ny, int nz, double dx, double dy, double dz, const unsigned char* d_mask,
                     const float* d_p, float* d_q, double* h_pq, void* stream)
{
    return apply_M_step<float>(nx, ny, nz, dx, dy, dz, d_mask, d_p, d_q, h_pq, stream);
}

int omni_residual_f64(int nx, int ny, int nz, double dx, double dy, double dz, const double* d_gx, const double* d_gy,
                      const double* d_gz, const unsigned char* d_mask, const double* d_P, double* d_r_out,
                      double* h_eps_R, void* stream)
{
    return residual_step<double>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P, d_r_out, h_eps_R, stream);
}
int omni_residual_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* d_gx, const float* d_gy,
                      const float* d_gz, const unsigned char* d_mask, const double* d_P, float* d_r_out,
                      double* h_eps_R, void* stream)
{
    return residual_step<float>(nx, ny, nz, dx, dy, dz, d_gx, d_gy, d_gz, d_mask, d_P, d_r_out, h_eps_R, stream);
}

long long omni_launch_count(int reset)
{
    return reset ? g_launches.exchange(0) : g_launches.load();
}

int omni_profile_enable(int on)
{
    return g_profile.exchange(on ? 1 : 0);
}

void omni_profile_read(double* h_ms3, long long* h_count3, int reset)
{
    std::lock_guard<std::mutex> lk(g_prof_mu);
    for (int i = 0; i < 3; ++i) {
        if (h_ms3) h_ms3[i] = g_prof_ms[i];
        if (h_count3) h_count3[i] = g_prof_n[i];
        if (reset) { g_prof_ms[i] = 0.0; g_prof_n[i] = 0; }
    }
}

#ifdef OMNI_TUNING
// tuning builds only: copy the per-CTA timeline of operator `which` (ticket index: 0 K3, 1 K4, 2 K2) to the host
int omni_debug_cta_trace(int which, unsigned long long* h_out, int n_ctas)
{
    if (which < 0 || which > 2 || n_ctas > 8192) return -1;
    cudaDeviceSynchronize();
    return cudaMemcpyFromSymbol(h_out, omni::g_cta_trace, (size_t)n_ctas * 24, (size_t)which * 3 * 8192 * 8) == cudaSuccess ? 0 : -2;
}
#endif

#ifdef OMNI_TUNING
// tuning builds only: `reps` V-cycles of the multigrid preconditioner on b = S, launched one by one on the stream (outside
// any graph, so that a profiler sees the level kernels by name)
int omni_debug_vcycle_f32(int nx, int ny, int nz, double dx, double dy, double dz, const float* gx, const float* gy,
                          const float* gz, const unsigned char* mask, int reps, void* stream)
{
    Geom g;
    if (!make_geom(nx, ny, nz, 4, g)) return OMNI_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = carve<float>(g, nullptr, nullptr);
    void* ws = nullptr;
    if (pool_alloc(&ws, bytes, st) != cudaSuccess) return OMNI_ERR_ALLOC;
    Workspace<float> w;
    carve<float>(g, (char*)ws, &w);
    HostConst H;
    host_constants(g.naxes, dx, dy, dz, H);
    const Coef<float> K = make_coef<float>(H, dx, dy, dz, g);
    init_scalars_kernel<<<1, 1, 0, st>>>(w.sc, 1e-5, 1, 1);
    int rc = setup_codes<float>(g, w, gx, gy, gz, mask, st);
    if (rc == OMNI_OK) rc = launch_source<float>(g, w, K, gx, gy, gz, st);
    MgHier<float> M;
    if (rc == OMNI_OK) rc = mg_build<float>(g, w, H, M, st);
    if (rc == OMNI_OK) {
        cudaMemcpyAsync(w.r, w.S, (size_t)g.npad * 4, cudaMemcpyDeviceToDevice, st);
        for (int i = 0; i < reps; ++i) mg_vcycle<float>(M, 0, st);
        cudaFreeAsync(M.mem, st);
    }
    cudaStreamSynchronize(st);
    cudaFreeAsync(ws, st);
    return cudaGetLastError() == cudaSuccess ? rc : OMNI_ERR_CUDA;
}

// tuning builds only: per-CTA timeline of the loop kernel's first phases: h_out[phase][cta][3], returns the phase count
int omni_debug_loop_trace(unsigned long long* h_out, int max_phases)
{
    cudaDeviceSynchronize();
    int n = 0;
    if (cudaMemcpyFromSymbol(&n, omni::g_loop_trace_n, sizeof(int)) != cudaSuccess) return -1;
    if (n > max_phases) n = max_phases;
    if (cudaMemcpyFromSymbol(h_out, omni::g_loop_trace, (size_t)n * 1024 * 3 * 8) != cudaSuccess) return -2;
    return n;
}
#endif

int omni_set_history(double* d_hist, int* d_cg_iters, int capacity)
{
    if (capacity < 0 || (d_hist == nullptr && (capacity > 0 || d_cg_iters != nullptr))) return OMNI_ERR_INVALID_ARG;
    g_hist.store(capacity > 0 ? d_hist : nullptr);
    g_hist_k.store(capacity > 0 ? d_cg_iters : nullptr);
    g_hist_cap.store(capacity > 0 ? capacity : 0);
    return OMNI_OK;
}

void omni_release_memory(void)
{
    reap_graphs(true);
    std::lock_guard<std::mutex> lk(g_pool_mu);
    for (auto& p : g_pools)
        if (p) cudaMemPoolTrimTo(p, 0);
}

int omni_set_loop_mode(int mode)
{
    if (mode < 0 || mode > 5) return g_loop_mode.load();
    return g_loop_mode.exchange(mode);
}

const char* omni_status_string(int status)
{
    switch (status) {
    case OMNI_OK: return "ok";
    case OMNI_NOT_CONVERGED: return "not converged: max_outer reached (last iterate written)";
    case OMNI_ERR_INVALID_ARG: return "invalid argument";
    case OMNI_ERR_CUDA: return "CUDA runtime error (or no CUDA device)";
    case OMNI_ERR_ALLOC: return "workspace allocation failed or workspace too small";
    case OMNI_ERR_BREAKDOWN: return "CG breakdown: non-finite scalar or p.Mp <= 0";
    case OMNI_ERR_TOO_LARGE: return "grid exceeds the fixed scratch of the no-allocation entry point (omni_source_noalloc_max_cells)";
    default: return "unknown status";
    }
}

int omni_resident_plan(int nx, int ny, int nz, int elem_size, int nsm, int lop, int* out)
{
    Geom g;
    if ((elem_size != 4 && elem_size != 8) || !out || nsm < 1 || !make_geom(nx, ny, nz, elem_size, g, 0)) return OMNI_ERR_INVALID_ARG;
    ResidentPlan pl;
    if (!resident_plan_auto(g, elem_size, nsm < 148 ? nsm : 148, lop != 0, pl)) return 0;
    const int v[13] = { pl.gy, pl.gz, pl.ly, pl.lz, (int)pl.smem_bytes, pl.rpt, pl.rreg, pl.dres, pl.qres, pl.wy, pl.wz, g.px, pl.rtm };
    for (int i = 0; i < 13; ++i) out[i] = v[i];
    return 1;
}

int omni_resident_split(int n, int parts, int i, int wface) { return res_split(n, parts, i, wface); }

int omni_version(void) { return 107; }   // 101: omni_solve_guess_*, omni_set_history, omni_rans_source_*, omni_compressible_rans_source_*

#ifdef OMNI_RES_TRACE
int omni_debug_res_trace(unsigned long long* out, int reset)
{
    unsigned long long z[16] = { 0 };
    if (cudaMemcpyFromSymbol(out, omni::g_res_trace, sizeof(z)) != cudaSuccess) return -1;
    z[15] = (unsigned long long)(reset > 0 ? reset - 1 : 0);      // reset = 1 + index of the CTA to trace
    if (reset && cudaMemcpyToSymbol(omni::g_res_trace, z, sizeof(z)) != cudaSuccess) return -1;
    return 0;
}
#endif
}  // extern "C"
