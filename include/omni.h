/* omni.h -- C ABI of the B200-native hot path of the matrix-based omnidirectional pressure integration
 * (Zigunov & Charonko, arXiv 2311.16935; citations are PAPER.md:<line>).
 *
 * Problem statement (PAPER.md:26, :51, :122, Algorithm 1 :128-150, :158): given a measured pressure-gradient field
 * f = grad P on a uniform rectangular grid with some cells missing, return P on the valid cells, up to an additive
 * constant per connected region, by iterating  [W^{n+1}]{P^{n+1}} = [W^n]{P^n} + {S}  (Eq. 12 :119) from P^0 = 0,
 * each system solved by conjugate gradients warm-started from P^n (:124, :489).
 *
 * Conventions for every entry point
 *   - x is the fastest index: idx = i + nx*(j + ny*k).  nz == 1 selects the 2D scheme (Eq. 8, 14-20); dz and gz are
 *     then ignored and gz may be NULL.  E/W = +/-x, N/S = +/-y, F/B = +/-z (:103).
 *   - a cell is MISSING if it is outside the box, or mask[idx] == 0, or any used component of g is NaN (Eq. 13 :176).
 *   - pointers named d_* are DEVICE memory owned by the caller (for example a torch tensor); pointers named h_* are
 *     HOST memory owned by the caller.  The library never frees or keeps caller memory.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  All device work is enqueued on it.
 *   - errors are return codes only: nothing is printed, thrown or exit()ed.  Invalid arguments are rejected before
 *     anything is enqueued.  Negative codes are errors; OMNI_NOT_CONVERGED (1) still writes the last iterate.
 *   - same inputs give bit-identical outputs (fixed reduction order, no floating-point atomics).
 *   - there is no CPU fallback: without a CUDA device every compute entry point returns OMNI_ERR_CUDA.
 */
#ifndef OMNI_H
#define OMNI_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    OMNI_OK = 0,
    OMNI_NOT_CONVERGED = 1,    /* max_outer reached with eps_R > tol; result written                      */
    OMNI_ERR_INVALID_ARG = -1,
    OMNI_ERR_CUDA = -2,        /* a CUDA runtime call failed (or no device)                                */
    OMNI_ERR_ALLOC = -3,       /* workspace allocation failed / caller workspace too small                 */
    OMNI_ERR_BREAKDOWN = -4,   /* non-finite scalar or p.Mp <= 0 seen on the device (M is not symmetric)   */
    OMNI_ERR_TOO_LARGE = -5    /* omni_source_noalloc_*: the grid exceeds the library's fixed scratch       */
} omni_status;

typedef struct {
    int outer_iters;           /* n: number of Eq. 12 solves performed (Algorithm 1 :141-149)              */
    long long cg_iters_total;  /* CG iterations summed over all outer iterations                           */
    double eps_R_final;        /* momentum residual of the returned field, Eq. 41 :442                     */
    double norm_S;             /* ||S||_2, the denominator of Eq. 41                                       */
    int status;                /* same value as the function's return code                                 */
} omni_info;

enum { OMNI_F32 = 0, OMNI_F64 = 1 };

/* ---- the whole hot path: Algorithm 1 (:128-150) -------------------------------------
 * d_gx, d_gy, d_gz : [nx*ny*nz] pressure-gradient components (Eq. 1 :23), NaN = missing (:158).
 * d_mask           : [nx*ny*nz] bytes, 1 = valid, 0 = missing; NULL = all cells valid.
 * d_P_out          : [nx*ny*nz] result; quiet NaN at missing cells.  Not mean-shifted (the caller pins the constant).
 * tol              : outer stop eps_R <= tol (Eq. 41); inner CG stops at ||r_k|| <= 0.1*tol*||S|| (A3).
 * max_outer,max_cg : caps on outer iterations / CG iterations per outer iteration (>= 0).  tol = 0 runs exactly
 *                    max_outer x max_cg iterations (fixed-count trajectories).
 * info             : host, may be NULL.  If NULL the call returns right after enqueueing (no synchronisation and
 *                    the return code covers argument / launch errors only); otherwise the call synchronises `stream`
 *                    once at the end and fills *info.
 * _f32: g, S, the CG vectors and the stencil arithmetic are fp32; dot products accumulate in fp64; the master
 * pressure and the outer residual (Eq. 41) are fp64 (A9).  dx, dy, dz, tol are double in both variants.
 * Workspace is taken from the stream-ordered allocator (cudaMallocAsync) and released before returning. */
int omni_solve_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                   const double* d_gx, const double* d_gy, const double* d_gz, const unsigned char* d_mask,
                   double* d_P_out, double tol, int max_outer, int max_cg, void* stream, omni_info* info);
int omni_solve_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                   const float* d_gx, const float* d_gy, const float* d_gz, const unsigned char* d_mask,
                   float* d_P_out, double tol, int max_outer, int max_cg, void* stream, omni_info* info);

/* Same with a caller-supplied device workspace (no allocation inside): d_workspace must hold at least
 * omni_workspace_bytes(nx, ny, nz, dtype) bytes, 256-byte aligned; contents are scratch. */
size_t omni_workspace_bytes(int nx, int ny, int nz, int dtype /* OMNI_F32 | OMNI_F64 */);
int omni_solve_f64_ws(int nx, int ny, int nz, double dx, double dy, double dz,
                      const double* d_gx, const double* d_gy, const double* d_gz, const unsigned char* d_mask,
                      double* d_P_out, double tol, int max_outer, int max_cg,
                      void* d_workspace, size_t workspace_bytes, void* stream, omni_info* info);
int omni_solve_f32_ws(int nx, int ny, int nz, double dx, double dy, double dz,
                      const float* d_gx, const float* d_gy, const float* d_gz, const unsigned char* d_mask,
                      float* d_P_out, double tol, int max_outer, int max_cg,
                      void* d_workspace, size_t workspace_bytes, void* stream, omni_info* info);

/* Same with HOST buffers: allocates device memory, copies h_g* / h_mask to the device, solves, copies P back and
 * synchronises.  h_* buffers may be pageable or pinned. */
int omni_solve_host_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                        const double* h_gx, const double* h_gy, const double* h_gz, const unsigned char* h_mask,
                        double* h_P_out, double tol, int max_outer, int max_cg, void* stream, omni_info* info);
int omni_solve_host_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                        const float* h_gx, const float* h_gy, const float* h_gz, const unsigned char* h_mask,
                        float* h_P_out, double tol, int max_outer, int max_cg, void* stream, omni_info* info);

/* ---- one entry point with per-call options ---------------------------------------------------------------------
 * omni_solve_ex_* runs Algorithm 1 (OMNI_METHOD_ALG1: what omni_solve_guess_* runs), CG on the fixed-point system
 * (OMNI_METHOD_DIRECT: omni_solve_direct_*) or its multigrid-preconditioned form (OMNI_METHOD_PCG: omni_solve_pcg_*)
 * with everything that is otherwise a process-wide setting passed IN THE CALL: two concurrent solves (threads,
 * streams) never share a history buffer or a loop mode.  options == NULL: the process-wide defaults.  All pointers in
 * omni_options are DEVICE memory owned by the caller and must stay valid until the solve has finished on `stream`.
 *   loop_mode       -1: the process-wide setting (omni_set_loop_mode); 0..5 as described there
 *   d_hist_eps_R    [hist_capacity] doubles: eps_R (Eq. 41 :442) at the i-th outer residual check (i = 0: first guess)
 *   d_hist_cg_iters [hist_capacity] ints: CG iterations of the outer iteration that led to check i (0 for i = 0)
 *   d_hist_eps_P    [hist_capacity] doubles: the pressure-update metric eps_P = ||P^i - P^(i-1)|| / ||P^i|| (Eq. 40 :438)
 *                   of the update that led to check i (0 for i = 0); any of the three may be NULL
 *   d_P64_out       [nx*ny*nz] doubles: the fp64 master pressure itself (NaN at missing cells).  The _f32 result
 *                   d_P_out is this field rounded to fp32, and that rounding alone leaves a residual of about
 *                   2^-24 |L||P| / ||S||, which on 1000-cell-wide grids exceeds tol = 1e-5; d_P64_out satisfies eps_R <= tol
 *   d_status        one int: the final status, written by the device when the solve ends -- the way to learn about
 *                   OMNI_NOT_CONVERGED / OMNI_ERR_BREAKDOWN after a call made with info == NULL (no synchronisation)
 *   single_reduction  OMNI_METHOD_DIRECT in the persistent loop (mode 3: grids up to 1.5 M cells by default) only: the
 *                   Chronopoulos-Gear recurrences, ONE grid barrier per CG iteration instead of two (SURVEY.md 8(f)
 *                   NEXT-2 i).  In exact arithmetic the same iterates; it relies on L = L^T, so it does not exist for
 *                   Algorithm 1, whose operator is not symmetric (A2).  Ignored elsewhere.  It selects mode 3 even
 *                   where the automatic choice would be the SM-resident loop (mode 5), which is faster with its two
 *                   relaxed barriers: a numerical variant, not a speed-up.
 * struct_size must be sizeof(omni_options) (omni_options_init sets it, loop_mode = -1 and everything else to 0 / NULL);
 * a mismatch, hist_capacity < 0, a history pointer with hist_capacity == 0 or an unknown method: OMNI_ERR_INVALID_ARG. */
enum { OMNI_METHOD_ALG1 = 0, OMNI_METHOD_DIRECT = 1, OMNI_METHOD_PCG = 2 };
typedef struct {
    size_t struct_size;
    int loop_mode;
    int hist_capacity;
    double* d_hist_eps_R;
    int* d_hist_cg_iters;
    double* d_hist_eps_P;
    double* d_P64_out;
    int* d_status;
    int single_reduction;
} omni_options;
void omni_options_init(omni_options* options);
int omni_solve_ex_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                      const double* d_gx, const double* d_gy, const double* d_gz, const unsigned char* d_mask,
                      const double* d_P_init, double* d_P_out, double tol, int max_outer, int max_cg, int method,
                      const omni_options* options, void* stream, omni_info* info);
int omni_solve_ex_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                      const float* d_gx, const float* d_gy, const float* d_gz, const unsigned char* d_mask,
                      const float* d_P_init, float* d_P_out, double tol, int max_outer, int max_cg, int method,
                      const omni_options* options, void* stream, omni_info* info);

/* ---- Algorithm 1 from a first guess ("initializing with a first guess for the pressure field") -------------
 * omni_solve_* with P^0 = d_P_init (device, [nz][ny][nx]; values at missing cells are ignored; NULL = zeros, i.e.
 * omni_solve_*) instead of P^0 = 0 (:139): the next volume of a time series starts from the previous one's pressure.
 * Same iteration, kernels, stopping rules, status codes and omni_info; the first residual check already counts, so a
 * guess that satisfies eps_R <= tol returns after zero outer iterations.  A constant added to the guess on a connected
 * component is added to the result on it (every row of M - W^n sums to zero, :631). */
int omni_solve_guess_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                         const double* d_gx, const double* d_gy, const double* d_gz, const unsigned char* d_mask,
                         const double* d_P_init, double* d_P_out, double tol, int max_outer, int max_cg, void* stream,
                         omni_info* info);
int omni_solve_guess_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                         const float* d_gx, const float* d_gy, const float* d_gz, const unsigned char* d_mask,
                         const float* d_P_init, float* d_P_out, double tol, int max_outer, int max_cg, void* stream,
                         omni_info* info);

/* ---- fixed point of Algorithm 1 without the boundary iteration (SURVEY.md 8(f) NEXT-2 iii) -----------------------------
 * NOT the paper's iteration: at a fixed point P^{n+1} = P^n of Alg. 1, Eq. 12 reads (M - W^n) P = S,
 * i.e. L P = S with L the symmetric positive semi-definite weighted graph Laplacian of the valid cells
 * ((L P)_C = sum_d v(C+d) (F_a / A_tot) (P_C - P_{C+d}), Eq. 10 :109: w^{n+1} + w^n = F_a / A_tot on a valid link).
 * These entry points run CG on that system directly -- same kernels, same S, same stopping rules, the CG kernels
 * applying L instead of M -- inside the same outer loop, which here is an fp64 iterative refinement (the true
 * residual S - L P is re-evaluated from the fp64 master pressure, eps_R of Eq. 41, and the CG restarted on it).
 * It returns the field Alg. 1 converges to (zero mean on every connected component) in O(n) instead of O(n^2) CG
 * iterations for an n-cell-wide domain.  Typical caps: max_outer 10, max_cg a few thousand.  d_P_init (device,
 * [nz][ny][nx], may be NULL = zeros) is the first guess; the returned field differs from the P_init = 0
 * one by a constant per connected component.  Other arguments, layout, ownership, status codes and omni_info as
 * omni_solve_*. */
int omni_solve_direct_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                          const double* d_gx, const double* d_gy, const double* d_gz, const unsigned char* d_mask,
                          const double* d_P_init, double* d_P_out, double tol, int max_outer, int max_cg, void* stream,
                          omni_info* info);
int omni_solve_direct_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                          const float* d_gx, const float* d_gy, const float* d_gz, const unsigned char* d_mask,
                          const float* d_P_init, float* d_P_out, double tol, int max_outer, int max_cg, void* stream,
                          omni_info* info);

/* omni_solve_direct_* with a cascadic first guess: the same system is first solved on up to `levels` grids coarsened by
 * 2 along every axis (a coarse cell is valid iff one of its children is; its gradient is the mean over the valid
 * children; coarsening stops before an axis would drop below 8 cells), coarsest first, each level's pressure being the
 * first guess of the next finer one.  The coarse levels only produce guesses: tol, max_outer, max_cg apply to every
 * level, info and the returned status are those of the finest level, whose solve alone decides the answer (the same
 * field as omni_solve_direct_* up to tol and a constant per connected component).  levels = 0 is omni_solve_direct_*. */
int omni_solve_cascade_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                           const double* d_gx, const double* d_gy, const double* d_gz, const unsigned char* d_mask,
                           double* d_P_out, double tol, int max_outer, int max_cg, int levels, void* stream, omni_info* info);
int omni_solve_cascade_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                           const float* d_gx, const float* d_gy, const float* d_gz, const unsigned char* d_mask,
                           float* d_P_out, double tol, int max_outer, int max_cg, int levels, void* stream, omni_info* info);

/* omni_solve_direct_* with the CG PRECONDITIONED by one geometric-multigrid V-cycle (SURVEY.md 8(f) NEXT-2 ii; reading
 * R-P1 of DESIGN.md; not the paper's iteration, which names only "CG").  Same system L P = S, same outer
 * loop (fp64 refinement: eps_R of Eq. 41 :442 re-evaluated from the fp64 master pressure, CG restarted on it), same
 * stopping rules, status codes and omni_info; cg_iters_total counts preconditioned iterations.  The V-cycle: levels
 * halving every axis that still has >= 8 cells and whose link weight is >= 0.7 of the largest such weight
 * (semi-coarsening: anisotropic spacings cost no extra iterations; a coarse cell is valid iff one of its children is), link weights
 * w_{l+1}[a] = w_l[a] 2^m (1/4 along halved axes), restriction = sum over the children, prolongation = its transpose,
 * damped Jacobi (omega = 0.8), 2 sweeps before and after the coarse-grid correction, 8 on the coarsest level.  The
 * iteration count is nearly independent of the grid size (about 10 to eps_R <= 1e-5, 15 to 1e-8) at about 4 times the
 * memory traffic of a plain CG iteration.  _f32: an inner solve also returns to the fp64 refinement once ||r|| <= 1e-2
 * ||r0|| (fp32 vectors cannot resolve more digits of one correction on 1000-cell-wide grids; 3 outer iterations of 3-5
 * preconditioned iterations reach 1e-5).  Typical caps: max_outer 10-20, max_cg 200.  Always runs under the CUDA graph
 * (omni_set_loop_mode does not apply).  Extra device memory: about 2.5 vectors, from the library's pool.
 * d_P_init: first guess or NULL.  The returned field has zero mean per connected component when d_P_init is NULL. */
int omni_solve_pcg_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                       const double* d_gx, const double* d_gy, const double* d_gz, const unsigned char* d_mask,
                       const double* d_P_init, double* d_P_out, double tol, int max_outer, int max_cg, void* stream,
                       omni_info* info);
int omni_solve_pcg_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                       const float* d_gx, const float* d_gy, const float* d_gz, const unsigned char* d_mask,
                       const float* d_P_init, float* d_P_out, double tol, int max_outer, int max_cg, void* stream,
                       omni_info* info);

/* The two combined: nb snapshots on one mask (arguments as omni_solve_batch2d_*), inner systems L P = S. */
int omni_solve_direct_batch2d_f64(int nx, int ny, int nb, double dx, double dy, const double* d_gx, const double* d_gy,
                                  const unsigned char* d_mask2d, const double* d_P_init, double* d_P_out, double tol,
                                  int max_outer, int max_cg, void* stream, omni_info* info);
int omni_solve_direct_batch2d_f32(int nx, int ny, int nb, double dx, double dy, const float* d_gx, const float* d_gy,
                                  const unsigned char* d_mask2d, const float* d_P_init, float* d_P_out, double tol,
                                  int max_outer, int max_cg, void* stream, omni_info* info);

/* ... and with the multigrid-preconditioned CG of omni_solve_pcg_* (the snapshot axis carries no links and is never
 * coarsened; joint CG scalars and stopping tests over the stack, as for omni_solve_batch2d_*). */
int omni_solve_pcg_batch2d_f64(int nx, int ny, int nb, double dx, double dy, const double* d_gx, const double* d_gy,
                               const unsigned char* d_mask2d, const double* d_P_init, double* d_P_out, double tol,
                               int max_outer, int max_cg, void* stream, omni_info* info);
int omni_solve_pcg_batch2d_f32(int nx, int ny, int nb, double dx, double dy, const float* d_gx, const float* d_gy,
                               const unsigned char* d_mask2d, const float* d_P_init, float* d_P_out, double tol,
                               int max_outer, int max_cg, void* stream, omni_info* info);

/* ---- batched 2D snapshots with an optional first guess (SURVEY.md 8(f) NEXT-1; time-resolved PIV: PAPER.md:365, :503) ----
 * nb independent 2D gradient fields [nb][ny][nx] on ONE mask [ny][nx] (NULL = all valid) are stacked and solved as one
 * block-diagonal system with the 2D scheme: stencil codes are built once, every stencil sweep serves all snapshots,
 * and the tile pipeline marches through the snapshots like through the planes of a volume.  The CG scalars and eps_R
 * (Eq. 41) are those of the stacked system: on return ||r|| <= tol ||S|| holds for the STACK, which bounds every
 * snapshot's own residual by ||r_b|| <= tol ||S||, i.e. eps_R,b <= tol ||S|| / ||S_b|| -- about tol sqrt(nb) for
 * snapshots of similar strength, but a snapshot whose source is much weaker than the others' can sit above tol by that
 * ratio (solve such a series one by one, or tighten tol).  Each converged P_b equals the single-snapshot result to
 * that accuracy.  d_P_init [nb][ny][nx] (may be NULL = zeros) is the
 * first guess P^0, e.g. the previous time step's pressure ("zero ... or any other arbitrary value");
 * its values at missing cells are ignored.  Everything else as omni_solve_*. */
int omni_solve_batch2d_f64(int nx, int ny, int nb, double dx, double dy, const double* d_gx, const double* d_gy,
                           const unsigned char* d_mask2d, const double* d_P_init, double* d_P_out, double tol,
                           int max_outer, int max_cg, void* stream, omni_info* info);
int omni_solve_batch2d_f32(int nx, int ny, int nb, double dx, double dy, const float* d_gx, const float* d_gy,
                           const unsigned char* d_mask2d, const float* d_P_init, float* d_P_out, double tol,
                           int max_outer, int max_cg, void* stream, omni_info* info);

/* ---- one solve on several ranks: z-slab sharding -------------------------------------
 * The paper stops at one 16 GB GPU and names memory as the limit.  Here the grid is cut along z:
 * rank s of nranks owns the planes [z0, z1) and works on the WINDOW [zlo, zhi) = its planes plus up to two halo planes
 * per side (the stencil codes of Eq. 25 :266 read validity two planes away); omni_slab_plan (host only) returns both
 * ranges: balanced, the first nz % nranks ranks own one plane more.  Per CG iteration each rank exchanges one halo
 * plane of p and one of r with each neighbour and two scalars are all-reduced; per outer iteration the halo planes of
 * delta, P and r and the four scalars of the boundary update.  Same kernels, same iteration, same stopping rules as
 * omni_solve_* (method OMNI_METHOD_ALG1) / omni_solve_direct_* (OMNI_METHOD_DIRECT); the reductions add per-rank
 * totals, so results equal the single-device ones to rounding and all ranks take identical decisions.
 *
 * omni_solve_slab_*: nlocal ranks of the solve live in THIS process on the current device; h_ranks[nlocal] are their
 * rank numbers; h_gx / h_gy / h_gz / h_mask / h_P_out are HOST arrays of nlocal DEVICE pointers to each rank's window
 * ([zhi - zlo][ny][nx], x fastest; h_mask may be NULL, or hold NULL entries = all valid).  P_out is written on the whole
 * window; the owned planes are the result (halo planes hold the neighbours' values of an earlier iteration).
 *   comm == NULL : all ranks are local (nlocal == nranks, h_ranks = 0..nranks-1): halo planes by device copies, the
 *                  scalars by a summing kernel -- the sharded algorithm on one GPU (tests, grids split for other reasons)
 *   comm != NULL : one rank per process (nlocal == 1), `comm` from omni_slab_comm_create: NCCL send / recv of the halo
 *                  planes and ncclAllReduce of the scalars over NVLink.  libnccl.so.2 is loaded at run time; without it
 *                  these calls return OMNI_ERR_CUDA.  omni_slab_unique_id (on rank 0) makes the 128-byte id every rank
 *                  passes to omni_slab_comm_create (ship it with any host-side broadcast).
 * nz >= nranks, nz >= 2 (3D only).  The loop is driven from the host (one synchronisation per outer iteration and per
 * 16 CG iterations), so the call always synchronises; info may be NULL.  Status codes as omni_solve_*. */
int omni_slab_plan(int nz, int nranks, int rank, int* z0, int* z1, int* zlo, int* zhi);
int omni_slab_unique_id(char* h_id128);
int omni_slab_comm_create(int rank, int nranks, const char* h_id128, void** comm);
void omni_slab_comm_destroy(void* comm);
int omni_solve_slab_f64(int nx, int ny, int nz, double dx, double dy, double dz, int nlocal, const int* h_ranks,
                        const double* const* h_gx, const double* const* h_gy, const double* const* h_gz,
                        const unsigned char* const* h_mask, double* const* h_P_out, double tol, int max_outer, int max_cg,
                        int method, int nranks, void* comm, void* stream, omni_info* info);
int omni_solve_slab_f32(int nx, int ny, int nz, double dx, double dy, double dz, int nlocal, const int* h_ranks,
                        const float* const* h_gx, const float* const* h_gy, const float* const* h_gz,
                        const unsigned char* const* h_mask, float* const* h_P_out, double tol, int max_outer, int max_cg,
                        int method, int nranks, void* comm, void* stream, omni_info* info);

/* ---- upstream of the path: the pressure gradient from a velocity field, Eq. 1 ----
 *   g = f(u) = -rho (du/dt + (u . grad) u) + mu lap u
 * with second-order central differences on the cell grid.  The paper does not fix the discretisation (reading R-V1,
 * DESIGN.md 13): a cell whose 2*naxes-neighbour stencil touches a missing cell (outside the box, mask == 0, a NaN
 * velocity component) gets NaN in every output component, which omni_solve_* treats as missing (Eq. 13 :176) -- so the
 * outputs can be fed to the solver with the same mask.  d_u, d_v, d_w: device, [nz][ny][nx] (d_w NULL iff nz == 1);
 * d_dudt, d_dvdt, d_dwdt: optional local accelerations (all NULL = steady flow); d_g*: device outputs (d_gz NULL iff
 * nz == 1).  Asynchronous on `stream`; returns an omni_status. */
int omni_velocity_source_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                             const double* d_u, const double* d_v, const double* d_w,
                             const double* d_dudt, const double* d_dvdt, const double* d_dwdt,
                             const unsigned char* d_mask, double rho, double mu,
                             double* d_gx, double* d_gy, double* d_gz, void* stream);
int omni_velocity_source_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                             const float* d_u, const float* d_v, const float* d_w,
                             const float* d_dudt, const float* d_dvdt, const float* d_dwdt,
                             const unsigned char* d_mask, double rho, double mu,
                             float* d_gx, float* d_gy, float* d_gz, void* stream);

/* ---- upstream, time-averaged flows: RANS source fields --------------------------------------
 * Incompressible RANS, viscous terms dropped, Eq. 42:
 *   f_i = -rho ( ubar_j d ubar_i / d x_j + d (u'_i u'_j) / d x_j )
 * d_u, d_v, d_w: mean velocity, device, [nz][ny][nx] (d_w NULL iff nz == 1).  h_stress: HOST array of 3 (nz == 1: xx,
 * yy, xy) or 6 (xx, yy, zz, xy, xz, yz) DEVICE pointers to the Reynolds stresses u'_i u'_j, or NULL / all entries NULL
 * for none.  d_f*: device outputs (d_fz NULL iff nz == 1).  Discretisation and missing cells as in
 * omni_velocity_source_* (reading R-V1): second-order central differences; a cell whose stencil touches a missing cell
 * (outside the box, mask == 0, NaN in any input) gets NaN in every component.  Asynchronous on `stream`; returns an
 * omni_status; invalid sizes / spacings / a partly given stress list: OMNI_ERR_INVALID_ARG, nothing enqueued. */
int omni_rans_source_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                         const double* d_u, const double* d_v, const double* d_w, const double* const* h_stress,
                         const unsigned char* d_mask, double rho, double* d_fx, double* d_fy, double* d_fz, void* stream);
int omni_rans_source_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                         const float* d_u, const float* d_v, const float* d_w, const float* const* h_stress,
                         const unsigned char* d_mask, double rho, float* d_fx, float* d_fy, float* d_fz, void* stream);

/* Compressible RANS for an adiabatic ideal gas with negligible density fluctuations, Eq. 43-44:
 *   T / T_inf = 1 + (gamma - 1)/2 M_inf^2 (1 - V^2 / V_inf^2),      uu_ij = ubar_i ubar_j + u'_i u'_j,
 *   (delta_ij + uu_ij / (R T)) g_j = -(1 / (R T)) ( d uu_ij / d x_j - (uu_ij / T) d T / d x_j ),
 * solved cell by cell for g = grad ln(P / P_inf); integrating g with omni_solve_* gives ln(P / P_inf) (:547).
 * rgas_t_inf = R T_inf (the only way the gas constant and T_inf enter); gamma > 1, v_inf > 0, rgas_t_inf > 0.
 * Arrays, h_stress, discretisation, missing cells and error behaviour as for omni_rans_source_*. */
int omni_compressible_rans_source_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                                      const double* d_u, const double* d_v, const double* d_w,
                                      const double* const* h_stress, const unsigned char* d_mask,
                                      double gamma, double mach_inf, double v_inf, double rgas_t_inf,
                                      double* d_gx, double* d_gy, double* d_gz, void* stream);
int omni_compressible_rans_source_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                                      const float* d_u, const float* d_v, const float* d_w,
                                      const float* const* h_stress, const unsigned char* d_mask,
                                      double gamma, double mach_inf, double v_inf, double rgas_t_inf,
                                      float* d_gx, float* d_gy, float* d_gz, void* stream);

/* ---- single steps of the path (each runs the same device code the solve runs; used by the parity tests) ----------
 * a0  geometry constants (host only, no device needed).  out[0..2] = face totals F_x,F_y,F_z (Eq. 5 :75 / Eq. 23 :258),
 *     out[3] = A_tot (Eq. 8 :94 / Eq. 24 :262), out[4..12] = c_jk row-major 3x3 (Eq. 17 :207 / Eq. 32-35 :314-326 /
 *     parallel-rectangle measure for general spacing, A7).  2D: every entry with a z index is 0. */
int omni_constants(int nx, int ny, int nz, double dx, double dy, double dz, double* h_out13);

/* a1+a2  source vector S (last sum of Eq. 9 :100; Eq. 49-50 :656-662), 0 at missing cells; *h_norm_S (host, may be
 *     NULL) receives ||S||_2.  Synchronises `stream`. */
int omni_source_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                    const double* d_gx, const double* d_gy, const double* d_gz, const unsigned char* d_mask,
                    double* d_S_out, double* h_norm_S, void* stream);
int omni_source_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                    const float* d_gx, const float* d_gy, const float* d_gz, const unsigned char* d_mask,
                    float* d_S_out, double* h_norm_S, void* stream);

/* a1+a2 WITHOUT ANY ALLOCATION -- for callers that cannot call cudaMalloc (code under CUDA-graph stream capture, tight
 *     serving loops, harnesses that forbid it).  Same S (last sum of Eq. 9 :100, 0 at missing cells; missing = outside
 *     the box, mask == 0 or NaN in a used component, Eq. 13 :176) as omni_source_*, from ONE kernel that evaluates the
 *     validity of a cell and its neighbours on the fly and writes straight to d_S_out; d_norm_S (DEVICE, one double, may
 *     be NULL) receives ||S||_2.  The call enqueues one 64-byte memset and one kernel on `stream`, never synchronises,
 *     and calls no cudaMalloc / cudaFree / pool or other allocating routine.  The only scratch (one reduction slot per
 *     4096 cells, a ticket) is a fixed 256 KiB static __device__ array that every GPU loading the library holds until the
 *     process exits; hence the limit nx*ny*nz <= omni_source_noalloc_max_cells() = 134 184 960 (500^3 fits): larger grids
 *     return OMNI_ERR_TOO_LARGE with nothing enqueued.  ALL calls on a device share that array: two calls that overlap
 *     on the GPU (different streams, or graph branches) race on it and give wrong norms -- serialise them; S itself does
 *     not go through the scratch.  Other arguments and errors as omni_source_*. */
int omni_source_noalloc_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                            const double* d_gx, const double* d_gy, const double* d_gz, const unsigned char* d_mask,
                            double* d_S_out, double* d_norm_S, void* stream);
int omni_source_noalloc_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                            const float* d_gx, const float* d_gy, const float* d_gz, const unsigned char* d_mask,
                            float* d_S_out, double* d_norm_S, void* stream);
long long omni_source_noalloc_max_cells(void);

/* a1+a4  q = [W^{n+1}] p = M p with M = I - W1_off (Eq. 9 rearranged, A1), through the CG operator kernel
 *     (K4's recomputation path); validity from d_mask only (NULL = full box); q = 0 at missing cells; values of p at
 *     missing cells are ignored.  *h_pq (host, may be NULL) receives p.Mp over valid cells.  Synchronises. */
int omni_apply_M_f64(int nx, int ny, int nz, double dx, double dy, double dz, const unsigned char* d_mask,
                     const double* d_p, double* d_q, double* h_pq, void* stream);
int omni_apply_M_f32(int nx, int ny, int nz, double dx, double dy, double dz, const unsigned char* d_mask,
                     const float* d_p, float* d_q, double* h_pq, void* stream);

/* a3  outer residual r = S + [W^n]P - [W^{n+1}]P = S - L P (Eq. 12 :119, Eq. 41 :442) for a given field P (values at
 *     missing cells ignored), r = 0 at missing cells; *h_eps_R (host, may be NULL) = ||r|| / ||S||.  Synchronises.
 *     _f32: g, S and r are fp32, P is fp64 (the fp32 solve keeps its master pressure in fp64, A9). */
int omni_residual_f64(int nx, int ny, int nz, double dx, double dy, double dz,
                      const double* d_gx, const double* d_gy, const double* d_gz, const unsigned char* d_mask,
                      const double* d_P, double* d_r_out, double* h_eps_R, void* stream);
int omni_residual_f32(int nx, int ny, int nz, double dx, double dy, double dz,
                      const float* d_gx, const float* d_gy, const float* d_gz, const unsigned char* d_mask,
                      const double* d_P, float* d_r_out, double* h_eps_R, void* stream);

/* ---- misc ---------------------------------------------------------------------------------------------------- */
/* Kernel launches issued by this library since the last reset (counts launches on any thread; for bench.py). */
long long omni_launch_count(int reset);
/* How the iteration (Alg. 1) is driven; every mode runs the same per-cell arithmetic.
 *   0  automatic (default): mode 5 where the grid fits it with r in shared memory, else mode 3 for grids of up to
 *      1.5 M padded cells, mode 2 above
 *   1  host-driven loop that synchronises once per outer iteration (debug / per-kernel profiling)
 *   2  CUDA graph with device-side conditional WHILE nodes around the tile kernels K2 / K3 / K4
 *   3  one persistent cooperative kernel: phases separated by grid barriers that double as the reductions
 *      (state is L2-resident; falls back to mode 2 if the device cannot co-schedule the grid)
 *   4  the whole iteration as ONE cooperative launch of the tile kernels' TMA pipeline (one column per CTA, the same
 *      grid barriers between the K2 / K3 / K4 phases); correct and deterministic, measured slower than mode 2 at every
 *      size (profiles/r2_loop_and_rows.md), never chosen automatically; falls back to mode 2 if its grid does not fit
 *   5  mode 3 with the CG vectors resident on the SMs for the whole inner solve: every CTA owns a box of grid rows, p of
 *      the box and its halo in shared memory, r and delta in the SM's tensor memory (tcgen05.ld / st as a thread-private
 *      scratchpad), else in shared memory or, where p alone fills it, behind L2;
 *      per CG iteration only the halo rows of r travel, as self-validating messages, and the two grid barriers carry
 *      nothing but the reduction (no fence).  For grids whose p fits the shared memory of the SMs (on a 148-SM B200 up to about
 *      5 M cells in fp32, 2.5 M in fp64: 2048^2, 160^3 / 1448 x 1024, 136^3) and whose rows are at most 2048 (fp32) / 1024
 *      (fp64) cells long; falls back to mode 3 where the grid does not fit.  Uses the workspace's two p vectors as
 *      message buffer.
 * The environment variable OMNI_PERSIST_MAX_CELLS overrides the threshold between modes 3 and 2, OMNI_RESIDENT=0 keeps mode
 * 5 out of the automatic choice, OMNI_RESIDENT_TMEM=0 keeps it out of tensor memory.  Modes 1 and 2 give bit-identical results; modes 3, 4 and 5 sum their reductions in a
 * different (fixed) order.  Returns the previous mode; other values are ignored. */
int omni_set_loop_mode(int mode);
/* The box decomposition loop mode 5 would use for this grid (host only, no CUDA call): 1 and
 * out[0..12] = { gy, gz (boxes along y and z, gy * gz CTAs), ly, lz (rows and planes of the largest box), dynamic shared
 * memory in bytes, rows per thread, r does not fit beside p (0 / 1), delta in shared memory, q in shared memory, weights of
 * the y and z cuts, padded row pitch in cells, r and delta in tensor memory (0 / 1) }; 0 if the grid does not fit the SMs (mode 5 then falls back to mode 3);
 * OMNI_ERR_INVALID_ARG for bad arguments.  elem_size 4 or 8, nsm = SMs to plan for, lop = 1 for the operator L of
 * omni_solve_direct.  omni_resident_split(n, parts, i, wface) = first cell of part i when an axis of n cells is cut into
 * `parts` boxes with that weight (i = parts: n). */
int omni_resident_plan(int nx, int ny, int nz, int elem_size, int nsm, int lop, int* out);
int omni_resident_split(int n, int parts, int i, int wface);
/* Convergence history (the momentum residual of Eq. 41, plotted in Fig. 10-13): registers a caller-owned
 * DEVICE buffer of `capacity` doubles that every solve enqueued afterwards fills on the device -- entry i = eps_R =
 * ||S - L P^i|| / ||S|| at the i-th outer residual check (i = 0: the first guess), written by the kernel that evaluates the
 * check; info.outer_iters + 1 entries for a completed solve, the first `capacity` of them if there are more.  d_cg_iters
 * (device, `capacity` ints, may be NULL) receives next to it the CG iterations of the outer iteration that led to the
 * check (0 for i = 0) -- the quantity behind the falling cost per iteration of Fig. 13 (:489).  No host
 * synchronisation is added.  (NULL, NULL, 0) switches it off.  Process-wide DEFAULT (like omni_set_loop_mode; the per-call form is
 * omni_options of omni_solve_ex_*, which also offers eps_P of Eq. 40); a cascade solve
 * leaves the history of its finest level.  Returns OMNI_OK, or OMNI_ERR_INVALID_ARG for capacity < 0 or a NULL d_hist
 * with capacity > 0 or with d_cg_iters given. */
int omni_set_history(double* d_hist, int* d_cg_iters, int capacity);
/* Workspace of the non-_ws entry points comes from a library-owned stream-ordered memory pool (one per device) that
 * keeps freed blocks mapped between calls; this returns the unused memory to the driver. */
void omni_release_memory(void);
/* Per-kernel timing of the host-driven loop (loop mode 1 only): when enabled, CUDA events bracket every launch of
 * K2 (outer boundary update), K3 (p update + operator + p.Mp) and K4 (operator recomputed + axpys + r.r) on `stream`;
 * launches that found the device loop flag cleared (no work) are left out.  omni_profile_read returns the summed
 * milliseconds and launch counts, index 0/1/2 = K2/K3/K4 (host arrays of 3, either may be NULL). */
int omni_profile_enable(int on);          /* returns the previous setting */
void omni_profile_read(double* h_ms3, long long* h_count3, int reset);
const char* omni_status_string(int status);
int omni_version(void);                  /* 100 * major + minor; 101 added the _guess, _rans_source and history entry points, 102 omni_solve_pcg_*, 103 omni_solve_ex_* / omni_options, 104 omni_solve_slab_*, 105 omni_source_noalloc_*, 106 omni_solve_pcg_batch2d_*, 107 loop mode 5, omni_resident_plan */

#ifdef __cplusplus
}
#endif
#endif /* OMNI_H */
