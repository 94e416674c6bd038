/* omni_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle of the matrix-based omnidirectional pressure
 * integration of Zigunov & Charonko (arXiv 2311.16935, "the paper"; citations are
 * PAPER.md:<line>).  Written from the paper only.  It shares no code, header,
 * table or constant generator with the CUDA path under paper_2311_16935_b200/ and
 * neither side includes or imports the other.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may build, load or call it.
 *
 * Design on purpose different from the GPU path: every weight of Eq. 10 is STORED
 * per cell (the paper's own layout, 6+6+1 fields), the operators are
 * explicit loops over the stored weights, the inner solver is the textbook CG
 * recurrence solving Eq. 12 for P^{n+1} directly (warm start from P^n, :489).
 *
 * Conventions:
 *   layout x-fastest: idx = i + nx*(j + ny*k);  nz == 1 selects the 2D scheme.
 *   directions d = 0..5 = E(+x) W(-x) N(+y) S(-y) F(+z) B(-z)     (:103)
 *   a cell is missing if outside the box, mask==0, or any used g is NaN (Eq. 13 :176)
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): Table 1 (:637-650), Eq. 5-7,
 * Eq. 17, Eq. 34-35, Eq. 49-50, the A_tot sum rule (:631), dense L^+ S fixed point,
 * dense LU inner solve, exactness on quadratics, 2nd-order refinement, Monte-Carlo
 * ray counts; oracle_solve_direct: dense pinv(L) S and the dense textbook CG iterates.
 * The per-iteration trajectory P^n (finite n) is "parity unpinned" by
 * the paper (it prints no intermediate values); it is pinned only through the pins
 * of every operator that generates it.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (no -ffast-math).
 * OpenMP is used on the grid loops only.  Dot products accumulate each x-row in
 * long double and add the row sums sequentially: results do not depend on threads.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long long i64;

/* grids smaller than this run the loops serially (fork/join would dominate the tiny pin cases) */
#define OMP_MIN_N 32768

/* ------------------------------------------------------------------ constants */

/* Legendre polynomial P_n(x) and derivative, for Gauss-Legendre nodes. */
static void legendre(int n, double x, double *p, double *dp)
{
    double p0 = 1.0, p1 = x;
    for (int m = 2; m <= n; ++m) {
        double p2 = ((2.0 * m - 1.0) * x * p1 - (m - 1.0) * p0) / m;
        p0 = p1; p1 = p2;
    }
    *p = p1;
    *dp = n * (x * p1 - p0) / (x * x - 1.0);
}

static void gauss_legendre(int n, double *x, double *w)
{
    for (int i = 0; i < n; ++i) {
        double z = cos(M_PI * (i + 0.75) / (n + 0.5)), p, dp;
        for (int it = 0; it < 100; ++it) {
            legendre(n, z, &p, &dp);
            double dz = p / dp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        legendre(n, z, &p, &dp);
        x[i] = z;
        w[i] = 2.0 / ((1.0 - z * z) * dp * dp);
    }
}

/* Far-face constant c_aa for general spacing (reading A7; PAPER.md:273,
 * Fig. 5b; Eq. 26 :275 is garbled and not transcribed).  Rays entering cell C through
 * its face a (area db*dc) came through cell Q = C + e_a; c_aa is the measure
 * (projected area integrated over direction, as in Eq. 22 :253) of those that entered
 * Q through its far face, a parallel db x dc rectangle at distance da:
 *   c_aa = 4 * int_0^db int_0^dc (db-u)(dc-v) da^2 / (u^2+v^2+da^2)^2 dv du.
 * Composite Gauss-Legendre: 16 points on each of 24 dyadic panels [L 2^-m, L 2^-(m-1)] per axis, refined
 * towards 0 where the integrand peaks (width ~ da), so strongly anisotropic spacings keep ~1e-13. */
static double far_face_constant(double da, double db, double dc)
{
    enum { NP = 24, NG = 16 };
    double gx[NG], gw[NG];
    gauss_legendre(NG, gx, gw);
    double lo[NP], hi[NP];                     /* panel bounds as fractions of the interval */
    for (int m = 0; m < NP; ++m) {
        hi[m] = ldexp(1.0, -m);
        lo[m] = (m == NP - 1) ? 0.0 : ldexp(1.0, -(m + 1));
    }
    long double acc = 0.0L;
    for (int pu = 0; pu < NP; ++pu)
        for (int iu = 0; iu < NG; ++iu) {
            double u = (lo[pu] + 0.5 * (gx[iu] + 1.0) * (hi[pu] - lo[pu])) * db;
            double wu = 0.5 * gw[iu] * (hi[pu] - lo[pu]) * db;
            for (int pv = 0; pv < NP; ++pv)
                for (int iv = 0; iv < NG; ++iv) {
                    double v = (lo[pv] + 0.5 * (gx[iv] + 1.0) * (hi[pv] - lo[pv])) * dc;
                    double wv = 0.5 * gw[iv] * (hi[pv] - lo[pv]) * dc;
                    double r2 = u * u + v * v + da * da;
                    acc += (long double)(wu * wv * (db - u) * (dc - v) * da * da / (r2 * r2));
                }
        }
    return (double)(4.0L * acc);
}

/* out[0..2]  = F_x, F_y, F_z      face totals (Eq. 5 :75 / Eq. 23 :258)
 * out[3]     = A_tot              (Eq. 8 :94 / Eq. 24 :262)
 * out[4..12] = c[a][b] row-major  (Eq. 17 :207-212 / Eq. 32-35 :314-326 / A7)
 * nz == 1 -> 2D scheme: F_z = 0 and every c with a z index = 0. */
/* Batched 2D snapshots (SURVEY NEXT-1; PAPER.md:365 "26 Taylor vortex snapshots", :503): nb independent 2D fields on
 * one mask are stacked along z and solved as ONE block-diagonal system with the 2D constants (scheme2d = 1 below although
 * nz > 1).  Every constant with a z index is then 0, so all weights across planes vanish (Eq. 16/18 with c_xz = c_yz =
 * c_zz = 0, F_z = 0) and no other routine needs to know.  The choices "2D scheme on a stack" and "inner systems L P = S"
 * are explicit arguments of the internal routines (constants_impl, weights_impl, solve_impl): no hidden state. */
static void constants_impl(int scheme2d, double dx, double dy, double dz, double *out);

void oracle_constants(int nx, int ny, int nz, double dx, double dy, double dz, double *out)
{
    (void)nx; (void)ny;
    constants_impl(nz == 1, dx, dy, dz, out);
}

static void constants_impl(int scheme2d, double dx, double dy, double dz, double *out)
{
    double F[3], c[3][3], Atot;
    memset(c, 0, sizeof c);
    if (scheme2d) {
        double dd = sqrt(dx * dx + dy * dy);          /* :214 */
        F[0] = 2.0 * dy; F[1] = 2.0 * dx; F[2] = 0.0; /* Eq. 5 :75, :96 */
        Atot = 4.0 * (dx + dy);                       /* Eq. 8 :94 */
        c[0][0] = 2.0 * (dd - dx);                    /* Eq. 17 */
        c[1][1] = 2.0 * (dd - dy);
        c[0][1] = c[1][0] = dx + dy - dd;
    } else {
        F[0] = M_PI * dy * dz; F[1] = M_PI * dx * dz; F[2] = M_PI * dx * dy; /* Eq. 23 :258-260 */
        Atot = 2.0 * M_PI * (dx * dy + dx * dz + dy * dz);                  /* Eq. 24 :262 */
        if (dx == dy && dy == dz) {
            double s2 = sqrt(2.0), D2 = dx * dx;
            double cjj = D2 * (log(4.0 / 3.0) - s2 * atan(s2) + 0.5 * s2 * atan(10.0 * s2 / 23.0)
                               + M_PI * (s2 - 1.0));                         /* Eq. 32 :314 */
            double cjk = D2 * (0.5 * M_PI - 0.25 * log(4.0 / 3.0) - 0.25 * s2 * atan(10.0 * s2 / 23.0)
                               - 0.5 * s2 * atan(s2));                       /* Eq. 33 :317 */
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) c[a][b] = (a == b) ? cjj : cjk;
        } else {
            double d[3] = { dx, dy, dz };
            double s[3];
            for (int a = 0; a < 3; ++a) {
                c[a][a] = far_face_constant(d[a], d[(a + 1) % 3], d[(a + 2) % 3]);
                s[a] = 0.5 * (F[a] - c[a][a]);  /* = c_ab + c_ac: all rays through face a sum to F_a (Eq. 23, 25) */
            }
            /* c_ab = c_ba (:304) closes the three sum rules */
            c[0][1] = c[1][0] = 0.5 * (s[0] + s[1] - s[2]);
            c[0][2] = c[2][0] = 0.5 * (s[0] + s[2] - s[1]);
            c[1][2] = c[2][1] = 0.5 * (s[1] + s[2] - s[0]);
        }
    }
    out[0] = F[0]; out[1] = F[1]; out[2] = F[2]; out[3] = Atot;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) out[4 + 3 * a + b] = c[a][b];
}

/* exposed for the pin test of the quadrature at dx=dy=dz against Eq. 34 */
double oracle_far_face_constant(double da, double db, double dc) { return far_face_constant(da, db, dc); }

/* ------------------------------------------------------------------ validity (Eq. 13 :176) */

void oracle_validity(int nx, int ny, int nz, const double *gx, const double *gy, const double *gz,
                     const unsigned char *mask, unsigned char *v)
{
    i64 N = (i64)nx * ny * nz;
#pragma omp parallel for if (N > OMP_MIN_N)
    for (i64 c = 0; c < N; ++c) {
        int ok = (mask == NULL) || (mask[c] != 0);
        if (isnan(gx[c]) || isnan(gy[c])) ok = 0;
        if (nz > 1 && gz != NULL && isnan(gz[c])) ok = 0;
        v[c] = (unsigned char)ok;
    }
}

static const int DIRV[6][3] = { { 1, 0, 0 }, { -1, 0, 0 }, { 0, 1, 0 }, { 0, -1, 0 }, { 0, 0, 1 }, { 0, 0, -1 } };

/* b~ of Eq. 13: 1 iff (i,j,k) is inside the box and has data */
static inline int val(const unsigned char *v, int nx, int ny, int nz, int i, int j, int k)
{
    if (i < 0 || j < 0 || k < 0 || i >= nx || j >= ny || k >= nz) return 0;
    return v[i + (i64)nx * (j + (i64)ny * k)];
}

/* ------------------------------------------------------------------ weights (Eq. 10, 11, 15, 16, 18-20, 25) */

/* w1[d*N + c] = w_d^{n+1}(c), w0[d*N + c] = w_d^{n}(c), w0C[c] = w_C^{n}(c); w_C^{n+1} = 0 (Eq. 11 :113).
 * Missing cells get all-zero weights. */
static void weights_impl(int scheme2d, int nx, int ny, int nz, double dx, double dy, double dz, const unsigned char *v,
                         double *w1, double *w0, double *w0C);

void oracle_weights(int nx, int ny, int nz, double dx, double dy, double dz, const unsigned char *v,
                    double *w1, double *w0, double *w0C)
{
    weights_impl(nz == 1, nx, ny, nz, dx, dy, dz, v, w1, w0, w0C);
}

static void weights_impl(int scheme2d, int nx, int ny, int nz, double dx, double dy, double dz, const unsigned char *v,
                         double *w1, double *w0, double *w0C)
{
    double K[13];
    constants_impl(scheme2d, dx, dy, dz, K);
    const double *F = K, Atot = K[3], *c = K + 4;
    i64 N = (i64)nx * ny * nz;
#pragma omp parallel for collapse(2) if (N > OMP_MIN_N)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                i64 C = i + (i64)nx * (j + (i64)ny * k);
                double AC = 0.0;
                for (int d = 0; d < 6; ++d) {
                    double A1 = 0.0, A0 = 0.0;
                    int a = d / 2;
                    int qi = i + DIRV[d][0], qj = j + DIRV[d][1], qk = k + DIRV[d][2];
                    if (v[C]) {
                        if (!val(v, nx, ny, nz, qi, qj, qk)) {
                            AC += F[a];              /* Eq. 15 :197 (3D: same form with Eq. 23 totals, reading A6) */
                        } else {
                            /* far cell Q+d, and the four side cells Q +/- e_b (b != a) (Eq. 16/18 :202/:218, Eq. 25 :266) */
                            int bt = val(v, nx, ny, nz, qi + DIRV[d][0], qj + DIRV[d][1], qk + DIRV[d][2]);
                            A1 += c[3 * a + a] * bt;
                            A0 += c[3 * a + a] * (1 - bt);
                            for (int b = 0; b < 3; ++b) {
                                if (b == a) continue;
                                for (int sgn = 0; sgn < 2; ++sgn) {
                                    const int *e = DIRV[2 * b + sgn];
                                    int bs = val(v, nx, ny, nz, qi + e[0], qj + e[1], qk + e[2]);
                                    A1 += c[3 * a + b] * bs;
                                    A0 += c[3 * a + b] * (1 - bs);
                                }
                            }
                        }
                    }
                    w1[(i64)d * N + C] = A1 / Atot;  /* Eq. 10 :109 */
                    w0[(i64)d * N + C] = A0 / Atot;
                }
                w0C[C] = AC / Atot;
            }
}

/* ------------------------------------------------------------------ source vector (last sum of Eq. 9 :100) */

/* S_C = - sum_j Delta_j (w_j^{n+1} + w_j^n) (f_j(j) + f_j(C)) / 2, Delta_E = +dx, Delta_W = -dx, ... (:105).
 * Missing neighbours have zero weights and contribute nothing (Eq. 49 :656). */
void oracle_source(int nx, int ny, int nz, double dx, double dy, double dz, const unsigned char *v,
                   const double *w1, const double *w0, const double *gx, const double *gy, const double *gz,
                   double *S)
{
    const double dl[3] = { dx, dy, dz };
    const double *g[3] = { gx, gy, gz };
    i64 N = (i64)nx * ny * nz;
    i64 st[3] = { 1, nx, (i64)nx * ny };
#pragma omp parallel for if (N > OMP_MIN_N)
    for (i64 C = 0; C < N; ++C) {
        double s = 0.0;
        if (v[C])
            for (int d = 0; d < 6; ++d) {
                double w = w1[(i64)d * N + C] + w0[(i64)d * N + C];
                if (w == 0.0) continue;              /* missing neighbour (or 2D z-direction) */
                int a = d / 2;
                double Dj = (d % 2 == 0) ? dl[a] : -dl[a];
                i64 Q = C + ((d % 2 == 0) ? st[a] : -st[a]);
                s -= Dj * w * (g[a][Q] + g[a][C]) / 2.0;
            }
        S[C] = s;
    }
}

/* ------------------------------------------------------------------ operators of Eq. 12 (reading A1) */

/* q = [W^{n+1}] p  with Eq. 9 rearranged: (M p)_C = p_C - sum_j w_j^{n+1} p_j   (diagonal +1) */
void oracle_apply_M(int nx, int ny, int nz, const unsigned char *v, const double *w1, const double *p, double *q)
{
    i64 N = (i64)nx * ny * nz;
    i64 st[3] = { 1, nx, (i64)nx * ny };
#pragma omp parallel for if (N > OMP_MIN_N)
    for (i64 C = 0; C < N; ++C) {
        double s = 0.0;
        if (v[C]) {
            s = p[C];
            for (int d = 0; d < 6; ++d) {
                double w = w1[(i64)d * N + C];
                if (w != 0.0) s -= w * p[C + ((d % 2 == 0) ? st[d / 2] : -st[d / 2])];
            }
        }
        q[C] = s;
    }
}

/* q = [W^n] p:  (W^n p)_C = w_C^n p_C + sum_j w_j^n p_j */
void oracle_apply_Wn(int nx, int ny, int nz, const unsigned char *v, const double *w0, const double *w0C,
                     const double *p, double *q)
{
    i64 N = (i64)nx * ny * nz;
    i64 st[3] = { 1, nx, (i64)nx * ny };
#pragma omp parallel for if (N > OMP_MIN_N)
    for (i64 C = 0; C < N; ++C) {
        double s = 0.0;
        if (v[C]) {
            s = w0C[C] * p[C];
            for (int d = 0; d < 6; ++d) {
                double w = w0[(i64)d * N + C];
                if (w != 0.0) s += w * p[C + ((d % 2 == 0) ? st[d / 2] : -st[d / 2])];
            }
        }
        q[C] = s;
    }
}

/* dot product: long-double row sums, rows added in order */
static double dot(i64 N, int nx, const double *a, const double *b)
{
    i64 rows = (N + nx - 1) / nx;
    long double *part = (long double *)malloc(sizeof(long double) * (size_t)rows);
#pragma omp parallel for if (N > OMP_MIN_N)
    for (i64 r = 0; r < rows; ++r) {
        long double s = 0.0L;
        i64 e = (r + 1) * nx < N ? (r + 1) * nx : N;
        for (i64 c = r * nx; c < e; ++c) s += (long double)a[c] * (long double)b[c];
        part[r] = s;
    }
    long double t = 0.0L;
    for (i64 r = 0; r < rows; ++r) t += part[r];
    free(part);
    return (double)t;
}

double oracle_dot(i64 N, int nx, const double *a, const double *b) { return dot(N, nx, a, b); }

/* ------------------------------------------------------------------ inner CG (textbook recurrences, O6) */

/* q = A p with A = M = I - W1_off (Eq. 12 :119), or, for the fixed-point solve below, A = L = M - W^n: moving the
 * boundary term W^n P of Eq. 12 to the left gives L P = S, the equation every fixed point of Alg. 1 satisfies
 * (L_CC = sum_d v t_a, L_C,C+d = -v t_a: w1 + w0 = t_a on every valid link, Eq. 10 :109).  tmp: N work doubles. */
static void apply_op(int direct, int nx, int ny, int nz, const unsigned char *v, const double *w1, const double *w0,
                     const double *w0C, const double *p, double *q, double *tmp)
{
    oracle_apply_M(nx, ny, nz, v, w1, p, q);
    if (direct) {
        i64 N = (i64)nx * ny * nz;
        oracle_apply_Wn(nx, ny, nz, v, w0, w0C, p, tmp);
#pragma omp parallel for if (N > OMP_MIN_N)
        for (i64 c = 0; c < N; ++c) q[c] -= tmp[c];
    }
}

/* Solves A x = rhs starting from x (in/out).  Stops when sqrt(rho) <= thresh, rho == 0, or k == max_cg.
 * Work arrays r, p, q (and tmp if direct) of size N.  Returns the number of iterations done. */
static int cg_op(int direct, int nx, int ny, int nz, const unsigned char *v, const double *w1, const double *w0,
                 const double *w0C, const double *rhs, double *x, double thresh, int max_cg, double *r, double *p,
                 double *q, double *tmp)
{
    i64 N = (i64)nx * ny * nz;
    apply_op(direct, nx, ny, nz, v, w1, w0, w0C, x, q, tmp);
#pragma omp parallel for if (N > OMP_MIN_N)
    for (i64 c = 0; c < N; ++c) { r[c] = rhs[c] - q[c]; p[c] = r[c]; }
    double rho = dot(N, nx, r, r);
    int k = 0;
    while (sqrt(rho) > thresh && rho != 0.0 && k < max_cg) {
        apply_op(direct, nx, ny, nz, v, w1, w0, w0C, p, q, tmp);
        double alpha = rho / dot(N, nx, p, q);
#pragma omp parallel for if (N > OMP_MIN_N)
        for (i64 c = 0; c < N; ++c) { x[c] += alpha * p[c]; r[c] -= alpha * q[c]; }
        double rho1 = dot(N, nx, r, r);
        double beta = rho1 / rho;
#pragma omp parallel for if (N > OMP_MIN_N)
        for (i64 c = 0; c < N; ++c) p[c] = r[c] + beta * p[c];
        rho = rho1;
        ++k;
    }
    return k;
}

/* Single-reduction CG (Chronopoulos & Gear 1989; SURVEY 8(d) V5, 8(f) NEXT-2 i) for the SYMMETRIC system L x = rhs:
 * the same iterates as cg_op in exact arithmetic, but both inner products of an iteration (r.r and (A r).r) are taken
 * at the same point, so a parallel implementation synchronises once per iteration instead of twice.  s tracks A p by
 * the recurrence s = A r + beta s; p.Ap is never formed: alpha = gamma / (delta - beta gamma / alpha_prev), which relies
 * on A = A^T (it is NOT valid for the paper's nonsymmetric M).  Same stopping rule.  Work arrays r, p, q (= s), tmp, w. */
static int cg1_op(int nx, int ny, int nz, const unsigned char *v, const double *w1, const double *w0,
                  const double *w0C, const double *rhs, double *x, double thresh, int max_cg, double *r, double *p,
                  double *s, double *tmp, double *w)
{
    i64 N = (i64)nx * ny * nz;
    apply_op(1, nx, ny, nz, v, w1, w0, w0C, x, w, tmp);
#pragma omp parallel for if (N > OMP_MIN_N)
    for (i64 c = 0; c < N; ++c) { r[c] = rhs[c] - w[c]; p[c] = 0.0; s[c] = 0.0; }
    apply_op(1, nx, ny, nz, v, w1, w0, w0C, r, w, tmp);
    double gamma = dot(N, nx, r, r), delta = dot(N, nx, w, r), beta = 0.0, alpha = gamma / delta;
    int k = 0;
    while (sqrt(gamma) > thresh && gamma != 0.0 && k < max_cg) {
#pragma omp parallel for if (N > OMP_MIN_N)
        for (i64 c = 0; c < N; ++c) {
            p[c] = r[c] + beta * p[c];
            s[c] = w[c] + beta * s[c];
            x[c] += alpha * p[c];
            r[c] -= alpha * s[c];
        }
        apply_op(1, nx, ny, nz, v, w1, w0, w0C, r, w, tmp);
        double gamma1 = dot(N, nx, r, r), delta1 = dot(N, nx, w, r);      /* the iteration's single reduction point */
        beta = gamma1 / gamma;
        double den = delta1 - beta * gamma1 / alpha;                      /* stands for p.Ap > 0 */
        gamma = gamma1;
        ++k;
        if (!(den > 0.0)) break;      /* the recurrences have lost their accuracy: the caller's outer loop restarts on the true residual */
        alpha = gamma1 / den;
    }
    return k;
}

int oracle_cg(int nx, int ny, int nz, const unsigned char *v, const double *w1, const double *rhs, double *x,
              double thresh, int max_cg, double *r, double *p, double *q)
{
    return cg_op(0, nx, ny, nz, v, w1, NULL, NULL, rhs, x, thresh, max_cg, r, p, q, NULL);
}

/* ------------------------------------------------------------------ Algorithm 1 (:128-150) */

typedef struct {
    int outer_iters;        /* n at exit = number of Eq. 12 solves performed */
    i64 cg_iters_total;
    double eps_R_final;     /* Eq. 41 :442 at the returned P */
    double norm_S;
    int converged;          /* 1 iff eps_R <= tol at exit */
} oracle_info;

/* P_out: pressure at valid cells, NaN at missing cells (:158).  hist (may be NULL) receives eps_R of every outer
 * iteration visited, up to hist_cap entries.  Returns 0, or -1 on allocation failure. */
/* scheme2d: 2D constants although nz > 1 (stacked snapshots); direct: 0 = Eq. 12 (Alg. 1), 1 = L P = S by textbook CG,
 * 2 = L P = S by the single-reduction recurrences of cg1_op */
static int solve_impl(int scheme2d, int direct, int nx, int ny, int nz, double dx, double dy, double dz,
                      const double *gx, const double *gy, const double *gz, const unsigned char *mask,
                      const double *P_init, double *P_out, double tol, int max_outer, int max_cg, oracle_info *info,
                      double *hist, int hist_cap, double *hist_P);

int oracle_solve(int nx, int ny, int nz, double dx, double dy, double dz,
                 const double *gx, const double *gy, const double *gz, const unsigned char *mask,
                 double *P_out, double tol, int max_outer, int max_cg, oracle_info *info,
                 double *hist, int hist_cap)
{
    return solve_impl(nz == 1, 0, nx, ny, nz, dx, dy, dz, gx, gy, gz, mask, NULL, P_out, tol, max_outer, max_cg, info, hist, hist_cap, NULL);
}

/* oracle_solve that also records the pressure-update metric of Eq. 40 (:438): hist_P[n] = ||P^n - P^{n-1}|| / ||P^n||
 * for n >= 1 (entry 0 = 0: no update yet), next to hist[n] = eps_R of Eq. 41 at the same check. */
int oracle_solve_hist(int nx, int ny, int nz, double dx, double dy, double dz,
                      const double *gx, const double *gy, const double *gz, const unsigned char *mask,
                      double *P_out, double tol, int max_outer, int max_cg, oracle_info *info,
                      double *hist, double *hist_P, int hist_cap)
{
    return solve_impl(nz == 1, 0, nx, ny, nz, dx, dy, dz, gx, gy, gz, mask, NULL, P_out, tol, max_outer, max_cg, info, hist, hist_cap, hist_P);
}

/* Algorithm 1 started from a first guess instead of P^0 = 0 ("initializing with a first guess for the pressure field",
 * PAPER.md:82; a volume of a time series starts from the previous one's pressure).  Same iteration, same stopping
 * rules; P_init at missing cells is ignored. */
int oracle_solve_guess(int nx, int ny, int nz, double dx, double dy, double dz,
                       const double *gx, const double *gy, const double *gz, const unsigned char *mask,
                       const double *P_init, double *P_out, double tol, int max_outer, int max_cg, oracle_info *info)
{
    return solve_impl(nz == 1, 0, nx, ny, nz, dx, dy, dz, gx, gy, gz, mask, P_init, P_out, tol, max_outer, max_cg, info, NULL, 0, NULL);
}

/* The fixed point of Alg. 1 computed without the boundary iteration: at convergence P^{n+1} = P^n, so Eq. 12 reads
 * (M - W^n) P = S, i.e. L P = S with L the symmetric positive semi-definite weighted graph Laplacian of the valid
 * cells (constant null space per connected component; S sums to zero on each).  CG on it from P = 0 returns the
 * solution with zero mean on every component.  NOT the paper's algorithm (SURVEY 8(f) NEXT-2 iii): same converged
 * field, a different iteration.  Same arguments and stopping rules as oracle_solve, plus an optional first guess
 * P_init (NULL = 0; :82), which shifts the result by a constant per component. */
int oracle_solve_direct(int nx, int ny, int nz, double dx, double dy, double dz,
                        const double *gx, const double *gy, const double *gz, const unsigned char *mask,
                        const double *P_init, double *P_out, double tol, int max_outer, int max_cg, oracle_info *info)
{
    return solve_impl(nz == 1, 1, nx, ny, nz, dx, dy, dz, gx, gy, gz, mask, P_init, P_out, tol, max_outer, max_cg, info, NULL, 0, NULL);
}

/* oracle_solve_direct with the single-reduction CG recurrences (cg1_op) in the inner solves: same system, same outer
 * loop and stopping rules; a different (in exact arithmetic identical) iteration. */
int oracle_solve_direct_cg1(int nx, int ny, int nz, double dx, double dy, double dz,
                            const double *gx, const double *gy, const double *gz, const unsigned char *mask,
                            const double *P_init, double *P_out, double tol, int max_outer, int max_cg, oracle_info *info)
{
    return solve_impl(nz == 1, 2, nx, ny, nz, dx, dy, dz, gx, gy, gz, mask, P_init, P_out, tol, max_outer, max_cg, info, NULL, 0, NULL);
}

/* nb snapshots [nb][ny][nx] on one mask [ny][nx] (NULL = all valid), optional first guess P_init [nb][ny][nx]
 * ("initialized to zero ... or any other arbitrary value"; NULL = 0).  eps_R and the CG scalars are those
 * of the stacked system. */
static int solve_batch2d_impl(int direct, int nx, int ny, int nb, double dx, double dy,
                              const double *gx, const double *gy, const unsigned char *mask2d, const double *P_init,
                              double *P_out, double tol, int max_outer, int max_cg, oracle_info *info)
{
    unsigned char *m = NULL;
    if (mask2d) {
        m = (unsigned char *)malloc((size_t)nx * ny * nb);
        if (!m) return -1;
        for (int b = 0; b < nb; ++b) memcpy(m + (size_t)b * nx * ny, mask2d, (size_t)nx * ny);
    }
    int rc = solve_impl(1, direct, nx, ny, nb, dx, dy, 1.0, gx, gy, NULL, m, P_init, P_out, tol, max_outer, max_cg, info, NULL, 0, NULL);
    free(m);
    return rc;
}

int oracle_solve_batch2d(int nx, int ny, int nb, double dx, double dy,
                         const double *gx, const double *gy, const unsigned char *mask2d, const double *P_init,
                         double *P_out, double tol, int max_outer, int max_cg, oracle_info *info)
{
    return solve_batch2d_impl(0, nx, ny, nb, dx, dy, gx, gy, mask2d, P_init, P_out, tol, max_outer, max_cg, info);
}

/* oracle_solve_batch2d with the inner systems of oracle_solve_direct: CG on the block-diagonal L P = S of the stack */
int oracle_solve_direct_batch2d(int nx, int ny, int nb, double dx, double dy,
                                const double *gx, const double *gy, const unsigned char *mask2d, const double *P_init,
                                double *P_out, double tol, int max_outer, int max_cg, oracle_info *info)
{
    return solve_batch2d_impl(1, nx, ny, nb, dx, dy, gx, gy, mask2d, P_init, P_out, tol, max_outer, max_cg, info);
}

static int solve_impl(int scheme2d, int direct, int nx, int ny, int nz, double dx, double dy, double dz,
                      const double *gx, const double *gy, const double *gz, const unsigned char *mask,
                      const double *P_init, double *P_out, double tol, int max_outer, int max_cg, oracle_info *info,
                      double *hist, int hist_cap, double *hist_P)
{
    i64 N = (i64)nx * ny * nz;
    size_t nb = sizeof(double) * (size_t)N;
    unsigned char *v = (unsigned char *)malloc((size_t)N);
    double *w1 = (double *)malloc(6 * nb), *w0 = (double *)malloc(6 * nb), *w0C = (double *)malloc(nb);
    double *S = (double *)malloc(nb), *P = (double *)calloc((size_t)N, sizeof(double));
    double *rhs = (double *)malloc(nb), *r = (double *)malloc(nb), *p = (double *)malloc(nb), *q = (double *)malloc(nb);
    double *tmp = (double *)malloc(nb);
    double *Pold = hist_P ? (double *)malloc(nb) : NULL;
    double *wv = (direct == 2) ? (double *)malloc(nb) : NULL;
    int rc = -1;
    if (!v || !w1 || !w0 || !w0C || !S || !P || !rhs || !r || !p || !q || !tmp || (hist_P && !Pold) || (direct == 2 && !wv)) goto done;
    rc = 0;

    oracle_validity(nx, ny, nz, gx, gy, gz, mask, v);
    weights_impl(scheme2d, nx, ny, nz, dx, dy, dz, v, w1, w0, w0C);
    oracle_source(nx, ny, nz, dx, dy, dz, v, w1, w0, gx, gy, gz ? gz : gx, S);
    double normS = sqrt(dot(N, nx, S, S));
    if (P_init)
        for (i64 c = 0; c < N; ++c) P[c] = v[c] ? P_init[c] : 0.0;

    int n = 0;
    i64 cg_total = 0;
    double epsR = 0.0;
    if (normS > 0.0) {
        for (;;) {
            /* rhs = W^n P^n + S ; r0 = rhs - M P^n ; eps_R = |r0| / |S|  (Eq. 12 :119, Eq. 41 :442) */
            oracle_apply_Wn(nx, ny, nz, v, w0, w0C, P, rhs);
            oracle_apply_M(nx, ny, nz, v, w1, P, q);
#pragma omp parallel for if (N > OMP_MIN_N)
            for (i64 c = 0; c < N; ++c) { rhs[c] += S[c]; r[c] = rhs[c] - q[c]; }
            epsR = sqrt(dot(N, nx, r, r)) / normS;
            if (hist && n < hist_cap) hist[n] = epsR;
            if (hist_P && n < hist_cap) {            /* Eq. 40 :438 for the update that led to this check */
                if (n == 0) hist_P[0] = 0.0;
                else {
#pragma omp parallel for if (N > OMP_MIN_N)
                    for (i64 c = 0; c < N; ++c) tmp[c] = P[c] - Pold[c];
                    double nP = sqrt(dot(N, nx, P, P));
                    hist_P[n] = nP > 0.0 ? sqrt(dot(N, nx, tmp, tmp)) / nP : 0.0;
                }
            }
            if (epsR <= tol || n == max_outer) break;
            if (hist_P) memcpy(Pold, P, nb);
            /* Solve Eq. 12 for P^{n+1} by CG, first guess P^n (:489); inner threshold: reading A3.
             * Fixed-point variant (oracle_solve_direct): the same loop with the system L P = S; eps_R above is its
             * residual too (r0 = S - L P^n), so the outer loop only restarts a CG that hit max_cg. */
            if (direct) memcpy(rhs, S, nb);
            if (direct == 2) cg_total += cg1_op(nx, ny, nz, v, w1, w0, w0C, rhs, P, 0.1 * tol * normS, max_cg, r, p, q, tmp, wv);
            else cg_total += cg_op(direct, nx, ny, nz, v, w1, w0, w0C, rhs, P, 0.1 * tol * normS, max_cg, r, p, q, tmp);
            ++n;
        }
    }
    for (i64 c = 0; c < N; ++c) P_out[c] = v[c] ? P[c] : NAN;
    if (info) {
        info->outer_iters = n; info->cg_iters_total = cg_total; info->eps_R_final = epsR;
        info->norm_S = normS; info->converged = (epsR <= tol);
    }
done:
    free(v); free(w1); free(w0); free(w0C); free(S); free(P); free(rhs); free(r); free(p); free(q); free(tmp); free(Pold); free(wv);
    return rc;
}

/* ------------------------------------------------------------------ per-cell evaluation at sampled cells
 * (full-size checks: the quantities below are local formulas, so the oracle can evaluate them one cell at a time
 * without storing 13 weight fields).  cells[] are linear indices; out-of-sample cost O(1) each. */

static void cell_weights(int nx, int ny, int nz, const double *K, const unsigned char *v, int i, int j, int k,
                         double *w1, double *w0, double *w0C)
{
    const double *F = K, Atot = K[3], *c = K + 4;
    double AC = 0.0;
    for (int d = 0; d < 6; ++d) {
        int a = d / 2;
        double A1 = 0.0, A0 = 0.0;
        int qi = i + DIRV[d][0], qj = j + DIRV[d][1], qk = k + DIRV[d][2];
        if (!val(v, nx, ny, nz, qi, qj, qk)) AC += F[a];
        else {
            int bt = val(v, nx, ny, nz, qi + DIRV[d][0], qj + DIRV[d][1], qk + DIRV[d][2]);
            A1 += c[3 * a + a] * bt; A0 += c[3 * a + a] * (1 - bt);
            for (int b = 0; b < 3; ++b) {
                if (b == a) continue;
                for (int sgn = 0; sgn < 2; ++sgn) {
                    const int *e = DIRV[2 * b + sgn];
                    int bs = val(v, nx, ny, nz, qi + e[0], qj + e[1], qk + e[2]);
                    A1 += c[3 * a + b] * bs; A0 += c[3 * a + b] * (1 - bs);
                }
            }
        }
        w1[d] = A1 / Atot; w0[d] = A0 / Atot;
    }
    *w0C = AC / Atot;
}

/* For each sampled cell: S_C (Eq. 9), (M x)_C, (W^n x)_C for a given field x (NULL -> zeros written).
 * Any of S_out, Mx_out, Wx_out may be NULL. */
void oracle_sample(int nx, int ny, int nz, double dx, double dy, double dz, const unsigned char *v,
                   const double *gx, const double *gy, const double *gz, const double *x,
                   i64 ncells, const i64 *cells, double *S_out, double *Mx_out, double *Wx_out)
{
    double K[13];
    oracle_constants(nx, ny, nz, dx, dy, dz, K);
    const double dl[3] = { dx, dy, dz };
    const double *g[3] = { gx, gy, gz };
    i64 st[3] = { 1, nx, (i64)nx * ny };
#pragma omp parallel for if (ncells > 1024)
    for (i64 s = 0; s < ncells; ++s) {
        i64 C = cells[s];
        int i = (int)(C % nx), j = (int)((C / nx) % ny), k = (int)(C / ((i64)nx * ny));
        double w1[6], w0[6], w0C, Sv = 0.0, Mv = 0.0, Wv = 0.0;
        if (v[C]) {
            cell_weights(nx, ny, nz, K, v, i, j, k, w1, w0, &w0C);
            if (x) { Mv = x[C]; Wv = w0C * x[C]; }
            for (int d = 0; d < 6; ++d) {
                double w = w1[d] + w0[d];
                if (w == 0.0) continue;
                int a = d / 2;
                i64 Q = C + ((d % 2 == 0) ? st[a] : -st[a]);
                if (gx) Sv -= ((d % 2 == 0) ? dl[a] : -dl[a]) * w * (g[a][Q] + g[a][C]) / 2.0;
                if (x) { Mv -= w1[d] * x[Q]; Wv += w0[d] * x[Q]; }
            }
        }
        if (S_out) S_out[s] = Sv;
        if (Mx_out) Mx_out[s] = Mv;
        if (Wx_out) Wx_out[s] = Wv;
    }
}

int oracle_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        n = omp_get_num_threads();
    }
#endif
    return n;
}
