"""oracle/omni_pcg.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain numpy fp64 oracle of omni_solve_pcg_* (SURVEY.md 8(f) NEXT-2 ii): the fixed point L P = S of Algorithm 1
(PAPER.md:119 at P^{n+1} = P^n; oracle_solve_direct in omni_oracle.c) by conjugate gradients PRECONDITIONED with one
geometric-multigrid V-cycle.  Not the paper's iteration (the paper names only "CG", :124); the reading taken is
DESIGN.md R-P1, restated step by step here.  Shares nothing with the CUDA path; only tests/, smoke() and bench.py's
oracle legs may import it.

Reading R-P1 (the algorithm, in the order executed):
  levels   level 0 is the grid.  Level l+1 halves (ceil) every axis a of level l that has >= 8 cells AND is strongly
           coupled on that level: w_l[a] >= 0.7 max_b w_l[b] (b over the axes with >= 8 cells).  Point smoothing only
           removes error along strongly coupled axes, so a weakly coupled axis (t_a is proportional to 1 / Delta_a: the
           axis with the larger spacing) is left alone until the halvings of the others -- each divides its own weight by
           4 relative to the rest -- have made it strong (semi-coarsening; on isotropic grids every axis is halved on every
           level).  A coarse cell is valid iff one of its children is; coarsening stops when no axis qualifies (or after
           24 levels).
  operator (L_l x)_C = sum_d v_l(C+d) w_l[a] (x_C - x_{C+d}) on valid cells, 0 elsewhere.  w_0[a] = t_a = F_a / A_tot
           (Eq. 10 :109: w^{n+1} + w^n on a valid link); w_{l+1}[a] = w_l[a] * 2^m * (1/4 if axis a was halved else 1),
           m = number of halved axes: the Galerkin weight of piecewise-constant transfers (number of fine links between
           two coarse cells), halved along the coarsened axes, where that Galerkin operator is twice too stiff.
  transfer restriction = plain sum over the children, prolongation = the parent's value (its transpose).
  smoother damped Jacobi  x <- x + omega D^-1 (b - L x),  omega = 0.8, D = diag(L) (D^-1 = 0 where D = 0).
  V-cycle  B_l(b): x = 2 sweeps from x = 0; b_c = restrict(b - L x); x += prolong(B_{l+1}(b_c)); 2 sweeps; return x.
           Coarsest level: 8 sweeps from 0.  Linear, symmetric (same smoother before and after, R = P^T), positive.
  PCG      on L delta = r0 from delta = 0:  z = B_0(r); rho = r.z; p = z + (rho/rho_old) p (p = z at first); q = L p;
           alpha = rho / p.q; delta += alpha p; r -= alpha q;  until sqrt(r.r) <= 0.1 tol ||S||, r.r = 0 or max_cg
           (fp32 library variant: also until sqrt(r.r) <= 1e-2 ||r0||, argument inner_rel -- fp32 vectors cannot
           resolve more digits of one correction on large grids; the fp64 outer loop restarts on the true residual).
  outer    as oracle_solve_direct: r0 = S - L P, eps_R = ||r0|| / ||S|| (Eq. 41 :442); stop at eps_R <= tol or
           max_outer; P += delta.  P_init (optional) is the first guess.

Pins (tests/test_oracle_pins.py): dense pinv(L) S; the V-cycle as a dense matrix is symmetric positive semi-definite
and the iterates equal a dense textbook PCG with that matrix; a grid too small to coarsen reduces to the Jacobi
polynomial in closed form; <restrict r, e> = <r, prolong e>; level-0 operator = M - W^n of the stored-weight oracle.
"""
import numpy as np

from . import omni_oracle as _o

OMEGA = 0.8
NU = 2            # sweeps before and after the coarse-grid correction
NU_COARSEST = 8
MIN_COARSEN = 8   # an axis is halved while it has at least this many cells ...
THETA = 0.7       # ... and its link weight is at least this fraction of the largest weight among such axes
MAX_LEVELS = 24


def _shift(x, ax, s):
    """y[C] = x[C + s e_ax], 0 outside the box (s = +1 / -1)."""
    y = np.zeros_like(x)
    a = [slice(None)] * x.ndim
    b = [slice(None)] * x.ndim
    if s > 0:
        a[ax], b[ax] = slice(0, -1), slice(1, None)
    else:
        a[ax], b[ax] = slice(1, None), slice(0, -1)
    y[tuple(a)] = x[tuple(b)]
    return y


class Level:
    """v: validity (bool, numpy order: x is the LAST axis); w[a]: link weight of axis a (a = 0 is x)."""

    def __init__(self, v, w):
        self.v, self.w = v, np.asarray(w, dtype=np.float64)
        nd = v.ndim
        self.link = []                                     # per axis a: (link to +e_a, link to -e_a)
        D = np.zeros(v.shape)
        for a in range(nd):
            ax = nd - 1 - a
            lp, lm = v & _shift(v, ax, +1), v & _shift(v, ax, -1)
            self.link.append((lp, lm))
            D += self.w[a] * (lp.astype(np.float64) + lm)
        self.Dinv = np.zeros(v.shape)
        self.Dinv[D > 0] = 1.0 / D[D > 0]

    def apply(self, x):
        nd = self.v.ndim
        y = np.zeros(self.v.shape)
        for a in range(nd):
            ax = nd - 1 - a
            lp, lm = self.link[a]
            y += self.w[a] * (lp * (x - _shift(x, ax, +1)) + lm * (x - _shift(x, ax, -1)))
        return y

    def sweep(self, x, b):
        return x + OMEGA * self.Dinv * (b - self.apply(x))


def coarsen_plan(shape, w, frozen_axes=()):
    """Which numpy axes of `shape` are halved to make the next level: those with >= MIN_COARSEN cells whose link weight
    (w[a], a = 0 is x = the LAST numpy axis) is >= THETA times the largest weight among the axes with >= MIN_COARSEN cells;
    numpy axes in `frozen_axes` (the snapshot axis of a stack of 2D fields) are never halved."""
    nd = len(shape)
    ok = [s >= MIN_COARSEN and ax not in frozen_axes for ax, s in enumerate(shape)]
    wax = [float(w[nd - 1 - ax]) for ax in range(nd)]
    wmax = max([wa for wa, o in zip(wax, ok) if o], default=0.0)
    return [bool(o and wa >= THETA * wmax) for wa, o in zip(wax, ok)]


def restrict(r, halve):
    """Sum over the children: axis halved -> pairs (2I, 2I+1) added (an odd last cell stands alone)."""
    for ax, h in enumerate(halve):
        if h:
            n = r.shape[ax]
            if n % 2:
                pad = [(0, 0)] * r.ndim
                pad[ax] = (0, 1)
                r = np.pad(r, pad)
            sh = list(r.shape)
            sh[ax:ax + 1] = [r.shape[ax] // 2, 2]
            r = r.reshape(sh).sum(axis=ax + 1)
    return r


def prolong(e, halve, fshape):
    """The parent's value: the transpose of restrict."""
    for ax, h in enumerate(halve):
        if h:
            e = np.repeat(e, 2, axis=ax)
    return e[tuple(slice(0, s) for s in fshape)]


def build_levels(v, w0, frozen_axes=()):
    levels, plans = [Level(v.astype(bool), w0)], []
    while len(levels) < MAX_LEVELS:
        f = levels[-1]
        halve = coarsen_plan(f.v.shape, f.w, frozen_axes)
        if not any(halve):
            break
        m = sum(halve)
        nd = f.v.ndim
        # axis a (x first) lives on numpy axis nd-1-a
        w = [f.w[a] * 2.0 ** m * (0.25 if halve[nd - 1 - a] else 1.0) for a in range(nd)]
        vc = restrict(f.v.astype(np.int64), halve) > 0
        plans.append(halve)
        levels.append(Level(vc, w))
    return levels, plans


def vcycle(levels, plans, l, b):
    L = levels[l]
    last = l + 1 == len(levels)
    x = OMEGA * L.Dinv * b                                 # first sweep from x = 0
    for _ in range((NU_COARSEST if last else NU) - 1):
        x = L.sweep(x, b)
    if last:
        return x
    rc = restrict((b - L.apply(x)) * L.v, plans[l])
    x = x + prolong(vcycle(levels, plans, l + 1, rc), plans[l], L.v.shape) * L.v
    for _ in range(NU):
        x = L.sweep(x, b)
    return x


def face_weights(nd, dx, dy, dz):
    """t_a = F_a / A_tot (Eq. 5 :75, Eq. 8 :94 in 2D; Eq. 23 :258, Eq. 24 :262 in 3D), from the oracle's constants."""
    K = _o.constants(4, 4, 4 if nd == 3 else 1, dx, dy, dz)
    return [K["F"][a] / K["A_tot"] for a in range(nd)]


def _pcg_core(v, S, w, tol, max_outer, max_cg, P_init, return_iterates, inner_rel, frozen_axes=()):
    """The iteration of reading R-P1 on validity v (bool), source S and level-0 link weights w (w[0] is x); numpy axes
    in `frozen_axes` are never coarsened (the snapshot axis of a stack)."""
    levels, plans = build_levels(v, w, frozen_axes)
    L0 = levels[0]
    P = np.zeros(v.shape) if P_init is None else np.where(v, np.nan_to_num(np.asarray(P_init, dtype=np.float64)), 0.0)
    normS = float(np.sqrt(np.sum(S * S)))
    n, cg_total, epsR, iterates = 0, 0, 0.0, []
    if normS > 0.0:
        while True:
            r = (S - L0.apply(P)) * v
            epsR = float(np.sqrt(np.sum(r * r))) / normS
            if epsR <= tol or n == max_outer:
                break
            delta, p, rho_old, k = np.zeros_like(P), np.zeros_like(P), 1.0, 0
            rr = float(np.sum(r * r))
            thresh = max(0.1 * tol * normS, inner_rel * np.sqrt(rr))
            while np.sqrt(rr) > thresh and rr != 0.0 and k < max_cg:
                z = vcycle(levels, plans, 0, r)
                rho = float(np.sum(r * z))
                p = z + ((rho / rho_old) if k > 0 else 0.0) * p
                q = L0.apply(p)
                alpha = rho / float(np.sum(p * q))
                delta = delta + alpha * p
                r = r - alpha * q
                rho_old = rho
                rr = float(np.sum(r * r))
                k += 1
                if return_iterates:
                    iterates.append((P + delta).copy())
            P = P + delta
            cg_total += k
            n += 1
    info = {"outer_iters": n, "cg_iters_total": cg_total, "eps_R_final": epsR, "norm_S": normS, "converged": epsR <= tol,
            "levels": len(levels)}
    out = np.where(v, P, np.nan)
    return (out, info, iterates) if return_iterates else (out, info)


def solve_pcg(gx, gy, gz, mask, dx, dy, dz, tol, max_outer, max_cg, P_init=None, return_iterates=False, inner_rel=0.0):
    """Returns (P with NaN at missing cells, info dict) -- same conventions as omni_oracle.solve_direct.
    inner_rel: an inner solve also stops once ||r|| <= inner_rel ||r0|| (0 = off; the fp32 library variant uses 1e-2,
    because fp32 vectors cannot resolve more digits of one correction on large grids -- the outer refinement restarts)."""
    gx = np.asarray(gx, dtype=np.float64)
    nd = gx.ndim
    v8 = _o.validity(gx, gy, gz, mask)
    w1, w0, w0C = _o.weights(v8, dx, dy, dz)
    z3 = lambda c: None if c is None else np.nan_to_num(np.asarray(c, dtype=np.float64))
    S = _o.source(v8, w1, w0, z3(gx), z3(gy), z3(gz), dx, dy, dz)
    return _pcg_core(v8.astype(bool), S, face_weights(nd, dx, dy, dz), tol, max_outer, max_cg, P_init, return_iterates, inner_rel)


def solve_pcg_batch2d(gx, gy, mask2d, dx, dy, tol, max_outer, max_cg, P_init=None, inner_rel=0.0):
    """nb stacked 2D snapshots (nb, ny, nx) on one mask (ny, nx), as omni_oracle.solve_batch2d with direct=True but with
    the preconditioned iteration: ONE block-diagonal system (2D scheme per plane, no links across planes: weight 0 along
    the snapshot axis, which is never coarsened), joint CG scalars and stopping tests over the stack."""
    gx, gy = np.asarray(gx, dtype=np.float64), np.asarray(gy, dtype=np.float64)
    nb = gx.shape[0]
    v8 = np.stack([_o.validity(gx[b], gy[b], None, mask2d) for b in range(nb)])
    S = np.zeros(gx.shape)
    for b in range(nb):
        w1, w0, w0C = _o.weights(v8[b], dx, dy)
        S[b] = _o.source(v8[b], w1, w0, np.nan_to_num(gx[b]), np.nan_to_num(gy[b]), None, dx, dy)
    w = face_weights(2, dx, dy, 1.0) + [0.0]
    return _pcg_core(v8.astype(bool), S, w, tol, max_outer, max_cg, P_init, False, inner_rel, frozen_axes=(0,))
