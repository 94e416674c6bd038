"""ctypes wrapper around oracle/omni_oracle.c  -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module.  It never imports paper_2311_16935_b200 and shares nothing with the CUDA path.
The solver path (constants, weights, S, operators, CG, Algorithm 1) is argument marshalling for the C functions of
omni_oracle.c, each citing the PAPER.md passage it follows.  The upstream source-field steps g = f(u) -- velocity_source
(Eq. 1), rans_source (Eq. 42), compressible_rans_source (Eq. 43-44) -- are written out here in plain numpy (fp64).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "omni_oracle.c")
_LIB = os.path.join(_HERE, "libomni_oracle.so")
_lib = None


def build(force=False):
    """gcc -O2 -ffp-contract=off -fopenmp (no fast-math); rebuilt when the source is newer."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class Info(C.Structure):
    _fields_ = [("outer_iters", C.c_int), ("cg_iters_total", C.c_longlong), ("eps_R_final", C.c_double),
                ("norm_S", C.c_double), ("converged", C.c_int)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_far_face_constant.restype = C.c_double
        _lib.oracle_far_face_constant.argtypes = [C.c_double] * 3
        _lib.oracle_dot.restype = C.c_double
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _dims(shape):
    """shape is numpy order (nz, ny, nx) or (ny, nx); returns nx, ny, nz."""
    if len(shape) == 2:
        return shape[1], shape[0], 1
    return shape[2], shape[1], shape[0]


def num_threads():
    return int(lib().oracle_num_threads())


def constants(nx, ny, nz, dx, dy, dz):
    """dict F[3], A_tot, c[3][3]  (Eq. 5/8/17 2D; Eq. 23/24/32-35 3D)."""
    out = np.zeros(13)
    lib().oracle_constants(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(dx), C.c_double(dy), C.c_double(dz), _p(out))
    return {"F": out[0:3].copy(), "A_tot": float(out[3]), "c": out[4:13].reshape(3, 3).copy()}


def far_face_constant(da, db, dc):
    return float(lib().oracle_far_face_constant(da, db, dc))


def validity(gx, gy, gz=None, mask=None):
    gx, gy, gz = _f64(gx), _f64(gy), _f64(gz)
    nx, ny, nz = _dims(gx.shape)
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    v = np.zeros(gx.shape, dtype=np.uint8)
    lib().oracle_validity(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(gx), _p(gy), _p(gz), _p(m), _p(v))
    return v


def weights(v, dx, dy, dz=1.0):
    """returns w1[6,...], w0[6,...], w0C[...] (Eq. 10) for a validity array v."""
    v = np.ascontiguousarray(v, dtype=np.uint8)
    nx, ny, nz = _dims(v.shape)
    w1 = np.zeros((6,) + v.shape)
    w0 = np.zeros((6,) + v.shape)
    w0C = np.zeros(v.shape)
    lib().oracle_weights(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(dx), C.c_double(dy), C.c_double(dz),
                         _p(v), _p(w1), _p(w0), _p(w0C))
    return w1, w0, w0C


def source(v, w1, w0, gx, gy, gz, dx, dy, dz=1.0):
    v = np.ascontiguousarray(v, dtype=np.uint8)
    nx, ny, nz = _dims(v.shape)
    gx, gy = _f64(gx), _f64(gy)
    gz = _f64(gz) if gz is not None else np.zeros_like(gx)
    S = np.zeros(v.shape)
    lib().oracle_source(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(dx), C.c_double(dy), C.c_double(dz),
                        _p(v), _p(w1), _p(w0), _p(gx), _p(gy), _p(gz), _p(S))
    return S


def apply_M(v, w1, p):
    v = np.ascontiguousarray(v, dtype=np.uint8)
    nx, ny, nz = _dims(v.shape)
    p = _f64(p)
    q = np.zeros(v.shape)
    lib().oracle_apply_M(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(v), _p(w1), _p(p), _p(q))
    return q


def apply_Wn(v, w0, w0C, p):
    v = np.ascontiguousarray(v, dtype=np.uint8)
    nx, ny, nz = _dims(v.shape)
    p = _f64(p)
    q = np.zeros(v.shape)
    lib().oracle_apply_Wn(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(v), _p(w0), _p(w0C), _p(p), _p(q))
    return q


def cg(v, w1, rhs, x0, thresh, max_cg):
    """textbook CG on M x = rhs from x0; returns (x, iterations)."""
    v = np.ascontiguousarray(v, dtype=np.uint8)
    nx, ny, nz = _dims(v.shape)
    rhs = _f64(rhs)
    x = np.array(x0, dtype=np.float64, order="C", copy=True)
    r, p, q = np.zeros(v.shape), np.zeros(v.shape), np.zeros(v.shape)
    f = lib().oracle_cg
    f.restype = C.c_int
    k = f(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(v), _p(w1), _p(rhs), _p(x), C.c_double(thresh), C.c_int(max_cg),
          _p(r), _p(p), _p(q))
    return x, int(k)


def solve(gx, gy, gz, mask, dx, dy, dz, tol, max_outer, max_cg, hist_cap=0):
    """Algorithm 1.  Arrays in numpy order (nz,ny,nx) or (ny,nx).  Returns (P, info dict[, hist])."""
    gx, gy = _f64(gx), _f64(gy)
    nx, ny, nz = _dims(gx.shape)
    gz = _f64(gz) if gz is not None else None
    if nz > 1 and gz is None:
        raise ValueError("gz required in 3D")
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    P = np.zeros(gx.shape)
    info = Info()
    hist = np.full(max(hist_cap, 1), np.nan)
    f = lib().oracle_solve
    f.restype = C.c_int
    rc = f(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(dx), C.c_double(dy), C.c_double(dz),
           _p(gx), _p(gy), _p(gz if gz is not None else gx), _p(m), _p(P), C.c_double(tol), C.c_int(max_outer),
           C.c_int(max_cg), C.byref(info), _p(hist) if hist_cap else None, C.c_int(hist_cap))
    if rc != 0:
        raise MemoryError("oracle_solve: allocation failed")
    d = {"outer_iters": info.outer_iters, "cg_iters_total": info.cg_iters_total, "eps_R_final": info.eps_R_final,
         "norm_S": info.norm_S, "converged": bool(info.converged)}
    return (P, d, hist) if hist_cap else (P, d)


def solve_hist(gx, gy, gz, mask, dx, dy, dz, tol, max_outer, max_cg, hist_cap):
    """Algorithm 1 with both convergence metrics recorded per outer check: eps_R (Eq. 41 :442) and the pressure-update
    metric eps_P (Eq. 40 :438; entry 0 = 0).  Returns (P, info dict, hist_R, hist_P)."""
    gx, gy = _f64(gx), _f64(gy)
    nx, ny, nz = _dims(gx.shape)
    gz = _f64(gz) if gz is not None else None
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    P = np.zeros(gx.shape)
    info = Info()
    hR, hP = np.full(hist_cap, np.nan), np.full(hist_cap, np.nan)
    f = lib().oracle_solve_hist
    f.restype = C.c_int
    rc = f(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(dx), C.c_double(dy), C.c_double(dz),
           _p(gx), _p(gy), _p(gz if gz is not None else gx), _p(m), _p(P), C.c_double(tol), C.c_int(max_outer),
           C.c_int(max_cg), C.byref(info), _p(hR), _p(hP), C.c_int(hist_cap))
    if rc != 0:
        raise MemoryError("oracle_solve_hist: allocation failed")
    d = {"outer_iters": info.outer_iters, "cg_iters_total": info.cg_iters_total, "eps_R_final": info.eps_R_final,
         "norm_S": info.norm_S, "converged": bool(info.converged)}
    return P, d, hR, hP


def solve_guess(gx, gy, gz, mask, dx, dy, dz, tol, max_outer, max_cg, P_init):
    """Algorithm 1 started from the first guess P_init (oracle_solve_guess).  Returns (P, info)."""
    gx, gy = _f64(gx), _f64(gy)
    nx, ny, nz = _dims(gx.shape)
    gz = _f64(gz) if gz is not None else None
    if nz > 1 and gz is None:
        raise ValueError("gz required in 3D")
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    P = np.zeros(gx.shape)
    info = Info()
    P0 = None if P_init is None else _f64(P_init)
    f = lib().oracle_solve_guess
    f.restype = C.c_int
    rc = f(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(dx), C.c_double(dy), C.c_double(dz),
           _p(gx), _p(gy), _p(gz if gz is not None else gx), _p(m), _p(P0), _p(P), C.c_double(tol), C.c_int(max_outer),
           C.c_int(max_cg), C.byref(info))
    if rc != 0:
        raise MemoryError("oracle_solve_guess: allocation failed")
    return P, {"outer_iters": info.outer_iters, "cg_iters_total": info.cg_iters_total, "eps_R_final": info.eps_R_final,
               "norm_S": info.norm_S, "converged": bool(info.converged)}


def solve_direct(gx, gy, gz, mask, dx, dy, dz, tol, max_outer, max_cg, P_init=None, single_reduction=False):
    """Fixed point of Algorithm 1 by CG on L P = S (oracle_solve_direct; not the paper's iteration).  Returns (P, info).
    single_reduction: the Chronopoulos-Gear recurrences (oracle_solve_direct_cg1) instead of the textbook ones."""
    gx, gy = _f64(gx), _f64(gy)
    nx, ny, nz = _dims(gx.shape)
    gz = _f64(gz) if gz is not None else None
    if nz > 1 and gz is None:
        raise ValueError("gz required in 3D")
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    P = np.zeros(gx.shape)
    info = Info()
    P0 = None if P_init is None else _f64(P_init)
    f = lib().oracle_solve_direct_cg1 if single_reduction else lib().oracle_solve_direct
    f.restype = C.c_int
    rc = f(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(dx), C.c_double(dy), C.c_double(dz),
           _p(gx), _p(gy), _p(gz if gz is not None else gx), _p(m), _p(P0), _p(P), C.c_double(tol), C.c_int(max_outer),
           C.c_int(max_cg), C.byref(info))
    if rc != 0:
        raise MemoryError("oracle_solve_direct: allocation failed")
    return P, {"outer_iters": info.outer_iters, "cg_iters_total": info.cg_iters_total, "eps_R_final": info.eps_R_final,
               "norm_S": info.norm_S, "converged": bool(info.converged)}


def sample(v, gx, gy, gz, x, cells, dx, dy, dz=1.0):
    """Per-cell S_C, (M x)_C, (W^n x)_C at linear indices `cells` (full-size spot checks)."""
    v = np.ascontiguousarray(v, dtype=np.uint8)
    nx, ny, nz = _dims(v.shape)
    gx, gy, gz, x = _f64(gx), _f64(gy), _f64(gz), _f64(x)
    if gx is not None and gz is None:
        gz = gx
    cells = np.ascontiguousarray(cells, dtype=np.int64)
    S, Mx, Wx = np.zeros(len(cells)), np.zeros(len(cells)), np.zeros(len(cells))
    lib().oracle_sample(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(dx), C.c_double(dy), C.c_double(dz),
                        _p(v), _p(gx), _p(gy), _p(gz), _p(x), C.c_longlong(len(cells)), _p(cells), _p(S), _p(Mx), _p(Wx))
    return S, Mx, Wx


def eps_R_of_field(gx, gy, gz, mask, P, dx, dy, dz=1.0, chunk=4_000_000):
    """Momentum residual of a GIVEN field (Eq. 41): eps_R = ||S + W^n P - M P||_2 / ||S||_2, evaluated cell by
    cell through oracle_sample in chunks of `chunk` cells, so that a full-size field (500^3) needs no stored weight
    arrays.  NaN / missing cells of P count as 0 (they carry zero weights).  Returns (eps_R, ||r||, ||S||).
    SURVEY 8(c) parity protocol iii: certifies a converged field the oracle itself cannot afford to compute."""
    v = validity(gx, gy, gz, mask)
    x = np.nan_to_num(_f64(P), nan=0.0) * v
    n = v.size
    rr = ss = 0.0
    for c0 in range(0, n, chunk):
        cells = np.arange(c0, min(n, c0 + chunk), dtype=np.int64)
        S, Mx, Wx = sample(v, gx, gy, gz, x, cells, dx, dy, dz)
        r = S + Wx - Mx
        rr += float(np.dot(r, r))
        ss += float(np.dot(S, S))
    return (float(np.sqrt(rr / ss)) if ss > 0 else 0.0), float(np.sqrt(rr)), float(np.sqrt(ss))


def solve_batch2d(gx, gy, mask2d, dx, dy, tol, max_outer, max_cg, P_init=None, direct=False):
    """nb stacked 2D snapshots (nb, ny, nx) on one mask (ny, nx), solved as one block-diagonal system
    (direct: with the inner systems of solve_direct)."""
    gx, gy = _f64(gx), _f64(gy)
    nb, ny, nx = gx.shape
    m = None if mask2d is None else np.ascontiguousarray(mask2d, dtype=np.uint8)
    P0 = None if P_init is None else _f64(P_init)
    P = np.zeros(gx.shape)
    info = Info()
    f = lib().oracle_solve_direct_batch2d if direct else lib().oracle_solve_batch2d
    f.restype = C.c_int
    rc = f(C.c_int(nx), C.c_int(ny), C.c_int(nb), C.c_double(dx), C.c_double(dy), _p(gx), _p(gy), _p(m), _p(P0), _p(P),
           C.c_double(tol), C.c_int(max_outer), C.c_int(max_cg), C.byref(info))
    if rc != 0:
        raise MemoryError("oracle_solve_batch2d: allocation failed")
    return P, {"outer_iters": info.outer_iters, "cg_iters_total": info.cg_iters_total, "eps_R_final": info.eps_R_final,
               "norm_S": info.norm_S, "converged": bool(info.converged)}


def velocity_source(u, v, w, mask, dx, dy, dz=1.0, rho=1.0, mu=0.0, dudt=None):
    """f(u) = grad P of Eq. 1: -rho (du/dt + (u . grad) u) + mu lap u, on the cell grid, written out with
    second-order central differences (plain numpy slicing, fp64).  u, v(, w): (ny, nx) or (nz, ny, nx); w = None in 2D.
    dudt: optional list of the local accelerations du_i/dt (same shapes; None = steady).  Reading R-V1:
    the paper does not fix the discretisation; a cell whose central stencil touches a missing cell (outside the box,
    mask == 0, NaN velocity) gets NaN in every component, which the solver treats as missing (Eq. 13 :176).
    Returns [gx, gy(, gz)]."""
    comps = [_f64(u), _f64(v)] + ([] if w is None else [_f64(w)])
    nd = comps[0].ndim
    assert nd == len(comps), "2D fields take (u, v), 3D fields (u, v, w)"
    h = [dx, dy, dz][:nd]                     # spacing of axis a = 0 (x), 1 (y), 2 (z); numpy axis of a is nd - 1 - a
    ok = np.ones(comps[0].shape, bool) if mask is None else (np.asarray(mask) != 0)
    for c in comps:
        ok &= ~np.isnan(c)
    acc = [np.zeros(comps[0].shape) if dudt is None else _f64(dudt[i]).copy() for i in range(nd)]
    lap = [np.zeros(comps[0].shape) for _ in range(nd)]
    good = ok.copy()
    for a in range(nd):
        ax = nd - 1 - a
        n = comps[0].shape[ax]
        ctr = [slice(None)] * nd; lo = [slice(None)] * nd; hi = [slice(None)] * nd
        ctr[ax] = slice(1, n - 1); lo[ax] = slice(0, n - 2); hi[ax] = slice(2, n)
        ctr, lo, hi = tuple(ctr), tuple(lo), tuple(hi)
        nb_ok = np.zeros_like(ok)
        nb_ok[ctr] = ok[lo] & ok[hi]
        good &= nb_ok
        for i in range(nd):
            d1 = np.zeros(comps[0].shape); d2 = np.zeros(comps[0].shape)
            with np.errstate(invalid="ignore"):
                d1[ctr] = (comps[i][hi] - comps[i][lo]) / (2.0 * h[a])
                d2[ctr] = (comps[i][hi] - 2.0 * comps[i][ctr] + comps[i][lo]) / (h[a] * h[a])
            acc[i] = acc[i] + np.nan_to_num(comps[a]) * np.nan_to_num(d1)
            lap[i] = lap[i] + np.nan_to_num(d2)
    out = []
    for i in range(nd):
        g = -rho * acc[i] + mu * lap[i]
        g[~good] = np.nan
        out.append(g)
    return out


def _central(f, a, h, nd):
    """d f / d x_a by second-order central differences on the interior of axis a (zero on its two end planes, which
    the callers mark missing); numpy axis of a is nd - 1 - a."""
    ax = nd - 1 - a
    n = f.shape[ax]
    ctr = [slice(None)] * nd; lo = [slice(None)] * nd; hi = [slice(None)] * nd
    ctr[ax] = slice(1, n - 1); lo[ax] = slice(0, n - 2); hi[ax] = slice(2, n)
    d = np.zeros(f.shape)
    with np.errstate(invalid="ignore"):
        d[tuple(ctr)] = (f[tuple(hi)] - f[tuple(lo)]) / (2.0 * h)
    return d


def _full_stencil(ok, nd):
    """cells whose 2 nd face neighbours are all inside the box and ok (and that are ok themselves)."""
    good = ok.copy()
    for a in range(nd):
        ax = nd - 1 - a
        n = ok.shape[ax]
        ctr = [slice(None)] * nd; lo = [slice(None)] * nd; hi = [slice(None)] * nd
        ctr[ax] = slice(1, n - 1); lo[ax] = slice(0, n - 2); hi[ax] = slice(2, n)
        nb = np.zeros_like(ok)
        nb[tuple(ctr)] = ok[tuple(lo)] & ok[tuple(hi)]
        good &= nb
    return good


def _stress_index(nd):
    """position of R_ij in the stress list: 2D [xx, yy, xy]; 3D [xx, yy, zz, xy, xz, yz]."""
    if nd == 2:
        return {(0, 0): 0, (1, 1): 1, (0, 1): 2, (1, 0): 2}
    return {(0, 0): 0, (1, 1): 1, (2, 2): 2, (0, 1): 3, (1, 0): 3, (0, 2): 4, (2, 0): 4, (1, 2): 5, (2, 1): 5}


def rans_source(u, v, w, stress, mask, dx, dy, dz=1.0, rho=1.0):
    """Eq. 42: f_i = -rho ( ubar_j d ubar_i / d x_j + d (u'_i u'_j) / d x_j ), viscous terms dropped, written
    out with second-order central differences (reading R-V1).  u, v(, w): mean velocity, (ny, nx) or
    (nz, ny, nx), w = None in 2D; stress: Reynolds stresses [xx, yy, xy] (2D) or [xx, yy, zz, xy, xz, yz] (3D).
    A cell whose stencil touches a missing cell (outside the box, mask == 0, NaN in any input) gets NaN in every component.
    Returns [fx, fy(, fz)]."""
    U = [_f64(u), _f64(v)] + ([] if w is None else [_f64(w)])
    nd = U[0].ndim
    R = [_f64(s) for s in stress]
    idx = _stress_index(nd)
    assert nd == len(U) and len(R) == (3 if nd == 2 else 6)
    h = [dx, dy, dz][:nd]
    ok = np.ones(U[0].shape, bool) if mask is None else (np.asarray(mask) != 0)
    for c in U + R:
        ok &= ~np.isnan(c)
    good = _full_stencil(ok, nd)
    out = []
    for i in range(nd):
        conv = np.zeros(U[0].shape)
        div = np.zeros(U[0].shape)
        for j in range(nd):
            conv = conv + np.nan_to_num(U[j]) * np.nan_to_num(_central(U[i], j, h[j], nd))
            div = div + np.nan_to_num(_central(R[idx[(i, j)]], j, h[j], nd))
        f = -rho * (conv + div)
        f[~good] = np.nan
        out.append(f)
    return out


def compressible_rans_source(u, v, w, stress, mask, dx, dy, dz=1.0, gamma=1.4, mach_inf=2.0, v_inf=1.0, rgas_t_inf=1.0):
    """Eq. 43-44: grad ln(P / P_inf) of the compressible RANS momentum equations for an adiabatic ideal
    gas with negligible density fluctuations.  Step by step:
      T / T_inf = 1 + (gamma - 1)/2 M_inf^2 (1 - V^2 / V_inf^2)                                   (Eq. 43)
      uu_ij = ubar_i ubar_j + (u'_i u'_j)                                                          (:545)
      (delta_ij + uu_ij / (R T)) g_j = -(1 / (R T)) ( d uu_ij / d x_j - (uu_ij / T) d T / d x_j )  (Eq. 44)
    solved for g = grad ln(P / P_inf) cell by cell (numpy.linalg.solve on the 2x2 / 3x3 systems).  rgas_t_inf = R T_inf
    (the only way R and T_inf enter); stress may be None (no Reynolds stresses).  Central differences and missing cells
    as in rans_source.  Returns [gx, gy(, gz)]."""
    U = [_f64(u), _f64(v)] + ([] if w is None else [_f64(w)])
    nd = U[0].ndim
    idx = _stress_index(nd)
    R = None if stress is None else [_f64(s) for s in stress]
    h = [dx, dy, dz][:nd]
    ok = np.ones(U[0].shape, bool) if mask is None else (np.asarray(mask) != 0)
    for c in U + ([] if R is None else R):
        ok &= ~np.isnan(c)
    good = _full_stencil(ok, nd)
    V2 = sum(c * c for c in U)
    theta = 1.0 + 0.5 * (gamma - 1.0) * mach_inf ** 2 * (1.0 - V2 / v_inf ** 2)         # T / T_inf
    RT = rgas_t_inf * theta
    uu = {}
    for i in range(nd):
        for j in range(i, nd):
            uu[(i, j)] = U[i] * U[j] + (0.0 if R is None else R[idx[(i, j)]])
            uu[(j, i)] = uu[(i, j)]
    dth = [_central(theta, j, h[j], nd) for j in range(nd)]
    A = np.zeros(U[0].shape + (nd, nd))
    b = np.zeros(U[0].shape + (nd,))
    with np.errstate(invalid="ignore", divide="ignore"):
        for i in range(nd):
            for j in range(nd):
                A[..., i, j] = (1.0 if i == j else 0.0) + uu[(i, j)] / RT
                b[..., i] += -(1.0 / RT) * (_central(uu[(i, j)], j, h[j], nd) - uu[(i, j)] / theta * dth[j])
    A[~good] = np.eye(nd)
    b[~good] = 0.0
    g = np.linalg.solve(A, b[..., None])[..., 0]
    out = []
    for i in range(nd):
        gi = g[..., i].copy()
        gi[~good] = np.nan
        out.append(gi)
    return out
