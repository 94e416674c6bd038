"""ctypes wrapper around oracle/omni_oracle.c  -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module.  It never imports paper_2311_16935_b200 and shares nothing with the CUDA path.
Everything here is argument marshalling for the C functions; the arithmetic lives in omni_oracle.c,
each function citing the PAPER.md passage it follows.
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


def solve_direct(gx, gy, gz, mask, dx, dy, dz, tol, max_outer, max_cg, P_init=None):
    """Fixed point of Algorithm 1 by CG on L P = S (oracle_solve_direct; not the paper's iteration).  Returns (P, info)."""
    gx, gy = _f64(gx), _f64(gy)
    nx, ny, nz = _dims(gx.shape)
    gz = _f64(gz) if gz is not None else None
    if nz > 1 and gz is None:
        raise ValueError("gz required in 3D")
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    P = np.zeros(gx.shape)
    info = Info()
    P0 = None if P_init is None else _f64(P_init)
    f = lib().oracle_solve_direct
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
