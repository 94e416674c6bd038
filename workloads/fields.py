"""Synthetic analytic pressure fields and their exact gradients.

Stand-ins for the paper's workloads (the paper's own data is not available and is not needed):
  gaussians2d  - smooth vortex-like blobs, like the Taylor vortex 101^2 case
  lamb_oseen2d - vortex + masked disc, like the masked planar PIV case
  fourier3d    - k^-5/3 random Fourier modes cut from a periodic box, like the JHU
                 isotropic-turbulence cut-outs 50^3..500^3
  sphere3d     - potential flow past a masked sphere, like the masked SSPIV volume
Noise levels 0-10 % follow PAPER.md:351, :404 (here added to the gradient, per BASELINE.json).

All fields: domain [0,1]^d, spacing 1/(n-1), cell centres at i/(n-1); P scaled to max|P| = 1 over valid
cells; then i.i.d. Gaussian noise N(0, (s*g_rms)^2) on every component at every cell,
g_rms = sqrt(sum_cells sum_comp g^2 / (d*N_valid)).  RNG: numpy default_rng(seed) (PCG64); parameters are
drawn first, then noise for gx, gy, gz as whole arrays in that order.
Arrays are numpy float64 in C order (nz, ny, nx) / (ny, nx): x is the fastest index.
"""
import math

import numpy as np

# index -> (kind, n, ndim, noise, tol_f64, tol_f32, dtypes) ; BASELINE.json configs[0..4]
CONFIGS = {
    0: dict(kind="gaussians2d", n=64, noise=0.05, dtypes=("f64",)),
    1: dict(kind="lamb_oseen2d", n=1024, noise=0.10, dtypes=("f32", "f64")),
    2: dict(kind="fourier3d", n=128, noise=0.05, dtypes=("f64",)),
    3: dict(kind="sphere3d", n=256, noise=0.05, dtypes=("f32", "f64")),
    4: dict(kind="fourier3d", n=500, noise=0.10, dtypes=("f32",)),
}
TOL = {"f64": 1e-8, "f32": 1e-5}


def _axes(shape):
    return [np.arange(m, dtype=np.float64) / max(m - 1, 1) for m in shape]


def _gaussians2d(shape, rng):
    ny, nx = shape
    c = rng.uniform(0.2, 0.8, size=(3, 2))
    sig = rng.uniform(0.05, 0.2, size=3)
    amp = np.where(rng.random(3) < 0.5, -1.0, 1.0)
    y, x = np.meshgrid(*_axes(shape), indexing="ij")
    P = np.zeros(shape)
    gx = np.zeros(shape)
    gy = np.zeros(shape)
    for m in range(3):
        e = amp[m] * np.exp(-((x - c[m, 0]) ** 2 + (y - c[m, 1]) ** 2) / (2 * sig[m] ** 2))
        P += e
        gx += -(x - c[m, 0]) / sig[m] ** 2 * e
        gy += -(y - c[m, 1]) / sig[m] ** 2 * e
    return P, [gx, gy], None


def _lamb_oseen2d(shape, rng):
    from scipy.special import exp1
    rc = 0.1
    y, x = np.meshgrid(*_axes(shape), indexing="ij")
    xr, yr = x - 0.5, y - 0.5
    r2 = xr * xr + yr * yr
    s = r2 / rc ** 2
    one_m = -np.expm1(-s)
    with np.errstate(divide="ignore", invalid="ignore"):
        P = -(one_m ** 2 / s + 2 * exp1(s) - 2 * exp1(2 * s))
        dPdr_over_r = 2.0 * one_m ** 2 / (rc ** 2 * s ** 2)   # (1/r) dP/dr, same units as P above
    zero = s == 0
    P[zero] = -2.0 * math.log(2.0)
    dPdr_over_r[zero] = 2.0 / rc ** 2
    small = (s < 1e-6) & ~zero
    dPdr_over_r[small] = 2.0 / rc ** 2 * (1 - s[small])
    gx, gy = dPdr_over_r * xr, dPdr_over_r * yr
    mask = ((x - 0.35) ** 2 + (y - 0.60) ** 2 >= 0.05 ** 2).astype(np.uint8)
    return P, [gx, gy], mask


def _fourier_modes(rng, nmodes=256, kmin=1.0, kmax=32.0):
    ks = []
    while len(ks) < nmodes:
        kmag = rng.uniform(kmin, kmax)
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        k = np.rint(kmag * d)
        kn = np.linalg.norm(k)
        if kn < kmin or kn > kmax:
            continue
        ks.append(k)
    k = np.array(ks)
    amp = np.linalg.norm(k, axis=1) ** (-5.0 / 3.0)
    phase = rng.uniform(0, 2 * np.pi, size=nmodes)
    return k, amp, phase


def _fourier3d(shape, rng, device="cpu", kmax=32.0):
    """P = sum_m A_m cos(2 pi k_m.x + phi_m) evaluated as real GEMMs over the mode index."""
    import torch
    nz, ny, nx = shape
    k, amp, phase = _fourier_modes(rng, kmax=kmax)
    dev = torch.device(device)
    z, y, x = [torch.from_numpy(a).to(dev) for a in _axes(shape)]
    kt = torch.from_numpy(k).to(dev)
    two_pi = 2 * math.pi
    ex = torch.exp(1j * two_pi * kt[:, 0:1] * x[None, :])                     # [m, nx]
    ey = torch.exp(1j * two_pi * kt[:, 1:2] * y[None, :])                     # [m, ny]
    ez = torch.exp(1j * (two_pi * kt[:, 2:3] * z[None, :] + torch.from_numpy(phase).to(dev)[:, None]))
    B = (ey[:, :, None] * ex[:, None, :]).reshape(len(amp), ny * nx)          # [m, ny*nx]
    Bs = torch.cat([B.real, B.imag], dim=0)                                   # [2m, ny*nx]
    a = torch.from_numpy(amp).to(dev)[:, None]
    outs = []
    # coefficient per output: P: a ; d/dx_c: i*2pi*k_c*a
    for coef in (a.to(torch.complex128), 1j * two_pi * kt[:, 0:1] * a, 1j * two_pi * kt[:, 1:2] * a, 1j * two_pi * kt[:, 2:3] * a):
        A = coef * ez                                                         # [m, nz]
        As = torch.cat([A.real, -A.imag], dim=0).T.contiguous()               # [nz, 2m]
        outs.append((As @ Bs).reshape(nz, ny, nx).cpu().numpy())
    P, gx, gy, gz = outs
    return P, [gx, gy, gz], None


def _sphere3d(shape, rng):
    a = 0.15
    z, y, x = np.meshgrid(*_axes(shape), indexing="ij", sparse=True)
    X = [x - 0.5, y - 0.5, z - 0.5]
    r2 = X[0] ** 2 + X[1] ** 2 + X[2] ** 2
    mask = (r2 >= a * a).astype(np.uint8)
    r2 = np.where(mask == 1, r2, 1.0)                 # keep the masked interior finite
    r = np.sqrt(r2)
    A = a ** 3 / 2
    # u_i = delta_ix (1 + A/r^3) - 3 A x x_i / r^5          (U = rho = 1)
    u = [(1 + A / r ** 3) - 3 * A * X[0] * X[0] / r ** 5, -3 * A * X[0] * X[1] / r ** 5, -3 * A * X[0] * X[2] / r ** 5]
    P = 0.5 * (1.0 - (u[0] ** 2 + u[1] ** 2 + u[2] ** 2))
    g = []
    for j in range(3):
        # d_j u_i = -3A delta_ix x_j/r^5 - 3A (delta_jx x_i + x delta_ij)/r^5 + 15 A x x_i x_j / r^7
        acc = 0.0
        for i in range(3):
            dj_ui = -3 * A * ((X[j] if i == 0 else 0.0) + (X[i] if j == 0 else 0.0) + (X[0] if i == j else 0.0)) / r ** 5 \
                    + 15 * A * X[0] * X[i] * X[j] / r ** 7
            acc = acc + u[i] * dj_ui
        g.append(-acc * np.ones(shape))
    P = P * np.ones(shape)
    return P, g, mask


_KINDS = {"gaussians2d": _gaussians2d, "lamb_oseen2d": _lamb_oseen2d, "fourier3d": _fourier3d, "sphere3d": _sphere3d}


def make_field(kind, shape, seed, noise, device="cpu", nan_mask=False, kmax=32.0):
    """Returns dict(P, g=[gx,gy(,gz)], mask (uint8 or None), d=(dx,dy,dz), shape, noise, seed).

    shape is numpy order.  The domain is [0,1] along every axis, so non-cubic shapes give anisotropic
    spacing.  kmax caps the fourier3d wavenumbers (small stand-in grids keep the field resolved).  nan_mask=True marks the missing cells by NaN in g instead of a mask array."""
    shape = tuple(int(s) for s in shape)
    rng = np.random.default_rng(seed)
    if kind == "fourier3d":
        P, g, mask = _fourier3d(shape, rng, device, kmax)
    else:
        P, g, mask = _KINDS[kind](shape, rng)
    valid = np.ones(shape, bool) if mask is None else mask.astype(bool)
    scale = 1.0 / np.max(np.abs(P[valid]))
    P = P * scale
    g = [c * scale for c in g]
    nvalid = int(valid.sum())
    g_rms = math.sqrt(sum(float(np.sum(c[valid] ** 2)) for c in g) / (len(g) * nvalid))
    if noise > 0:
        for c in g:
            c += rng.normal(0.0, noise * g_rms, size=shape)
    if mask is not None:
        for c in g:
            c[~valid] = np.nan if nan_mask else 0.0
        P = np.where(valid, P, np.nan)
        if nan_mask:
            mask = None
    sp = [1.0 / max(m - 1, 1) for m in shape]
    d = (sp[-1], sp[-2], sp[-3] if len(shape) == 3 else 1.0)
    return dict(P=P, g=g, mask=mask, d=d, shape=shape, noise=noise, seed=seed, kind=kind, g_rms=g_rms)


def make_config(idx, n=None, device="cpu", noise=None):
    """BASELINE.json configs[idx]; n overrides the edge length (small stand-ins for tests; the fourier3d
    wavenumber cap then shrinks to n/4 so the stand-in stays as well resolved as the full-size field)."""
    c = CONFIGS[idx]
    n = n or c["n"]
    ndim = 2 if c["kind"].endswith("2d") else 3
    kmax = 32.0 if n >= 128 else max(2.0, n / 4.0)
    f = make_field(c["kind"], (n,) * ndim, seed=idx, noise=c["noise"] if noise is None else noise, device=device,
                   kmax=kmax)
    f["config"] = idx
    return f
