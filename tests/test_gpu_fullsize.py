"""BASELINE.json's full-size configs, in the launch configuration bench.py times, against the oracle:
* test_fullsize_config: step outputs at sampled cells (the oracle evaluates S_C, (M x)_C, (W^n x)_C one cell at a
  time) and the device reductions against fp64 sums of the full device arrays;
* test_fullsize_trajectory_vs_oracle: a short fixed-count trajectory against a FULL oracle solve (SURVEY 8(c) parity
  protocol i); skipped BY NAME, with the reason, only if the host cannot hold the oracle's 19 fp64 fields;
* test_converged_parity_fullsize: converged on both sides with the same stopping rules (protocol ii) where the oracle
  finishes in minutes -- configs[2] always, configs[1] / configs[3] fp32 with OMNI_TEST_LONG=1;
* test_converged_field_certified_by_oracle: every config converged on the GPU (Alg. 1 and the cascade solve), then
  eps_R of Eq. 41 re-evaluated by the oracle's per-cell operators over ALL cells (protocol iii)."""
import os

import numpy as np
import pytest

import paper_2311_16935_b200 as omni
from workloads import CONFIGS, make_config

from util import rel_l2_after_mean_removal

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

NSAMP = 20000
CASES = [(1, "f32"), (1, "f64"), (2, "f64"), (3, "f32"), (3, "f64"), (4, "f32")]
TOL_STEP = {"f64": 1e-12, "f32": 4e-6}
TOL_SOLVE = {"f64": 1e-9, "f32": 2e-4}


def _host_mem_gb():
    try:
        import psutil
        return psutil.virtual_memory().available / 2**30
    except Exception:
        pass
    try:
        with open("/proc/meminfo") as fh:
            for line in fh:
                if line.startswith("MemAvailable:"):
                    return int(line.split()[1]) / 2**20
    except Exception:
        pass
    return float("nan")                   # unknown: the callers then try, they do not skip silently


def _load(idx, dtype):
    """Device tensors of configs[idx] in `dtype` and the values the oracle must consume (what the device consumed)."""
    f = make_config(idx, device="cuda")
    tdt = torch.float32 if dtype == "f32" else torch.float64
    g_dev = [torch.from_numpy(c).to(tdt).cuda() for c in f["g"]]
    g_or = [c.cpu().numpy().astype(np.float64) for c in g_dev]
    g_dev += [None] * (3 - len(g_dev))
    g_or += [None] * (3 - len(g_or))
    mask = f["mask"]
    m_dev = None if mask is None else torch.from_numpy(mask).cuda()
    return f, g_dev, g_or, mask, m_dev


@pytest.mark.parametrize("idx,dtype", CASES)
def test_fullsize_config(oracle, idx, dtype):
    f, g_dev, g_or, mask, m_dev = _load(idx, dtype)
    d = f["d"]
    tdt = torch.float32 if dtype == "f32" else torch.float64
    shape = f["g"][0].shape
    N = int(np.prod(shape))
    v = oracle.validity(g_or[0], g_or[1], g_or[2], mask)
    rng = np.random.default_rng(100 + idx)
    # sampled cells: uniform + every kind of boundary (box faces, edges, corners, mask surface)
    cells = rng.choice(N, NSAMP, replace=False)
    edge = np.array([0, 1, shape[-1] - 2, shape[-1] - 1, shape[-1], N - 1, N - 2, N - shape[-1], N // 2])
    cells = np.unique(np.concatenate([cells, edge]))
    if mask is not None:
        from scipy import ndimage
        surf = np.flatnonzero((ndimage.binary_dilation(mask == 0) & (mask == 1)).ravel())
        cells = np.unique(np.concatenate([cells, rng.choice(surf, min(len(surf), 4000), replace=False)]))

    # a2: source term
    S, nS = omni.source(g_dev[0], g_dev[1], g_dev[2], m_dev, d)
    x = rng.standard_normal(shape)
    x_dev = torch.from_numpy(x).to(tdt).cuda()
    x_or = x_dev.cpu().numpy().astype(np.float64) * v
    S_or, Mx_or, Wx_or = oracle.sample(v, g_or[0], g_or[1], g_or[2], x_or, cells, *d)
    S_s = S.flatten()[torch.from_numpy(cells).cuda()].cpu().numpy().astype(np.float64)
    assert np.abs(S_s - S_or).max() <= TOL_STEP[dtype] * np.abs(S_or).max() * 4
    assert nS == pytest.approx(float(torch.linalg.vector_norm(S.double())), rel=1e-12)
    # a4: operator through the CG kernel
    q, pq = omni.apply_M(x_dev, m_dev, d)
    q_s = q.flatten()[torch.from_numpy(cells).cuda()].cpu().numpy().astype(np.float64)
    assert np.abs(q_s - Mx_or).max() <= TOL_STEP[dtype] * np.abs(Mx_or).max() * 8
    xv = x_dev.double() * torch.from_numpy(v).cuda()
    # fp32: the products of a 16-byte chunk are summed in fp32 before the fp64 accumulator (chunk_dot), 2e-7 relative
    # per 4-term partial, averaging down over the 2.6e5+ chunks of a config
    assert pq == pytest.approx(float((xv * q.double()).sum()), rel=1e-10 if dtype == "f64" else 1e-8)
    del q, xv

    # the whole path in bench.py's launch configuration (fixed caps, graph loop)
    tol = 1e-5 if dtype == "f32" else 1e-8
    P, info = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 8, 25)
    assert info["status"] in (0, 1) and info["cg_iters_total"] > 0
    assert info["norm_S"] == pytest.approx(nS, rel=1e-12)
    Pn = torch.nan_to_num(P.double(), nan=0.0)
    assert bool((torch.isnan(P) == (torch.from_numpy(v).cuda() == 0)).all())
    # a3 on the returned field: r at sampled cells against the oracle, eps_R against the full device arrays
    r, eps = omni.residual(g_dev[0], g_dev[1], g_dev[2], m_dev, Pn, d)
    _, MP, WP = oracle.sample(v, None, None, None, Pn.cpu().numpy(), cells, *d)
    r_or = S_or + WP - MP
    r_s = r.flatten()[torch.from_numpy(cells).cuda()].cpu().numpy().astype(np.float64)
    scale = max(np.abs(r_or).max(), np.abs(MP).max() * 1e-3)
    assert np.abs(r_s - r_or).max() <= TOL_STEP[dtype] * 16 * max(np.abs(MP).max(), np.abs(S_or).max())
    assert eps == pytest.approx(float(torch.linalg.vector_norm(r.double())) / nS, rel=1e-6 if dtype == "f32" else 1e-10)
    # the solve's own eps_R (fp64 master pressure) agrees with the residual of the (rounded) returned field
    assert info["eps_R_final"] == pytest.approx(eps, rel=5e-2 if dtype == "f32" else 1e-6)
    assert scale > 0
    del r, Pn, S, x_dev

    # omni_solve_direct at full size: its eps_R against the residual kernel on the returned field, the residual at the
    # sampled cells against the oracle
    Pd, idd = omni.solve_direct(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 2, 60)
    assert idd["status"] in (0, 1) and idd["cg_iters_total"] > 0
    Pn = torch.nan_to_num(Pd.double(), nan=0.0)
    r, eps = omni.residual(g_dev[0], g_dev[1], g_dev[2], m_dev, Pn, d)
    assert idd["eps_R_final"] == pytest.approx(eps, rel=5e-2 if dtype == "f32" else 1e-6)
    _, MP, WP = oracle.sample(v, None, None, None, Pn.cpu().numpy(), cells, *d)
    r_s = r.flatten()[torch.from_numpy(cells).cuda()].cpu().numpy().astype(np.float64)
    assert np.abs(r_s - (S_or + WP - MP)).max() <= TOL_STEP[dtype] * 16 * max(np.abs(MP).max(), np.abs(S_or).max())


@pytest.mark.parametrize("idx,dtype", CASES)
def test_fullsize_trajectory_vs_oracle(oracle, idx, dtype):
    """Short fixed-count trajectory (tol = 0: identical steps on both sides) of Alg. 1 and of the fixed-point solve at the
    FULL size of every config, against a full oracle solve.  The oracle holds 19 fp64 fields plus inputs and outputs
    (24 x 8 x N bytes: 24 GB at 500^3)."""
    f, g_dev, g_or, mask, m_dev = _load(idx, dtype)
    d = f["d"]
    N = int(np.prod(f["g"][0].shape))
    need, have = N * 8 * 24 / 2**30, _host_mem_gb()
    if have == have and have < 1.2 * need:
        pytest.skip(f"host memory: the oracle needs {need:.1f} GiB for configs[{idx}], {have:.1f} GiB available")
    v = oracle.validity(g_or[0], g_or[1], g_or[2], mask)
    mo, mc = (2, 5) if N > 5e7 else (3, 8)
    Pg, ig = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, d, 0.0, mo, mc)
    Po, io = oracle.solve(g_or[0], g_or[1], g_or[2], mask, *d, tol=0.0, max_outer=mo, max_cg=mc)
    assert ig["cg_iters_total"] == io["cg_iters_total"] == mo * mc
    err = rel_l2_after_mean_removal(Pg.cpu().numpy(), Po, v == 1)
    assert err <= TOL_SOLVE[dtype], err
    assert ig["eps_R_final"] == pytest.approx(io["eps_R_final"], rel=1e-3 if dtype == "f32" else 1e-8)
    # the fixed-point solve (omni_solve_direct) on the same footing
    Pg, ig = omni.solve_direct(g_dev[0], g_dev[1], g_dev[2], m_dev, d, 0.0, mo, mc)
    Po, io = oracle.solve_direct(g_or[0], g_or[1], g_or[2], mask, *d, tol=0.0, max_outer=mo, max_cg=mc)
    assert ig["cg_iters_total"] == io["cg_iters_total"] == mo * mc
    err = rel_l2_after_mean_removal(Pg.cpu().numpy(), Po, v == 1)
    assert err <= TOL_SOLVE[dtype], err
    assert ig["eps_R_final"] == pytest.approx(io["eps_R_final"], rel=1e-3 if dtype == "f32" else 1e-8)


LONG = os.environ.get("OMNI_TEST_LONG") == "1"
TOL_CONV = {"f64": 1e-8, "f32": 1e-5}


@pytest.mark.parametrize("idx,dtype,always", [(2, "f64", True), (1, "f32", False), (3, "f32", False)])
def test_converged_parity_fullsize(oracle, idx, dtype, always):
    """SURVEY 8(c) parity protocol ii at full size: BASELINE's tolerance, max_cg = 16 (the tuned cap of BASELINE.md 5a:
    the same converged field), the same stopping rules on both sides; rel-L2 after mean removal <= 1e-9 / 2e-4 and the
    outer-iteration counts within 2 (eps_R carries ~10 % of tol of inner-solve noise near the end).
    The oracle needs about 3 min (configs[2]) / 5 min (configs[1] fp32) / 10 min (configs[3] fp32) on 16 host threads."""
    if not always and not LONG:
        pytest.skip(f"configs[{idx}] {dtype}: the oracle needs 5-10 min to converge; set OMNI_TEST_LONG=1 to run")
    f, g_dev, g_or, mask, m_dev = _load(idx, dtype)
    d, tol = f["d"], TOL_CONV[dtype]
    P, info = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 200000, 16)
    assert info["status"] == 0 and info["eps_R_final"] <= tol
    Po, io = oracle.solve(g_or[0], g_or[1], g_or[2], mask, *d, tol=tol, max_outer=200000, max_cg=16)
    assert io["converged"]
    valid = ~np.isnan(Po)
    assert np.array_equal(np.isnan(P.cpu().numpy()), ~valid)
    err = rel_l2_after_mean_removal(P.cpu().numpy(), Po, valid)
    print(f"configs[{idx}] {dtype}: GPU {info['outer_iters']} outer / {info['cg_iters_total']} CG, oracle "
          f"{io['outer_iters']} / {io['cg_iters_total']}, rel-L2 {err:.3e}")
    assert err <= TOL_SOLVE[dtype], err
    assert abs(info["outer_iters"] - io["outer_iters"]) <= 2, (info, io)
    Pa = f["P"]
    assert rel_l2_after_mean_removal(P.cpu().numpy(), Pa, valid) == pytest.approx(rel_l2_after_mean_removal(Po, Pa, valid), rel=1e-3)


@pytest.mark.parametrize("idx,dtype", [(0, "f64")] + CASES)
def test_converged_field_certified_by_oracle(oracle, idx, dtype):
    """SURVEY 8(c) parity protocol iii (north_star "Target"): the CONVERGED GPU field of every config -- by Alg. 1
    (max_cg 16), by omni_solve_cascade and by omni_solve_pcg -- has its eps_R (Eq. 41 :442) re-evaluated by the oracle's per-cell operators
    over all cells (oracle.eps_R_of_field).  fp64: the oracle must see eps_R <= 1.05 tol.  fp32: the returned field is
    the fp64 master pressure rounded to fp32, and that rounding alone leaves a residual u |L||P| that grows with the
    grid (SURVEY 7 hard part 3), so the oracle's figure is bounded by tol plus that floor, the floor being evaluated by
    the oracle on the same field (the residual change under one more fp32 rounding of P_out has the same statistics).
    configs[4] by Alg. 1 takes about two minutes of GPU time (10 500 outer iterations): here only with OMNI_TEST_LONG=1;
    the default bench.py line runs it and has the oracle certify it (section `converged`)."""
    f, g_dev, g_or, mask, m_dev = _load(idx, dtype)
    d, tol = f["d"], TOL_CONV[dtype]
    P64 = torch.zeros(f["g"][0].shape, dtype=torch.float64, device="cuda") if dtype == "f32" else None
    runs = [("alg1", lambda: omni.solve_ex(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 400000, 16, method="alg1", P64_out=P64)),
            ("cascade", lambda: omni.solve_cascade(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 20, 30000, levels=4)),
            ("pcg", lambda: omni.solve_ex(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 20, 300, method="pcg", P64_out=P64))]
    for name, fn in runs:
        if name == "alg1" and idx == 4 and not LONG:
            # two minutes of GPU time (10 500 outer iterations); the same run, oracle-certified, is part of the default
            # bench.py line (section `converged`)
            print("configs[4] by Alg. 1: set OMNI_TEST_LONG=1 to run it here; bench.py runs and certifies it")
            continue
        P, info = fn()
        assert info["status"] == 0 and info["eps_R_final"] <= tol, (name, info)
        Pn = P.cpu().numpy()
        eps, nr, nS = oracle.eps_R_of_field(g_or[0], g_or[1], g_or[2], mask, Pn, *d)
        assert nS == pytest.approx(info["norm_S"], rel=1e-5 if dtype == "f32" else 1e-11)
        if P64 is not None and name != "cascade":
            # the fp64 master pressure of the fp32 solve (omni_options::d_P64_out) meets tol in the oracle's eyes
            e64, _, _ = oracle.eps_R_of_field(g_or[0], g_or[1], g_or[2], mask, P64.cpu().numpy(), *d)
            print(f"configs[{idx}] {dtype} {name}: oracle eps_R of the fp64 master pressure {e64:.3e}")
            assert e64 <= 1.05 * tol, (name, e64)
        if dtype == "f64":
            bound = 1.05 * tol
        else:
            # floor of an fp32 field: perturb P_out by a relative 2^-24 per cell with alternating sign pattern drawn
            # once (seeded), and let the oracle measure the residual change
            rng = np.random.default_rng(5)
            Pp = Pn.astype(np.float64) * (1.0 + 2.0 ** -24 * rng.uniform(-1.0, 1.0, size=Pn.shape))
            eps_p, _, _ = oracle.eps_R_of_field(g_or[0], g_or[1], g_or[2], mask, Pp, *d)
            floor = abs(eps_p ** 2 - eps ** 2) ** 0.5
            bound = 1.05 * tol + 2.0 * floor
            print(f"  fp32 rounding floor of eps_R on this field: {floor:.3e}")
        print(f"configs[{idx}] {dtype} {name}: GPU eps_R {info['eps_R_final']:.3e} ({info['outer_iters']} outer, "
              f"{info['cg_iters_total']} CG), oracle eps_R of P_out {eps:.3e} (bound {bound:.3e})")
        assert eps <= bound, (name, eps, bound)
        valid = ~np.isnan(Pn)
        assert rel_l2_after_mean_removal(Pn, f["P"], valid) < 0.05


def _quadratic_case(nx, ny, nz, dev):
    """Exact gradient of a quadratic pressure on [0,1]^3, generated on the device slab by slab (fp32), plus a function
    returning the analytic pressure of a z range in fp64.  Pin P7: the trapezoid face rule is exact on
    quadratics, so the fixed point of Alg. 1 IS this pressure up to a constant -- a property that holds at any size."""
    dx, dy, dz = 1.0 / (nx - 1), 1.0 / (ny - 1), 1.0 / (nz - 1)
    x = (torch.arange(nx, device=dev, dtype=torch.float64) * dx).view(1, 1, nx)
    y = (torch.arange(ny, device=dev, dtype=torch.float64) * dy).view(1, ny, 1)
    z = (torch.arange(nz, device=dev, dtype=torch.float64) * dz).view(nz, 1, 1)
    a = dict(xx=1.3, yy=-0.7, zz=0.9, xy=0.5, xz=-0.4, yz=0.8, x=0.2, y=-0.3, z=0.1)

    def slabs(fn):
        out = torch.empty((nz, ny, nx), device=dev, dtype=torch.float32)
        for k0 in range(0, nz, 64):
            k1 = min(nz, k0 + 64)
            out[k0:k1] = fn(z[k0:k1]).expand(k1 - k0, ny, nx).to(torch.float32)
        return out
    g = [slabs(lambda zz: a["xx"] * x + a["xy"] * y + a["xz"] * zz + a["x"]),
         slabs(lambda zz: a["yy"] * y + a["xy"] * x + a["yz"] * zz + a["y"]),
         slabs(lambda zz: a["zz"] * zz + a["xz"] * x + a["yz"] * y + a["z"])]

    def analytic(k0, k1):
        zz = z[k0:k1]
        return (0.5 * (a["xx"] * x * x + a["yy"] * y * y + a["zz"] * zz * zz) + a["xy"] * x * y + a["xz"] * x * zz
                + a["yz"] * y * zz + a["x"] * x + a["y"] * y + a["z"] * zz)
    return g, (dx, dy, dz), analytic


@pytest.mark.parametrize("shape", [(160, 96, 72), (2048, 1024, 1024)])
def test_quadratic_exactness_up_to_maximum_size(shape):
    """Property at any size (no oracle run needed): quadratic P -> exact gradient -> omni_solve_cascade -> P up to a
    constant.  The second shape has 2^31 cells (8.6 GB per fp32 vector, ~125 GB in total): it takes the 64-bit index paths
    of every kernel and anisotropic 3D constants; it runs only with OMNI_TEST_HUGE=1 on a device with >= 150 GB free
    (measured on a B200: 4781 CG iterations, 63 s, rel-L2 5.9e-8)."""
    import os
    nx, ny, nz = shape
    if nx * ny * nz >= 2 ** 31:
        if os.environ.get("OMNI_TEST_HUGE") != "1":
            pytest.skip("set OMNI_TEST_HUGE=1 to run the 2^31-cell case")
        if torch.cuda.mem_get_info()[0] < 150e9:
            pytest.skip("needs 150 GB of free device memory")
    g, d, analytic = _quadratic_case(nx, ny, nz, "cuda")
    P, info = omni.solve_cascade(g[0], g[1], g[2], None, d, 1e-6, 20, 30000, levels=5)
    assert info["status"] == 0 and info["eps_R_final"] <= 1e-6
    del g
    s1 = s2 = sa = saa = 0.0
    n = 0
    for k0 in range(0, nz, 32):
        k1 = min(nz, k0 + 32)
        Pa = analytic(k0, k1)
        dd = P[k0:k1].double() - Pa
        assert not torch.isnan(dd).any()
        s1 += float(dd.sum()); s2 += float((dd * dd).sum()); sa += float(Pa.sum()); saa += float((Pa * Pa).sum())
        n += dd.numel()
    var_d, var_a = s2 / n - (s1 / n) ** 2, saa / n - (sa / n) ** 2
    assert (max(var_d, 0.0) / var_a) ** 0.5 <= 5e-6
