"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element, on seeded inputs.

Tolerances: fp64 rel-L2 after mean removal <= 1e-9, fp32 <= 2e-4 (north_star); single-step
operators are compared entry-wise with a bound derived from the arithmetic (a handful of roundings of terms of size
max|term|): 1e-13 relative to the largest entry in fp64, 2e-6 in fp32.
"""
import numpy as np
import pytest

import paper_2311_16935_b200 as omni
from workloads import make_config, make_field

from util import rel_l2_after_mean_removal, to_dev

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_STEP = {"f64": 1e-13, "f32": 2e-6}
TOL_SOLVE = {"f64": 1e-9, "f32": 2e-4}
TDT = {"f64": torch.float64, "f32": torch.float32}


def _inputs(f, dtype, mask=None):
    """Device tensors + the values the oracle must consume (fp32 runs: the fp32-rounded inputs)."""
    np_dt = np.float32 if dtype == "f32" else np.float64
    g_host = [np.ascontiguousarray(c.astype(np_dt)) for c in f["g"]]
    g_dev = [to_dev(c) for c in g_host] + [None] * (3 - len(g_host))
    g_or = [c.astype(np.float64) for c in g_host] + [None] * (3 - len(g_host))
    m = f["mask"] if mask is None else mask
    return g_dev, g_or, (None if m is None else to_dev(m.astype(np.uint8))), m


def _random_mask(shape, seed, frac):
    rng = np.random.default_rng(seed)
    return (rng.random(shape) > frac).astype(np.uint8)


SHAPES = [((37, 300), 0.1), ((9, 31, 150), 0.1), ((5, 16, 264), 0.0), ((17, 29, 9), 0.3), ((1, 77), 0.0), ((40, 3, 20), 0.05)]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape,frac", SHAPES)
def test_source_and_operator_steps(oracle, dtype, shape, frac):
    """a1+a2 (S), a4 (q = M p) and a3 (r = S - L P) against the oracle's stored-weight operators: ragged sizes
    spanning several tiles, random masks, anisotropic spacing."""
    kind = "gaussians2d" if len(shape) == 2 else "fourier3d"
    f = make_field(kind, shape, seed=11, noise=0.1, kmax=3.0)
    mask = _random_mask(shape, 5, frac) if frac > 0 else None
    g_dev, g_or, m_dev, m = _inputs(f, dtype, mask)
    d = f["d"]
    v = oracle.validity(g_or[0], g_or[1], g_or[2], m)
    w1, w0, w0C = oracle.weights(v, *d)
    S_or = oracle.source(v, w1, w0, g_or[0], g_or[1], g_or[2], *d)

    S, nS = omni.source(g_dev[0], g_dev[1], g_dev[2], m_dev, d)
    S = S.cpu().numpy().astype(np.float64)
    scale = np.abs(S_or).max()
    assert np.abs(S - S_or).max() <= TOL_STEP[dtype] * scale * 4
    assert nS == pytest.approx(np.linalg.norm(S_or), rel=10 * TOL_STEP[dtype])
    assert np.all(S[v == 0] == 0)

    rng = np.random.default_rng(3)
    p = rng.normal(size=shape)
    p_dev = to_dev(p, TDT[dtype])
    p_or = p_dev.cpu().numpy().astype(np.float64) * v
    q, pq = omni.apply_M(p_dev, m_dev if m is not None else None, d)
    # validity for apply_M comes from the mask alone; these inputs carry no NaN so it equals v
    q = q.cpu().numpy().astype(np.float64)
    q_or = oracle.apply_M(v, w1, p_or)
    assert np.abs(q - q_or).max() <= TOL_STEP[dtype] * np.abs(q_or).max() * 8
    assert pq == pytest.approx(float(np.sum(p_or * q_or)), rel=1e-5 if dtype == "f32" else 1e-11)
    assert np.all(q[v == 0] == 0)

    P = rng.normal(size=shape)
    r, eps = omni.residual(g_dev[0], g_dev[1], g_dev[2], m_dev, to_dev(P), d)
    r = r.cpu().numpy().astype(np.float64)
    Pv = P * v
    r_or = S_or + oracle.apply_Wn(v, w0, w0C, Pv) - oracle.apply_M(v, w1, Pv)
    assert np.abs(r - r_or).max() <= TOL_STEP[dtype] * max(np.abs(r_or).max(), np.abs(Pv).max()) * 8
    assert eps == pytest.approx(np.linalg.norm(r_or) / np.linalg.norm(S_or), rel=1e-5 if dtype == "f32" else 1e-10)


# omni_set_loop_mode; the default (0) picks one of the three by grid size
LOOPS = {"graph": 2, "persistent": 3, "loopk": 4, "resident": 5}


@pytest.fixture(params=list(LOOPS))
def forced_loop(request):
    """Runs a test once per loop driver (the grids here are small enough that the default would always pick one)."""
    prev = omni.set_loop_mode(LOOPS[request.param])
    yield request.param
    omni.set_loop_mode(prev)


def _solve_both(oracle, f, dtype, tol, max_outer, max_cg, mask=None, nan_mask=False, loop=None):
    g_dev, g_or, m_dev, m = _inputs(f, dtype, mask)
    d = f["d"]
    prev = omni.set_loop_mode(LOOPS[loop]) if loop else None
    try:
        P, info = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, max_outer, max_cg)
        torch.cuda.synchronize()
    finally:
        if loop:
            omni.set_loop_mode(prev)
    Po, io = oracle.solve(g_or[0], g_or[1], g_or[2], m, *d, tol=tol, max_outer=max_outer, max_cg=max_cg)
    return P.cpu().numpy(), info, Po, io


TRAJ = [("gaussians2d", (64, 64), None), ("lamb_oseen2d", (150, 130), None), ("fourier3d", (20, 33, 140), None),
        ("sphere3d", (40, 36, 44), None), ("fourier3d", (12, 30, 270), 0.15),
        # rows that end with a chunk made only of pad cells (nx = 4 mod 8 in fp32, 2 mod 4 in fp64), like 500^3
        ("gaussians2d", (21, 132), None), ("fourier3d", (9, 19, 66), None)]


@pytest.mark.parametrize("loop", list(LOOPS))
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("kind,shape,frac", TRAJ)
def test_trajectory_parity(oracle, dtype, kind, shape, frac, loop):
    """Same inputs, tol = 0, fixed iteration counts: both sides execute identical steps (SURVEY 8c protocol i)."""
    f = make_field(kind, shape, seed=7, noise=0.05, kmax=4.0)
    mask = None
    if frac:
        mask = _random_mask(shape, 9, frac)
    P, info, Po, io = _solve_both(oracle, f, dtype, 0.0, 6, 20, mask, loop=loop)
    valid = ~np.isnan(Po)
    assert np.array_equal(np.isnan(P), ~valid)
    assert info["outer_iters"] == io["outer_iters"] == 6
    assert info["cg_iters_total"] == io["cg_iters_total"]
    assert info["status"] == omni.binding.OMNI_NOT_CONVERGED
    err = rel_l2_after_mean_removal(P, Po, valid)
    assert err <= TOL_SOLVE[dtype], err
    assert info["norm_S"] == pytest.approx(io["norm_S"], rel=1e-5 if dtype == "f32" else 1e-12)
    assert info["eps_R_final"] == pytest.approx(io["eps_R_final"], rel=2e-3 if dtype == "f32" else 1e-7)


SMALL = [(4, 4, 4), (5, 4, 9), (3, 7, 12), (2, 6, 10), (4, 9), (3, 5), (2, 2), (6, 1, 7), (1, 1, 9), (7, 5, 4), (9, 4, 5)]


@pytest.mark.parametrize("loop", list(LOOPS))
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape", SMALL)
def test_small_and_thin_grids(oracle, dtype, shape, loop):
    """Axes of length 1..5: every cell is a face / edge / corner cell, the per-axis face corrections overlap, and
    axes shorter than 4 fall back to flagged groups (coded path).  With and without a masked cell."""
    rng = np.random.default_rng(sum(shape))
    g = [rng.normal(size=shape) for _ in range(len(shape))]
    f = dict(g=g, mask=None, d=tuple(0.3 + 0.2 * a for a in range(3)))
    for with_mask in (False, True):
        mask = None
        if with_mask:
            mask = np.ones(shape, np.uint8)
            mask[tuple(s // 2 for s in shape)] = 0
            if mask.sum() == 0:
                continue
        P, info, Po, io = _solve_both(oracle, f, dtype, 0.0, 4, 6, mask, loop=loop)
        valid = ~np.isnan(Po)
        assert np.array_equal(np.isnan(P), ~valid)
        assert info["cg_iters_total"] == io["cg_iters_total"]
        if valid.sum() > 1 and np.nanmax(np.abs(Po)) > 0:
            Pz, Poz = np.nan_to_num(P), np.nan_to_num(Po)
            assert np.abs(Pz - Poz).max() <= (1e-10 if dtype == "f64" else 2e-4) * np.abs(Poz).max(), (shape, with_mask)


@pytest.mark.parametrize("loop", list(LOOPS))
@pytest.mark.parametrize("seed", range(24))
def test_fuzz_random_shapes_masks_spacings(oracle, seed, loop):
    """Seeded fuzz: random 2D/3D shapes (tile tails, pad-only chunks, thin axes), random mask densities including
    masks touching the box faces, random anisotropic spacing; operator, residual and a short solve against the oracle."""
    rng = np.random.default_rng(1000 + seed)
    nd = 2 if seed % 3 == 0 else 3
    shape = tuple(int(rng.integers(1, 12)) for _ in range(nd - 1)) + (int(rng.integers(1, 200)),)
    dtype = "f64" if seed % 2 == 0 else "f32"
    d = tuple(float(rng.uniform(0.2, 2.0)) for _ in range(3))
    frac = [0.0, 0.05, 0.3][seed % 3]
    mask = (rng.random(shape) > frac).astype(np.uint8) if frac > 0 else None
    g = [rng.normal(size=shape) for _ in range(nd)]
    f = dict(g=g, mask=mask, d=d)
    g_dev, g_or, m_dev, m = _inputs(f, dtype, mask)
    v = oracle.validity(g_or[0], g_or[1], g_or[2], m)
    if v.sum() == 0:
        pytest.skip("everything masked")
    w1, w0, w0C = oracle.weights(v, *d)
    p = rng.normal(size=shape)
    p_dev = to_dev(p, TDT[dtype])
    p_or = p_dev.cpu().numpy().astype(np.float64) * v
    q, _ = omni.apply_M(p_dev, m_dev, d)
    q_or = oracle.apply_M(v, w1, p_or)
    assert np.abs(q.cpu().numpy() - q_or).max() <= TOL_STEP[dtype] * 8 * max(np.abs(q_or).max(), 1e-30), (shape, dtype)
    P, info, Po, io = _solve_both(oracle, f, dtype, 0.0, 3, 5, mask, loop=loop)
    assert info["cg_iters_total"] == io["cg_iters_total"]
    assert np.array_equal(np.isnan(P), np.isnan(Po))
    scale = np.nanmax(np.abs(Po)) if np.isfinite(Po).any() else 0.0
    if scale > 0:
        assert np.nanmax(np.abs(np.nan_to_num(P) - np.nan_to_num(Po))) <= (1e-10 if dtype == "f64" else 2e-4) * scale, (shape, dtype)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_batch2d_and_first_guess(oracle, dtype, forced_loop):
    """omni_solve_batch2d_*: stacked 2D snapshots on one mask against the oracle's stacked solve (same joint CG scalars),
    with and without a first guess; nb = 1 is bit-identical to omni_solve_*; a converged first guess stops at once."""
    fs = [make_field("lamb_oseen2d", (45, 140), seed=s, noise=0.05) for s in range(5)]
    np_dt = np.float32 if dtype == "f32" else np.float64
    gx = np.stack([f["g"][0] for f in fs]).astype(np_dt); gy = np.stack([f["g"][1] for f in fs]).astype(np_dt)
    m, d = fs[0]["mask"], fs[0]["d"]
    gxd, gyd, md = to_dev(gx), to_dev(gy), to_dev(m)
    tolp = 1e-9 if dtype == "f64" else 2e-4
    rng = np.random.default_rng(5)
    P0 = (0.1 * rng.normal(size=gx.shape)).astype(np_dt)
    for init in (None, P0):
        P, info = omni.solve_batch2d(gxd, gyd, md, d, 0.0, 5, 12, P_init=None if init is None else to_dev(init))
        Po, io = oracle.solve_batch2d(gx.astype(np.float64), gy.astype(np.float64), m, d[0], d[1], 0.0, 5, 12,
                                      P_init=None if init is None else init.astype(np.float64))
        assert info["cg_iters_total"] == io["cg_iters_total"] == 60
        Pn = P.cpu().numpy()
        assert np.array_equal(np.isnan(Pn), np.isnan(Po))
        for b in range(5):
            valid = ~np.isnan(Po[b])
            assert rel_l2_after_mean_removal(Pn[b], Po[b], valid) <= tolp
        assert info["eps_R_final"] == pytest.approx(io["eps_R_final"], rel=2e-3 if dtype == "f32" else 1e-7)
    # nb = 1: same bits as the plain 2D entry point
    Pb, ib = omni.solve_batch2d(gxd[:1].contiguous(), gyd[:1].contiguous(), md, d, 1e-4, 50, 12)
    Ps, is_ = omni.solve(gxd[0].contiguous(), gyd[0].contiguous(), None, md, d, 1e-4, 50, 12)
    assert ib == is_ and np.array_equal(Pb[0].cpu().numpy(), Ps.cpu().numpy(), equal_nan=True)
    # converged field as first guess: no iteration; P returned unchanged (to the dtype)
    tol = 1e-5 if dtype == "f32" else 1e-8
    Pc, ic = omni.solve_batch2d(gxd, gyd, md, d, tol, 100000, 32)
    assert ic["status"] == 0
    # what the joint stopping rule guarantees per snapshot (include/omni.h): ||r_b|| <= tol ||S|| of the STACK, i.e.
    # eps_R,b <= tol ||S|| / ||S_b||, with eps_R,b (Eq. 41) evaluated by the oracle's stored-weight operators
    v2 = oracle.validity(gx[0].astype(np.float64), gy[0].astype(np.float64), None, m)
    w1, w0, w0C = oracle.weights(v2, d[0], d[1])
    rb, Sb = [], []
    for b in range(5):
        S_b = oracle.source(v2, w1, w0, gx[b].astype(np.float64), gy[b].astype(np.float64), None, d[0], d[1])
        P_b = np.nan_to_num(Pc[b].cpu().numpy().astype(np.float64))
        r_b = S_b + oracle.apply_Wn(v2, w0, w0C, P_b) - oracle.apply_M(v2, w1, P_b)
        rb.append(np.linalg.norm(r_b)); Sb.append(np.linalg.norm(S_b))
    normS = float(np.sqrt(np.sum(np.square(Sb))))
    assert ic["norm_S"] == pytest.approx(normS, rel=1e-5 if dtype == "f32" else 1e-12)
    slack = 3.0 if dtype == "f32" else 1.05           # fp32: P_out is the fp64 master pressure rounded to fp32
    for b in range(5):
        assert rb[b] <= slack * tol * normS, (b, rb[b] / Sb[b])          # eps_R,b <= tol ||S|| / ||S_b||
    assert np.sqrt(np.sum(np.square(rb))) / normS <= slack * tol
    Pw, iw = omni.solve_batch2d(gxd, gyd, md, d, 2 * tol, 100, 32, P_init=torch.nan_to_num(Pc))
    assert iw["outer_iters"] == 0 and iw["cg_iters_total"] == 0
    assert torch.allclose(torch.nan_to_num(Pw), torch.nan_to_num(Pc), rtol=0, atol=1e-6 if dtype == "f32" else 1e-13)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_direct_batch2d(oracle, dtype, forced_loop):
    """omni_solve_direct_batch2d_*: the stacked snapshots with the inner systems L P = S, against the oracle's, with
    and without a first guess; converged, every snapshot meets the tolerance of the joint system."""
    fs = [make_field("lamb_oseen2d", (45, 140), seed=s, noise=0.05) for s in range(4)]
    np_dt = np.float32 if dtype == "f32" else np.float64
    gx = np.stack([f["g"][0] for f in fs]).astype(np_dt); gy = np.stack([f["g"][1] for f in fs]).astype(np_dt)
    m, d = fs[0]["mask"], fs[0]["d"]
    gxd, gyd, md = to_dev(gx), to_dev(gy), to_dev(m)
    rng = np.random.default_rng(6)
    P0 = (0.1 * rng.normal(size=gx.shape)).astype(np_dt)
    for init in (None, P0):
        P, info = omni.solve_batch2d(gxd, gyd, md, d, 0.0, 2, 30, P_init=None if init is None else to_dev(init), direct=True)
        Po, io = oracle.solve_batch2d(gx.astype(np.float64), gy.astype(np.float64), m, d[0], d[1], 0.0, 2, 30,
                                      P_init=None if init is None else init.astype(np.float64), direct=True)
        assert info["cg_iters_total"] == io["cg_iters_total"] == 60
        Pn = P.cpu().numpy()
        assert np.array_equal(np.isnan(Pn), np.isnan(Po))
        for b in range(4):
            assert rel_l2_after_mean_removal(Pn[b], Po[b], ~np.isnan(Po[b])) <= TOL_SOLVE[dtype]
    tol = 1e-5 if dtype == "f32" else 1e-8
    Pc, ic = omni.solve_batch2d(gxd, gyd, md, d, tol, 20, 3000, direct=True)
    assert ic["status"] == 0 and ic["eps_R_final"] <= tol
    P2, i2 = omni.solve_batch2d(gxd, gyd, md, d, tol, 200000, 16)
    assert i2["status"] == 0 and ic["cg_iters_total"] * 5 < i2["cg_iters_total"]
    for b in range(4):
        valid = ~torch.isnan(Pc[b]).cpu().numpy()
        assert rel_l2_after_mean_removal(P2[b].cpu().numpy(), Pc[b].cpu().numpy(), valid) <= (1e-4 if dtype == "f64" else 5e-3)


def test_converged_parity_config0(oracle):
    """BASELINE configs[0]: 64^2 fp64, tol 1e-8, converged on both sides with the same stopping rules; and the
    recovered field matches the analytic P up to a constant at the discretisation + noise level."""
    f = make_config(0)
    P, info, Po, io = _solve_both(oracle, f, "f64", 1e-8, 100000, 1000)
    assert info["status"] == 0 and io["converged"]
    # the inner solves stop at 0.1*tol*|S|, so eps_R carries ~10 % of tol of inner-solve noise near the end and the
    # two sides may cross tol one outer iteration apart; the fields still agree to 1e-9
    assert abs(info["outer_iters"] - io["outer_iters"]) <= 1
    valid = np.ones(P.shape, bool)
    assert rel_l2_after_mean_removal(P, Po, valid) <= 1e-9
    assert info["eps_R_final"] <= 1e-8
    assert rel_l2_after_mean_removal(P, f["P"], valid) < 0.05


@pytest.mark.parametrize("dtype,tol", [("f64", 1e-8), ("f32", 1e-5)])
def test_converged_parity_small_standins(oracle, dtype, tol):
    """Small stand-ins of configs 1 and 3 (masked 2D vortex 96^2, masked sphere flow 32^3), converged."""
    for idx, n in ((1, 96), (3, 32)):
        f = make_config(idx, n)
        P, info, Po, io = _solve_both(oracle, f, dtype, tol, 200000, 400)
        assert info["status"] == 0 and io["converged"], (idx, info, io)
        valid = ~np.isnan(Po)
        assert rel_l2_after_mean_removal(P, Po, valid) <= TOL_SOLVE[dtype]
        if dtype == "f64":
            assert abs(info["outer_iters"] - io["outer_iters"]) <= 2


def test_graph_and_host_loops_are_bit_identical():
    f = make_field("sphere3d", (24, 30, 40), seed=2, noise=0.05)
    for dtype in ("f64", "f32"):
        g_dev, _, m_dev, _ = _inputs(f, dtype)
        res = []
        for mode in (2, 1):
            prev = omni.set_loop_mode(mode)
            try:
                P, info = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, f["d"], 1e-4, 50, 12)
            finally:
                omni.set_loop_mode(prev)
            res.append((P.cpu().numpy(), info))
        assert res[0][1] == res[1][1]
        assert np.array_equal(res[0][0], res[1][0], equal_nan=True)
        # determinism: same call twice, same bits -- in the graph loop, in the persistent kernel and in the cooperative
        # tile-loop kernel, whose reductions run in another (fixed) order: same iteration counts, fields equal to rounding
        for mode in (2, 3, 4):
            prev = omni.set_loop_mode(mode)
            try:
                Pa, ia = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, f["d"], 1e-4, 50, 12)
                Pb, ib = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, f["d"], 1e-4, 50, 12)
            finally:
                omni.set_loop_mode(prev)
            assert ia == ib and np.array_equal(Pa.cpu().numpy(), Pb.cpu().numpy(), equal_nan=True)
            if mode == 2:
                assert np.array_equal(res[0][0], Pa.cpu().numpy(), equal_nan=True)
            else:
                assert ia["outer_iters"] == res[0][1]["outer_iters"] and ia["cg_iters_total"] == res[0][1]["cg_iters_total"]
                valid = ~np.isnan(res[0][0])
                assert rel_l2_after_mean_removal(Pa.cpu().numpy(), res[0][0], valid) <= (1e-11 if dtype == "f64" else 1e-5)


def _direct_both(oracle, f, dtype, tol, max_outer, max_cg, mask=None, loop=None, P_init=None):
    g_dev, g_or, m_dev, m = _inputs(f, dtype, mask)
    d = f["d"]
    p_dev = p_or = None
    if P_init is not None:
        p_dev = to_dev(P_init, TDT[dtype])
        p_or = p_dev.cpu().numpy().astype(np.float64)
    prev = omni.set_loop_mode(LOOPS[loop]) if loop else None
    try:
        P, info = omni.solve_direct(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, max_outer, max_cg, P_init=p_dev)
        torch.cuda.synchronize()
    finally:
        if loop:
            omni.set_loop_mode(prev)
    Po, io = oracle.solve_direct(g_or[0], g_or[1], g_or[2], m, *d, tol=tol, max_outer=max_outer, max_cg=max_cg, P_init=p_or)
    return P.cpu().numpy(), info, Po, io


@pytest.mark.parametrize("loop", list(LOOPS))
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("kind,shape,frac", TRAJ + [("fourier3d", (5, 4, 9), 0.2), ("gaussians2d", (3, 70), None)])
def test_direct_solve_trajectory_parity(oracle, dtype, kind, shape, frac, loop):
    """omni_solve_direct (CG on L P = S, SURVEY 8(f) NEXT-2 iii) against oracle.solve_direct: tol = 0 and fixed caps,
    both sides execute the same 2 x 25 CG steps (the second outer iteration restarts from the fp64 residual)."""
    f = make_field(kind, shape, seed=7, noise=0.05, kmax=4.0)
    mask = _random_mask(shape, 9, frac) if frac else None
    # every other case starts from a first guess instead of zero
    P_init = np.random.default_rng(3).normal(size=shape) * 0.1 if (len(shape) + shape[-1]) % 2 else None
    P, info, Po, io = _direct_both(oracle, f, dtype, 0.0, 2, 25, mask, loop=loop, P_init=P_init)
    valid = ~np.isnan(Po)
    assert np.array_equal(np.isnan(P), ~valid)
    assert info["outer_iters"] == io["outer_iters"] == 2
    assert info["cg_iters_total"] == io["cg_iters_total"]
    err = rel_l2_after_mean_removal(P, Po, valid)
    assert err <= TOL_SOLVE[dtype], err
    assert info["eps_R_final"] == pytest.approx(io["eps_R_final"], rel=5e-3 if dtype == "f32" else 1e-6)


@pytest.mark.parametrize("dtype,tol", [("f64", 1e-8), ("f32", 1e-5)])
def test_direct_solve_converged(oracle, dtype, tol, forced_loop):
    """Converged: the direct solve meets Eq. 41 with the oracle's operators, agrees with the oracle's direct solve and
    lands on the field Algorithm 1 converges to (configs[0], and masked stand-ins of configs 1 and 3)."""
    for idx, n in ((0, None), (1, 96), (3, 32)):
        f = make_config(idx, n) if n else make_config(idx)
        P, info, Po, io = _direct_both(oracle, f, dtype, tol, 20, 3000)
        assert info["status"] == 0 and io["converged"], (idx, info, io)
        assert info["eps_R_final"] <= tol
        if dtype == "f64":
            assert abs(info["cg_iters_total"] - io["cg_iters_total"]) <= max(3, io["cg_iters_total"] // 50), (info, io)
        else:   # fp32 CG: the recursive residual drifts from the true one, the fp64 outer check restarts it once or twice
            assert info["cg_iters_total"] <= 1.5 * io["cg_iters_total"] + 10 and info["outer_iters"] <= io["outer_iters"] + 3, (info, io)
        valid = ~np.isnan(Po)
        assert rel_l2_after_mean_removal(P, Po, valid) <= TOL_SOLVE[dtype] * (100 if dtype == "f64" else 1)
        # the residual of the GPU field, re-evaluated by the oracle's stored-weight operators in fp64 (r0 = W^n P + S - M P)
        g_dev, g_or, m_dev, m = _inputs(f, dtype)
        v = oracle.validity(g_or[0], g_or[1], g_or[2], m)
        w1, w0, w0C = oracle.weights(v, *f["d"])
        S = oracle.source(v, w1, w0, g_or[0], g_or[1], g_or[2], *f["d"])
        Pz = np.nan_to_num(P.astype(np.float64))
        r0 = oracle.apply_Wn(v, w0, w0C, Pz) + S - oracle.apply_M(v, w1, Pz)
        assert np.linalg.norm(r0) / np.linalg.norm(S) <= (1.05 * tol if dtype == "f64" else 3 * tol)
        # same fixed point as the two-level iteration
        P2, i2 = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, f["d"], tol, 200000, 16)
        assert i2["status"] == 0
        assert info["cg_iters_total"] * 5 < i2["cg_iters_total"]
        assert rel_l2_after_mean_removal(P2.cpu().numpy(), P, valid) <= (1e-4 if dtype == "f64" else 5e-3)


@pytest.mark.parametrize("dtype,tol", [("f64", 1e-8), ("f32", 1e-5)])
def test_cascade_first_guess(oracle, dtype, tol, forced_loop):
    """omni_solve_cascade_*: the coarse levels only supply a first guess, so what is checked is what is unique -- the
    returned field meets Eq. 41 with the oracle's operators and equals the direct solve's (hence the oracle's) to the
    tolerance -- plus that the guess pays (fewer finest-level CG iterations at the fp32 tolerance).  levels = 0 is the direct solve, bitwise.
    Odd sizes (ragged children), a masked 3D case, a 2D case."""
    cases = [("sphere3d", (45, 51, 67), 3), ("lamb_oseen2d", (150, 131), 4), ("fourier3d", (33, 40, 38), 2)]
    for kind, shape, levels in cases:
        f = make_field(kind, shape, seed=4, noise=0.05, kmax=3.0)
        g_dev, g_or, m_dev, m = _inputs(f, dtype)
        d = f["d"]
        Pd, idd = omni.solve_direct(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 20, 5000)
        P0, i0 = omni.solve_cascade(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 20, 5000, levels=0)
        assert i0 == idd and np.array_equal(P0.cpu().numpy(), Pd.cpu().numpy(), equal_nan=True)
        Pc, ic = omni.solve_cascade(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 20, 5000, levels=levels)
        assert ic["status"] == 0 and ic["eps_R_final"] <= tol
        # the guess pays at the fp32 tolerance (the smooth part of the error is gone); at 1e-8 on these small noisy cases
        # the finest level still has to resolve the noise and the count is about the same
        if dtype == "f32":
            assert ic["cg_iters_total"] < idd["cg_iters_total"], (kind, ic, idd)
        else:
            assert ic["cg_iters_total"] <= 1.15 * idd["cg_iters_total"] + 5, (kind, ic, idd)
        Pn, Pdn = Pc.cpu().numpy().astype(np.float64), Pd.cpu().numpy().astype(np.float64)
        valid = ~np.isnan(Pdn)
        assert np.array_equal(np.isnan(Pn), ~valid)
        v = oracle.validity(g_or[0], g_or[1], g_or[2], m)
        assert np.array_equal(v == 1, valid)
        w1, w0, w0C = oracle.weights(v, *d)
        S = oracle.source(v, w1, w0, g_or[0], g_or[1], g_or[2], *d)
        Pz = np.nan_to_num(Pn)
        r0 = oracle.apply_Wn(v, w0, w0C, Pz) + S - oracle.apply_M(v, w1, Pz)
        assert np.linalg.norm(r0) / np.linalg.norm(S) <= (1.05 * tol if dtype == "f64" else 3 * tol)
        # same field as the direct solve (one connected component in these cases): tolerance-level agreement
        assert rel_l2_after_mean_removal(Pn, Pdn, valid) <= (1e-5 if dtype == "f64" else 5e-3)
        Po, io = oracle.solve_direct(g_or[0], g_or[1], g_or[2], m, *d, tol=tol, max_outer=20, max_cg=5000)
        assert rel_l2_after_mean_removal(Pn, Po, valid) <= (1e-5 if dtype == "f64" else 5e-3)


@pytest.mark.parametrize("coop", [3, 5])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_persistent_loop_stress(dtype, coop):
    """The cooperative kernels' grid barriers (3: the persistent loop's fenced ones; 5: the SM-resident loop's fenced
    and relaxed ones plus its halo messages) under every mix of phases (max_cg = 0, 1, 2, 3, 16: the outer and the inner
    barriers interleave differently, the lazy delta is flushed at even and odd counts), on grids from one CTA to one CTA
    per SM, repeated: every repetition gives the same bits, the same iteration counts as the graph loop, and the same
    field to rounding.  (1030 x 1000 in fp64: r and delta beside p, no room for q; 100 x 108 x 120 in fp64: r beside p,
    delta lazy in global memory; r outside the SM is covered at 128^3 fp64 by tests/test_gpu_fullsize.py.)"""
    cases = [("gaussians2d", (64, 64)), ("lamb_oseen2d", (700, 300)), ("sphere3d", (48, 40, 36)), ("fourier3d", (9, 19, 66))]
    if coop == 5:
        cases += [("lamb_oseen2d", (1030, 1000)), ("fourier3d", (100, 108, 120))]
    for kind, shape in cases:
        f = make_field(kind, shape, seed=3, noise=0.05, kmax=4.0)
        g_dev, _, m_dev, _ = _inputs(f, dtype)
        for max_outer, max_cg in ((3, 0), (12, 1), (9, 2), (7, 3), (5, 16)):
            out = {}
            for mode, reps in ((2, 1), (coop, 4)):
                prev = omni.set_loop_mode(mode)
                try:
                    out[mode] = [omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, f["d"], 0.0, max_outer, max_cg) for _ in range(reps)]
                finally:
                    omni.set_loop_mode(prev)
            Pg, ig = out[2][0]
            Pg = Pg.cpu().numpy()
            valid = ~np.isnan(Pg)
            P0 = out[coop][0][0].cpu().numpy()
            for P, info in out[coop]:
                assert info == out[coop][0][1], (kind, shape, max_outer, max_cg)
                assert np.array_equal(P.cpu().numpy(), P0, equal_nan=True), (kind, shape, max_outer, max_cg)
            assert out[coop][0][1]["cg_iters_total"] == ig["cg_iters_total"] and out[coop][0][1]["outer_iters"] == ig["outer_iters"]
            if max_cg > 0:
                assert rel_l2_after_mean_removal(P0, Pg, valid) <= (1e-11 if dtype == "f64" else 1e-5), (kind, shape, max_outer, max_cg)
            else:
                assert np.array_equal(P0, Pg, equal_nan=True)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_velocity_source_parity(oracle, dtype):
    """omni_velocity_source_* (g = f(u), Eq. 1 :23) against oracle.velocity_source, entry by entry: 3D and 2D, ragged
    sizes, random masks plus NaN velocities, steady and with local accelerations; the NaN pattern is identical.  Then
    the whole chain on a Taylor-Green vortex: velocity -> g on the GPU -> omni_solve_direct -> the analytic pressure."""
    rng = np.random.default_rng(12)
    np_dt = np.float32 if dtype == "f32" else np.float64
    for shape, frac, unsteady in (((13, 21, 70), 0.05, True), ((37, 150), 0.03, False), ((6, 5, 9), 0.0, True), ((3, 40), 0.0, False)):
        nd = len(shape)
        d = (0.4, 0.7, 1.1)
        vel = [rng.normal(size=shape).astype(np_dt) for _ in range(nd)]
        if frac > 0:
            vel[0][rng.random(shape) < 0.01] = np.nan
        mask = (rng.random(shape) > frac).astype(np.uint8) if frac > 0 else None
        acc = [rng.normal(size=shape).astype(np_dt) for _ in range(nd)] if unsteady else None
        vd = [to_dev(c) for c in vel] + [None] * (3 - nd)
        g = omni.velocity_source(vd[0], vd[1], vd[2], None if mask is None else to_dev(mask), d, rho=1.3, mu=0.02,
                                 dudt=None if acc is None else [to_dev(c) for c in acc])
        v64 = [c.astype(np.float64) for c in vel] + [None] * (3 - nd)
        go = oracle.velocity_source(v64[0], v64[1], v64[2], mask, *d[:nd], rho=1.3, mu=0.02,
                                    dudt=None if acc is None else [c.astype(np.float64) for c in acc])
        assert len(g) == nd
        for i in range(nd):
            gi = g[i].cpu().numpy().astype(np.float64)
            assert np.array_equal(np.isnan(gi), np.isnan(go[i])), (shape, i)
            scale = np.nanmax(np.abs(go[i])) if np.isfinite(go[i]).any() else 1.0
            assert np.nanmax(np.abs(gi - go[i]), initial=0.0) <= (1e-12 if dtype == "f64" else 2e-5) * scale, (shape, i)
    # chain: Taylor-Green (steady, inviscid): P = rho/4 (cos 2x + cos 2y)
    n = 96
    h = 2 * np.pi / n
    yy, xx = np.meshgrid(np.arange(n) * h, np.arange(n) * h, indexing="ij")
    rho = 1.2
    u, v = (np.sin(xx) * np.cos(yy)).astype(np_dt), (-np.cos(xx) * np.sin(yy)).astype(np_dt)
    gx, gy = omni.velocity_source(to_dev(u), to_dev(v), None, None, (h, h), rho=rho)
    tol = 1e-8 if dtype == "f64" else 1e-5
    P, info = omni.solve_direct(gx, gy, None, None, (h, h), tol, 20, 5000)
    assert info["status"] == 0
    Pa = 0.25 * rho * (np.cos(2 * xx) + np.cos(2 * yy))
    Pn = P.cpu().numpy().astype(np.float64)
    valid = ~np.isnan(Pn)
    assert valid.sum() == (n - 2) ** 2                      # the one-cell rim has no central stencil
    assert rel_l2_after_mean_removal(Pn, Pa, valid) < 5e-3


def test_solve_without_info_is_asynchronous():
    """include/omni.h: with info == NULL the call returns after enqueueing.  The graph loop parks its executable graph
    instead of destroying it in flight (that blocks the host for the whole solve); the persistent loop is one launch."""
    import time
    f = make_config(3, 160)
    g_dev, _, m_dev, _ = _inputs(f, "f32")
    for mode in (2, 3):
        prev = omni.set_loop_mode(mode)
        try:
            for _ in range(2):
                omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, f["d"], 0.0, 6, 50)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            e0.record()
            P, info = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, f["d"], 0.0, 6, 50, want_info=False)
            host_ms = (time.perf_counter() - t0) * 1e3
            e1.record()
            torch.cuda.synchronize()
            gpu_ms = e0.elapsed_time(e1)
        finally:
            omni.set_loop_mode(prev)
        assert info is None
        assert host_ms < 0.5 * gpu_ms, (mode, host_ms, gpu_ms)
    omni.release_memory()


def test_edge_cases(oracle):
    dev = "cuda"
    # zero gradient -> P = 0, no iterations
    z = torch.zeros(6, 7, 8, dtype=torch.float64, device=dev)
    m = torch.ones(6, 7, 8, dtype=torch.uint8, device=dev)
    m[2, 3, 4] = 0
    P, info = omni.solve(z, z, z, m, (1.0, 1.0, 1.0), 1e-8, 10, 10)
    assert info["outer_iters"] == 0 and info["cg_iters_total"] == 0 and info["norm_S"] == 0 and info["status"] == 0
    Pn = P.cpu().numpy()
    assert np.isnan(Pn[2, 3, 4]) and np.all(Pn[m.cpu().numpy() == 1] == 0)
    # everything masked
    P, info = omni.solve(z, z, z, torch.zeros_like(m), (1.0, 1.0, 1.0), 1e-8, 10, 10)
    assert np.all(np.isnan(P.cpu().numpy())) and info["outer_iters"] == 0
    # single cell, single row, single column
    one = torch.ones(1, 1, dtype=torch.float64, device=dev)
    P, info = omni.solve(one, one, None, None, (1.0, 1.0), 1e-8, 10, 10)
    assert float(P[0, 0]) == 0.0 and info["outer_iters"] == 0
    # NaN-marked missing data equals mask-marked missing data (Eq. 13)
    f = make_field("lamb_oseen2d", (60, 70), seed=1, noise=0.05)
    fn = make_field("lamb_oseen2d", (60, 70), seed=1, noise=0.05, nan_mask=True)
    Pm, im = omni.solve(to_dev(f["g"][0]), to_dev(f["g"][1]), None, to_dev(f["mask"]), f["d"], 1e-6, 500, 20)
    Pn, inn = omni.solve(to_dev(fn["g"][0]), to_dev(fn["g"][1]), None, None, fn["d"], 1e-6, 500, 20)
    assert im == inn and np.array_equal(Pm.cpu().numpy(), Pn.cpu().numpy(), equal_nan=True)
    # max_outer = 0 and max_cg = 0 terminate
    g = to_dev(f["g"][0])
    P, info = omni.solve(g, to_dev(f["g"][1]), None, to_dev(f["mask"]), f["d"], 1e-6, 0, 5)
    assert info["outer_iters"] == 0 and info["status"] == 1 and info["eps_R_final"] == pytest.approx(1.0)
    P, info = omni.solve(g, to_dev(f["g"][1]), None, to_dev(f["mask"]), f["d"], 1e-6, 3, 0)
    assert info["outer_iters"] == 3 and info["cg_iters_total"] == 0
    # the 3x3 appendix example runs (all cells are boundary cells)
    rng = np.random.default_rng(0)
    fx, fy = rng.normal(size=(3, 3)), rng.normal(size=(3, 3))
    P, info = omni.solve(to_dev(fx), to_dev(fy), None, None, (0.5, 0.5), 0.0, 4, 9)
    Po, io = oracle.solve(fx, fy, None, None, 0.5, 0.5, 1.0, tol=0.0, max_outer=4, max_cg=9)
    assert rel_l2_after_mean_removal(P.cpu().numpy(), Po, np.ones((3, 3), bool)) < 1e-9


def test_host_buffers_and_workspace_entry_points(oracle):
    f = make_field("fourier3d", (10, 20, 30), seed=4, noise=0.05, kmax=2.0)
    g = [torch.from_numpy(c) for c in f["g"]]
    Ph, ih = omni.solve(g[0], g[1], g[2], None, f["d"], 1e-6, 100, 10)          # host path
    gd = [c.cuda() for c in g]
    Pd, idv = omni.solve(gd[0], gd[1], gd[2], None, f["d"], 1e-6, 100, 10)
    assert ih == idv and np.array_equal(Ph.numpy(), Pd.cpu().numpy())
    ws = torch.empty(omni.workspace_bytes(30, 20, 10, "f64"), dtype=torch.uint8, device="cuda")
    Pw, iw = omni.solve(gd[0], gd[1], gd[2], None, f["d"], 1e-6, 100, 10, workspace=ws)
    assert iw == idv and np.array_equal(Pw.cpu().numpy(), Pd.cpu().numpy())
    # a workspace full of NaN bit patterns must not leak into the result (every array is initialised by the solve)
    ws.fill_(0xFF)
    Pw2, iw2 = omni.solve(gd[0], gd[1], gd[2], None, f["d"], 1e-6, 100, 10, workspace=ws)
    assert iw2 == idv and np.array_equal(Pw2.cpu().numpy(), Pd.cpu().numpy())
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(omni.OmniError):
        omni.solve(gd[0], gd[1], gd[2], None, f["d"], 1e-6, 100, 10, workspace=small)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_rans_source_parity(oracle, dtype):
    """omni_rans_source_* (Eq. 42 :507) and omni_compressible_rans_source_* (Eq. 43-44 :540-545) against the oracle,
    entry by entry: 3D and 2D, ragged sizes, random masks plus NaN inputs, with and without Reynolds stresses; the NaN
    pattern is identical.  fp32 bound: the central differences of O(1) fields over h ~ 0.4 keep ~1e-6 of the largest
    entry; the 3x3 systems of Eq. 44 are diagonally dominated here (|uu| / RT < 1/2).  Then the chain on the compressible
    free vortex: velocity -> g on the GPU -> omni_solve_direct -> ln(P / P_inf) = gamma/(gamma-1) ln(T / T_inf)."""
    rng = np.random.default_rng(21)
    np_dt = np.float32 if dtype == "f32" else np.float64
    tol = 1e-12 if dtype == "f64" else 3e-5
    for shape, frac, with_R in (((11, 19, 70), 0.05, True), ((33, 150), 0.03, True), ((6, 5, 9), 0.0, False), ((3, 40), 0.0, True)):
        nd = len(shape)
        d = (0.4, 0.7, 1.1)
        vel = [rng.normal(size=shape).astype(np_dt) for _ in range(nd)]
        nR = 3 if nd == 2 else 6
        R = [(0.3 * rng.normal(size=shape)).astype(np_dt) for _ in range(nR)] if with_R else None
        if frac > 0:
            vel[1][rng.random(shape) < 0.01] = np.nan
            R[nR - 1][rng.random(shape) < 0.01] = np.nan
        mask = (rng.random(shape) > frac).astype(np.uint8) if frac > 0 else None
        vd = [to_dev(c) for c in vel] + [None] * (3 - nd)
        Rd = None if R is None else [to_dev(c) for c in R]
        md = None if mask is None else to_dev(mask)
        v64 = [c.astype(np.float64) for c in vel] + [None] * (3 - nd)
        R64 = None if R is None else [c.astype(np.float64) for c in R]
        got = omni.rans_source(vd[0], vd[1], vd[2], Rd, md, d, rho=1.3)
        ref = oracle.rans_source(v64[0], v64[1], v64[2], R64 if R64 is not None else [np.zeros(shape)] * nR, mask, *d[:nd], rho=1.3)
        kw = dict(gamma=1.4, mach_inf=0.9, v_inf=2.5, rgas_t_inf=6.0)
        gotc = omni.compressible_rans_source(vd[0], vd[1], vd[2], Rd, md, d, **kw)
        refc = oracle.compressible_rans_source(v64[0], v64[1], v64[2], R64, mask, *d[:nd], **kw)
        for name, g, go in (("rans", got, ref), ("compressible", gotc, refc)):
            assert len(g) == nd
            for i in range(nd):
                gi = g[i].cpu().numpy().astype(np.float64)
                assert np.array_equal(np.isnan(gi), np.isnan(go[i])), (name, shape, i)
                scale = max(np.nanmax(np.abs(c)) for c in go) if np.isfinite(go[i]).any() else 1.0
                assert np.nanmax(np.abs(gi - go[i]), initial=0.0) <= tol * scale, (name, shape, i)
    # a partly given stress list is rejected
    with pytest.raises(omni.OmniError):
        omni.rans_source(vd[0], vd[1], None, [vd[0], None, vd[1]], None, d)
    # chain: compressible free vortex (homentropic): ln(P/P_inf) = gamma/(gamma-1) ln(T/T_inf)
    gam, G, Minf = 1.4, 0.5, 0.4
    n = 129
    h = 2.0 / (n - 1)
    y, x = np.meshgrid(-1 + np.arange(n) * h, -1 + np.arange(n) * h, indexing="ij")
    r2 = x * x + y * y
    mask = (r2 >= 0.5 ** 2).astype(np.uint8)
    Vinf = G
    RTinf = Vinf ** 2 / (gam * Minf ** 2)
    with np.errstate(divide="ignore", invalid="ignore"):
        u, v = (-G * y / r2).astype(np_dt), (G * x / r2).astype(np_dt)
    u[mask == 0] = 0; v[mask == 0] = 0
    gx, gy = omni.compressible_rans_source(to_dev(u), to_dev(v), None, None, to_dev(mask), (h, h), gamma=gam, mach_inf=Minf,
                                           v_inf=Vinf, rgas_t_inf=RTinf)
    P, info = omni.solve_direct(gx, gy, None, to_dev(mask), (h, h), 1e-8 if dtype == "f64" else 1e-5, 20, 5000)
    assert info["status"] == 0
    with np.errstate(divide="ignore", invalid="ignore"):
        lnP = gam / (gam - 1) * np.log(1 + 0.5 * (gam - 1) * Minf ** 2 * (1 - G * G / r2 / Vinf ** 2))
    Pn = P.cpu().numpy().astype(np.float64)
    valid = ~np.isnan(Pn)
    assert valid.sum() > 0.6 * n * n
    assert rel_l2_after_mean_removal(Pn, lnP, valid) < 5e-3


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_solve_guess_parity(oracle, dtype, forced_loop):
    """omni_solve_guess_* (Alg. 1 from a first guess) against oracle.solve_guess: trajectory parity from a
    random guess in 3D (masked) and 2D, garbage at the missing cells ignored; a NULL guess is bit-identical to omni_solve;
    a restart from the converged field of omni_solve stops at the first residual check."""
    rng = np.random.default_rng(31)
    np_dt = np.float32 if dtype == "f32" else np.float64
    bound = 1e-9 if dtype == "f64" else 2e-4
    for kind, shape in (("sphere3d", (20, 26, 70)), ("lamb_oseen2d", (40, 150))):
        f = make_field(kind, shape, seed=8, noise=0.05)
        gh = [c.astype(np_dt) for c in f["g"]]
        g = [to_dev(c) for c in gh] + [None] * (3 - len(gh))
        g64 = [c.astype(np.float64) for c in gh] + [None] * (3 - len(gh))
        m = None if f["mask"] is None else to_dev(f["mask"])
        guess = rng.normal(size=shape).astype(np_dt)
        if f["mask"] is not None:
            guess[f["mask"] == 0] = 1e30
        P, info = omni.solve_guess(g[0], g[1], g[2], m, f["d"], 0.0, 5, 20, to_dev(guess))
        Po, io = oracle.solve_guess(g64[0], g64[1], g64[2], f["mask"], *f["d"], tol=0.0, max_outer=5, max_cg=20,
                                    P_init=guess.astype(np.float64))
        assert info["cg_iters_total"] == io["cg_iters_total"] == 100
        assert rel_l2_after_mean_removal(P.cpu().numpy(), Po, ~np.isnan(Po)) <= bound
        # raw values too: the guess fixes the additive constant (no mean removal), up to the trajectory bound
        v = ~np.isnan(Po)
        assert np.abs(P.cpu().numpy()[v] - Po[v]).max() <= (1e-9 if dtype == "f64" else 5e-4) * max(1.0, np.abs(Po[v]).max())
        P0, i0 = omni.solve(g[0], g[1], g[2], m, f["d"], 0.0, 3, 10)
        Pn, i_n = omni.solve_guess(g[0], g[1], g[2], m, f["d"], 0.0, 3, 10, None)
        assert torch.equal(torch.nan_to_num(P0), torch.nan_to_num(Pn)) and i0 == i_n
    tol = 1e-8 if dtype == "f64" else 1e-5
    Pc, ic = omni.solve(g[0], g[1], g[2], m, f["d"], tol, 200000, 16)
    assert ic["status"] == 0
    # fp32: the returned field is the fp64 master pressure rounded to fp32, which perturbs eps_R at the 1e-6 level
    Pr, ir = omni.solve_guess(g[0], g[1], g[2], m, f["d"], tol * (1.01 if dtype == "f64" else 3.0), 200000, 16, torch.nan_to_num(Pc))
    assert ir["status"] == 0 and ir["outer_iters"] == 0 and ir["cg_iters_total"] == 0
    vv = ~torch.isnan(Pc)
    assert torch.allclose(Pr[vv], Pc[vv], rtol=0, atol=(1e-12 if dtype == "f64" else 1e-6) * float(Pc[vv].abs().max()))


@pytest.mark.parametrize("loop", list(LOOPS))
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_residual_history_parity(oracle, dtype, loop):
    """omni_set_history: eps_R (Eq. 41 :442) of every outer residual check against the oracle's history of the same run
    (fixed caps, both loop drivers, Alg. 1 and the direct solve): outer_iters + 1 entries, each within the trajectory
    bound relative to its value; entries beyond stay untouched; a short buffer keeps the first entries only."""
    f = make_field("sphere3d", (18, 22, 40), seed=4, noise=0.05)
    np_dt = np.float32 if dtype == "f32" else np.float64
    gh = [c.astype(np_dt) for c in f["g"]]
    g = [to_dev(c) for c in gh]
    g64 = [c.astype(np.float64) for c in gh]
    m = to_dev(f["mask"])
    rel = 1e-9 if dtype == "f64" else 2e-4
    prev = omni.set_loop_mode(LOOPS[loop])
    try:
        hist = torch.full((16,), -1.0, dtype=torch.float64, device="cuda")
        its = torch.full((16,), -1, dtype=torch.int32, device="cuda")
        omni.set_history(hist, its)
        P, info = omni.solve(g[0], g[1], g[2], m, f["d"], 0.0, 6, 15)
        h = hist.cpu().numpy()
        assert its.cpu().tolist() == [0] + [15] * 6 + [-1] * 9           # CG iterations per outer iteration (fixed caps)
        _, io, ho = oracle.solve(*g64, f["mask"], *f["d"], tol=0.0, max_outer=6, max_cg=15, hist_cap=16)
        n = info["outer_iters"] + 1
        assert n == 7 and np.all(h[n:] == -1.0) and np.all(np.isnan(ho[n:]))
        assert h[0] == pytest.approx(1.0, abs=1e-6)                 # P^0 = 0: r_0 = S
        assert np.all(np.abs(h[:n] - ho[:n]) <= rel * np.maximum(ho[:n], 1e-3)), (h[:n], ho[:n])
        assert h[n - 1] == pytest.approx(info["eps_R_final"], rel=1e-12)
        short = torch.full((3,), -1.0, dtype=torch.float64, device="cuda")
        omni.set_history(short)
        omni.solve(g[0], g[1], g[2], m, f["d"], 0.0, 6, 15)
        assert np.array_equal(short.cpu().numpy(), h[:3])
        # the direct solve records its refinement checks the same way
        omni.set_history(hist.fill_(-1.0))
        Pd, idd = omni.solve_direct(g[0], g[1], g[2], m, f["d"], 0.0, 2, 40)
        hd = hist.cpu().numpy()
        assert np.all(hd[:3] > 0) and np.all(hd[3:] == -1.0) and hd[2] == pytest.approx(idd["eps_R_final"], rel=1e-12)
        assert hd[1] < 1e-2 * hd[0]
        omni.set_history(None)
        hist.fill_(-1.0)
        omni.solve(g[0], g[1], g[2], m, f["d"], 0.0, 2, 5)
        assert float(hist.max()) == -1.0                           # switched off: nothing written
    finally:
        omni.set_history(None)
        omni.set_loop_mode(prev)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_disconnected_components_and_isolated_cells(oracle, dtype, forced_loop):
    """Reading A12: P is fixed up to one constant PER connected component of the valid set.  A masked wall splits the box
    in two, one valid cell is walled in on its own.  Both sides start from P^0 = 0 and take identical steps, so the RAW
    values agree (no mean removal at all); the isolated cell has no link and stays 0; the direct solve returns zero mean
    on each component separately."""
    f = make_field("fourier3d", (14, 18, 40), seed=9, noise=0.05, kmax=3.0)
    mask = np.ones((14, 18, 40), np.uint8)
    mask[:, :, 19:21] = 0                       # wall normal to x: two components
    mask[6:9, 8:11, 4:7] = 0
    mask[7, 9, 5] = 1                           # a valid cell with six missing neighbours
    np_dt = np.float32 if dtype == "f32" else np.float64
    gh = [c.astype(np_dt) for c in f["g"]]
    g = [to_dev(c) for c in gh]
    g64 = [c.astype(np.float64) for c in gh]
    P, info = omni.solve(g[0], g[1], g[2], to_dev(mask), f["d"], 0.0, 5, 20)
    Po, io = oracle.solve(*g64, mask, *f["d"], tol=0.0, max_outer=5, max_cg=20)
    Pn = P.cpu().numpy().astype(np.float64)
    v = mask == 1
    assert np.array_equal(np.isnan(Pn), ~v) and np.array_equal(np.isnan(Po), ~v)
    assert Pn[7, 9, 5] == 0.0 and Po[7, 9, 5] == 0.0
    bound = 1e-9 if dtype == "f64" else 2e-4
    assert np.abs(Pn[v] - Po[v]).max() <= bound * np.abs(Po[v]).max()
    left, right = v.copy(), v.copy()
    left[:, :, 19:] = False; left[7, 9, 5] = False
    right[:, :, :21] = False
    for comp in (left, right):
        assert rel_l2_after_mean_removal(Pn, Po, comp) <= bound
    Pd, idd = omni.solve_direct(g[0], g[1], g[2], to_dev(mask), f["d"], 1e-8 if dtype == "f64" else 1e-5, 10, 3000)
    assert idd["status"] == 0
    Pdn = Pd.cpu().numpy().astype(np.float64)
    scale = np.abs(Pdn[v]).max()
    for comp in (left, right):
        assert abs(Pdn[comp].mean()) <= (1e-9 if dtype == "f64" else 1e-4) * scale
    assert Pdn[7, 9, 5] == 0.0


PENCILS = [(2000, 1, 4), (500, 1, 1), (4000, 4, 4), (2000, 1, 8), (1200, 9, 3)]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape", PENCILS)
def test_pencil_shapes_long_z_axis(oracle, dtype, shape):
    """Thin cross-sections with a long z axis: the tile kernels launch (x tiles) x (y tiles) x (z segments) CTAs with
    z segments as short as ~4 planes, many more reduction slots than npad / 256 (the per-CTA partial buffer
    must be sized from the launch geometry).  Through apply_M and residual (always the tile kernels) and through the
    host-driven and graph loops."""
    rng = np.random.default_rng(sum(shape))
    g = [rng.normal(size=shape) for _ in range(3)]
    mask = (rng.random(shape) > 0.03).astype(np.uint8)
    f = dict(g=g, mask=mask, d=(0.7, 1.1, 0.4))
    g_dev, g_or, m_dev, m = _inputs(f, dtype, mask)
    d = f["d"]
    v = oracle.validity(g_or[0], g_or[1], g_or[2], m)
    w1, w0, w0C = oracle.weights(v, *d)
    S_or = oracle.source(v, w1, w0, g_or[0], g_or[1], g_or[2], *d)
    p = rng.normal(size=shape)
    p_dev = to_dev(p, TDT[dtype])
    p_or = p_dev.cpu().numpy().astype(np.float64) * v
    q, pq = omni.apply_M(p_dev, m_dev, d)
    q_or = oracle.apply_M(v, w1, p_or)
    assert np.abs(q.cpu().numpy() - q_or).max() <= TOL_STEP[dtype] * 8 * np.abs(q_or).max()
    assert pq == pytest.approx(float(np.sum(p_or * q_or)), rel=1e-5 if dtype == "f32" else 1e-11)
    P = rng.normal(size=shape)
    r, eps = omni.residual(g_dev[0], g_dev[1], g_dev[2], m_dev, to_dev(P), d)
    Pv = P * v
    r_or = S_or + oracle.apply_Wn(v, w0, w0C, Pv) - oracle.apply_M(v, w1, Pv)
    assert np.abs(r.cpu().numpy() - r_or).max() <= TOL_STEP[dtype] * 8 * max(np.abs(r_or).max(), np.abs(Pv).max())
    assert eps == pytest.approx(np.linalg.norm(r_or) / np.linalg.norm(S_or), rel=1e-5 if dtype == "f32" else 1e-10)
    Po, io = oracle.solve(g_or[0], g_or[1], g_or[2], m, *d, tol=0.0, max_outer=3, max_cg=7)
    for mode in (1, 2):
        prev = omni.set_loop_mode(mode)
        try:
            Pg, ig = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, d, 0.0, 3, 7)
        finally:
            omni.set_loop_mode(prev)
        assert ig["cg_iters_total"] == io["cg_iters_total"] == 21 and ig["outer_iters"] == io["outer_iters"]
        assert np.array_equal(np.isnan(Pg.cpu().numpy()), np.isnan(Po))
        assert rel_l2_after_mean_removal(Pg.cpu().numpy(), Po, ~np.isnan(Po)) <= TOL_SOLVE[dtype]
        assert ig["eps_R_final"] == pytest.approx(io["eps_R_final"], rel=2e-3 if dtype == "f32" else 1e-7)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_outer_iterations_whose_inner_loop_does_not_start(oracle, dtype, forced_loop):
    """When an outer iteration's CG does not start (max_cg = 0; or an fp32-rounded r0 that underflows below the inner
    threshold while the fp64 residual is still above tol) no new correction exists, and K2 must not fold whatever the
    delta array holds into P (Scalars::dzero).  The oracle then repeats the same residual check until max_outer
    (P unchanged, no CG iterations).  Reachable here through max_cg = 0, from zero and from a first guess."""
    f = make_field("sphere3d", (20, 24, 36), seed=4, noise=0.05)
    g_dev, g_or, m_dev, m = _inputs(f, dtype)
    d = f["d"]
    # (1) max_cg = 0: nothing may move
    P, info = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, d, 1e-12, 5, 0)
    Po, io = oracle.solve(g_or[0], g_or[1], g_or[2], m, *d, tol=1e-12, max_outer=5, max_cg=0)
    assert info["outer_iters"] == io["outer_iters"] == 5 and info["cg_iters_total"] == io["cg_iters_total"] == 0
    assert info["status"] == omni.binding.OMNI_NOT_CONVERGED
    assert np.array_equal(np.nan_to_num(P.cpu().numpy()), np.nan_to_num(Po)) and not np.nan_to_num(Po).any()
    assert info["eps_R_final"] == pytest.approx(1.0, rel=1e-6) and io["eps_R_final"] == pytest.approx(1.0, rel=1e-12)
    # (2) a first guess plus max_cg = 0 comes back unchanged after several outer iterations, every check seeing the
    # same residual
    P1, i1 = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, d, 0.0, 2, 9)
    guess = torch.nan_to_num(P1)
    hist = torch.zeros(8, dtype=torch.float64, device="cuda")
    omni.set_history(hist)
    try:
        P2, i2 = omni.solve_guess(g_dev[0], g_dev[1], g_dev[2], m_dev, d, 1e-12, 4, 0, guess)
    finally:
        omni.set_history(None)
    assert i2["outer_iters"] == 4 and i2["cg_iters_total"] == 0
    assert torch.equal(torch.nan_to_num(P2), guess)
    h = hist.cpu().numpy()
    assert np.all(h[:5] == h[0]) and h[0] > 0          # the same residual at every check
    Po2, io2 = oracle.solve_guess(g_or[0], g_or[1], g_or[2], m, *d, tol=1e-12, max_outer=4, max_cg=0,
                                  P_init=guess.cpu().numpy().astype(np.float64))
    assert io2["outer_iters"] == 4 and h[0] == pytest.approx(io2["eps_R_final"], rel=1e-4 if dtype == "f32" else 1e-9)


PCG_CASES = [("gaussians2d", (64, 64), None), ("lamb_oseen2d", (150, 130), None), ("fourier3d", (20, 33, 140), None),
             ("sphere3d", (40, 36, 44), None), ("fourier3d", (12, 30, 270), 0.15), ("gaussians2d", (21, 132), None),
             ("fourier3d", (9, 19, 66), None), ("fourier3d", (5, 4, 9), 0.2), ("gaussians2d", (3, 70), None), ("gaussians2d", (6, 7), None)]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("kind,shape,frac", PCG_CASES)
def test_pcg_trajectory_parity(oracle, dtype, kind, shape, frac):
    """omni_solve_pcg_* (multigrid-preconditioned CG on L P = S, reading R-P1) against oracle/omni_pcg.py with fixed
    iteration counts (tol = 0): identical steps on both sides -- level plan (odd sizes, axes that stop coarsening, grids
    too small to coarsen at all), coarse validity and link weights, transfers, Jacobi sweeps, the preconditioned
    recurrence, the fp64 outer refinement."""
    from oracle import omni_pcg
    f = make_field(kind, shape, seed=7, noise=0.05, kmax=4.0)
    mask = _random_mask(shape, 9, frac) if frac else None
    g_dev, g_or, m_dev, m = _inputs(f, dtype, mask)
    d = f["d"]
    # fp32: an inner solve returns to the fp64 refinement after two digits (inner_rel = 1e-2), which 2 iterations do not
    # reach: 4 x 2 iterations there, 2 x 6 in fp64
    mo, mc = (2, 6) if dtype == "f64" else (4, 2)
    rel = 0.0 if dtype == "f64" else 1e-2
    P, info = omni.solve_pcg(g_dev[0], g_dev[1], g_dev[2], m_dev, d, 0.0, mo, mc)
    Po, io = omni_pcg.solve_pcg(g_or[0], g_or[1], g_or[2], m, *d, tol=0.0, max_outer=mo, max_cg=mc, inner_rel=rel)
    valid = ~np.isnan(Po)
    assert np.array_equal(np.isnan(P.cpu().numpy()), ~valid)
    assert info["outer_iters"] == io["outer_iters"] == mo and info["cg_iters_total"] == io["cg_iters_total"]
    err = rel_l2_after_mean_removal(P.cpu().numpy(), Po, valid)
    assert err <= TOL_SOLVE[dtype], err
    # eps_R of the returned field: equal up to rounding, above the floor the fp32 field's own rounding leaves
    assert abs(info["eps_R_final"] - io["eps_R_final"]) <= (5e-3 if dtype == "f32" else 1e-6) * io["eps_R_final"] + (5e-5 if dtype == "f32" else 1e-12)
    # from a first guess (raw values: the guess fixes the constant)
    rng = np.random.default_rng(3)
    P0 = (0.1 * rng.normal(size=shape)).astype(np.float32 if dtype == "f32" else np.float64)
    Pg, ig = omni.solve_pcg(g_dev[0], g_dev[1], g_dev[2], m_dev, d, 0.0, 2, 2, P_init=to_dev(P0))
    Pog, iog = omni_pcg.solve_pcg(g_or[0], g_or[1], g_or[2], m, *d, tol=0.0, max_outer=2, max_cg=2, P_init=P0.astype(np.float64),
                                  inner_rel=rel)
    assert ig["cg_iters_total"] == iog["cg_iters_total"] == 4
    scale = np.nanmax(np.abs(Pog))
    assert np.nanmax(np.abs(Pg.cpu().numpy() - Pog)) <= (1e-10 if dtype == "f64" else 2e-4) * scale


@pytest.mark.parametrize("dtype,tol", [("f64", 1e-8), ("f32", 1e-5)])
def test_pcg_converged(oracle, dtype, tol):
    """Converged omni_solve_pcg_* on stand-ins of configs 1 - 4: the oracle's operators certify eps_R of the returned
    field (Eq. 41), the field equals the oracle's PCG result and omni_solve_direct's to tolerance level, and the
    iteration count is the grid-independent handful the preconditioner is there for."""
    from oracle import omni_pcg
    for idx, n in ((1, 160), (3, 48), (2, 64), (4, 72)):
        f = make_config(idx, n)
        g_dev, g_or, m_dev, m = _inputs(f, dtype)
        d = f["d"]
        P, info = omni.solve_pcg(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 10, 100)
        assert info["status"] == 0 and info["eps_R_final"] <= tol, (idx, info)
        assert info["cg_iters_total"] <= 30, info
        eps, _, _ = oracle.eps_R_of_field(g_or[0], g_or[1], g_or[2], m, P.cpu().numpy(), *d)
        assert eps <= (1.05 if dtype == "f64" else 3.0) * tol, (idx, eps)
        Po, io = omni_pcg.solve_pcg(g_or[0], g_or[1], g_or[2], m, *d, tol=tol, max_outer=10, max_cg=100,
                                    inner_rel=0.0 if dtype == "f64" else 1e-2)
        assert io["converged"] and abs(io["cg_iters_total"] - info["cg_iters_total"]) <= 2
        valid = ~np.isnan(Po)
        # both sides stop anywhere below tol: the fields agree to the accuracy tol buys (cf. test_direct_solve_converged)
        bound = 2e-6 if dtype == "f64" else 2e-3
        assert rel_l2_after_mean_removal(P.cpu().numpy(), Po, valid) <= bound
        Pd, idd = omni.solve_direct(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 10, 5000)
        assert idd["status"] == 0 and idd["cg_iters_total"] > 3 * info["cg_iters_total"]
        assert rel_l2_after_mean_removal(P.cpu().numpy(), Pd.cpu().numpy(), valid) <= bound


@pytest.mark.parametrize("loop", list(LOOPS))
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_solve_ex_options(oracle, dtype, loop):
    """omni_solve_ex_* with per-call omni_options: the three history columns (eps_R of Eq. 41, CG iterations, eps_P of
    Eq. 40) against oracle.solve_hist through every loop driver; the fp64 master pressure d_P64_out (the fp32 result
    is its rounding, and the ORACLE's eps_R of it meets tol where the fp32 field's cannot); the device status word after
    a call without info; the per-call loop mode leaves the process-wide one alone."""
    f = make_field("lamb_oseen2d", (40, 52), seed=3, noise=0.05)
    g_dev, g_or, m_dev, m = _inputs(f, dtype)
    d = f["d"]
    cap = 16
    hR = torch.full((cap,), -1.0, dtype=torch.float64, device="cuda")
    hP = torch.full((cap,), -1.0, dtype=torch.float64, device="cuda")
    hK = torch.full((cap,), -1, dtype=torch.int32, device="cuda")
    P64 = torch.zeros(f["g"][0].shape, dtype=torch.float64, device="cuda")
    st = torch.full((1,), 77, dtype=torch.int32, device="cuda")
    before = omni.set_loop_mode(0); omni.set_loop_mode(before)
    P, info = omni.solve_ex(g_dev[0], g_dev[1], None, m_dev, d, 0.0, 12, 15, method="alg1", loop_mode=LOOPS[loop],
                            hist_eps_R=hR, hist_cg_iters=hK, hist_eps_P=hP, P64_out=P64, status=st)
    after = omni.set_loop_mode(0); omni.set_loop_mode(after)
    assert before == after
    Po, io, oR, oP = oracle.solve_hist(g_or[0], g_or[1], None, m, *d, tol=0.0, max_outer=12, max_cg=15, hist_cap=cap)
    assert info["outer_iters"] == io["outer_iters"] == 12 and int(st.item()) == info["status"] == 1
    r, p, k = hR.cpu().numpy(), hP.cpu().numpy(), hK.cpu().numpy()
    rel = 2e-3 if dtype == "f32" else 1e-7
    assert np.allclose(r[:13], oR[:13], rtol=rel) and np.all(r[13:] == -1.0)
    assert p[0] == 0.0 and np.allclose(p[1:13], oP[1:13], rtol=rel) and np.all(p[13:] == -1.0)
    assert k[0] == 0 and np.all(k[1:13] == 15)
    valid = ~np.isnan(Po)
    P64n = P64.cpu().numpy()
    assert np.array_equal(np.isnan(P64n), ~valid)
    assert np.array_equal(P.cpu().numpy(), P64n.astype(np.float32 if dtype == "f32" else np.float64), equal_nan=True)
    assert rel_l2_after_mean_removal(P64n, Po, valid) <= TOL_SOLVE[dtype]
    # no info: the call does not synchronise; the status word tells how it ended
    st.fill_(77)
    _, none = omni.solve_ex(g_dev[0], g_dev[1], None, m_dev, d, 1e-3, 100000, 16, method="pcg" if loop == "graph" else "direct",
                            loop_mode=LOOPS[loop], status=st, want_info=False)
    assert none is None
    torch.cuda.synchronize()
    assert int(st.item()) == 0


@pytest.mark.parametrize("method", ["alg1", "direct", "pcg"])
def test_fp64_master_pressure_meets_tol_where_fp32_output_cannot(oracle, method):
    """configs[1] stand-in 384^2 in fp32, tol 1e-5: the oracle's eps_R (Eq. 41) of d_P64_out is <= 1.05 tol; of the fp32
    result it is the larger rounding floor 2^-24 |L||P| / ||S|| (SURVEY 7 hard part 3) -- which is why the option exists."""
    f = make_config(1, 384)
    g_dev, g_or, m_dev, m = _inputs(f, "f32")
    d, tol = f["d"], 1e-5
    P64 = torch.zeros(f["g"][0].shape, dtype=torch.float64, device="cuda")
    caps = {"alg1": (200000, 16), "direct": (20, 20000), "pcg": (20, 100)}[method]
    P, info = omni.solve_ex(g_dev[0], g_dev[1], None, m_dev, d, tol, caps[0], caps[1], method=method, P64_out=P64)
    assert info["status"] == 0 and info["eps_R_final"] <= tol
    e64, _, _ = oracle.eps_R_of_field(g_or[0], g_or[1], None, m, P64.cpu().numpy(), *d)
    e32, _, _ = oracle.eps_R_of_field(g_or[0], g_or[1], None, m, P.cpu().numpy(), *d)
    # the device forms S and r in fp32 (2^-24 relative per entry of S): the two figures agree to a few 1e-7 of ||S||
    assert abs(e64 - info["eps_R_final"]) <= 5e-7 and e64 <= 1.05 * tol
    assert e32 > e64


SLAB_CASES = [("sphere3d", (37, 20, 70), None, 2), ("sphere3d", (37, 20, 70), None, 3), ("fourier3d", (24, 33, 140), 0.1, 4),
              ("fourier3d", (5, 9, 40), 0.05, 4), ("fourier3d", (9, 19, 66), None, 2), ("fourier3d", (16, 12, 270), 0.15, 5)]


@pytest.mark.parametrize("method", ["alg1", "direct"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("kind,shape,frac,nslabs", SLAB_CASES)
def test_slab_sharded_solve(oracle, dtype, method, kind, shape, frac, nslabs):
    """NEXT-3: one solve cut into z-slabs (all ranks on this device: plane copies for the halos, a summing kernel for the
    scalars) against the oracle's single-grid solve with identical iteration counts, and against the single-device
    library result to rounding.  Masks crossing slab boundaries, slabs of one or two planes, odd sizes, fp32 / fp64,
    Alg. 1 (stencil codes read validity two planes into the neighbour slab) and the fixed-point solve."""
    f = make_field(kind, shape, seed=7, noise=0.05, kmax=4.0)
    mask = _random_mask(shape, 9, frac) if frac else None
    g_dev, g_or, m_dev, m = _inputs(f, dtype, mask)
    d = f["d"]
    mo, mc = 3, 7
    P, info = omni.solve_slab(g_dev[0], g_dev[1], g_dev[2], m_dev, d, 0.0, mo, mc, nslabs, method=method)
    fn_or = oracle.solve if method == "alg1" else oracle.solve_direct
    Po, io = fn_or(g_or[0], g_or[1], g_or[2], m, *d, tol=0.0, max_outer=mo, max_cg=mc)
    valid = ~np.isnan(Po)
    assert np.array_equal(np.isnan(P.cpu().numpy()), ~valid)
    assert info["outer_iters"] == io["outer_iters"] == mo and info["cg_iters_total"] == io["cg_iters_total"] == mo * mc
    assert rel_l2_after_mean_removal(P.cpu().numpy(), Po, valid) <= TOL_SOLVE[dtype]
    assert info["eps_R_final"] == pytest.approx(io["eps_R_final"], rel=2e-3 if dtype == "f32" else 1e-7)
    assert info["norm_S"] == pytest.approx(io["norm_S"], rel=1e-5 if dtype == "f32" else 1e-12)
    prev = omni.set_loop_mode(2)
    try:
        fn1 = omni.solve if method == "alg1" else omni.solve_direct
        P1, i1 = fn1(g_dev[0], g_dev[1], g_dev[2], m_dev, d, 0.0, mo, mc)
    finally:
        omni.set_loop_mode(prev)
    assert i1["cg_iters_total"] == info["cg_iters_total"]
    assert rel_l2_after_mean_removal(P.cpu().numpy(), P1.cpu().numpy(), valid) <= (1e-11 if dtype == "f64" else 1e-5)


@pytest.mark.parametrize("dtype,tol", [("f64", 1e-8), ("f32", 1e-5)])
def test_slab_sharded_solve_converged(oracle, dtype, tol):
    """The sharded fixed-point solve run to tolerance on a stand-in of configs[3] (masked sphere, 3 slabs): every rank
    stops at the same iteration, the oracle certifies eps_R of the assembled field, and it matches the one-device result."""
    f = make_config(3, 48)
    g_dev, g_or, m_dev, m = _inputs(f, dtype)
    d = f["d"]
    P, info = omni.solve_slab(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 10, 2000, 3, method="direct")
    assert info["status"] == 0 and info["eps_R_final"] <= tol
    eps, _, _ = oracle.eps_R_of_field(g_or[0], g_or[1], g_or[2], m, P.cpu().numpy(), *d)
    assert eps <= (1.05 if dtype == "f64" else 3.0) * tol
    P1, i1 = omni.solve_direct(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 10, 2000)
    assert abs(i1["cg_iters_total"] - info["cg_iters_total"]) <= 2
    valid = ~torch.isnan(P1).cpu().numpy()
    assert rel_l2_after_mean_removal(P.cpu().numpy(), P1.cpu().numpy(), valid) <= (2e-6 if dtype == "f64" else 2e-3)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("kind,shape,frac", [("gaussians2d", (64, 64), None), ("lamb_oseen2d", (150, 130), None),
                                             ("sphere3d", (40, 36, 44), None), ("fourier3d", (12, 30, 270), 0.15),
                                             ("gaussians2d", (21, 132), None), ("fourier3d", (5, 4, 9), 0.2)])
def test_single_reduction_cg_parity(oracle, dtype, kind, shape, frac):
    """omni_options::single_reduction (Chronopoulos-Gear CG for the symmetric L in the persistent kernel, one grid barrier
    per iteration; NEXT-2 i) against oracle_solve_direct_cg1 with fixed iteration counts, against the two-reduction
    library result (same iterates in exact arithmetic: the drift is rounding), and converged."""
    f = make_field(kind, shape, seed=7, noise=0.05, kmax=4.0)
    mask = _random_mask(shape, 9, frac) if frac else None
    g_dev, g_or, m_dev, m = _inputs(f, dtype, mask)
    d = f["d"]
    P, info = omni.solve_ex(g_dev[0], g_dev[1], g_dev[2], m_dev, d, 0.0, 2, 15, method="direct", loop_mode=3, single_reduction=True)
    Po, io = oracle.solve_direct(g_or[0], g_or[1], g_or[2], m, *d, tol=0.0, max_outer=2, max_cg=15, single_reduction=True)
    valid = ~np.isnan(Po)
    assert np.array_equal(np.isnan(P.cpu().numpy()), ~valid)
    assert info["outer_iters"] == io["outer_iters"] == 2 and info["cg_iters_total"] == io["cg_iters_total"] == 30
    assert rel_l2_after_mean_removal(P.cpu().numpy(), Po, valid) <= TOL_SOLVE[dtype]
    assert info["eps_R_final"] == pytest.approx(io["eps_R_final"], rel=5e-3 if dtype == "f32" else 1e-7)
    P2, i2 = omni.solve_ex(g_dev[0], g_dev[1], g_dev[2], m_dev, d, 0.0, 2, 15, method="direct", loop_mode=3)
    assert rel_l2_after_mean_removal(P.cpu().numpy(), P2.cpu().numpy(), valid) <= (1e-10 if dtype == "f64" else 2e-4)
    tol = 1e-8 if dtype == "f64" else 1e-5
    Pc, ic = omni.solve_ex(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 10, 5000, method="direct", loop_mode=3, single_reduction=True)
    Pd, idd = omni.solve_ex(g_dev[0], g_dev[1], g_dev[2], m_dev, d, tol, 10, 5000, method="direct", loop_mode=3)
    assert ic["status"] == 0 and ic["eps_R_final"] <= tol
    # the single-reduction recurrences are numerically weaker: in fp32 the recurred s = A p drifts and
    # costs up to ~10 % more iterations (711 vs 653 on the 150 x 130 case); fp64 stays within a few iterations
    assert abs(ic["cg_iters_total"] - idd["cg_iters_total"]) <= max(3, idd["cg_iters_total"] // (5 if dtype == "f32" else 20))
    assert rel_l2_after_mean_removal(Pc.cpu().numpy(), Pd.cpu().numpy(), valid) <= (2e-6 if dtype == "f64" else 2e-3)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_pcg_batch2d(oracle, dtype):
    """omni_solve_pcg_batch2d_*: the stacked snapshots with the multigrid-preconditioned CG against
    oracle/omni_pcg.solve_pcg_batch2d (fixed counts, with and without a first guess), and converged: every snapshot's own
    eps_R (oracle operators) within the bound the joint stopping rule gives, the fields equal to the unpreconditioned
    stacked solve's."""
    from oracle import omni_pcg
    fs = [make_field("lamb_oseen2d", (45, 140), seed=s, noise=0.05) for s in range(4)]
    np_dt = np.float32 if dtype == "f32" else np.float64
    gx = np.stack([f["g"][0] for f in fs]).astype(np_dt); gy = np.stack([f["g"][1] for f in fs]).astype(np_dt)
    m, d = fs[0]["mask"], fs[0]["d"]
    gxd, gyd, md = to_dev(gx), to_dev(gy), to_dev(m)
    mo, mc, rel = (2, 5, 0.0) if dtype == "f64" else (4, 2, 1e-2)
    rng = np.random.default_rng(6)
    P0 = (0.1 * rng.normal(size=gx.shape)).astype(np_dt)
    for init in (None, P0):
        P, info = omni.solve_batch2d(gxd, gyd, md, d, 0.0, mo, mc, P_init=None if init is None else to_dev(init), pcg=True)
        Po, io = omni_pcg.solve_pcg_batch2d(gx.astype(np.float64), gy.astype(np.float64), m, d[0], d[1], 0.0, mo, mc,
                                            P_init=None if init is None else init.astype(np.float64), inner_rel=rel)
        assert info["cg_iters_total"] == io["cg_iters_total"] and info["outer_iters"] == io["outer_iters"] == mo
        Pn = P.cpu().numpy()
        assert np.array_equal(np.isnan(Pn), np.isnan(Po))
        for b in range(4):
            if init is None:
                assert rel_l2_after_mean_removal(Pn[b], Po[b], ~np.isnan(Po[b])) <= TOL_SOLVE[dtype]
            else:
                assert np.nanmax(np.abs(Pn[b] - Po[b])) <= (1e-10 if dtype == "f64" else 2e-4) * np.nanmax(np.abs(Po[b]))
    tol = 1e-5 if dtype == "f32" else 1e-8
    Pc, ic = omni.solve_batch2d(gxd, gyd, md, d, tol, 20, 200, pcg=True)
    assert ic["status"] == 0 and ic["eps_R_final"] <= tol and ic["cg_iters_total"] <= 40
    Pd, idd = omni.solve_batch2d(gxd, gyd, md, d, tol, 20, 5000, direct=True)
    assert idd["status"] == 0 and idd["cg_iters_total"] > 5 * ic["cg_iters_total"]
    for b in range(4):
        valid = ~torch.isnan(Pd[b]).cpu().numpy()
        assert rel_l2_after_mean_removal(Pc[b].cpu().numpy(), Pd[b].cpu().numpy(), valid) <= (2e-6 if dtype == "f64" else 2e-3)
        e_b, _, nS_b = oracle.eps_R_of_field(gx[b].astype(np.float64), gy[b].astype(np.float64), None, m, Pc[b].cpu().numpy(), d[0], d[1])
        assert e_b * nS_b <= (1.05 if dtype == "f64" else 3.0) * tol * ic["norm_S"]


def test_automatic_loop_choice():
    """Which loop the automatic mode takes, shown by bit-identical results: the SM-resident kernel (5) where the grid fits
    the SMs, the persistent kernel (3) where its rows are too long for one chunk per thread, the CUDA graph over the tile
    kernels (2) where p no longer fits the shared memory of the SMs."""
    cases = [("gaussians2d", (96, 80), "f32", 5), ("fourier3d", (20, 33, 140), "f64", 5),
             ("lamb_oseen2d", (40, 2100), "f64", 3), ("fourier3d", (200, 190, 200), "f32", 2)]
    for kind, shape, dtype, expect in cases:
        f = make_field(kind, shape, seed=2, noise=0.05, kmax=4.0)
        g_dev, _, m_dev, _ = _inputs(f, dtype)
        nx = shape[-1]
        plan = omni.resident_plan(nx, shape[-2], shape[0] if len(shape) == 3 else 1, dtype)
        assert (plan is not None) == (expect == 5), (shape, dtype, plan)
        P0, i0 = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, f["d"], 0.0, 3, 7)
        out = {}
        for mode in (2, 3, 5):
            prev = omni.set_loop_mode(mode)
            try:
                out[mode] = omni.solve(g_dev[0], g_dev[1], g_dev[2], m_dev, f["d"], 0.0, 3, 7)[0]
            finally:
                omni.set_loop_mode(prev)
        assert torch.equal(torch.nan_to_num(P0), torch.nan_to_num(out[expect])), (shape, dtype, expect)
        assert i0["cg_iters_total"] == 21
