"""CPU-side checks of the CUDA library: it loads, exports every symbol of include/omni.h, validates arguments, and
its host-side geometry constants (step a0) agree with the oracle's independent computation."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2311_16935_b200 as omni

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "omni.h")).read()
    declared = set(re.findall(r"\b(omni_[a-z0-9_A-Z]+)\s*\(", hdr))
    assert declared == set(omni.SYMBOLS), declared ^ set(omni.SYMBOLS)
    L = omni.lib()
    for s in declared:
        assert hasattr(L, s), s
    assert omni.version() >= 100
    assert "invalid" in omni.status_string(-1)


def test_argument_validation_needs_no_device():
    L = omni.lib()
    bad = [dict(nx=0), dict(dx=0.0), dict(dx=float("nan")), dict(tol=-1.0), dict(max_outer=-1), dict(gx=0), dict(P=0)]
    for b in bad:
        a = dict(nx=4, ny=4, nz=1, dx=1.0, dy=1.0, dz=1.0, gx=8, gy=8, gz=0, mask=0, P=8, tol=1e-8, max_outer=1, max_cg=1)
        a.update(b)
        rc = L.omni_solve_f64(C.c_int(a["nx"]), C.c_int(a["ny"]), C.c_int(a["nz"]), C.c_double(a["dx"]), C.c_double(a["dy"]),
                              C.c_double(a["dz"]), C.c_void_p(a["gx"]), C.c_void_p(a["gy"]), C.c_void_p(a["gz"]),
                              C.c_void_p(a["mask"]), C.c_void_p(a["P"]), C.c_double(a["tol"]), C.c_int(a["max_outer"]),
                              C.c_int(a["max_cg"]), None, None)
        assert rc == -1, b
    # 3D needs gz
    rc = L.omni_solve_f32(C.c_int(4), C.c_int(4), C.c_int(4), C.c_double(1), C.c_double(1), C.c_double(1), C.c_void_p(8),
                          C.c_void_p(8), C.c_void_p(0), None, C.c_void_p(8), C.c_double(0), C.c_int(1), C.c_int(1), None, None)
    assert rc == -1
    assert omni.workspace_bytes(64, 64, 1, "f64") > 64 * 64 * 8 * 6
    assert omni.workspace_bytes(500, 500, 500, "f32") < 6 * 2**30


@pytest.mark.parametrize("dims,sp", [((9, 9, 1), (0.3, 0.7, 1.0)), ((5, 5, 5), (1.0, 1.0, 1.0)), ((5, 5, 5), (0.25, 0.25, 0.25)),
                                     ((5, 6, 7), (1.0, 0.7, 1.9)), ((4, 4, 4), (0.01, 0.013, 0.0047)),
                                     ((264, 16, 5), (1 / 263, 1 / 15, 1 / 4)), ((5, 16, 264), (0.25, 1 / 15, 1 / 263))])
def test_constants_a0_match_oracle(oracle, dims, sp):
    """Two independent routes to c_jk: closed-form parallel-rectangle measure (library) vs Eq. 17 / Eq. 32-33 /
    Gauss-Legendre quadrature of the defining integral (oracle)."""
    K = omni.constants(*dims, *sp)
    Ko = oracle.constants(*dims, *sp)
    assert np.allclose(K["F"], Ko["F"], rtol=1e-14)
    assert K["A_tot"] == pytest.approx(Ko["A_tot"], rel=1e-14)
    # what enters the stencil is c / A_tot (Eq. 10): relative 2e-12, or 1e-15 absolute for the tiny far-face
    # constants of strongly anisotropic cells, where the closed form loses digits to cancellation
    assert np.allclose(np.array(K["c"]) / K["A_tot"], Ko["c"] / Ko["A_tot"], rtol=2e-12, atol=1e-15)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    g = torch.zeros(8, 8, dtype=torch.float64)
    with pytest.raises(RuntimeError):
        omni.solve(g, g, None, None, (1.0, 1.0), 1e-8, 1, 1)


def test_binding_rejects_mismatched_tensors_before_the_call():
    """A gy / gz / mask / out tensor whose shape or dtype differs from gx would make the kernels index out of bounds:
    the binding raises before anything reaches the library (no device needed)."""
    import torch
    g = torch.zeros(6, 8, dtype=torch.float64)
    for bad in (dict(gy=torch.zeros(6, 8, dtype=torch.float32)), dict(gy=torch.zeros(6, 9, dtype=torch.float64)),
                dict(mask=torch.ones(8, 6, dtype=torch.uint8)), dict(mask=torch.ones(6, 8, dtype=torch.bool)),
                dict(out=torch.zeros(6, 8, dtype=torch.float32))):
        a = dict(gy=g, mask=None, out=None)
        a.update(bad)
        with pytest.raises(TypeError):
            omni.solve(g, a["gy"], None, a["mask"], (1.0, 1.0), 1e-8, 1, 1, out=a["out"])
    g3 = torch.zeros(4, 6, 8, dtype=torch.float32)
    with pytest.raises(TypeError):
        omni.solve(g3, g3, g3, torch.ones(6, 8, dtype=torch.uint8), (1.0, 1.0, 1.0), 1e-5, 1, 1)


@pytest.mark.parametrize("dims", [(4, 1, 2000), (1, 1, 500), (4, 4, 4000), (8, 1, 2000), (500, 500, 500), (1024, 1024, 1)])
def test_workspace_holds_one_reduction_slot_per_tile_cta(dims):
    """thin cross-sections with a long z axis launch far more tile CTAs (x tiles * y tiles * z segments, four
    accumulators in K2) than npad / 256; the workspace must grow with that bound, whatever segment count the device
    picks (at most nz)."""
    nx, ny, nz = dims
    for dt, cell, pad in (("f32", 4, 8), ("f64", 8, 4)):
        px = (nx + pad - 1) // pad * pad
        npad = px * ny * nz
        vectors = 5 * npad * cell + 2 * npad * 8 + npad * 5          # S r p0 p1 delta, P P1, link + wcode
        worst_ctas = 4 * ((px + 63) // 64) * ((ny + 7) // 8) * nz
        assert omni.workspace_bytes(nx, ny, nz, dt) >= vectors + 8 * worst_ctas


def test_solve_ex_rejects_bad_options_before_enqueueing():
    """omni_solve_ex_*: unknown method, a struct_size that is not this library's, a history pointer without capacity."""
    L = omni.lib()
    o = omni.Options()
    L.omni_options_init(C.byref(o))
    assert o.struct_size == C.sizeof(omni.Options) and o.loop_mode == -1 and o.hist_capacity == 0

    def call(method, opt):
        return L.omni_solve_ex_f64(C.c_int(4), C.c_int(4), C.c_int(1), C.c_double(1), C.c_double(1), C.c_double(1), C.c_void_p(8),
                                   C.c_void_p(8), C.c_void_p(0), None, None, C.c_void_p(8), C.c_double(1e-8), C.c_int(1), C.c_int(1),
                                   C.c_int(method), C.byref(opt) if opt is not None else None, None, None)
    assert call(7, o) == -1
    bad = omni.Options(); L.omni_options_init(C.byref(bad)); bad.struct_size = 8
    assert call(0, bad) == -1
    bad = omni.Options(); L.omni_options_init(C.byref(bad)); bad.d_hist_eps_R = 256
    assert call(0, bad) == -1
    bad = omni.Options(); L.omni_options_init(C.byref(bad)); bad.loop_mode = 9
    assert call(0, bad) == -1


def test_resident_plan_invariants():
    """The box decomposition of the SM-resident loop (host code of omni_resident.cuh through omni_resident_plan): the cuts
    tile every axis with non-empty boxes, the largest box is the one the plan reports, the shared memory fits an SM, the
    rows per thread cover the largest box; weighted cuts (operator M) never give a face box more rows than an interior one;
    grids that cannot fit are refused."""
    import paper_2311_16935_b200 as omni
    cases = [(64, 64, 1), (130, 150, 1), (1024, 1024, 1), (2048, 700, 1), (32, 32, 32), (66, 19, 9), (128, 128, 128),
             (130, 110, 101), (96, 96, 96), (500, 37, 41), (8, 3, 2)]
    seen = 0
    for nx, ny, nz in cases:
        for dtype, esz in (("f32", 4), ("f64", 8)):
            for lop in (False, True):
                for nsm in (148, 132, 20):
                    pl = omni.resident_plan(nx, ny, nz, dtype, nsm, lop)
                    if pl is None:
                        continue
                    seen += 1
                    V = 16 // esz
                    assert pl["gy"] * pl["gz"] <= nsm and pl["gy"] <= ny and pl["gz"] <= nz
                    assert pl["smem_bytes"] <= 222 * 1024
                    cpr = pl["px"] // V
                    assert pl["px"] % V == 0 and cpr <= 512
                    nrg = 512 // cpr
                    assert pl["rows_per_thread"] * nrg >= pl["ly"] * pl["lz"]
                    three = nz > 1
                    p_bytes = (pl["lz"] + (2 if three else 0)) * (pl["ly"] + 2) * (pl["px"] + 2 * V) * esz
                    extra = (0 if pl["r_outside_smem"] else 1) + pl["delta_in_smem"] + pl["q_in_smem"]
                    assert pl["smem_bytes"] == p_bytes + extra * pl["rows_per_thread"] * 512 * 16
                    assert not (pl["r_outside_smem"] and pl["delta_in_smem"])
                    assert not (pl["q_in_smem"] and pl["r_outside_smem"] and not pl["r_delta_in_tmem"])
                    if pl["r_delta_in_tmem"]:                         # a thread's share of tensor memory: 16 + 16 chunks
                        assert pl["rows_per_thread"] <= 16 and pl["r_outside_smem"] == 1
                    for n, parts, w, big in ((ny, pl["gy"], pl["wy"], pl["ly"]), (nz, pl["gz"], pl["wz"], pl["lz"])):
                        cuts = [omni.resident_split(n, parts, i, w) for i in range(parts + 1)]
                        assert cuts[0] == 0 and cuts[-1] == n
                        sizes = np.diff(cuts)
                        assert (sizes >= 1).all() and sizes.max() == big
                        if w > 0 and parts > 2:
                            assert sizes[0] <= sizes[1:-1].min() + 1 and sizes[-1] <= sizes[1:-1].min() + 1
    assert seen > 60
    # rows longer than one chunk per thread, and grids whose p array cannot fit: no plan
    assert omni.resident_plan(4096, 64, 1, "f32") is None and omni.resident_plan(1100, 900, 1, "f64") is None
    assert omni.resident_plan(256, 256, 256, "f32") is None and omni.resident_plan(500, 500, 500, "f32") is None
    # the weighted cut equalises cost: 128 cells in 8 parts, face cells cost 7 instead of 4
    cuts = [omni.resident_split(128, 8, i, 3) for i in range(9)]
    cost = lambda a, b: sum(7 if x in (0, 1, 126, 127) else 4 for x in range(a, b))
    costs = [cost(cuts[i], cuts[i + 1]) for i in range(8)]
    assert max(costs) - min(costs) <= 7 and cuts[1] < 16 and cuts[8] - cuts[7] < 16
    assert [omni.resident_split(128, 8, i, 0) for i in range(9)] == list(range(0, 129, 16))
