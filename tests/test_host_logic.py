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
