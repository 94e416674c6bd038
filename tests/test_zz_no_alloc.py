"""omni_source_noalloc_* -- the source-vector step for callers that cannot allocate (include/omni.h): its output against
the existing path's (omni_source_*, which builds link codes in a pool-allocated workspace), on two calls in a row that share
the library's static scratch array.  Collected last on purpose (the suite runs with pytest -x)."""
import ctypes as C

import numpy as np
import pytest

import paper_2311_16935_b200 as omni
from workloads import make_field

torch = pytest.importorskip("torch")

TOL_STEP = {"f64": 1e-13, "f32": 2e-6}           # as tests/test_gpu_parity.py: a handful of roundings of the largest entry
TDT = {"f64": torch.float64, "f32": torch.float32}


def _case(kind, shape, dtype, seed, frac, nan_cell):
    f = make_field(kind, shape, seed=seed, noise=0.1, kmax=3.0)
    rng = np.random.default_rng(seed)
    mask = (rng.random(shape) > frac).astype(np.uint8) if frac > 0 else None
    np_dt = np.float32 if dtype == "f32" else np.float64
    g = [np.ascontiguousarray(c.astype(np_dt)) for c in f["g"]]
    if nan_cell is not None:
        g[1][nan_cell] = np.nan                   # NaN marks a missing cell as well (Eq. 13)
    g_dev = [torch.from_numpy(c).cuda() for c in g] + [None] * (3 - len(g))
    m_dev = None if mask is None else torch.from_numpy(mask).cuda()
    return g_dev, m_dev, f["d"]


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_source_noalloc_matches_allocating_path_on_two_calls_in_a_row(dtype):
    """Two different problems back to back through the same static scratch (the second one smaller, so stale partials of
    the first stay behind it): S entry by entry and ||S|| against omni_source_*; then the first problem again, bit-identical
    to its first run (nothing of the call in between leaks)."""
    cases = [("fourier3d", (9, 31, 150), 3, 0.1, (4, 7, 20)), ("gaussians2d", (37, 300), 5, 0.05, None),
             ("fourier3d", (5, 16, 264), 7, 0.0, None)]
    first = None
    for kind, shape, seed, frac, nan_cell in cases + cases[:1]:
        g, m, d = _case(kind, shape, dtype, seed, frac, nan_cell)
        out = torch.full(shape, 123.0, dtype=TDT[dtype], device="cuda")
        nrm = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
        S = omni.source_noalloc(g[0], g[1], g[2], m, d, out, nrm)
        torch.cuda.synchronize()
        S_ref, n_ref = omni.source(g[0], g[1], g[2], m, d)
        a, b = S.cpu().numpy().astype(np.float64), S_ref.cpu().numpy().astype(np.float64)
        assert np.isfinite(a).all()
        assert np.abs(a - b).max() <= TOL_STEP[dtype] * 4 * np.abs(b).max()
        assert np.array_equal(a == 0, b == 0)                          # the missing-cell pattern
        assert float(nrm.item()) == pytest.approx(n_ref, rel=1e-12)
        assert float(nrm.item()) == pytest.approx(float(torch.linalg.vector_norm(S.double())), rel=1e-12)
        if first is None:
            first = (a.copy(), float(nrm.item()))
    assert np.array_equal(a, first[0]) and float(nrm.item()) == first[1]
    # norm output is optional
    S2 = omni.source_noalloc(g[0], g[1], g[2], m, d, torch.empty_like(out), None)
    assert torch.equal(S2, S)


@pytest.mark.gpu
def test_source_noalloc_allocates_nothing_and_rejects_oversize():
    """No device memory is taken by the call (the driver's free-memory figure does not move, the library's pool stays as
    trimmed); a grid beyond the fixed scratch is rejected with OMNI_ERR_TOO_LARGE before anything is enqueued."""
    g, m, d = _case("fourier3d", (24, 40, 96), "f32", 11, 0.1, None)
    out = torch.empty_like(g[0])
    nrm = torch.zeros(1, dtype=torch.float64, device="cuda")
    omni.source_noalloc(g[0], g[1], g[2], m, d, out, nrm)               # first call: symbol address looked up
    torch.cuda.synchronize()
    omni.release_memory()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        omni.source_noalloc(g[0], g[1], g[2], m, d, out, nrm)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    cap = omni.source_noalloc_max_cells()
    assert cap == 32760 * 4096
    L = omni.lib()
    rc = L.omni_source_noalloc_f32(C.c_int(1024), C.c_int(1024), C.c_int(129), C.c_double(1), C.c_double(1), C.c_double(1),
                                   C.c_void_p(256), C.c_void_p(256), C.c_void_p(256), None, C.c_void_p(256), None, None)
    assert 1024 * 1024 * 129 > cap and rc == -5 and "no-allocation" in omni.status_string(rc)
    torch.cuda.synchronize()                                             # nothing was enqueued: no fault to collect


def test_source_noalloc_argument_validation_needs_no_device():
    L = omni.lib()
    rc = L.omni_source_noalloc_f64(C.c_int(0), C.c_int(4), C.c_int(1), C.c_double(1), C.c_double(1), C.c_double(1),
                                   C.c_void_p(8), C.c_void_p(8), None, None, C.c_void_p(8), None, None)
    assert rc == -1
    rc = L.omni_source_noalloc_f64(C.c_int(4), C.c_int(4), C.c_int(4), C.c_double(1), C.c_double(1), C.c_double(1),
                                   C.c_void_p(8), C.c_void_p(8), None, None, C.c_void_p(8), None, None)
    assert rc == -1                                                      # 3D needs gz
    rc = L.omni_source_noalloc_f32(C.c_int(2048), C.c_int(2048), C.c_int(64), C.c_double(1), C.c_double(1), C.c_double(1),
                                   C.c_void_p(8), C.c_void_p(8), C.c_void_p(8), None, C.c_void_p(8), None, None)
    assert rc == -5                                                      # 268 M cells > 134 184 960: before any CUDA call
