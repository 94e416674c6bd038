"""Thin ctypes binding of include/omni.h: argument marshalling only.

Every step of the path runs in the CUDA kernels of libomni.so; torch is used for device memory and streams.
There is no CPU fallback: a missing library or a missing CUDA device raises.
Arrays are torch tensors in C order with x the fastest index: shape (nz, ny, nx) or (ny, nx).
"""
import ctypes as C
import os

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None

OMNI_OK, OMNI_NOT_CONVERGED = 0, 1
STATUS_NAMES = {0: "OMNI_OK", 1: "OMNI_NOT_CONVERGED", -1: "OMNI_ERR_INVALID_ARG", -2: "OMNI_ERR_CUDA",
                -3: "OMNI_ERR_ALLOC", -4: "OMNI_ERR_BREAKDOWN", -5: "OMNI_ERR_TOO_LARGE"}
# every symbol include/omni.h declares
SYMBOLS = ["omni_solve_f64", "omni_solve_f32", "omni_workspace_bytes", "omni_solve_f64_ws", "omni_solve_f32_ws",
           "omni_solve_host_f64", "omni_solve_host_f32", "omni_solve_batch2d_f64", "omni_solve_batch2d_f32", "omni_solve_guess_f64", "omni_solve_guess_f32", "omni_solve_direct_f64", "omni_solve_direct_f32", "omni_solve_pcg_f64", "omni_solve_pcg_f32", "omni_solve_pcg_batch2d_f64", "omni_solve_pcg_batch2d_f32", "omni_solve_ex_f64", "omni_solve_ex_f32", "omni_options_init", "omni_slab_plan", "omni_slab_unique_id", "omni_slab_comm_create", "omni_slab_comm_destroy",
           "omni_solve_slab_f64", "omni_solve_slab_f32", "omni_source_noalloc_f64", "omni_source_noalloc_f32",
           "omni_source_noalloc_max_cells", "omni_solve_direct_batch2d_f64", "omni_solve_direct_batch2d_f32", "omni_solve_cascade_f64", "omni_solve_cascade_f32", "omni_velocity_source_f64", "omni_velocity_source_f32", "omni_rans_source_f64", "omni_rans_source_f32",
           "omni_compressible_rans_source_f64", "omni_compressible_rans_source_f32", "omni_constants", "omni_source_f64", "omni_source_f32",
           "omni_apply_M_f64", "omni_apply_M_f32", "omni_residual_f64", "omni_residual_f32", "omni_launch_count",
           "omni_set_loop_mode", "omni_resident_plan", "omni_resident_split", "omni_set_history", "omni_release_memory", "omni_profile_enable", "omni_profile_read", "omni_status_string", "omni_version"]


class OmniError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"{what}: {STATUS_NAMES.get(code, code)} ({status_string(code)})")
        self.code = code


class Info(C.Structure):
    _fields_ = [("outer_iters", C.c_int), ("cg_iters_total", C.c_longlong), ("eps_R_final", C.c_double),
                ("norm_S", C.c_double), ("status", C.c_int)]

    def as_dict(self):
        return {"outer_iters": self.outer_iters, "cg_iters_total": self.cg_iters_total,
                "eps_R_final": self.eps_R_final, "norm_S": self.norm_S, "status": self.status}


def lib():
    """Loads libomni.so (building it in-tree first if nvcc is available and the sources are newer)."""
    global _lib
    if _lib is None:
        path = os.environ.get("OMNI_LIB")          # debug: load an alternative build of the same library
        if not path:
            path = os.path.join(_HERE, "libomni.so")
            try:
                path = _build.build()
            except Exception:
                if not os.path.exists(path):
                    raise
        L = C.CDLL(path)
        L.omni_workspace_bytes.restype = C.c_size_t
        L.omni_launch_count.restype = C.c_longlong
        L.omni_source_noalloc_max_cells.restype = C.c_longlong
        L.omni_status_string.restype = C.c_char_p
        _lib = L
    return _lib


def status_string(code):
    return lib().omni_status_string(C.c_int(code)).decode()


def version():
    return int(lib().omni_version())


def launch_count(reset=False):
    return int(lib().omni_launch_count(C.c_int(1 if reset else 0)))


def set_loop_mode(mode):
    """0 = automatic (default), 1 = host-driven debug loop, 2 = CUDA-graph loop, 3 = persistent cooperative kernel
    (include/omni.h).  Returns the previous mode."""
    return int(lib().omni_set_loop_mode(C.c_int(mode)))


def resident_plan(nx, ny, nz, dtype="f32", nsm=148, lop=False):
    """omni_resident_plan: the box decomposition of the SM-resident loop (loop mode 5) for this grid, or None if the grid
    does not fit the SMs.  Host only."""
    out = (C.c_int * 13)()
    rc = lib().omni_resident_plan(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_int(4 if dtype == "f32" else 8), C.c_int(nsm),
                                  C.c_int(1 if lop else 0), out)
    if rc < 0:
        raise OmniError(rc, "omni_resident_plan")
    if rc == 0:
        return None
    keys = ("gy", "gz", "ly", "lz", "smem_bytes", "rows_per_thread", "r_outside_smem", "delta_in_smem", "q_in_smem", "wy", "wz", "px", "r_delta_in_tmem")
    return dict(zip(keys, list(out)))


def resident_split(n, parts, i, wface=0):
    return int(lib().omni_resident_split(C.c_int(n), C.c_int(parts), C.c_int(i), C.c_int(wface)))


def set_history(buf, cg_iters=None):
    """omni_set_history: buf = CUDA float64 tensor that the next solves fill with eps_R of every outer residual check,
    cg_iters = optional CUDA int32 tensor of the same length for the CG iterations per outer iteration (None switches it
    off).  The caller keeps the tensors alive while they are registered."""
    if buf is None:
        rc = lib().omni_set_history(C.c_void_p(0), C.c_void_p(0), C.c_int(0))
    else:
        import torch
        if buf.dtype != torch.float64 or not buf.is_cuda or not buf.is_contiguous():
            raise TypeError("history buffer must be a contiguous CUDA float64 tensor")
        if cg_iters is not None and (cg_iters.dtype != torch.int32 or not cg_iters.is_cuda or not cg_iters.is_contiguous()
                                     or cg_iters.numel() != buf.numel()):
            raise TypeError("cg_iters must be a contiguous CUDA int32 tensor as long as the history buffer")
        rc = lib().omni_set_history(_ptr(buf), _ptr(cg_iters), C.c_int(buf.numel()))
    if rc < 0:
        raise OmniError(rc, "omni_set_history")


def release_memory():
    lib().omni_release_memory()


def profile_enable(on):
    return int(lib().omni_profile_enable(C.c_int(1 if on else 0)))


def profile_read(reset=False):
    """{'K2': (ms, launches), 'K3': ..., 'K4': ...} accumulated by host-loop solves while profiling was on."""
    ms = (C.c_double * 3)()
    n = (C.c_longlong * 3)()
    lib().omni_profile_read(ms, n, C.c_int(1 if reset else 0))
    return {k: (ms[i], n[i]) for i, k in enumerate(("K2", "K3", "K4"))}


def constants(nx, ny, nz, dx, dy, dz):
    out = (C.c_double * 13)()
    rc = lib().omni_constants(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(dx), C.c_double(dy), C.c_double(dz), out)
    if rc != 0:
        raise OmniError(rc, "omni_constants")
    v = list(out)
    return {"F": v[0:3], "A_tot": v[3], "c": [v[4:7], v[7:10], v[10:13]]}


def workspace_bytes(nx, ny, nz, dtype):
    return int(lib().omni_workspace_bytes(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_int(0 if dtype == "f32" else 1)))


# ----------------------------------------------------------------------------------------------- marshalling

def _dims(t):
    if t.dim() == 2:
        return t.shape[1], t.shape[0], 1
    if t.dim() == 3:
        return t.shape[2], t.shape[1], t.shape[0]
    raise ValueError("expected a 2D (ny, nx) or 3D (nz, ny, nx) tensor")


def _suffix(t):
    import torch
    if t.dtype == torch.float32:
        return "f32"
    if t.dtype == torch.float64:
        return "f64"
    raise TypeError("fp32 or fp64 tensors only")


def _ptr(t):
    return C.c_void_p(0 if t is None else t.data_ptr())


def _check(ts, device_type):
    for t in ts:
        if t is None:
            continue
        if not t.is_contiguous():
            raise ValueError("tensors must be contiguous")
        if t.device.type != device_type:
            raise ValueError(f"tensor on {t.device}, expected {device_type}")


def _check_like(ref, fields, mask=None, mask_shape=None, what="gx"):
    """Every field tensor must match `ref` in shape and dtype (the C entry points take one nx, ny, nz and one element
    type for all of them); the mask is uint8 with the grid's shape (`mask_shape` for the batched entry points)."""
    import torch
    for name, t in fields:
        if t is None:
            continue
        if t.dtype != ref.dtype or tuple(t.shape) != tuple(ref.shape):
            raise TypeError(f"{name}: shape {tuple(t.shape)} / {t.dtype} does not match {what} {tuple(ref.shape)} / {ref.dtype}")
    if mask is not None:
        want = tuple(ref.shape) if mask_shape is None else tuple(mask_shape)
        if mask.dtype != torch.uint8 or tuple(mask.shape) != want:
            raise TypeError(f"mask must be uint8 with shape {want}, got {mask.dtype} {tuple(mask.shape)}")


def _stream(dev):
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2311_16935_b200 needs a CUDA device: there is no CPU fallback")
    return C.c_void_p(torch.cuda.current_stream(dev).cuda_stream)


def _geom(gx, d):
    nx, ny, nz = _dims(gx)
    dx, dy = float(d[0]), float(d[1])
    dz = float(d[2]) if len(d) > 2 else 1.0
    return (C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(dx), C.c_double(dy), C.c_double(dz))


def solve(gx, gy, gz, mask, d, tol, max_outer, max_cg, out=None, workspace=None, want_info=True):
    """Algorithm 1 (omni_solve_f32/f64[_ws]) on device tensors, or omni_solve_host_* on CPU tensors.

    d = (dx, dy[, dz]).  Returns (P, info dict or None).  Raises OmniError on negative status codes."""
    import torch
    sfx = _suffix(gx)
    host = gx.device.type == "cpu"
    _check([gx, gy, gz, mask, out], "cpu" if host else "cuda")
    _check_like(gx, [("gy", gy), ("gz", gz), ("out", out)], mask)
    if workspace is not None and (not workspace.is_cuda or not workspace.is_contiguous() or workspace.data_ptr() % 256):
        raise ValueError("workspace must be a contiguous CUDA tensor aligned to 256 bytes")
    P = out if out is not None else torch.empty_like(gx)
    info = Info()
    geom = _geom(gx, d)
    tail = (C.c_double(tol), C.c_int(max_outer), C.c_int(max_cg))
    if host:
        dev = torch.device("cuda", torch.cuda.current_device()) if torch.cuda.is_available() else None
        fn = getattr(lib(), f"omni_solve_host_{sfx}")
        rc = fn(*geom, _ptr(gx), _ptr(gy), _ptr(gz), _ptr(mask), _ptr(P), *tail, _stream(dev), C.byref(info))
    else:
        with torch.cuda.device(gx.device):
            st = _stream(gx.device)
            ip = C.byref(info) if want_info else None
            if workspace is not None:
                fn = getattr(lib(), f"omni_solve_{sfx}_ws")
                rc = fn(*geom, _ptr(gx), _ptr(gy), _ptr(gz), _ptr(mask), _ptr(P), *tail, _ptr(workspace),
                        C.c_size_t(workspace.numel() * workspace.element_size()), st, ip)
            else:
                fn = getattr(lib(), f"omni_solve_{sfx}")
                rc = fn(*geom, _ptr(gx), _ptr(gy), _ptr(gz), _ptr(mask), _ptr(P), *tail, st, ip)
    if rc < 0:
        raise OmniError(rc, f"omni_solve_{sfx}")
    return P, (info.as_dict() if (want_info or host) else None)


def solve_guess(gx, gy, gz, mask, d, tol, max_outer, max_cg, P_init, out=None):
    """omni_solve_guess_*: Algorithm 1 started from the first guess P_init.  Returns (P, info dict)."""
    return solve_direct(gx, gy, gz, mask, d, tol, max_outer, max_cg, out=out, P_init=P_init, _entry="omni_solve_guess")


def solve_direct(gx, gy, gz, mask, d, tol, max_outer, max_cg, out=None, P_init=None, _entry="omni_solve_direct"):
    """omni_solve_direct_*: the fixed point of Algorithm 1 by CG on L P = S (not the paper's iteration; include/omni.h).
    CUDA tensors; d = (dx, dy[, dz]).  Returns (P, info dict).  (`_entry` selects the C entry point with the same
    argument list: omni_solve_guess_* shares the marshalling.)"""
    import torch
    sfx = _suffix(gx)
    _check([gx, gy, gz, mask, out, P_init], "cuda")
    _check_like(gx, [("gy", gy), ("gz", gz), ("out", out), ("P_init", P_init)], mask)
    P = out if out is not None else torch.empty_like(gx)
    info = Info()
    with torch.cuda.device(gx.device):
        fn = getattr(lib(), f"{_entry}_{sfx}")
        rc = fn(*_geom(gx, d), _ptr(gx), _ptr(gy), _ptr(gz), _ptr(mask), _ptr(P_init), _ptr(P), C.c_double(tol), C.c_int(max_outer),
                C.c_int(max_cg), _stream(gx.device), C.byref(info))
    if rc < 0:
        raise OmniError(rc, f"{_entry}_{sfx}")
    return P, info.as_dict()


def solve_pcg(gx, gy, gz, mask, d, tol, max_outer, max_cg, out=None, P_init=None):
    """omni_solve_pcg_*: the fixed point L P = S by multigrid-preconditioned CG (include/omni.h).  Returns (P, info dict)."""
    return solve_direct(gx, gy, gz, mask, d, tol, max_outer, max_cg, out=out, P_init=P_init, _entry="omni_solve_pcg")


class Options(C.Structure):
    """omni_options of include/omni.h."""
    _fields_ = [("struct_size", C.c_size_t), ("loop_mode", C.c_int), ("hist_capacity", C.c_int),
                ("d_hist_eps_R", C.c_void_p), ("d_hist_cg_iters", C.c_void_p), ("d_hist_eps_P", C.c_void_p),
                ("d_P64_out", C.c_void_p), ("d_status", C.c_void_p), ("single_reduction", C.c_int)]


METHODS = {"alg1": 0, "direct": 1, "pcg": 2}


def solve_ex(gx, gy, gz, mask, d, tol, max_outer, max_cg, method="alg1", P_init=None, out=None, loop_mode=-1,
             hist_eps_R=None, hist_cg_iters=None, hist_eps_P=None, P64_out=None, status=None, want_info=True,
             single_reduction=False):
    """omni_solve_ex_*: one solve with per-call options (omni_options): loop mode, history buffers (CUDA float64 /
    int32 tensors of one common length), the fp64 master pressure (CUDA float64 tensor shaped like gx) and a device
    status word (CUDA int32 tensor with one element).  Returns (P, info dict or None)."""
    import torch
    sfx = _suffix(gx)
    _check([gx, gy, gz, mask, out, P_init, hist_eps_R, hist_cg_iters, hist_eps_P, P64_out, status], "cuda")
    _check_like(gx, [("gy", gy), ("gz", gz), ("out", out), ("P_init", P_init)], mask)
    hs = [t for t in (hist_eps_R, hist_cg_iters, hist_eps_P) if t is not None]
    cap = hs[0].numel() if hs else 0
    for t, dt in ((hist_eps_R, torch.float64), (hist_cg_iters, torch.int32), (hist_eps_P, torch.float64)):
        if t is not None and (t.dtype != dt or t.numel() != cap):
            raise TypeError("history tensors: float64 / int32 / float64, one common length")
    if P64_out is not None and (P64_out.dtype != torch.float64 or tuple(P64_out.shape) != tuple(gx.shape)):
        raise TypeError("P64_out must be float64 with the shape of gx")
    if status is not None and (status.dtype != torch.int32 or status.numel() != 1):
        raise TypeError("status must be one int32")
    o = Options()
    lib().omni_options_init(C.byref(o))
    o.loop_mode, o.hist_capacity = loop_mode, cap
    o.d_hist_eps_R, o.d_hist_cg_iters, o.d_hist_eps_P = (None if t is None else t.data_ptr() for t in (hist_eps_R, hist_cg_iters, hist_eps_P))
    o.d_P64_out = None if P64_out is None else P64_out.data_ptr()
    o.d_status = None if status is None else status.data_ptr()
    o.single_reduction = 1 if single_reduction else 0
    P = out if out is not None else torch.empty_like(gx)
    info = Info()
    with torch.cuda.device(gx.device):
        fn = getattr(lib(), f"omni_solve_ex_{sfx}")
        rc = fn(*_geom(gx, d), _ptr(gx), _ptr(gy), _ptr(gz), _ptr(mask), _ptr(P_init), _ptr(P), C.c_double(tol), C.c_int(max_outer),
                C.c_int(max_cg), C.c_int(METHODS[method]), C.byref(o), _stream(gx.device), C.byref(info) if want_info else None)
    if rc < 0:
        raise OmniError(rc, f"omni_solve_ex_{sfx}")
    return P, (info.as_dict() if want_info else None)


def slab_plan(nz, nranks, rank):
    """omni_slab_plan: (z0, z1, zlo, zhi) -- owned planes [z0, z1) and window [zlo, zhi) of `rank` (host only)."""
    v = [C.c_int(0) for _ in range(4)]
    rc = lib().omni_slab_plan(C.c_int(nz), C.c_int(nranks), C.c_int(rank), *[C.byref(x) for x in v])
    if rc != 0:
        raise OmniError(rc, "omni_slab_plan")
    return tuple(x.value for x in v)


def _slab_call(sfx, nx, ny, nz, d, ranks, wins, tol, max_outer, max_cg, method, nranks, comm, dev):
    """wins: per local rank (gx, gy, gz, mask or None, P_out) window tensors.  Marshals the pointer arrays."""
    n = len(ranks)
    arr = lambda i: (C.c_void_p * n)(*[None if w[i] is None else w[i].data_ptr() for w in wins])
    masks = arr(3) if any(w[3] is not None for w in wins) else None
    info = Info()
    fn = getattr(lib(), f"omni_solve_slab_{sfx}")
    rc = fn(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(float(d[0])), C.c_double(float(d[1])), C.c_double(float(d[2])),
            C.c_int(n), (C.c_int * n)(*ranks), arr(0), arr(1), arr(2), masks, arr(4), C.c_double(tol), C.c_int(max_outer),
            C.c_int(max_cg), C.c_int(METHODS[method]), C.c_int(nranks), C.c_void_p(comm), _stream(dev), C.byref(info))
    if rc < 0:
        raise OmniError(rc, f"omni_solve_slab_{sfx}")
    return info.as_dict()


def solve_slab(gx, gy, gz, mask, d, tol, max_outer, max_cg, nslabs, method="alg1"):
    """omni_solve_slab_* with all `nslabs` ranks on this device (comm = NULL): the global CUDA tensors are cut into the
    ranks' windows, solved as z-slabs with halo exchange, and the owned planes are put together again.  Returns (P, info)."""
    import torch
    sfx = _suffix(gx)
    _check([gx, gy, gz, mask], "cuda")
    _check_like(gx, [("gy", gy), ("gz", gz)], mask)
    if gx.dim() != 3:
        raise ValueError("z-slab sharding needs a 3D grid")
    nz, ny, nx = gx.shape
    plans = [slab_plan(nz, nslabs, r) for r in range(nslabs)]
    wins = []
    for (z0, z1, zlo, zhi) in plans:
        wins.append((gx[zlo:zhi].contiguous(), gy[zlo:zhi].contiguous(), gz[zlo:zhi].contiguous(),
                     None if mask is None else mask[zlo:zhi].contiguous(), torch.empty((zhi - zlo, ny, nx), dtype=gx.dtype, device=gx.device)))
    with torch.cuda.device(gx.device):
        info = _slab_call(sfx, nx, ny, nz, d, list(range(nslabs)), wins, tol, max_outer, max_cg, method, nslabs, None, gx.device)
    P = torch.empty_like(gx)
    for (z0, z1, zlo, zhi), w in zip(plans, wins):
        P[z0:z1] = w[4][z0 - zlo:z1 - zlo]
    return P, info


def slab_comm_create(rank, nranks, broadcast):
    """One NCCL communicator for omni_solve_slab_* with one rank per process.  `broadcast(bytes_or_None) -> bytes`
    ships rank 0's 128-byte id to every rank (e.g. through torch.distributed.broadcast_object_list)."""
    buf = C.create_string_buffer(128)
    if rank == 0:
        rc = lib().omni_slab_unique_id(buf)
        if rc != 0:
            raise OmniError(rc, "omni_slab_unique_id")
    raw = broadcast(buf.raw if rank == 0 else None)
    comm = C.c_void_p(0)
    rc = lib().omni_slab_comm_create(C.c_int(rank), C.c_int(nranks), C.create_string_buffer(raw, 128), C.byref(comm))
    if rc != 0:
        raise OmniError(rc, "omni_slab_comm_create")
    return comm.value


def slab_comm_destroy(comm):
    lib().omni_slab_comm_destroy(C.c_void_p(comm))


def solve_slab_rank(gx_win, gy_win, gz_win, mask_win, d, nz, rank, nranks, comm, tol, max_outer, max_cg, method="alg1"):
    """This process's rank of a sharded solve: *_win are the CUDA tensors of its window [zlo, zhi) (slab_plan); `comm` from
    slab_comm_create.  Returns (P on the owned planes, info)."""
    import torch
    sfx = _suffix(gx_win)
    _check([gx_win, gy_win, gz_win, mask_win], "cuda")
    _check_like(gx_win, [("gy", gy_win), ("gz", gz_win)], mask_win)
    z0, z1, zlo, zhi = slab_plan(nz, nranks, rank)
    if gx_win.shape[0] != zhi - zlo:
        raise ValueError(f"rank {rank} of {nranks}: the window holds planes [{zlo}, {zhi})")
    _, ny, nx = gx_win.shape
    out = torch.empty_like(gx_win)
    with torch.cuda.device(gx_win.device):
        info = _slab_call(sfx, nx, ny, nz, d, [rank], [(gx_win, gy_win, gz_win, mask_win, out)], tol, max_outer, max_cg, method,
                          nranks, comm, gx_win.device)
    return out[z0 - zlo:z1 - zlo], info


def velocity_source(u, v, w, mask, d, rho=1.0, mu=0.0, dudt=None):
    """omni_velocity_source_*: g = f(u) of Eq. 1 on CUDA tensors (w = None in 2D; dudt = optional list of local
    accelerations).  Returns [gx, gy(, gz)]."""
    import torch
    sfx = _suffix(u)
    acc = list(dudt) if dudt is not None else [None, None, None]
    acc += [None] * (3 - len(acc))
    _check([u, v, w, mask] + acc, "cuda")
    _check_like(u, [("v", v), ("w", w)] + [("dudt", t) for t in acc], mask, what="u")
    g = [torch.empty_like(u), torch.empty_like(u), None if w is None else torch.empty_like(u)]
    with torch.cuda.device(u.device):
        fn = getattr(lib(), f"omni_velocity_source_{sfx}")
        rc = fn(*_geom(u, d), _ptr(u), _ptr(v), _ptr(w), _ptr(acc[0]), _ptr(acc[1]), _ptr(acc[2]), _ptr(mask),
                C.c_double(rho), C.c_double(mu), _ptr(g[0]), _ptr(g[1]), _ptr(g[2]), _stream(u.device))
    if rc < 0:
        raise OmniError(rc, f"omni_velocity_source_{sfx}")
    return g[:2] if w is None else g


def _stress_array(stress, nd):
    """HOST array of device pointers to the Reynolds stresses (2D: xx, yy, xy; 3D: xx, yy, zz, xy, xz, yz), or None."""
    if stress is None:
        return None
    if len(stress) != (3 if nd == 2 else 6):
        raise ValueError("stress: 3 components (xx, yy, xy) in 2D, 6 (xx, yy, zz, xy, xz, yz) in 3D")
    return (C.c_void_p * len(stress))(*[_ptr(t) for t in stress])


def rans_source(u, v, w, stress, mask, d, rho=1.0):
    """omni_rans_source_*: f of Eq. 42 from the mean velocity and the Reynolds stresses (CUDA tensors; w = None in 2D;
    stress = list of tensors or None).  Returns [fx, fy(, fz)]."""
    import torch
    sfx = _suffix(u)
    _check([u, v, w, mask] + (list(stress) if stress is not None else []), "cuda")
    _check_like(u, [("v", v), ("w", w)] + [("stress", t) for t in (stress or [])], mask, what="u")
    g = [torch.empty_like(u), torch.empty_like(u), None if w is None else torch.empty_like(u)]
    arr = _stress_array(stress, 2 if w is None else 3)
    with torch.cuda.device(u.device):
        rc = getattr(lib(), f"omni_rans_source_{sfx}")(*_geom(u, d), _ptr(u), _ptr(v), _ptr(w), arr, _ptr(mask), C.c_double(rho),
                                                       _ptr(g[0]), _ptr(g[1]), _ptr(g[2]), _stream(u.device))
    if rc < 0:
        raise OmniError(rc, f"omni_rans_source_{sfx}")
    return g[:2] if w is None else g


def compressible_rans_source(u, v, w, stress, mask, d, gamma=1.4, mach_inf=2.0, v_inf=1.0, rgas_t_inf=1.0):
    """omni_compressible_rans_source_*: g = grad ln(P / P_inf) of Eq. 43-44.  Returns [gx, gy(, gz)]."""
    import torch
    sfx = _suffix(u)
    _check([u, v, w, mask] + (list(stress) if stress is not None else []), "cuda")
    _check_like(u, [("v", v), ("w", w)] + [("stress", t) for t in (stress or [])], mask, what="u")
    g = [torch.empty_like(u), torch.empty_like(u), None if w is None else torch.empty_like(u)]
    arr = _stress_array(stress, 2 if w is None else 3)
    with torch.cuda.device(u.device):
        fn = getattr(lib(), f"omni_compressible_rans_source_{sfx}")
        rc = fn(*_geom(u, d), _ptr(u), _ptr(v), _ptr(w), arr, _ptr(mask), C.c_double(gamma), C.c_double(mach_inf),
                C.c_double(v_inf), C.c_double(rgas_t_inf), _ptr(g[0]), _ptr(g[1]), _ptr(g[2]), _stream(u.device))
    if rc < 0:
        raise OmniError(rc, f"omni_compressible_rans_source_{sfx}")
    return g[:2] if w is None else g


def solve_cascade(gx, gy, gz, mask, d, tol, max_outer, max_cg, levels=3, out=None):
    """omni_solve_cascade_*: omni_solve_direct_* started from a guess computed on `levels` coarser grids."""
    import torch
    sfx = _suffix(gx)
    _check([gx, gy, gz, mask, out], "cuda")
    _check_like(gx, [("gy", gy), ("gz", gz), ("out", out)], mask)
    P = out if out is not None else torch.empty_like(gx)
    info = Info()
    with torch.cuda.device(gx.device):
        fn = getattr(lib(), f"omni_solve_cascade_{sfx}")
        rc = fn(*_geom(gx, d), _ptr(gx), _ptr(gy), _ptr(gz), _ptr(mask), _ptr(P), C.c_double(tol), C.c_int(max_outer),
                C.c_int(max_cg), C.c_int(levels), _stream(gx.device), C.byref(info))
    if rc < 0:
        raise OmniError(rc, f"omni_solve_cascade_{sfx}")
    return P, info.as_dict()


def solve_batch2d(gx, gy, mask2d, d, tol, max_outer, max_cg, P_init=None, out=None, direct=False, pcg=False):
    """omni_solve_batch2d_* (direct=True: omni_solve_direct_batch2d_*; pcg=True: omni_solve_pcg_batch2d_*): gx, gy
    (nb, ny, nx) CUDA tensors, mask2d (ny, nx) uint8 or None, d = (dx, dy)."""
    import torch
    sfx = _suffix(gx)
    _check([gx, gy, mask2d, P_init, out], "cuda")
    if gx.dim() != 3:
        raise ValueError("expected (nb, ny, nx) tensors")
    nb, ny, nx = gx.shape
    _check_like(gx, [("gy", gy), ("P_init", P_init), ("out", out)], mask2d, mask_shape=(ny, nx))
    P = out if out is not None else torch.empty_like(gx)
    info = Info()
    with torch.cuda.device(gx.device):
        name = "omni_solve_pcg_batch2d" if pcg else "omni_solve_direct_batch2d" if direct else "omni_solve_batch2d"
        fn = getattr(lib(), f"{name}_{sfx}")
        rc = fn(C.c_int(nx), C.c_int(ny), C.c_int(nb), C.c_double(float(d[0])), C.c_double(float(d[1])), _ptr(gx), _ptr(gy),
                _ptr(mask2d), _ptr(P_init), _ptr(P), C.c_double(tol), C.c_int(max_outer), C.c_int(max_cg),
                _stream(gx.device), C.byref(info))
    if rc < 0:
        raise OmniError(rc, f"omni_solve_batch2d_{sfx}")
    return P, info.as_dict()


def source(gx, gy, gz, mask, d):
    """S of Eq. 9 (omni_source_*).  Returns (S, ||S||)."""
    import torch
    sfx = _suffix(gx)
    _check([gx, gy, gz, mask], "cuda")
    _check_like(gx, [("gy", gy), ("gz", gz)], mask)
    S = torch.empty_like(gx)
    nrm = C.c_double(0.0)
    with torch.cuda.device(gx.device):
        rc = getattr(lib(), f"omni_source_{sfx}")(*_geom(gx, d), _ptr(gx), _ptr(gy), _ptr(gz), _ptr(mask), _ptr(S),
                                                  C.byref(nrm), _stream(gx.device))
    if rc < 0:
        raise OmniError(rc, f"omni_source_{sfx}")
    return S, nrm.value


def source_noalloc(gx, gy, gz, mask, d, out, norm_out=None):
    """omni_source_noalloc_*: S of Eq. 9 into the caller's `out` (and ||S|| into the one-element CUDA float64 tensor
    `norm_out`) with no allocation anywhere: the caller passes every output, the library's only scratch is its fixed
    static device array.  Asynchronous.  Returns `out`."""
    import torch
    sfx = _suffix(gx)
    _check([gx, gy, gz, mask, out, norm_out], "cuda")
    _check_like(gx, [("gy", gy), ("gz", gz), ("out", out)], mask)
    if norm_out is not None and (norm_out.dtype != torch.float64 or norm_out.numel() != 1):
        raise TypeError("norm_out must be one float64")
    with torch.cuda.device(gx.device):
        rc = getattr(lib(), f"omni_source_noalloc_{sfx}")(*_geom(gx, d), _ptr(gx), _ptr(gy), _ptr(gz), _ptr(mask), _ptr(out),
                                                          _ptr(norm_out), _stream(gx.device))
    if rc < 0:
        raise OmniError(rc, f"omni_source_noalloc_{sfx}")
    return out


def source_noalloc_max_cells():
    return int(lib().omni_source_noalloc_max_cells())


def apply_M(p, mask, d):
    """q = M p (omni_apply_M_*).  Returns (q, p.Mp)."""
    sfx = _suffix(p)
    _check([p, mask], "cuda")
    _check_like(p, [], mask, what="p")
    import torch
    q = torch.empty_like(p)
    pq = C.c_double(0.0)
    with torch.cuda.device(p.device):
        rc = getattr(lib(), f"omni_apply_M_{sfx}")(*_geom(p, d), _ptr(mask), _ptr(p), _ptr(q), C.byref(pq),
                                                   _stream(p.device))
    if rc < 0:
        raise OmniError(rc, f"omni_apply_M_{sfx}")
    return q, pq.value


def residual(gx, gy, gz, mask, P, d):
    """r = S - L P and eps_R of Eq. 41 (omni_residual_*); P is fp64.  Returns (r, eps_R)."""
    import torch
    sfx = _suffix(gx)
    _check([gx, gy, gz, mask, P], "cuda")
    _check_like(gx, [("gy", gy), ("gz", gz)], mask)
    if P.dtype != torch.float64 or tuple(P.shape) != tuple(gx.shape):
        raise TypeError("P must be fp64 with the shape of gx")
    r = torch.empty_like(gx)
    eps = C.c_double(0.0)
    with torch.cuda.device(gx.device):
        rc = getattr(lib(), f"omni_residual_{sfx}")(*_geom(gx, d), _ptr(gx), _ptr(gy), _ptr(gz), _ptr(mask), _ptr(P),
                                                    _ptr(r), C.byref(eps), _stream(gx.device))
    if rc < 0:
        raise OmniError(rc, f"omni_residual_{sfx}")
    return r, eps.value
