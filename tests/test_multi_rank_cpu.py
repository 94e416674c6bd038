"""N > 1 path of bench.py (replicas only) on CPU: gloo, world_size 2.

The data path has no collective; what is shared between ranks is the timing reduction (max over ranks) and the
aggregation of the replicas' work, plus the rule that only rank 0 of the reference arm does anything."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms, e2e = bench.max_over_ranks([100.0 + 50.0 * rank, 2.0 - rank], world)
    dist.barrier()
    q.put((rank, ms, e2e, bench.aggregate_value(1000, 3, world, ms * 1e-3)))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, e2e, val in res:
        assert ms == 150.0 and e2e == 2.0                    # the slowest rank decides
        assert val == pytest.approx(2 * 1000 * 3 / 0.150)    # all replicas' units over that time


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                          "--steps", "1", "--warmup", "0", "--gpus", "2"], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env["RANK"] = "0"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                          "--steps", "1", "--warmup", "0", "--gpus", "2"], env=env, capture_output=True, text=True, timeout=300)
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["metric"] == "grid-point CG updates/s"


def _slab_worker(rank, world, port, q):
    """One rank of a z-slab sharded solve, host side only: its plan from the C library, its window cut from the global
    array, and one halo exchange with its neighbours through the process group (gloo) with the plane indices
    omni_solve_slab_* uses (paper_2311_16935_b200/csrc/omni_api.cu slab_exchange)."""
    import numpy as np
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import paper_2311_16935_b200 as omni
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    nz, ny, nx = 11, 3, 4
    glob = np.arange(nz * ny * nx, dtype=np.float64).reshape(nz, ny, nx)
    z0, z1, zlo, zhi = omni.slab_plan(nz, world, rank)
    plans = [None] * world
    dist.all_gather_object(plans, (z0, z1, zlo, zhi))
    win = torch.from_numpy(glob[zlo:zhi].copy())
    kz0, kz1 = z0 - zlo, z1 - zlo
    own_before = win[kz0:kz1].clone()
    # stale halos, then the exchange: my plane just above / below the owned range <- the neighbour's outermost owned plane
    if kz0 > 0:
        win[:kz0] = -1.0
    if kz1 < win.shape[0]:
        win[kz1:] = -1.0
    reqs = []
    if rank > 0:
        reqs.append(dist.isend(win[kz0].clone(), rank - 1))
        reqs.append(dist.irecv(win[kz0 - 1], rank - 1))
    if rank + 1 < world:
        reqs.append(dist.isend(win[kz1 - 1].clone(), rank + 1))
        reqs.append(dist.irecv(win[kz1], rank + 1))
    for r in reqs:
        r.wait()
    # a scalar all-reduce in rank order, as every reduction of the sharded solve
    part = torch.tensor([float(own_before.sum())], dtype=torch.float64)
    dist.all_reduce(part)
    dist.barrier()
    q.put((rank, plans, win.numpy().copy(), float(part)))
    dist.destroy_process_group()


def test_slab_plan_and_halo_exchange_gloo_world2():
    """NEXT-3 host logic on CPU, two processes: the ranks' plans tile the z axis without gap or overlap, windows reach at
    most two planes beyond the owned range and never outside the grid, the exchanged halo plane is the neighbour's
    outermost owned plane (the window's first halo plane equals the global array there), and the all-reduced total is the
    global one on both ranks."""
    import numpy as np
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_slab_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=180) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    nz, ny, nx = 11, 3, 4
    glob = np.arange(nz * ny * nx, dtype=np.float64).reshape(nz, ny, nx)
    plans = res[0][1]
    assert plans == res[1][1] and plans[0][0] == 0 and plans[-1][1] == nz
    for (a, b) in zip(plans[:-1], plans[1:]):
        assert a[1] == b[0]                                          # no gap, no overlap
    for rank, _, win, total in res:
        z0, z1, zlo, zhi = plans[rank]
        assert 0 <= zlo <= z0 < z1 <= zhi <= nz and z0 - zlo <= 2 and zhi - z1 <= 2
        assert zlo == max(0, z0 - 2) and zhi == min(nz, z1 + 2)
        assert np.array_equal(win[z0 - zlo:z1 - zlo], glob[z0:z1])
        if z0 > 0:
            assert np.array_equal(win[z0 - zlo - 1], glob[z0 - 1])      # first halo plane below: current
        if z1 < nz:
            assert np.array_equal(win[z1 - zlo], glob[z1])              # first halo plane above: current
        assert total == glob.sum()


def test_slab_plan_edge_cases():
    import paper_2311_16935_b200 as omni
    assert omni.slab_plan(5, 1, 0) == (0, 5, 0, 5)
    assert [omni.slab_plan(5, 4, r)[:2] for r in range(4)] == [(0, 2), (2, 3), (3, 4), (4, 5)]
    assert omni.slab_plan(5, 4, 1) == (2, 3, 0, 5)
    for bad in ((3, 4, 0), (8, 2, 2), (8, 0, 0)):
        with pytest.raises(omni.OmniError):
            omni.slab_plan(*bad)
