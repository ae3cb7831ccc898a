"""The N > 1 path: the box cut into z slabs, one per rank (section 3.4).

CPU (gloo, world_size 2): the partition, the neighbour wiring, the handle exchange, the local <-> whole-box
array plumbing and bench.py's max-over-ranks / aggregate helpers -- everything of the multi-rank path that
is not a kernel.
GPU (marked gpu): two processes on ONE GPU, each holding one slab, attach each other's device memory by
CUDA IPC and advance the decomposed step; the result equals the single-domain run bit for bit.  The ranks
synchronise on the host (gloo), no kernel ever waits for another rank's kernel.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _spawn(target, world, *args, timeout=300):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=target, args=(r, world, port, out) + args) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=timeout) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    return res


def _init(rank, world, port, backend="gloo"):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    if backend == "nccl":
        torch.cuda.set_device(0)
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", 0))
    else:
        dist.init_process_group("gloo", rank=rank, world_size=world)


# ---------------------------------------------------------------- CPU: host-side logic

def _worker_timing(rank, world, port, out):
    _init(rank, world, port)
    import bench
    mine = 2.0 + 3.0 * rank                     # ms per K steps measured by this rank
    slowest = bench.max_over_ranks(mine, dist, "cpu")
    value = bench.aggregate_throughput(1000, 4, slowest, world)
    dist.barrier()
    out.put((rank, slowest, value))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_two_ranks():
    for rank, slowest, value in _spawn(_worker_timing, 2):
        assert slowest == 5.0                                  # the slower rank sets the job time
        assert abs(value - 2 * 1000 * 4 / 5.0e-3) < 1e-6       # both slabs' zones over that time


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(1.25, None) == 1.25


def test_slab_partition_covers_the_box():
    """pluto_slab_planes (no device needed): contiguous, disjoint, sizes differ by at most one plane"""
    from paper_2511_20337_b200.distributed import slab_planes
    for nz, nslab in [(256, 8), (26, 4), (19, 2), (352, 4), (7, 7), (12, 1)]:
        parts = [slab_planes(nz, nslab, s) for s in range(nslab)]
        assert parts[0][0] == 0 and sum(n for _, n in parts) == nz
        for (k0, n), (k1, _) in zip(parts, parts[1:]):
            assert k0 + n == k1
        sizes = [n for _, n in parts]
        assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)


def test_neighbours_are_periodic():
    from paper_2511_20337_b200.distributed import neighbour_ranks
    assert neighbour_ranks(0, 4) == (3, 1) and neighbour_ranks(3, 4) == (2, 0)
    assert neighbour_ranks(0, 2) == (1, 1) and neighbour_ranks(1, 2) == (0, 0)
    assert neighbour_ranks(0, 1) == (0, 0)


def _worker_plumbing(rank, world, port, out):
    """what SlabPluto.init / load do around the library calls, with fake handles: every rank ends up with
    the handles of the slab below and above it, and the local parts tile the whole-box state"""
    _init(rank, world, port)
    from paper_2511_20337_b200 import workloads as wl
    from paper_2511_20337_b200.distributed import local_part, neighbour_ranks, slab_planes
    w = wl.random_smooth(10, 6, 9, seed=5)
    k0, nzl = slab_planes(w.nz, world, rank)
    mine = (bytes([rank]) * 64, 1000 + rank, nzl)
    everyone = [None] * world
    dist.all_gather_object(everyone, mine)
    lo, hi = neighbour_ranks(rank, world)
    Ul, Bl = local_part(w.U, w.Bface, w.nx, w.ny, w.nz, k0, nzl)
    # the dt all-reduce of the host-synchronous path: MAX of bit patterns of positive doubles
    bits = torch.tensor([np.float64(1.5 + rank).view(np.int64)], dtype=torch.int64)
    dist.all_reduce(bits, op=dist.ReduceOp.MAX)
    out.put((rank, k0, nzl, everyone[lo][0][0], everyone[hi][0][0], everyone[lo][1], Ul, Bl,
             float(np.int64(bits.item()).view(np.float64))))
    dist.barrier()
    dist.destroy_process_group()


def test_handle_exchange_and_array_plumbing_two_ranks():
    from paper_2511_20337_b200 import workloads as wl
    from paper_2511_20337_b200.distributed import join_parts
    w = wl.random_smooth(10, 6, 9, seed=5)
    res = _spawn(_worker_plumbing, 2)
    for rank, k0, nzl, lo_id, hi_id, lo_sa, Ul, Bl, dtmax in res:
        assert lo_id == hi_id == 1 - rank and lo_sa == 1000 + (1 - rank)
        assert dtmax == 2.5                                    # the larger of 1.5 and 2.5 on both ranks
    U, Bf = join_parts([(k0, nzl, Ul, Bl) for _, k0, nzl, _, _, _, Ul, Bl, _ in res], w.nx, w.ny, w.nz)
    assert np.array_equal(U, w.U) and np.array_equal(Bf, w.Bface)


# ---------------------------------------------------------------- GPU: two slabs, two processes, one device

def _worker_slab(rank, world, port, out, case, backend="gloo"):
    _init(rank, world, port, backend)
    from paper_2511_20337_b200 import workloads as wl
    from paper_2511_20337_b200.distributed import SlabPluto
    name, rk, ghost, steps = case
    w = _case(name)
    sim = SlabPluto(dist, device=0)
    sim.set_integrator(rk)
    sim.load(w, ghost=ghost)
    sim.step(steps)
    dt, t = sim.get_dt(), sim.get_time()
    sim.step(1, fixed_dt=0.5 * dt)
    Ul, Bl = sim.get_state()
    out.put((rank, sim.k0, sim.nzl, Ul, Bl, dt, t))
    sim.finalize()
    dist.barrier()
    dist.destroy_process_group()


def _case(name):
    from paper_2511_20337_b200 import workloads as wl
    if name == "smooth_mc":
        return wl.random_smooth(64, 20, 26, seed=61, limiter=1, box=(1.0, 0.4, 0.5))
    if name == "blast":
        return wl.blast_3d(32)
    w = wl.orszag_tang_3d(32, noise=1e-3)
    w.limiter = 2
    return w


@pytest.mark.gpu
@pytest.mark.parametrize("case", [("smooth_mc", 2, 2, 3), ("blast", 3, 2, 2), ("ot3d_wenoz", 3, 3, 2)], ids=lambda c: c[0])
def test_two_processes_one_slab_each_match_the_single_domain(case):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    sys.path.insert(0, ROOT)
    from paper_2511_20337_b200.binding import Pluto
    from paper_2511_20337_b200.distributed import join_parts
    name, rk, ghost, steps = case
    w = _case(name)
    ref = Pluto()
    ref.set_integrator(rk)
    ref.load(w, ghost=ghost)
    ref.step(steps)
    dt, t = ref.get_dt(), ref.get_time()
    ref.step_fixed_dt(1, 0.5 * dt)
    Ur, Br = ref.get_state()
    ref.set_integrator(2)
    ref.finalize()
    res = _spawn(_worker_slab, 2, case, timeout=600)
    for _, _, _, _, _, dts, ts in res:
        assert dts == dt and ts == t
    U, Bf = join_parts([(k0, nzl, Ul, Bl) for _, k0, nzl, Ul, Bl, _, _ in res], w.nx, w.ny, w.nz)
    assert np.array_equal(U, Ur) and np.array_equal(Bf, Br)


@pytest.mark.gpu
@pytest.mark.parametrize("case", [("smooth_mc", 2, 2, 3), ("ot3d_wenoz", 3, 3, 2)], ids=lambda c: c[0])
def test_nccl_branch_one_rank_matches_the_single_domain(case):
    """the device-side collectives of SlabPluto (backend nccl: the MAX all-reduce on a tensor wrapped around the raw
    pluto_dt_max_bits pointer, and the token all-reduce that serves as the barrier, both ordered on the library's
    stream) in a group of ONE rank: one GPU is all this box has, and ranks whose kernels wait on one another must not
    share a GPU.  The decomposed step with the whole box as its single slab equals the single-domain run bit for bit."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    sys.path.insert(0, ROOT)
    from paper_2511_20337_b200.binding import Pluto
    name, rk, ghost, steps = case
    w = _case(name)
    ref = Pluto()
    ref.set_integrator(rk)
    ref.load(w, ghost=ghost)
    ref.step(steps)
    dt, t = ref.get_dt(), ref.get_time()
    ref.step_fixed_dt(1, 0.5 * dt)
    Ur, Br = ref.get_state()
    ref.set_integrator(2)
    ref.finalize()
    (_, k0, nzl, Ul, Bl, dts, ts), = _spawn(_worker_slab, 1, case, "nccl", timeout=600)
    assert (k0, nzl) == (0, w.nz) and dts == dt and ts == t
    assert np.array_equal(Ul.reshape(Ur.shape), Ur) and np.array_equal(Bl, Br)


@pytest.mark.gpu
def test_bench_refuses_more_gpus_than_the_box_has_and_runs_the_slab_path():
    """`python bench.py --gpus N` without a launcher starts its own ranks; with fewer than N devices it must fail
    loudly instead of timing one GPU.  `--gpus 1 --slab-path` runs the decomposed step (one-rank NCCL group)."""
    import json
    import subprocess
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    too_many = torch.cuda.device_count() + 1
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", str(too_many), "--steps", "1"],
                       capture_output=True, text=True, env=env, timeout=600)
    assert p.returncode != 0 and f"needs {too_many} CUDA devices" in p.stderr and not p.stdout.strip()
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "1", "--slab-path", "--steps", "3",
                        "--warmup", "3", "--repeats", "1", "--e2e-steps", "1"],
                       capture_output=True, text=True, env=env, timeout=900)
    assert p.returncode == 0, p.stderr[-2000:]
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["n_gpus"] == 1 and line["value"] > 0 and line["gpu_launches"] > 0
    assert "z-slab" in line["config"]["parallelism"] and line["config"]["zones"] == 256 ** 3
