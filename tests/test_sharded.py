"""NEXT-4: block sharding over the GPUs of one node.

CPU (`-m "not gpu"`): the host logic -- the block partition, the list of remote faces / pulled bytes, and the
collectives of the sharded stage on gloo with world_size 2.
GPU (`-m gpu`, ONE device): (1) two sharded contexts in one process, each owning half of the C4 blocks and seeing the
other half through plain device pointers (what a peer mapping is to the kernels), advanced in lock step, must reproduce
the unsharded 8-block context BIT FOR BIT; (2) the same with two PROCESSES on the one GPU, the buffers exchanged through
CUDA IPC and the control plane on gloo (no kernel of one process ever waits on the other: the ranks meet at host
barriers between the phases of a stage).
"""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ------------------------------------------------------------------------------------------------- host logic
def test_partition_blocks_balanced_and_deterministic():
    from paper_2006_07964_b200.sharded import partition_blocks

    dims = [(96, 96, 96)] * 8
    assert partition_blocks(dims, 1) == [0] * 8
    o2 = partition_blocks(dims, 2)
    assert sorted(o2) == [0] * 4 + [1] * 4 and o2 == partition_blocks(dims, 2)
    o3 = partition_blocks(dims, 3)
    assert sorted(np.bincount(o3).tolist()) == [2, 3, 3]
    o8 = partition_blocks(dims, 8)
    assert sorted(o8) == list(range(8))
    # unequal blocks: largest first onto the least loaded rank; loads within one largest block of each other
    dims = [(64, 64, 64), (32, 32, 32), (32, 32, 64), (64, 32, 32), (16, 16, 16), (48, 48, 48)]
    o = partition_blocks(dims, 2)
    pts = np.array([a * b * c for a, b, c in dims])
    load = [pts[np.array(o) == r].sum() for r in range(2)]
    assert abs(load[0] - load[1]) <= pts.max()
    with pytest.raises(ValueError):
        partition_blocks(dims, 0)


def test_remote_faces_and_halo_bytes_c4(W):
    from paper_2006_07964_b200.sharded import halo_bytes_per_stage, partition_blocks, remote_faces

    case = W.c4_multiblock(nb=8)
    owner = partition_blocks(case.dims, 2)
    nconn = sum(1 for f in case.faces if f["type"] in (1, 2))
    assert nconn == 48
    rf = [remote_faces(case.faces, owner, r) for r in range(2)]
    # every connecting face is local or remote for exactly its owner; a remote face's neighbour is on the other rank
    for r in range(2):
        for t, nr in rf[r]:
            f = case.faces[t]
            assert owner[f["block"]] == r and nr == 1 - r and owner[f["nbr_block"]] == 1 - r
    # the remote relation is symmetric: face (b, f) remote <=> its neighbour's face remote
    pairs = {(case.faces[t]["block"], case.faces[t]["face"]) for r in range(2) for t, _ in rf[r]}
    for r in range(2):
        for t, _ in rf[r]:
            f = case.faces[t]
            assert (f["nbr_block"], f["nbr_face"]) in pairs
    assert len(rf[0]) == len(rf[1]) > 0
    # 6 layers x 8 x 8 face x 5 doubles per remote face
    assert halo_bytes_per_stage(case.dims, case.faces, owner, 0) == len(rf[0]) * 6 * 64 * 5 * 8
    # one rank: nothing is remote
    assert remote_faces(case.faces, [0] * 8, 0) == []


def _comm_worker(rank, world, port, out):
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    from paper_2006_07964_b200.sharded import Comm, partition_blocks

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group(backend="gloo", rank=rank, world_size=world)
    comm = Comm(dist, "cpu")
    res = comm.allreduce(np.arange(5.0) + 10.0 * rank, "sum")       # the stage-1 residual: SUM over the ranks
    dt = comm.allreduce([0.5 - 0.1 * rank], "min")                   # the CFL time step: MIN over the ranks
    comm.stream_barrier(None)                                        # gloo: host barrier
    owners = comm.all_gather_object(partition_blocks([(8, 8, 8)] * 8, world))
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, res.tolist(), float(dt[0]), owners, comm.on_device))


def test_comm_collectives_gloo_world2():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 33500 + os.getpid() % 2000
    procs = [ctx.Process(target=_comm_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, res, dt, owners, on_device in got:
        assert res == [10.0 + 2 * m for m in range(5)]
        assert dt == pytest.approx(0.4)
        assert owners[0] == owners[1] and sorted(owners[0]) == [0] * 4 + [1] * 4   # same map on every rank
        assert on_device is False


# ------------------------------------------------------------------------------------------------- GPU, one device
def _single(case, steps):
    from paper_2006_07964_b200 import binding as B

    g = B.Context(case.dims, case.faces, case.params, device="cuda:0")
    g.load_case(case)
    res = None
    for _ in range(steps):
        res = g.step(case.dt, want_res=True)
    q = [g.to_numpy(b, "q") for b in range(len(case.dims))]
    gq = [g.to_numpy(b, "q", interior=False) for b in range(len(case.dims))]
    dt = g.cfl_dt(0.5)
    g.close()
    return q, gq, res, dt


@pytest.mark.gpu
@pytest.mark.parametrize("world", [2, 3])
def test_sharded_contexts_in_one_process_match_unsharded_bit_for_bit(W, po, world):
    import ctypes as C

    from paper_2006_07964_b200 import binding as B
    from paper_2006_07964_b200.sharded import NG, ShardedContext, partition_blocks

    case = W.c4_multiblock(nb=12, mach=0.3)
    steps = 2
    q1, gq1, res1, dt1 = _single(case, steps)
    owner = partition_blocks(case.dims, world)

    class FakeComm:   # rank identity only: the test itself plays the collectives by calling the phases in turn
        def __init__(self, r):
            self.rank, self.world = r, world

    ctxs = [ShardedContext(case.dims, case.faces, case.params, owner, FakeComm(r), device="cuda:0", defer_create=True)
            for r in range(world)]
    for r, c in enumerate(ctxs):
        peers = {}
        for o in ctxs:
            if o is not c:
                peers.update({b: {n: o.fields[b][n] for n in ("q", "qn", "r", "xyz")} for b in o.local})
        c.create(peer_fields=peers)
        c.comm = None   # no communicator: every "collective" is the loop structure below (one stream, in order)
    for c in ctxs:
        c.load_local(case)
    for phase in range(3):
        for c in ctxs:
            c.finish_load(phase)
    # the single-call stages would run the P2P ghost fill with no cross-process barrier after the sweeps: refused on a
    # context with peer-owned blocks (include/cfd.h), and nothing is enqueued
    for c in ctxs:
        n0 = c.launch_count
        dummy = (C.c_void_p * len(case.dims))(*[1] * len(case.dims))
        for name, call in (("cfd_stage", lambda: B.lib.cfd_stage(c.h, 1, case.dt, None)),
                           ("cfd_stage_fused", lambda: B.lib.cfd_stage_fused(c.h, 1, case.dt, None)),
                           ("cfd_step_host", lambda: B.lib.cfd_step_host(c.h, dummy, dummy, case.dt, None))):
            assert call() == -1, name
            msg = B.lib.cfd_last_error(c.h).decode()
            assert name + ":" in msg and "peer" in msg and "cfd_stage_fused_local" in msg, msg
        assert c.launch_count == n0
    res = None
    for _ in range(steps):
        for s in (1, 2, 3):
            parts = [c.stage_local(s, case.dt, want_res=(s == 1)) for c in ctxs]
            for c in ctxs:
                c.exchange()
            for c in ctxs:
                c.apply_bc()
            if s == 1:
                res = np.sum(parts, axis=0)
    dts = [c.cfl_dt(0.5) for c in ctxs]
    for c in ctxs:
        for b in c.local:
            got = c.interior(b, "q").cpu().numpy()
            assert np.array_equal(got, q1[b]), f"block {b} (rank {c.rank})"
            # the ghost layers the stencils read (3 deep, incl. edges) were pulled from the peers' interiors: identical too
            full = c.field(b, "q").cpu().numpy()
            sl = (slice(None),) + (slice(NG - 3, -(NG - 3)),) * 3
            assert np.array_equal(full[sl], gq1[b][sl]), f"ghosts of block {b}"
    assert np.allclose(res, res1, rtol=1e-13, atol=0.0)      # same terms, the per-rank partial sums are added in another order
    assert min(dts) == dt1                                     # MAX reduction: exact
    # ... and the sharded path beside the ORACLE itself (not only beside the unsharded CUDA path)
    o = po.Oracle(case.dims, case.faces, case.params)
    o.load_case(case)
    for _ in range(steps):
        ro = o.step(case.dt)
    assert np.allclose(res, ro, rtol=1e-10, atol=0.0)
    for c in ctxs:
        for b in c.local:
            qo = o.interior(b, "q")
            assert np.abs(c.interior(b, "q").cpu().numpy() - qo).max() < 1e-11 * np.abs(qo).max(), f"block {b} vs oracle"
    assert abs(min(dts) / o.cfl_dt(0.5) - 1) < 1e-13
    for c in ctxs:
        c.close()


def _ipc_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    from paper_2006_07964_b200 import workloads as W
    from paper_2006_07964_b200.sharded import Comm, ShardedContext, partition_blocks

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group(backend="gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    case = W.c4_multiblock(nb=12, mach=0.3)
    owner = partition_blocks(case.dims, world)
    comm = Comm(dist, "cuda:0")
    c = ShardedContext(case.dims, case.faces, case.params, owner, comm, device="cuda:0")
    c.load_case(case)
    res = None
    for _ in range(2):
        res = c.step(case.dt, want_res=True)
    dt = c.cfl_dt(0.5)
    torch.cuda.synchronize()
    dist.barrier()
    state = {b: c.interior(b, "q").cpu().numpy() for b in c.local}
    dist.barrier()   # nobody unmaps a buffer a peer may still read
    c.close()
    out.put((rank, state, res.tolist(), dt))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.gpu
def test_sharded_two_processes_cuda_ipc_on_one_gpu(W, po):
    import torch.multiprocessing as mp

    case = W.c4_multiblock(nb=12, mach=0.3)
    q1, _, res1, dt1 = _single(case, 2)
    o = po.Oracle(case.dims, case.faces, case.params)   # the oracle beside the two-process run itself
    o.load_case(case)
    for _ in range(2):
        ro = o.step(case.dt)
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 35500 + os.getpid() % 2000
    procs = [ctx.Process(target=_ipc_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    try:
        got = sorted((out.get(timeout=240) for _ in procs), key=lambda x: x[0])
    finally:
        for p in procs:
            p.join(timeout=60)
            if p.is_alive():
                p.kill()
    for p in procs:
        assert p.exitcode == 0
    seen = set()
    for rank, state, res, dt in got:
        for b, q in state.items():
            assert np.array_equal(q, q1[b]), f"block {b} (rank {rank})"
            qo = o.interior(b, "q")
            assert np.abs(q - qo).max() < 1e-11 * np.abs(qo).max(), f"block {b} (rank {rank}) vs oracle"
            seen.add(b)
        assert np.allclose(res, res1, rtol=1e-13, atol=0.0)   # all-reduced over the two ranks
        assert np.allclose(res, ro, rtol=1e-10, atol=0.0)
        assert dt == dt1
    assert seen == set(range(8))


@pytest.mark.gpu
def test_bench_sharded_line_on_one_gpu():
    """`bench.py --sharded` at N = 1 (all blocks local, nothing pulled): the JSON line of the sharded arm."""
    import json
    import subprocess

    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--sharded", "--workload", "c4", "--steps", "2", "--warmup", "3",
                        "--repeats", "1"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads([ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1])
    assert d["scaling"] == "strong" and d["n_gpus"] == 1 and d["unit"] == "Gpts/s"
    assert d["config"]["owner"] == [0] * 8 and d["config"]["halo_bytes_pulled_per_stage_rank0"] == 0
    assert d["state_finite"] and d["value"] > 0.5 and d["e2e"]["value"] > 0 and d["gpu_launches"] > 0


@pytest.mark.gpu
def test_sharded_contexts_with_physical_bcs_match_unsharded(W):
    """The second collective of the sharded stage (between the P2P ghost fill and the BCs): the cylinder cut into four
    blocks, two per "rank", wall and far field next to remote interfaces."""
    from paper_2006_07964_b200.sharded import ShardedContext, partition_blocks

    case = W.c5_cylinder_split(4, ni=96, nj=20, nk=10, noise=1e-2)
    q1, _, res1, dt1 = _single(case, 2)
    owner = partition_blocks(case.dims, 2)

    class FakeComm:
        def __init__(self, r):
            self.rank, self.world = r, 2

    ctxs = [ShardedContext(case.dims, case.faces, case.params, owner, FakeComm(r), device="cuda:0", defer_create=True) for r in range(2)]
    assert all(c.has_bc for c in ctxs)
    for c in ctxs:
        o = ctxs[1 - c.rank]
        c.create(peer_fields={b: {n: o.fields[b][n] for n in ("q", "qn", "r", "xyz")} for b in o.local})
        c.comm = None
    for c in ctxs:
        c.load_local(case)
    for phase in range(3):
        for c in ctxs:
            c.finish_load(phase)
    for _ in range(2):
        for s in (1, 2, 3):
            parts = [c.stage_local(s, case.dt, want_res=(s == 1)) for c in ctxs]
            for c in ctxs:
                c.exchange()
            for c in ctxs:
                c.apply_bc()
            if s == 1:
                res = np.sum(parts, axis=0)
    for c in ctxs:
        for b in c.local:
            assert np.array_equal(c.interior(b, "q").cpu().numpy(), q1[b]), f"block {b}"
    assert np.allclose(res, res1, rtol=1e-13, atol=0.0)
    for c in ctxs:
        c.close()
