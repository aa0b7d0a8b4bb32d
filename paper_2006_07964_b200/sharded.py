"""NEXT-4: block sharding over the GPUs of one NVLink / NVSwitch node, one process per GPU.

The paper gives every GPU one sub-block set and exchanges halos through MPI / GPUDirect P2P over PCIe, placing the
processes by PCIe topology.  Here:

  * `partition_blocks` spreads the blocks over the ranks by point count (largest first onto the least loaded rank);
    on NVSwitch every peer is equidistant, so there is no placement problem left;
  * every rank allocates the fields of ITS blocks with torch, exports q, qn, r, xyz through CUDA IPC and maps the
    buffers of all other ranks (`exchange_ipc_handles`): torch.distributed is only the control plane;
  * the C ABI (`cfd_create_blocks_sharded`) gets the whole topology, the local blocks' pointers and the peer-mapped
    pointers of the remote blocks: its ghost-fill kernel pulls the ghost layers of the local blocks straight out of the
    owners' interior cells with P2P loads over NVLink -- nothing is packed, staged or copied through the host;
  * per stage:  cfd_stage_fused_local  ->  collective on the compute stream (every rank has written its new state)
    ->  cfd_exchange_interfaces  ->  [collective, only if physical faces exist]  ->  cfd_apply_bc;
    the stage-1 residual is all-reduced (SUM), the CFL time step all-reduced (MIN).

This module is argument marshalling and torch.distributed plumbing only; every step of the path runs in the kernels of
csrc/.  There is no CPU fallback: `ShardedContext` needs a CUDA device and the extension.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

NG = 6


def partition_blocks(dims, world):
    """owner[b] in [0, world): blocks sorted by point count (ties by index), each onto the currently least loaded rank
    (ties by rank).  Deterministic, so every rank computes the same map without communication."""
    if world < 1:
        raise ValueError("world must be >= 1")
    pts = [int(d[0]) * int(d[1]) * int(d[2]) for d in dims]
    load = [0] * world
    owner = [0] * len(dims)
    for b in sorted(range(len(dims)), key=lambda b: (-pts[b], b)):
        r = min(range(world), key=lambda r: (load[r], r))
        owner[b] = r
        load[r] += pts[b]
    if world <= len(dims) and any(l == 0 for l in load):
        raise ValueError("partition_blocks: a rank received no block")
    return owner


def remote_faces(faces, owner, rank):
    """The connecting faces of `rank`'s blocks whose neighbour lives on another rank: [(face index, neighbour rank)]."""
    out = []
    for t, f in enumerate(faces):
        if owner[f["block"]] == rank and f["type"] in (1, 2) and owner[f["nbr_block"]] != rank:
            out.append((t, owner[f["nbr_block"]]))
    return out


def halo_bytes_per_stage(dims, faces, owner, rank):
    """Bytes this rank pulls from peers per stage: 6 ghost layers x face area x 5 doubles per remote face (edge and corner
    regions not counted)."""
    n = 0
    for t, _ in remote_faces(faces, owner, rank):
        f = faces[t]
        d = dims[f["block"]]
        a = f["face"] // 2
        area = int(d[(a + 1) % 3]) * int(d[(a + 2) % 3])
        n += NG * area * 5 * 8
    return n


class Comm:
    """The collectives the sharded stage needs, on top of torch.distributed (nccl on the GPUs; gloo in the CPU tests and
    in the single-GPU IPC test, where the device-side barrier degrades to stream synchronise + host barrier)."""

    def __init__(self, dist, device="cpu"):
        import torch

        self.torch, self.dist, self.device = torch, dist, torch.device(device)
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        self.backend = dist.get_backend()
        self.on_device = self.backend == "nccl"
        self._tok = torch.zeros(1, dtype=torch.float64, device=self.device if self.on_device else "cpu")

    def stream_barrier(self, stream=None):
        """Every rank's work enqueued so far on `stream` completes before any rank's later work on it starts."""
        if self.on_device:
            with self.torch.cuda.stream(stream):
                self.dist.all_reduce(self._tok)       # ordered on the compute stream, no host synchronisation
        else:
            if stream is not None:
                stream.synchronize()
            self.dist.barrier()

    def allreduce(self, values, op="sum", stream=None):
        """values: 1-D numpy fp64 (host) -> reduced copy on every rank."""
        t = self.torch.from_numpy(np.array(values, dtype=np.float64, copy=True))
        if self.on_device:
            t = t.to(self.device)
        o = {"sum": self.dist.ReduceOp.SUM, "min": self.dist.ReduceOp.MIN, "max": self.dist.ReduceOp.MAX}[op]
        self.dist.all_reduce(t, op=o)
        return t.cpu().numpy()

    def all_gather_object(self, obj):
        out = [None] * self.world
        self.dist.all_gather_object(out, obj)
        return out


def exchange_ipc_handles(comm, local_fields, names=("q", "qn", "r", "xyz")):
    """local_fields: {block: {name: CUDA tensor}} of this rank.  Returns {block: {name: tensor}} for EVERY block of every
    other rank, viewing the owner's memory through CUDA IPC (peer access over NVLink is enabled by the driver when the
    handle is opened).  The returned tensors keep the mappings alive."""
    import torch

    mine = {}
    for b, fl in local_fields.items():
        mine[b] = {}
        for n in names:
            t = fl[n]
            mine[b][n] = (t.untyped_storage()._share_cuda_(), tuple(t.shape), t.storage_offset())
    everyone = comm.all_gather_object(mine)
    peers = {}
    for r, blocks in enumerate(everyone):
        if r == comm.rank:
            continue
        for b, fl in blocks.items():
            peers[b] = {}
            for n, (h, shape, off) in fl.items():
                st = torch.UntypedStorage._new_shared_cuda(*h)
                t = torch.empty(0, dtype=torch.float64, device=st.device)
                t.set_(st, off, shape)
                peers[b][n] = t
    return peers


class ShardedContext:
    """A rank's share of a multi-block case.  `peer_fields` ({block: {q, qn, r, xyz: tensor}}) may be given directly
    (single-process tests hand in another context's tensors); otherwise the buffers are exchanged through CUDA IPC."""

    NV = dict(q=5, qn=5, r=5, xyz=3, khat=9, jac=1)

    def __init__(self, dims, faces, params, owner, comm, device="cuda:0", stream=None, peer_fields=None, defer_create=False):
        import torch

        from . import binding as B

        if not torch.cuda.is_available():
            raise B.CfdError(-6, "no CUDA device: this library has no CPU fallback")
        self.torch, self.B, self.comm = torch, B, comm
        self.device = torch.device(device)
        self.dims = [tuple(int(x) for x in d) for d in dims]
        self.faces, self.params, self.owner = faces, params, list(owner)
        self.rank = comm.rank if comm is not None else 0
        self.local = [b for b in range(len(self.dims)) if self.owner[b] == self.rank]
        self.has_bc = any(f["type"] in (3, 4) for f in faces)
        self.fields = {}
        with torch.cuda.device(self.device):
            for b in self.local:
                ni, nj, nk = self.dims[b]
                shp = (nk + 2 * NG, nj + 2 * NG, ni + 2 * NG)
                self.fields[b] = {n: torch.zeros((nv,) + shp, dtype=torch.float64, device=self.device) for n, nv in self.NV.items()}
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.peer_fields = peer_fields
        self.h = None
        if not defer_create:
            self.create()

    def create(self, peer_fields=None):
        """Maps the peers' buffers (CUDA IPC unless given) and builds the C-ABI context."""
        torch, B = self.torch, self.B
        if peer_fields is not None:
            self.peer_fields = peer_fields
        if self.peer_fields is None:
            self.peer_fields = exchange_ipc_handles(self.comm, self.fields) if len(self.local) < len(self.dims) else {}
        nb = len(self.dims)
        d = (B._Dims * nb)(*[B._Dims(*dd) for dd in self.dims])
        p = B._Params()
        for k in ("gamma", "mach", "reynolds", "prandtl", "weno_eps", "viscous", "scheme"):
            setattr(p, k, self.params[k])
        for a in range(5):
            p.q_inf[a] = self.params["q_inf"][a]
        p.sutherland = float(self.params.get("sutherland", 0.0))
        fa = (B._Face * max(1, len(self.faces)))()
        for t, f in enumerate(self.faces):
            fa[t].block, fa[t].face, fa[t].type = f["block"], f["face"], f["type"]
            fa[t].nbr_block, fa[t].nbr_face = f["nbr_block"], f["nbr_face"]
            for a in range(3):
                fa[t].perm[a], fa[t].sign[a], fa[t].shift[a] = f["perm"][a], f["sign"][a], f["shift"][a]
        ptrs = (B._Ptrs * nb)()
        loc = (C.c_int * nb)()
        for b in range(nb):
            if b in self.fields:
                loc[b] = 1
                for n in self.NV:
                    setattr(ptrs[b], n, self.fields[b][n].data_ptr())
            else:
                loc[b] = 0
                for n in ("q", "qn", "r", "xyz"):
                    setattr(ptrs[b], n, self.peer_fields[b][n].data_ptr())
        with torch.cuda.device(self.device):
            wsb = B.lib.cfd_workspace_bytes_sharded(nb, d, loc, C.byref(p))
            self.workspace = torch.empty((wsb + 7) // 8, dtype=torch.float64, device=self.device)
            h = C.c_void_p()
            rc = B.lib.cfd_create_blocks_sharded(C.byref(h), nb, d, ptrs, loc, len(self.faces), fa, C.byref(p),
                                                 self.workspace.data_ptr(), wsb, C.c_void_p(self.stream.cuda_stream))
        if rc != 0:
            raise B.CfdError(rc, B.lib.cfd_last_error(None).decode())
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            with self.torch.cuda.device(self.device):
                self.B.lib.cfd_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc):
        if rc != 0:
            raise self.B.CfdError(rc, self.B.lib.cfd_last_error(self.h).decode())

    def _call(self, fn, *args):
        """A library call that enqueues work: made with THIS context's device current (its stream and buffers belong to
        self.device; the process-wide current device may be another one, e.g. with several contexts in one process)."""
        with self.torch.cuda.device(self.device):
            self._chk(fn(self.h, *args))

    def _barrier(self):
        if self.comm is not None:
            self.comm.stream_barrier(self.stream)

    # ---- harness helpers ----
    def buffer_roles(self):
        r = (C.c_int * 3)()
        self._chk(self.B.lib.cfd_buffer_roles(self.h, r))
        return tuple(r[:])

    def field(self, b, name):
        if name in ("q", "qn", "r"):
            name = ("q", "qn", "r")[self.buffer_roles()[("q", "qn", "r").index(name)]]
        return self.fields[b][name]

    def interior(self, b, name):
        return self.field(b, name)[:, NG:-NG, NG:-NG, NG:-NG]

    def load_local(self, case):
        """Interior coordinates and state of the local blocks (step 1 of load_case; no communication)."""
        t = self.torch
        for b in self.local:
            self.interior(b, "xyz").copy_(t.from_numpy(np.ascontiguousarray(case.xyz[b])))
            self.interior(b, "q").copy_(t.from_numpy(np.ascontiguousarray(case.q0[b])))

    def finish_load(self, phase):
        """Steps 2..4 of load_case; between them every rank must have reached the same point (single-process tests call
        the phases of all their contexts in turn; `load_case` does it with the communicator)."""
        lib = self.B.lib
        if phase == 0:
            self._call(lib.cfd_compute_metrics)     # pulls the peers' xyz interiors
        elif phase == 1:
            self._call(lib.cfd_exchange_interfaces)  # pulls the peers' q interiors
        else:
            self._call(lib.cfd_apply_bc)

    def load_case(self, case):
        self.load_local(case)
        for phase in range(3):
            self._barrier()
            self.finish_load(phase)
        self._barrier()

    # ---- the sharded stage ----
    def stage_local(self, stage, dt, want_res=False):
        res = (C.c_double * 5)()
        self._call(self.B.lib.cfd_stage_fused_local, int(stage), float(dt), res if want_res else None)
        return np.array(res[:]) if want_res else None

    def exchange(self):
        self._call(self.B.lib.cfd_exchange_interfaces)

    def apply_bc(self):
        self._call(self.B.lib.cfd_apply_bc)

    def stage(self, stage, dt, want_res=False):
        """cfd_stage_fused over all ranks: local sweeps + RK, collective, P2P ghost fill, BCs; the stage-1 residual
        (sum of R_m^2 over ALL blocks) is all-reduced."""
        res = self.stage_local(stage, dt, want_res and stage == 1)
        self._barrier()
        self.exchange()
        if self.has_bc:
            self._barrier()
            self.apply_bc()
        if res is not None and self.comm is not None:
            res = self.comm.allreduce(res, "sum", self.stream)
        return res

    def step(self, dt, want_res=False):
        res = None
        for s in (1, 2, 3):
            r = self.stage(s, dt, want_res)
            if s == 1:
                res = r
        return res

    def step_host(self, q_in, q_out, dt):
        """End to end with HOST buffers: {block: pinned host tensor (5, nk, nj, ni)} for the local blocks in, one RK3 step,
        the same out (may alias); the copies ride on the compute stream, the call returns after a synchronise."""
        t = self.torch
        with t.cuda.stream(self.stream):
            for b in self.local:
                self.interior(b, "q").copy_(q_in[b], non_blocking=True)
        self._barrier()
        self.exchange()
        if self.has_bc:
            self._barrier()
            self.apply_bc()
        self.step(dt)
        with t.cuda.stream(self.stream):
            for b in self.local:
                q_out[b].copy_(self.interior(b, "q"), non_blocking=True)
        self.stream.synchronize()

    def cfl_dt(self, cfl):
        """min over the ranks of the local cfd_cfl_dt."""
        dt = C.c_double()
        self._call(self.B.lib.cfd_cfl_dt, float(cfl), C.byref(dt), None)
        if self.comm is None:
            return dt.value
        return float(self.comm.allreduce([dt.value], "min", self.stream)[0])

    @property
    def launch_count(self):
        return int(self.B.lib.cfd_launch_count(self.h))
