"""Driver of a grid sharded over the GPUs of one node (section 4.4,
Alg. 4): argument marshalling and the collectives between the parts of a step.  Every step of
the path itself runs in the kernels of libbatl (include/batl.h, "Sharding").

One process per GPU.  Every rank builds the same grid and owns a contiguous Morton segment of its
blocks.  There are no message buffers and no packing: the ranks map one another's state buffers (CUDA
IPC; NVLink peer access) and the stage kernel writes the outer cell layers of its blocks straight into
the ghost slots of neighbours on other GPUs.  What is left between the parts of a step is

    a barrier after each stage            (all ghost writes of a stage have landed before anyone reads)
    an all-reduce(min) of the time step   (8 bytes; dt_mode global; doubles as the barrier of stage 2)

both enqueued on the grid's stream through ``torch.distributed`` (NCCL).  ``Transport`` abstracts these
two calls, so that the same step loop drives (a) real ranks and (b) several ranks emulated in ONE
process on ONE GPU (``LocalTransport``), which is how the kernels' sharded path is tested on a single
B200: the launches of the emulated ranks are simply enqueued one after the other on one stream.

NOT measured on several GPUs: this environment has one.  What HAS run on it: ranks emulated in one
process, and two PROCESSES sharing the GPU with the IPC mapping below (torch.multiprocessing's own
mechanism, ``UntypedStorage._share_cuda_`` / ``_new_shared_cuda``) and gloo collectives
(tests/test_sharded.py); NCCL and NVLink themselves have not.
"""
from __future__ import annotations

import numpy as np

from . import Grid

PART_DT0, PART_TICK_START, PART_STAGE1, PART_FILL_B, PART_STAGE2, PART_FILL_A, PART_TICK_END = range(7)
DT_GLOBAL = 0


class Transport:
    """The two collectives of a sharded step, on the stream of the grid(s)."""

    def barrier(self, grids):
        raise NotImplementedError

    def allreduce_min_i64(self, grids, slots):
        """slots: one int64 device tensor (1 element) per local grid; every one ends up holding the minimum
        over all ranks."""
        raise NotImplementedError


class LocalTransport(Transport):
    """All ranks live in this process and share one stream: launches are already ordered, the minimum is
    taken on the device."""

    def barrier(self, grids):
        pass

    def allreduce_min_i64(self, grids, slots):
        import torch
        m = slots[0].clone()
        for s in slots[1:]:
            torch.minimum(m, s, out=m)
        for s in slots:
            s.copy_(m)


class TorchDistTransport(Transport):
    """One rank per process over ``torch.distributed``: NCCL between the GPUs of a node; gloo also works
    (it stages CUDA tensors through the host and blocks until done), which is how two processes sharing
    ONE GPU are tested.  The collectives are issued with the grid's stream current, so they are ordered
    after the kernels enqueued before them and before those enqueued after."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group

    def barrier(self, grids):
        import torch
        g = grids[0]
        with torch.cuda.stream(g.stream):
            flag = torch.zeros(1, dtype=torch.int32, device=g._bufs[2].device)
            self.dist.all_reduce(flag, group=self.group)

    def allreduce_min_i64(self, grids, slots):
        import torch
        with torch.cuda.stream(grids[0].stream):
            self.dist.all_reduce(slots[0], op=self.dist.ReduceOp.MIN, group=self.group)


NcclTransport = TorchDistTransport


def positive_double_bits_min(values):
    """The rule the all-reduce relies on, as host arithmetic (used by the CPU tests): for positive doubles
    the order of the int64 bit patterns is the order of the values."""
    bits = np.asarray(values, dtype=np.float64).view(np.int64)
    return np.int64(bits.min()).view(np.float64)


class ShardedStepper:
    """Drives `grids` (the local ranks: one for real multi-GPU runs, all of them in the single-process
    emulation) through whole steps."""

    def __init__(self, grids, transport: Transport):
        self.grids, self.tr = list(grids), transport
        self.global_dt = int(self.grids[0].cfg["dt_mode"]) == DT_GLOBAL
        self.two_stage = int(self.grids[0].cfg.get("n_stage", 2)) == 2
        self.started = False

    def _all(self, part):
        for g in self.grids:
            g.step_part(part)

    def _reduce_dt(self):
        if self.global_dt:
            self.tr.allreduce_min_i64(self.grids, [g.dt_next_slot() for g in self.grids])
        else:
            self.tr.barrier(self.grids)

    def step(self, n_steps=1):
        for _ in range(int(n_steps)):
            if not self.started:                 # dt of the first step from the initial state (Q-T2)
                self._all(PART_DT0)
                self._reduce_dt()
                self._all(PART_TICK_START)
                self.started = True
            self._all(PART_STAGE1)
            self.tr.barrier(self.grids)
            self._all(PART_FILL_B)
            if self.two_stage:
                self._all(PART_STAGE2)
                self.tr.barrier(self.grids)
                self._all(PART_FILL_A)
            self._reduce_dt()
            self._all(PART_TICK_END)


def make_local_ranks(cfg: dict, world: int, device="cuda:0", stream=None):
    """`world` ranks of one sharded grid in this process, on one device and one stream (emulation for
    tests on a single GPU): every rank's buffers are visible to every other as plain device pointers."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream(torch.device(device))
    grids = [Grid(cfg).set_partition(world, r).bind(device, st) for r in range(world)]
    ptrs = [g.state_pointers() for g in grids]
    for g in grids:
        g.bind_peers([p[0] for p in ptrs], [p[1] for p in ptrs])
    return grids


def make_rank(cfg: dict, device, stream=None, group=None):
    """This process's rank of a grid sharded over the ranks of `group` (default: the world): builds the
    grid, binds it, exchanges CUDA IPC handles of the state buffers and maps the peers'."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    g = Grid(cfg).set_partition(world, rank).bind(device, stream)
    A, B = g._bufs[0], g._bufs[1]
    mine = (A.untyped_storage()._share_cuda_(), B.untyped_storage()._share_cuda_())
    handles = [None] * world
    dist.all_gather_object(handles, mine, group=group)
    g._peer_storages = []                        # keep the mappings alive
    pa, pb = [], []
    for r, (ha, hb) in enumerate(handles):
        if r == rank:
            pa.append(A.data_ptr()); pb.append(B.data_ptr())
            continue
        sa = torch.UntypedStorage._new_shared_cuda(*ha)
        sb = torch.UntypedStorage._new_shared_cuda(*hb)
        g._peer_storages += [sa, sb]
        pa.append(sa.data_ptr())
        pb.append(sb.data_ptr())
    g.bind_peers(pa, pb)
    return g


def gather_state(grids):
    """The whole state [nB][8][8][8][8] assembled from the own segments of the local ranks."""
    first = grids[0].partition()
    out = None
    for g in grids:
        U = g.get_state()
        if out is None:
            out = np.zeros_like(U)
        lo, hi = first[g.rank], first[g.rank + 1]
        out[lo:hi] = U[lo:hi]
    return out
