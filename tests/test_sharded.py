"""Row f4 (section 4.4, Alg. 4): a grid sharded over several GPUs.
This environment has ONE GPU, so the multi-rank path is covered in two halves:

* `-m gpu`: the ranks of a sharded grid are emulated in one process on one device (their launches are
  enqueued one after the other on one stream, nothing waits on anything): the kernels' sharded code --
  own-block lists, ghost writes into the buffers of other ranks, fills that read other ranks' blocks,
  the min-reduction of the time step -- must give the state of the unsharded grid;
* `-m "not gpu"`: the partition tables, the refusal of unsupported combinations, and, with two gloo
  processes, that an all-reduce(MIN) of the int64 bit patterns is the minimum of the positive doubles.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ----------------------------------------------------------------------------- CPU
def test_partition_is_contiguous_and_balanced():
    import paper_2501_06717_b200 as batl
    cfg = wl.brio_wu_amr()
    nB = batl.Grid(cfg).n_blocks
    for world in (1, 2, 3, 8):
        firsts = []
        for rank in range(world):
            g = batl.Grid(cfg).set_partition(world, rank)
            firsts.append(g.partition())
        assert all(np.array_equal(f, firsts[0]) for f in firsts)
        f = firsts[0]
        assert f[0] == 0 and f[-1] == nB and np.all(np.diff(f) >= nB // world) and np.all(np.diff(f) <= nB // world + 1)


def test_unsupported_combinations_are_refused():
    import paper_2501_06717_b200 as batl
    for extra in (dict(prolong_order=2), dict(flux_correction=1)):
        g = batl.Grid(dict(wl.fast_wave((2, 2, 2)), **extra))
        with pytest.raises(batl.BatlError):
            g.set_partition(2, 0)
        g.set_partition(1, 0)                          # one rank is the unsharded grid
    with pytest.raises(batl.BatlError):
        batl.Grid(wl.alfven()).set_partition(2, 2)


def test_bit_pattern_order_of_positive_doubles():
    from paper_2501_06717_b200.dist import positive_double_bits_min
    rng = np.random.default_rng(5)
    x = np.concatenate([rng.uniform(1e-300, 1e300, 1000), 10.0 ** rng.uniform(-300, 300, 1000), [np.inf, 5e-324]])
    assert positive_double_bits_min(x) == x.min()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = np.array([0.0125 * (rank + 1) + 1e-9 * rank, np.inf if rank else 3.0e-7])   # two "dt_next" slots
    t = torch.from_numpy(mine.view(np.int64).copy())
    dist.all_reduce(t, op=dist.ReduceOp.MIN)
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, t.numpy().view(np.float64).tolist()))


def test_allreduce_min_of_bit_patterns_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0] == res[1] == [0.0125, 3.0e-7]


# ----------------------------------------------------------------------------- GPU
SHARD_CASES = {
    "uniform_4x2x2": (lambda: wl.random_uniform((4, 2, 2)), 6),
    "fast_wave_15_amr": (lambda: wl.fast_wave((2, 2, 2), amplitude_scale=5.0), 6),
    "brio_wu_amr_352": (lambda: wl.brio_wu_amr(), 5),
    "uniform_local_dt": (lambda: wl.random_uniform((3, 2, 2), dt_mode=wl.DT_LOCAL), 4),
    # the paper's operational time stepping (L391-397): one stage, first order; the buffers trade roles every step
    "fast_wave_15_one_stage": (lambda: dict(wl.fast_wave((2, 2, 2), amplitude_scale=5.0), n_stage=1, n_order=1, cfl=0.4), 5),
    "uniform_one_stage_2nd_order": (lambda: dict(wl.random_uniform((4, 2, 2)), n_stage=1, cfl=0.4), 5),
}


@pytest.mark.gpu
@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("name", sorted(SHARD_CASES))
def test_emulated_ranks_reproduce_the_unsharded_grid(name, world):
    import paper_2501_06717_b200 as batl
    from paper_2501_06717_b200 import dist as bd
    make, n = SHARD_CASES[name]
    cfg = make()
    ref = batl.Grid(cfg).bind()
    U0 = wl.initial_conserved(cfg, ref.blocks())
    ref.set_state(U0)
    _, t_ref, dt_ref = ref.step(n)
    want = ref.get_state()
    ref.close()

    grids = bd.make_local_ranks(cfg, world)
    for g in grids:
        g.set_state(U0)
    st = bd.ShardedStepper(grids, bd.LocalTransport())
    st.step(n)
    got = bd.gather_state(grids)
    scal = [g.step(0) for g in grids]                    # (warn, t, dt_last) of every rank
    for g in grids:
        g.close()
    # same arithmetic per block: the states agree to the last bit (a different kernel instantiation takes the
    # blocks from a list; should a compiler ever contract it differently, round-off is the bar)
    err = np.abs(got - want).max() / np.abs(want).max()
    assert err <= 1e-14, err
    assert np.isfinite(got).all()
    for _, t, dt in scal:
        assert t == scal[0][1] and dt == scal[0][2]
        assert abs(t - t_ref) <= 1e-14 * max(abs(t_ref), 1e-300) and abs(dt - dt_ref) <= 1e-14 * max(abs(dt_ref), 1e-300)


@pytest.mark.gpu
def test_sharded_grid_against_the_oracle():
    # the sharded path against the CPU oracle directly (not only against the unsharded kernels): config 3's grid
    # and physics (two levels, float x boundaries), three ranks, the north_star's 10 steps and 1e-11
    import oracle
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from util import rel_err_O9
    from paper_2501_06717_b200 import dist as bd
    cfg = wl.brio_wu_amr()
    o = oracle.Oracle(cfg)
    o.set_primitive(wl.initial_primitive(cfg, o.blocks()))
    U0 = o.get_state()
    wo, to, dto = o.step(10)
    grids = bd.make_local_ranks(cfg, 3)
    for g in grids:
        g.set_state(U0)
    bd.ShardedStepper(grids, bd.LocalTransport()).step(10)
    got = bd.gather_state(grids)
    scal = [g.step(0) for g in grids]
    for g in grids:
        g.close()
    assert rel_err_O9(got, o.get_state()) <= 1e-11
    for w, t, dt in scal:
        assert abs(t - to) <= 1e-12 * abs(to) and abs(dt - dto) <= 1e-12 * abs(dto)


@pytest.mark.gpu
def test_sharded_config5_two_ranks():
    # configs[4]: four levels, B0 dipole, body blocks (general kernel on the own body blocks), local dt
    import paper_2501_06717_b200 as batl
    from paper_2501_06717_b200 import dist as bd
    cfg = wl.magnetosphere()
    ref = batl.Grid(cfg).bind()
    U0 = wl.initial_conserved(cfg, ref.blocks())
    ref.set_state(U0)
    ref.step(2)
    want = ref.get_state()
    ref.close()
    grids = bd.make_local_ranks(cfg, 2)
    for g in grids:
        g.set_state(U0)
    bd.ShardedStepper(grids, bd.LocalTransport()).step(2)
    got = bd.gather_state(grids)
    for g in grids:
        g.close()
    scale = np.abs(want).reshape(want.shape[0], 8, -1).max(axis=(0, 2))
    assert (np.abs(got - want).reshape(want.shape[0], 8, -1).max(axis=(0, 2)) / scale).max() <= 1e-11


# ------------------------------------------------- two PROCESSES on one GPU: the IPC mapping for real
def _ipc_worker(rank, world, port, name, n_steps, out):
    """One rank of a sharded grid in its own process.  Both processes use cuda:0 (time-sliced; no kernel
    waits on another process: the ranks synchronise on the host through gloo), so the CUDA IPC mapping of
    the peers' buffers, the cross-process ghost writes and the all-reduce of the dt bit pattern run as on
    several GPUs -- only NCCL and NVLink are missing."""
    try:
        import torch
        import torch.distributed as dist
        sys.path.insert(0, ROOT)
        import paper_2501_06717_b200 as batl
        from paper_2501_06717_b200 import dist as bd
        os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        dist.init_process_group("gloo", rank=rank, world_size=world)
        cfg = SHARD_CASES[name][0]()
        g = bd.make_rank(cfg, "cuda:0")
        U0 = wl.initial_conserved(cfg, g.blocks())
        g.set_state(U0)
        torch.cuda.synchronize()
        dist.barrier()
        bd.ShardedStepper([g], bd.NcclTransport()).step(n_steps)
        torch.cuda.synchronize()
        first = g.partition()
        mine = g.get_state()[first[rank]:first[rank + 1]]
        _, t, dt = g.step(0)
        dist.barrier()                                   # nobody unmaps while a peer may still write
        g.close()
        dist.destroy_process_group()
        out.put((rank, mine, t, dt, None))
    except Exception as e:                               # pragma: no cover
        out.put((rank, None, 0.0, 0.0, repr(e)))


@pytest.mark.gpu
@pytest.mark.parametrize("name", ["fast_wave_15_amr", "uniform_4x2x2"])
def test_two_processes_one_gpu_ipc_mapping(name):
    import paper_2501_06717_b200 as batl
    n = 4
    cfg = SHARD_CASES[name][0]()
    ref = batl.Grid(cfg).bind()
    ref.set_state(wl.initial_conserved(cfg, ref.blocks()))
    _, t_ref, dt_ref = ref.step(n)
    want = ref.get_state()
    ref.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_ipc_worker, args=(r, 2, port, name, n, q)) for r in range(2)]
    for p in procs:
        p.start()
    try:
        res = [q.get(timeout=240) for _ in procs]
    finally:
        for p in procs:
            p.join(timeout=60)
            if p.is_alive():
                p.kill()
    res.sort(key=lambda r: r[0])
    for r in res:
        assert r[4] is None, r[4]
    got = np.concatenate([r[1] for r in res], axis=0)
    assert got.shape == want.shape
    assert np.abs(got - want).max() <= 1e-14 * np.abs(want).max()
    for r in res:
        assert abs(r[2] - t_ref) <= 1e-14 * abs(t_ref) and abs(r[3] - dt_ref) <= 1e-14 * abs(dt_ref)
