"""World-size-2 gloo test of the sink-sharding host logic (paper_2011_14984_b200/sharding.py).
The compute callables are the oracle's sweeps on CPU tensors (the CUDA kernels cannot run here);
what is tested is the partition of the sinks, the all-gather of a between the sweeps and the
assembly -- the result must be bit-identical to the unsharded call."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import frost_inputs as fi


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, n, out_dir):
    import oracle
    from paper_2011_14984_b200 import sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    oracle.set_num_threads(2)
    pos, vel, mass = fi.plummer(n, 5)
    acc = torch.zeros((3, n), dtype=torch.float64); grad = torch.zeros((3, n), dtype=torch.float64)

    def acc_fn(sink_idx, a):
        oracle.forces(pos, mass, sink_idx=sink_idx.numpy(), flags=oracle.ACC, acc=a.numpy(),
                      grad=grad.numpy())

    def grad_fn(sink_idx, a, g):
        oracle.forces(pos, mass, sink_idx=sink_idx.numpy(), flags=oracle.GRAD, acc=a.numpy(),
                      grad=g.numpy())

    lo, hi = sharding.sharded_acc_grad(n, rank, world, acc_fn, grad_fn, acc, grad)
    g_full = sharding.all_gather_planes(grad[:, lo:hi].contiguous(), n, rank, world,
                                        torch.zeros_like(grad))
    np.save(os.path.join(out_dir, f"acc{rank}.npy"), acc.numpy())
    np.save(os.path.join(out_dir, f"grad{rank}.npy"), g_full.numpy())
    dist.destroy_process_group()


def test_shard_ranges_cover_and_balance():
    from paper_2011_14984_b200.sharding import shard_range
    for n in (0, 1, 7, 1000, 1 << 20):
        for w in (1, 2, 3, 8):
            r = [shard_range(n, k, w) for k in range(w)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(w - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1


def test_two_rank_sharded_pass_matches_unsharded(tmp_path, oracle):
    n, world = 301, 2
    port = _free_port()
    mp.spawn(_worker, args=(world, port, n, str(tmp_path)), nprocs=world, join=True)
    pos, vel, mass = fi.plummer(n, 5)
    a_ref, g_ref = oracle.forces(pos, mass)
    for r in range(world):
        assert np.array_equal(np.load(tmp_path / f"acc{r}.npy"), a_ref)
        assert np.array_equal(np.load(tmp_path / f"grad{r}.npy"), g_ref)


def _pair_worker(rank, world, port, n, out_dir):
    import oracle
    from paper_2011_14984_b200 import sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    oracle.set_num_threads(2)
    pos, vel, mass = fi.plummer(n, 5)
    mine = np.arange(rank, n, world).astype(np.int32)      # stands in for this rank's tile pairs
    acc = torch.zeros((3, n), dtype=torch.float64); grad = torch.zeros((3, n), dtype=torch.float64)

    def acc_fn(a):
        a.zero_()
        oracle.forces(pos, mass, sink_idx=mine, flags=oracle.ACC, acc=a.numpy(), grad=grad.numpy())

    def grad_fn(a, g):
        g.zero_()
        oracle.forces(pos, mass, sink_idx=mine, flags=oracle.GRAD, acc=a.numpy().copy(), grad=g.numpy())

    sharding.pair_sharded_acc_grad(world, acc_fn, grad_fn, acc, grad)
    np.save(os.path.join(out_dir, f"pacc{rank}.npy"), acc.numpy())
    np.save(os.path.join(out_dir, f"pgrad{rank}.npy"), grad.numpy())
    dist.destroy_process_group()


def test_two_rank_pair_sharded_pass_matches_unsharded(tmp_path, oracle):
    """Host logic of the pair-sharded pass: partial sums, all-reduce of a, gradient on the complete
    a, all-reduce of g (the partial sums here have disjoint support, so the result is exact)."""
    n, world = 257, 2
    port = _free_port()
    mp.spawn(_pair_worker, args=(world, port, n, str(tmp_path)), nprocs=world, join=True)
    pos, vel, mass = fi.plummer(n, 5)
    a_ref, g_ref = oracle.forces(pos, mass)
    for r in range(world):
        assert np.array_equal(np.load(tmp_path / f"pacc{r}.npy"), a_ref)
        assert np.array_equal(np.load(tmp_path / f"pgrad{r}.npy"), g_ref)
