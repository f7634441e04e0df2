"""World-size-2 gloo test of the N>1 host logic: states sharded across ranks, tensors replicated, no
collective on the data path, result assembled by all-gather; distribution sharded over an output-bit prefix.  The compute
on each rank is the CPU oracle (this is a `-m "not gpu"` test: it checks the sharding, not the kernels)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import reconstruct as R
from tqc_inputs import configs, random_states, random_tensors

# the package needs libtqc.so; sharding.py itself is plain Python
from paper_2502_03445_b200.sharding import shard_prefixes, shard_states


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    net = configs.random_network(m=4, K=5, seed=3, o_lo=1, o_hi=3)
    T = random_tensors(net, 5)
    B = 257                                                    # ragged split
    bits = random_states(net.n_qubits, B, 9)
    lo, hi = shard_states(B, rank, world)
    mine = torch.from_numpy(R.direct_sum(net, T, bits[lo:hi]))
    sizes = [shard_states(B, r, world) for r in range(world)]
    parts = [torch.zeros(b - a, dtype=torch.float64) for a, b in sizes]
    dist.all_gather(parts, mine) if len({b - a for a, b in sizes}) == 1 else _gather_ragged(parts, mine, rank, world)
    states_full = torch.cat(parts).numpy()
    # distribution: prefix chunks
    pb, vals = shard_prefixes(net.n_qubits, rank, world)
    allbits = R.full_distribution_bits(net.n_qubits)
    chunk = 1 << (net.n_qubits - pb)
    local = {v: R.direct_sum(net, T, allbits[v * chunk:(v + 1) * chunk]) for v in vals}
    gathered = [None] * world
    dist.all_gather_object(gathered, local)
    if rank == 0:
        full = np.zeros(1 << net.n_qubits)
        for d in gathered:
            for v, arr in d.items():
                full[v * chunk:(v + 1) * chunk] = arr
        q.put((states_full, full))
    dist.barrier()
    dist.destroy_process_group()


def _gather_ragged(parts, mine, rank, world):
    for r in range(world):
        buf = mine.clone() if r == rank else parts[r]
        dist.broadcast(buf, src=r)
        parts[r].copy_(buf)


def test_two_ranks_shard_states_and_prefixes():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, PORT, q)) for r in range(world)]
    for p in procs:
        p.start()
    states_full, dist_full = q.get()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    net = configs.random_network(m=4, K=5, seed=3, o_lo=1, o_hi=3)
    T = random_tensors(net, 5)
    bits = random_states(net.n_qubits, 257, 9)
    np.testing.assert_allclose(states_full, R.direct_sum(net, T, bits), rtol=0, atol=0)
    np.testing.assert_allclose(dist_full, R.direct_sum(net, T, R.full_distribution_bits(net.n_qubits)), rtol=0, atol=0)


PORT = _free_port()


def test_shard_arithmetic():
    for n, w in [(0, 2), (1, 2), (257, 2), (1000, 8), (7, 8)]:
        cover = []
        for r in range(w):
            lo, hi = shard_states(n, r, w)
            assert 0 <= lo <= hi <= n
            cover += list(range(lo, hi))
        assert cover == list(range(n))
    for w in (1, 2, 3, 4, 8):
        seen = []
        for r in range(w):
            pb, vals = shard_prefixes(10, r, w)
            seen += vals
        assert sorted(seen) == list(range(1 << pb))
