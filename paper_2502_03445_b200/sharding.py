"""Multi-GPU sharding of the path: pure index arithmetic, no compute.

States mode: the batch is split into contiguous, nearly equal ranges, one per rank; tensors are
replicated; no collective on the data path (an optional all-gather assembles the result).
Distribution mode: rank r computes the chunk whose top `prefix_bits` qubits equal r
(tqc_contract_distribution's prefix arguments); world sizes that are not powers of two hand the
2^prefix_bits chunks out round-robin.
"""
from __future__ import annotations


def shard_states(n_states: int, rank: int, world: int):
    """[lo, hi) of the caller's batch that `rank` contracts; sizes differ by at most one."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, extra = divmod(n_states, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_prefixes(n_qubits: int, rank: int, world: int):
    """(prefix_bits, [prefix values]) of the distribution chunks `rank` computes."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    bits = 0
    while (1 << bits) < world and bits < n_qubits:
        bits += 1
    return bits, list(range(rank, 1 << bits, world))
