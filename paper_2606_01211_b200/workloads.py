"""The five synthetic workloads of BASELINE.json (`configs`) as plain data.

Holds parameters and seeded *generic* random-input helpers only -- none of the
method's arithmetic (no AES, no sampling rules, no modular products): the CUDA
path and the oracle each implement those independently.  Both tests/ and bench.py
read the table from here.

The paper uses no dataset: its workloads are parameter sets and iteration counts
(Table 1); C1-C3 span Table 2's n range, C4 is
"many concurrent key exchanges", C5 the n=32768 runs.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Workload:
    name: str
    n: int
    m: int
    k: int
    q: int
    eta: int
    batch: int
    seed: int
    note: str = ""

    @property
    def a_bytes(self) -> int:
        return 2 * self.m * self.n

    def ops_keygen(self) -> int:
        """modular ops (1 mul + 1 add per A element), SURVEY 8(c) S18"""
        return 2 * self.m * self.n * self.batch

    def ops_encaps(self) -> int:
        return (2 * self.m * self.n * self.k + 2 * self.m * self.k) * self.batch

    def ops_decaps(self) -> int:
        return 2 * self.n * self.k * self.batch


C1 = Workload("C1", 256, 512, 256, 65536, 4, 1, 1, "tiny single KEM")
C2 = Workload("C2", 1024, 2048, 256, 65536, 4, 1, 2, "small KEM")
C3 = Workload("C3", 4096, 8192, 256, 65521, 8, 1, 3, "prime modulus, Barrett path")
C4 = Workload("C4", 8192, 16384, 256, 65536, 4, 32, 4, "32 instances sharing one stored A")
C5 = Workload("C5", 32768, 65536, 256, 65536, 4, 1, 5, "A = 4 GiB, stored and regenerated")

CONFIGS = {w.name: w for w in (C1, C2, C3, C4, C5)}

# object tags of the seeded streams -- labels, not arithmetic
TAG_A, TAG_S, TAG_E, TAG_R, TAG_MU = 1, 2, 3, 4, 5
TAG_RG, TAG_E1, TAG_E2 = 6, 7, 8                      # N2: Gaussian r, e1 and centred-uniform e2 (paper's own PKE)

# Table 1 of the paper, the rows whose modulus fits uint16: (n, q, sigma, k of e2); eta = 3 for s
PAPER_TABLE1 = [(512, 3329, 2.3, 3), (1024, 12289, 2.3, 3), (2048, 12289, 2.3, 3), (4096, 12289, 1.7, 3)]


def shard_instances(batch: int, rank: int, world_size: int) -> range:
    """Instance ids owned by `rank` when `batch` independent instances are split
    over `world_size` processes (contiguous, remainder to the low ranks).  The KEM
    instances share nothing but the public matrix A (regenerable from its seed on
    every rank), so this is the whole multi-GPU story: no data-path collective."""
    if world_size <= 0 or not (0 <= rank < world_size):
        raise ValueError("bad rank/world_size")
    base, rem = divmod(batch, world_size)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))


# ---- generic seeded inputs for unit-level parity tests (not drawn by the method) ----

def random_u16(shape, q: int, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return rng.integers(0, q, size=shape, dtype=np.uint32).astype(np.uint16)


def random_bytes(n: int, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return rng.integers(0, 256, size=n, dtype=np.uint16).astype(np.uint8)
