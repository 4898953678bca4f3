"""Helpers for the -m gpu parity tests: device buffers as torch tensors, oracle
objects as numpy arrays.  No arithmetic of the method lives here."""
from __future__ import annotations

import numpy as np
import torch

import oracle as O
from paper_2606_01211_b200 import binding as B
from paper_2606_01211_b200 import workloads as W


def dev(a: np.ndarray) -> torch.Tensor:
    """numpy (uint8 / uint16) -> device tensor with the same bytes"""
    a = np.ascontiguousarray(a)
    if a.dtype == np.uint16:
        return torch.from_numpy(a.view(np.int16)).cuda()
    assert a.dtype == np.uint8
    return torch.from_numpy(a).cuda()


def dev_empty_u16(*shape) -> torch.Tensor:
    return torch.empty(*shape, dtype=torch.int16, device="cuda")


def dev_empty_u8(*shape) -> torch.Tensor:
    return torch.empty(*shape, dtype=torch.uint8, device="cuda")


def host_u16(t: torch.Tensor) -> np.ndarray:
    torch.cuda.synchronize()
    return t.cpu().numpy().view(np.uint16)


def host_u8(t: torch.Tensor) -> np.ndarray:
    torch.cuda.synchronize()
    return t.cpu().numpy()


def unpack_bits(packed, n) -> np.ndarray:
    return np.unpackbits(np.asarray(packed, dtype=np.uint8), bitorder="little")[:n]


class OracleInstance:
    """All seeded objects of one KEM instance of a workload, drawn by the ORACLE."""

    def __init__(self, w: W.Workload, inst: int, n=None, m=None, with_A=True):
        self.w, self.inst = w, inst
        self.n, self.m = n or w.n, m or w.m
        self.A = (O.sample_uniform(0, self.m * self.n, w.seed, O.TAG_A, 0, w.q).reshape(self.m, self.n)
                  if with_A else None)
        self.s = O.sample_uniform(0, self.n, w.seed, O.TAG_S, inst, w.q)
        self.e = O.sample_cbd(0, self.m, w.seed, O.TAG_E, inst, w.q, w.eta)
        self.Rbits = O.sample_bits(0, self.m * w.k, w.seed, O.TAG_R, inst)
        self.mubits = O.sample_bits(0, w.k, w.seed, O.TAG_MU, inst)


def make_ctx(w: W.Workload, n=None, m=None, k=None, q=None, max_batch=None) -> B.Context:
    return B.Context(n or w.n, m or w.m, k or w.k, q or w.q, w.eta, max_batch or w.batch)
