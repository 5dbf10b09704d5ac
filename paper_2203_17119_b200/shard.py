"""Sharding by Dirichlet blocks (host logic only; no operator arithmetic).

With cut links zeroed the operator is block diagonal, D_dirichlet = D_Omega (+) D_Omegabar
(eqs. 3-4), and "these solves can be performed independently on each node"
(PAPER.md:123).  So the path shards with NO data-path collective: each rank owns whole blocks, solves on
them with its own dwf context (dims = block extents, dirichlet_cut = block extents, so the wrap link of the
block is cut: open boundaries), and only the final gather of a global field is an exchange.

A block is the cuboid {x : b_mu*B_mu <= x_mu < (b_mu+1)*B_mu}.  Block extents must be even so that the
parity of a site is the same in the block's coordinates as in the lattice's.

Field layouts are the canonical ones of include/dwf.h: gauge U[t,z,y,x,mu,3,3], FULL psi[t,z,y,x,s,4,3].
"""
from __future__ import annotations

import itertools

import numpy as np


def block_extents(dims, cut):
    """Block length per direction (Lx,Ly,Lz,Lt order); a direction without a cut is one block."""
    ext = tuple(int(c) if c else int(d) for d, c in zip(dims, cut))
    for d, e in zip(dims, ext):
        if d % e or e % 2:
            raise ValueError(f"block extent {e} must be even and divide {d}")
    return ext


def block_grid(dims, cut):
    ext = block_extents(dims, cut)
    return tuple(d // e for d, e in zip(dims, ext))


def blocks(dims, cut):
    """All block coordinates (bx,by,bz,bt), x fastest."""
    nb = block_grid(dims, cut)
    return [tuple(reversed(c)) for c in itertools.product(*[range(n) for n in reversed(nb)])]


def blocks_of_rank(dims, cut, rank, world):
    """Round-robin ownership: block i belongs to rank i % world."""
    return [b for i, b in enumerate(blocks(dims, cut)) if i % world == rank]


def _slices(dims, cut, block):
    ext = block_extents(dims, cut)
    sl = [slice(b * e, (b + 1) * e) for b, e in zip(block, ext)]
    return tuple(reversed(sl))          # arrays are indexed [t,z,y,x,...]


def extract_block(field, dims, cut, block):
    """Sub-array of a [t,z,y,x,...] field (gauge or FULL spinor) on one block (a contiguous copy)."""
    return np.ascontiguousarray(field[_slices(dims, cut, block)])


def insert_block(field, sub, dims, cut, block):
    field[_slices(dims, cut, block)] = sub
    return field


def block_context_args(dims, cut):
    """(dims, dirichlet_cut) of the dwf context a rank creates for one block.

    In a cut direction the block's own wrap link must be cut too (open boundary): cut = extent.  In an
    uncut direction the block spans the lattice and keeps its periodic wrap: cut = 0."""
    ext = block_extents(dims, cut)
    return ext, tuple(e if c else 0 for e, c in zip(ext, cut))


def needs_antiperiodic_t(dims, cut):
    """The antiperiodic sign lives on the t wrap link; it only survives when t is not cut."""
    return not cut[3]


def max_over_ranks(value: float, dist=None) -> float:
    """bench.py's timing rule: the step time of a multi-rank run is the maximum over ranks."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_blocks(local: dict, dims, cut, shape_tail, dtype, dist=None):
    """Assemble a global [t,z,y,x,...] field on every rank from per-rank {block: sub-array} dicts.
    The only exchange of the sharded path (an all-gather of results, outside the solve)."""
    Lx, Ly, Lz, Lt = dims
    out = np.zeros((Lt, Lz, Ly, Lx) + tuple(shape_tail), dtype=dtype)
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        parts = [local]
    else:
        parts = [None] * dist.get_world_size()
        dist.all_gather_object(parts, local)
    for part in parts:
        for block, sub in part.items():
            insert_block(out, sub, dims, cut, block)
    return out
