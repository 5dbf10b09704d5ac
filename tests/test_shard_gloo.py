"""N > 1 path on CPU (gloo, world_size 2): the path shards by Dirichlet blocks with no data-path collective
("these solves can be performed independently on each node", eqs. 3-4).
Each rank extracts its own block, solves on it alone (here with the oracle standing in for the per-rank
dwf context -- the sharding host logic is what is under test), and only the final gather exchanges data.
The assembled solution must equal the whole-lattice solve of the cut operator."""
import os
import socket

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2203_17119_b200 import inputs, shard

DIMS, LS, CUT = (4, 4, 4, 8), 4, (0, 0, 0, 4)
PAR = dict(M5=1.8, mf=0.05, b5=1.5, c5=0.5)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    # each rank's oracle gets its share of the cores (set before libgomp loads): two ranks with all cores each spin against
    # one another and the test takes a minute instead of seconds
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      OMP_NUM_THREADS=str(max(1, (os.cpu_count() or 2) // world)), OMP_WAIT_POLICY="passive")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle.dwf_oracle import Oracle, solve_redblack
        U = inputs.gauge_weak(DIMS, 0.4, 11)
        eta = inputs.source_full(DIMS, LS, 12)
        bdims, bcut = shard.block_context_args(DIMS, CUT)
        local = {}
        for blk in shard.blocks_of_rank(DIMS, CUT, rank, world):
            Ub = shard.extract_block(U, DIMS, CUT, blk)
            eb = shard.extract_block(eta, DIMS, CUT, blk)
            orc = Oracle(bdims, LS, antiperiodic_t=shard.needs_antiperiodic_t(DIMS, CUT), cut=bcut, **PAR).set_gauge(Ub)
            psi_b, info = solve_redblack(orc, eb, 1e-11, 4000)
            assert info["converged"]
            local[blk] = psi_b
        psi = shard.gather_blocks(local, DIMS, CUT, (LS, 4, 3), np.complex128, dist)
        tmax = shard.max_over_ranks(10.0 + rank, dist)
        np.save(os.path.join(out_dir, f"psi_{rank}.npy"), psi)
        np.save(os.path.join(out_dir, f"tmax_{rank}.npy"), np.array([tmax, len(local)]))
    finally:
        dist.destroy_process_group()


def test_blocks_enumeration_and_roundtrip():
    assert shard.block_extents(DIMS, CUT) == (4, 4, 4, 4)
    assert shard.block_grid(DIMS, CUT) == (1, 1, 1, 2)
    assert shard.blocks(DIMS, CUT) == [(0, 0, 0, 0), (0, 0, 0, 1)]
    assert shard.blocks((8, 4, 4, 8), (4, 0, 0, 4)) == [(0, 0, 0, 0), (1, 0, 0, 0), (0, 0, 0, 1), (1, 0, 0, 1)]
    assert shard.blocks_of_rank((8, 4, 4, 8), (4, 0, 0, 4), 1, 2) == [(1, 0, 0, 0), (1, 0, 0, 1)]
    assert shard.block_context_args((8, 4, 4, 8), (4, 0, 0, 0)) == ((4, 4, 4, 8), (4, 0, 0, 0))
    with pytest.raises(ValueError):
        shard.block_extents((6, 4, 4, 4), (3, 0, 0, 0))      # odd block extent breaks the parity
    f = inputs.source_full(DIMS, 2, 1)
    g = np.zeros_like(f)
    for b in shard.blocks(DIMS, CUT):
        shard.insert_block(g, shard.extract_block(f, DIMS, CUT, b), DIMS, CUT, b)
    assert np.array_equal(f, g)
    # a block keeps the lattice's site parity: its even sites are the lattice's even sites
    pm = inputs.parity_mask(DIMS)
    pb = shard.extract_block(pm, DIMS, CUT, (0, 0, 0, 1))
    assert np.array_equal(pb, inputs.parity_mask(shard.block_extents(DIMS, CUT)))
    assert shard.max_over_ranks(3.5) == 3.5


def test_two_ranks_solve_their_blocks_independently(tmp_path, oracle_built):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    psi0, psi1 = np.load(tmp_path / "psi_0.npy"), np.load(tmp_path / "psi_1.npy")
    assert np.array_equal(psi0, psi1)                           # every rank holds the gathered field
    for r in (0, 1):
        tmax, nblk = np.load(tmp_path / f"tmax_{r}.npy")
        assert tmax == 11.0 and nblk == 1                       # max over ranks; one block each
    # whole-lattice solve of the cut operator D_Omega (+) D_Omegabar
    from oracle.dwf_oracle import Oracle, solve_redblack
    U = inputs.gauge_weak(DIMS, 0.4, 11)
    eta = inputs.source_full(DIMS, LS, 12)
    orc = Oracle(DIMS, LS, antiperiodic_t=True, cut=CUT, **PAR).set_gauge(U)
    want, info = solve_redblack(orc, eta, 1e-11, 4000)
    assert info["converged"]
    assert np.linalg.norm((psi0 - want).ravel()) / np.linalg.norm(want.ravel()) < 1e-8
    # and the assembled field solves the cut system: |eta - M_cut psi| small
    assert np.sqrt(orc.norm2(eta - orc.M(psi0)) / orc.norm2(eta)) < 1e-8
