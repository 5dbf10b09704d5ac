"""The N > 1 path on the PRODUCT: one dwf context per Dirichlet block, built from
shard.block_context_args exactly as a rank would build it, each block solved on its own with no exchange
("these solves can be performed independently on each node"; eqs. 3-4), the blocks
gathered -- against ONE context holding the whole lattice with the cut and against the oracle.
One GPU runs the blocks one after the other; they never wait on one another."""
import numpy as np
import pytest

from paper_2203_17119_b200 import inputs, shard

pytestmark = pytest.mark.gpu

PAR = dict(M5=1.8, mf=0.01, b5=1.5, c5=0.5)
CASES = {
    # c2's geometry scaled down: cut in t into two blocks
    "t2": dict(dims=(8, 8, 8, 16), Ls=8, cut=(0, 0, 0, 8)),
    # a 2 x 2 checkerboard of blocks (cut in x and t), ragged tile shapes inside the blocks
    "xt4": dict(dims=(12, 4, 4, 8), Ls=4, cut=(6, 0, 0, 4)),
}


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def _solve_full(api, g, dims, eta, tol):
    import torch
    e, o = inputs.split_parity(eta, dims)
    nat = torch.cat([g.pack(e, api.F64, api.EVEN), g.pack(o, api.F64, api.ODD)])
    psi, info, st = g.solve(nat, tol, 20000, api.CG_F64)
    assert st == api.OK, info
    n = psi.numel() // 2
    return inputs.merge_parity(g.unpack(psi[:n], api.F64, api.EVEN), g.unpack(psi[n:], api.F64, api.ODD), dims), info


@pytest.mark.parametrize("name", list(CASES))
def test_blocks_solved_independently_equal_the_cut_lattice_solve(name, oracle_built):
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2203_17119_b200 import api
    from oracle.dwf_oracle import Oracle
    dims, Ls, cut = CASES[name]["dims"], CASES[name]["Ls"], CASES[name]["cut"]
    U = inputs.gauge_weak(dims, 0.35, 61)
    eta = inputs.source_full(dims, Ls, 62)
    tol = 1e-11
    bdims, bcut = shard.block_context_args(dims, cut)
    world = 2
    gathered = np.zeros_like(eta)
    owners = {}
    for rank in range(world):
        local = {}
        for blk in shard.blocks_of_rank(dims, cut, rank, world):
            g = api.Dwf(bdims, Ls, PAR["M5"], PAR["mf"], PAR["b5"], PAR["c5"], cut=bcut,
                        antiperiodic_t=int(shard.needs_antiperiodic_t(dims, cut)))
            g.set_gauge(shard.extract_block(U, dims, cut, blk))
            local[blk], _ = _solve_full(api, g, bdims, shard.extract_block(eta, dims, cut, blk), tol)
            g.close()
            owners[blk] = rank
        part = shard.gather_blocks(local, dims, cut, (Ls, 4, 3), np.complex128)
        gathered += part
    assert sorted(owners) == sorted(shard.blocks(dims, cut)) and set(owners.values()) == {0, 1}
    # one context for the whole lattice with the cut
    g = api.Dwf(dims, Ls, PAR["M5"], PAR["mf"], PAR["b5"], PAR["c5"], cut=cut)
    g.set_gauge(U)
    whole, _ = _solve_full(api, g, dims, eta, tol)
    g.close()
    assert rel(gathered, whole) < 1e-8
    # the oracle applies the cut operator to the gathered field
    orc = Oracle(dims, Ls, PAR["M5"], PAR["mf"], PAR["b5"], PAR["c5"], antiperiodic_t=True, cut=cut).set_gauge(U)
    assert np.sqrt(orc.norm2(eta - orc.M(gathered)) / orc.norm2(eta)) < 1e-8
