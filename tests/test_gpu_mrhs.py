"""SURVEY 8f NEXT-3 through the C ABI: batched (multi right-hand side) Dhop, Mpc, Mpc^dag Mpc and CG ("four PV
local solves, and two non-local light quark solves").  The oracle has nothing new to compute: it applies the
single-system operator / CG to every right-hand side in turn, and each system of the batch is compared with it element by
element (operators) or by iteration count +-2 and oracle-recomputed true residual (CG).  Also: the batched result equals the
single-system GPU result bit for bit (same kernels, same order of operations per system)."""
import numpy as np
import pytest

from paper_2203_17119_b200 import inputs

pytestmark = pytest.mark.gpu

MOEB = dict(M5=1.8, mf=0.01, b5=1.5, c5=0.5)
SHAM = dict(M5=1.8, mf=0.1, b5=1.0, c5=0.0)
CASES = {
    # fused TMA path (4^4 tiles), Ls with an unrolled column kernel, cut lattice
    "fused_cut": dict(dims=(8, 8, 4, 8), Ls=8, par=MOEB, eps=0.4, cut=(0, 0, 0, 4), nrhs=3),
    "fused_shamir": dict(dims=(4, 4, 8, 8), Ls=12, par=SHAM, eps=0.3, nrhs=2),
    # ragged tiles -> cp.async tile kernel and the unfused column kernels, generic Ls
    "ragged_ls5": dict(dims=(4, 6, 4, 8), Ls=5, par=MOEB, eps=0.5, nrhs=4),
    # 18-real links (unfused), six systems
    "g18": dict(dims=(4, 4, 4, 8), Ls=4, par=MOEB, eps=0.6, compress12=0, nrhs=6),
    # the largest batch the ABI accepts, on the fused path
    "max16": dict(dims=(4, 4, 4, 4), Ls=4, par=SHAM, eps=0.3, nrhs=16),
}


def rel(a, b):
    a = np.asarray(a, dtype=np.complex128)
    b = np.asarray(b, dtype=np.complex128)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


@pytest.fixture(scope="module", params=list(CASES))
def case(request, oracle_built):
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2203_17119_b200 import api
    from oracle.dwf_oracle import Oracle
    kw = dict(CASES[request.param])
    dims, Ls, par, nrhs = kw["dims"], kw["Ls"], kw["par"], kw["nrhs"]
    cut = kw.get("cut", (0, 0, 0, 0))
    U = inputs.gauge_weak(dims, kw["eps"], 31)
    g = api.Dwf(dims, Ls, par["M5"], par["mf"], par["b5"], par["c5"], cut=cut, compress12=kw.get("compress12", 1))
    g.set_gauge(U)
    orc = Oracle(dims, Ls, par["M5"], par["mf"], par["b5"], par["c5"], antiperiodic_t=True, cut=cut).set_gauge(U)
    U32 = U.astype(np.complex64).astype(np.complex128)
    orc32 = Oracle(dims, Ls, par["M5"], par["mf"], par["b5"], par["c5"], antiperiodic_t=True, cut=cut).set_gauge(U32)
    # sources of different size, so that the systems converge at different iterations; one of them is a multiple of another
    srcs = [inputs.source_half(dims, Ls, 500 + j, parity=1) * (10.0 ** (-j)) for j in range(nrhs)]
    yield dict(api=api, g=g, orc=orc, orc32=orc32, srcs=srcs, nrhs=nrhs, dims=dims, Ls=Ls, U=U, par=par, cut=cut)
    g.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_batched_operators_match_oracle_per_system(case, prec):
    A, g, n = case["api"], case["g"], case["nrhs"]
    P = A.F64 if prec == "f64" else A.F32
    tol = 1e-12 if prec == "f64" else 1e-5
    orc = case["orc"] if prec == "f64" else case["orc32"]
    srcs = [s if prec == "f64" else s.astype(np.complex64).astype(np.complex128) for s in case["srcs"]]
    nat = [g.pack(s, P, A.ODD) for s in srcs]
    batched = g.mrhs_gather(nat, P)
    # insert / extract round trip
    back = g.mrhs_scatter(batched, n, P)
    import torch
    assert all(torch.equal(a, b) for a, b in zip(back, nat))
    for dagger in (False, True):
        outs = g.mrhs_scatter(g.dhop_mrhs(batched, n, A.EVEN, dagger, P), n, P)
        for j in range(n):
            assert rel(g.unpack(outs[j], P, A.EVEN), orc.dhop(srcs[j], 0, dagger)) < tol, (j, dagger)
            assert torch.equal(outs[j], g.dhop(nat[j], A.EVEN, dagger, P))          # = the single-system kernel, bit for bit
        outs = g.mrhs_scatter(g.mpc_mrhs(batched, n, dagger, P), n, P)
        for j in range(n):
            assert rel(g.unpack(outs[j], P, A.ODD), orc.mpc(srcs[j], dagger=dagger)) < tol, (j, dagger)
            assert torch.equal(outs[j], g.mpc(nat[j], dagger, P))
    outs = g.mrhs_scatter(g.mdagm_mrhs(batched, n, P), n, P)
    for j in range(n):
        assert rel(g.unpack(outs[j], P, A.ODD), orc.mdagm(srcs[j])) < 2 * tol, j
        assert torch.equal(outs[j], g.mdagm(nat[j], P))


@pytest.mark.parametrize("mode", ["f64", "mixed"])
def test_batched_cg_matches_oracle_per_system(case, mode):
    from oracle.dwf_oracle import Oracle, cg, cg_mixed
    A, g, n, orc = case["api"], case["g"], case["nrhs"], case["orc"]
    tol = 1e-10
    srcs = list(case["srcs"])
    # systems that need different iteration counts: system 1 is solved to the same relative tolerance from a smoother source
    if n >= 2:
        srcs[1] = orc.mdagm(srcs[1])
    nat = [g.pack(s, A.F64, A.ODD) for s in srcs]
    batched = g.mrhs_gather(nat)
    x, infos, st = g.cg_mrhs(batched, n, tol, 20000, A.CG_MIXED if mode == "mixed" else A.CG_F64)
    assert st == A.OK
    xs = g.mrhs_scatter(x, n)
    if mode == "mixed":
        par = case["par"]
        o32 = Oracle(case["dims"], case["Ls"], par["M5"], par["mf"], par["b5"], par["c5"], antiperiodic_t=True, cut=case["cut"],
                     prec="f32").set_gauge(case["U"])
    for j in range(n):
        if mode == "f64":
            _, ref = cg(orc, srcs[j], tol, 20000)
            assert abs(infos[j]["iters_total"] - ref["iters"]) <= 2, (j, infos[j], ref)
        else:
            _, ref = cg_mixed(orc, o32, srcs[j], tol, 20000)
            assert infos[j]["restarts"] == ref["restarts"], (j, infos[j], ref)
            slack = max(2 * ref["restarts"], int(0.02 * ref["iters"]) + 1)         # reading C9
            assert abs(infos[j]["iters_total"] - ref["iters"]) <= slack, (j, infos[j], ref)
        got = g.unpack(xs[j], A.F64, A.ODD)
        true_res = np.sqrt(orc.norm2(srcs[j] - orc.mdagm(got)) / orc.norm2(srcs[j]))
        assert true_res <= tol * (1 + 1e-6) and abs(true_res - infos[j]["resid_true"]) <= 1e-3 * true_res + 1e-16
    if mode == "f64":
        # the batch is N independent CGs sharing launches: every system equals its single-system solve bit for bit
        import torch
        for j in range(n):
            x1, i1, st1 = g.cg(nat[j], tol, 20000, A.CG_F64)
            assert st1 == A.OK and i1["iters_total"] == infos[j]["iters_total"]
            assert torch.equal(x1, xs[j])


def test_batched_edge_cases(case):
    A, g, n = case["api"], case["g"], case["nrhs"]
    nat = [g.pack(s, A.F64, A.ODD) for s in case["srcs"]]
    # a vanishing right-hand side inside a batch: x_j = 0, zero iterations, the others unaffected
    import torch
    zero = torch.zeros_like(nat[0])
    batched = g.mrhs_gather([nat[0], zero] + nat[2:n])
    x, infos, st = g.cg_mrhs(batched, n, 1e-9, 20000)
    assert st == A.OK and infos[1]["iters_total"] == 0
    xs = g.mrhs_scatter(x, n)
    assert float(xs[1].abs().max()) == 0.0
    x0, i0, _ = g.cg(nat[0], 1e-9, 20000)
    assert torch.equal(xs[0], x0) and i0["iters_total"] == infos[0]["iters_total"]
    # max_iter reached: every system reports it, x holds the iterate
    x, infos, st = g.cg_mrhs(g.mrhs_gather(nat), n, 1e-30, 3)
    assert st == A.ENOTCONV and all(i["iters_total"] == 3 for i in infos)
    # nrhs = 1 is the plain path
    x1, inf1, st = g.cg_mrhs(nat[0], 1, 1e-9, 20000)
    assert st == A.OK and torch.equal(x1, x0)
    with pytest.raises(A.DwfError):
        g.cg_mrhs(batched, 17, 1e-9, 10)
    with pytest.raises(A.DwfError):
        g.dhop_mrhs(batched, n, A.FULL)


@pytest.mark.parametrize("mode", ["f64", "mixed"])
def test_system_frozen_long_before_the_rest_of_its_batch(case, mode):
    """A system whose stopping test fires at once (its initial guess is already the solution) stays frozen while the other
    systems of the batch run their full course.  On the fused path its Dhop chain then carries zeros and cg_r leaves its
    residual alone (csrc/dwf_fived.cu: cg_xp_kernel / cg_r_kernel); its x must come out finite, untouched by the others'
    iterations, and equal to what the single-system solve with the same guess returns, bit for bit."""
    import torch
    A, g, n = case["api"], case["g"], case["nrhs"]
    M = A.CG_MIXED if mode == "mixed" else A.CG_F64
    tol = 1e-10
    nat = [g.pack(s, A.F64, A.ODD) for s in case["srcs"]]
    x_done, i_done, st = g.cg(nat[0], 1e-12, 20000, A.CG_F64)
    assert st == A.OK
    guesses = [x_done.clone()] + [torch.zeros_like(nat[0]) for _ in range(n - 1)]
    x, infos, st = g.cg_mrhs(g.mrhs_gather(nat), n, tol, 20000, M, x=g.mrhs_gather(guesses), use_guess=True)
    assert st == A.OK
    xs = g.mrhs_scatter(x, n)
    assert infos[0]["iters_total"] == 0 and torch.equal(xs[0], x_done)             # never moved
    assert max(i["iters_total"] for i in infos[1:]) >= 20                            # while the others iterated
    for j in range(n):
        assert bool(torch.isfinite(xs[j]).all()), j
        x1, i1, st1 = g.cg(nat[j], tol, 20000, M, x=guesses[j].clone(), use_guess=True)
        assert st1 == A.OK
        if mode == "f64":
            assert i1["iters_total"] == infos[j]["iters_total"], (j, i1, infos[j])
            assert torch.equal(x1, xs[j]), j
        else:
            assert abs(i1["iters_total"] - infos[j]["iters_total"]) <= max(2, infos[j]["iters_total"] // 50), (j, i1, infos[j])
        assert infos[j]["resid_true"] <= tol
