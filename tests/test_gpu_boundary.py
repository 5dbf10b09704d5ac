"""SURVEY 8f NEXT-1 through the C ABI: the domain and boundary projectors and the paper's boundary operators R (eqs. 9-10) and
R^-1 (eqs. 13-14) against oracle/boundary.py on small lattices, and the identity R R^-1 = P
on the GPU alone at BASELINE configs[1] (c2, 16^4 x 16, two 16^3 x 8 domains)."""
import numpy as np
import pytest

from paper_2203_17119_b200 import inputs

pytestmark = pytest.mark.gpu

MOEB = dict(M5=1.8, mf=0.05, b5=1.5, c5=0.5)
SHAM = dict(M5=1.8, mf=0.1, b5=1.0, c5=0.0)
CASES = {
    "shamir_t": dict(dims=(4, 4, 4, 8), Ls=4, par=SHAM, cut=(0, 0, 0, 4)),
    "moebius_t": dict(dims=(4, 4, 4, 8), Ls=4, par=MOEB, cut=(0, 0, 0, 4)),
    "shamir_zt_corners": dict(dims=(4, 4, 8, 8), Ls=4, par=SHAM, cut=(0, 0, 4, 4)),
    "shamir_thin_blocks": dict(dims=(4, 4, 4, 8), Ls=8, par=SHAM, cut=(0, 0, 0, 2)),
}


def rel(a, b):
    return float(np.linalg.norm((np.asarray(a) - np.asarray(b)).ravel()) / max(np.linalg.norm(np.asarray(b).ravel()), 1e-300))


class Ctx:
    def __init__(self, api, dims, Ls, par, cut, eps=0.3, seed=21):
        from oracle.boundary import Boundary
        self.api, self.dims, self.Ls = api, tuple(dims), Ls
        self.U = inputs.gauge_weak(dims, eps, seed)
        self.g = api.Dwf(dims, Ls, par["M5"], par["mf"], par["b5"], par["c5"], cut=cut)
        self.g.set_gauge(self.U)
        self.bd = Boundary(dims, Ls, par["M5"], par["mf"], par["b5"], par["c5"], cut, self.U)
        self.phi = inputs.source_full(dims, Ls, seed + 1)

    def nat(self, v):
        import torch
        A, g = self.api, self.g
        e, o = inputs.split_parity(v, self.dims)
        return torch.cat([g.pack(e, A.F64, A.EVEN), g.pack(o, A.F64, A.ODD)])

    def canon(self, nat):
        A, g = self.api, self.g
        n = nat.numel() // 2
        return inputs.merge_parity(g.unpack(nat[:n], A.F64, A.EVEN), g.unpack(nat[n:], A.F64, A.ODD), self.dims)


@pytest.fixture(scope="module", params=list(CASES))
def ctx(request, oracle_built):
    import torch
    assert torch.cuda.is_available()
    from paper_2203_17119_b200 import api
    c = Ctx(api, **CASES[request.param])
    yield c
    c.g.close()


def test_domain_and_boundary_projectors(ctx):
    g, bd, phi = ctx.g, ctx.bd, ctx.phi
    nat = ctx.nat(phi)
    assert np.array_equal(ctx.canon(g.domain_project(nat, 0)), bd.P_domain(phi, True))
    assert np.array_equal(ctx.canon(g.domain_project(nat, 1)), bd.P_domain(phi, False))
    got = ctx.canon(g.domain_project(nat, 2))
    assert rel(got, bd.P_boundary(phi)) < 1e-15
    # a projector: applying it twice changes nothing beyond rounding; it lives on Omega
    twice = ctx.canon(g.domain_project(g.domain_project(nat, 2), 2))
    assert rel(twice, got) < 1e-15
    assert np.count_nonzero(bd.P_domain(got, False)) == 0


def test_R_and_Rinv_match_oracle(ctx):
    A, g, bd, phi = ctx.api, ctx.g, ctx.bd, ctx.phi
    nat = ctx.nat(phi)
    out, info, st = g.boundary_op(nat, True, 1e-11, 20000)
    assert st == A.OK and info["resid_full"] < 1e-9
    assert rel(ctx.canon(out), bd.R_inv(phi)) < 1e-7
    out, info, st = g.boundary_op(nat, False, 1e-11, 20000)
    assert st == A.OK
    assert rel(ctx.canon(out), bd.R(phi)) < 1e-7
    # the operators of the context still see the CUT links afterwards
    Mc = ctx.canon(g.m(nat, False, A.F64))
    assert rel(Mc, bd.dir.M(phi)) < 1e-12


def test_R_Rinv_is_P_on_the_gpu(ctx):
    A, g, phi = ctx.api, ctx.g, ctx.phi
    nat = ctx.nat(phi)
    rinv, _, st1 = g.boundary_op(nat, True, 1e-11, 20000)
    rr, _, st2 = g.boundary_op(rinv, False, 1e-11, 20000)
    assert st1 == A.OK and st2 == A.OK
    assert rel(ctx.canon(rr), ctx.canon(g.domain_project(nat, 2))) < 1e-7


def test_boundary_ops_need_a_two_colourable_cut(oracle_built):
    from paper_2203_17119_b200 import api
    U = inputs.gauge_weak((4, 4, 4, 8), 0.3, 3)
    for cut in ((0, 0, 0, 0), (0, 0, 0, 8)):            # no cut; one block (only the wrap link is cut)
        g = api.Dwf((4, 4, 4, 8), 4, 1.8, 0.1, 1.0, 0.0, cut=cut)
        g.set_gauge(U)
        f = g.new_native(api.F64, api.FULL).normal_()
        with pytest.raises(api.DwfError) as e:
            g.domain_project(f, 2)
        assert e.value.status == api.EINVAL
        with pytest.raises(api.DwfError) as e:
            g.boundary_op(f, True, 1e-8, 100)
        assert e.value.status == api.EINVAL
        g.close()


def test_c2_R_Rinv_is_P_full_size(oracle_built):
    """BASELINE configs[1] at full size, GPU only: R R^-1 phi = P phi with three solves (one uncut, two Dirichlet)."""
    import torch
    from paper_2203_17119_b200 import api
    cfg = inputs.CONFIGS["c2"]
    g = api.from_config(cfg)
    g.set_gauge(inputs.make_gauge(cfg))
    phi = g.new_native(api.F64, api.FULL).normal_()
    rinv, i1, st1 = g.boundary_op(phi, True, 1e-10, 50000, api.CG_MIXED)
    rr, i2, st2 = g.boundary_op(rinv, False, 1e-10, 50000, api.CG_MIXED)
    assert st1 == api.OK and st2 == api.OK
    p = g.domain_project(phi, 2)
    err = float(torch.linalg.norm(rr - p) / torch.linalg.norm(p))
    assert err < 1e-7, (err, i1, i2)
    g.close()
