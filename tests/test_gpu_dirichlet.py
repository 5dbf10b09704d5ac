"""Row a10: the Dirichlet checks, through the C ABI.

PAPER.md:175 -- the Dirichlet condition is applied to the gauge-field argument; eqs. 3-4 -- with the
cut D = [[D_Omega, D_d], [D_dbar, D_Omegabar]] loses its off-diagonal blocks; eq. 5 -- the Schur
(UDL) factorisation of D in terms of D_Omega, D_Omegabar^-1 and the two boundary blocks.

On BASELINE configs[1] (c2: 16^4 x Ls=16 Moebius, cut in t into two 16^3 x 8 blocks) at full size:
  * M_cut has exactly zero Omega <-> Omegabar blocks, and its Omega block equals the Omega block of the uncut M bit
    for bit (reading C7);
  * eq. 5 applied to a random vector, matrix-free with two Dirichlet solves, reproduces M v to solver accuracy.
The same two checks against the oracle's operators run on a scaled-down copy (8^3 x 16, Ls = 8).
The masks / projections are plain numpy on canonical arrays: projectors are "performance non-critical"
and not part of the hot path."""
import numpy as np
import pytest

from paper_2203_17119_b200 import inputs

pytestmark = pytest.mark.gpu


def rel(a, b):
    return float(np.linalg.norm((np.asarray(a) - np.asarray(b)).ravel()) / np.linalg.norm(np.asarray(b).ravel()))


class Pair:
    """The uncut and the Dirichlet-cut operator on one gauge field; canonical FULL fields in and out."""

    def __init__(self, api, dims, Ls, par, eps, seed, Bt):
        self.api, self.dims, self.Ls, self.par = api, tuple(dims), Ls, par
        self.U = inputs.gauge_weak(dims, eps, seed)
        mk = lambda cut: api.Dwf(dims, Ls, par["M5"], par["mf"], par["b5"], par["c5"], cut=cut)
        self.full, self.cut = mk((0, 0, 0, 0)), mk((0, 0, 0, Bt))
        self.full.set_gauge(self.U)
        self.cut.set_gauge(self.U)
        Lt = dims[3]
        t = np.arange(Lt)
        self.om = ((t // Bt) % 2 == 0).reshape(Lt, 1, 1, 1, 1, 1, 1)     # Omega = first block (c2: t < 8)

    def close(self):
        self.full.close()
        self.cut.close()

    def P(self, v, omega=True):
        return np.where(self.om if omega else ~self.om, v, 0.0)

    def _nat(self, g, v):
        import torch
        A = self.api
        e, o = inputs.split_parity(v, self.dims)
        return torch.cat([g.pack(e, A.F64, A.EVEN), g.pack(o, A.F64, A.ODD)])

    def _canon(self, g, nat):
        A = self.api
        n = nat.numel() // 2
        return inputs.merge_parity(g.unpack(nat[:n], A.F64, A.EVEN), g.unpack(nat[n:], A.F64, A.ODD), self.dims)

    def M(self, v, cut):
        g = self.cut if cut else self.full
        return self._canon(g, g.m(self._nat(g, v), False, self.api.F64))

    def Mcut_inv(self, eta, tol=1e-11):
        g = self.cut
        psi, info, st = g.solve(self._nat(g, eta), tol, 20000, self.api.CG_F64)
        assert st == self.api.OK, info
        return self._canon(g, psi)


MOEB = dict(M5=1.8, mf=0.01, b5=1.5, c5=0.5)


@pytest.fixture(scope="module", params=["c2", "small"])
def pair(request, oracle_built):
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2203_17119_b200 import api
    if request.param == "c2":
        cfg = inputs.CONFIGS["c2"]
        p = Pair(api, cfg.dims, cfg.Ls, dict(M5=cfg.M5, mf=cfg.mf, b5=cfg.b5, c5=cfg.c5), cfg.eps, cfg.gauge_seed, cfg.cut[3])
        p.with_oracle = True
    else:
        p = Pair(api, (8, 8, 8, 16), 8, MOEB, 0.3, 11, 8)
        p.with_oracle = True
    p.v = inputs.source_full(p.dims, p.Ls, 4242)
    yield p
    p.close()


def test_cut_operator_is_block_diagonal_and_restricts_D(pair):
    v = pair.v
    v_om = pair.P(v, True)
    Mc = pair.M(v_om, cut=True)
    # eqs. 3-4: no Omega -> Omegabar block at all once the crossing links are zero (exact zeros, not small numbers)
    assert np.count_nonzero(pair.P(Mc, False)) == 0
    # D_Omega = P_Omega D P_Omega, bit for bit (only the gauge-field argument changed)
    Mf = pair.M(v_om, cut=False)
    assert np.array_equal(pair.P(Mc, True), pair.P(Mf, True))
    # and the uncut operator does couple the two domains
    assert np.count_nonzero(pair.P(Mf, False)) > 0
    if pair.with_oracle:
        from oracle.dwf_oracle import Oracle
        par = pair.par
        orc = Oracle(pair.dims, pair.Ls, par["M5"], par["mf"], par["b5"], par["c5"], antiperiodic_t=True,
                     cut=(0, 0, 0, 8)).set_gauge(pair.U)
        want = orc.M(v_om)
        assert rel(Mc, want) < 1e-12 and float(np.abs(Mc - want).max() / np.abs(want).max()) < 1e-12


def test_eq5_schur_factorisation_on_a_random_vector(pair):
    """eq. 5, in the matrix-free form of SURVEY 8(c)-C7: with X = M - M_cut (the two boundary blocks),
    w_b = v_b + D_b^-1 D_dbar v_o ; y_o = D_o v_o - D_d D_b^-1 D_dbar v_o ; y_b = D_b w_b ; z_o = y_o + D_d D_b^-1 y_b ;
    z_b = y_b ; then z = M v   (o = Omega, b = Omegabar)."""
    v = pair.v
    X = lambda u: pair.M(u, cut=False) - pair.M(u, cut=True)
    v_o, v_b = pair.P(v, True), pair.P(v, False)
    a = pair.P(X(v_o), False)                      # D_dbar v_o
    b = pair.Mcut_inv(a)                           # D_b^-1 D_dbar v_o   (supported on Omegabar)
    assert np.count_nonzero(pair.P(b, True)) == 0
    y_o = pair.P(pair.M(v_o, cut=True), True) - pair.P(X(b), True)
    y_b = pair.P(pair.M(v_b + b, cut=True), False)
    c = pair.Mcut_inv(y_b)                         # D_b^-1 y_b
    z = y_o + pair.P(X(c), True) + y_b
    Mv = pair.M(v, cut=False)
    assert rel(z, Mv) < 1e-8
    if pair.with_oracle:
        from oracle.dwf_oracle import Oracle
        par = pair.par
        orc = Oracle(pair.dims, pair.Ls, par["M5"], par["mf"], par["b5"], par["c5"], antiperiodic_t=True).set_gauge(pair.U)
        assert rel(z, orc.M(v)) < 1e-8


@pytest.mark.slow
def test_c2_cg_to_completion_matches_oracle(oracle_built):
    """"oracle CG run to completion" -- BASELINE configs[1] at full size (16^4 x 16 Moebius, cut B_t = 8,
    tol 1e-10): Mpc^dag Mpc of the cut operator whole-field against the oracle, then the red-black CG on both sides with the
    iteration count within +-2 (north_star) and the oracle recomputing the true residual of the GPU solution."""
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2203_17119_b200 import api as A
    from oracle.dwf_oracle import Oracle, cg
    cfg = inputs.CONFIGS["c2"]
    U = inputs.make_gauge(cfg)
    g = A.from_config(cfg, device="cuda:0")
    g.set_gauge(U)
    orc = Oracle(cfg.dims, cfg.Ls, cfg.M5, cfg.mf, cfg.b5, cfg.c5, antiperiodic_t=cfg.antiperiodic_t, cut=cfg.cut).set_gauge(U)
    odd = inputs.source_half(cfg.dims, cfg.Ls, cfg.source_seed, parity=1)
    nat = g.pack(odd, A.F64, A.ODD)
    got, want = g.unpack(g.mdagm(nat, A.F64), A.F64, A.ODD), orc.mdagm(odd)
    assert rel(got, want) < 2e-12 and float(np.abs(got - want).max() / np.abs(want).max()) < 2e-12
    x_ref, info_ref = cg(orc, odd, cfg.tol, 5000)
    x, info, st = g.cg(nat, cfg.tol, 5000, A.CG_F64)
    assert st == A.OK and info_ref["converged"] and info["resid_true"] <= cfg.tol
    assert abs(info["iters_total"] - info_ref["iters"]) <= 2, (info, info_ref)
    xs = g.unpack(x, A.F64, A.ODD)
    assert np.sqrt(orc.norm2(odd - orc.mdagm(xs)) / orc.norm2(odd)) <= cfg.tol * (1 + 1e-6)
    assert rel(xs, x_ref) < 1e-5
    g.close()
