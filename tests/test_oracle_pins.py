"""Pins for the oracle (`-m "not gpu"`): the oracle is checked against what the paper and the
mathematics fix, never against itself or the CUDA path.

The paper prints no worked numerical example, so the pins are:
  dense Kronecker brute force (tests/dense_ref.py, independent construction),
  the free-field plane-wave closed form, gauge covariance, gamma5-R5 hermiticity,
  the Mooee^{-1} closed form, the Schur/determinant identities, the paper's eq. 5 and
  eq. 6 on a Dirichlet-cut lattice, D_Omega = restricted D,
  and CG against a dense solve.
"""
import numpy as np
import pytest

import dense_ref as dr
from oracle.dwf_oracle import Oracle, cg, cg_mixed, solve_redblack, split, merge
from paper_2203_17119_b200 import inputs

DIMS = (2, 2, 2, 4)
LS = 4
V = int(np.prod(DIMS))
MOEB = dict(M5=1.8, mf=0.05, b5=1.5, c5=0.5)
SHAM = dict(M5=1.8, mf=0.1, b5=1.0, c5=0.0)


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


@pytest.fixture(scope="module")
def U():
    return inputs.gauge_weak(DIMS, 0.4, 77)


@pytest.fixture(scope="module")
def psi():
    return inputs.source_full(DIMS, LS, 78)


def make(par, U, cut=(0, 0, 0, 0), dims=DIMS, Ls=LS, apbc=True, prec="f64"):
    return Oracle(dims, Ls, antiperiodic_t=apbc, cut=cut, prec=prec, **par).set_gauge(U)


# ---------------------------------------------------------------- gamma algebra (C1)
def test_gamma_clifford_hermitian_gamma5(oracle_built):
    o = Oracle(DIMS, LS, **SHAM)
    g = [o.gamma(mu) for mu in range(4)]
    for mu in range(4):
        assert np.allclose(g[mu], g[mu].conj().T)
        for nu in range(4):
            assert np.allclose(g[mu] @ g[nu] + g[nu] @ g[mu], 2 * (mu == nu) * np.eye(4))
    assert np.allclose(g[0] @ g[1] @ g[2] @ g[3], np.diag([1, 1, -1, -1]))


# ---------------------------------------------------------------- inputs
def test_gauge_is_su3_and_plaquette_fingerprint():
    Ug = inputs.gauge_weak((4, 4, 4, 4), 0.2, 1001)
    UU = Ug @ np.conj(np.swapaxes(Ug, -1, -2))
    assert np.allclose(UU, np.eye(3), atol=1e-13)
    assert np.allclose(np.linalg.det(Ug), 1.0, atol=1e-13)
    # <plaq> ~ 0.80 at eps=0.2, 0.61 at 0.3, ~0.05 at 0.7 for this generator
    assert abs(inputs.plaquette(Ug) - 0.80) < 0.02
    assert abs(inputs.plaquette(inputs.gauge_weak((4, 4, 4, 4), 0.3, 5)) - 0.61) < 0.02
    assert abs(inputs.plaquette(inputs.gauge_weak((4, 4, 4, 4), 0.7, 5)) - 0.05) < 0.03
    assert abs(inputs.plaquette(inputs.gauge_unit((4, 4, 4, 4))) - 1.0) < 1e-15
    Uh = inputs.ape_smear(inputs.gauge_haar((4, 4, 4, 4), 3), 0.5, 2)
    assert np.allclose(Uh @ np.conj(np.swapaxes(Uh, -1, -2)), np.eye(3), atol=1e-13)


def test_haar_ape_generator_of_c5():
    """The c5 gauge recipe (Haar SU(3) + 4 APE passes, alpha = 0.5) against what is known without running it:
    Haar links have <Re tr P>/3 = 0 and <|U_ij|^2> = 1/3; a pure-gauge field is a fixed point of the smearing (every staple
    equals the link); each pass raises the plaquette.  The value after 4 passes, 0.60 (0.597 on 8^4, 0.604 on the c5
    lattice), is the recipe's fingerprint, kept to +-1 % so a changed alpha, staple or pass count shows."""
    dims = (8, 8, 8, 8)
    cfg = inputs.CONFIGS["c5"]
    U0 = inputs.gauge_haar(dims, cfg.gauge_seed)
    assert np.allclose(U0 @ np.conj(np.swapaxes(U0, -1, -2)), np.eye(3), atol=1e-13)
    assert np.allclose(np.linalg.det(U0), 1.0, atol=1e-13)
    nplaq = 6 * int(np.prod(dims))
    assert abs(inputs.plaquette(U0)) < 4.0 / np.sqrt(nplaq)          # variance of Re tr P / 3 for Haar links is 1/18 < 1
    assert abs(np.mean(np.abs(U0) ** 2) - 1.0 / 3.0) < 1e-12
    plaq = [inputs.plaquette(U0)]
    Us = U0
    for _ in range(4):
        Us = inputs.ape_smear(Us, 0.5, 1)
        plaq.append(inputs.plaquette(Us))
    assert all(b > a for a, b in zip(plaq, plaq[1:]))
    assert np.allclose(Us @ np.conj(np.swapaxes(Us, -1, -2)), np.eye(3), atol=1e-13)
    assert abs(plaq[-1] - 0.60) < 0.006
    assert np.array_equal(inputs.make_gauge(inputs.small_variant(cfg, dims)), Us)          # make_gauge(c5) is this recipe
    g = inputs.gauge_haar((4, 4, 4, 4), 7)[..., 0, :, :]
    Ug = np.stack([g @ np.conj(np.swapaxes(np.roll(g, -1, axis=3 - mu), -1, -2)) for mu in range(4)], axis=4)
    assert abs(inputs.plaquette(Ug) - 1.0) < 1e-14
    assert np.abs(inputs.ape_smear(Ug, 0.5, 2) - Ug).max() < 1e-14


def test_split_merge_roundtrip():
    f = inputs.source_full(DIMS, LS, 5)
    e, o = inputs.split_parity(f, DIMS)
    assert np.array_equal(inputs.merge_parity(e, o, DIMS), f)
    e2, o2 = split(f, DIMS)
    assert np.array_equal(e, e2) and np.array_equal(o, o2)
    # cb = lex/2 in increasing lex order
    pm = inputs.parity_mask(DIMS).reshape(-1)
    lex_odd = np.nonzero(pm == 1)[0]
    assert np.array_equal(lex_odd // 2, np.arange(V // 2))


# ---------------------------------------------------------------- dense brute force
@pytest.mark.parametrize("apbc", [True, False])
@pytest.mark.parametrize("dagger", [False, True])
def test_dhop_vs_dense(U, psi, apbc, dagger, oracle_built):
    o = make(MOEB, U, apbc=apbc)
    D4 = dr.dhop4(U, DIMS, apbc, dagger)
    want = (dr.lift5(D4, V, LS) @ psi.reshape(-1)).reshape(psi.shape)
    assert rel(o.dhop(psi, 2, dagger), want) < 1e-14


def test_dhop_vs_dense_asymmetric_lattice(oracle_built):
    dims = (4, 2, 2, 4)                     # forward and backward x-neighbours differ
    Ug = inputs.gauge_weak(dims, 0.5, 9)
    f = inputs.source_full(dims, 2, 10)
    o = make(MOEB, Ug, dims=dims, Ls=2)
    Vv = int(np.prod(dims))
    want = dr.lift5(dr.dhop4(Ug, dims, True), Vv, 2) @ f.reshape(-1)
    assert rel(o.dhop(f, 2), want) < 1e-14
    M = dr.dwf_matrix(Ug, dims, 2, 1.8, 0.05, 1.5, 0.5)
    assert rel(o.M(f), M @ f.reshape(-1)) < 1e-14


@pytest.mark.parametrize("par", [MOEB, SHAM])
def test_M_and_Mdag_vs_dense(U, psi, par, oracle_built):
    o = make(par, U)
    M = dr.dwf_matrix(U, DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    v = psi.reshape(-1)
    assert rel(o.M(psi), M @ v) < 1e-14
    assert rel(o.M(psi, dagger=True), M.conj().T @ v) < 1e-14


def test_parity_dhop_is_restriction_of_full(U, psi, oracle_built):
    o = make(MOEB, U)
    e, od = split(psi, DIMS)
    z = np.zeros_like(e)
    for dag in (False, True):
        full_from_odd = o.dhop(merge(z, od, DIMS), 2, dag)
        fe, fo = split(full_from_odd, DIMS)
        assert rel(o.dhop(od, 0, dag), fe) < 1e-15 and np.abs(fo).max() == 0
        fe, fo = split(o.dhop(merge(e, z, DIMS), 2, dag), DIMS)
        assert rel(o.dhop(e, 1, dag), fo) < 1e-15 and np.abs(fe).max() == 0


@pytest.mark.parametrize("par", [MOEB, SHAM])
def test_redblack_blocks_vs_dense(U, psi, par, oracle_built):
    """Mooee, Meooe, Mooee^{-1}, Mpc built from dense blocks of M (C5, C6)."""
    o = make(par, U)
    M = dr.dwf_matrix(U, DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    ev, od = dr.parity_index(DIMS, LS)
    Mee, Meo, Moe, Moo = M[np.ix_(ev, ev)], M[np.ix_(ev, od)], M[np.ix_(od, ev)], M[np.ix_(od, od)]
    pe, po = split(psi, DIMS)
    ve, vo = pe.reshape(-1), po.reshape(-1)
    for dag in (False, True):
        H = (lambda A: A.conj().T) if dag else (lambda A: A)
        assert rel(o.mooee(po, dag), H(Moo) @ vo) < 1e-14
        assert rel(o.mooee(pe, dag), H(Mee) @ ve) < 1e-14
        assert rel(o.mooee_inv(pe, dag), np.linalg.solve(H(Mee), ve)) < 1e-13
    assert rel(o.meooe(po, 0), Meo @ vo) < 1e-14
    assert rel(o.meooe(pe, 1), Moe @ ve) < 1e-14
    # (Meooe)^dag with output parity p = dagger of the block that maps p -> other
    assert rel(o.meooe(po, 0, dagger=True), Moe.conj().T @ vo) < 1e-14
    assert rel(o.meooe(pe, 1, dagger=True), Meo.conj().T @ ve) < 1e-14
    Mpc = Moo - Moe @ np.linalg.solve(Mee, Meo)
    assert rel(o.mpc(po), Mpc @ vo) < 1e-13
    assert rel(o.mpc(po, dagger=True), Mpc.conj().T @ vo) < 1e-13
    assert rel(o.mdagm(po), Mpc.conj().T @ (Mpc @ vo)) < 1e-13
    # det M = det Mee det Mpc
    s0, l0 = np.linalg.slogdet(M)
    s1, l1 = np.linalg.slogdet(Mee)
    s2, l2 = np.linalg.slogdet(Mpc)
    assert abs(l0 - l1 - l2) < 1e-9 and abs(s0 - s1 * s2) < 1e-9
    # the blocks sum to M and Mooee is parity diagonal
    assert np.abs(M[np.ix_(ev, od)] - Meo).max() == 0


# ---------------------------------------------------------------- Mooee^{-1} closed form
def closed_form_T(Ls, M5, mf, b5, c5):
    bee, cee = 1 + b5 * (4 - M5), 1 - c5 * (4 - M5)
    r = cee / bee
    d = bee * (1 + mf * r ** Ls)
    Tp = np.zeros((Ls, Ls)); Tm = np.zeros((Ls, Ls))
    for s in range(Ls):
        for sp in range(Ls):
            Tp[s, sp] = r ** ((s - sp) % Ls) * (1.0 if s >= sp else -mf) / d
            Tm[s, sp] = r ** ((sp - s) % Ls) * (1.0 if sp >= s else -mf) / d
    return Tp, Tm


@pytest.mark.parametrize("par", [MOEB, SHAM, dict(M5=1.8, mf=1.0, b5=1.5, c5=0.5), dict(M5=1.4, mf=0.0, b5=2.0, c5=1.0)])
@pytest.mark.parametrize("Ls", [1, 2, 5, 12, 16])
def test_mooee_inv_closed_form_and_identity(par, Ls, oracle_built):
    o = Oracle(DIMS, Ls, **par)
    x = inputs.complex_gaussian((6, Ls, 4, 3), 31 + Ls)
    Tp, Tm = closed_form_T(Ls, **par)
    for dag in (False, True):
        y = o.mooee_inv(x, dag)
        A, B = (Tm, Tp) if dag else (Tp, Tm)
        want = np.empty_like(x)
        want[:, :, :2] = np.einsum("st,ntac->nsac", A, x[:, :, :2])
        want[:, :, 2:] = np.einsum("st,ntac->nsac", B, x[:, :, 2:])
        assert rel(y, want) < 1e-13
        assert rel(o.mooee(y, dag), x) < 1e-13
        assert rel(o.mooee_inv(o.mooee(x, dag), dag), x) < 1e-13


# ---------------------------------------------------------------- free field closed form (C3)
@pytest.mark.parametrize("n", [(0, 0, 0, 0), (1, 0, 1, 2), (3, 1, 0, 1)])
@pytest.mark.parametrize("apbc", [True, False])
def test_free_field_plane_wave(n, apbc, oracle_built):
    dims, Ls = (4, 2, 2, 4), 3
    par = MOEB
    o = make(par, inputs.gauge_unit(dims), dims=dims, Ls=Ls, apbc=apbc)
    p = [2 * np.pi * n[mu] / dims[mu] for mu in range(3)] + [2 * np.pi * (n[3] + (0.5 if apbc else 0.0)) / dims[3]]
    # D_W(p) = (4 - M5 - sum cos p) + i sum gamma sin p ;  Dhop(p) = sum (2 cos p - 2 i gamma sin p)
    DWp = (4 - par["M5"] - sum(np.cos(p))) * np.eye(4) + 1j * sum(np.sin(p[mu]) * dr.GAMMA[mu] for mu in range(4))
    Dhp = sum(2 * np.cos(p[mu]) * np.eye(4) - 2j * np.sin(p[mu]) * dr.GAMMA[mu] for mu in range(4))
    up, dn = dr.s_shifts(Ls, par["mf"])
    Qs = np.kron(up, dr.PM) + np.kron(dn, dr.PP)
    Mp = np.kron(np.eye(Ls), par["b5"] * DWp + np.eye(4)) + np.kron(np.eye(Ls), par["c5"] * DWp - np.eye(4)) @ Qs
    u = inputs.complex_gaussian((Ls, 4, 3), 44)
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    psi = phase[..., None, None, None] * u
    want_M = phase[..., None, None, None] * np.einsum("ij,jc->ic", Mp, u.reshape(Ls * 4, 3)).reshape(Ls, 4, 3)
    want_D = phase[..., None, None, None] * np.einsum("ab,sbc->sac", Dhp, u)
    assert rel(o.dhop(psi, 2), want_D) < 1e-13
    assert rel(o.M(psi), want_M) < 1e-13


# ---------------------------------------------------------------- gauge covariance
def test_gauge_covariance(U, psi, oracle_built):
    g = inputs.gauge_haar(DIMS, 123)[..., 0, :, :]          # one SU(3) per site
    Ug = np.empty_like(U)
    for mu in range(4):
        gshift = np.roll(g, -1, axis=3 - mu)                # g(x+mu)
        Ug[..., mu, :, :] = g @ U[..., mu, :, :] @ np.conj(np.swapaxes(gshift, -1, -2))
    o, og = make(MOEB, U, apbc=False), make(MOEB, Ug, apbc=False)
    gpsi = np.einsum("tzyxab,tzyxsib->tzyxsia", g, psi)
    lhs = og.M(gpsi)
    rhs = np.einsum("tzyxab,tzyxsib->tzyxsia", g, o.M(psi))
    assert rel(lhs, rhs) < 1e-13


# ---------------------------------------------------------------- gamma5 R5 hermiticity (C4')
def G5R5(f):
    out = f[..., ::-1, :, :].copy()
    out[..., 2:, :] *= -1
    return out


def test_gamma5R5_hermiticity(U, psi, oracle_built):
    o = make(SHAM, U)
    assert rel(o.M(psi, dagger=True), G5R5(o.M(G5R5(psi)))) < 1e-14          # Shamir: exact
    o = make(MOEB, U)
    assert rel(o.M(psi, dagger=True), G5R5(o.M(G5R5(psi)))) > 1e-3           # Moebius c5 != 0: not Gamma5-hermitian

    def Dminus(f):                                                            # D_- = c5 D_W - 1
        return MOEB["c5"] * ((4 - MOEB["M5"]) * f - 0.5 * o.dhop(f, 2)) - f
    lhs = o.M(Dminus(psi))
    rhs = Dminus(G5R5(o.M(G5R5(psi), dagger=True)))
    assert rel(lhs, rhs) < 1e-13
    # <u, M v> = <M^dag u, v>
    u = inputs.source_full(DIMS, LS, 79)
    assert abs(np.vdot(u, o.M(psi)) - np.vdot(o.M(u, dagger=True), psi)) < 1e-11 * abs(np.vdot(u, o.M(psi)))
    # dhop^dag = gamma5 dhop gamma5
    g5 = lambda f: np.concatenate([f[..., :2, :], -f[..., 2:, :]], axis=-2)
    assert rel(o.dhop(psi, 2, True), g5(o.dhop(g5(psi), 2))) < 1e-14


# ---------------------------------------------------------------- Dirichlet (eqs. 3-6)
def test_dirichlet_blocks_schur_eq5_det_eq6(U, psi, oracle_built):
    cut = (0, 0, 0, 2)
    par = MOEB
    o_cut, o = make(par, U, cut=cut), make(par, U)
    M = dr.dwf_matrix(U, DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    Mc = dr.dwf_matrix(dr.cut_gauge(U, DIMS, cut), DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    om, ob = dr.domain_index(DIMS, LS, 3, 2)
    v = psi.reshape(-1)
    # oracle with cut == dense with cut gauge
    assert rel(o_cut.M(psi), Mc @ v) < 1e-14
    # D_dirichlet is block diagonal and its Omega block equals the Omega block of D, bit for bit
    assert np.abs(Mc[np.ix_(om, ob)]).max() == 0 and np.abs(Mc[np.ix_(ob, om)]).max() == 0
    assert np.array_equal(Mc[np.ix_(om, om)], M[np.ix_(om, om)])
    assert np.array_equal(Mc[np.ix_(ob, ob)], M[np.ix_(ob, ob)])
    # matrix-free: D_cut (P_Omega v) == P_Omega D P_Omega v
    vO = np.zeros_like(v); vO[om] = v[om]
    got = o_cut.M(vO.reshape(psi.shape)).reshape(-1)
    full = o.M(vO.reshape(psi.shape)).reshape(-1)
    assert np.abs(got[ob]).max() == 0
    assert rel(got[om], full[om]) < 1e-15
    # eq. 5 applied to a vector, using the oracle for every operator application
    DO, DOb = M[np.ix_(om, om)], M[np.ix_(ob, ob)]
    Dd, Ddb = M[np.ix_(om, ob)], M[np.ix_(ob, om)]           # D_partial, D_partial-bar
    w_ob = v[ob] + np.linalg.solve(DOb, Ddb @ v[om])
    y_om = (DO - Dd @ np.linalg.solve(DOb, Ddb)) @ v[om]
    y_ob = DOb @ w_ob
    z = np.empty_like(v)
    z[om] = y_om + Dd @ np.linalg.solve(DOb, y_ob)
    z[ob] = y_ob
    assert rel(z, o.M(psi).reshape(-1)) < 1e-12
    # D_partial from the oracle: P_Omega (M - M_cut) P_Omegabar
    vOb = np.zeros_like(v); vOb[ob] = v[ob]
    dpar = (o.M(vOb.reshape(psi.shape)) - o_cut.M(vOb.reshape(psi.shape))).reshape(-1)
    assert rel(dpar[om], Dd @ v[ob]) < 1e-13
    # eq. 6: det D = det D_Omega det D_Omegabar det(1 - D_Omega^-1 D_d D_Omegabar^-1 D_dbar)
    chi = np.eye(len(om)) - np.linalg.solve(DO, Dd @ np.linalg.solve(DOb, Ddb))
    s, l = np.linalg.slogdet(M)
    parts = [np.linalg.slogdet(A) for A in (DO, DOb, chi)]
    assert abs(l - sum(p[1] for p in parts)) < 1e-9
    assert abs(s - np.prod([p[0] for p in parts])) < 1e-9


# ---------------------------------------------------------------- solvers
def test_cg_vs_dense_solve(U, psi, oracle_built):
    par = MOEB
    o = make(par, U)
    M = dr.dwf_matrix(U, DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    ev, od = dr.parity_index(DIMS, LS)
    Mpc = M[np.ix_(od, od)] - M[np.ix_(od, ev)] @ np.linalg.solve(M[np.ix_(ev, ev)], M[np.ix_(ev, od)])
    A = Mpc.conj().T @ Mpc
    _, b = split(psi, DIMS)
    xs = np.linalg.solve(A, b.reshape(-1))
    hist = []
    x, info = cg(o, b, 1e-11, 2000, history=hist)
    assert info["converged"] and info["resid_true"] <= 1e-11
    assert rel(x, xs) < 1e-9
    assert abs(hist[-1] - info["resid_iter"]) < 1e-30 and len(hist) == info["iters"]
    # A-norm of the error decreases monotonically (CG optimality)
    errs = []
    for k in (2, 5, 10, 20):
        xk, _ = cg(o, b, 1e-30, k, restart_on_true=False)
        e = xk.reshape(-1) - xs
        errs.append(np.real(np.vdot(e, A @ e)))
    assert all(errs[i + 1] < errs[i] for i in range(len(errs) - 1))
    # initial guess: starting from the solution converges immediately
    x2, info2 = cg(o, b, 1e-9, 100, x0=x)
    assert info2["iters"] == 0 and info2["converged"]


def test_norm2_is_the_plain_sum_of_squares(psi, oracle_built):
    """orc_norm2 pinned directly: every other pin uses it only in ratios, where a wrong normalisation (a half-summed array,
    |re|^2 only) would cancel.  numpy's vdot on the same values, both precisions (the fp32 oracle accumulates in fp64, C8)."""
    _, b = split(psi, DIMS)
    o64, o32 = Oracle(DIMS, LS, **SHAM), Oracle(DIMS, LS, prec="f32", **SHAM)
    want = float(np.vdot(b, b).real)
    assert abs(o64.norm2(b) - want) <= 1e-14 * want
    b32 = b.astype(np.complex64)
    want32 = float(np.vdot(b32.astype(np.complex128), b32.astype(np.complex128)).real)
    assert abs(o32.norm2(b32) - want32) <= 1e-14 * want32
    e = np.zeros_like(b)
    e.reshape(-1)[-1] = 3 - 4j                                     # the last element counts, re and im both
    assert o64.norm2(e) == 25.0 and o64.norm2(np.zeros_like(b)) == 0.0


def test_cg_restarts_from_the_true_residual(U, psi, oracle_built):
    """Reading C8's restart rule, entered for real: at tol = 4e-15 the recurrence residual passes the test while the true
    residual b - A x (~5e-15 here, fp64 rounding of 160 iterations) does not, so the solve must recompute r = b - A x, go
    on from the current x, keep counting iterations, and stop once the TRUE residual is below tol.  Checked against the
    same rule written around numpy's dense Mpc (independent construction, tests/dense_ref.py), and against what holds
    whatever the rule's details: the answer satisfies the dense system to tol, at least one restart happened, and the
    restarted solve took more iterations than the recurrence alone asks for (restart_on_true=False)."""
    par = MOEB
    o = make(par, U)
    M = dr.dwf_matrix(U, DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    ev, od = dr.parity_index(DIMS, LS)
    Mpc = M[np.ix_(od, od)] - M[np.ix_(od, ev)] @ np.linalg.solve(M[np.ix_(ev, ev)], M[np.ix_(ev, od)])
    Mh = Mpc.conj().T
    _, b = split(psi, DIMS)
    bv = b.reshape(-1)
    tol, max_iter = 4e-15, 2000
    n2 = lambda v: float(np.vdot(v, v).real)
    bn2 = n2(bv)
    target = tol * tol * bn2
    x = np.zeros_like(bv)
    iters = restarts = 0
    while True:
        r = bv - Mh @ (Mpc @ x) if restarts else bv.copy()
        p, c = r.copy(), n2(r)
        while c > target and iters < max_iter:
            q = Mpc @ p
            alpha = c / n2(q)
            x += alpha * p
            r -= alpha * (Mh @ q)
            cn = n2(r)
            iters += 1
            if cn <= target:
                break
            p = r + (cn / c) * p
            c = cn
        true = np.sqrt(n2(bv - Mh @ (Mpc @ x)) / bn2)
        if true <= tol or iters >= max_iter:
            break
        restarts += 1
    assert true <= tol and restarts >= 1
    xo, info = cg(o, b, tol, max_iter)
    assert info["converged"] and info["restarts"] >= 1
    assert info["restarts"] == restarts and abs(info["iters"] - iters) <= 2, (info, restarts, iters)
    # independent of the rule's wording: the dense system is solved to tol, and the reported true residual is the real one
    dense_true = np.sqrt(n2(bv - Mh @ (Mpc @ xo.reshape(-1))) / bn2)
    # (to the rounding of evaluating b - A x itself, ~1e-15 relative here: two evaluations differ by that much)
    assert dense_true <= 1.5 * tol and abs(dense_true - info["resid_true"]) <= 0.5 * tol
    _, plain = cg(o, b, tol, max_iter, restart_on_true=False)
    assert plain["restarts"] == 0 and not plain["converged"] and plain["resid_true"] > tol
    assert info["iters"] > plain["iters"]                          # iterations of all passes are counted


def test_multishift_cg_vs_dense_solves(U, psi, oracle_built):
    """NEXT-2: every shifted solution against numpy's dense solve of (Mpc^dag Mpc + sigma) x = b, the matrix built
    from dense blocks (independent of the oracle's loops); one shared iteration count; sigma = 0 reproduces plain CG."""
    from oracle.dwf_oracle import multishift_cg
    par = MOEB
    o = make(par, U)
    M = dr.dwf_matrix(U, DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    ev, od = dr.parity_index(DIMS, LS)
    Mpc = M[np.ix_(od, od)] - M[np.ix_(od, ev)] @ np.linalg.solve(M[np.ix_(ev, ev)], M[np.ix_(ev, od)])
    A = Mpc.conj().T @ Mpc
    _, b = split(psi, DIMS)
    shifts = [0.0, 0.01, 0.3, 5.0]
    xs, info = multishift_cg(o, b, shifts, 1e-11, 2000)
    assert info["converged"] and max(info["resid_true"]) <= 1.01e-11
    for x, sg in zip(xs, shifts):
        want = np.linalg.solve(A + sg * np.eye(A.shape[0]), b.reshape(-1))
        assert rel(x.reshape(-1), want) < 1e-9
    # the larger the shift the better conditioned the system: true residuals do not increase with sigma
    assert all(info["resid_true"][i + 1] <= info["resid_true"][i] * (1 + 1e-6) + 1e-15 for i in range(3))
    x0, info0 = cg(o, b, 1e-11, 2000)
    assert abs(info["iters"] - info0["iters"]) <= 1 and rel(xs[0], x0) < 1e-9


def test_chebyshev_filter_vs_spectral_decomposition(U, psi, oracle_built):
    """NEXT-4: T_n((2A - hi - lo)/(hi - lo)) v against the spectral definition sum_i T_n(l_i) <u_i, v> u_i from numpy's
    eigh of the dense Mpc^dag Mpc and numpy's own Chebyshev evaluation (no recurrence shared with the oracle)."""
    from numpy.polynomial import chebyshev as npcheb
    from oracle.dwf_oracle import chebyshev
    par = MOEB
    o = make(par, U)
    M = dr.dwf_matrix(U, DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    ev, od = dr.parity_index(DIMS, LS)
    Mpc = M[np.ix_(od, od)] - M[np.ix_(od, ev)] @ np.linalg.solve(M[np.ix_(ev, ev)], M[np.ix_(ev, od)])
    lam, Uv = np.linalg.eigh(Mpc.conj().T @ Mpc)
    _, b = split(psi, DIMS)
    lo, hi = 0.5 * lam[-1], 1.05 * lam[-1]          # a window on the upper part of the spectrum: low modes are amplified
    for n in (0, 1, 2, 7, 16):
        coef = np.zeros(n + 1)
        coef[n] = 1.0
        tl = npcheb.chebval((2 * lam - (hi + lo)) / (hi - lo), coef)
        want = Uv @ (tl * (Uv.conj().T @ b.reshape(-1)))
        got = chebyshev(o, b, lo, hi, n).reshape(-1)
        assert rel(got, want) < 1e-9, n
    # inside the window |T_n| <= 1, below it the filter grows: the lowest mode is enhanced relative to the top one
    gain = npcheb.chebval((2 * lam[[0, -1]] - (hi + lo)) / (hi - lo), coef)
    assert abs(gain[0]) > 1e3 * abs(gain[1])


def test_redblack_solve_vs_dense(U, psi, oracle_built):
    par = SHAM
    o = make(par, U)
    M = dr.dwf_matrix(U, DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    want = np.linalg.solve(M, psi.reshape(-1))
    sol, info = solve_redblack(o, psi, 1e-11, 2000)
    assert info["converged"] and info["resid_full"] < 1e-9
    assert rel(sol, want) < 1e-9


def test_mixed_cg(U, psi, oracle_built):
    par = MOEB
    o64, o32 = make(par, U), make(par, U, prec="f32")
    _, b = split(psi, DIMS)
    x, info = cg_mixed(o64, o32, b, 1e-10, 5000)
    assert info["converged"] and info["resid_true"] <= 1e-10 and info["restarts"] >= 2
    x64, _ = cg(o64, b, 1e-12, 5000)
    assert rel(x, x64) < 1e-8
    # the fp32 oracle is the fp64 oracle in lower precision
    assert rel(o32.mpc(b.astype(np.complex64)).astype(np.complex128), o64.mpc(b)) < 1e-6


def test_mixed_cg_restarts_and_deltas_vs_dense_defect_correction(U, psi, oracle_built):
    """Reading C9 pinned through its constants, not only its answer: the same defect correction written out around numpy's
    dense matrices (fp64 outer residual with the dense Mpc^dag Mpc, inner CG with the complex64 copy of the dense Mpc and
    fp64 reductions, delta = max(inner_tol, tol |b| / |r|)) must give the oracle's restart count, its delta sequence and
    its inner iteration counts.  A wrong delta rule, a missing restart or an inner solve that does not start from e = 0
    changes these numbers even when the final answer still converges."""
    par = MOEB
    o64, o32 = make(par, U), make(par, U, prec="f32")
    M = dr.dwf_matrix(U, DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    ev, od = dr.parity_index(DIMS, LS)
    Mpc = M[np.ix_(od, od)] - M[np.ix_(od, ev)] @ np.linalg.solve(M[np.ix_(ev, ev)], M[np.ix_(ev, od)])
    Mpc32 = Mpc.astype(np.complex64)
    Mpc32h = np.ascontiguousarray(Mpc32.conj().T)
    _, b = split(psi, DIMS)
    bv = b.reshape(-1)
    for tol, inner_tol in ((1e-10, 1e-4), (1e-9, 1e-2), (1e-12, 1e-5)):
        n2 = lambda v: float(np.sum(np.abs(v.astype(np.complex128)) ** 2))
        x = np.zeros_like(bv)
        bn2 = n2(bv)
        deltas, inner, restarts = [], [], 0
        while True:
            r = bv - Mpc.conj().T @ (Mpc @ x)
            rn2 = n2(r)
            if np.sqrt(rn2 / bn2) <= tol or restarts >= 20:
                break
            delta = max(inner_tol, tol * np.sqrt(bn2 / rn2))
            rf = r.astype(np.complex64)
            e = np.zeros_like(rf)
            p = rf.copy()
            c = n2(rf)
            target = delta * delta * c
            k = 0
            while c > target:
                q = Mpc32 @ p
                alpha = np.float32(c / n2(q))
                e += alpha * p
                rf -= alpha * (Mpc32h @ q)
                cn = n2(rf)
                k += 1
                if cn <= target:
                    break
                p = rf + np.float32(cn / c) * p
                c = cn
            x = x + e.astype(np.complex128)
            deltas.append(delta)
            inner.append(k)
            restarts += 1
        xo, info = cg_mixed(o64, o32, b, tol, 5000, inner_tol=inner_tol)
        assert info["converged"] and info["restarts"] == restarts and restarts >= 2, (info, restarts)
        assert len(info["deltas"]) == restarts
        # a delta above inner_tol is tol |b| / |r| with |r| at the fp32 rounding floor of the previous inner solve, which
        # depends on the rounding order of the two operator implementations: same value within a factor 1.5
        for dg, dw in zip(info["deltas"], deltas):
            assert dg == dw if dw == inner_tol else (dg > inner_tol and 1 / 1.5 < dg / dw < 1.5), (info["deltas"], deltas)
        assert all(abs(a - b_) <= 1 for a, b_ in zip(info["per_restart"], inner)), (info["per_restart"], inner)
        assert rel(xo.reshape(-1), x) < 1e-7


def test_zero_rhs_and_zero_links(oracle_built):
    o = make(MOEB, np.zeros(tuple(reversed(DIMS)) + (4, 3, 3), dtype=complex))
    f = inputs.source_full(DIMS, LS, 3)
    assert np.abs(o.dhop(f, 2)).max() == 0          # all links cut: Dhop vanishes, M is site-local
    e, od = split(f, DIMS)
    assert rel(o.mpc(od), o.mooee(od)) == 0
    x, info = cg(o, np.zeros_like(od), 1e-10, 10)
    assert info["iters"] == 0 and np.abs(x).max() == 0
