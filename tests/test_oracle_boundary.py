"""Pins of oracle/boundary.py (the boundary projector and R, R^-1 of eqs. 8-14)
against dense linear algebra.  Geometry "t": a 2x2x2x4, Ls = 4 lattice cut in t into two 2^3 x 2 domains (every site of
Omega on exactly one cut face).  Geometry "xt": a 4x2x2x6, Ls = 2 lattice cut in x (blocks of 2) AND t (blocks of 3) into a
2 x 2 checkerboard of blocks: Omega is coloured by two block indices, the sites with t mod 3 = 1 sit on one cut face (x)
and all others on two (corner sites: the multi-face branch of Boundary.P_boundary).  The dense side (tests/dense_ref.py +
numpy SVD / solve / slogdet) shares nothing with the oracle; in "xt" even Omega is read off the dense matrices."""
import numpy as np
import pytest

import dense_ref as dr
from paper_2203_17119_b200 import inputs

GEOMS = {"t": ((2, 2, 2, 4), 4, (0, 0, 0, 2)), "xt": ((4, 2, 2, 6), 2, (2, 0, 0, 3))}
MOEB = dict(M5=1.8, mf=0.05, b5=1.5, c5=0.5)
SHAM = dict(M5=1.8, mf=0.1, b5=1.0, c5=0.0)


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a).ravel() - np.asarray(b).ravel()) / np.linalg.norm(np.asarray(b).ravel()))


@pytest.fixture(scope="module", params=["t-shamir", "t-moebius", "xt-shamir", "xt-moebius"])
def setup(request, oracle_built):
    from oracle.boundary import Boundary
    geom, kind = request.param.split("-")
    DIMS, LS, CUT = GEOMS[geom]
    par = SHAM if kind == "shamir" else MOEB
    U = inputs.gauge_weak(DIMS, 0.4, 77)
    bd = Boundary(DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"], CUT, U)
    M = dr.dwf_matrix(U, DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    Mcut = dr.dwf_matrix(dr.cut_gauge(U, DIMS, CUT), DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    om, ob, nblocks = dr.domains_from_matrices(M, Mcut, DIMS, LS)
    if geom == "t":
        om1, ob1 = dr.domain_index(DIMS, LS, 3, 2)
        assert np.array_equal(om, om1) and np.array_equal(ob, ob1) and nblocks == 2
    else:
        assert nblocks == 4
    n = M.shape[0]
    shape = (DIMS[3], DIMS[2], DIMS[1], DIMS[0], LS, 4, 3)
    # the oracle's projector as a matrix (columns = images of the unit vectors)
    P = np.zeros((n, n), dtype=complex)
    eye = np.eye(n, dtype=complex)
    for j0 in range(0, n, 96):
        for j in range(j0, min(j0 + 96, n)):
            P[:, j] = bd.P_boundary(eye[:, j].reshape(shape)).reshape(-1)
    Ddb_hat = np.zeros_like(M)
    Ddb_hat[np.ix_(ob, om)] = M[np.ix_(ob, om)]
    return dict(kind=kind, geom=geom, dims=DIMS, Ls=LS, cut=CUT, bd=bd, M=M, Mcut=Mcut, om=om, ob=ob, P=P, Ddb_hat=Ddb_hat,
                shape=shape, n=n)


def test_omega_is_the_block_colouring_of_the_dense_cut_operator(setup):
    """Boundary.omega (sum of block indices even) against the domains read off the dense matrices: the cut operator is
    block-diagonal on them (eq. 3 with D_d = D_dbar = 0) and every removed link joins Omega to Omegabar."""
    bd, om, ob, Mcut, M, shape = (setup[k] for k in ("bd", "om", "ob", "Mcut", "M", "shape"))
    mask = np.zeros(setup["n"], dtype=bool)
    mask[om] = True
    want = mask.reshape(shape)[..., 0, 0, 0]
    assert np.array_equal(bd.omega, want)
    assert np.abs(Mcut[np.ix_(om, ob)]).max() == 0 and np.abs(Mcut[np.ix_(ob, om)]).max() == 0
    diff = M - Mcut
    assert np.abs(diff[np.ix_(om, om)]).max() == 0 and np.abs(diff[np.ix_(ob, ob)]).max() == 0
    assert np.abs(diff).max() > 0


def test_projector_covers_what_D_dbar_touches(setup):
    P, Dh, om, ob = setup["P"], setup["Ddb_hat"], setup["om"], setup["ob"]
    assert np.allclose(P @ P, P, atol=1e-14) and np.allclose(P, P.conj().T, atol=1e-14)
    assert np.abs(P[np.ix_(ob, ob)]).max() == 0 and np.abs(P[np.ix_(om, ob)]).max() == 0      # lives on Omega
    assert rel(Dh @ P, Dh) < 1e-14                                                              # eq. 8: D_dbar P = D_dbar
    # the minimal projector = orthogonal projector on the row space of D_dbar (numpy SVD)
    _, sv, Vh = np.linalg.svd(Dh)
    rank = int((sv > 1e-10 * sv[0]).sum())
    Pmin = Vh[:rank].conj().T @ Vh[:rank]
    assert rel(P @ Pmin, Pmin) < 1e-12                                                          # contains it
    nbnd = len(om)                     # in both geometries every site of Omega is a boundary site (thin blocks)
    if setup["geom"] == "t":
        assert rank == nbnd // 2       # half of the face components: the (1 +- gamma_mu)/2 structure of PAPER.md:87
    elif setup["kind"] == "shamir":
        # sites on one face (t mod 3 = 1: a third of Omega) keep half of their components; corner sites are read through
        # (1 +- gamma_x) and (1 +- gamma_t), whose ranges together span the whole spinor: all components
        assert rank == (nbnd // 3) // 2 + 2 * (nbnd // 3)
    if setup["kind"] == "shamir":
        assert rel(P, Pmin) < 1e-12    # Shamir: the oracle's projector IS the minimal one, corner sites included
    else:
        assert round(np.trace(P).real) == nbnd


def test_domain_blocks_and_edge_detection(setup):
    bd, M, om, ob, shape, n = (setup[k] for k in ("bd", "M", "om", "ob", "shape", "n"))
    rng = np.random.default_rng(3)
    v = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    vO = np.zeros_like(v); vO[om] = v[om]
    vB = np.zeros_like(v); vB[ob] = v[ob]
    assert rel(bd.P_domain(v.reshape(shape), True).reshape(-1), vO) == 0
    assert rel(bd.P_domain(v.reshape(shape), False).reshape(-1), vB) == 0
    want = np.zeros_like(v); want[ob] = M[np.ix_(ob, om)] @ v[om]
    assert rel(bd.D_dbar_hat(v.reshape(shape)).reshape(-1), want) < 1e-14
    want = np.zeros_like(v); want[om] = M[np.ix_(om, ob)] @ v[ob]
    assert rel(bd.D_d_hat(v.reshape(shape)).reshape(-1), want) < 1e-14
    faces = {(mu, sg): m for m, mu, sg in bd.faces()}
    if setup["geom"] == "t":
        # mask-and-shift: t = 1 has its forward link cut, t = 0 its backward (wrap) link; t = 2, 3 are Omegabar
        assert faces[(3, +1)][1].all() and not faces[(3, +1)][[0, 2, 3]].any()
        assert faces[(3, -1)][0].all() and not faces[(3, -1)][[1, 2, 3]].any()
    else:
        # every face mask against the dense operators: y in Omega is on the (mu, +) face iff the block (y + mu, y) of
        # M - Mcut is non-zero (its forward link was cut), on the (mu, -) face iff the block (y - mu, y) is
        dims, Ls = setup["dims"], setup["Ls"]
        V, nn = int(np.prod(dims)), Ls * 12
        rem = np.abs((M - setup["Mcut"]).reshape(V, nn, V, nn)).max(axis=(1, 3)) > 0
        for (mu, sg), m in faces.items():
            for x in dr.sites(dims):
                y2 = list(x); y2[mu] = (x[mu] + sg) % dims[mu]
                want = bool(bd.omega[x[3], x[2], x[1], x[0]]) and bool(rem[dr.lex(y2, dims), dr.lex(x, dims)])
                assert bool(m[x[3], x[2], x[1], x[0]]) == want, (mu, sg, x)


def test_R_and_Rinv_eqs_13_14(setup):
    bd, M, om, ob, P, Dh, shape, n = (setup[k] for k in ("bd", "M", "om", "ob", "P", "Ddb_hat", "shape", "n"))
    DO, DOb, Dd, Ddb = M[np.ix_(om, om)], M[np.ix_(ob, ob)], M[np.ix_(om, ob)], M[np.ix_(ob, om)]
    X = np.zeros_like(M)
    X[np.ix_(om, om)] = np.linalg.solve(DO, Dd @ np.linalg.solve(DOb, Ddb))
    R = P - P @ X                                                   # eqs. 9-10
    Rinv = P - P @ np.linalg.solve(M, Dh)                           # eqs. 13-14
    assert rel(R @ Rinv, P) < 1e-11 and rel(Rinv @ R, P) < 1e-11    # "R R^-1 = P"
    rng = np.random.default_rng(5)
    phi = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    assert rel(bd.R_inv(phi.reshape(shape)).reshape(-1), Rinv @ phi) < 1e-9
    assert rel(bd.R(phi.reshape(shape)).reshape(-1), R @ phi) < 1e-9
    # eqs. 11-12: det chi = det R = det(1 - X), R taken on the range of P
    w, Vp = np.linalg.eigh(P)
    B = Vp[:, w > 0.5]
    s1, l1 = np.linalg.slogdet(B.conj().T @ R @ B)
    s2, l2 = np.linalg.slogdet(np.eye(n) - X)
    assert abs(l1 - l2) < 1e-9 and abs(s1 - s2) < 1e-9
    # eq. 6 in this language: det D = det D_O det D_Ob det R
    s, l = np.linalg.slogdet(M)
    parts = [np.linalg.slogdet(A) for A in (DO, DOb)]
    assert abs(l - (parts[0][1] + parts[1][1] + l1)) < 1e-8
