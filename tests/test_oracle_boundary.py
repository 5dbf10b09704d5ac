"""Pins of oracle/boundary.py (the boundary projector and R, R^-1 of eqs. 8-14)
against dense linear algebra on a 2x2x2x4, Ls = 4 lattice cut in t into two 2^3 x 2 domains.  The dense side
(tests/dense_ref.py + numpy SVD / solve / slogdet) shares nothing with the oracle."""
import numpy as np
import pytest

import dense_ref as dr
from paper_2203_17119_b200 import inputs

DIMS, LS, CUT = (2, 2, 2, 4), 4, (0, 0, 0, 2)
MOEB = dict(M5=1.8, mf=0.05, b5=1.5, c5=0.5)
SHAM = dict(M5=1.8, mf=0.1, b5=1.0, c5=0.0)


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a).ravel() - np.asarray(b).ravel()) / np.linalg.norm(np.asarray(b).ravel()))


@pytest.fixture(scope="module", params=["shamir", "moebius"])
def setup(request, oracle_built):
    from oracle.boundary import Boundary
    par = SHAM if request.param == "shamir" else MOEB
    U = inputs.gauge_weak(DIMS, 0.4, 77)
    bd = Boundary(DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"], CUT, U)
    M = dr.dwf_matrix(U, DIMS, LS, par["M5"], par["mf"], par["b5"], par["c5"])
    om, ob = dr.domain_index(DIMS, LS, 3, 2)
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
    return dict(kind=request.param, bd=bd, M=M, om=om, ob=ob, P=P, Ddb_hat=Ddb_hat, shape=shape, n=n)


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
    nbnd = len(om)                     # here every site of Omega is a boundary site (blocks are 2 thick)
    assert rank == nbnd // 2           # half of the face components: the (1 +- gamma_mu)/2 structure of PAPER.md:87
    if setup["kind"] == "shamir":
        assert rel(P, Pmin) < 1e-12    # Shamir: the oracle's projector IS the minimal one
    else:
        assert round(np.trace(P).real) == nbnd


def test_domain_blocks_and_edge_detection(setup):
    bd, M, om, ob, shape, n = (setup[k] for k in ("bd", "M", "om", "ob", "shape", "n"))
    rng = np.random.default_rng(3)
    v = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    vO = np.zeros_like(v); vO[om] = v[om]
    vB = np.zeros_like(v); vB[ob] = v[ob]
    assert rel(bd.P_domain(v.reshape(shape), True).reshape(-1), vO) == 0
    want = np.zeros_like(v); want[ob] = M[np.ix_(ob, om)] @ v[om]
    assert rel(bd.D_dbar_hat(v.reshape(shape)).reshape(-1), want) < 1e-14
    want = np.zeros_like(v); want[om] = M[np.ix_(om, ob)] @ v[ob]
    assert rel(bd.D_d_hat(v.reshape(shape)).reshape(-1), want) < 1e-14
    # mask-and-shift: t = 1 has its forward link cut, t = 0 its backward (wrap) link; t = 2, 3 are Omegabar
    faces = {(mu, sg): m for m, mu, sg in bd.faces()}
    assert faces[(3, +1)][1].all() and not faces[(3, +1)][[0, 2, 3]].any()
    assert faces[(3, -1)][0].all() and not faces[(3, -1)][[1, 2, 3]].any()


def test_R_and_Rinv_eqs_13_14(setup):
    bd, M, om, ob, P, Dh, shape, n = (setup[k] for k in ("bd", "M", "om", "ob", "P", "Ddb_hat", "shape", "n"))
    DO, DOb, Dd, Ddb = M[np.ix_(om, om)], M[np.ix_(ob, ob)], M[np.ix_(om, ob)], M[np.ix_(ob, om)]
    X = np.zeros_like(M)
    X[np.ix_(om, om)] = np.linalg.solve(DO, Dd @ np.linalg.solve(DOb, Ddb))
    R = P - P @ X                                                   # eq. 13
    Rinv = P - P @ np.linalg.solve(M, Dh)                           # eq. 14
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
