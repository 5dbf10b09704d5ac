"""Dense Kronecker-product construction of the DWF operator on tiny lattices.

Independent of oracle/ (no shared code): the matrices are assembled from shift
matrices, s-matrices and gamma matrices (SURVEY.md §8(c) "Dense recipe"), so that a
wrong sign, index or transposed operand in the loop oracle shows up as a mismatch.
Index order of every dense matrix: (site lex, s, spin, colour), the flattening of the
canonical FULL layout.
"""
import numpy as np

I2 = np.eye(2)
# chiral basis, gamma5 = diag(1,1,-1,-1) (C1)
GX = np.array([[0, 0, 0, 1j], [0, 0, 1j, 0], [0, -1j, 0, 0], [-1j, 0, 0, 0]])
GY = np.array([[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]], dtype=complex)
GZ = np.array([[0, 0, 1j, 0], [0, 0, 0, -1j], [-1j, 0, 0, 0], [0, 1j, 0, 0]])
GT = np.array([[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]], dtype=complex)
GAMMA = [GX, GY, GZ, GT]
G5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(complex)
PP = (np.eye(4) + G5) / 2
PM = (np.eye(4) - G5) / 2


def lex(x, dims):
    Lx, Ly, Lz, Lt = dims
    return ((x[3] * Lz + x[2]) * Ly + x[1]) * Lx + x[0]


def sites(dims):
    Lx, Ly, Lz, Lt = dims
    for t in range(Lt):
        for z in range(Lz):
            for y in range(Ly):
                for x in range(Lx):
                    yield (x, y, z, t)


def cut_gauge(U, dims, cut):
    """C7: zero U_mu(x) where x_mu mod B == B-1."""
    U = U.copy()
    for x in sites(dims):
        for mu in range(4):
            B = cut[mu]
            if B > 0 and x[mu] % B == B - 1:
                U[x[3], x[2], x[1], x[0], mu] = 0
    return U


def dhop4(U, dims, antiperiodic_t=True, dagger=False):
    """(12 V4)^2 matrix: block (x, x+mu) = (1-g_mu) (x) U_mu(x), block (x, x-mu) = (1+g_mu) (x) U_mu(x-mu)^dag."""
    V = int(np.prod(dims))
    D = np.zeros((V, 12, V, 12), dtype=complex)
    sg = -1.0 if dagger else 1.0
    for x in sites(dims):
        ix = lex(x, dims)
        for mu in range(4):
            xp = list(x); xp[mu] = (x[mu] + 1) % dims[mu]
            xm = list(x); xm[mu] = (x[mu] - 1) % dims[mu]
            bcp = -1.0 if (antiperiodic_t and mu == 3 and x[3] == dims[3] - 1) else 1.0
            bcm = -1.0 if (antiperiodic_t and mu == 3 and x[3] == 0) else 1.0
            Uf = U[x[3], x[2], x[1], x[0], mu]
            Ub = U[xm[3], xm[2], xm[1], xm[0], mu].conj().T
            D[ix, :, lex(xp, dims), :] += bcp * np.kron(np.eye(4) - sg * GAMMA[mu], Uf)
            D[ix, :, lex(xm, dims), :] += bcm * np.kron(np.eye(4) + sg * GAMMA[mu], Ub)
    return D.reshape(V * 12, V * 12)


def s_shifts(Ls, mf):
    up = np.zeros((Ls, Ls)); dn = np.zeros((Ls, Ls))
    for s in range(Ls):
        if s + 1 < Ls:
            up[s, s + 1] = 1
        else:
            up[s, 0] = -mf
        if s - 1 >= 0:
            dn[s, s - 1] = 1
        else:
            dn[s, Ls - 1] = -mf
    return up, dn


def lift5(D4, V, Ls):
    """4-D matrix acting identically on every s-slice, 5-D index order (site, s, spin*colour)."""
    D = D4.reshape(V, 12, V, 12)
    return np.einsum("xiyj,st->xsiytj", D, np.eye(Ls)).reshape(V * Ls * 12, V * Ls * 12)


def Qmat(V, Ls, mf):
    up, dn = s_shifts(Ls, mf)
    q = np.kron(up, PM) + np.kron(dn, PP)
    return np.kron(np.eye(V), np.kron(q, np.eye(3)))


def dwf_matrix(U, dims, Ls, M5, mf, b5, c5, antiperiodic_t=True):
    """M = (b5 D_W + 1) + (c5 D_W - 1) Q, D_W = (4-M5) - Dhop/2   (C4)."""
    V = int(np.prod(dims))
    N = V * Ls * 12
    DW = lift5((4.0 - M5) * np.eye(V * 12) - 0.5 * dhop4(U, dims, antiperiodic_t), V, Ls)
    Q = Qmat(V, Ls, mf)
    return (b5 * DW + np.eye(N)) + (c5 * DW - np.eye(N)) @ Q


def parity_index(dims, Ls):
    """Indices (into the 5-D dense vector) of even and odd sites, each in lex order."""
    ev, od = [], []
    for x in sites(dims):
        base = lex(x, dims) * Ls * 12
        (od if (sum(x) & 1) else ev).extend(range(base, base + Ls * 12))
    return np.array(ev), np.array(od)


def domain_index(dims, Ls, mu, B):
    """Omega = blocks with even block index along mu (x_mu // B even), Omega_bar = the rest."""
    om, ob = [], []
    for x in sites(dims):
        base = lex(x, dims) * Ls * 12
        ((om if (x[mu] // B) % 2 == 0 else ob)).extend(range(base, base + Ls * 12))
    return np.array(om), np.array(ob)


def Gamma5R5(V, Ls):
    R5 = np.eye(Ls)[::-1]
    return np.kron(np.eye(V), np.kron(R5, np.kron(G5, np.eye(3))))


def domains_from_matrices(M, Mcut, dims, Ls):
    """Omega / Omegabar read off the dense operators alone (eqs. 1-4): the sites fall into the connected
    components of the Dirichlet-cut operator Mcut (its blocks), and every link that the cut removed (a non-zero site block
    of M - Mcut) must join the two domains, which 2-colours the blocks; the block holding the origin is in Omega.
    Returns (om, ob) index arrays into the 5-D dense vector, or raises if no such colouring exists."""
    V = int(np.prod(dims))
    n = Ls * 12

    def site_adj(A):
        return np.abs(A.reshape(V, n, V, n)).max(axis=(1, 3)) > 0

    conn, removed = site_adj(Mcut), site_adj(M - Mcut)
    comp = -np.ones(V, dtype=int)
    nc = 0
    for s0 in range(V):
        if comp[s0] >= 0:
            continue
        stack = [s0]
        comp[s0] = nc
        while stack:
            a = stack.pop()
            for b in np.nonzero(conn[a])[0]:
                if comp[b] < 0:
                    comp[b] = nc
                    stack.append(b)
        nc += 1
    colour = -np.ones(nc, dtype=int)
    colour[comp[0]] = 0
    changed = True
    while changed:
        changed = False
        for a, b in zip(*np.nonzero(removed)):
            ca, cb = comp[a], comp[b]
            if colour[ca] >= 0 and colour[cb] < 0:
                colour[cb] = 1 - colour[ca]
                changed = True
            elif colour[ca] >= 0 and colour[cb] >= 0 and colour[ca] == colour[cb]:
                raise ValueError("a cut link joins two blocks of the same domain")
    assert (colour >= 0).all()
    site_dom = colour[comp]
    om = np.concatenate([np.arange(s * n, (s + 1) * n) for s in range(V) if site_dom[s] == 0])
    ob = np.concatenate([np.arange(s * n, (s + 1) * n) for s in range(V) if site_dom[s] == 1])
    return om, ob, nc
