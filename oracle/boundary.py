"""ORACLE -- TEST INFRASTRUCTURE ONLY.  The paper's boundary operator, plain numpy on canonical
FULL fields psi[t,z,y,x,s,spin,colour], written from eqs. 1-4 and 8-14 and the implementation
notes PAPER.md:175-177.  Nothing here is shared with, or imported by, the CUDA path.

Partition (eqs. 1-2): with Dirichlet block lengths B_mu (cut[mu], 0 = direction not cut) a site belongs to Omega when
sum_mu floor(x_mu / B_mu) over the cut directions is even, else to Omegabar (L_mu / B_mu must be even, so that every cut
link joins the two domains).  Block form (eq. 3): D = [[D_O, D_d], [D_dbar, D_Ob]], D_dbar = P_Ob D P_O maps Omega to
Omegabar; the hatted operators of eq. 4 are these blocks zero-padded to the whole lattice.

Projector (eq. 8): P_dbar projects on the components of Omega that D_dbar touches, D_dbar P = D_dbar.  It
is found as the paper says, "mask and shift by one in each direction": a site y of Omega whose forward
link in a cut direction mu is cut (y_mu mod B = B-1) is read by x = y + mu through (1 + gamma_mu) U^dag psi(y); one whose
backward link is cut (y_mu mod B = 0) is read by x = y - mu through (1 - gamma_mu) U psi(y).
Reading where the paper is silent ("P_dbar"): for Shamir (c5 = 0) and a site on exactly one cut
face the projector is the boundary mask times (1 +- gamma_mu)/2 -- the minimal one; for Moebius (c5 != 0: D_dbar =
-1/2 Dhop A, and A = b5 + c5 Q mixes s and chirality) and for sites on several cut faces it is the boundary mask times the
identity in spin and s, the smallest coordinate projector that contains the minimal one.  Eqs. 13-14 hold for any
projector with D_dbar P = D_dbar (R R^-1 = P follows from X P = X, X = D_O^-1 D_d D_Ob^-1 D_dbar).

    R    phi = P phi - P D_O^-1 D_d D_Ob^-1 D_dbar phi        (eqs. 9-10)
    R^-1 phi = P phi - P D^-1 D_dbar_hat phi                  (eqs. 13-14)
"""
from __future__ import annotations

import numpy as np

from .dwf_oracle import Oracle, solve_redblack


class Boundary:
    def __init__(self, dims, Ls, M5, mf, b5, c5, cut, U, antiperiodic_t=True):
        self.dims, self.Ls, self.cut = tuple(dims), int(Ls), tuple(int(c) for c in cut)
        assert any(self.cut)
        for L, B in zip(self.dims, self.cut):
            assert B == 0 or (L % B == 0 and (L // B) % 2 == 0), "every cut direction needs an even number of blocks"
        self.shamir = (c5 == 0.0)
        self.full = Oracle(dims, Ls, M5, mf, b5, c5, antiperiodic_t=antiperiodic_t).set_gauge(U)
        self.dir = Oracle(dims, Ls, M5, mf, b5, c5, antiperiodic_t=antiperiodic_t, cut=cut).set_gauge(U)
        Lx, Ly, Lz, Lt = self.dims
        t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
        self.coord = (x, y, z, t)
        blk = np.zeros_like(x)
        for mu in range(4):
            if self.cut[mu]:
                blk = blk + self.coord[mu] // self.cut[mu]
        self.omega = (blk % 2 == 0)                                   # [t,z,y,x]

    # ---- projectors --------------------------------------------------------------------------------------------
    def _site(self, m):
        return m.reshape(m.shape + (1, 1, 1))

    def P_domain(self, psi, omega=True):
        return np.where(self._site(self.omega if omega else ~self.omega), psi, 0.0)

    def faces(self):
        """list of (mask[t,z,y,x], mu, sign): sites of Omega whose forward (sign +1) / backward (-1) link in mu is cut."""
        out = []
        for mu in range(4):
            B = self.cut[mu]
            if not B:
                continue
            c = self.coord[mu] % B
            out.append((self.omega & (c == B - 1), mu, +1))
            out.append((self.omega & (c == 0), mu, -1))
        return out

    def P_boundary(self, psi):
        """P_dbar psi (eq. 8; reading above)."""
        faces = self.faces()
        nface = sum(m.astype(int) for m, _, _ in faces)
        out = np.zeros_like(psi)
        many = nface > 1
        if not self.shamir:
            many = nface > 0
        out += np.where(self._site(many), psi, 0.0)
        if self.shamir:
            for m, mu, sg in faces:
                one = m & (nface == 1)
                proj = 0.5 * (np.eye(4) + sg * self.full.gamma(mu))
                out += np.where(self._site(one), np.einsum("ab,...bc->...ac", proj, psi), 0.0)
        return out

    # ---- blocks ------------------------------------------------------------------------------------------------
    def D_dbar_hat(self, psi):
        """P_Ob D P_O psi (eqs. 3-4)."""
        return self.P_domain(self.full.M(self.P_domain(psi, True)), False)

    def D_d_hat(self, psi):
        """P_O D P_Ob psi."""
        return self.P_domain(self.full.M(self.P_domain(psi, False)), True)

    # ---- eqs. 13-14 (R^-1) and eqs. 9-10 (R) -------------------------------------------------------------------------------------------
    def R_inv(self, phi, tol=1e-12, max_iter=20000):
        u = self.D_dbar_hat(phi)
        v, info = solve_redblack(self.full, u, tol, max_iter)
        assert info["converged"]
        return self.P_boundary(phi) - self.P_boundary(v)

    def R(self, phi, tol=1e-12, max_iter=20000):
        u = self.D_dbar_hat(phi)                                       # on Omegabar
        v, i1 = solve_redblack(self.dir, u, tol, max_iter)             # D_Ob^-1 u  (the cut operator is D_O + D_Ob)
        w = self.D_d_hat(v)                                            # on Omega
        z, i2 = solve_redblack(self.dir, w, tol, max_iter)             # D_O^-1 w
        assert i1["converged"] and i2["converged"]
        return self.P_boundary(phi) - self.P_boundary(z)
