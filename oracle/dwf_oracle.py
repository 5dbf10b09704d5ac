"""ORACLE — TEST INFRASTRUCTURE ONLY.  Python face of oracle/dwf_oracle.c plus the solvers.

Operators run in the plain C loops of dwf_oracle.c (one function per definition);
the Krylov solvers below are written out step by step in the order of
SURVEY.md §8(c) C8 (CG on Mpc^dag Mpc), C9 (fp32-inner / fp64-outer defect
correction) and C6 (red-black wrap of M psi = eta; "usual red-black
preconditioned").  Nothing here is shared with, or imported by, the CUDA path.

Fields are complex numpy arrays in the canonical layouts:
    FULL  psi[t,z,y,x,s,spin,colour]     half  psi[cb,s,spin,colour]
    gauge U[t,z,y,x,mu,row,col]
"""
from __future__ import annotations

import ctypes
import os
import numpy as np

from . import build as _build


class _Params(ctypes.Structure):
    _fields_ = [("L", ctypes.c_int * 4), ("Ls", ctypes.c_int),
                ("M5", ctypes.c_double), ("mf", ctypes.c_double),
                ("b5", ctypes.c_double), ("c5", ctypes.c_double),
                ("antiperiodic_t", ctypes.c_int)]


_LIBS = {}


def _lib(prec: str):
    if prec not in _LIBS:
        _build.build()
        _LIBS[prec] = ctypes.CDLL(_build.lib_path(prec))
        _LIBS[prec].__getattr__(f"orc_norm2_{prec}").restype = ctypes.c_double
    return _LIBS[prec]


class Oracle:
    """Moebius/Shamir DWF operator on one lattice, canonical layouts, CPU."""

    def __init__(self, dims, Ls, M5, mf, b5, c5, antiperiodic_t=True, cut=(0, 0, 0, 0), prec="f64"):
        assert prec in ("f64", "f32")
        self.dims = tuple(int(d) for d in dims)
        assert all(d % 2 == 0 for d in self.dims)
        self.Ls, self.M5, self.mf, self.b5, self.c5 = int(Ls), float(M5), float(mf), float(b5), float(c5)
        self.cut = tuple(int(c) for c in cut)
        for d, c in zip(self.dims, self.cut):
            assert c == 0 or d % c == 0
        self.prec = prec
        self.cdtype = np.complex128 if prec == "f64" else np.complex64
        self.lib = _lib(prec)
        self.p = _Params((ctypes.c_int * 4)(*self.dims), self.Ls, self.M5, self.mf, self.b5, self.c5,
                         1 if antiperiodic_t else 0)
        self.V4 = int(np.prod(self.dims))
        self.U = None

    # ---- helpers -------------------------------------------------------
    def _fn(self, name):
        return getattr(self.lib, f"{name}_{self.prec}")

    def _c(self, a):
        a = np.ascontiguousarray(a, dtype=self.cdtype)
        return a

    @staticmethod
    def _ptr(a):
        return a.ctypes.data_as(ctypes.c_void_p)

    def full_shape(self):
        Lx, Ly, Lz, Lt = self.dims
        return (Lt, Lz, Ly, Lx, self.Ls, 4, 3)

    def half_shape(self):
        return (self.V4 // 2, self.Ls, 4, 3)

    # ---- gauge ---------------------------------------------------------
    def set_gauge(self, U):
        """Stores the Dirichlet-cut gauge field (C7); U[t,z,y,x,mu,3,3]."""
        U = self._c(U)
        assert U.shape == tuple(reversed(self.dims)) + (4, 3, 3)
        out = np.empty_like(U)
        cut = (ctypes.c_int * 4)(*self.cut)
        self._fn("orc_apply_cut")(ctypes.byref(self.p), cut, self._ptr(U), self._ptr(out))
        self.U = out
        return self

    # ---- operators -----------------------------------------------------
    def dhop(self, psi, out_parity=2, dagger=False):
        psi = self._c(psi)
        assert psi.shape == (self.full_shape() if out_parity == 2 else self.half_shape())
        out = np.empty_like(psi)
        self._fn("orc_dhop")(ctypes.byref(self.p), self._ptr(self.U), self._ptr(psi), self._ptr(out),
                             int(out_parity), int(bool(dagger)))
        return out

    def _site_local(self, name, psi, dagger):
        psi = self._c(psi)
        n4 = psi.size // (self.Ls * 12)
        out = np.empty_like(psi)
        self._fn(name)(ctypes.byref(self.p), ctypes.c_long(n4), self._ptr(psi), self._ptr(out), int(bool(dagger)))
        return out

    def meooe5d(self, psi, dagger=False):
        return self._site_local("orc_meooe5d", psi, dagger)

    def mooee(self, psi, dagger=False):
        return self._site_local("orc_mooee", psi, dagger)

    def mooee_inv(self, psi, dagger=False):
        return self._site_local("orc_mooee_inv", psi, dagger)

    def M(self, psi, dagger=False):
        psi = self._c(psi)
        assert psi.shape == self.full_shape()
        out = np.empty_like(psi)
        self._fn("orc_M")(ctypes.byref(self.p), self._ptr(self.U), self._ptr(psi), self._ptr(out), int(bool(dagger)))
        return out

    def meooe(self, psi, out_parity, dagger=False):
        psi = self._c(psi)
        assert psi.shape == self.half_shape()
        out = np.empty_like(psi)
        self._fn("orc_meooe")(ctypes.byref(self.p), self._ptr(self.U), self._ptr(psi), self._ptr(out),
                              int(out_parity), int(bool(dagger)))
        return out

    def mpc(self, psi, dagger=False):
        psi = self._c(psi)
        assert psi.shape == self.half_shape()
        out = np.empty_like(psi)
        self._fn("orc_mpc")(ctypes.byref(self.p), self._ptr(self.U), self._ptr(psi), self._ptr(out), int(bool(dagger)))
        return out

    def mdagm(self, psi):
        psi = self._c(psi)
        out = np.empty_like(psi)
        self._fn("orc_mdagm")(ctypes.byref(self.p), self._ptr(self.U), self._ptr(psi), self._ptr(out))
        return out

    def gamma(self, mu):
        """The oracle's 4x4 gamma_mu (C1), for the Clifford-algebra pin."""
        out = np.zeros((4, 4, 2))
        self._fn("orc_gamma")(int(mu), self._ptr(out))
        return out[..., 0] + 1j * out[..., 1]

    def norm2(self, v):
        """sum |v|^2, accumulated in fp64 whatever the field precision (C8)."""
        v = np.ascontiguousarray(v)
        return float(self._fn("orc_norm2")(self._ptr(v), ctypes.c_long(v.size * 2)))


# ---------------------------------------------------------------------------
# C8: CG on A = Mpc^dag Mpc
# ---------------------------------------------------------------------------
def cg(orc: Oracle, b, tol, max_iter, x0=None, history=None, restart_on_true=True):
    """r=b-Ax, p=r, c=|r|^2; loop: q=Mpc p; d=|q|^2; alpha=c/d; x+=alpha p;
    r-=alpha Mpc^dag q; c'=|r|^2; stop if c' <= tol^2 |b|^2; beta=c'/c; p=r+beta p.

    If the true residual exceeds tol at exit the solve restarts from the current x
    (C8 reading of "true residual <= stated tolerance"); all iterations are counted.
    Returns (x, info) with info = dict(iters, resid_iter, resid_true, restarts, converged).
    """
    b = np.ascontiguousarray(b, dtype=orc.cdtype)
    x = np.zeros_like(b) if x0 is None else np.array(x0, dtype=orc.cdtype, copy=True)
    bnorm2 = orc.norm2(b)
    if bnorm2 == 0.0:
        return np.zeros_like(b), dict(iters=0, resid_iter=0.0, resid_true=0.0, restarts=0, converged=True)
    target = tol * tol * bnorm2
    rdt = np.float64 if orc.prec == "f64" else np.float32
    iters, restarts = 0, 0
    resid_iter = resid_true = float("inf")
    converged = False
    while True:
        r = b - orc.mdagm(x) if (x0 is not None or restarts > 0) else b.copy()
        p = r.copy()
        c = orc.norm2(r)
        resid_iter = np.sqrt(c / bnorm2)
        inner_done = c <= target
        while not inner_done and iters < max_iter:
            q = orc.mpc(p)
            d = orc.norm2(q)
            alpha = rdt(c / d)
            x += alpha * p
            r -= alpha * orc.mpc(q, dagger=True)
            cn = orc.norm2(r)
            iters += 1
            resid_iter = np.sqrt(cn / bnorm2)
            if history is not None:
                history.append(resid_iter)
            if cn <= target:
                inner_done = True
                break
            beta = rdt(cn / c)
            p = r + beta * p
            c = cn
        resid_true = np.sqrt(orc.norm2(b - orc.mdagm(x)) / bnorm2)
        if resid_true <= tol:
            converged = True
            break
        if iters >= max_iter or not restart_on_true:
            break
        restarts += 1
    return x, dict(iters=iters, resid_iter=float(resid_iter), resid_true=float(resid_true),
                   restarts=restarts, converged=converged)


# ---------------------------------------------------------------------------
# NEXT-2: multishift CG on A + sigma_i, A = Mpc^dag Mpc -- the solver behind the rational
# functions of D^dag D in the DD-RHMC one-flavour action (eqs. 20-21)
# ---------------------------------------------------------------------------
def multishift_cg(orc: Oracle, b, shifts, tol, max_iter):
    """Solves (A + sigma_i) x_i = b for all shifts with ONE Krylov space (Jegerlehner, hep-lat/9612014), written out
    in the CG form of C8.  The base system is the smallest shift sigma_0 (slowest to converge), delta_i = sigma_i - sigma_0;
    the residual of system i is zeta_i r, so only r is stored:
        q = (A + sigma_0) p_0; d = <p_0, q>; alpha = c/d
        zeta_i' = zeta_i zeta_i^old alpha^old / (alpha beta^old (zeta_i^old - zeta_i) + zeta_i^old alpha^old (1 + delta_i alpha))
        x_i += alpha (zeta_i'/zeta_i) p_i ;  r -= alpha q ; c' = |r|^2 ; beta = c'/c
        p_i = zeta_i' r + beta (zeta_i'/zeta_i)^2 p_i
    stops when |r| <= tol |b| for the base system.  Returns ([x_i], info) with the true residual of every system."""
    b = np.ascontiguousarray(b, dtype=np.complex128)
    shifts = [float(s) for s in shifts]
    assert all(shifts[i] <= shifts[i + 1] for i in range(len(shifts) - 1)), "shifts ascending"
    n = len(shifts)
    s0 = shifts[0]
    delta = [s - s0 for s in shifts]
    bn2 = orc.norm2(b)
    x = [np.zeros_like(b) for _ in shifts]
    if bn2 == 0.0:
        return x, dict(iters=0, resid_true=[0.0] * n, converged=True)
    r = b.copy()
    p = [b.copy() for _ in shifts]
    zeta, zeta_old = [1.0] * n, [1.0] * n
    alpha_old, beta_old = 1.0, 0.0
    c = bn2
    target = tol * tol * bn2
    iters = 0
    while c > target and iters < max_iter:
        q = orc.mdagm(p[0]) + s0 * p[0]
        d = float(np.real(np.vdot(p[0], q)))
        alpha = c / d
        znew = [0.0] * n
        for i in range(n):
            znew[i] = zeta[i] * zeta_old[i] * alpha_old / (
                alpha * beta_old * (zeta_old[i] - zeta[i]) + zeta_old[i] * alpha_old * (1.0 + delta[i] * alpha))
            x[i] += (alpha * znew[i] / zeta[i]) * p[i]
        r -= alpha * q
        cn = orc.norm2(r)
        beta = cn / c
        for i in range(n):
            p[i] = znew[i] * r + (beta * (znew[i] / zeta[i]) ** 2) * p[i]
        zeta_old, zeta, alpha_old, beta_old, c = zeta, znew, alpha, beta, cn
        iters += 1
    res = [float(np.sqrt(orc.norm2(b - orc.mdagm(x[i]) - shifts[i] * x[i]) / bn2)) for i in range(n)]
    return x, dict(iters=iters, resid_iter=float(np.sqrt(c / bn2)), resid_true=res, converged=bool(c <= target))


# ---------------------------------------------------------------------------
# NEXT-4: Chebyshev polynomial of A = Mpc^dag Mpc applied to a vector -- the "filter functions ... which
# can be obtained recursively" of the paper's multigrid set-up (Fig. 4 caption PAPER.md:191).  The paper
# gives neither window nor order: both are arguments.
# ---------------------------------------------------------------------------
def chebyshev(orc: Oracle, v, lo, hi, order):
    """T_n(a) v with a = (2A - (hi + lo)) / (hi - lo), by the three-term recurrence
    t_0 = v, t_1 = a v, t_{k+1} = 2 a t_k - t_{k-1}."""
    v = np.ascontiguousarray(v, dtype=np.complex128)
    s, o = 2.0 / (hi - lo), -(hi + lo) / (hi - lo)
    amul = lambda x: s * orc.mdagm(x) + o * x
    if order == 0:
        return v.copy()
    t0, t1 = v, amul(v)
    for _ in range(order - 1):
        t0, t1 = t1, 2.0 * amul(t1) - t0
    return t1


# ---------------------------------------------------------------------------
# C9: fp32 inner / fp64 outer defect correction
# ---------------------------------------------------------------------------
def cg_mixed(orc64: Oracle, orc32: Oracle, b, tol, max_iter, inner_tol=1e-4, max_restarts=20, x0=None):
    """outer (fp64): r = b - A x; stop if |r| <= tol |b|; inner (fp32 fields and gauge, fp64
    reductions): CG for A_f e = r_f from e = 0 to relative tolerance
    delta = max(inner_tol, tol |b| / |r|); x += e; repeat."""
    b = np.ascontiguousarray(b, dtype=np.complex128)
    x = np.zeros_like(b) if x0 is None else np.array(x0, dtype=np.complex128, copy=True)
    bnorm2 = orc64.norm2(b)
    iters_inner, restarts = 0, 0
    per_restart, deltas = [], []
    while True:
        r = b - orc64.mdagm(x)
        rn2 = orc64.norm2(r)
        resid_true = np.sqrt(rn2 / bnorm2)
        if resid_true <= tol or restarts >= max_restarts or iters_inner >= max_iter:
            break
        delta = max(inner_tol, tol * np.sqrt(bnorm2 / rn2))
        e, info = cg(orc32, r.astype(np.complex64), delta, max_iter - iters_inner, restart_on_true=False)
        iters_inner += info["iters"]
        per_restart.append(info["iters"])
        deltas.append(float(delta))
        x += e.astype(np.complex128)
        restarts += 1
    return x, dict(iters=iters_inner, iters_inner=iters_inner, restarts=restarts, resid_true=float(resid_true),
                   per_restart=per_restart, deltas=deltas, converged=bool(resid_true <= tol))


# ---------------------------------------------------------------------------
# C6: red-black solve of the full system M psi = eta
# ---------------------------------------------------------------------------
def split(full, dims):
    """FULL [t,z,y,x,...] -> (even, odd) half fields in lex order (cb = lex/2)."""
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    par = ((x + y + z + t) & 1).reshape(-1)
    flat = full.reshape((par.size,) + full.shape[4:])
    return np.ascontiguousarray(flat[par == 0]), np.ascontiguousarray(flat[par == 1])


def merge(even, odd, dims):
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    par = ((x + y + z + t) & 1).reshape(-1)
    flat = np.empty((par.size,) + even.shape[1:], dtype=even.dtype)
    flat[par == 0] = even
    flat[par == 1] = odd
    return flat.reshape((Lt, Lz, Ly, Lx) + even.shape[1:])


def solve_redblack(orc: Oracle, eta_full, tol, max_iter, orc32: Oracle | None = None):
    """eta' = eta_o - Moe Mee^{-1} eta_e; solve Mpc^dag Mpc psi_o = Mpc^dag eta';
    psi_e = Mee^{-1}(eta_e - Meo psi_o).  Returns (psi_full, info)."""
    eta_e, eta_o = split(np.asarray(eta_full, dtype=np.complex128), orc.dims)
    src = eta_o - orc.meooe(orc.mooee_inv(eta_e), 1)
    rhs = orc.mpc(src, dagger=True)
    if orc32 is None:
        psi_o, info = cg(orc, rhs, tol, max_iter)
    else:
        psi_o, info = cg_mixed(orc, orc32, rhs, tol, max_iter)
    psi_e = orc.mooee_inv(eta_e - orc.meooe(psi_o, 0))
    psi = merge(psi_e, psi_o, orc.dims)
    info = dict(info)
    info["resid_full"] = float(np.sqrt(orc.norm2(eta_full - orc.M(psi)) / orc.norm2(np.asarray(eta_full, dtype=np.complex128))))
    return psi, info
