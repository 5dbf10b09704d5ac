"""Seeded synthetic inputs shared by the oracle side and the CUDA side.

This module holds NONE of the method's arithmetic (no Dirac operator, no
projector, no solver): it only draws numbers and shapes them into SU(3) links
and Gaussian spinors, in the canonical interchange layouts of DESIGN.md §3.

Synthetic gauge fields stand in for the paper's Iwasaki beta=2.13 ensemble
(not in the container); recipes follow BASELINE.json `configs`
and SURVEY.md §8(d).

Canonical layouts (fp64, C order):
  gauge   U[t, z, y, x, mu, row, col]  complex128, mu = 0..3 = x,y,z,t,
          U_mu(x) is the link from x to x+mu_hat   (18 reals per link)
  spinor  psi[t, z, y, x, s, spin, colour] complex128 (FULL), or
          psi[cb, s, spin, colour] for one parity, cb = lex/2 with
          lex = ((t*Lz+z)*Ly+y)*Lx+x and parity = (x+y+z+t) mod 2.
All RNG is counter-based (Philox keyed by the seed) so values do not depend on
thread count or call order.
"""
from __future__ import annotations

import dataclasses
import numpy as np


# --------------------------------------------------------------------------
# workload table (BASELINE.json configs[0..4] -> c1..c5)
# --------------------------------------------------------------------------
@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    dims: tuple            # (Lx, Ly, Lz, Lt)
    Ls: int
    M5: float
    mf: float
    b5: float
    c5: float
    cut: tuple             # Dirichlet block length per direction, 0 = no cut
    gauge: str             # "weak" (exp(i eps H)) or "haar_ape"
    eps: float
    tol: float
    gauge_seed: int
    source_seed: int
    antiperiodic_t: bool = True

    @property
    def V4(self):
        return int(np.prod(self.dims))


CONFIGS = {
    "c1": Config("c1", (4, 4, 4, 4), 8, 1.8, 0.1, 1.0, 0.0, (0, 0, 0, 0), "weak", 0.2, 1e-10, 1001, 2001),
    "c2": Config("c2", (16, 16, 16, 16), 16, 1.8, 0.01, 1.5, 0.5, (0, 0, 0, 8), "weak", 0.3, 1e-10, 1002, 2002),
    "c3": Config("c3", (24, 24, 24, 24), 16, 1.8, 0.01, 1.5, 0.5, (0, 0, 0, 0), "weak", 0.5, 1e-10, 1003, 2003),
    "c4": Config("c4", (32, 32, 32, 32), 12, 1.8, 0.005, 1.5, 0.5, (0, 0, 0, 0), "weak", 0.7, 1e-8, 1004, 2004),
    "c5": Config("c5", (32, 32, 32, 64), 16, 1.8, 0.005, 1.5, 0.5, (0, 0, 0, 32), "haar_ape", 0.0, 1e-8, 1005, 2005),
}


def small_variant(cfg: Config, dims, Ls=None, cut=None) -> Config:
    """Same physics parameters on a smaller lattice (for oracle-speed parity cases)."""
    return dataclasses.replace(cfg, name=cfg.name + "_small", dims=tuple(dims),
                               Ls=cfg.Ls if Ls is None else Ls,
                               cut=cfg.cut if cut is None else tuple(cut))


# --------------------------------------------------------------------------
# RNG
# --------------------------------------------------------------------------
def _rng(seed: int, stream: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed), int(stream)]))


def complex_gaussian(shape, seed: int, stream: int = 0) -> np.ndarray:
    """N(0,1) + i N(0,1), complex128."""
    g = _rng(seed, stream)
    re = g.standard_normal(shape)
    im = g.standard_normal(shape)
    return re + 1j * im


# --------------------------------------------------------------------------
# SU(3) helpers (input shaping only)
# --------------------------------------------------------------------------
def reunitarise(U: np.ndarray) -> np.ndarray:
    """Row Gram-Schmidt on rows 0,1; row 2 = conj(row0 x row1). Shape (...,3,3)."""
    r0 = U[..., 0, :]
    r1 = U[..., 1, :]
    r0 = r0 / np.sqrt(np.sum(np.abs(r0) ** 2, axis=-1, keepdims=True))
    r1 = r1 - r0 * np.sum(np.conj(r0) * r1, axis=-1, keepdims=True)
    r1 = r1 / np.sqrt(np.sum(np.abs(r1) ** 2, axis=-1, keepdims=True))
    r2 = np.conj(np.cross(r0, r1))
    return np.stack([r0, r1, r2], axis=-2)


def _expi_hermitian(H: np.ndarray, eps: float) -> np.ndarray:
    """exp(i eps H) for Hermitian H (...,3,3) through its eigen-decomposition."""
    w, V = np.linalg.eigh(H)
    ph = np.exp(1j * eps * w)
    return np.einsum("...ij,...j,...kj->...ik", V, ph, np.conj(V), optimize=True)


def gauge_weak(dims, eps: float, seed: int, chunk: int = 1 << 18) -> np.ndarray:
    """U = exp(i eps H), H = (G+G^dag)/2 - tr/3, G_ij = N(0,1)+iN(0,1); reunitarised.

    Returns U[t,z,y,x,mu,3,3] complex128.
    """
    Lx, Ly, Lz, Lt = dims
    n = Lx * Ly * Lz * Lt * 4
    out = np.empty((n, 3, 3), dtype=np.complex128)
    g = _rng(seed, 0)
    for lo in range(0, n, chunk):
        hi = min(n, lo + chunk)
        G = g.standard_normal((hi - lo, 3, 3)) + 1j * g.standard_normal((hi - lo, 3, 3))
        H = 0.5 * (G + np.conj(np.swapaxes(G, -1, -2)))
        tr = np.trace(H, axis1=-2, axis2=-1).real / 3.0
        H[:, 0, 0] -= tr
        H[:, 1, 1] -= tr
        H[:, 2, 2] -= tr
        out[lo:hi] = reunitarise(_expi_hermitian(H, eps))
    return out.reshape(Lt, Lz, Ly, Lx, 4, 3, 3)


def gauge_unit(dims) -> np.ndarray:
    Lx, Ly, Lz, Lt = dims
    U = np.zeros((Lt, Lz, Ly, Lx, 4, 3, 3), dtype=np.complex128)
    U[..., 0, 0] = U[..., 1, 1] = U[..., 2, 2] = 1.0
    return U


def gauge_haar(dims, seed: int) -> np.ndarray:
    """Haar-like SU(3): row Gram-Schmidt of a complex Gaussian 3x3, row 2 by cross product."""
    Lx, Ly, Lz, Lt = dims
    G = complex_gaussian((Lt, Lz, Ly, Lx, 4, 3, 3), seed, 0)
    return reunitarise(G)


def _shift(F: np.ndarray, mu: int, sign: int) -> np.ndarray:
    """F(x) -> F(x + sign*mu_hat), periodic. Axis order is (t,z,y,x,...)."""
    return np.roll(F, -sign, axis=3 - mu)


def _dag(M):
    return np.conj(np.swapaxes(M, -1, -2))


def ape_smear(U: np.ndarray, alpha: float = 0.5, passes: int = 4) -> np.ndarray:
    """U' = Proj[(1-alpha) U + (alpha/6) sum staples], Proj = row Gram-Schmidt."""
    for _ in range(passes):
        new = np.empty_like(U)
        for mu in range(4):
            Umu = U[..., mu, :, :]
            st = np.zeros_like(Umu)
            for nu in range(4):
                if nu == mu:
                    continue
                Unu = U[..., nu, :, :]
                # upper staple: U_nu(x) U_mu(x+nu) U_nu(x+mu)^dag
                st += Unu @ _shift(Umu, nu, +1) @ _dag(_shift(Unu, mu, +1))
                # lower staple: U_nu(x-nu)^dag U_mu(x-nu) U_nu(x-nu+mu)
                Unu_m = _shift(Unu, nu, -1)
                st += _dag(Unu_m) @ _shift(Umu, nu, -1) @ _shift(Unu_m, mu, +1)
            new[..., mu, :, :] = reunitarise((1.0 - alpha) * Umu + (alpha / 6.0) * st)
        U = new
    return U


def make_gauge(cfg: Config) -> np.ndarray:
    if cfg.gauge == "weak":
        return gauge_weak(cfg.dims, cfg.eps, cfg.gauge_seed)
    if cfg.gauge == "haar_ape":
        return ape_smear(gauge_haar(cfg.dims, cfg.gauge_seed), alpha=0.5, passes=4)
    raise ValueError(cfg.gauge)


def plaquette(U: np.ndarray) -> float:
    """Average of Re tr U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag / 3 (input fingerprint)."""
    tot, n = 0.0, 0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            Um, Un = U[..., mu, :, :], U[..., nu, :, :]
            P = Um @ _shift(Un, mu, +1) @ _dag(_shift(Um, nu, +1)) @ _dag(Un)
            tot += np.trace(P, axis1=-2, axis2=-1).real.mean() / 3.0
            n += 1
    return tot / n


# --------------------------------------------------------------------------
# spinor sources
# --------------------------------------------------------------------------
def source_full(dims, Ls: int, seed: int) -> np.ndarray:
    """Complex Gaussian psi[t,z,y,x,s,4,3]."""
    Lx, Ly, Lz, Lt = dims
    return complex_gaussian((Lt, Lz, Ly, Lx, Ls, 4, 3), seed, 1)


def parity_mask(dims) -> np.ndarray:
    """(x+y+z+t) mod 2 as an int array [t,z,y,x]."""
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return ((x + y + z + t) & 1).astype(np.int8)


def split_parity(full: np.ndarray, dims):
    """FULL field [t,z,y,x,...] -> (even, odd) half fields [cb,...] in lex order."""
    pm = parity_mask(dims).reshape(-1)
    flat = full.reshape((pm.size,) + full.shape[4:])
    return np.ascontiguousarray(flat[pm == 0]), np.ascontiguousarray(flat[pm == 1])


def merge_parity(even: np.ndarray, odd: np.ndarray, dims) -> np.ndarray:
    Lx, Ly, Lz, Lt = dims
    pm = parity_mask(dims).reshape(-1)
    flat = np.empty((pm.size,) + even.shape[1:], dtype=even.dtype)
    flat[pm == 0] = even
    flat[pm == 1] = odd
    return flat.reshape((Lt, Lz, Ly, Lx) + even.shape[1:])


def source_half(dims, Ls: int, seed: int, parity: int = 1) -> np.ndarray:
    """Complex Gaussian half field [cb,s,4,3] (the given parity of source_full)."""
    e, o = split_parity(source_full(dims, Ls, seed), dims)
    return o if parity else e
