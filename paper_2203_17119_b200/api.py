"""Thin Python binding of the C-ABI library (include/dwf.h): argument marshalling only.

Every step of the hot path runs inside libdwf_b200.so (hand-written CUDA, sm_100a).  PyTorch is used
for device memory and streams, nothing else.  There is NO CPU fallback: importing this module
without the compiled library raises, and so does any call without a CUDA device.

Names mirror the C ABI: Dwf.dhop <-> dwf_dhop, Dwf.mooee_inv <-> dwf_mooee_inv, Dwf.mpc <-> dwf_mpc,
Dwf.mdagm <-> dwf_mdagm, Dwf.cg <-> dwf_cg, Dwf.solve <-> dwf_solve, ...
"""
from __future__ import annotations

import ctypes
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libdwf_b200.so")

F32, F64 = 0, 1
EVEN, ODD, FULL = 0, 1, 2
CG_F64, CG_MIXED = 0, 1
OK, EINVAL, ENOMEM, ECUDA, ESTATE, ENOTCONV = 0, 1, 2, 3, 4, 5

# every symbol include/dwf.h declares (tests check the library exports all of them)
SYMBOLS = [
    "dwf_create", "dwf_destroy", "dwf_set_option", "dwf_get_option", "dwf_set_stream", "dwf_set_gauge",
    "dwf_field_bytes", "dwf_pack", "dwf_unpack", "dwf_convert", "dwf_dhop", "dwf_meooe5d", "dwf_mooee",
    "dwf_mooee_inv", "dwf_m", "dwf_mpc", "dwf_mdagm", "dwf_norm2", "dwf_cg", "dwf_multishift_cg", "dwf_chebyshev", "dwf_domain_project", "dwf_boundary_op", "dwf_solve", "dwf_dhop_host",
    "dwf_mdagm_host", "dwf_cg_host", "dwf_solve_host", "dwf_launch_count", "dwf_last_error", "dwf_version",
    "dwf_mrhs_reserve", "dwf_mrhs_field_bytes", "dwf_mrhs_insert", "dwf_mrhs_extract", "dwf_dhop_mrhs", "dwf_mpc_mrhs",
    "dwf_mdagm_mrhs", "dwf_cg_mrhs", "dwf_norm2_static",
]


class CgInfo(ctypes.Structure):
    _fields_ = [("iters_total", ctypes.c_int), ("iters_inner", ctypes.c_int), ("restarts", ctypes.c_int),
                ("resid_iter", ctypes.c_double), ("resid_true", ctypes.c_double), ("resid_full", ctypes.c_double),
                ("seconds", ctypes.c_double), ("launches", ctypes.c_int)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class DwfError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"dwf status {status}: {msg}")
        self.status = status


_LIB = None


def load_library():
    """Loads libdwf_b200.so; fails loudly when it has not been built."""
    global _LIB
    if _LIB is not None:
        return _LIB
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2203_17119_b200.build` "
                          "(there is no CPU or PyTorch fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    P = ctypes.POINTER
    lib.dwf_create.argtypes = [P(vp), P(ci), ci, cd, cd, cd, cd, P(ci)]
    lib.dwf_destroy.argtypes = [vp]
    lib.dwf_set_option.argtypes = [vp, ctypes.c_char_p, cd]
    lib.dwf_get_option.argtypes = [vp, ctypes.c_char_p, P(cd)]
    lib.dwf_set_stream.argtypes = [vp, vp]
    lib.dwf_set_gauge.argtypes = [vp, vp]
    lib.dwf_field_bytes.argtypes = [vp, ci, ci]
    lib.dwf_field_bytes.restype = ctypes.c_size_t
    lib.dwf_pack.argtypes = [vp, vp, vp, ci, ci]
    lib.dwf_unpack.argtypes = [vp, vp, vp, ci, ci]
    lib.dwf_convert.argtypes = [vp, vp, ci, vp, ci, ci]
    lib.dwf_dhop.argtypes = [vp, vp, vp, ci, ci, ci]
    for name in ("dwf_meooe5d", "dwf_mooee", "dwf_mooee_inv"):
        getattr(lib, name).argtypes = [vp, vp, vp, ci, ci, ci]
    lib.dwf_m.argtypes = [vp, vp, vp, ci, ci]
    lib.dwf_mpc.argtypes = [vp, vp, vp, ci, ci]
    lib.dwf_mdagm.argtypes = [vp, vp, vp, ci]
    lib.dwf_norm2.argtypes = [vp, vp, ci, ci, P(cd)]
    lib.dwf_norm2_static.argtypes = [vp, ctypes.c_size_t, ci, vp, vp, ctypes.c_char_p, ctypes.c_size_t]
    lib.dwf_cg.argtypes = [vp, vp, vp, cd, ci, ci, ci, P(CgInfo)]
    lib.dwf_domain_project.argtypes = [vp, vp, vp, ci, ci]
    lib.dwf_boundary_op.argtypes = [vp, vp, vp, ci, cd, ci, ci, P(CgInfo)]
    lib.dwf_chebyshev.argtypes = [vp, vp, vp, cd, cd, ci, ci]
    lib.dwf_multishift_cg.argtypes = [vp, vp, vp, P(cd), ci, cd, ci, P(CgInfo), P(cd)]
    lib.dwf_solve.argtypes = [vp, vp, vp, cd, ci, ci, P(CgInfo)]
    lib.dwf_dhop_host.argtypes = [vp, vp, vp, ci, ci, ci]
    lib.dwf_mdagm_host.argtypes = [vp, vp, vp, ci]
    lib.dwf_solve_host.argtypes = [vp, vp, vp, cd, ci, ci, P(CgInfo)]
    lib.dwf_cg_host.argtypes = [vp, vp, vp, cd, ci, ci, P(CgInfo)]
    lib.dwf_mrhs_reserve.argtypes = [vp, ci]
    lib.dwf_mrhs_field_bytes.argtypes = [vp, ci, ci]
    lib.dwf_mrhs_field_bytes.restype = ctypes.c_size_t
    lib.dwf_mrhs_insert.argtypes = [vp, vp, ci, ci, vp, ci]
    lib.dwf_mrhs_extract.argtypes = [vp, vp, vp, ci, ci, ci]
    lib.dwf_dhop_mrhs.argtypes = [vp, vp, vp, ci, ci, ci, ci]
    lib.dwf_mpc_mrhs.argtypes = [vp, vp, vp, ci, ci, ci]
    lib.dwf_mdagm_mrhs.argtypes = [vp, vp, vp, ci, ci]
    lib.dwf_cg_mrhs.argtypes = [vp, vp, vp, ci, cd, ci, ci, ci, P(CgInfo)]
    lib.dwf_launch_count.argtypes = [vp]
    lib.dwf_launch_count.restype = ctypes.c_longlong
    lib.dwf_last_error.argtypes = [vp]
    lib.dwf_last_error.restype = ctypes.c_char_p
    lib.dwf_version.restype = ctypes.c_char_p
    _LIB = lib
    return lib


def _rdtype(prec):
    return torch.float64 if prec == F64 else torch.float32


def _npdtype(prec):
    return np.float64 if prec == F64 else np.float32


class Dwf:
    """One dwf_ctx.  Fields are torch CUDA tensors: `native` ones are opaque 1-D real tensors of
    dwf_field_bytes bytes; `canonical` ones have the layouts of include/dwf.h viewed as reals."""

    def __init__(self, dims, Ls, M5, mf, b5, c5, cut=(0, 0, 0, 0), device="cuda:0", **options):
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2203_17119_b200 needs a CUDA device (no CPU fallback)")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.dims, self.Ls = tuple(int(d) for d in dims), int(Ls)
        self.V4 = int(np.prod(self.dims))
        self._h = ctypes.c_void_p()
        d = (ctypes.c_int * 4)(*self.dims)
        c = (ctypes.c_int * 4)(*[int(x) for x in cut])
        st = self.lib.dwf_create(ctypes.byref(self._h), d, self.Ls, M5, mf, b5, c5, c)
        if st != OK:
            self._h = ctypes.c_void_p()
            raise DwfError(st, "dwf_create failed (bad dims / Ls / cut?)")
        for k, v in options.items():
            self.set_option(k, v)
        self.use_current_stream()

    # ---- plumbing ----------------------------------------------------------------------------
    def _chk(self, st, allow=()):
        if st != OK and st not in allow:
            raise DwfError(st, self.lib.dwf_last_error(self._h).decode())
        return st

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self.lib.dwf_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key, val):
        self._chk(self.lib.dwf_set_option(self._h, key.encode(), float(val)))

    def get_option(self, key):
        v = ctypes.c_double()
        self._chk(self.lib.dwf_get_option(self._h, key.encode(), ctypes.byref(v)))
        return v.value

    def use_current_stream(self):
        self.set_stream(torch.cuda.current_stream(self.device).cuda_stream)

    def set_stream(self, cuda_stream_handle):
        self._chk(self.lib.dwf_set_stream(self._h, ctypes.c_void_p(cuda_stream_handle)))

    def launch_count(self):
        return int(self.lib.dwf_launch_count(self._h))

    def field_bytes(self, prec, parity):
        return int(self.lib.dwf_field_bytes(self._h, prec, parity))

    def new_native(self, prec=F64, parity=ODD):
        n = self.field_bytes(prec, parity) // (8 if prec == F64 else 4)
        return torch.zeros(n, dtype=_rdtype(prec), device=self.device)

    def canonical_shape(self, parity):
        n4 = self.V4 if parity == FULL else self.V4 // 2
        return (n4, self.Ls, 4, 3, 2)

    @staticmethod
    def _p(t):
        return ctypes.c_void_p(t.data_ptr())

    # ---- gauge and layout ----------------------------------------------------------------------
    def set_gauge(self, U):
        """U: complex128 numpy [t,z,y,x,mu,3,3] or a CUDA fp64 tensor of V4*4*18 reals (canonical)."""
        if isinstance(U, np.ndarray):
            U = torch.from_numpy(np.ascontiguousarray(U, dtype=np.complex128).view(np.float64).reshape(-1))
        U = U.to(self.device, dtype=torch.float64).contiguous()
        assert U.numel() == self.V4 * 4 * 18
        self._chk(self.lib.dwf_set_gauge(self._h, self._p(U)))
        torch.cuda.current_stream(self.device).synchronize()

    def pack(self, canonical, prec=F64, parity=ODD, out=None):
        """canonical numpy complex / torch real array -> native CUDA tensor."""
        if isinstance(canonical, np.ndarray):
            cd = np.complex128 if prec == F64 else np.complex64
            canonical = torch.from_numpy(np.ascontiguousarray(canonical, dtype=cd).view(_npdtype(prec)).reshape(-1))
        canonical = canonical.to(self.device, dtype=_rdtype(prec)).contiguous().reshape(-1)
        assert canonical.numel() == int(np.prod(self.canonical_shape(parity)))
        out = self.new_native(prec, parity) if out is None else out
        self._chk(self.lib.dwf_pack(self._h, self._p(out), self._p(canonical), prec, parity))
        return out

    def unpack(self, native, prec=F64, parity=ODD, numpy=True):
        canon = torch.empty(int(np.prod(self.canonical_shape(parity))), dtype=_rdtype(prec), device=self.device)
        self._chk(self.lib.dwf_unpack(self._h, self._p(canon), self._p(native), prec, parity))
        if not numpy:
            return canon
        a = canon.cpu().numpy().reshape(self.canonical_shape(parity))
        return a[..., 0] + 1j * a[..., 1]

    def convert(self, src, src_prec, dst_prec, parity=ODD, out=None):
        out = self.new_native(dst_prec, parity) if out is None else out
        self._chk(self.lib.dwf_convert(self._h, self._p(out), dst_prec, self._p(src), src_prec, parity))
        return out

    # ---- operators on native fields --------------------------------------------------------------
    def dhop(self, inp, out_parity=FULL, dagger=False, prec=F64, out=None):
        out = self.new_native(prec, out_parity) if out is None else out
        self._chk(self.lib.dwf_dhop(self._h, self._p(out), self._p(inp), out_parity, int(dagger), prec))
        return out

    def _op5(self, fn, inp, parity, dagger, prec, out):
        out = self.new_native(prec, parity) if out is None else out
        self._chk(fn(self._h, self._p(out), self._p(inp), parity, int(dagger), prec))
        return out

    def meooe5d(self, inp, parity=ODD, dagger=False, prec=F64, out=None):
        return self._op5(self.lib.dwf_meooe5d, inp, parity, dagger, prec, out)

    def mooee(self, inp, parity=ODD, dagger=False, prec=F64, out=None):
        return self._op5(self.lib.dwf_mooee, inp, parity, dagger, prec, out)

    def mooee_inv(self, inp, parity=ODD, dagger=False, prec=F64, out=None):
        return self._op5(self.lib.dwf_mooee_inv, inp, parity, dagger, prec, out)

    def m(self, inp, dagger=False, prec=F64, out=None):
        out = self.new_native(prec, FULL) if out is None else out
        self._chk(self.lib.dwf_m(self._h, self._p(out), self._p(inp), int(dagger), prec))
        return out

    def mpc(self, inp, dagger=False, prec=F64, out=None):
        out = self.new_native(prec, ODD) if out is None else out
        self._chk(self.lib.dwf_mpc(self._h, self._p(out), self._p(inp), int(dagger), prec))
        return out

    def mdagm(self, inp, prec=F64, out=None):
        out = self.new_native(prec, ODD) if out is None else out
        self._chk(self.lib.dwf_mdagm(self._h, self._p(out), self._p(inp), prec))
        return out

    def norm2(self, v, prec=F64, parity=ODD):
        r = ctypes.c_double()
        self._chk(self.lib.dwf_norm2(self._h, self._p(v), prec, parity, ctypes.byref(r)))
        return r.value

    # ---- solvers ---------------------------------------------------------------------------------
    def cg(self, b, tol, max_iter, mode=CG_F64, x=None, use_guess=None):
        """Mpc^dag Mpc x = b on native fp64 ODD fields.  Returns (x, info dict, status).
        x given: it is the output buffer and, unless use_guess=False, the initial guess."""
        use_guess = (x is not None) if use_guess is None else bool(use_guess)
        x = self.new_native(F64, ODD) if x is None else x
        info = CgInfo()
        st = self._chk(self.lib.dwf_cg(self._h, self._p(x), self._p(b), tol, max_iter, mode, int(use_guess),
                                       ctypes.byref(info)), allow=(ENOTCONV,))
        return x, info.as_dict(), st

    # ---- batched (multi right-hand side) fields: SURVEY 8f NEXT-3 ---------------------------------
    def mrhs_reserve(self, nrhs):
        self._chk(self.lib.dwf_mrhs_reserve(self._h, int(nrhs)))

    def new_mrhs(self, nrhs, prec=F64):
        nb = self.lib.dwf_mrhs_field_bytes(self._h, int(nrhs), prec)
        return torch.empty(nb // (8 if prec == F64 else 4), dtype=_rdtype(prec), device=self.device)

    def mrhs_gather(self, fields, prec=F64):
        """list of native half fields -> one batched field"""
        n = len(fields)
        out = self.new_mrhs(n, prec)
        for j, f in enumerate(fields):
            self._chk(self.lib.dwf_mrhs_insert(self._h, self._p(out), n, j, self._p(f), prec))
        return out

    def mrhs_scatter(self, batched, nrhs, prec=F64):
        """one batched field -> list of native half fields"""
        outs = []
        for j in range(nrhs):
            f = self.new_native(prec, ODD)
            self._chk(self.lib.dwf_mrhs_extract(self._h, self._p(f), self._p(batched), nrhs, j, prec))
            outs.append(f)
        return outs

    def dhop_mrhs(self, inp, nrhs, out_parity, dagger=False, prec=F64, out=None):
        out = self.new_mrhs(nrhs, prec) if out is None else out
        self._chk(self.lib.dwf_dhop_mrhs(self._h, self._p(out), self._p(inp), int(nrhs), out_parity, int(dagger), prec))
        return out

    def mpc_mrhs(self, inp, nrhs, dagger=False, prec=F64, out=None):
        out = self.new_mrhs(nrhs, prec) if out is None else out
        self._chk(self.lib.dwf_mpc_mrhs(self._h, self._p(out), self._p(inp), int(nrhs), int(dagger), prec))
        return out

    def mdagm_mrhs(self, inp, nrhs, prec=F64, out=None):
        out = self.new_mrhs(nrhs, prec) if out is None else out
        self._chk(self.lib.dwf_mdagm_mrhs(self._h, self._p(out), self._p(inp), int(nrhs), prec))
        return out

    def cg_mrhs(self, b, nrhs, tol, max_iter, mode=CG_F64, x=None, use_guess=None):
        """nrhs independent CGs on a batched fp64 ODD field.  Returns (x batched, [info dict per system], status)."""
        use_guess = (x is not None) if use_guess is None else bool(use_guess)
        x = self.new_mrhs(nrhs, F64) if x is None else x
        infos = (CgInfo * nrhs)()
        st = self._chk(self.lib.dwf_cg_mrhs(self._h, self._p(x), self._p(b), int(nrhs), tol, max_iter, mode, int(use_guess),
                                            infos), allow=(ENOTCONV,))
        return x, [i.as_dict() for i in infos], st

    def domain_project(self, inp, which, prec=F64, out=None):
        """which = 0: P_Omega, 1: P_Omegabar, 2: boundary projector P_dbar; FULL native fields."""
        out = self.new_native(prec, FULL) if out is None else out
        self._chk(self.lib.dwf_domain_project(self._h, self._p(out), self._p(inp), int(which), prec))
        return out

    def boundary_op(self, phi, inverse, tol, max_iter, mode=CG_F64, out=None):
        """R phi (inverse False, eqs. 9-10) or R^-1 phi (inverse True, eqs. 13-14); FULL fp64 native fields."""
        out = self.new_native(F64, FULL) if out is None else out
        info = CgInfo()
        st = self._chk(self.lib.dwf_boundary_op(self._h, self._p(out), self._p(phi), int(bool(inverse)), tol, max_iter, mode,
                                                ctypes.byref(info)), allow=(ENOTCONV,))
        return out, info.as_dict(), st

    def chebyshev(self, inp, lo, hi, order, prec=F64, out=None):
        out = self.new_native(prec, ODD) if out is None else out
        self._chk(self.lib.dwf_chebyshev(self._h, self._p(out), self._p(inp), float(lo), float(hi), int(order), prec))
        return out

    def multishift_cg(self, b, shifts, tol, max_iter):
        """(Mpc^dag Mpc + shifts[i]) x_i = b, fp64.  Returns (list of native x_i, info dict, per-shift true residuals, status)."""
        n = len(shifts)
        per = self.field_bytes(F64, ODD) // 8
        x = torch.empty(n * per, dtype=torch.float64, device=self.device)
        sh = (ctypes.c_double * n)(*[float(s) for s in shifts])
        res = (ctypes.c_double * n)()
        info = CgInfo()
        st = self._chk(self.lib.dwf_multishift_cg(self._h, self._p(x), self._p(b), sh, n, tol, max_iter, ctypes.byref(info), res),
                       allow=(ENOTCONV,))
        return [x[i * per:(i + 1) * per] for i in range(n)], info.as_dict(), list(res), st

    def solve(self, eta, tol, max_iter, mode=CG_F64, out=None):
        """M psi = eta on native fp64 FULL fields.  Returns (psi, info dict, status)."""
        psi = self.new_native(F64, FULL) if out is None else out
        info = CgInfo()
        st = self._chk(self.lib.dwf_solve(self._h, self._p(psi), self._p(eta), tol, max_iter, mode,
                                          ctypes.byref(info)), allow=(ENOTCONV,))
        return psi, info.as_dict(), st

    # ---- end-to-end entry points: HOST canonical buffers (numpy / pinned torch CPU tensors) ---------
    @staticmethod
    def _hp(a):
        if isinstance(a, np.ndarray):
            assert a.flags["C_CONTIGUOUS"]
            return ctypes.c_void_p(a.ctypes.data)
        assert a.device.type == "cpu" and a.is_contiguous()
        return ctypes.c_void_p(a.data_ptr())

    def dhop_host(self, out_host, in_host, out_parity=FULL, dagger=False, prec=F64):
        self._chk(self.lib.dwf_dhop_host(self._h, self._hp(out_host), self._hp(in_host), out_parity, int(dagger), prec))
        return out_host

    def mdagm_host(self, out_host, in_host, prec=F64):
        self._chk(self.lib.dwf_mdagm_host(self._h, self._hp(out_host), self._hp(in_host), prec))
        return out_host

    def cg_host(self, x_host, b_host, tol, max_iter, mode=CG_F64):
        info = CgInfo()
        st = self._chk(self.lib.dwf_cg_host(self._h, self._hp(x_host), self._hp(b_host), tol, max_iter, mode,
                                            ctypes.byref(info)), allow=(ENOTCONV,))
        return x_host, info.as_dict(), st

    def solve_host(self, psi_host, eta_host, tol, max_iter, mode=CG_F64):
        info = CgInfo()
        st = self._chk(self.lib.dwf_solve_host(self._h, self._hp(psi_host), self._hp(eta_host), tol, max_iter, mode,
                                               ctypes.byref(info)), allow=(ENOTCONV,))
        return psi_host, info.as_dict(), st


NORM2_STATIC_MAX_BYTES = 1 << 32      # DWF_NORM2_STATIC_MAX_BYTES of include/dwf.h


def norm2_static(v, out, prec=None, stream=None):
    """dwf_norm2_static: sum |v|^2 of a CUDA tensor into the one-element fp64 CUDA tensor `out`, for callers whose device
    memory is all spoken for.  Unlike Dwf.norm2 it needs no context and the library allocates nothing for it: the partial
    sums go to a fixed 512 KiB array built into libdwf_b200.so, which is why `v` may hold at most NORM2_STATIC_MAX_BYTES
    (4 GiB; DwfError otherwise).  `v`: contiguous real tensor (float64 / float32) on the current device, any layout.  Two
    kernels are enqueued on `stream` (default: torch's current stream) and nothing waits for them: `out.item()` or a stream
    synchronise gives the value.  Calls on one device share the array, so do not let two of them overlap on the GPU.  This
    wrapper only marshals the arguments (it allocates nothing either; `out` is the caller's)."""
    lib = load_library()
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2203_17119_b200 needs a CUDA device (no CPU fallback)")
    prec = (F64 if v.dtype == torch.float64 else F32) if prec is None else prec
    assert v.is_cuda and v.is_contiguous() and v.dtype == _rdtype(prec)
    assert out.is_cuda and out.dtype == torch.float64 and out.numel() >= 1 and out.device == v.device
    s = torch.cuda.current_stream(v.device).cuda_stream if stream is None else int(stream)
    err = ctypes.create_string_buffer(256)
    with torch.cuda.device(v.device):
        st = lib.dwf_norm2_static(ctypes.c_void_p(v.data_ptr()), v.numel(), prec, ctypes.c_void_p(out.data_ptr()),
                                  ctypes.c_void_p(s), err, len(err))
    if st != OK:
        raise DwfError(st, err.value.decode())
    return out


def from_config(cfg, **options) -> Dwf:
    """Context for an inputs.Config (BASELINE.json configs)."""
    o = dict(options)
    o.setdefault("antiperiodic_t", 1 if cfg.antiperiodic_t else 0)
    return Dwf(cfg.dims, cfg.Ls, cfg.M5, cfg.mf, cfg.b5, cfg.c5, cut=cfg.cut, **o)
