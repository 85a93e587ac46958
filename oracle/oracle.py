"""ctypes front end of oracle/acm_oracle.c (TEST INFRASTRUCTURE, not the product).

Mirrors the call list of include/acm.h with host (numpy) arrays so that one test
harness can drive both the oracle and the CUDA library.  No arithmetic of the
method lives here: every number comes out of acm_oracle.c.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        lib.oracle_create.argtypes = [C.POINTER(C.c_void_p)] + [C.c_int] * 5 + [C.c_double] * 7 + [dp, C.c_uint]
        lib.oracle_destroy.argtypes = [C.c_void_p]
        lib.oracle_destroy.restype = None
        lib.oracle_init.argtypes = [C.c_void_p, dp, dp]
        lib.oracle_step.argtypes = [C.c_void_p, C.c_int]
        lib.oracle_fields.argtypes = [C.c_void_p, dp, dp, dp]
        lib.oracle_phi_mass.argtypes = [C.c_void_p, dp]
        lib.oracle_get_pdfs.argtypes = [C.c_void_p, dp, dp]
        lib.oracle_set_pdfs.argtypes = [C.c_void_p, dp, dp]
        lib.oracle_lattice.argtypes = [C.c_int, ip, dp, ip, dp, dp, ip]
        lib.oracle_fd.argtypes = [C.c_void_p, C.c_int, dp, dp, dp]
        lib.oracle_set_threads.argtypes = [C.c_int]
        lib.oracle_set_variant.argtypes = [C.c_void_p, C.c_uint]
        lib.oracle_set_subiter.argtypes = [C.c_void_p, C.c_int]
        lib.oracle_bubble_diag.argtypes = [C.c_void_p, dp]
        lib.oracle_bubble_params.argtypes = [C.c_double] * 7 + [dp]
        lib.oracle_drag_lbm.argtypes = [C.c_double] * 5
        lib.oracle_drag_lbm.restype = C.c_double
        lib.oracle_drag_exp.argtypes = [C.c_double]
        lib.oracle_drag_exp.restype = C.c_double
        _lib = lib
    return _lib


def _dp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def set_threads(n: int) -> int:
    return _load().oracle_set_threads(int(n))


def lattice(Q: int, bulk_split: bool = False):
    """Direction table, weights, opposite index, moment matrix M, M^-1 and row orders.
    bulk_split: the basis of variant A26 (the bulk moment is a row of its own, order ORDER_BULK)."""
    lib = _load()
    e = np.zeros((Q, 3), dtype=np.int32)
    w = np.zeros(Q)
    opp = np.zeros(Q, dtype=np.int32)
    M = np.zeros((Q, Q))
    Minv = np.zeros((Q, Q))
    order = np.zeros(Q, dtype=np.int32)
    ip = C.POINTER(C.c_int)
    rc = lib.oracle_lattice(-Q if bulk_split else Q, e.ctypes.data_as(ip), _dp(w), opp.ctypes.data_as(ip), _dp(M), _dp(Minv),
                            order.ctypes.data_as(ip))
    if rc:
        raise ValueError(f"unsupported stencil D3Q{Q}")
    return e, w, opp, M, Minv, order


VAR_PHASE_SRT, VAR_BULK_ONE = 1, 2
ORDER_BULK = 20


def bubble_params(Re_Gr, Eo, D, t_ref, rho_H=1.0, rho_star=1000.0, mu_star=100.0):
    """eqs. 31-33 solved for the lattice parameters: dict(gy, sigma, nu_H, nu_L, rho_L)."""
    out = np.zeros(5)
    rc = _load().oracle_bubble_params(Re_Gr, Eo, D, t_ref, rho_H, rho_star, mu_star, _dp(out))
    if rc:
        raise ValueError("bubble_params: all arguments must be positive")
    return dict(gy=out[0], sigma=out[1], nu_H=out[2], nu_L=out[3], rho_L=out[4])


def drag_lbm(gy, rho_H, rho_L, D, u_t):
    return _load().oracle_drag_lbm(gy, rho_H, rho_L, D, u_t)


def drag_exp(Re_Gr):
    return _load().oracle_drag_exp(Re_Gr)


class Oracle:
    """Host-side twin of the acm_* call list."""

    def __init__(self, nx, ny, nz, stencil_phase=15, stencil_hydro=19, rho_H=1.0, rho_L=1e-3, sigma=1e-4, xi=5.0,
                 M=0.02, nu_H=1 / 60, nu_L=1 / 60, gravity=(0.0, 0.0, 0.0), wall_flags=0, phase_srt=False, bulk_one=False,
                 subiter=1):
        self._lib = _load()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.Qh, self.Qg = int(stencil_phase), int(stencil_hydro)
        self.N = self.nx * self.ny * self.nz
        self.shape = (self.nz, self.ny, self.nx)
        g = (C.c_double * 3)(*[float(v) for v in gravity])
        h = C.c_void_p()
        rc = self._lib.oracle_create(C.byref(h), self.nx, self.ny, self.nz, self.Qh, self.Qg, rho_H, rho_L, sigma, xi,
                                     M, nu_H, nu_L, g, int(wall_flags))
        if rc:
            raise ValueError(f"oracle_create failed with code {rc}")
        self._h = h
        flags = (VAR_PHASE_SRT if phase_srt else 0) | (VAR_BULK_ONE if bulk_one else 0)
        if flags:
            assert self._lib.oracle_set_variant(h, flags) == 0
        if subiter != 1:
            assert self._lib.oracle_set_subiter(h, int(subiter)) == 0

    @classmethod
    def from_params(cls, p, **kw):
        kw.setdefault("phase_srt", getattr(p, "phase_srt", False))
        return cls(p.nx, p.ny, p.nz, p.stencil_phase, p.stencil_hydro, p.rho_H, p.rho_L, p.sigma, p.xi, p.M,
                   p.nu_H, p.nu_L, p.gravity, p.wall_flags, **kw)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.oracle_destroy(self._h)
            self._h = None

    __del__ = close

    def init(self, phi, u):
        phi = np.ascontiguousarray(phi, dtype=np.float64).reshape(self.shape)
        u = np.ascontiguousarray(u, dtype=np.float64).reshape((3,) + self.shape)
        rc = self._lib.oracle_init(self._h, _dp(phi), _dp(u))
        assert rc == 0, rc

    def step(self, n=1):
        rc = self._lib.oracle_step(self._h, int(n))
        if rc:
            raise RuntimeError(f"oracle_step failed with code {rc}")

    def fields(self, want_p=True):
        phi = np.empty(self.shape)
        u = np.empty((3,) + self.shape)
        p = np.empty(self.shape) if want_p else None
        self._lib.oracle_fields(self._h, _dp(phi), _dp(u), _dp(p))
        return phi, u, p

    def phi_mass(self):
        t = C.c_double()
        rc = self._lib.oracle_phi_mass(self._h, C.byref(t))
        if rc:
            raise FloatingPointError("sum(phi) is not finite")
        return t.value

    def bubble_diag(self):
        """(V, centroid[3] as (x,y,z), velocity[3]) of the light phase, weighted with 1 - phi."""
        out = np.zeros(7)
        assert self._lib.oracle_bubble_diag(self._h, _dp(out)) == 0
        return out[0], out[1:4].copy(), out[4:7].copy()

    def get_pdfs(self):
        h = np.empty((self.Qh,) + self.shape)
        g = np.empty((self.Qg,) + self.shape)
        self._lib.oracle_get_pdfs(self._h, _dp(h), _dp(g))
        return h, g

    def set_pdfs(self, h=None, g=None):
        h = None if h is None else np.ascontiguousarray(h, dtype=np.float64).reshape((self.Qh,) + self.shape)
        g = None if g is None else np.ascontiguousarray(g, dtype=np.float64).reshape((self.Qg,) + self.shape)
        self._lib.oracle_set_pdfs(self._h, _dp(h), _dp(g))

    def fd(self, field, hydro_stencil=False):
        field = np.ascontiguousarray(field, dtype=np.float64).reshape(self.shape)
        grad = np.empty((3,) + self.shape)
        lap = np.empty(self.shape)
        self._lib.oracle_fd(self._h, int(hydro_stencil), _dp(field), _dp(grad), _dp(lap))
        return grad, lap
