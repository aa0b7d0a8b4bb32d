"""ctypes wrapper around oracle/liboracle.so — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It shares nothing with the CUDA binding (paper_2006_07964_b200/binding.py): the two
define their own ctypes structs and neither imports the other.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, HERE)
import build as _build  # noqa: E402  (oracle/build.py)

sys.path.pop(0)

NG = 6


class _Params(C.Structure):
    _fields_ = [("gamma", C.c_double), ("mach", C.c_double), ("reynolds", C.c_double), ("prandtl", C.c_double),
                ("weno_eps", C.c_double), ("viscous", C.c_int), ("scheme", C.c_int), ("q_inf", C.c_double * 5),
                ("sutherland", C.c_double)]


class _Face(C.Structure):
    _fields_ = [("block", C.c_int), ("face", C.c_int), ("type", C.c_int), ("nbr_block", C.c_int),
                ("nbr_face", C.c_int), ("perm", C.c_int * 3), ("sign", C.c_int * 3), ("shift", C.c_double * 3)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.POINTER(C.c_int), C.c_int, C.POINTER(_Face), C.POINTER(_Params)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_threads.argtypes = [C.c_void_p, C.c_int]
        L.orc_max_threads.restype = C.c_int
        L.orc_field.restype = C.POINTER(C.c_double)
        L.orc_field.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_last_error.restype = C.c_char_p
        L.orc_last_error.argtypes = [C.c_void_p]
        for name in ("orc_compute_metrics", "orc_rhs", "orc_exchange_interfaces", "orc_apply_bc"):
            getattr(L, name).argtypes = [C.c_void_p]
            getattr(L, name).restype = C.c_int
        L.orc_rk_stage.argtypes = [C.c_void_p, C.c_int, C.c_double, C.POINTER(C.c_double)]
        L.orc_rk_stage.restype = C.c_int
        L.orc_cfl_dt.argtypes = [C.c_void_p, C.c_double]
        L.orc_cfl_dt.restype = C.c_double
        dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
        L.orc_d6.argtypes = [dp]
        L.orc_d6.restype = C.c_double
        L.orc_weno5.argtypes = [dp, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_weno5_beta.argtypes = [dp, dp]
        L.orc_eig.argtypes = [dp, dp, C.c_double, dp, dp]
        L.orc_sw_flux.argtypes = [dp, dp, C.c_double, C.c_int, dp]
        L.orc_point_flux.argtypes = [dp, dp, C.c_double, dp]
        L.orc_khat_half.argtypes = [dp]
        L.orc_khat_half.restype = C.c_double
        L.orc_inviscid_line.argtypes = [C.c_int, dp, dp, C.c_double, C.c_double, C.c_int, dp]
        L.orc_visc_flux_point.argtypes = [dp, dp, dp, C.c_double, C.c_double, dp]
        L.orc_grad_point.argtypes = [dp, dp, C.c_double, dp]
        L.orc_sutherland_mu.argtypes = [C.c_double, C.c_double]
        L.orc_sutherland_mu.restype = C.c_double
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


# ---- per-point routines -----------------------------------------------------------------------
def d6(a7):
    return lib().orc_d6(_f64(a7))


def weno5(s5, eps=1e-6):
    vL, vR = C.c_double(), C.c_double()
    lib().orc_weno5(_f64(s5), eps, C.byref(vL), C.byref(vR))
    return vL.value, vR.value


def weno5_beta(s5):
    b = np.zeros(3)
    lib().orc_weno5_beta(_f64(s5), b)
    return b


def eig(Q, n, gamma=1.4):
    L, R = np.zeros((5, 5)), np.zeros((5, 5))
    lib().orc_eig(_f64(Q), _f64(n), gamma, L, R)
    return L, R


def sw_flux(Q, k, sgn, gamma=1.4):
    F = np.zeros(5)
    lib().orc_sw_flux(_f64(Q), _f64(k), gamma, int(sgn), F)
    return F


def point_flux(Q, k, gamma=1.4):
    F = np.zeros(5)
    lib().orc_point_flux(_f64(Q), _f64(k), gamma, F)
    return F


def khat_half(a6):
    return lib().orc_khat_half(_f64(a6))


def inviscid_line(Ql, kl, gamma=1.4, eps=1e-6, scheme=0):
    """Ql: (5, n+12), kl: (3, n+12) -> D (5, n)."""
    Ql, kl = _f64(Ql), _f64(kl)
    n = Ql.shape[1] - 2 * NG
    D = np.zeros((5, n))
    lib().orc_inviscid_line(n, Ql, kl, gamma, eps, scheme, D)
    return D


def visc_flux_point(vel, g, k, mu, kappa):
    Fv = np.zeros(5)
    lib().orc_visc_flux_point(_f64(vel), _f64(g), _f64(k), mu, kappa, Fv)
    return Fv


def sutherland_mu(T, S):
    return lib().orc_sutherland_mu(float(T), float(S))


def grad_point(dphi, kh, J):
    g = np.zeros((3, 4))
    lib().orc_grad_point(_f64(dphi), _f64(kh), J, g)
    return g


# ---- block-level solver -----------------------------------------------------------------------
class Oracle:
    """Owns its (host) arrays; `field(b, name)` returns a numpy view [nv, mk, mj, mi] with ghosts."""

    FIELDS = dict(q=(0, 5), qn=(1, 5), r=(2, 5), xyz=(3, 3), khat=(4, 9), jac=(5, 1))

    def __init__(self, dims, faces, params, threads=None):
        L = lib()
        self.dims = [tuple(int(x) for x in d) for d in dims]
        nb = len(self.dims)
        d = (C.c_int * (3 * nb))(*[x for dd in self.dims for x in dd])
        fa = (_Face * max(1, len(faces)))()
        for t, f in enumerate(faces):
            fa[t].block, fa[t].face, fa[t].type = f["block"], f["face"], f["type"]
            fa[t].nbr_block, fa[t].nbr_face = f["nbr_block"], f["nbr_face"]
            for a in range(3):
                fa[t].perm[a], fa[t].sign[a], fa[t].shift[a] = f["perm"][a], f["sign"][a], f["shift"][a]
        p = _Params()
        for k in ("gamma", "mach", "reynolds", "prandtl", "weno_eps", "viscous", "scheme"):
            setattr(p, k, params[k])
        for a in range(5):
            p.q_inf[a] = params["q_inf"][a]
        p.sutherland = float(params.get("sutherland", 0.0))
        self.h = L.orc_create(nb, d, len(faces), fa, C.byref(p))
        if not self.h:
            raise ValueError("orc_create failed (see stderr)")
        self.threads = threads or L.orc_max_threads()
        L.orc_set_threads(self.h, self.threads)

    def __del__(self):
        if getattr(self, "h", None):
            lib().orc_destroy(self.h)
            self.h = None

    def set_threads(self, n):
        self.threads = int(n)
        lib().orc_set_threads(self.h, self.threads)

    def field(self, b, name):
        fid, nv = self.FIELDS[name]
        ni, nj, nk = self.dims[b]
        shape = (nv, nk + 2 * NG, nj + 2 * NG, ni + 2 * NG)
        ptr = lib().orc_field(self.h, b, fid)
        return np.ctypeslib.as_array(ptr, shape=(int(np.prod(shape)),)).reshape(shape)

    def interior(self, b, name):
        return self.field(b, name)[:, NG:-NG, NG:-NG, NG:-NG]

    def _chk(self, rc):
        if rc != 0:
            raise RuntimeError(lib().orc_last_error(self.h).decode())

    def load_case(self, case):
        for b in range(len(self.dims)):
            self.interior(b, "xyz")[...] = case.xyz[b]
            self.interior(b, "q")[...] = case.q0[b]
        self.compute_metrics()
        self.exchange_interfaces()
        self.apply_bc()

    def compute_metrics(self):
        self._chk(lib().orc_compute_metrics(self.h))

    def rhs(self):
        self._chk(lib().orc_rhs(self.h))

    def rk_stage(self, stage, dt, want_res=False):
        res = (C.c_double * 5)()
        self._chk(lib().orc_rk_stage(self.h, stage, dt, res if want_res else None))
        return np.array(res[:]) if want_res else None

    def exchange_interfaces(self):
        self._chk(lib().orc_exchange_interfaces(self.h))

    def apply_bc(self):
        self._chk(lib().orc_apply_bc(self.h))

    def cfl_dt(self, cfl):
        return lib().orc_cfl_dt(self.h, cfl)

    def stage(self, s, dt, want_res=False):
        """One RK stage in the order of Fig. 2: RHS, Eq. 20, ghost fill, physical BCs."""
        self.rhs()
        r = self.rk_stage(s, dt, want_res=want_res)
        self.exchange_interfaces()
        self.apply_bc()
        return r

    def step(self, dt):
        """One TVD-RK3 step in the order of Fig. 2."""
        res = None
        for s in (1, 2, 3):
            r = self.stage(s, dt, want_res=(s == 1))
            if s == 1:
                res = r
        return res
