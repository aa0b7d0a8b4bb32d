"""Thin ctypes binding of the C ABI in include/cfd.h (argument marshalling only).

PyTorch is used for device memory and the CUDA stream — plumbing, not the product: every step of
the path runs in the kernels of csrc/.  There is NO CPU fallback: importing this module raises if
libcfd_b200.so is missing, and `Context` raises if there is no CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

NG = 6
HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libcfd_b200.so")

ABI_SYMBOLS = (
    "cfd_workspace_bytes", "cfd_create_blocks", "cfd_compute_metrics", "cfd_rhs", "cfd_rk_stage",
    "cfd_exchange_interfaces", "cfd_apply_bc", "cfd_stage", "cfd_destroy", "cfd_last_error",
    "cfd_launch_count", "cfd_fp64_peak_probe", "cfd_step_host", "cfd_profile_enable", "cfd_profile_read",
    "cfd_profile_name", "cfd_selftest_fastmath", "cfd_set_sweep_plan", "cfd_stage_fused", "cfd_buffer_roles",
    "cfd_cfl_dt", "cfd_create_blocks_sharded", "cfd_workspace_bytes_sharded", "cfd_stage_fused_local",
    "cfd_profile_only", "cfd_set_visc_tile", "cfd_rk_stage1_static", "cfd_static_last_error",
)
STATIC_MAX_POINTS = 2097152  # CFD_STATIC_MAX_POINTS of include/cfd.h
PROF_NCLASS = 12


class CfdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"cfd error {code}: {msg}")
        self.code = code


class _Dims(C.Structure):
    _fields_ = [("ni", C.c_int), ("nj", C.c_int), ("nk", C.c_int)]


class _Params(C.Structure):
    _fields_ = [("gamma", C.c_double), ("mach", C.c_double), ("reynolds", C.c_double), ("prandtl", C.c_double),
                ("weno_eps", C.c_double), ("viscous", C.c_int), ("scheme", C.c_int), ("q_inf", C.c_double * 5),
                ("sutherland", C.c_double)]


class _Face(C.Structure):
    _fields_ = [("block", C.c_int), ("face", C.c_int), ("type", C.c_int), ("nbr_block", C.c_int),
                ("nbr_face", C.c_int), ("perm", C.c_int * 3), ("sign", C.c_int * 3), ("shift", C.c_double * 3)]


class _Ptrs(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("q", "qn", "r", "xyz", "khat", "jac")]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2006_07964_b200.build` "
            "(nvcc, sm_100a). There is no CPU fallback for this library.")
    L = C.CDLL(LIB_PATH)
    L.cfd_workspace_bytes.restype = C.c_size_t
    L.cfd_workspace_bytes.argtypes = [C.c_int, C.POINTER(_Dims), C.POINTER(_Params)]
    L.cfd_create_blocks.restype = C.c_int
    L.cfd_create_blocks.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.POINTER(_Dims), C.POINTER(_Ptrs), C.c_int,
                                    C.POINTER(_Face), C.POINTER(_Params), C.c_void_p, C.c_size_t, C.c_void_p]
    for n in ("cfd_compute_metrics", "cfd_rhs", "cfd_exchange_interfaces", "cfd_apply_bc", "cfd_destroy"):
        getattr(L, n).restype = C.c_int
        getattr(L, n).argtypes = [C.c_void_p]
    L.cfd_buffer_roles.restype = C.c_int
    L.cfd_buffer_roles.argtypes = [C.c_void_p, C.POINTER(C.c_int)]
    L.cfd_workspace_bytes_sharded.restype = C.c_size_t
    L.cfd_workspace_bytes_sharded.argtypes = [C.c_int, C.POINTER(_Dims), C.POINTER(C.c_int), C.POINTER(_Params)]
    L.cfd_create_blocks_sharded.restype = C.c_int
    L.cfd_create_blocks_sharded.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.POINTER(_Dims), C.POINTER(_Ptrs), C.POINTER(C.c_int),
                                            C.c_int, C.POINTER(_Face), C.POINTER(_Params), C.c_void_p, C.c_size_t, C.c_void_p]
    for n in ("cfd_rk_stage", "cfd_stage", "cfd_stage_fused", "cfd_stage_fused_local"):
        getattr(L, n).restype = C.c_int
        getattr(L, n).argtypes = [C.c_void_p, C.c_int, C.c_double, C.POINTER(C.c_double)]
    L.cfd_cfl_dt.restype = C.c_int
    L.cfd_cfl_dt.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_void_p)]
    L.cfd_last_error.restype = C.c_char_p
    L.cfd_last_error.argtypes = [C.c_void_p]
    L.cfd_launch_count.restype = C.c_longlong
    L.cfd_launch_count.argtypes = [C.c_void_p]
    L.cfd_step_host.restype = C.c_int
    L.cfd_step_host.argtypes = [C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.c_double, C.POINTER(C.c_double)]
    L.cfd_profile_enable.restype = C.c_int
    L.cfd_profile_enable.argtypes = [C.c_void_p, C.c_int]
    L.cfd_profile_read.restype = C.c_int
    L.cfd_profile_read.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
    L.cfd_profile_name.restype = C.c_char_p
    L.cfd_profile_name.argtypes = [C.c_int]
    L.cfd_set_visc_tile.restype = C.c_int
    L.cfd_set_visc_tile.argtypes = [C.c_void_p, C.c_int]
    L.cfd_profile_only.restype = C.c_int
    L.cfd_profile_only.argtypes = [C.c_void_p, C.c_uint]
    L.cfd_set_sweep_plan.restype = C.c_int
    L.cfd_set_sweep_plan.argtypes = [C.c_void_p, C.c_int]
    L.cfd_selftest_fastmath.restype = C.c_int
    L.cfd_selftest_fastmath.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.cfd_fp64_peak_probe.restype = C.c_int
    L.cfd_fp64_peak_probe.argtypes = [C.c_int, C.POINTER(C.c_double)]
    L.cfd_rk_stage1_static.restype = C.c_int
    L.cfd_rk_stage1_static.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double,
                                       C.c_void_p, C.c_void_p]
    L.cfd_static_last_error.restype = C.c_char_p
    L.cfd_static_last_error.argtypes = []
    return L


lib = _load()


def device_peak_probe(iters=4096):
    """Measured FP64 FMA throughput of the current device in TFLOP/s (FMA = 2 flops)."""
    t = C.c_double()
    rc = lib.cfd_fp64_peak_probe(int(iters), C.byref(t))
    if rc != 0:
        raise CfdError(rc, "cfd_fp64_peak_probe failed")
    return t.value


def selftest_fastmath(x):
    """(1/x, 1/sqrt(x)) as the hot kernels compute them (csrc/fastmath.cuh), for a host fp64 array x > 0."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    r, s = np.empty_like(x), np.empty_like(x)
    dp = C.POINTER(C.c_double)
    rc = lib.cfd_selftest_fastmath(int(x.size), x.ctypes.data_as(dp), r.ctypes.data_as(dp), s.ctypes.data_as(dp))
    if rc != 0:
        raise CfdError(rc, "cfd_selftest_fastmath failed")
    return r, s


def rk_stage1_static(q, qn, r, dims, dt, res5, stream=None):
    """cfd_rk_stage1_static: RK3 stage 1 (q^n := q, q := q + dt r) and res_m = sum r_m^2 of ONE block without a context,
    a workspace or any device allocation -- for callers that cannot allocate (a plug-in inside an application that has
    reserved all device memory, a loop that may not stall the GPU on cudaMalloc, a callback that owns no allocator): the
    partial sums live in a fixed array inside the library.  q, qn, r: device fp64 tensors of shape (5, nk+12, nj+12, ni+12);
    res5: device fp64 tensor of 5 elements (output); dims = (ni, nj, nk) with ni*nj*nk <= STATIC_MAX_POINTS.  Enqueues on
    `stream` (default: torch's current stream of q's device) and returns at once.  All calls on one device share that array:
    keep them on one stream.  This wrapper only checks and passes pointers."""
    import torch

    ni, nj, nk = (int(x) for x in dims)
    shp = (5, nk + 2 * NG, nj + 2 * NG, ni + 2 * NG)
    for name, a in (("q", q), ("qn", qn), ("r", r)):
        if not (a.is_cuda and a.dtype == torch.float64 and a.is_contiguous() and tuple(a.shape) == shp):
            raise CfdError(-1, f"rk_stage1_static: {name} must be a contiguous device fp64 tensor of shape {shp}")
    if not (res5.is_cuda and res5.dtype == torch.float64 and res5.is_contiguous() and res5.numel() == 5):
        raise CfdError(-1, "rk_stage1_static: res5 must be a contiguous device fp64 tensor of 5 elements")
    with torch.cuda.device(q.device):
        st = stream if stream is not None else torch.cuda.current_stream(q.device)
        rc = lib.cfd_rk_stage1_static(q.data_ptr(), qn.data_ptr(), r.data_ptr(), ni, nj, nk, float(dt), res5.data_ptr(),
                                      C.c_void_p(st.cuda_stream))
    if rc != 0:
        raise CfdError(rc, lib.cfd_static_last_error().decode())


class Context:
    """One solver context over `dims` blocks.  Allocates the device fields with torch (fp64,
    [var][k][j][i] with 6 ghost layers) and hands raw pointers to the C ABI."""

    NV = dict(q=5, qn=5, r=5, xyz=3, khat=9, jac=1)

    def __init__(self, dims, faces, params, device="cuda:0", stream=None):
        import torch

        if not torch.cuda.is_available():
            raise CfdError(-6, "no CUDA device: this library has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        self.dims = [tuple(int(x) for x in d) for d in dims]
        nb = len(self.dims)
        self.fields = []
        with torch.cuda.device(self.device):
            for (ni, nj, nk) in self.dims:
                shp = (nk + 2 * NG, nj + 2 * NG, ni + 2 * NG)
                self.fields.append({n: torch.zeros((nv,) + shp, dtype=torch.float64, device=self.device)
                                    for n, nv in self.NV.items()})
            d = (_Dims * nb)(*[_Dims(*dd) for dd in self.dims])
            p = _Params()
            for k in ("gamma", "mach", "reynolds", "prandtl", "weno_eps", "viscous", "scheme"):
                setattr(p, k, params[k])
            for a in range(5):
                p.q_inf[a] = params["q_inf"][a]
            p.sutherland = float(params.get("sutherland", 0.0))
            fa = (_Face * max(1, len(faces)))()
            for t, f in enumerate(faces):
                fa[t].block, fa[t].face, fa[t].type = f["block"], f["face"], f["type"]
                fa[t].nbr_block, fa[t].nbr_face = f["nbr_block"], f["nbr_face"]
                for a in range(3):
                    fa[t].perm[a], fa[t].sign[a], fa[t].shift[a] = f["perm"][a], f["sign"][a], f["shift"][a]
            ptrs = (_Ptrs * nb)()
            for b in range(nb):
                for n in self.NV:
                    setattr(ptrs[b], n, self.fields[b][n].data_ptr())
            wsb = lib.cfd_workspace_bytes(nb, d, C.byref(p))
            self.workspace = torch.empty((wsb + 7) // 8, dtype=torch.float64, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            rc = lib.cfd_create_blocks(C.byref(h), nb, d, ptrs, len(faces), fa, C.byref(p), self.workspace.data_ptr(),
                                       wsb, C.c_void_p(self.stream.cuda_stream))
            if rc != 0:
                raise CfdError(rc, lib.cfd_last_error(None).decode())
            self.h = h

    # ---- lifetime ----
    def close(self):
        if getattr(self, "h", None):
            lib.cfd_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc):
        if rc != 0:
            raise CfdError(rc, lib.cfd_last_error(self.h).decode())

    # ---- data movement helpers (harness side) ----
    def buffer_roles(self):
        """cfd_buffer_roles: which of the buffers allocated as (q, qn, r) currently holds Q, Q^n, R."""
        r = (C.c_int * 3)()
        self._chk(lib.cfd_buffer_roles(self.h, r))
        return tuple(r[:])

    def field(self, b, name):
        """The tensor that currently plays the role `name` (cfd_stage_fused exchanges the roles of q, qn, r)."""
        if name in ("q", "qn", "r"):
            name = ("q", "qn", "r")[self.buffer_roles()[("q", "qn", "r").index(name)]]
        return self.fields[b][name]

    def interior(self, b, name):
        return self.field(b, name)[:, NG:-NG, NG:-NG, NG:-NG]

    def load_case(self, case):
        t = self.torch
        for b in range(len(self.dims)):
            self.interior(b, "xyz").copy_(t.from_numpy(np.ascontiguousarray(case.xyz[b])))
            self.interior(b, "q").copy_(t.from_numpy(np.ascontiguousarray(case.q0[b])))
        self.compute_metrics()
        self.exchange_interfaces()
        self.apply_bc()

    def to_numpy(self, b, name, interior=True):
        a = self.interior(b, name) if interior else self.field(b, name)
        return a.detach().cpu().numpy()

    # ---- the C ABI, same names ----
    def compute_metrics(self):
        self._chk(lib.cfd_compute_metrics(self.h))

    def rhs(self):
        self._chk(lib.cfd_rhs(self.h))

    def rk_stage(self, stage, dt, want_res=False):
        res = (C.c_double * 5)()
        self._chk(lib.cfd_rk_stage(self.h, int(stage), float(dt), res if want_res else None))
        return np.array(res[:]) if want_res else None

    def exchange_interfaces(self):
        self._chk(lib.cfd_exchange_interfaces(self.h))

    def apply_bc(self):
        self._chk(lib.cfd_apply_bc(self.h))

    def cfl_dt(self, cfl, dt_local=None):
        """cfd_cfl_dt: dt = cfl / max over all interior points of sum_d(|k_d.u| + c|k_d|) from the current q; dt_local:
        optional list (one per block) of device fp64 tensors of shape (nk+12, nj+12, ni+12) receiving cfl / s_i."""
        dt = C.c_double()
        loc = None
        if dt_local is not None:
            for b, a in enumerate(dt_local):
                ni, nj, nk = self.dims[b]
                if not (a.is_cuda and a.dtype == self.torch.float64 and a.is_contiguous()
                        and tuple(a.shape) == (nk + 2 * NG, nj + 2 * NG, ni + 2 * NG)):
                    raise CfdError(-1, f"cfl_dt: block {b} needs a contiguous device fp64 tensor of shape (nk+12, nj+12, ni+12)")
            loc = (C.c_void_p * len(self.dims))(*[a.data_ptr() for a in dt_local])
        self._chk(lib.cfd_cfl_dt(self.h, float(cfl), C.byref(dt), loc))
        return dt.value

    def stage(self, stage, dt, want_res=False):
        res = (C.c_double * 5)()
        self._chk(lib.cfd_stage(self.h, int(stage), float(dt), res if want_res else None))
        return np.array(res[:]) if want_res else None

    def stage_fused(self, stage, dt, want_res=False):
        res = (C.c_double * 5)()
        self._chk(lib.cfd_stage_fused(self.h, int(stage), float(dt), res if want_res else None))
        return np.array(res[:]) if want_res else None

    def step(self, dt, want_res=False, fused=True):
        """One TVD-RK3 step = three stages in the order of Fig. 2; fused: cfd_stage_fused (the RK update
        inside the last sweep, buffer roles exchanged) instead of cfd_stage."""
        res = None
        for s in (1, 2, 3):
            r = (self.stage_fused if fused else self.stage)(s, dt, want_res=(want_res and s == 1))
            if s == 1:
                res = r
        return res

    def step_host(self, q_in, q_out, dt, want_res=False):
        """cfd_step_host: q_in / q_out are lists (one per block) of HOST fp64 tensors or numpy arrays of shape
        (5, nk, nj, ni), C-contiguous (pinned torch tensors recommended); returns res5 or None."""
        nb = len(self.dims)
        pin = (C.c_void_p * nb)(*[self._host_ptr(a, b) for b, a in enumerate(q_in)])
        pout = (C.c_void_p * nb)(*[self._host_ptr(a, b) for b, a in enumerate(q_out)])
        res = (C.c_double * 5)()
        self._chk(lib.cfd_step_host(self.h, pin, pout, float(dt), res if want_res else None))
        return np.array(res[:]) if want_res else None

    def _host_ptr(self, a, b):
        ni, nj, nk = self.dims[b]
        if isinstance(a, np.ndarray):
            ok = a.dtype == np.float64 and a.flags["C_CONTIGUOUS"] and a.shape == (5, nk, nj, ni)
            ptr = a.ctypes.data
        else:
            ok = (a.dtype == self.torch.float64 and a.is_contiguous() and tuple(a.shape) == (5, nk, nj, ni)
                  and a.device.type == "cpu")
            ptr = a.data_ptr()
        if not ok:
            raise CfdError(-1, f"step_host: block {b} needs a C-contiguous host fp64 array of shape (5,{nk},{nj},{ni})")
        return ptr

    def set_sweep_plan(self, plan):
        self._chk(lib.cfd_set_sweep_plan(self.h, int(plan)))

    def set_visc_tile(self, tile=-1):
        self._chk(lib.cfd_set_visc_tile(self.h, int(tile)))

    def profile_only(self, mask=0xFFFFFFFF):
        """cfd_profile_only: launch only the hot kernel classes in mask (measurement aid; results invalid unless all ones)."""
        self._chk(lib.cfd_profile_only(self.h, int(mask) & 0xFFFFFFFF))

    def profile_enable(self, on=True):
        self._chk(lib.cfd_profile_enable(self.h, 1 if on else 0))

    def profile_read(self):
        """{kernel class: (summed device ms, launches)} since the last read (synchronises)."""
        ms = (C.c_double * PROF_NCLASS)()
        n = (C.c_longlong * PROF_NCLASS)()
        self._chk(lib.cfd_profile_read(self.h, ms, n))
        return {lib.cfd_profile_name(i).decode(): (ms[i], int(n[i])) for i in range(PROF_NCLASS) if n[i]}

    @property
    def launch_count(self):
        return int(lib.cfd_launch_count(self.h))
