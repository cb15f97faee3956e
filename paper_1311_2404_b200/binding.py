"""Thin ctypes binding of include/lbm.h -- argument marshalling only.

Same names as the C ABI (lbm_create, lbm_set_geometry, lbm_init_equilibrium, lbm_step,
lbm_macro, ...) plus a small `Lbm` convenience class that owns the torch workspace tensor.
PyTorch is used for device memory and the CUDA stream only; every step of the path runs in the
library's kernels.  There is NO fallback: if liblbm_b200.so is missing, loading raises.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblbm_b200.so")

LBM_OK, LBM_EINVAL, LBM_EUNSUPPORTED, LBM_ENOMEM, LBM_ECUDA, LBM_ESTATE = 0, -1, -2, -3, -4, -5
LBM_D2Q9, LBM_D3Q19 = 0, 1
LBM_BGK, LBM_MRT, LBM_SC2, LBM_BGK_REG, LBM_BGK_LES = 0, 1, 2, 3, 4
LBM_F32, LBM_F64 = 0, 1
LBM_PSI_RHO, LBM_PSI_1MEXP = 0, 1
LBM_STORE_AB, LBM_STORE_AA = 0, 1
LBM_FORCE_GUO, LBM_FORCE_EDM = 0, 1
LBM_NODE_FLUID, LBM_NODE_SOLID, LBM_NODE_WALL_FULLWAY, LBM_NODE_VELOCITY = 0, 1, 2, 3
LBM_QMAX = 19

EXPORTS = ("lbm_lattice_info", "lbm_workspace_bytes", "lbm_create", "lbm_destroy", "lbm_set_geometry",
           "lbm_get_geometry", "lbm_init_equilibrium", "lbm_step", "lbm_macro", "lbm_get_distributions",
           "lbm_set_distributions", "lbm_get_stream_map", "lbm_run_host", "lbm_get_counters",
           "lbm_get_dispatch", "lbm_step_slabs", "lbm_step_noalloc", "lbm_noalloc_last_error", "lbm_last_error")


class lbm_params(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32),
        ("lattice", C.c_int32), ("model", C.c_int32), ("precision", C.c_int32),
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("tau", C.c_double * 2),
        ("rates", C.c_double * LBM_QMAX),
        ("force", C.c_double * 3),
        ("sc_G", C.c_double),
        ("sc_psi", C.c_int32),
        ("store", C.c_int32),
        ("bc_velocity", C.c_double * 3),
        ("force_scheme", C.c_int32),
        ("reserved_", C.c_int32),
        ("smagorinsky_cs", C.c_double),
    ]


class LbmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("lbm error %d: %s" % (code, msg))
        self.code = code


_lib = None


def load():
    """Load liblbm_b200.so (raises if it has not been built; there is no CPU path)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s is missing: run `python -m paper_1311_2404_b200.build` "
                          "(the CUDA library is the only implementation)" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp, i32, i64p = C.c_void_p, C.c_int32, C.c_void_p
    L.lbm_lattice_info.argtypes = [i32, vp, vp, vp, vp, vp]
    L.lbm_workspace_bytes.argtypes = [C.POINTER(lbm_params), C.POINTER(C.c_size_t)]
    L.lbm_create.argtypes = [C.POINTER(lbm_params), vp, C.c_size_t, vp, C.POINTER(vp)]
    L.lbm_destroy.argtypes = [vp]
    L.lbm_set_geometry.argtypes = [vp, vp]
    L.lbm_get_geometry.argtypes = [vp, vp]
    L.lbm_init_equilibrium.argtypes = [vp, C.c_int, vp, vp]
    L.lbm_step.argtypes = [vp, C.c_int]
    L.lbm_macro.argtypes = [vp, C.c_int, vp, vp]
    L.lbm_get_distributions.argtypes = [vp, C.c_int, vp]
    L.lbm_set_distributions.argtypes = [vp, C.c_int, vp]
    L.lbm_get_stream_map.argtypes = [vp, i64p]
    L.lbm_run_host.argtypes = [vp, vp, C.POINTER(vp), C.POINTER(vp), C.c_int, vp, vp]
    L.lbm_get_counters.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.lbm_get_dispatch.argtypes = [vp, C.POINTER(lbm_dispatch)]
    L.lbm_step_slabs.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int]
    L.lbm_last_error.argtypes = [vp]
    L.lbm_last_error.restype = C.c_char_p
    L.lbm_step_noalloc.argtypes = [C.POINTER(lbm_params), vp, vp, vp, C.c_int, vp]
    L.lbm_noalloc_last_error.argtypes = []
    L.lbm_noalloc_last_error.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("lbm_last_error", "lbm_noalloc_last_error"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


class lbm_dispatch(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("nodes_per_thread", "index_bits", "graph_replay", "resident_nodes_per_cta",
                                         "resident_ctas", "rows_per_block", "block_threads", "sc_split", "rows_strided")]


def make_params(lattice, model, precision, nx, ny, nz=1, tau=(1.0, 1.0), rates=None,
                force=(0.0, 0.0, 0.0), sc_G=0.0, sc_psi=LBM_PSI_RHO, store=LBM_STORE_AB,
                bc_velocity=(0.0, 0.0, 0.0), force_scheme=0, smagorinsky_cs=0.0) -> lbm_params:
    p = lbm_params()
    p.struct_size = C.sizeof(lbm_params)
    p.lattice, p.model, p.precision = int(lattice), int(model), int(precision)
    p.nx, p.ny, p.nz = int(nx), int(ny), int(nz)
    tau = (tau, tau) if isinstance(tau, (int, float)) else tuple(tau)
    p.tau[0], p.tau[1] = float(tau[0]), float(tau[1] if len(tau) > 1 else tau[0])
    if rates is not None:
        for k, r in enumerate(rates):
            p.rates[k] = float(r)
    for a in range(3):
        p.force[a] = float(force[a]) if a < len(force) else 0.0
    p.sc_G, p.sc_psi, p.store = float(sc_G), int(sc_psi), int(store)
    p.force_scheme = int(force_scheme)
    p.smagorinsky_cs = float(smagorinsky_cs)
    for a in range(3):
        p.bc_velocity[a] = float(bc_velocity[a]) if a < len(bc_velocity) else 0.0
    return p


def _check(rc, ctx=None):
    if rc != LBM_OK:
        msg = load().lbm_last_error(ctx)
        raise LbmError(rc, msg.decode() if msg else "")


# ---- C-ABI names, raw pointers in / error codes raised ------------------------------------------
def lbm_lattice_info(lattice):
    import numpy as np
    Q, D = C.c_int32(), C.c_int32()
    _check(load().lbm_lattice_info(lattice, C.addressof(Q), C.addressof(D), None, None, None))
    e = np.zeros((Q.value, 3), np.int32)
    w = np.zeros(Q.value, np.float64)
    opp = np.zeros(Q.value, np.int32)
    _check(load().lbm_lattice_info(lattice, None, None, e.ctypes.data, w.ctypes.data, opp.ctypes.data))
    return Q.value, D.value, e, w, opp


def lbm_workspace_bytes(params: lbm_params) -> int:
    n = C.c_size_t()
    _check(load().lbm_workspace_bytes(C.byref(params), C.byref(n)))
    return n.value


def lbm_create(params: lbm_params, d_workspace: int, nbytes: int, cuda_stream: int = 0) -> int:
    out = C.c_void_p()
    _check(load().lbm_create(C.byref(params), d_workspace, nbytes, cuda_stream or None, C.byref(out)))
    return out.value


def lbm_destroy(ctx): _check(load().lbm_destroy(ctx))
def lbm_set_geometry(ctx, d_mask): _check(load().lbm_set_geometry(ctx, d_mask), ctx)
def lbm_get_geometry(ctx, d_mask): _check(load().lbm_get_geometry(ctx, d_mask), ctx)
def lbm_init_equilibrium(ctx, comp, d_rho, d_u): _check(load().lbm_init_equilibrium(ctx, comp, d_rho, d_u), ctx)
def lbm_step(ctx, n): _check(load().lbm_step(ctx, n), ctx)
def lbm_macro(ctx, comp, d_rho, d_u): _check(load().lbm_macro(ctx, comp, d_rho, d_u), ctx)
def lbm_get_distributions(ctx, comp, d_f): _check(load().lbm_get_distributions(ctx, comp, d_f), ctx)
def lbm_set_distributions(ctx, comp, d_f): _check(load().lbm_set_distributions(ctx, comp, d_f), ctx)
def lbm_get_stream_map(ctx, d_map): _check(load().lbm_get_stream_map(ctx, d_map), ctx)


def lbm_run_host(ctx, h_mask, h_rho0, h_u0, n, h_rho_out, h_u_out):
    """h_rho0 / h_u0: sequences of host addresses (one per component)."""
    k = len(h_rho0)
    rho = (C.c_void_p * k)(*h_rho0)
    u = (C.c_void_p * k)(*h_u0)
    _check(load().lbm_run_host(ctx, h_mask, rho, u, n, h_rho_out, h_u_out), ctx)


def lbm_get_counters(ctx):
    s, l = C.c_int64(), C.c_int64()
    _check(load().lbm_get_counters(ctx, C.byref(s), C.byref(l)), ctx)
    return s.value, l.value


def lbm_step_slabs(ctxs, periodic_z: bool, n: int):
    arr = (C.c_void_p * len(ctxs))(*ctxs)
    _check(load().lbm_step_slabs(arr, len(ctxs), 1 if periodic_z else 0, int(n)), ctxs[0])


LBM_NOALLOC_MAX_BYTES = 64 << 20


def lbm_step_noalloc(params, d_mask, d_f_in, d_f_out, n: int, cuda_stream=None):
    """Raw pointers in (ints; d_mask may be None); raises LbmError with lbm_noalloc_last_error's message."""
    rc = load().lbm_step_noalloc(C.byref(params), d_mask, d_f_in, d_f_out, int(n), cuda_stream)
    if rc != LBM_OK:
        msg = load().lbm_noalloc_last_error()
        raise LbmError(rc, msg.decode() if msg else "")


def lbm_get_dispatch(ctx) -> dict:
    d = lbm_dispatch()
    _check(load().lbm_get_dispatch(ctx, C.byref(d)), ctx)
    return {n: getattr(d, n) for n, _ in lbm_dispatch._fields_ if n != "reserved_"}


# ---- convenience wrapper: owns the torch workspace, takes/returns torch tensors ------------------
class Lbm:
    """One context.  Tensors are torch CUDA tensors, C-order [z][y][x] / [D][z][y][x] / [Q][z][y][x]."""

    def __init__(self, lattice, model, precision, nx, ny, nz=1, device="cuda:0", stream=None, **kw):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1311_2404_b200 needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.device = torch.device(device)
        self.params = make_params(lattice, model, precision, nx, ny, nz, **kw)
        self.Q, self.D = (9, 2) if lattice == LBM_D2Q9 else (19, 3)
        self.shape = (nz, ny, nx)
        self.N = nx * ny * nz
        self.ncomp = 2 if model == LBM_SC2 else 1
        self.dtype = torch.float32 if precision == LBM_F32 else torch.float64
        nbytes = lbm_workspace_bytes(self.params)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.ctx = lbm_create(self.params, self.workspace.data_ptr(), nbytes, self.stream.cuda_stream)

    def close(self):
        if getattr(self, "ctx", None):
            lbm_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _dev(self, a, dtype):
        t = self.torch.as_tensor(a)
        return t.to(device=self.device, dtype=dtype).contiguous()

    def set_geometry(self, mask):
        m = self._dev(mask, self.torch.uint8)
        assert m.numel() == self.N
        lbm_set_geometry(self.ctx, m.data_ptr())
        self.stream.synchronize()  # m may be a temporary

    def get_geometry(self):
        m = self.torch.empty(self.shape, dtype=self.torch.uint8, device=self.device)
        lbm_get_geometry(self.ctx, m.data_ptr())
        return m

    def init_equilibrium(self, rho, u, comp=0):
        r, v = self._dev(rho, self.dtype), self._dev(u, self.dtype)
        assert r.numel() == self.N and v.numel() == self.D * self.N
        lbm_init_equilibrium(self.ctx, comp, r.data_ptr(), v.data_ptr())
        self.stream.synchronize()

    def step(self, n=1):
        lbm_step(self.ctx, int(n))

    def macro(self, comp=0):
        rho = self.torch.empty(self.shape, dtype=self.dtype, device=self.device)
        u = self.torch.empty((self.D,) + self.shape, dtype=self.dtype, device=self.device)
        lbm_macro(self.ctx, comp, rho.data_ptr(), u.data_ptr())
        return rho, u

    def get_distributions(self, comp=0):
        f = self.torch.empty((self.Q,) + self.shape, dtype=self.dtype, device=self.device)
        lbm_get_distributions(self.ctx, comp, f.data_ptr())
        return f

    def set_distributions(self, f, comp=0):
        t = self._dev(f, self.dtype)
        assert t.numel() == self.Q * self.N
        lbm_set_distributions(self.ctx, comp, t.data_ptr())
        self.stream.synchronize()

    def get_stream_map(self):
        m = self.torch.empty((self.Q, self.N), dtype=self.torch.int64, device=self.device)
        lbm_get_stream_map(self.ctx, m.data_ptr())
        return m

    def run_host(self, mask, rho0, u0, n, want_rho=True, want_u=True):
        """Whole path on HOST tensors (pinned recommended): returns (rho, u) host tensors of comp 0."""
        torch = self.torch
        rho_out = torch.empty(self.shape, dtype=self.dtype).pin_memory() if want_rho is True else want_rho
        u_out = torch.empty((self.D,) + self.shape, dtype=self.dtype).pin_memory() if want_u is True else want_u
        lbm_run_host(self.ctx, mask.data_ptr() if mask is not None else None,
                     [r.data_ptr() for r in rho0], [v.data_ptr() for v in u0], int(n),
                     rho_out.data_ptr() if rho_out is not None else None,
                     u_out.data_ptr() if u_out is not None else None)
        return rho_out, u_out

    def counters(self):
        return lbm_get_counters(self.ctx)

    def dispatch(self) -> dict:
        return lbm_get_dispatch(self.ctx)


def from_workload(w, device="cuda:0", **kw) -> "Lbm":
    """Context for a workloads.Workload (parameters only; arrays are passed separately)."""
    return Lbm(w.lattice, w.model, w.precision, w.nx, w.ny, w.nz, device=device, tau=w.tau, rates=w.rates,
               force=w.force, sc_G=w.sc_G, sc_psi=w.sc_psi, bc_velocity=w.bc_velocity, force_scheme=w.force_scheme, smagorinsky_cs=w.smagorinsky_cs, **kw)
