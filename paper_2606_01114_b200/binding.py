"""Thin Python binding of the C ABI in include/mm_b200.h.

Argument marshalling only: every numeric step runs in the library's CUDA kernels.  PyTorch is
used for device memory (the workspaces and the field tensors) and for the CUDA stream.  There
is no CPU fallback: if libmm_b200.so is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmm_b200.so")

MM_F32, MM_F64 = 0, 1
TERM_DEMAG, TERM_EXCHANGE, TERM_ANISOTROPY, TERM_ZEEMAN, TERM_DMI, TERM_STT = 1, 2, 4, 8, 16, 32
# DMI vectors e_k^DMI of PAPER.md:39 (rows k = x, y, z)
DMI_INTERFACIAL = ((0.0, 1.0, 0.0), (-1.0, 0.0, 0.0), (0.0, 0.0, 0.0))
DMI_BULK = ((1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0))
STATUS = {0: "MM_OK", 1: "MM_ERR_INVALID_ARG", 2: "MM_ERR_UNSUPPORTED_SIZE",
          3: "MM_ERR_NOT_INITIALISED", 4: "MM_ERR_WORKSPACE", 5: "MM_ERR_CUDA",
          6: "MM_ERR_NOT_IMPLEMENTED"}


class MMError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"{STATUS.get(status, status)}: {text}")
        self.status = status


_lib = None


def load_library():
    """dlopen libmm_b200.so; raises if it has not been built (python -m paper_2606_01114_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: build it with "
                          "`python -m paper_2606_01114_b200.build` (no CPU fallback exists)")
    lib = C.CDLL(LIB_PATH)
    vp, dbl, i32, sz = C.c_void_p, C.c_double, C.c_int, C.c_size_t
    sigs = {
        "mm_ctx_create": [i32, i32, i32, dbl, dbl, dbl, i32, C.POINTER(vp)],
        "mm_ctx_destroy": [vp],
        "mm_ctx_set_stream": [vp, vp],
        "mm_ctx_workspace_bytes": [vp, C.POINTER(sz), C.POINTER(sz)],
        "mm_ctx_set_workspace": [vp, vp, sz, vp, sz],
        "mm_set_material": [vp, dbl, dbl, dbl, C.POINTER(dbl), dbl, dbl],
        "mm_set_zeeman": [vp, C.POINTER(dbl)],
        "mm_set_material_cells": [vp, vp, vp],
        "mm_set_dmi": [vp, dbl, C.POINTER(dbl)],
        "mm_set_stt": [vp, C.POINTER(dbl), dbl, dbl],
        "mm_set_terms": [vp, C.c_uint],
        "mm_demag_init": [vp],
        "mm_demag_nhat_export": [vp, vp],
        "mm_demag_field": [vp, vp, vp],
        "mm_exchange_field": [vp, vp, vp],
        "mm_heff": [vp, vp, vp],
        "mm_dmi_field": [vp, vp, vp],
        "mm_llg_rhs": [vp, vp, vp],
        "mm_rk_step": [vp, vp, dbl],
        "mm_rk_steps": [vp, vp, dbl, i32],
        "mm_rkf45_init": [vp, dbl, dbl, dbl, dbl, dbl],
        "mm_rkf45_step": [vp, vp],
        "mm_rkf45_state": [vp, C.POINTER(dbl), C.POINTER(dbl), C.POINTER(dbl), C.POINTER(dbl),
                           C.POINTER(i32), C.POINTER(C.c_ulonglong), C.POINTER(C.c_ulonglong)],
        "mm_minimize_init": [vp, dbl, dbl, dbl, dbl],
        "mm_minimize_step": [vp, vp],
        "mm_minimize_state": [vp, C.POINTER(C.c_ulonglong), C.POINTER(dbl), C.POINTER(dbl), C.POINTER(i32)],
        "mm_minimize": [vp, vp, i32, i32, C.POINTER(C.c_ulonglong), C.POINTER(i32)],
        "mm_demag_field_static": [vp, vp, vp],
        "mm_static_scratch_info": [vp, C.POINTER(sz), C.POINTER(sz)],
        "mm_demag_field_host": [vp, vp, vp],
        "mm_heff_host": [vp, vp, vp],
        "mm_llg_rhs_host": [vp, vp, vp],
        "mm_rk_step_host": [vp, vp, dbl],
        "mm_llg_rhs_host_batch": [vp, C.POINTER(vp), C.POINTER(vp), i32],
        "mm_demag_field_host_batch": [vp, C.POINTER(vp), C.POINTER(vp), i32],
        "mm_heff_host_batch": [vp, C.POINTER(vp), C.POINTER(vp), i32],
        "mm_ctx_launch_count": [vp, C.POINTER(C.c_ulonglong)],
        "mm_ctx_set_tiles": [vp, i32, i32, i32],
        "mm_ctx_set_path": [vp, i32],
        "mm_ctx_set_slabs": [vp, i32],
        "mm_ctx_path": [vp, C.POINTER(i32)],
        "mm_ctx_set_profiling": [vp, i32],
        "mm_ctx_kernel_times": [vp, i32, C.POINTER(dbl), C.POINTER(C.c_ulonglong)],
    }
    for name, args in sigs.items():
        fn = getattr(lib, name)
        fn.argtypes = args
        fn.restype = i32
    lib.mm_last_error.argtypes = [vp]
    lib.mm_last_error.restype = C.c_char_p
    lib.mm_ctx_kernel_name.argtypes = [vp, i32]
    lib.mm_ctx_kernel_name.restype = C.c_char_p
    _lib = lib
    return lib


def _dt_code(dtype):
    if dtype in (torch.float32, "f32", np.float32):
        return MM_F32, torch.float32
    if dtype in (torch.float64, "f64", np.float64):
        return MM_F64, torch.float64
    raise ValueError(f"unsupported dtype {dtype}")


class Context:
    """One mesh on one GPU (mm_ctx).  Mirrors Mesh(n, dx) + State.material + the field-term
    list of the paper's scripts."""

    def __init__(self, n, d, dtype=torch.float32, device="cuda:0", tiles=None, allocate=True, path=0, slabs=0):
        self.lib = load_library()
        self.n = tuple(int(v) for v in n)
        self.d = tuple(float(v) for v in d)
        self.code, self.dtype = _dt_code(dtype)
        self.device = torch.device(device)
        self._h = C.c_void_p()
        st = self.lib.mm_ctx_create(*self.n, *self.d, self.code, C.byref(self._h))
        if st != 0:
            raise MMError(st, self.lib.mm_last_error(None).decode())
        if tiles is not None:
            self._call("mm_ctx_set_tiles", *[int(t) for t in tiles])
        if path:
            self._call("mm_ctx_set_path", int(path))
        if slabs:
            self._call("mm_ctx_set_slabs", int(slabs))
        self._ws = None
        if allocate:
            self.allocate()

    # -- plumbing
    def _call(self, name, *args):
        st = getattr(self.lib, name)(self._h, *args)
        if st != 0:
            raise MMError(st, self.lib.mm_last_error(self._h).decode())

    def workspace_bytes(self):
        p, s = C.c_size_t(), C.c_size_t()
        self._call("mm_ctx_workspace_bytes", C.byref(p), C.byref(s))
        return p.value, s.value

    def allocate(self):
        """torch owns the workspaces; the library only carves them up."""
        p, s = self.workspace_bytes()
        with torch.cuda.device(self.device):
            pers = torch.empty(p + 256, dtype=torch.uint8, device=self.device)
            scr = torch.empty(s + 256, dtype=torch.uint8, device=self.device)
        self._ws = (pers, scr)
        a = lambda t: (t.data_ptr() + 255) // 256 * 256
        self._call("mm_ctx_set_workspace", a(pers), p, a(scr), s)
        self.use_current_stream()

    def use_current_stream(self):
        self._call("mm_ctx_set_stream", torch.cuda.current_stream(self.device).cuda_stream)

    def close(self):
        if self._h:
            self.lib.mm_ctx_destroy(self._h)
            self._h = C.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- configuration
    def set_material(self, Ms, Aex=0.0, Ku=0.0, axis=(0.0, 0.0, 1.0), alpha=0.0, gamma=2.211e5):
        ax = (C.c_double * 3)(*axis)
        self._call("mm_set_material", Ms, Aex, Ku, ax, alpha, gamma)

    def set_zeeman(self, Hext):
        self._call("mm_set_zeeman", (C.c_double * 3)(*Hext))

    def set_material_cells(self, Ms_cells=None, A_cells=None):
        """Per-cell Ms / A as cuda tensors of shape n in the context dtype (kept alive by the context)."""
        for t in (Ms_cells, A_cells):
            if t is not None and not (t.is_cuda and t.dtype == self.dtype and t.is_contiguous()
                                      and tuple(t.shape) == self.n):
                raise ValueError(f"expected contiguous cuda {self.dtype} tensor of shape {self.n}")
        self._cells = (Ms_cells, A_cells)
        self._call("mm_set_material_cells", Ms_cells.data_ptr() if Ms_cells is not None else None,
                   A_cells.data_ptr() if A_cells is not None else None)

    def set_dmi(self, D, e=DMI_INTERFACIAL):
        self._call("mm_set_dmi", float(D), (C.c_double * 9)(*[float(v) for row in e for v in row]))

    def set_stt(self, p, a_damp, a_field=0.0):
        self._call("mm_set_stt", (C.c_double * 3)(*p), float(a_damp), float(a_field))

    def set_terms(self, mask):
        self._call("mm_set_terms", int(mask))

    def demag_init(self):
        self._call("mm_demag_init")

    PATH_NAMES = ("generic", "fast", "mixed", "embedded")

    @property
    def path_name(self):
        """'generic' (z-first passes), 'fast' (x-first register-stage kernels), 'mixed' (mixed-radix x-first,
        shared-memory stages) or 'embedded' (x-first kernels on an enclosing mesh)."""
        f = C.c_int()
        self._call("mm_ctx_path", C.byref(f))
        return self.PATH_NAMES[f.value]

    @property
    def launch_count(self):
        v = C.c_ulonglong()
        self._call("mm_ctx_launch_count", C.byref(v))
        return v.value

    def set_profiling(self, on=True):
        self._call("mm_ctx_set_profiling", 1 if on else 0)

    KERNEL_KINDS = ("S1", "S2", "S3", "S4", "S5", "S6")   # mm_ctx_kernel_times kinds 0..5

    def kernel_name(self, kind):
        """__global__ function launched for kernel kind 0..5 (as in an ncu launch list)."""
        return self.lib.mm_ctx_kernel_name(self._h, int(kind)).decode()

    def kernel_times(self, reset=True):
        """{kind: (total ms, launches)} since the last reset, kinds 'S1'..'S6'; synchronises."""
        ms = (C.c_double * 8)()
        cnt = (C.c_ulonglong * 8)()
        self._call("mm_ctx_kernel_times", 1 if reset else 0, ms, cnt)
        return {k: (ms[i], cnt[i]) for i, k in enumerate(self.KERNEL_KINDS)}

    # -- device calls
    def _check(self, t):
        if not (t.is_cuda and t.dtype == self.dtype and t.is_contiguous()
                and tuple(t.shape) == self.n + (3,)):
            raise ValueError(f"expected contiguous cuda {self.dtype} tensor of shape {self.n + (3,)}")
        return t

    def _field(self, name, m, out):
        self._check(m)
        out = torch.empty_like(m) if out is None else self._check(out)
        self._call(name, m.data_ptr(), out.data_ptr())
        return out

    def demag_field(self, m, out=None):
        return self._field("mm_demag_field", m, out)

    def demag_field_static(self, m, out=None):
        """mm_demag_field with the spectra in the library's static device array (no allocation in the library;
        pass `out` to allocate nothing here either).  Calls that overlap on the GPU race on that array."""
        return self._field("mm_demag_field_static", m, out)

    def static_scratch_info(self):
        """(capacity, needed) in bytes; also resolves the static array's address on the current device."""
        cap, need = C.c_size_t(0), C.c_size_t(0)
        self._call("mm_static_scratch_info", C.byref(cap), C.byref(need))
        return cap.value, need.value

    def exchange_field(self, m, out=None):
        return self._field("mm_exchange_field", m, out)

    def dmi_field(self, m, out=None):
        return self._field("mm_dmi_field", m, out)

    def heff(self, m, out=None):
        return self._field("mm_heff", m, out)

    def llg_rhs(self, m, out=None):
        return self._field("mm_llg_rhs", m, out)

    def rk_step(self, m, dt):
        self._check(m)
        self._call("mm_rk_step", m.data_ptr(), float(dt))
        return m

    def rk_steps(self, m, dt, n):
        """n RK4 steps as replays of a CUDA graph the library captures and caches (mm_rk_steps)."""
        self._check(m)
        self._call("mm_rk_steps", m.data_ptr(), float(dt), int(n))
        return m

    def rkf45_init(self, t0=0.0, dt0=1e-13, tol=1e-6, dt_min=0.0, dt_max=1.0):
        self._call("mm_rkf45_init", float(t0), float(dt0), float(tol), float(dt_min), float(dt_max))

    def rkf45_step(self, m):
        """Enqueues one attempted RKF45 step (accept/reject and the next dt are decided on the device)."""
        self._check(m)
        self._call("mm_rkf45_step", m.data_ptr())
        return m

    def rkf45_state(self):
        """Synchronises; dict(t, dt_next, err, dt_last, accepted, n_accepted, n_rejected)."""
        t, dn, er, dl = C.c_double(), C.c_double(), C.c_double(), C.c_double()
        acc, na, nr = C.c_int(), C.c_ulonglong(), C.c_ulonglong()
        self._call("mm_rkf45_state", C.byref(t), C.byref(dn), C.byref(er), C.byref(dl), C.byref(acc),
                   C.byref(na), C.byref(nr))
        return {"t": t.value, "dt_next": dn.value, "err": er.value, "dt_last": dl.value,
                "accepted": bool(acc.value), "n_accepted": na.value, "n_rejected": nr.value}

    def minimize_init(self, tau0=1e-6, tau_min=1e-9, tau_max=1e-3, tol=1e-8):
        self._call("mm_minimize_init", tau0, tau_min, tau_max, tol)

    def minimize_step(self, m):
        self._check(m)
        self._call("mm_minimize_step", m.data_ptr())

    def minimize_state(self):
        """(iterations, tau_last, dm_max, converged); synchronises."""
        n, tau, dm, cv = C.c_ulonglong(), C.c_double(), C.c_double(), C.c_int()
        self._call("mm_minimize_state", C.byref(n), C.byref(tau), C.byref(dm), C.byref(cv))
        return n.value, tau.value, dm.value, bool(cv.value)

    def minimize(self, m, max_iter=10000, check_every=10):
        """Runs the minimiser in place; returns (iterations, converged)."""
        self._check(m)
        n, cv = C.c_ulonglong(), C.c_int()
        self._call("mm_minimize", m.data_ptr(), int(max_iter), int(check_every), C.byref(n), C.byref(cv))
        return n.value, bool(cv.value)

    def nhat_export(self):
        o = tuple(1 if v == 1 else v + 1 for v in self.n)
        out = torch.empty((6,) + o, dtype=self.dtype, device=self.device)
        self._call("mm_demag_nhat_export", out.data_ptr())
        return out

    # -- host-buffer calls (numpy arrays or CPU tensors; copies happen inside the library)
    def _host(self, name, m_host, out_host):
        a = m_host if isinstance(m_host, np.ndarray) else m_host.numpy()
        if out_host is None:
            out_host = np.empty_like(a)
        b = out_host if isinstance(out_host, np.ndarray) else out_host.numpy()
        want = np.float32 if self.dtype == torch.float32 else np.float64
        for x in (a, b):
            if x.dtype != want or not x.flags.c_contiguous or x.shape != self.n + (3,):
                raise ValueError("host buffers must be C-contiguous, context dtype, [nx,ny,nz,3]")
        self._call(name, a.ctypes.data, b.ctypes.data)
        return out_host

    def demag_field_host(self, m_host, out_host=None):
        return self._host("mm_demag_field_host", m_host, out_host)

    def heff_host(self, m_host, out_host=None):
        return self._host("mm_heff_host", m_host, out_host)

    def llg_rhs_host(self, m_host, out_host=None):
        return self._host("mm_llg_rhs_host", m_host, out_host)

    def llg_rhs_host_batch(self, m_hosts, out_hosts):
        """Independent evaluations on lists of host buffers, copies pipelined beside the kernels (pinned memory)."""
        return self._host_batch("mm_llg_rhs_host_batch", m_hosts, out_hosts)

    def demag_field_host_batch(self, m_hosts, out_hosts):
        return self._host_batch("mm_demag_field_host_batch", m_hosts, out_hosts)

    def heff_host_batch(self, m_hosts, out_hosts):
        return self._host_batch("mm_heff_host_batch", m_hosts, out_hosts)

    def _host_batch(self, name, m_hosts, out_hosts):
        want = np.float32 if self.dtype == torch.float32 else np.float64
        arrs = []
        for lst in (m_hosts, out_hosts):
            a = [x if isinstance(x, np.ndarray) else x.numpy() for x in lst]
            for x in a:
                if x.dtype != want or not x.flags.c_contiguous or x.shape != self.n + (3,):
                    raise ValueError("host buffers must be C-contiguous, context dtype, [nx,ny,nz,3]")
            arrs.append(a)
        if len(arrs[0]) != len(arrs[1]):
            raise ValueError("as many outputs as inputs")
        k = len(arrs[0])
        pin = (C.c_void_p * max(k, 1))(*[x.ctypes.data for x in arrs[0]])
        pout = (C.c_void_p * max(k, 1))(*[x.ctypes.data for x in arrs[1]])
        self._call(name, pin, pout, k)
        return out_hosts

    def rk_step_host(self, m_host, dt):
        a = m_host if isinstance(m_host, np.ndarray) else m_host.numpy()
        self._call("mm_rk_step_host", a.ctypes.data, float(dt))
        return m_host
