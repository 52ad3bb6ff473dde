"""ctypes front end of the CPU oracle (oracle/mm_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the
CUDA package and the CUDA package imports nothing from here.

All arrays are fp64 numpy arrays of shape [nx, ny, nz, 3] (PAPER.md:130-132 layout).
Function-by-function citations are in the header of mm_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mm_oracle.c")
_LIB = os.path.join(_HERE, "libmm_oracle.so")

MU0 = 4.0e-7 * np.pi  # reading Q8

TERM_DEMAG, TERM_EXCHANGE, TERM_ANISOTROPY, TERM_ZEEMAN, TERM_DMI, TERM_STT = 1, 2, 4, 8, 16, 32

# DMI vectors e_k^DMI of PAPER.md:39, rows k = x, y, z
DMI_INTERFACIAL = ((0.0, 1.0, 0.0), (-1.0, 0.0, 0.0), (0.0, 0.0, 0.0))
DMI_BULK = ((1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0))


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (quadmath + OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC,
               "-lquadmath", "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


class _Problem(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("Ms", C.c_double), ("Aex", C.c_double), ("Ku", C.c_double),
                ("axis", C.c_double * 3), ("alpha", C.c_double), ("gamma", C.c_double),
                ("Hext", C.c_double * 3), ("terms", C.c_uint), ("Nhat", C.c_void_p),
                ("D", C.c_double), ("edmi", C.c_double * 9),
                ("stt_p", C.c_double * 3), ("stt_damp", C.c_double), ("stt_field", C.c_double),
                ("Ms_cells", C.c_void_p), ("A_cells", C.c_void_p)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def num_threads() -> int:
    return int(lib().orc_num_threads())


def newell_point(d, i, j, k):
    """N(xx,yy,zz,xy,xz,yz) at cell offset (i,j,k) by the literal 27-point definition (O1)."""
    out = np.zeros(6)
    lib().orc_newell_point(C.c_double(d[0]), C.c_double(d[1]), C.c_double(d[2]),
                           C.c_int(i), C.c_int(j), C.c_int(k), _p(out))
    return out


def newell_octant(n, d):
    """Octant table N[6, nx, ny, nz] (O1)."""
    N = np.zeros((6, n[0], n[1], n[2]))
    _chk(lib().orc_newell_octant(C.c_int(n[0]), C.c_int(n[1]), C.c_int(n[2]), C.c_double(d[0]),
                                 C.c_double(d[1]), C.c_double(d[2]), _p(N)), "newell_octant")
    return N


def demag_direct(N, Ms, m):
    """O3: full O(n^2) real-space sum."""
    m = _f64(m)
    nx, ny, nz = m.shape[:3]
    H = np.zeros_like(m)
    _chk(lib().orc_demag_direct(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(N), C.c_double(Ms),
                                _p(m), _p(H)), "demag_direct")
    return H


def demag_direct_sampled(N, Ms, m, cells):
    """O3 at chosen flat cell indices; returns [nsamp, 3]."""
    m = _f64(m)
    nx, ny, nz = m.shape[:3]
    cells = np.ascontiguousarray(cells, dtype=np.int64)
    Hs = np.zeros((len(cells), 3))
    _chk(lib().orc_demag_direct_sampled(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(N),
                                        C.c_double(Ms), _p(m), C.c_int(len(cells)), _p(cells),
                                        _p(Hs)), "demag_direct_sampled")
    return Hs


def demag_dft(N, Ms, m):
    """O4: literal-DFT zero-padded convolution (tiny meshes only)."""
    m = _f64(m)
    nx, ny, nz = m.shape[:3]
    H = np.zeros_like(m)
    _chk(lib().orc_demag_dft(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(N), C.c_double(Ms), _p(m),
                             _p(H)), "demag_dft")
    return H


def padded(n):
    """Period of the paper's zero-padding: 2n, or 1 for a one-cell axis (Q10)."""
    return 1 if n == 1 else 2 * n


def fft_period(n):
    """Period the oracle's radix-2 FFT path uses: 2n for powers of two, else the next power of
    two above 2n (same linear convolution, reading Q27)."""
    return int(lib().orc_fft_period(C.c_int(n)))


def demag_fft_nhat(N, return_max_imag=False):
    """O5 set-up: real Fourier-space tensor Nhat[6, Px, Py, Pz]."""
    _, nx, ny, nz = N.shape
    Nhat = np.zeros((6, fft_period(nx), fft_period(ny), fft_period(nz)))
    mi = C.c_double(0.0)
    _chk(lib().orc_demag_fft_nhat(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(N), _p(Nhat),
                                  C.byref(mi)), "demag_fft_nhat")
    return (Nhat, mi.value) if return_max_imag else Nhat


def demag_fft(Nhat, Ms, m):
    """O5: demag field by the oracle's own FFT path."""
    m = _f64(m)
    nx, ny, nz = m.shape[:3]
    H = np.zeros_like(m)
    _chk(lib().orc_demag_fft(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(Nhat), C.c_double(Ms),
                             _p(m), _p(H)), "demag_fft")
    return H


def exchange(d, Ms, Aex, m):
    """O6."""
    m = _f64(m)
    nx, ny, nz = m.shape[:3]
    H = np.zeros_like(m)
    _chk(lib().orc_exchange(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(d[0]),
                            C.c_double(d[1]), C.c_double(d[2]), C.c_double(Ms), C.c_double(Aex),
                            _p(m), _p(H)), "exchange")
    return H


def anisotropy(Ms, Ku, axis, m):
    """O7."""
    m = _f64(m)
    u = _f64(axis)
    H = np.zeros_like(m)
    _chk(lib().orc_anisotropy(C.c_size_t(m.size // 3), C.c_double(Ms), C.c_double(Ku), _p(u),
                              _p(m), _p(H)), "anisotropy")
    return H


def dmi(d, Ms, D, e, m):
    """O11: DMI field of eq. 3 for the DMI vectors e[k] (3 x 3)."""
    m = _f64(m)
    nx, ny, nz = m.shape[:3]
    ev = _f64(np.asarray(e).reshape(9))
    H = np.zeros_like(m)
    _chk(lib().orc_dmi(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(d[0]), C.c_double(d[1]),
                       C.c_double(d[2]), C.c_double(Ms), C.c_double(D), _p(ev), _p(m), _p(H)), "dmi")
    return H


def stt(p, a_damp, a_field, m):
    """O12: spin-torque effective field a_damp (m x p) + a_field p."""
    m = _f64(m)
    pv = _f64(p)
    H = np.zeros_like(m)
    _chk(lib().orc_stt(C.c_size_t(m.size // 3), _p(pv), C.c_double(a_damp), C.c_double(a_field),
                       _p(m), _p(H)), "stt")
    return H


def llg_torque(alpha, gamma, m, H):
    """O8 on a given field."""
    m = _f64(m)
    H = _f64(H)
    out = np.zeros_like(m)
    _chk(lib().orc_llg_torque(C.c_size_t(m.size // 3), C.c_double(alpha), C.c_double(gamma),
                              _p(m), _p(H), _p(out)), "llg_torque")
    return out


class _BBState(C.Structure):
    _fields_ = [("n", C.c_long), ("tau0", C.c_double), ("tau_min", C.c_double), ("tau_max", C.c_double),
                ("tol", C.c_double), ("tau", C.c_double), ("dm_max", C.c_double), ("converged", C.c_int),
                ("m_prev", C.c_void_p), ("g_prev", C.c_void_p)]


class BBMinimizer:
    """O13: Barzilai-Borwein minimiser state around orc_bb_step (reading Q30)."""

    def __init__(self, problem, m, tau0=1e-6, tau_min=1e-9, tau_max=1e-3, tol=1e-8):
        self.problem = problem
        self.m = _f64(m).copy()
        self._mp = np.zeros_like(self.m)
        self._gp = np.zeros_like(self.m)
        self.st = _BBState(0, tau0, tau_min, tau_max, tol, 0.0, 0.0, 0, self._mp.ctypes.data,
                           self._gp.ctypes.data)

    def step(self):
        _chk(lib().orc_bb_step(C.byref(self.problem._c()), _p(self.m), C.byref(self.st)), "bb_step")
        return self.st.tau, self.st.dm_max, bool(self.st.converged)

    def minimize(self, max_iter=10000):
        while self.st.n < max_iter and not self.st.converged:
            self.step()
        return self.m, int(self.st.n), bool(self.st.converged)


@dataclass
class Problem:
    """Mesh + material + enabled terms; mirrors the paper's state.material / field-term list
    (PAPER.md:84-161)."""
    n: tuple
    d: tuple
    Ms: float
    Aex: float = 0.0
    Ku: float = 0.0
    axis: tuple = (0.0, 0.0, 1.0)
    alpha: float = 0.0
    gamma: float = 2.211e5
    Hext: tuple = (0.0, 0.0, 0.0)
    terms: int = TERM_DEMAG | TERM_EXCHANGE
    D: float = 0.0
    edmi: tuple = DMI_INTERFACIAL
    stt_p: tuple = (0.0, 0.0, 1.0)
    stt_damp: float = 0.0
    stt_field: float = 0.0
    Ms_cells: np.ndarray | None = field(default=None, repr=False)   # [nx, ny, nz] or None (uniform Ms)
    A_cells: np.ndarray | None = field(default=None, repr=False)    # [nx, ny, nz] or None (uniform Aex)
    N: np.ndarray | None = field(default=None, repr=False)
    Nhat: np.ndarray | None = field(default=None, repr=False)

    def prepare(self):
        """One-off: Newell table and its transform (excluded from any timing)."""
        if self.terms & TERM_DEMAG and self.Nhat is None:
            if self.N is None:
                self.N = newell_octant(self.n, self.d)
            self.Nhat = demag_fft_nhat(self.N)
        return self

    def _c(self):
        s = _Problem()
        s.nx, s.ny, s.nz = self.n
        s.dx, s.dy, s.dz = self.d
        s.Ms, s.Aex, s.Ku = self.Ms, self.Aex, self.Ku
        s.axis[:] = list(self.axis)
        s.alpha, s.gamma = self.alpha, self.gamma
        s.Hext[:] = list(self.Hext)
        s.terms = self.terms
        s.Nhat = self.Nhat.ctypes.data if self.Nhat is not None else None
        s.D = self.D
        s.edmi[:] = [float(v) for row in self.edmi for v in row]
        s.stt_p[:] = list(self.stt_p)
        s.stt_damp, s.stt_field = self.stt_damp, self.stt_field
        if self.Ms_cells is not None:
            self.Ms_cells = _f64(self.Ms_cells)
            s.Ms_cells = self.Ms_cells.ctypes.data
        if self.A_cells is not None:
            self.A_cells = _f64(self.A_cells)
            s.A_cells = self.A_cells.ctypes.data
        return s

    def heff(self, m):
        m = _f64(m)
        H = np.zeros_like(m)
        _chk(lib().orc_heff(C.byref(self._c()), _p(m), _p(H)), "heff")
        return H

    def llg_rhs(self, m):
        m = _f64(m)
        out = np.zeros_like(m)
        _chk(lib().orc_llg_rhs(C.byref(self._c()), _p(m), _p(out)), "llg_rhs")
        return out

    def rkf45_step(self, m, dt, tol, dt_min=0.0, dt_max=1.0):
        """O10; one attempted RKF45 step.  Returns (m_new, err, accepted, dt_next); m_new is the
        input when the attempt is rejected."""
        m = _f64(m).copy()
        err, acc, dtn = C.c_double(), C.c_int(), C.c_double()
        _chk(lib().orc_rkf45_step(C.byref(self._c()), _p(m), C.c_double(dt), C.c_double(tol),
                                  C.c_double(dt_min), C.c_double(dt_max), C.byref(err),
                                  C.byref(acc), C.byref(dtn)), "rkf45_step")
        return m, err.value, bool(acc.value), dtn.value

    def rk4_step(self, m, dt):
        """O9; returns the new m (input untouched)."""
        m = _f64(m).copy()
        _chk(lib().orc_rk4_step(C.byref(self._c()), _p(m), C.c_double(dt)), "rk4_step")
        return m
