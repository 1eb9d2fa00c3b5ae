"""CPU oracle for the Fourier split-operator step -- TEST INFRASTRUCTURE, NOT PRODUCT.

Thin ctypes wrapper around ``oracle/sso_oracle.c`` (plain C, fp64, written from
the paper; see that file's header for the citations and the pins).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_1012_3911_b200`` and that package imports nothing from here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "sso_oracle.c"
_LIB = _HERE / "libsso_oracle.so"

FIELD_NONE, FIELD_E, FIELD_A = 0, 1, 2


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (``-O2 -fopenmp``; no -ffast-math)."""
    if force or (not _LIB.exists()) or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.{os.getpid()}.tmp")
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


class _Params(ctypes.Structure):
    _fields_ = [
        ("ndim", ctypes.c_int32),
        ("ncomp", ctypes.c_int32),
        ("n", ctypes.c_int64 * 3),
        ("dx", ctypes.c_double * 3),
        ("dt", ctypes.c_double),
        ("mass", ctypes.c_double),
        ("c", ctypes.c_double),
        ("charge", ctypes.c_double),
        ("field_kind", ctypes.c_int32),
        ("pad_", ctypes.c_int32),
        ("nvals", ctypes.c_int64),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(str(build()))
        dp = ctypes.POINTER(ctypes.c_double)
        i64p = ctypes.POINTER(ctypes.c_int64)
        L.orc_max_threads.restype = ctypes.c_int
        L.orc_set_threads.argtypes = [ctypes.c_int]
        L.orc_fft.argtypes = [dp, ctypes.c_int, i64p, ctypes.c_int]
        L.orc_grids.argtypes = [ctypes.c_int64, ctypes.c_double, dp, dp]
        L.orc_dirac_matrices.argtypes = [ctypes.c_int, dp]
        L.orc_dirac_kinetic_matrix.argtypes = [ctypes.c_int, ctypes.c_int, dp, ctypes.c_double, ctypes.c_double, ctypes.c_double, dp]
        L.orc_dirac_u.argtypes = [ctypes.c_int, ctypes.c_int, dp, ctypes.c_double, ctypes.c_double, dp]
        L.orc_step.argtypes = [ctypes.POINTER(_Params), dp, dp, dp, ctypes.c_int64, ctypes.c_int64]
        L.orc_step.restype = ctypes.c_int
        L.orc_step_apos.argtypes = [ctypes.POINTER(_Params), dp, dp, dp, dp, ctypes.c_int64, ctypes.c_int64]
        L.orc_step_apos.restype = ctypes.c_int
        L.orc_alpha_rotation.argtypes = [ctypes.c_int, ctypes.c_int, dp, dp]
        L.orc_norm.argtypes = [ctypes.POINTER(_Params), dp]
        L.orc_norm.restype = ctypes.c_double
        L.orc_inverse_sample.argtypes = [ctypes.POINTER(_Params), dp, dp, dp, ctypes.c_int64, dp]
        L.orc_half_step_to_k.argtypes = [ctypes.POINTER(_Params), dp, dp, dp, ctypes.c_int64]
        L.orc_half_step_to_k.restype = ctypes.c_int
        L.orc_overlap.argtypes = [ctypes.POINTER(_Params), dp, dp, dp]
        L.orc_expect_r.argtypes = [ctypes.POINTER(_Params), dp, dp]
        L.orc_expect_p.argtypes = [ctypes.POINTER(_Params), dp, dp]
        L.orc_spectrum.argtypes = [dp, ctypes.c_int64, ctypes.c_double, dp, ctypes.c_int64, dp]
        L.orc_filter_accumulate.argtypes = [ctypes.POINTER(_Params), dp, dp, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if a is not None else None


def max_threads() -> int:
    return int(lib().orc_max_threads())


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def fft(x: np.ndarray, sign: int) -> np.ndarray:
    """N-d DFT of a complex128 array: sign=-1 unnormalised forward, +1 inverse with 1/N."""
    y = np.ascontiguousarray(x, dtype=np.complex128).copy()
    n = (ctypes.c_int64 * y.ndim)(*y.shape)
    lib().orc_fft(_dp(y), y.ndim, n, int(sign))
    return y


def grids(n: int, dx: float):
    r = np.empty(n)
    k = np.empty(n)
    lib().orc_grids(n, dx, _dp(r), _dp(k))
    return r, k


def dirac_matrices(ncomp: int):
    """(alpha[3], beta) as the oracle uses them (eq. 16 / eq. 17 of the paper)."""
    out = np.zeros((4, ncomp, ncomp), dtype=np.complex128)
    lib().orc_dirac_matrices(ncomp, _dp(out))
    return out[:3], out[3]


def dirac_kinetic_matrix(ncomp: int, p, mass: float, c: float, tau: float) -> np.ndarray:
    p = np.ascontiguousarray(p, dtype=np.float64)
    U = np.zeros((ncomp, ncomp), dtype=np.complex128)
    lib().orc_dirac_kinetic_matrix(ncomp, p.size, _dp(p), mass, c, tau, _dp(U))
    return U


def dirac_u(ncomp: int, p, mass: float, c: float) -> np.ndarray:
    p = np.ascontiguousarray(p, dtype=np.float64)
    u = np.zeros((ncomp, ncomp), dtype=np.complex128)
    lib().orc_dirac_u(ncomp, p.size, _dp(p), mass, c, _dp(u))
    return u


def alpha_rotation(ncomp: int, a) -> np.ndarray:
    """exp(i sum_i a_i alpha_i) in the closed form of eq. 23/24, as the oracle evaluates it."""
    a = np.ascontiguousarray(a, dtype=np.float64)
    M = np.zeros((ncomp, ncomp), dtype=np.complex128)
    lib().orc_alpha_rotation(ncomp, a.size, _dp(a), _dp(M))
    return M


def spectrum(chi, dts: float, E) -> np.ndarray:
    """chi~(E) of eq. 41 from samples chi(n dts), n < len(chi), T = len(chi) dts."""
    chi = np.ascontiguousarray(chi, dtype=np.complex128)
    E = np.ascontiguousarray(E, dtype=np.float64)
    out = np.zeros(E.size, dtype=np.complex128)
    lib().orc_spectrum(_dp(chi), chi.size, float(dts), _dp(E), E.size, _dp(out))
    return out


class Solver:
    """The oracle's view of one problem: grid, constants, potential, field table."""

    def __init__(self, sizes, dx, dt, ncomp=1, mass=1.0, c=137.036, charge=-1.0):
        sizes = [int(s) for s in sizes]
        dx = [float(d) for d in dx]
        assert 1 <= len(sizes) <= 3 and len(dx) == len(sizes)
        self.sizes = tuple(sizes)
        self.p = _Params()
        self.p.ndim = len(sizes)
        self.p.ncomp = ncomp
        for a in range(3):
            self.p.n[a] = sizes[a] if a < len(sizes) else 1
            self.p.dx[a] = dx[a] if a < len(sizes) else 1.0
        self.p.dt = dt
        self.p.mass, self.p.c, self.p.charge = mass, c, charge
        self.p.field_kind = FIELD_NONE
        self.p.nvals = 0
        self.V = None
        self.step_avg = None
        self.A_pos = None
        self.time_index = 0

    def set_potential(self, V):
        self.V = None if V is None else np.ascontiguousarray(V, dtype=np.float64).reshape(self.sizes).copy()

    def set_field(self, kind, step_avg):
        self.p.field_kind = int(kind)
        if kind == FIELD_NONE:
            self.step_avg, self.p.nvals = None, 0
        else:
            self.step_avg = np.ascontiguousarray(step_avg, dtype=np.float64).reshape(-1, len(self.sizes)).copy()
            self.p.nvals = self.step_avg.shape[0]

    def set_vector_potential(self, A):
        """Step-averaged position-dependent A(r), shape (ndim, *sizes), applied in position space (eq. 26); None = off."""
        self.A_pos = None if A is None else np.ascontiguousarray(A, dtype=np.float64).reshape((len(self.sizes),) + self.sizes).copy()

    def set_time_index(self, n):
        self.time_index = int(n)

    def step(self, psi: np.ndarray, nsteps: int) -> np.ndarray:
        """Returns a new array; psi has shape (ncomp, *sizes) or sizes when ncomp == 1."""
        out = np.ascontiguousarray(psi, dtype=np.complex128).copy()
        assert out.size == self.p.ncomp * int(np.prod(self.sizes))
        if self.A_pos is not None:
            rc = lib().orc_step_apos(ctypes.byref(self.p), _dp(out), _dp(self.V), _dp(self.step_avg), _dp(self.A_pos), self.time_index, int(nsteps))
            if rc == -2:
                raise ValueError("oracle: the position-space vector potential needs a Dirac spinor (ncomp 2 or 4)")
        else:
            rc = lib().orc_step(ctypes.byref(self.p), _dp(out), _dp(self.V), _dp(self.step_avg), self.time_index, int(nsteps))
        if rc != 0:
            raise ValueError("oracle: field table shorter than the steps requested")
        self.time_index += int(nsteps)
        return out

    def norm(self, psi: np.ndarray) -> float:
        a = np.ascontiguousarray(psi, dtype=np.complex128)
        return float(lib().orc_norm(ctypes.byref(self.p), _dp(a)))

    def half_step_to_k(self, psi: np.ndarray, n: int) -> np.ndarray:
        out = np.ascontiguousarray(psi, dtype=np.complex128).copy()
        rc = lib().orc_half_step_to_k(ctypes.byref(self.p), _dp(out), _dp(self.V), _dp(self.step_avg), int(n))
        if rc != 0:
            raise ValueError("oracle: field table shorter than the steps requested")
        return out

    def inverse_sample(self, psik: np.ndarray, n: int, flat_index: int) -> np.ndarray:
        """psi_c(r_j) after steps 4+5 of step n, by the O(N) definition sum, for one flat grid index."""
        a = np.ascontiguousarray(psik, dtype=np.complex128)
        out = np.zeros(self.p.ncomp, dtype=np.complex128)
        Ebar = None
        if self.p.field_kind == FIELD_E:
            Ebar = np.ascontiguousarray(self.step_avg[n])
        lib().orc_inverse_sample(ctypes.byref(self.p), _dp(a), _dp(self.V), _dp(Ebar), int(flat_index), _dp(out))
        return out

    # observables
    def overlap(self, a: np.ndarray, b: np.ndarray) -> complex:
        """<a|b> = sum conj(a) b prod dx  (chi(t) of eq. 40 with a = psi(0), b = psi(t))."""
        a = np.ascontiguousarray(a, dtype=np.complex128)
        b = np.ascontiguousarray(b, dtype=np.complex128)
        out = np.zeros(2)
        lib().orc_overlap(ctypes.byref(self.p), _dp(a), _dp(b), _dp(out))
        return complex(out[0], out[1])

    def expect_r(self, psi: np.ndarray) -> np.ndarray:
        a = np.ascontiguousarray(psi, dtype=np.complex128)
        out = np.zeros(len(self.sizes))
        lib().orc_expect_r(ctypes.byref(self.p), _dp(a), _dp(out))
        return out

    def expect_p(self, psi: np.ndarray) -> np.ndarray:
        a = np.ascontiguousarray(psi, dtype=np.complex128)
        out = np.zeros(len(self.sizes))
        lib().orc_expect_p(ctypes.byref(self.p), _dp(a), _dp(out))
        return out

    def filter_accumulate(self, acc: np.ndarray, psi: np.ndarray, t: float, T: float, E: float, dts: float) -> None:
        """acc += psi (1 - cos(2 pi t/T)) exp(i E t) dts, in place (one term of eq. 42)."""
        assert acc.dtype == np.complex128 and acc.flags.c_contiguous
        a = np.ascontiguousarray(psi, dtype=np.complex128)
        lib().orc_filter_accumulate(ctypes.byref(self.p), _dp(acc), _dp(a), float(t), float(T), float(E), float(dts))
