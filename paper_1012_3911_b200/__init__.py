"""paper_1012_3911_b200 -- Python binding of libsso.so, the B200-native Fourier split-operator library.

Argument marshalling only: every step of the path (potential phases, FFTs, kinetic factors, norm)
runs in the CUDA kernels behind the C ABI declared in ``include/sso.h``.  PyTorch is used by callers
for device memory and streams; this module needs neither torch nor numpy to load.  There is no CPU
fallback: if the shared library is missing the import of :func:`lib` fails loudly.

The operation is one Fourier split-operator step (eq. 7, 76 eq. 8) -- see
``include/sso.h`` for the conventions.
"""
from __future__ import annotations

import ctypes
from pathlib import Path
from typing import Optional, Sequence

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libsso.so"

OK, ERR_INVALID, ERR_UNSUPPORTED, ERR_ALLOC, ERR_CUDA, ERR_STATE = 0, 1, 2, 3, 4, 5
C64, C128 = 0, 1
FIELD_NONE, FIELD_E, FIELD_A = 0, 1, 2
OPT_LINES_PER_TILE_CONTIG, OPT_LINES_PER_TILE_STRIDED, OPT_POTENTIAL_PHASE = 1, 2, 3
OPT_GROUPS_PER_CTA, OPT_RING_BUFFERS, OPT_THREADS_PER_CTA, OPT_STRIDED_RING, OPT_DIRAC_TABLE, OPT_TILE_ORDER, OPT_LINES_PER_TILE_MIDDLE, OPT_CLUSTER_1D = 4, 5, 6, 7, 8, 9, 10, 11

# every symbol include/sso.h declares
SYMBOLS = (
    "sso_plan_create", "sso_set_constants", "sso_set_potential", "sso_set_field", "sso_set_time_index",
    "sso_get_time_index", "sso_step", "sso_step_host", "sso_norm", "sso_set_option", "sso_launch_count",
    "sso_destroy", "sso_last_error", "sso_version", "sso_profile_step", "sso_pass_name",
    "sso_set_vector_potential", "sso_overlap", "sso_expect_position", "sso_expect_momentum", "sso_spectrum",
    "sso_filter_accumulate", "sso_step_observe", "sso_norm_static",
)
PASS_KINDS = 9
NORM_STATIC_CHUNK, NORM_STATIC_MAX_COUNT = 8192, 1 << 28  # SSO_NORM_STATIC_* of include/sso.h


class SsoError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"sso error {code}: {msg}")
        self.code = code


_lib = None


def lib() -> ctypes.CDLL:
    """Load libsso.so (built in-tree by ``paper_1012_3911_b200.build``); raises if it is missing."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise ImportError(f"{LIB_PATH} not found: run `python -m paper_1012_3911_b200.build` (there is no CPU fallback)")
        L = ctypes.CDLL(str(LIB_PATH))
        vp, i64, dbl, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int
        L.sso_plan_create.argtypes = [ctypes.POINTER(vp), ci, ctypes.POINTER(i64), ctypes.POINTER(dbl), dbl, ci, ci]
        L.sso_set_constants.argtypes = [vp, dbl, dbl, dbl]
        L.sso_set_potential.argtypes = [vp, vp, ci, vp]
        L.sso_set_field.argtypes = [vp, ci, vp, i64]
        L.sso_set_vector_potential.argtypes = [vp, vp, ci, vp]
        L.sso_set_time_index.argtypes = [vp, i64]
        L.sso_get_time_index.argtypes = [vp, ctypes.POINTER(i64)]
        L.sso_step.argtypes = [vp, vp, i64, vp]
        L.sso_step_host.argtypes = [vp, vp, i64]
        L.sso_norm.argtypes = [vp, vp, ctypes.POINTER(dbl), vp]
        L.sso_set_option.argtypes = [vp, ci, i64]
        L.sso_launch_count.argtypes = [vp, i64, ctypes.POINTER(i64)]
        L.sso_destroy.argtypes = [vp]
        L.sso_last_error.argtypes = [vp]
        L.sso_last_error.restype = ctypes.c_char_p
        L.sso_version.restype = ctypes.c_char_p
        L.sso_profile_step.argtypes = [vp, vp, i64, vp, ctypes.POINTER(i64), ctypes.POINTER(dbl)]
        L.sso_pass_name.argtypes = [ci]
        L.sso_overlap.argtypes = [vp, vp, vp, ctypes.POINTER(dbl), vp]
        L.sso_expect_position.argtypes = [vp, vp, ctypes.POINTER(dbl), vp]
        L.sso_expect_momentum.argtypes = [vp, vp, ctypes.POINTER(dbl), vp]
        L.sso_spectrum.argtypes = [vp, vp, i64, dbl, vp, i64, vp, vp]
        L.sso_filter_accumulate.argtypes = [vp, vp, vp, dbl, dbl, dbl, dbl, vp]
        L.sso_step_observe.argtypes = [vp, vp, i64, vp, vp, dbl, dbl, dbl, dbl, ctypes.POINTER(dbl), vp]
        L.sso_pass_name.restype = ctypes.c_char_p
        L.sso_norm_static.argtypes = [vp, ci, i64, dbl, vp, vp]
        for name in SYMBOLS:
            if name not in ("sso_last_error", "sso_version", "sso_pass_name"):
                getattr(L, name).restype = ci
        _lib = L
    return _lib


def version() -> str:
    return lib().sso_version().decode()


def _ptr(x) -> Optional[int]:
    """Address of a torch tensor / numpy array / raw int; None stays NULL."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError(f"cannot take the address of {type(x)}")


def _check_buffer(x, want_bytes: int, elem_bytes: int, device: Optional[bool], what: str) -> None:
    """The C ABI takes bare pointers and cannot check them: refuse a tensor/array whose size, element width,
    contiguity or residence does not match the plan.  Raw integer addresses are the caller's responsibility."""
    if x is None or isinstance(x, int):
        return
    if hasattr(x, "data_ptr"):  # torch tensor
        if device is not None and bool(x.is_cuda) != device:
            raise ValueError(f"{what}: expected a {'CUDA' if device else 'host'} tensor")
        if not x.is_contiguous():
            raise ValueError(f"{what}: tensor must be contiguous")
        nbytes, esz = x.numel() * x.element_size(), x.element_size()
    elif hasattr(x, "ctypes"):  # numpy array
        if device:
            raise ValueError(f"{what}: expected a CUDA tensor, got a host array")
        if not x.flags["C_CONTIGUOUS"]:
            raise ValueError(f"{what}: array must be C-contiguous")
        nbytes, esz = x.nbytes, x.itemsize
    else:
        return
    if esz != elem_bytes:
        raise ValueError(f"{what}: element size {esz} bytes, the plan expects {elem_bytes}")
    if nbytes != want_bytes:
        raise ValueError(f"{what}: {nbytes} bytes, the plan expects {want_bytes}")


def _stream(s) -> Optional[int]:
    if s is None:
        return None
    if isinstance(s, int):
        return s or None
    return s.cuda_stream  # torch.cuda.Stream


def norm_static(psi, vol: float, out, precision: Optional[int] = None, count: Optional[int] = None, stream=None) -> None:
    """``sso_norm_static``: out[0] = vol * sum |psi|^2 for callers that must not allocate device memory.

    No plan is involved and the library calls neither cudaMalloc nor cudaFree: the partial sums go to an array
    built into libsso.so (256 KiB per GPU, which is why ``count`` may not exceed ``NORM_STATIC_MAX_COUNT``).  Use it
    when the application's arena already owns all of HBM, when the time loop cannot afford the device-wide wait of
    an allocation, or when there is only a pointer to somebody else's wavefunction and no plan.  ``psi`` is a
    contiguous CUDA tensor of complex64/complex128 (or a raw device address, then ``precision`` and ``count`` are
    required), ``out`` a CUDA float64 tensor with at least one element (or a raw address) that receives the result;
    the caller allocates both.  Nothing is synchronised or copied to the host: read ``out`` after the stream has
    finished.  All calls on a device share the built-in array, so calls whose kernels could overlap on the GPU must
    be ordered by the caller; make the first call on a device during set-up (it resolves the array's address).
    """
    if hasattr(psi, "data_ptr"):
        if not psi.is_cuda or not psi.is_contiguous():
            raise ValueError("psi: expected a contiguous CUDA tensor")
        if not psi.is_complex():
            raise ValueError("psi: expected a complex64 or complex128 tensor")
        if precision is None:
            precision = C128 if psi.element_size() == 16 else C64
        if count is None:
            count = psi.numel()
    if precision is None or count is None:
        raise ValueError("precision and count are required with a raw psi address")
    if hasattr(out, "data_ptr") and (not out.is_cuda or out.element_size() != 8 or out.numel() < 1):
        raise ValueError("out: expected a CUDA float64 tensor with at least one element")
    rc = lib().sso_norm_static(_ptr(psi), int(precision), int(count), float(vol), _ptr(out), _stream(stream))
    if rc != OK:
        raise SsoError(rc, (lib().sso_last_error(None) or b"").decode())


class Plan:
    """Thin owner of an ``sso_plan*``; method names follow the C ABI (sso_<name>)."""

    def __init__(self, sizes: Sequence[int], dx: Sequence[float], dt: float, ncomp: int = 1, precision: int = C128):
        L = lib()
        nd = len(sizes)
        self._h = ctypes.c_void_p()
        szs = (ctypes.c_int64 * max(nd, 1))(*[int(s) for s in sizes])
        dxs = (ctypes.c_double * max(nd, 1))(*[float(d) for d in dx])
        rc = L.sso_plan_create(ctypes.byref(self._h), nd, szs, dxs, float(dt), int(ncomp), int(precision))
        if rc != OK:
            raise SsoError(rc, L.sso_last_error(None).decode())
        self.sizes, self.ncomp, self.precision = tuple(int(s) for s in sizes), int(ncomp), int(precision)
        self._npts = 1
        for n in self.sizes:
            self._npts *= n
        self._esz = 16 if self.precision == C128 else 8
        self._psi_bytes = self._npts * self.ncomp * self._esz

    def _ck(self, rc: int) -> None:
        if rc != OK:
            raise SsoError(rc, lib().sso_last_error(self._h).decode())

    def set_constants(self, mass: float, c: float, charge: float) -> None:
        self._ck(lib().sso_set_constants(self._h, mass, c, charge))

    def set_potential(self, V, on_device: bool = False, stream=None) -> None:
        """V: float64 array of shape sizes (numpy on host, or a torch CUDA tensor with on_device=True); None = 0."""
        _check_buffer(V, self._npts * 8, 8, bool(on_device), "V")
        self._ck(lib().sso_set_potential(self._h, _ptr(V), int(bool(on_device)), _stream(stream)))

    def set_field(self, kind: int, step_avg=None) -> None:
        """step_avg: contiguous float64 host array [nvals][ndim]."""
        if kind == FIELD_NONE or step_avg is None:
            self._ck(lib().sso_set_field(self._h, int(kind), None, 0))
            return
        nvals = step_avg.shape[0]
        _check_buffer(step_avg, nvals * len(self.sizes) * 8, 8, False, "step_avg")
        self._ck(lib().sso_set_field(self._h, int(kind), _ptr(step_avg), int(nvals)))

    def set_vector_potential(self, A, on_device: bool = False, stream=None) -> None:
        """A: float64 step-averaged A(r), shape (ndim, *sizes) (numpy on host, or a torch CUDA tensor); None = off."""
        _check_buffer(A, self._npts * len(self.sizes) * 8, 8, bool(on_device), "A")
        self._ck(lib().sso_set_vector_potential(self._h, _ptr(A), int(bool(on_device)), _stream(stream)))

    def set_time_index(self, n: int) -> None:
        self._ck(lib().sso_set_time_index(self._h, int(n)))

    def get_time_index(self) -> int:
        n = ctypes.c_int64()
        self._ck(lib().sso_get_time_index(self._h, ctypes.byref(n)))
        return n.value

    def set_option(self, option: int, value: int) -> None:
        self._ck(lib().sso_set_option(self._h, int(option), int(value)))

    def step(self, psi, nsteps: int, stream=None) -> None:
        """psi: device buffer (torch CUDA tensor, complex64/complex128, shape (ncomp, *sizes)); in place, asynchronous."""
        _check_buffer(psi, self._psi_bytes, self._esz, True, "psi")
        self._ck(lib().sso_step(self._h, _ptr(psi), int(nsteps), _stream(stream)))

    def step_host(self, psi_host, nsteps: int) -> None:
        """psi_host: host buffer (numpy array or pinned torch tensor); copied up, stepped, copied back."""
        _check_buffer(psi_host, self._psi_bytes, self._esz, False, "psi_host")
        self._ck(lib().sso_step_host(self._h, _ptr(psi_host), int(nsteps)))

    def norm(self, psi, stream=None) -> float:
        out = ctypes.c_double()
        _check_buffer(psi, self._psi_bytes, self._esz, True, "psi")
        self._ck(lib().sso_norm(self._h, _ptr(psi), ctypes.byref(out), _stream(stream)))
        return out.value

    # observables
    def overlap(self, psi_a, psi_b, stream=None) -> complex:
        """<a|b> = sum conj(a) b prod dx (chi(t) of eq. 40 for a = psi(0), b = psi(t))."""
        _check_buffer(psi_a, self._psi_bytes, self._esz, True, "psi_a")
        _check_buffer(psi_b, self._psi_bytes, self._esz, True, "psi_b")
        out = (ctypes.c_double * 2)()
        self._ck(lib().sso_overlap(self._h, _ptr(psi_a), _ptr(psi_b), out, _stream(stream)))
        return complex(out[0], out[1])

    def expect_position(self, psi, stream=None):
        _check_buffer(psi, self._psi_bytes, self._esz, True, "psi")
        out = (ctypes.c_double * 3)()
        self._ck(lib().sso_expect_position(self._h, _ptr(psi), out, _stream(stream)))
        return [out[a] for a in range(len(self.sizes))]

    def expect_momentum(self, psi, stream=None):
        _check_buffer(psi, self._psi_bytes, self._esz, True, "psi")
        out = (ctypes.c_double * 3)()
        self._ck(lib().sso_expect_momentum(self._h, _ptr(psi), out, _stream(stream)))
        return [out[a] for a in range(len(self.sizes))]

    def spectrum(self, chi, dts: float, E, out, stream=None) -> None:
        """chi: complex128 host array [nt]; E: float64 host array [nE]; out: complex128 host array [nE], filled."""
        nt, nE = chi.shape[0], E.shape[0]
        _check_buffer(chi, nt * 16, 16, False, "chi")
        _check_buffer(E, nE * 8, 8, False, "E")
        _check_buffer(out, nE * 16, 16, False, "out")
        self._ck(lib().sso_spectrum(self._h, _ptr(chi), int(nt), float(dts), _ptr(E), int(nE), _ptr(out), _stream(stream)))

    def filter_accumulate(self, acc, psi, t: float, T: float, E: float, dts: float, stream=None) -> None:
        """acc (complex128 CUDA tensor, shape of psi) += psi (1 - cos(2 pi t/T)) exp(i E t) dts (one term of eq. 42)."""
        _check_buffer(acc, self._npts * self.ncomp * 16, 16, True, "acc")
        _check_buffer(psi, self._psi_bytes, self._esz, True, "psi")
        self._ck(lib().sso_filter_accumulate(self._h, _ptr(acc), _ptr(psi), float(t), float(T), float(E), float(dts), _stream(stream)))

    def step_observe(self, psi, nsteps: int, psi_ref=None, filter_acc=None, filter_t: float = 0.0, filter_T: float = 1.0,
                     filter_E: float = 0.0, filter_dts: float = 0.0, stream=None):
        """sso_step_observe: step, and return (norm, <psi_ref|psi>, [<r_a>]) of the result from the closing pass."""
        _check_buffer(psi, self._psi_bytes, self._esz, True, "psi")
        _check_buffer(psi_ref, self._psi_bytes, self._esz, True, "psi_ref")
        _check_buffer(filter_acc, self._npts * self.ncomp * 16, 16, True, "filter_acc")
        out = (ctypes.c_double * 6)()
        self._ck(lib().sso_step_observe(self._h, _ptr(psi), int(nsteps), _ptr(psi_ref), _ptr(filter_acc), float(filter_t), float(filter_T),
                                        float(filter_E), float(filter_dts), out, _stream(stream)))
        return out[0], complex(out[1], out[2]), [out[3 + a] for a in range(len(self.sizes))]

    def profile_step(self, psi, nsteps: int, stream=None):
        """sso_profile_step: [(pass name, launches, mean microseconds)] for the pass kinds that ran."""
        _check_buffer(psi, self._psi_bytes, self._esz, True, "psi")
        cnt = (ctypes.c_int64 * PASS_KINDS)()
        us = (ctypes.c_double * PASS_KINDS)()
        self._ck(lib().sso_profile_step(self._h, _ptr(psi), int(nsteps), _stream(stream), cnt, us))
        return [(lib().sso_pass_name(k).decode(), int(cnt[k]), float(us[k])) for k in range(PASS_KINDS) if cnt[k]]

    def launch_count(self, nsteps: int) -> int:
        n = ctypes.c_int64()
        self._ck(lib().sso_launch_count(self._h, int(nsteps), ctypes.byref(n)))
        return n.value

    def destroy(self) -> None:
        if getattr(self, "_h", None) is not None and self._h:
            lib().sso_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
