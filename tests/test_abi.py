"""The C-ABI boundary without a GPU: the library builds, loads and exports every symbol include/sso.h declares;
argument validation that happens before any CUDA call; the host-side radix schedule / digit reversal."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

import paper_1012_3911_b200 as sso
from paper_1012_3911_b200 import build as sso_build

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def L():
    sso_build.build()
    return sso.lib()


def test_header_symbols_are_exported(L):
    header = (ROOT / "include" / "sso.h").read_text()
    declared = set(re.findall(r"\b(sso_[a-z_]+)\s*\(", header))
    assert declared, "no declarations found in include/sso.h"
    assert declared == set(sso.SYMBOLS), declared ^ set(sso.SYMBOLS)
    for name in declared:
        assert hasattr(L, name), f"libsso.so does not export {name}"


def test_version(L):
    assert "sm_100a" in sso.version()


def _create(L, ndim, sizes, dx, dt, ncomp, prec):
    h = ctypes.c_void_p()
    szs = (ctypes.c_int64 * 3)(*(list(sizes) + [0] * (3 - len(sizes))))
    dxs = (ctypes.c_double * 3)(*(list(dx) + [0.0] * (3 - len(dx))))
    rc = L.sso_plan_create(ctypes.byref(h), ndim, szs, dxs, dt, ncomp, prec)
    return rc, h


@pytest.mark.parametrize(
    "args,code",
    [
        ((0, (64,), (0.1,), 0.01, 1, sso.C128), sso.ERR_INVALID),          # ndim out of range
        ((4, (64,), (0.1,), 0.01, 1, sso.C128), sso.ERR_INVALID),
        ((1, (48,), (0.1,), 0.01, 1, sso.C128), sso.ERR_INVALID),          # not a power of two
        ((1, (8,), (0.1,), 0.01, 1, sso.C128), sso.ERR_UNSUPPORTED),       # below SSO_MIN_AXIS
        ((1, (65536,), (0.1,), 0.01, 1, sso.C128), sso.ERR_UNSUPPORTED),   # above SSO_MAX_AXIS_1D
        ((1, (8192,), (0.1,), 0.01, 2, sso.C128), sso.ERR_UNSUPPORTED),    # above SSO_MAX_AXIS for a 1D Dirac spinor
        ((2, (16384, 64), (0.1, 0.1), 0.01, 1, sso.C128), sso.ERR_UNSUPPORTED),  # above SSO_MAX_AXIS for a 2D lattice
        ((2, (64, 64), (0.1, -0.1), 0.01, 1, sso.C128), sso.ERR_INVALID),  # dx <= 0
        ((2, (64, 64), (0.1, float("nan")), 0.01, 1, sso.C128), sso.ERR_INVALID),
        ((1, (64,), (0.1,), float("inf"), 1, sso.C128), sso.ERR_INVALID),  # dt not finite
        ((1, (64,), (0.1,), 0.01, 3, sso.C128), sso.ERR_INVALID),          # ncomp
        ((3, (16, 16, 16), (0.1,) * 3, 0.01, 2, sso.C128), sso.ERR_INVALID),  # 2 components in 3D
        ((1, (64,), (0.1,), 0.01, 1, 7), sso.ERR_INVALID),                 # precision
        ((1, (4096,), (0.1,), 0.01, 4, sso.C128), sso.ERR_UNSUPPORTED),    # 1D Dirac line too long for one CTA
    ],
)
def test_plan_create_rejects_bad_arguments(L, args, code):
    rc, h = _create(L, *args)
    assert rc == code
    assert not h.value
    assert L.sso_last_error(None)  # a message is recorded


def test_null_arguments(L):
    assert L.sso_plan_create(None, 1, None, None, 0.1, 1, 1) == sso.ERR_INVALID
    h = ctypes.c_void_p()
    assert L.sso_plan_create(ctypes.byref(h), 1, None, None, 0.1, 1, 1) == sso.ERR_INVALID
    assert L.sso_destroy(None) == sso.OK
    assert L.sso_step(None, None, 1, None) == sso.ERR_INVALID
    assert L.sso_norm(None, None, None, None) == sso.ERR_INVALID
    assert L.sso_set_potential(None, None, 0, None) == sso.ERR_INVALID
    assert L.sso_set_field(None, 0, None, 0) == sso.ERR_INVALID
    assert L.sso_set_time_index(None, 0) == sso.ERR_INVALID


def test_no_cpu_fallback_without_a_device(L):
    """On a box without a GPU a valid request must fail loudly with SSO_ERR_CUDA, never run on the CPU."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    rc, h = _create(L, 1, (64,), (0.1,), 0.01, 1, sso.C128)
    assert rc == sso.ERR_CUDA
    assert b"no CPU fallback" in L.sso_last_error(None)
    with pytest.raises(sso.SsoError):
        sso.Plan((64,), (0.1,), 0.01)


# ---------------------------------------------------------------------------------------------------------
# host logic: the digit-reversed order the plan builder assumes is the order the DIF network really produces
# ---------------------------------------------------------------------------------------------------------

def _schedule(n):
    log = n.bit_length() - 1
    rem = log - 4
    m = 1 + (rem + 3) // 4
    return [4 if i == m - 1 else (rem - 4 * (m - 2) if i == 0 else 4) for i in range(m)]


def _dif_network(x):
    """In-place mixed-radix decimation in frequency exactly as the kernel's stages do it (numpy, complex128)."""
    n = x.size
    y = x.astype(np.complex128).copy()
    NP = n
    for lr in _schedule(n):
        R = 1 << lr
        NI = NP // R
        y = y.reshape(n // NP, R, NI)                      # [block][j][l]
        W = np.exp(-2j * np.pi * np.outer(np.arange(R), np.arange(R)) / R)
        y = np.einsum("kj,bjl->bkl", W, y)                 # butterflies over the top digit
        tw = np.exp(-2j * np.pi * np.outer(np.arange(R), np.arange(NI)) / NP)
        y = (y * tw[None]).reshape(n)                      # twiddles w_NP^(l k)
        NP = NI
    return y


@pytest.mark.parametrize("n", [16, 32, 64, 128, 256, 512, 1024, 2048, 4096])
def test_layout_tables_match_the_dif_network(L, n):
    L.sso_debug_layout.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int)]
    L.sso_debug_layout.restype = ctypes.c_int
    pos_freq = (ctypes.c_int * n)()
    slot_nat = (ctypes.c_int * n)()
    assert L.sso_debug_layout(n, pos_freq, slot_nat) == sso.OK
    pf = np.array(pos_freq[:])
    sn = np.array(slot_nat[:])
    assert sorted(pf) == list(range(n)) and sorted(sn) == list(range(n))
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    X = np.fft.fft(x)
    y = _dif_network(x)
    np.testing.assert_allclose(y, X[pf], rtol=0, atol=1e-10)
    # permuted-layout slot q*U + B' holds network position 16 B' + q
    U = n // 16
    q, B = np.divmod(np.arange(n), U)
    np.testing.assert_array_equal(sn, pf[16 * B + q])
    assert L.sso_debug_layout(24, pos_freq, slot_nat) == sso.ERR_INVALID
