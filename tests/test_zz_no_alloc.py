"""sso_norm_static -- the norm for callers that are not allowed to allocate device memory.

Who that is: an application (or the framework around it) whose own arena already holds all of HBM, so that a
cudaMalloc issued by this library fails; a time loop that cannot take the device-wide wait cudaMalloc / cudaFree
imply; a monitor that only holds a pointer to a wavefunction and has no plan (sso_plan_create allocates tables).
The entry point keeps its partial sums in an array built into libsso.so instead, which is why it has a size limit
and why every call on a device shares -- and finds the leftovers of -- the same scratch.

The GPU test checks it against the existing path (a plan's sso_norm) on two calls in a row, the second on a
shorter and different state, so that anything the first call left in the shared array would show.  It depends on
no other test: it runs alone in a fresh process as well as at the end of the whole suite (the file name sorts
last on purpose, so that with `pytest -x` a failure here hides no other test).
"""
import ctypes

import numpy as np
import pytest

import paper_1012_3911_b200 as sso
from paper_1012_3911_b200 import build as sso_build

REL_TOL = 1e-14  # the tolerance test_norm_matches_oracle puts on sso_norm


@pytest.fixture(scope="module")
def L():
    sso_build.build()
    return sso.lib()


def test_rejects_what_the_builtin_scratch_cannot_hold(L):
    """Argument errors are found before any CUDA call (so this runs without a GPU) and say what the limit is."""
    out = ctypes.c_double()
    fake = ctypes.addressof(out)  # 8-byte aligned stand-in; never dereferenced on these paths
    rc = L.sso_norm_static(fake & ~15, sso.C128, sso.NORM_STATIC_MAX_COUNT + 1, 1.0, fake, None)
    assert rc == sso.ERR_INVALID
    msg = L.sso_last_error(None).decode()
    assert "SSO_NORM_STATIC_MAX_COUNT" in msg and str(sso.NORM_STATIC_MAX_COUNT) in msg
    assert L.sso_norm_static(fake & ~15, 7, 16, 1.0, fake, None) == sso.ERR_INVALID         # precision
    assert L.sso_norm_static(fake & ~15, sso.C128, -1, 1.0, fake, None) == sso.ERR_INVALID  # count
    assert L.sso_norm_static(None, sso.C128, 16, 1.0, fake, None) == sso.ERR_INVALID         # psi NULL
    assert L.sso_norm_static(fake & ~15, sso.C128, 16, 1.0, None, None) == sso.ERR_INVALID  # out NULL
    assert L.sso_norm_static((fake & ~15) + 8, sso.C128, 16, 1.0, fake, None) == sso.ERR_INVALID  # psi misaligned
    assert L.sso_norm_static(fake & ~15, sso.C128, 16, float("nan"), fake, None) == sso.ERR_INVALID
    with pytest.raises(sso.SsoError, match="SSO_NORM_STATIC_MAX_COUNT"):
        sso.norm_static(fake & ~15, 1.0, fake, precision=sso.C64, count=sso.NORM_STATIC_MAX_COUNT + 8192)


def test_header_states_the_limit():
    """The binding's copy of the limits is the header's."""
    import re
    from pathlib import Path

    h = (Path(__file__).resolve().parent.parent / "include" / "sso.h").read_text()
    chunk = int(re.search(r"#define SSO_NORM_STATIC_CHUNK (\d+)", h).group(1))
    shift = int(re.search(r"#define SSO_NORM_STATIC_MAX_COUNT \(1LL << (\d+)\)", h).group(1))
    assert (chunk, 1 << shift) == (sso.NORM_STATIC_CHUNK, sso.NORM_STATIC_MAX_COUNT)


@pytest.mark.gpu
@pytest.mark.parametrize("prec", [sso.C128, sso.C64], ids=["c128", "c64"])
def test_two_calls_in_a_row_match_the_plan_norm(L, prec):
    import torch

    torch.cuda.set_device(0)
    dt = torch.complex128 if prec == sso.C128 else torch.complex64
    g = torch.Generator(device="cpu").manual_seed(1012_3911 + prec)
    # first call: 512 x 1024 points = 64 chunks; second call: a 2-component spinor on 64 x 128 points = 2 chunks,
    # other values, after the first call has left 64 partial sums behind in the shared array
    cases = [((1, 512, 1024), (0.05, 0.07)), ((2, 64, 128), (0.3, 0.11))]
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")  # caller-owned result slots
    want = []
    for i, (shape, dx) in enumerate(cases):
        re_, im_ = torch.randn(shape, generator=g, dtype=torch.float64), torch.randn(shape, generator=g, dtype=torch.float64)
        psi = torch.complex(re_, im_).mul_(1.0 + i).to(dt).cuda()
        plan = sso.Plan(shape[1:], dx, 0.01, ncomp=shape[0], precision=prec)
        want.append(plan.norm(psi))  # the existing path: plan-owned partial sums, result copied to the host
        plan.destroy()
        sso.norm_static(psi, dx[0] * dx[1], out[i:])
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    for i in range(2):
        assert np.isfinite(got[i]) and want[i] > 0
        assert abs(got[i] - want[i]) <= REL_TOL * want[i], (i, got[i], want[i])


@pytest.mark.gpu
def test_ragged_tail_empty_input_and_side_stream(L):
    """count that is no multiple of the chunk or of the CTA size, count = 0, and a caller-owned stream."""
    import torch

    torch.cuda.set_device(0)
    g = torch.Generator(device="cpu").manual_seed(7)
    n = 3 * sso.NORM_STATIC_CHUNK + 1237
    psi = torch.complex(torch.randn(n, generator=g, dtype=torch.float64), torch.randn(n, generator=g, dtype=torch.float64)).cuda()
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        sso.norm_static(psi, 0.25, out, stream=st)
        sso.norm_static(psi, 0.25, out[1:], count=0, stream=st)
    st.synchronize()
    want = 0.25 * float((psi.real.double() ** 2 + psi.imag.double() ** 2).sum().item())
    got = out.cpu().numpy()
    assert abs(got[0] - want) <= 1e-13 * want
    assert got[1] == 0.0
