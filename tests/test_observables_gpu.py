"""GPU parity of the observables (autocorrelation eq. 40, spectrum eq. 41, eigenfunction filter
eq. 42, <r>, <p>) through the C ABI against the CPU oracle on the same seeded inputs; plus the paper's soft-core
ground-state energy obtained with the GPU chain alone."""
from pathlib import Path

import numpy as np
import pytest

import oracle
import paper_1012_3911_b200 as sso

pytestmark = pytest.mark.gpu
GOLDEN = Path(__file__).resolve().parent / "golden"


@pytest.fixture(scope="module")
def torch():
    import torch as t

    assert t.cuda.is_available()
    t.cuda.set_device(0)
    sso.lib()
    return t


def packet(rng, ncomp, sizes, dx):
    """Seeded smooth packets with momentum plus noise, a different one per component, normalised."""
    grids = np.meshgrid(*[(np.arange(n) - n // 2) * d for n, d in zip(sizes, dx)], indexing="ij")
    psi = np.empty((ncomp,) + tuple(sizes), dtype=np.complex128)
    for c in range(ncomp):
        x0 = rng.uniform(-1.0, 1.0, size=len(sizes))
        p0 = rng.uniform(-1.5, 1.5, size=len(sizes))
        arg = sum(-((g - a) ** 2) / 3.0 + 1j * p * g for g, a, p in zip(grids, x0, p0))
        psi[c] = rng.uniform(0.5, 1.5) * np.exp(arg) + 1e-3 * (rng.normal(size=sizes) + 1j * rng.normal(size=sizes))
    psi /= np.sqrt(np.sum(np.abs(psi) ** 2) * np.prod(dx))
    return psi


CASES = [
    ("1d-c128", 1, (512,), (0.1,), sso.C128),
    ("2d-c128", 1, (64, 128), (0.2, 0.1), sso.C128),
    ("3d-dirac4-c128", 4, (16, 32, 64), (0.3, 0.2, 0.1), sso.C128),
    ("2d-dirac2-c64", 2, (32, 256), (0.25, 0.1), sso.C64),
    ("3d-c64", 1, (32, 16, 64), (0.3, 0.3, 0.2), sso.C64),
]


@pytest.mark.parametrize("name,ncomp,sizes,dx,prec", CASES, ids=[c[0] for c in CASES])
def test_overlap_position_momentum_match_the_oracle(torch, name, ncomp, sizes, dx, prec):
    rng = np.random.default_rng(4000 + [c[0] for c in CASES].index(name))
    cdt = np.complex128 if prec == sso.C128 else np.complex64
    a = packet(rng, ncomp, sizes, dx).astype(cdt)
    b = packet(rng, ncomp, sizes, dx).astype(cdt)
    o = oracle.Solver(sizes, dx, 0.01, ncomp)
    p = sso.Plan(sizes, dx, 0.01, ncomp, prec)
    ta, tb = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
    a64, b64 = a.astype(np.complex128), b.astype(np.complex128)
    exact = 1e-12  # sums of products formed in double on both sides
    fft_tol = 1e-11 if prec == sso.C128 else 2e-5
    assert abs(p.overlap(ta, tb) - o.overlap(a64, b64)) < exact
    assert abs(p.overlap(tb, ta) - o.overlap(b64, a64)) < exact
    np.testing.assert_allclose(p.expect_position(tb), o.expect_r(b64), atol=exact * 10)
    np.testing.assert_allclose(p.expect_momentum(tb), o.expect_p(b64), atol=fft_tol * 10)
    assert np.array_equal(tb.cpu().numpy(), b)  # psi is not modified
    assert abs(p.norm(ta) - o.norm(a64)) < exact
    p.destroy()


def test_spectrum_matches_the_oracle(torch):
    rng = np.random.default_rng(41)
    nt, dts = 777, 0.05
    t = np.arange(nt) * dts
    chi = sum(w * np.exp(-1j * e * t) for w, e in ((0.6, -0.5), (0.3, -0.12), (0.1 + 0.05j, 0.4))) + 1e-3 * rng.normal(size=nt)
    chi = np.ascontiguousarray(chi, dtype=np.complex128)
    E = np.ascontiguousarray(np.linspace(-1.0, 1.0, 301))
    p = sso.Plan((16,), (0.1,), 0.01)
    out = np.zeros(E.size, dtype=np.complex128)
    p.spectrum(chi, dts, E, out)
    want = oracle.spectrum(chi, dts, E)
    assert np.abs(out - want).max() < 1e-11 * np.abs(want).max()
    p.destroy()


@pytest.mark.parametrize("prec", [sso.C128, sso.C64], ids=["c128", "c64"])
def test_filter_accumulation_matches_the_oracle(torch, prec):
    sizes, dx, ncomp = (32, 64), (0.2, 0.1), 2
    rng = np.random.default_rng(42)
    cdt = np.complex128 if prec == sso.C128 else np.complex64
    o = oracle.Solver(sizes, dx, 0.01, ncomp)
    p = sso.Plan(sizes, dx, 0.01, ncomp, prec)
    acc = torch.zeros((ncomp,) + sizes, dtype=torch.complex128, device="cuda")
    want = np.zeros((ncomp,) + sizes, dtype=np.complex128)
    T, E, dts = 3.0, -0.37, 0.25
    for k in range(12):
        psi = packet(rng, ncomp, sizes, dx).astype(cdt)
        p.filter_accumulate(acc, torch.from_numpy(psi).cuda(), k * dts, T, E, dts)
        o.filter_accumulate(want, psi.astype(np.complex128), k * dts, T, E, dts)
    torch.cuda.synchronize()
    assert np.abs(acc.cpu().numpy() - want).max() < 1e-13 * np.abs(want).max() * 12
    p.destroy()


def test_soft_core_ground_state_energy_on_the_gpu(torch):
    """PAPER.md:357-367 end to end on the device: propagate, record chi(t) (sso_overlap), transform (sso_spectrum),
    locate the peak; the paper's statement is E0 ~ -Z^2/2 for zeta = 1.4133.  The same chain on the
    oracle gives the same chi(t) and the same peak."""
    pc = {ln.split()[0]: float(ln.split()[1]) for ln in (GOLDEN / "paper_constants.txt").read_text().splitlines() if ln and not ln.startswith("#")}
    n, dx, tau, nt = 512, 0.2, 0.05, 4096
    x = (np.arange(n) - n // 2) * dx
    V = -1.0 / np.sqrt(x * x + pc["softcore_zeta_1d"] ** 2)
    psi0 = np.exp(-x * x / 2).astype(np.complex128)
    psi0 /= np.sqrt(np.sum(np.abs(psi0) ** 2) * dx)
    p = sso.Plan((n,), (dx,), tau)
    p.set_potential(V)
    o = oracle.Solver((n,), (dx,), tau)
    o.set_potential(V)
    ref = torch.from_numpy(psi0).cuda()
    psi = ref.clone()
    chi = np.empty(nt, dtype=np.complex128)
    chi_o = np.empty(nt, dtype=np.complex128)
    po = psi0
    for k in range(nt):
        chi[k] = p.overlap(ref, psi)
        p.step(psi, 1)
        if k < 256:
            chi_o[k] = o.overlap(psi0, po)
            po = o.step(po, 1)
    assert np.abs(chi[:256] - chi_o[:256]).max() < 1e-11
    E = np.ascontiguousarray(np.linspace(-0.7, -0.3, 4001))
    sp = np.zeros(E.size, dtype=np.complex128)
    p.spectrum(chi, tau, E, sp)
    E0 = E[int(np.argmax(np.abs(sp)))]
    assert abs(E0 - pc["softcore_groundstate_energy_over_Z2"]) < 2e-3, E0
    assert E0 == E[int(np.argmax(np.abs(oracle.spectrum(chi, tau, E))))]
    p.destroy()


def test_observable_argument_errors(torch):
    p = sso.Plan((64,), (0.1,), 0.01)
    L = sso.lib()
    import ctypes

    out = (ctypes.c_double * 3)()
    assert L.sso_overlap(p._h, None, None, out, None) == sso.ERR_INVALID
    assert L.sso_expect_position(p._h, None, out, None) == sso.ERR_INVALID
    assert L.sso_expect_momentum(p._h, None, out, None) == sso.ERR_INVALID
    assert L.sso_spectrum(p._h, None, 4, 0.1, None, 4, None, None) == sso.ERR_INVALID
    assert L.sso_filter_accumulate(p._h, None, None, 0.0, 1.0, 0.0, 0.1, None) == sso.ERR_INVALID
    assert L.sso_overlap(None, None, None, out, None) == sso.ERR_INVALID
    p.destroy()


FUSED = [
    ("2d-c128-field", 1, (64, 128), (0.2, 0.1), sso.C128, True),
    ("3d-dirac4-c128", 4, (16, 32, 64), (0.3, 0.2, 0.1), sso.C128, False),
    ("2d-dirac2-c64", 2, (32, 256), (0.25, 0.1), sso.C64, False),
    ("3d-c128", 1, (32, 16, 64), (0.3, 0.3, 0.2), sso.C128, False),
    ("1d-c128", 1, (1024,), (0.1,), sso.C128, False),
]


@pytest.mark.parametrize("name,ncomp,sizes,dx,prec,field", FUSED, ids=[c[0] for c in FUSED])
def test_observables_fused_into_the_closing_pass(torch, name, ncomp, sizes, dx, prec, field):
    """sso_step_observe: norm, <ref|psi>, <r> and one filter term come out of the closing pass of the call; they equal
    the oracle's observables of the oracle's psi after the same steps, and psi itself equals plain sso_step."""
    rng = np.random.default_rng(5000 + [c[0] for c in FUSED].index(name))
    cdt = np.complex128 if prec == sso.C128 else np.complex64
    tau = 0.01 if ncomp == 1 else 1e-4
    psi0 = packet(rng, ncomp, sizes, dx).astype(cdt)
    ref = packet(rng, ncomp, sizes, dx).astype(cdt)
    V = rng.uniform(-1.0, 1.0, size=sizes)
    nsteps = 7
    p = sso.Plan(sizes, dx, tau, ncomp, prec)
    o = oracle.Solver(sizes, dx, tau, ncomp)
    p.set_potential(V)
    o.set_potential(V)
    if field:
        avg = rng.uniform(-0.3, 0.3, size=(nsteps, len(sizes)))
        p.set_field(sso.FIELD_E, np.ascontiguousarray(avg))
        o.set_field(oracle.FIELD_E, avg)
    want = o.step(psi0.astype(np.complex128), nsteps)
    acc0 = (rng.normal(size=(ncomp,) + tuple(sizes)) + 1j * rng.normal(size=(ncomp,) + tuple(sizes)))
    want_acc = acc0.copy()
    ft, fT, fE, fdts = 0.35, 1.3, -0.42, 0.05
    o.filter_accumulate(want_acc, want, ft, fT, fE, fdts)
    psi = torch.from_numpy(psi0).cuda()
    tref = torch.from_numpy(ref).cuda()
    acc = torch.from_numpy(acc0).cuda()
    nrm, chi, r = p.step_observe(psi, nsteps, tref, acc, ft, fT, fE, fdts)
    torch.cuda.synchronize()
    tol = 1e-11 if prec == sso.C128 else 2e-5
    got = psi.cpu().numpy()
    assert np.linalg.norm((got - want).ravel()) / np.linalg.norm(want.ravel()) < tol
    assert abs(nrm - o.norm(want)) < tol * 10
    assert abs(chi - o.overlap(ref.astype(np.complex128), want)) < tol * 10
    np.testing.assert_allclose(r, o.expect_r(want), atol=tol * 100)
    assert np.abs(acc.cpu().numpy() - want_acc).max() < tol * 10 * np.abs(want_acc).max()
    # the same psi as plain stepping, and the same numbers as the separate kernels on it
    psi2 = torch.from_numpy(psi0).cuda()
    p.set_time_index(0)
    p.step(psi2, nsteps)
    assert np.array_equal(psi2.cpu().numpy(), got)
    assert abs(p.norm(psi2) - nrm) < 1e-13
    assert abs(p.overlap(tref, psi2) - chi) < 1e-13
    np.testing.assert_allclose(p.expect_position(psi2), r, atol=1e-12)
    p.destroy()
