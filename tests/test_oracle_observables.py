"""Pins for the oracle's observables (section V.2: autocorrelation chi(t) eq. 40, windowed spectrum
eq. 41, eigenfunction filter eq. 42; <r>, <p>).  Expected values are closed forms, exact discrete identities and the
paper's own soft-core ground-state statement; nothing here needs a GPU.
"""
from pathlib import Path

import numpy as np
import pytest

import oracle

GOLDEN = Path(__file__).resolve().parent / "golden"


def paper_constants():
    return {ln.split()[0]: float(ln.split()[1]) for ln in (GOLDEN / "paper_constants.txt").read_text().splitlines() if ln and not ln.startswith("#")}


def axis(n, dx):
    return (np.arange(n) - n // 2) * dx


def gaussian(x, x0, p0, sigma):
    return (np.pi * sigma**2) ** -0.25 * np.exp(-((x - x0) ** 2) / (2 * sigma**2) + 1j * p0 * x)


def test_overlap_of_two_gaussians_closed_form():
    """<g1|g2> = exp(-(x1-x2)^2/4s^2 - s^2 (p2-p1)^2/4 + i (p2-p1)(x1+x2)/2): the conjugate sits on the FIRST argument."""
    n, dx, s = 512, 0.1, 1.3
    x = axis(n, dx)
    x1, p1, x2, p2 = -0.4, 0.4, 1.1, -0.5
    o = oracle.Solver((n,), (dx,), 0.01)
    want = np.exp(-((x1 - x2) ** 2) / (4 * s**2) - s**2 * (p2 - p1) ** 2 / 4 + 1j * (p2 - p1) * (x1 + x2) / 2)
    got = o.overlap(gaussian(x, x1, p1, s), gaussian(x, x2, p2, s))
    assert abs(got - want) < 1e-13
    assert abs(want.imag) > 0.05  # the case does distinguish <a|b> from <b|a>
    assert abs(o.overlap(gaussian(x, x2, p2, s), gaussian(x, x1, p1, s)) - np.conj(want)) < 1e-13


def test_overlap_sums_all_components_and_uses_the_cell_volume():
    sizes, dx = (8, 4, 16), (0.3, 0.5, 0.2)
    rng = np.random.default_rng(40)
    o = oracle.Solver(sizes, dx, 0.01, ncomp=4)
    a = rng.normal(size=(4,) + sizes) + 1j * rng.normal(size=(4,) + sizes)
    # <a | i^c a_c> = sum_c i^c ||a_c||^2: every component enters with its own weight
    b = np.stack([(1j**c) * a[c] for c in range(4)])
    per = [float(np.sum(np.abs(a[c]) ** 2)) * 0.3 * 0.5 * 0.2 for c in range(4)]
    want = sum((1j**c) * per[c] for c in range(4))
    assert abs(o.overlap(a, b) - want) < 1e-12 * abs(want)


def test_autocorrelation_of_a_free_plane_wave_and_of_a_dirac_plane_wave():
    """chi(t) = <psi(0)|psi(t)> (eq. 40).  A plane wave at a grid momentum is an eigenstate of the V = 0 step:
    Schroedinger chi(n tau) = exp(-i k^2 n tau / 2); Dirac u^+(k) e_1: chi = exp(-i E n tau), E = +sqrt(c^2 k^2 + c^4)."""
    n, dx, tau = 64, 0.25, 0.02
    x = axis(n, dx)
    L = n * dx
    k = 2 * np.pi * (-5) / L
    o = oracle.Solver((n,), (dx,), tau)
    psi0 = np.exp(1j * k * x) / np.sqrt(L)
    psi = o.step(psi0, 37)
    assert abs(o.overlap(psi0, psi) - np.exp(-1j * k * k * 37 * tau / 2)) < 1e-13
    c = 137.036
    tau = 1e-4
    od = oracle.Solver((n,), (dx,), tau, ncomp=2, c=c)
    u = oracle.dirac_u(2, [k], 1.0, c)
    spinor = u.conj().T[:, 0]  # column 1 of u^+: positive energy (reading G8)
    psi0 = spinor[:, None] * np.exp(1j * k * x)[None, :] / np.sqrt(L)
    psi = od.step(psi0, 11)
    E = np.sqrt(c * c * k * k + c**4)
    assert abs(od.overlap(psi0, psi) - np.exp(-1j * E * 11 * tau)) < 1e-12


@pytest.mark.parametrize("sizes,dx", [((256,), (0.1,)), ((64, 128), (0.2, 0.1)), ((32, 64, 16), (0.3, 0.15, 0.6))])
def test_position_and_momentum_of_a_gaussian_packet(sizes, dx):
    """<r_a> = x0_a and <p_a> = p0_a for a Gaussian packet, distinct per axis (an axis mix-up or a sign fails)."""
    nd = len(sizes)
    x0 = [0.7, -1.1, 0.9][:nd]
    p0 = [-0.8, 1.3, 0.5][:nd]
    psi = np.ones(sizes, dtype=np.complex128)
    for a in range(nd):
        g = gaussian(axis(sizes[a], dx[a]), x0[a], p0[a], 0.9)
        psi = psi * g.reshape([-1 if b == a else 1 for b in range(nd)])
    o = oracle.Solver(sizes, dx, 0.01)
    np.testing.assert_allclose(o.expect_r(psi), x0, atol=1e-12)
    np.testing.assert_allclose(o.expect_p(psi), p0, atol=1e-12)


def test_momentum_of_grid_plane_waves_including_negative_and_nyquist():
    n, dx = 32, 0.4
    x = axis(n, dx)
    o = oracle.Solver((n,), (dx,), 0.01)
    for j in (3, -7, -16):
        k = 2 * np.pi * j / (n * dx)
        psi = np.exp(1j * k * x) / np.sqrt(n * dx)
        assert abs(o.expect_p(psi)[0] - k) < 1e-12  # Nyquist counts as -pi/dx (reading G14)


def test_spinor_expectations_weight_every_component():
    n, dx = 256, 0.1
    x = axis(n, dx)
    o = oracle.Solver((n,), (dx,), 1e-4, ncomp=2)
    psi = np.stack([np.sqrt(0.3) * gaussian(x, 2.0, 1.0, 1.0), np.sqrt(0.7) * gaussian(x, -1.0, -2.0, 1.0)])
    assert abs(o.expect_r(psi)[0] - (0.3 * 2.0 + 0.7 * -1.0)) < 1e-12
    assert abs(o.expect_p(psi)[0] - (0.3 * 1.0 + 0.7 * -2.0)) < 1e-12


def test_momentum_kick_by_a_constant_field():
    """Constant Ebar on a free particle: every step changes <p> by -Ebar tau exactly (Stoermer-Verlet kick) and
    <r> by the mean of the old and new momentum times tau."""
    n, dx, tau, Eb = 512, 0.1, 0.05, 0.3
    x = axis(n, dx)
    o = oracle.Solver((n,), (dx,), tau)
    o.set_field(oracle.FIELD_E, np.full((20, 1), Eb))
    psi = gaussian(x, -3.0, 0.5, 1.5)
    p, r = o.expect_p(psi)[0], o.expect_r(psi)[0]
    for _ in range(20):
        psi = o.step(psi, 1)
        pn, rn = o.expect_p(psi)[0], o.expect_r(psi)[0]
        assert abs(pn - (p - Eb * tau)) < 1e-12
        assert abs(rn - (r + 0.5 * (p + pn) * tau)) < 1e-11
        p, r = pn, rn


def test_spectrum_of_a_single_exponential_is_the_hann_window_transform():
    """chi(t) = exp(-i E0 t): eq. 41 gives T at E = E0, -T/2 at E0 +- 2 pi/T, 0 at E0 + 2 pi m/T (|m| >= 2) exactly for
    the sum over samples; between those points it follows the closed form of the integral."""
    nt, dts, E0 = 400, 0.05, -0.73
    T = nt * dts
    t = np.arange(nt) * dts
    chi = np.exp(-1j * E0 * t)
    m = np.array([0, 1, -1, 2, -3, 7])
    got = oracle.spectrum(chi, dts, E0 + 2 * np.pi * m / T)
    np.testing.assert_allclose(got, T * np.array([1, -0.5, -0.5, 0, 0, 0]), atol=1e-12)
    # the peak sits at +E0 for exp(-i E0 t) (sign of the exponent in eq. 41)
    assert abs(oracle.spectrum(chi, dts, np.array([-E0]))[0]) < 0.05 * T
    # closed form of the integral off the grid: f(d) - f(d+W)/2 - f(d-W)/2, f(a) = (exp(i a T) - 1)/(i a), W = 2 pi/T
    f = lambda a: (np.exp(1j * a * T) - 1) / (1j * a)
    W = 2 * np.pi / T
    d = np.array([0.13, -0.41, 0.9])
    want = f(d) - 0.5 * f(d + W) - 0.5 * f(d - W)
    np.testing.assert_allclose(oracle.spectrum(chi, dts, E0 + d), want, atol=2e-5 * T)


def test_filter_accumulation_projects_on_one_term():
    """psi(x,t) = a phi1 exp(-i E1 t) + b phi2 exp(-i E2 t) with E2 - E1 = 2 pi m/T, m >= 2: the sum of eq. 42's terms
    at E = E1 over the samples is a T phi1 exactly (discrete orthogonality of the Hann-windowed exponentials)."""
    n, dx = 64, 0.3
    x = axis(n, dx)
    nt, dts = 128, 0.1
    T = nt * dts
    E1 = -0.5
    E2 = E1 + 2 * np.pi * 5 / T
    phi1 = gaussian(x, 0.0, 0.0, 1.0)
    phi2 = x * gaussian(x, 0.0, 0.0, 1.0)
    o = oracle.Solver((n,), (dx,), dts, ncomp=2)
    a, b = 0.8 - 0.2j, 0.3 + 0.5j
    acc = np.zeros((2, n), dtype=np.complex128)
    for k in range(nt):
        t = k * dts
        psi = a * phi1 * np.exp(-1j * E1 * t) + b * phi2 * np.exp(-1j * E2 * t)
        o.filter_accumulate(acc, np.stack([psi, 2 * psi]), t, T, E1, dts)
    np.testing.assert_allclose(acc[0], a * T * phi1, atol=1e-12)
    np.testing.assert_allclose(acc[1], 2 * a * T * phi1, atol=1e-12)


def soft_core(r2, zeta, Z=1.0):
    return -Z / np.sqrt(r2 + (zeta / Z) ** 2)


def ground_state_energy(sizes, dx, zeta, tau, nt):
    """The paper's procedure: propagate a trial function, record chi(t), locate the lowest peak of
    |chi~(E)|; then the eigenfunction by eq. 42.  Returns (E0, Psi_E0, solver, V)."""
    nd = len(sizes)
    grids = np.meshgrid(*[axis(n, d) for n, d in zip(sizes, dx)], indexing="ij")
    r2 = sum(g * g for g in grids)
    V = soft_core(r2, zeta)
    o = oracle.Solver(sizes, dx, tau)
    o.set_potential(V)
    psi0 = np.exp(-r2 / 2).astype(np.complex128)
    psi0 /= np.sqrt(o.norm(psi0))
    chi = np.empty(nt, dtype=np.complex128)
    psi = psi0
    states = []
    for k in range(nt):
        chi[k] = o.overlap(psi0, psi)
        states.append(psi)
        psi = o.step(psi, 1)
    E = np.linspace(-0.7, -0.3, 4001)
    sp = np.abs(oracle.spectrum(chi, tau, E))
    E0 = E[int(np.argmax(sp))]
    acc = np.zeros(sizes, dtype=np.complex128)
    T = nt * tau
    for k, s in enumerate(states):
        o.filter_accumulate(acc, s, k * tau, T, E0, tau)
    return E0, acc, o, V


def check_eigenfunction(acc, V, sizes, dx, E0, tol):
    """||H Psi - E0 Psi|| / ||Psi|| with H = -laplace/2 + V applied spectrally by numpy (independent of the oracle)."""
    ks = np.meshgrid(*[2 * np.pi * np.fft.fftfreq(n, d) for n, d in zip(sizes, dx)], indexing="ij")
    k2 = sum(k * k for k in ks)
    H = np.fft.ifftn(0.5 * k2 * np.fft.fftn(acc)) + V * acc
    res = np.linalg.norm(H - E0 * acc) / np.linalg.norm(acc)
    assert res < tol, res


def test_soft_core_ground_state_1d_paper_value():
    """the 1D soft-core potential with zeta = 1.4133 has approximately the Coulomb ground-state energy
    -Z^2/2.  The whole chain chi(t) -> chi~(E) -> peak -> eq. 42 eigenfunction is exercised."""
    pc = paper_constants()
    sizes, dx, tau, nt = (512,), (0.2,), 0.05, 4096
    E0, acc, o, V = ground_state_energy(sizes, dx, pc["softcore_zeta_1d"], tau, nt)
    assert abs(E0 - pc["softcore_groundstate_energy_over_Z2"]) < 2e-3, E0
    check_eigenfunction(acc, V, sizes, dx, E0, 5e-3)


def test_soft_core_ground_state_2d_paper_value():
    """in two dimensions zeta = 0.791 matches the ground-state energies."""
    pc = paper_constants()
    sizes, dx, tau, nt = (128, 128), (0.3, 0.3), 0.05, 2048
    E0, acc, o, V = ground_state_energy(sizes, dx, pc["softcore_zeta_2d"], tau, nt)
    assert abs(E0 - pc["softcore_groundstate_energy_over_Z2"]) < 5e-3, E0
    check_eigenfunction(acc, V, sizes, dx, E0, 2e-2)
