"""Pins for the CPU oracle: what the paper and the mathematics fix, independent of the oracle's own code.

Each test names the passage of PAPER.md (or the DESIGN.md reading) it pins.  None of them needs a GPU.
"""
from pathlib import Path

import numpy as np
import pytest
import scipy.linalg

import oracle
import workloads as wl

GOLDEN = Path(__file__).resolve().parent / "golden"


# ---------------------------------------------------------------------------
# helpers that do NOT call the oracle
# ---------------------------------------------------------------------------

def naive_dft(x: np.ndarray, sign: int) -> np.ndarray:
    """O(N^2) definition, axis by axis: X_l = sum_j x_j exp(sign 2 pi i j l / n); exponent reduced in integers."""
    y = np.asarray(x, dtype=np.complex128)
    for ax, n in enumerate(y.shape):
        j = np.arange(n)
        M = np.exp(sign * 2j * np.pi * ((j[:, None] * j[None, :]) % n) / n)
        y = np.moveaxis(np.tensordot(M, np.moveaxis(y, ax, 0), axes=(1, 0)), 0, ax)
    return y


def parse_matrices(path: Path, dim: int):
    tok = {"0": 0, "1": 1, "-1": -1, "i": 1j, "-i": -1j}
    rows = [[tok[t] for t in ln.split()] for ln in path.read_text().splitlines() if ln.strip() and not ln.startswith("#")]
    arr = np.array(rows, dtype=np.complex128)
    return arr.reshape(-1, dim, dim)


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(np.asarray(b).ravel()))


# ---------------------------------------------------------------------------
# 1. the FFT against the DFT definition (eq. 12 sign)
# ---------------------------------------------------------------------------

@pytest.mark.parametrize("shape", [(1,), (2,), (4,), (8,), (16,), (64,), (8, 16), (32, 4), (4, 8, 2), (16, 2, 8)])
def test_fft_matches_naive_dft(shape):
    rng = np.random.default_rng(7)
    x = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    N = x.size
    fwd = oracle.fft(x, -1)
    np.testing.assert_allclose(fwd, naive_dft(x, -1), rtol=0, atol=1e-12 * np.sqrt(N))
    inv = oracle.fft(x, +1)
    np.testing.assert_allclose(inv, naive_dft(x, +1) / N, rtol=0, atol=1e-12)


def test_fft_single_mode_and_sign():
    # x_j = exp(+2 pi i 3 j / n) must land in bin 3 of the *forward* (minus-sign) transform (eq. 12)
    n = 32
    j = np.arange(n)
    X = oracle.fft(np.exp(2j * np.pi * 3 * j / n), -1)
    want = np.zeros(n, complex)
    want[3] = n
    np.testing.assert_allclose(X, want, atol=1e-12)


@pytest.mark.parametrize("shape", [(4096,), (256, 128), (32, 64, 16)])
def test_fft_roundtrip_and_parseval(shape):
    rng = np.random.default_rng(11)
    x = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    X = oracle.fft(x, -1)
    assert abs(np.sum(np.abs(X) ** 2) / x.size - np.sum(np.abs(x) ** 2)) < 1e-10 * np.sum(np.abs(x) ** 2)
    assert rel_l2(oracle.fft(X, +1), x) < 1e-14


def test_grids_convention():
    # G14: r_{n/2} = 0, half open; k Nyquist negative; k dx n / 2 pi are the signed integers
    r, k = oracle.grids(16, 0.25)
    assert r[8] == 0.0 and r[0] == -2.0 and r[-1] == 1.75
    m = k * 16 * 0.25 / (2 * np.pi)
    np.testing.assert_allclose(m, [0, 1, 2, 3, 4, 5, 6, 7, -8, -7, -6, -5, -4, -3, -2, -1], atol=1e-14)
    np.testing.assert_allclose(r, wl.axis_r(16, 0.25))
    np.testing.assert_allclose(k, wl.axis_k(16, 0.25))


# ---------------------------------------------------------------------------
# 2. free Gaussian packet: k-grid, sign and 1/2 of the kinetic phase, 1/N (eq. 13)
# ---------------------------------------------------------------------------

def free_gaussian(x, t, x0, p0, sigma):
    """Textbook solution of i psi_t = -psi_xx/2 for psi(x,0) = (pi sigma^2)^(-1/4) exp(-(x-x0)^2/(2 sigma^2) + i p0 (x-x0))."""
    z = 1.0 + 1j * t / sigma**2
    return (np.pi * sigma**2) ** (-0.25) * z ** (-0.5) * np.exp(
        -((x - x0 - p0 * t) ** 2) / (2.0 * sigma**2 * z) + 1j * p0 * (x - x0) - 0.5j * p0**2 * t)


@pytest.mark.parametrize("p0", [0.0, 1.5, -2.0])
def test_free_gaussian_closed_form(p0):
    n, dx, dt, steps = 4096, 400.0 / 4096.0, 0.01, 1000
    x = wl.axis_r(n, dx)
    x0, sigma = 5.0, 1.0
    s = oracle.Solver((n,), (dx,), dt)
    psi = s.step(free_gaussian(x, 0.0, x0, p0, sigma)[None], steps)[0]
    want = free_gaussian(x, steps * dt, x0, p0, sigma)
    assert rel_l2(psi, want) < 2e-12
    # variance of |psi|^2: sigma^2/2 (1 + t^2/sigma^4)
    rho = np.abs(psi) ** 2 * dx
    mean = np.sum(x * rho)
    var = np.sum((x - mean) ** 2 * rho)
    t = steps * dt
    assert abs(mean - (x0 + p0 * t)) < 1e-11
    assert abs(var - 0.5 * sigma**2 * (1 + t**2 / sigma**4)) < 1e-11


def test_free_gaussian_2d_axis_order():
    # different sizes, spacings and momenta per axis: a transposed axis or swapped k-grid fails
    sizes, dx, dt, steps = (256, 128), (0.25, 0.4), 0.02, 50
    X, Y = wl.mesh(sizes, dx)
    f = lambda t: free_gaussian(X, t, -2.0, 1.0, 1.5) * free_gaussian(Y, t, 3.0, -0.5, 2.0)
    s = oracle.Solver(sizes, dx, dt)
    psi = s.step(f(0.0)[None], steps)[0]
    assert rel_l2(psi, f(steps * dt)) < 1e-11


def test_mass_enters_kinetic_phase():
    n, dx, dt, steps, m = 2048, 0.1, 0.01, 100, 2.5
    x = wl.axis_r(n, dx)
    # mass m: the free solution is the m=1 one at time t/m with momentum p0 (velocity p0/m)
    s = oracle.Solver((n,), (dx,), dt, mass=m)
    psi = s.step(free_gaussian(x, 0.0, 1.0, 2.0, 1.0)[None], steps)[0]
    want = free_gaussian(x, steps * dt / m, 1.0, 2.0, 1.0)
    assert rel_l2(psi, want) < 1e-11


# ---------------------------------------------------------------------------
# 3. harmonic well: V phase + Strang ordering (eq. 7, 11).  For a quadratic
# potential <x>,<p> follow the Stoermer-Verlet map exactly:
# x_n = x0 cos(n w~ tau), cos(w~ tau) = 1 - w^2 tau^2 / 2.
# ---------------------------------------------------------------------------

def test_harmonic_centroid_follows_verlet_period():
    w = wl.config1(noise=0.0)
    s = oracle.Solver(w.sizes, w.dx, w.dt)
    s.set_potential(w.V)
    x = wl.axis_r(w.sizes[0], w.dx[0])
    wt = np.arccos(1.0 - 0.5 * w.dt**2)
    psi = w.psi0
    worst = 0.0
    done = 0
    for chunk in [1, 9, 90, 400, 500]:
        psi = s.step(psi, chunk)
        done += chunk
        mean = np.sum(x * np.abs(psi[0]) ** 2) * w.dx[0]
        worst = max(worst, abs(mean - 5.0 * np.cos(done * wt)))
    assert worst < 2e-11
    # against the continuous-time cos(t) the discrepancy is ~1e-4: the pin is the Verlet period, not omega
    assert abs(5.0 * np.cos(1000 * wt) - 5.0 * np.cos(10.0)) > 1e-5


def test_coherent_state_width_is_constant():
    # G9: sigma = 1 amplitude width is the m = omega = 1 coherent state: density variance stays 1/2
    w = wl.config1(noise=0.0)
    s = oracle.Solver(w.sizes, w.dx, w.dt)
    s.set_potential(w.V)
    x = wl.axis_r(w.sizes[0], w.dx[0])
    psi = s.step(w.psi0, 157)  # a quarter period
    rho = np.abs(psi[0]) ** 2 * w.dx[0]
    mean = np.sum(x * rho)
    assert abs(np.sum((x - mean) ** 2 * rho) - 0.5) < 1e-4


# ---------------------------------------------------------------------------
# 4/5. unitarity and reversibility (product of unitary factors, eq. 7/8)
# ---------------------------------------------------------------------------

def test_norm_conserved_1000_steps():
    w = wl.config1()
    s = oracle.Solver(w.sizes, w.dx, w.dt)
    s.set_potential(w.V)
    n0 = s.norm(w.psi0)
    assert abs(n0 - 1.0) < 1e-13
    psi = s.step(w.psi0, 1000)
    assert abs(s.norm(psi) - n0) < 1e-12


@pytest.mark.parametrize("ncomp,sizes", [(1, (64, 32)), (2, (32, 64)), (4, (16, 16, 8)), (2, (128,)), (4, (64,))])
def test_reversibility_and_norm(ncomp, sizes):
    dx = (0.3,) * len(sizes)
    rng = np.random.default_rng(5)
    V = rng.uniform(-2, 2, size=sizes)
    psi0 = wl.random_state(sizes, ncomp, 3, dx)
    f = oracle.Solver(sizes, dx, 0.01, ncomp=ncomp)
    b = oracle.Solver(sizes, dx, -0.01, ncomp=ncomp)
    f.set_potential(V)
    b.set_potential(V)
    psi = f.step(psi0, 7)
    assert abs(f.norm(psi) - f.norm(psi0)) < 1e-13
    assert rel_l2(psi, psi0) > 1e-3
    assert rel_l2(b.step(psi, 7), psi0) < 1e-13


# ---------------------------------------------------------------------------
# 6. Dirac matrices: the paper's printed eq. 16 / 17 and the algebra eq. 15
# ---------------------------------------------------------------------------

def test_dirac_matrices_are_the_papers():
    g16 = parse_matrices(GOLDEN / "dirac_matrices_eq16.txt", 4)
    al, be = oracle.dirac_matrices(4)
    np.testing.assert_array_equal(al, g16[:3])
    np.testing.assert_array_equal(be, g16[3])
    g17 = parse_matrices(GOLDEN / "dirac_matrices_eq17.txt", 2)
    al2, be2 = oracle.dirac_matrices(2)
    np.testing.assert_array_equal(al2[0], g17[0])
    np.testing.assert_array_equal(be2, g17[1])
    # G7: the second 2x2 matrix is sigma_y = the {1,4} block of alpha_2
    np.testing.assert_array_equal(al2[1], g16[1][np.ix_([0, 3], [0, 3])])
    np.testing.assert_array_equal(al2[0], g16[0][np.ix_([0, 3], [0, 3])])
    np.testing.assert_array_equal(be2, g16[3][np.ix_([0, 3], [0, 3])])


@pytest.mark.parametrize("C", [2, 4])
def test_dirac_algebra_eq15(C):
    al, be = oracle.dirac_matrices(C)
    nal = 3 if C == 4 else 2
    I = np.eye(C)
    np.testing.assert_array_equal(be @ be, I)
    for i in range(nal):
        np.testing.assert_array_equal(al[i] @ be + be @ al[i], 0 * I)
        for k in range(nal):
            np.testing.assert_array_equal(al[i] @ al[k] + al[k] @ al[i], 2 * I * (i == k))


# ---------------------------------------------------------------------------
# 7. Dirac kinetic factor: eq. 29-33 against brute-force expm(-i H tau) with H
# assembled from the *golden* matrices, not the oracle's
# ---------------------------------------------------------------------------

def golden_hamiltonian(C, p, m, c):
    g16 = parse_matrices(GOLDEN / "dirac_matrices_eq16.txt", 4)
    if C == 4:
        al, be = g16[:3], g16[3]
    else:
        sel = np.ix_([0, 3], [0, 3])
        al, be = [g[sel] for g in g16[:3]], g16[3][sel]
    return sum(c * pi * a for pi, a in zip(p, al)) + m * c * c * be


@pytest.mark.parametrize("C,ndim", [(2, 1), (2, 2), (4, 1), (4, 2), (4, 3)])
def test_dirac_kinetic_equals_expm(C, ndim):
    rng = np.random.default_rng(100 + 10 * C + ndim)
    m, c = 1.0, 137.036
    for trial in range(12):
        p = rng.uniform(-60, 60, size=ndim) if trial else np.zeros(ndim)
        if trial == 1:
            p = np.array([1e-9] + [0.0] * (ndim - 1))
        tau = rng.choice([1e-4, -1e-4, 3e-5])
        H = golden_hamiltonian(C, p, m, c)
        want = scipy.linalg.expm(-1j * tau * H)
        U = oracle.dirac_kinetic_matrix(C, p, m, c, tau)
        np.testing.assert_allclose(U, want, atol=5e-14)
        np.testing.assert_allclose(U @ oracle.dirac_kinetic_matrix(C, p, m, c, -tau), np.eye(C), atol=1e-14)
        # eq. 30/31: u unitary and diagonalising
        u = oracle.dirac_u(C, p, m, c)
        E = np.sqrt(m * m * c**4 + np.dot(p, p) * c * c)
        np.testing.assert_allclose(u @ u.conj().T, np.eye(C), atol=1e-14)
        D = np.diag([E] * (C // 2) + [-E] * (C // 2))
        np.testing.assert_allclose(u @ H @ u.conj().T, D, atol=1e-9)


def test_dirac_kinetic_other_mass_and_c():
    p = np.array([0.7, -1.1, 0.4])
    H = golden_hamiltonian(4, p, 2.0, 10.0)
    np.testing.assert_allclose(oracle.dirac_kinetic_matrix(4, p, 2.0, 10.0, 0.013), scipy.linalg.expm(-0.013j * H), atol=1e-14)


def test_dirac_four_component_block_is_two_component():
    # G7: with p3 = 0 the {1,4} block of eq. 16 is the 2-component problem
    p = np.array([3.0, -4.0])
    U4 = oracle.dirac_kinetic_matrix(4, p, 1.0, 137.036, 1e-4)
    U2 = oracle.dirac_kinetic_matrix(2, p, 1.0, 137.036, 1e-4)
    np.testing.assert_allclose(U4[np.ix_([0, 3], [0, 3])], U2, atol=1e-15)
    np.testing.assert_allclose(U4[np.ix_([0, 3], [1, 2])], 0, atol=1e-15)


def test_dirac_2d_four_vs_two_component_propagation():
    sizes, dx = (32, 64), (0.1, 0.1)
    w = wl.config4(sizes=sizes, nsteps=5)
    s2 = oracle.Solver(sizes, dx, w.dt, ncomp=2)
    s4 = oracle.Solver(sizes, dx, w.dt, ncomp=4)
    for s in (s2, s4):
        s.set_potential(w.V)
        s.set_field(oracle.FIELD_A, w.step_avg)
    psi4 = np.zeros((4,) + sizes, complex)
    psi4[0], psi4[3] = w.psi0[0], w.psi0[1]
    out2 = s2.step(w.psi0, 5)
    out4 = s4.step(psi4, 5)
    assert rel_l2(out4[[0, 3]], out2) < 1e-13
    assert np.max(np.abs(out4[[1, 2]])) < 1e-14


# ---------------------------------------------------------------------------
# 8. free Dirac dispersion E = +-sqrt(c^2 k^2 + c^4) (eq. 32) on the grid
# ---------------------------------------------------------------------------

@pytest.mark.parametrize("C,sizes,idx", [(2, (64,), (5,)), (2, (32, 16), (3, 13)), (4, (16, 8, 8), (2, 7, 1)), (4, (32, 32), (30, 4))])
def test_dirac_plane_wave_dispersion(C, sizes, idx):
    dx = (0.1,) * len(sizes)
    c, m, dt, steps = 137.036, 1.0, 1e-4, 100
    kax = [wl.axis_k(n, d) for n, d in zip(sizes, dx)]
    k0 = np.array([ka[i] for ka, i in zip(kax, idx)])
    R = wl.mesh(sizes, dx)
    wave = np.exp(1j * sum(k * Ra for k, Ra in zip(k0, R)))
    E = np.sqrt(c * c * np.dot(k0, k0) + m * m * c**4)
    spin = wl.positive_energy_spinor([np.array(k) for k in k0], C, m, c)  # textbook spinor, not the oracle's u
    psi0 = np.stack([sp * wave for sp in spin])
    s = oracle.Solver(sizes, dx, dt, ncomp=C, mass=m, c=c)
    out = s.step(psi0, steps)
    assert rel_l2(out, np.exp(-1j * E * steps * dt) * psi0) < 2e-12
    # a negative-energy state picks up e^{+iEt}: charge-conjugate-like spinor orthogonal to the positive ones
    H = golden_hamiltonian(C, k0, m, c)
    evals, evecs = np.linalg.eigh(H)
    neg = evecs[:, 0]
    assert abs(evals[0] + E) < 1e-8
    psin = np.stack([a * wave for a in neg])
    outn = s.step(psin, steps)
    assert rel_l2(outn, np.exp(+1j * E * steps * dt) * psin) < 2e-12


# ---------------------------------------------------------------------------
# 9. time-dependent field plumbing (G12, G16)
# ---------------------------------------------------------------------------

def test_field_E_is_a_momentum_kick():
    # V = 0, constant Ebar: each step changes <p> by -Ebar tau exactly (two half kicks), any psi
    sizes, dx, dt = (512,), (0.1,), 0.02
    x = wl.axis_r(*sizes, *dx)
    k = wl.axis_k(*sizes, *dx)
    psi0 = wl.gaussian_packet(sizes, dx, (1.0,), (0.7,), 1.5)[None]
    s = oracle.Solver(sizes, dx, dt)
    Ebar = 0.35
    s.set_field(oracle.FIELD_E, np.full((10, 1), Ebar))

    def mean_p(psi):
        ph = np.fft.fft(psi[0])
        return float(np.sum(k * np.abs(ph) ** 2) / np.sum(np.abs(ph) ** 2))

    p_before = mean_p(psi0)
    out = s.step(psi0, 10)
    assert abs((mean_p(out) - p_before) - (-Ebar * dt * 10)) < 1e-10
    with pytest.raises(ValueError):
        s.step(out, 1)  # table exhausted


def test_field_E_time_index_and_axis():
    sizes, dx, dt = (32, 64), (0.2, 0.1), 0.02
    w = wl.config2(sizes=sizes, nsteps=6)
    s = oracle.Solver(sizes, dx, dt)
    s.set_potential(w.V)
    s.set_field(oracle.FIELD_E, w.step_avg)
    a = s.step(s.step(w.psi0, 2), 4)
    s.set_time_index(0)
    b = s.step(w.psi0, 6)
    assert rel_l2(a, b) < 1e-15
    # the same evolution with the field folded into V by hand, step by step (axis 0 is "x", G26)
    X, _ = wl.mesh(sizes, dx)
    psi = w.psi0
    for n in range(6):
        t = oracle.Solver(sizes, dx, dt)
        t.set_potential(w.V + X * w.step_avg[n, 0])
        psi = t.step(psi, 1)
    assert rel_l2(psi, b) < 1e-14


def test_field_A_shifts_the_kinetic_momentum():
    # Dirac + constant Abar: a plane wave at grid momentum k0 with the spinor of pi = k0 - q Abar is stationary
    sizes, dx = (32, 16), (0.1, 0.1)
    c, m, q, dt, steps = 137.036, 1.0, -1.0, 1e-4, 20
    kax = [wl.axis_k(n, d) for n, d in zip(sizes, dx)]
    k0 = np.array([kax[0][3], kax[1][14]])
    A = np.array([5.0, -2.0])
    pi = k0 - q * A
    R = wl.mesh(sizes, dx)
    wave = np.exp(1j * sum(k * Ra for k, Ra in zip(k0, R)))
    spin = wl.positive_energy_spinor([np.array(p) for p in pi], 2, m, c)
    psi0 = np.stack([sp * wave for sp in spin])
    E = np.sqrt(c * c * np.dot(pi, pi) + m * m * c**4)
    s = oracle.Solver(sizes, dx, dt, ncomp=2, mass=m, c=c, charge=q)
    s.set_field(oracle.FIELD_A, np.tile(A, (steps, 1)))
    out = s.step(psi0, steps)
    assert rel_l2(out, np.exp(-1j * E * steps * dt) * psi0) < 1e-12
    # Schroedinger: phase exp(-i (k0 - qA)^2 t / 2)
    s1 = oracle.Solver(sizes, dx, 0.01)
    s1.set_field(oracle.FIELD_A, np.tile(A, (steps, 1)))
    out1 = s1.step(wave[None], steps)
    assert rel_l2(out1, np.exp(-0.5j * np.dot(pi, pi) * steps * 0.01) * wave[None]) < 1e-12


# ---------------------------------------------------------------------------
# 10. loose physics sanity from the paper's text, and the sampled inverse
# ---------------------------------------------------------------------------

def test_classical_velocity_quoted_in_the_paper():
    vals = {ln.split()[0]: float(ln.split()[1]) for ln in (GOLDEN / "paper_constants.txt").read_text().splitlines() if ln and not ln.startswith("#")}
    v = 40.0 / np.sqrt(1 + 40.0**2 / 137.036**2)
    assert abs(v - vals["classical_packet_velocity_au"]) < 0.5


def test_inverse_sample_matches_full_step():
    w = wl.config4(sizes=(16, 32), nsteps=3)
    s = oracle.Solver(w.sizes, w.dx, w.dt, ncomp=2)
    s.set_potential(w.V)
    s.set_field(oracle.FIELD_A, w.step_avg)
    full = s.step(w.psi0, 1)
    psik = s.half_step_to_k(w.psi0, 0)
    for j in [0, 17, 16 * 32 - 1, 200]:
        got = s.inverse_sample(psik, 0, j)
        np.testing.assert_allclose(got, full.reshape(2, -1)[:, j], atol=1e-14)
    w2 = wl.config2(sizes=(16, 8), nsteps=3)
    s2 = oracle.Solver(w2.sizes, w2.dx, w2.dt)
    s2.set_potential(w2.V)
    s2.set_field(oracle.FIELD_E, w2.step_avg)
    s2.set_time_index(1)
    full = s2.step(w2.psi0, 1)
    psik = s2.half_step_to_k(w2.psi0, 1)
    np.testing.assert_allclose(s2.inverse_sample(psik, 1, 77), full.reshape(1, -1)[:, 77], atol=1e-14)


def test_workload_generators_are_normalised_and_seeded():
    for mk, kw in [(wl.config1, {}), (wl.config2, dict(sizes=(64, 32))), (wl.config3, dict(sizes=(16, 32, 8))),
                   (wl.config4, dict(sizes=(32, 64))), (wl.config5, dict(sizes=(16, 8, 16)))]:
        a, b = mk(**kw), mk(**kw)
        np.testing.assert_array_equal(a.psi0, b.psi0)
        assert abs(np.sum(np.abs(a.psi0) ** 2) * np.prod(a.dx) - 1.0) < 1e-12
        assert a.psi0.shape == (a.ncomp,) + a.sizes and a.V.shape == a.sizes
