"""Pins for the oracle's position-space vector-potential factor (the paper's own Dirac interaction factor):
PAPER.md:138-144 (eq. 18a), 168-184 (eq. 23/24), 188-198 (eq. 25/26), 236 (eq. 34).  Nothing here needs a GPU and
nothing but the comparisons calls the oracle: matrices come from tests/golden/, exponentials from scipy.
"""
import numpy as np
import pytest
import scipy.linalg

import oracle
import workloads as wl
from test_oracle_dense_step import alpha_beta, dense_step, lattice


def exp_i_a_alpha(C, ndim, a):
    al, _ = alpha_beta(C, ndim)
    return scipy.linalg.expm(1j * sum(ai * m for ai, m in zip(a, al)))


@pytest.mark.parametrize("C,ndim", [(2, 1), (2, 2), (4, 1), (4, 2), (4, 3)])
def test_closed_form_equals_matrix_exponential(C, ndim):
    """eq. 23/24: exp(i sum a_i alpha_i) = cos a + i (sum a_i alpha_i / a) sin a, including a = 0 and tiny a."""
    rng = np.random.default_rng(50 + 10 * C + ndim)
    for trial in range(10):
        a = rng.uniform(-4.0, 4.0, size=ndim)
        if trial == 0:
            a = np.zeros(ndim)
        if trial == 1:
            a = np.array([1e-12] + [0.0] * (ndim - 1))
        M = oracle.alpha_rotation(C, a)
        np.testing.assert_allclose(M, exp_i_a_alpha(C, ndim, a), atol=2e-15)
        np.testing.assert_allclose(M @ M.conj().T, np.eye(C), atol=2e-15)


def test_equation_26_as_printed_is_the_electron_case():
    """eq. 26 has no q: (cos(-delta c Abar) + i sum (Abar_i/Abar) alpha_i sin(-delta c Abar)) psi.
    With a_i = delta q c Abar_i that is the general closed form for q = -1 (reading G4) -- and not for q = +1."""
    g16 = alpha_beta(4, 3)[0]
    rng = np.random.default_rng(26)
    Abar = rng.uniform(-1e-3, 1e-3, size=3)  # time integral of A over a step
    delta, c = 0.5, 137.036
    An = np.linalg.norm(Abar)
    printed = np.cos(-delta * c * An) * np.eye(4) + 1j * sum(A / An * m for A, m in zip(Abar, g16)) * np.sin(-delta * c * An)
    np.testing.assert_allclose(oracle.alpha_rotation(4, delta * (-1.0) * c * Abar), printed, atol=1e-15)
    assert np.abs(oracle.alpha_rotation(4, delta * (+1.0) * c * Abar) - printed).max() > 1e-3


CASES = [(2, (8,), oracle.FIELD_NONE), (2, (4, 8), oracle.FIELD_A), (4, (4, 4), oracle.FIELD_E), (4, (2, 4, 2), oracle.FIELD_NONE), (4, (8,), oracle.FIELD_A)]


@pytest.mark.parametrize("C,sizes,kind", CASES, ids=[f"C{c}-{'x'.join(map(str, s))}-field{k}" for c, s, k in CASES])
def test_step_with_position_space_factor_equals_dense_matrix(C, sizes, kind):
    """One step = R P F^-1 K F P R with R = blockdiag_r exp(i (tau/2) q c sum_i A_i(r) alpha_i) (eq. 7 with eq. 18a),
    built from scipy's expm on the paper's matrices and the naive DFT (dense_step of test_oracle_dense_step)."""
    nd, N = len(sizes), int(np.prod(sizes))
    rng = np.random.default_rng(7 * C + N + kind)
    dx = tuple(rng.uniform(0.05, 0.3, size=nd))
    tau, m, c, q = 1e-4, 1.2, 137.036, -1.0
    V = rng.uniform(-2000.0, 2000.0, size=sizes)
    A = rng.uniform(-60.0, 60.0, size=(nd,) + sizes)   # c tau |A| / 2 of order 0.4
    avg = rng.uniform(-3.0, 3.0, size=(5, nd))
    psi0 = rng.standard_normal((C,) + sizes) + 1j * rng.standard_normal((C,) + sizes)
    s = oracle.Solver(sizes, dx, tau, ncomp=C, mass=m, c=c, charge=q)
    s.set_potential(V)
    s.set_vector_potential(A)
    if kind != oracle.FIELD_NONE:
        s.set_field(kind, avg)
    got = s.step(psi0, 2).reshape(-1)
    R = np.zeros((C * N, C * N), dtype=np.complex128)
    Aflat = A.reshape(nd, N)
    for j in range(N):
        M = exp_i_a_alpha(C, nd, 0.5 * tau * q * c * Aflat[:, j])
        for r_ in range(C):
            for s_ in range(C):
                R[r_ * N + j, s_ * N + j] = M[r_, s_]
    want = psi0.reshape(-1)
    for n in range(2):
        want = R @ (dense_step(sizes, dx, tau, C, V, kind, avg[n], m, c, q) @ (R @ want))
    np.testing.assert_allclose(got, want, rtol=0, atol=2e-13 * np.abs(want).max())


def test_homogeneous_field_agrees_with_the_kinetic_variant_to_second_order():
    """For a homogeneous A the paper's splitting (A in position space) and BASELINE's (A in the kinetic factor,
    reading G16) are both second order: their difference after a fixed time falls like tau^2."""
    sizes, dx = (64,), (0.05,)
    T, A0 = 8e-4, 30.0
    w = wl.dirac1d(sizes=sizes, nsteps=1, ncomp=2)
    diffs = []
    for nsteps in (32, 64, 128):
        tau = T / nsteps
        kin = oracle.Solver(sizes, dx, tau, ncomp=2)
        kin.set_potential(w.V * 200.0)
        kin.set_field(oracle.FIELD_A, np.full((nsteps, 1), A0))
        pos = oracle.Solver(sizes, dx, tau, ncomp=2)
        pos.set_potential(w.V * 200.0)
        pos.set_vector_potential(np.full((1,) + sizes, A0))
        a, b = kin.step(w.psi0, nsteps), pos.step(w.psi0, nsteps)
        diffs.append(np.linalg.norm(a - b) / np.linalg.norm(a))
    assert diffs[0] > 1e-9                      # the two splittings are not the same thing
    assert 3.6 < diffs[0] / diffs[1] < 4.5 and 3.8 < diffs[1] / diffs[2] < 4.2, diffs


def test_position_space_factor_is_unitary_and_needs_a_spinor():
    w = wl.config4(sizes=(16, 32), nsteps=5)
    rng = np.random.default_rng(3)
    s = oracle.Solver(w.sizes, w.dx, w.dt, ncomp=2)
    s.set_potential(w.V)
    s.set_vector_potential(rng.uniform(-50, 50, size=(2,) + w.sizes))
    out = s.step(w.psi0, 5)
    assert abs(s.norm(out) - 1.0) < 1e-13
    s1 = oracle.Solver((16,), (0.1,), 0.01, ncomp=1)
    s1.set_vector_potential(np.ones((1, 16)))
    with pytest.raises(ValueError):
        s1.step(np.ones((1, 16), complex), 1)


def test_pulse_of_equation_46():
    """workloads.pulse_*: eq. 46c envelope, E = omega dA/deta (eq. 46a with E = -dA/dt), A = 0 ahead
    of the pulse, constant behind it, continuous everywhere."""
    j, l, E0, omega = 8, 2, 3000.0, 2 * np.pi * 137.036 / 40.0
    eta = np.linspace(-9 * np.pi, np.pi, 20001)
    f = wl.pulse_envelope(eta, j, l)
    assert f.max() == 1.0 and f.min() == 0.0
    assert np.allclose(wl.pulse_envelope(np.array([-8 * np.pi, -7 * np.pi, -6 * np.pi, -4 * np.pi, -2 * np.pi, -np.pi, 0.0, 1.0, -30.0]), j, l),
                       [0.0, 0.5, 1.0, 1.0, 1.0, 0.5, 0.0, 0.0, 0.0])
    A = wl.pulse_vector_potential(eta, E0, omega, j, l)
    dA = np.gradient(A, eta)
    E = wl.pulse_field(eta, E0, j, l)
    assert np.abs(omega * dA - E)[5:-5].max() < 2e-3 * E0  # second-order finite differences on a 5e-4 pi grid
    assert np.all(A[eta >= 0] == 0.0)
    behind = A[eta <= -j * np.pi]
    assert np.ptp(behind) < 1e-9 * E0 / omega
    # the step average tends to the midpoint value
    x = np.linspace(-40.0, 0.0, 64)
    k = omega / 137.036
    avg = wl.pulse_step_average(x, 0.01, 1e-5, E0, omega, j, l, k)
    mid = wl.pulse_vector_potential(k * x - omega * (0.01 + 0.5e-5), E0, omega, j, l)
    assert np.abs(avg - mid).max() < 1e-6 * np.abs(mid).max()
