"""Dense one-step pin for the CPU oracle: the whole step as one matrix, built without the oracle.

For tiny lattices the step of PAPER.md:71 (eq. 7) in its Fourier form PAPER.md:76-78 (eq. 8) is the matrix

    S_n = P_n . F^-1 . K_n . F . P_n ,      P_n = diag(exp(-i Vbar_n(r) tau/2)) (x) 1_C     (eq. 11, eq. 22)

with F the naive O(N^2) DFT matrix of the lattice (eq. 12: forward = minus sign, 1/N on the inverse), and K_n
block diagonal over k: the scalar exp(-i tau |k - q Abar_n|^2 / 2m) (eq. 13) for one component, and
scipy's expm(-i tau H(k - q Abar_n)) with H = c sum_a alpha_a pi_a + m c^2 beta (eq. 14/18b) assembled from the
matrices typed from the paper in tests/golden/ for a spinor.  Everything here is numpy/scipy; nothing calls the
oracle except the comparison.  This pins, in one test: the component loop of the potential half step for
ncomp > 1 (eq. 22: the same phase on every component), the component indexing of the Dirac kinetic factor, the
3D kinetic and 3D field paths, the r.Ebar term of SSO_FIELD_E and the k - q Abar shift of SSO_FIELD_A, and the
step-index bookkeeping of the field table over several steps.
"""
import itertools
from pathlib import Path

import numpy as np
import pytest
import scipy.linalg

import oracle

GOLDEN = Path(__file__).resolve().parent / "golden"
TOK = {"0": 0, "1": 1, "-1": -1, "i": 1j, "-i": -1j}


def golden(name: str, dim: int) -> np.ndarray:
    rows = [[TOK[t] for t in ln.split()] for ln in (GOLDEN / name).read_text().splitlines() if ln.strip() and not ln.startswith("#")]
    return np.array(rows, dtype=np.complex128).reshape(-1, dim, dim)


def alpha_beta(C: int, ndim: int):
    """alpha_1..alpha_ndim and beta as printed in the paper: eq. 16 for four components; eq. 17 for two components
    in one dimension; the {1,4} block of eq. 16 for two components in two dimensions (reading G7)."""
    g16 = golden("dirac_matrices_eq16.txt", 4)
    if C == 4:
        return list(g16[:ndim]), g16[3]
    if ndim == 1:
        g17 = golden("dirac_matrices_eq17.txt", 2)
        return [g17[0]], g17[1]
    sel = np.ix_([0, 3], [0, 3])
    return [g[sel] for g in g16[:ndim]], g16[3][sel]


def lattice(sizes, dx):
    """r_j = (j - n/2) dx and k_j in DFT order with the Nyquist frequency negative (reading G14), per axis."""
    r = [(np.arange(n) - n // 2) * d for n, d in zip(sizes, dx)]
    k = [2.0 * np.pi * np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n) / (n * d) for n, d in zip(sizes, dx)]
    return r, k


def dft_matrix(sizes) -> np.ndarray:
    """Forward DFT of the whole lattice as one N x N matrix (Kronecker product of the per-axis definitions)."""
    F = np.ones((1, 1), dtype=np.complex128)
    for n in sizes:
        j = np.arange(n)
        F = np.kron(F, np.exp(-2j * np.pi * ((j[:, None] * j[None, :]) % n) / n))
    return F


def dense_step(sizes, dx, tau, C, V, kind, avg_row, m, c, q) -> np.ndarray:
    """The (C N) x (C N) matrix of one step; component-major ordering like psi[ncomp][n0][n1][n2]."""
    nd, N = len(sizes), int(np.prod(sizes))
    r, k = lattice(sizes, dx)
    idx = list(itertools.product(*[range(n) for n in sizes]))  # C order: last axis fastest
    vbar = V.reshape(-1).astype(np.float64).copy()
    if kind == oracle.FIELD_E:
        vbar += np.array([sum(r[a][j[a]] * avg_row[a] for a in range(nd)) for j in idx])
    P = np.kron(np.eye(C), np.diag(np.exp(-0.5j * tau * vbar)))
    F1 = dft_matrix(sizes)
    F = np.kron(np.eye(C), F1)
    Finv = np.kron(np.eye(C), F1.conj().T / N)
    shift = q * np.asarray(avg_row) if kind == oracle.FIELD_A else np.zeros(nd)
    K = np.zeros((C * N, C * N), dtype=np.complex128)
    al, be = (None, None) if C == 1 else alpha_beta(C, nd)
    for col, j in enumerate(idx):
        pi = np.array([k[a][j[a]] for a in range(nd)]) - shift
        if C == 1:
            K[col, col] = np.exp(-1j * tau * np.dot(pi, pi) / (2.0 * m))
        else:
            H = sum(c * p * a for p, a in zip(pi, al)) + m * c * c * be
            U = scipy.linalg.expm(-1j * tau * H)
            for s in range(C):
                for t in range(C):
                    K[s * N + col, t * N + col] = U[s, t]
    return P @ Finv @ K @ F @ P


CASES = [
    # C, sizes, field kind
    (1, (8,), oracle.FIELD_NONE), (1, (4, 8), oracle.FIELD_E), (1, (2, 4, 4), oracle.FIELD_E), (1, (4, 2, 4), oracle.FIELD_A),
    (2, (8,), oracle.FIELD_A), (2, (4, 8), oracle.FIELD_A), (2, (8, 4), oracle.FIELD_E), (2, (16,), oracle.FIELD_NONE),
    (4, (8,), oracle.FIELD_E), (4, (4, 4), oracle.FIELD_A), (4, (2, 4, 4), oracle.FIELD_A), (4, (4, 2, 2), oracle.FIELD_E),
    (4, (2, 2, 8), oracle.FIELD_NONE),
]


@pytest.mark.parametrize("C,sizes,kind", CASES, ids=[f"C{c}-{'x'.join(map(str, s))}-field{k}" for c, s, k in CASES])
def test_oracle_step_equals_dense_matrix(C, sizes, kind):
    nd, N = len(sizes), int(np.prod(sizes))
    rng = np.random.default_rng(1000 * C + 10 * N + kind)
    dx = tuple(rng.uniform(0.05, 0.3, size=nd))
    # Dirac: c tau |k| and m c^2 tau of order one so that every entry of the 4x4 unitary matters
    tau = 1e-4 * (1 if rng.random() < 0.5 else -1) if C > 1 else 0.013
    m, c, q = (1.3, 137.036, -1.0) if C > 1 else (0.8, 137.036, 0.7)
    V = rng.uniform(-40.0, 40.0, size=sizes) / (abs(tau) * 100.0 if C > 1 else 1.0)
    nsteps = 3
    avg = rng.uniform(-3.0, 3.0, size=(nsteps + 2, nd)) * (50.0 if kind == oracle.FIELD_E and C > 1 else 1.0)
    psi0 = rng.standard_normal((C,) + sizes) + 1j * rng.standard_normal((C,) + sizes)
    s = oracle.Solver(sizes, dx, tau, ncomp=C, mass=m, c=c, charge=q)
    s.set_potential(V)
    if kind != oracle.FIELD_NONE:
        s.set_field(kind, avg)
    n0 = 1  # start at a non-zero step index: the rows used are n0, n0+1, ...
    s.set_time_index(n0)
    got = s.step(psi0, nsteps)
    want = psi0.reshape(-1)
    for n in range(n0, n0 + nsteps):
        want = dense_step(sizes, dx, tau, C, V, kind, avg[n], m, c, q) @ want
    scale = np.abs(want).max()
    np.testing.assert_allclose(got.reshape(-1), want, rtol=0, atol=2e-13 * scale)


def test_dense_step_detects_a_phase_on_one_component_only():
    """The pin has teeth: the same matrix with the potential phase on component 0 only (the mistake eq. 22 rules
    out) differs from the oracle by far more than the tolerance."""
    C, sizes = 4, (4, 4)
    rng = np.random.default_rng(5)
    dx, tau = (0.1, 0.2), 1e-4
    V = rng.uniform(-4000.0, 4000.0, size=sizes)
    psi0 = rng.standard_normal((C,) + sizes) + 1j * rng.standard_normal((C,) + sizes)
    s = oracle.Solver(sizes, dx, tau, ncomp=C)
    s.set_potential(V)
    got = s.step(psi0, 1).reshape(-1)
    N = 16
    S = dense_step(sizes, dx, tau, C, V, oracle.FIELD_NONE, None, 1.0, 137.036, -1.0)
    assert np.abs(S @ psi0.reshape(-1) - got).max() < 1e-12 * np.abs(got).max()
    Pbad = np.eye(C * N, dtype=np.complex128)
    Pbad[:N, :N] = np.diag(np.exp(-0.5j * tau * V.reshape(-1)))
    Pgood = np.kron(np.eye(C), np.diag(np.exp(-0.5j * tau * V.reshape(-1))))
    Sbad = Pbad @ np.linalg.solve(Pgood, S @ np.linalg.solve(Pgood, Pbad))
    assert np.abs(Sbad @ psi0.reshape(-1) - got).max() > 1e-3 * np.abs(got).max()
