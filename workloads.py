"""Seeded synthetic inputs for the five BASELINE.json configs (and reduced-size variants).

This module only *generates inputs* (grids, potentials, initial wavefunctions,
step-averaged field tables) and hands them, as plain numpy arrays, to both the
CPU oracle and the CUDA library.  It holds none of the split-operator step's
arithmetic and imports neither ``oracle`` nor ``paper_1012_3911_b200``.

The paper benchmarks "one- and two-dimensional Gaussian wave packets in a
harmonic potential over 128 time steps" and gives no dx, dt or
widths (G10); BASELINE.json's configs supply them and DESIGN.md
("Input recipe") lists every remaining choice (G22-G27).  No public dataset is
involved.  Seeds: 10123911 + config number.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

FIELD_NONE, FIELD_E, FIELD_A = 0, 1, 2
C_LIGHT = 137.036  # a.u. (BASELINE.json)
SEED0 = 10123911


@dataclass
class Workload:
    name: str
    sizes: tuple
    dx: tuple
    dt: float
    ncomp: int
    nsteps: int
    psi0: np.ndarray                      # complex128, shape (ncomp, *sizes)
    V: Optional[np.ndarray] = None        # float64, shape sizes
    field_kind: int = FIELD_NONE
    step_avg: Optional[np.ndarray] = None  # float64 [nvals][ndim]
    mass: float = 1.0
    c: float = C_LIGHT
    charge: float = -1.0
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def ndim(self) -> int:
        return len(self.sizes)

    @property
    def npoints(self) -> int:
        return int(np.prod(self.sizes))


def axis_r(n: int, dx: float) -> np.ndarray:
    """r_j = (j - n/2) dx, half-open grid (G14)."""
    return (np.arange(n) - n // 2) * dx


def axis_k(n: int, dx: float) -> np.ndarray:
    """k_j in DFT order, Nyquist negative (numpy fftfreq convention, G14)."""
    return 2.0 * np.pi * np.fft.fftfreq(n, d=dx)


def mesh(sizes: Sequence[int], dx: Sequence[float]):
    return np.meshgrid(*[axis_r(n, d) for n, d in zip(sizes, dx)], indexing="ij")


def kmesh(sizes: Sequence[int], dx: Sequence[float]):
    return np.meshgrid(*[axis_k(n, d) for n, d in zip(sizes, dx)], indexing="ij")


def normalise(psi: np.ndarray, dx: Sequence[float]) -> np.ndarray:
    vol = float(np.prod(dx))
    return psi / np.sqrt(np.sum(np.abs(psi) ** 2) * vol)


def sinus_step_average(F0: float, omega: float, dt: float, nvals: int) -> np.ndarray:
    """Exact average of F0 sin(omega t) over [n dt, (n+1) dt] (G12)."""
    n = np.arange(nvals)
    half = 0.5 * omega * dt
    return F0 * np.sin(omega * (n * dt + 0.5 * dt)) * (np.sin(half) / half)


def gaussian_packet(sizes, dx, r0, p0, sigma) -> np.ndarray:
    """exp(-|r-r0|^2/(2 sigma^2) + i p0.r), normalised (G9, G24)."""
    R = mesh(sizes, dx)
    arg = sum(-((Ra - a) ** 2) / (2.0 * sigma**2) for Ra, a in zip(R, r0))
    ph = sum(Ra * p for Ra, p in zip(R, p0))
    return normalise(np.exp(arg + 1j * ph), dx)


def positive_energy_spinor(K, ncomp: int, mass: float, c: float):
    """Textbook free positive-energy, spin-up spinor of H = c alpha.p + m c^2 beta:
    (E + m c^2, 0, c p_z, c (p_x + i p_y)) / sqrt(2 E (E + m c^2)) in the Dirac
    representation (ncomp = 4); its {1,4} components for ncomp = 2 (G7, G8).
    K: list of ndim momentum meshes.  Returns an array (ncomp, *grid)."""
    ndim = len(K)
    px = K[0]
    py = K[1] if ndim >= 2 else np.zeros_like(px)
    pz = K[2] if ndim >= 3 else np.zeros_like(px)
    p2 = px**2 + py**2 + pz**2
    E = np.sqrt(mass**2 * c**4 + p2 * c**2)
    nrm = np.sqrt(2.0 * E * (E + mass * c**2))
    up = (E + mass * c**2) / nrm
    dn = c * (px + 1j * py) / nrm
    if ncomp == 2:
        return np.stack([up.astype(np.complex128), dn])
    return np.stack([up.astype(np.complex128), np.zeros_like(dn), (c * pz / nrm).astype(np.complex128), dn])


def dirac_packet(sizes, dx, kbar, sigma_p, ncomp, mass, c) -> np.ndarray:
    """psi0 = F^-1{ u_+(k) exp(-|k-kbar|^2/(4 sigma_p^2)) } (eq. 36/37 with an isotropic width), normalised."""
    K = kmesh(sizes, dx)
    g = np.exp(-sum((Ka - kb) ** 2 for Ka, kb in zip(K, kbar)) / (4.0 * sigma_p**2))
    spin = positive_energy_spinor(K, ncomp, mass, c)
    R0 = [n // 2 for n in sizes]
    # centre the packet at r = 0, which sits at index n/2 on the half-open grid
    shift = np.ones(sizes, dtype=np.complex128)
    for a, (Ka, n, d) in enumerate(zip(K, sizes, dx)):
        shift = shift * np.exp(-1j * Ka * (R0[a] * d))
    psi = np.stack([np.fft.ifftn(spin[s] * g * shift) for s in range(ncomp)])
    return normalise(psi, dx)


# ---------------------------------------------------------------------------
# the five configs; `sizes` overrides give the reduced parity cases
# ---------------------------------------------------------------------------

def config1(sizes=(4096,), nsteps=1000, noise=1e-3) -> Workload:
    """1D Schroedinger, harmonic well, coherent state (sigma=1, x0=5, p0=0) with 1e-3 phase noise (G9, G25)."""
    rng = np.random.default_rng(SEED0 + 1)
    n = sizes[0]
    dx = (400.0 / 4096.0,)  # x in [-200, 200) at n = 4096
    x = axis_r(n, dx[0])
    psi = np.pi ** (-0.25) * np.exp(-((x - 5.0) ** 2) / 2.0)
    xi = rng.uniform(-1.0, 1.0, size=n)
    psi = psi * np.exp(1j * noise * xi)
    psi = normalise(psi, dx)[None, :]
    return Workload("cfg1_schroedinger1d", tuple(sizes), dx, 0.01, 1, nsteps, psi, V=0.5 * x**2,
                    note="harmonic V=x^2/2, coherent state x0=5")


def config2(sizes=(2048, 2048), nsteps=500) -> Workload:
    """2D Schroedinger, soft-core Coulomb + dipole field along axis 0 (G22, G24, G26)."""
    rng = np.random.default_rng(SEED0 + 2)
    dx = (0.1, 0.1)
    dt = 0.02
    X, Y = mesh(sizes, dx)
    V = -1.0 / np.sqrt(X**2 + Y**2 + 1.0)
    L = min(n * d for n, d in zip(sizes, dx))
    span = min(5.0, L / 8.0)
    r0 = rng.uniform(-span, span, size=2)
    p0 = rng.uniform(-1.0, 1.0, size=2)
    psi = gaussian_packet(sizes, dx, r0, p0, 1.5)[None]
    avg = np.zeros((nsteps + 8, 2))
    avg[:, 0] = sinus_step_average(0.05, 0.057, dt, nsteps + 8)
    return Workload("cfg2_schroedinger2d", tuple(sizes), dx, dt, 1, nsteps, psi, V=V,
                    field_kind=FIELD_E, step_avg=avg, note="soft-core + x.E0 sin(wt), E0=0.05, w=0.057")


def config3(sizes=(256, 256, 256), nsteps=200) -> Workload:
    """3D Schroedinger, smooth random potential = sum of 32 Gaussians (G23)."""
    rng = np.random.default_rng(SEED0 + 3)
    dx = (0.2, 0.2, 0.2)
    axes = [axis_r(n, d) for n, d in zip(sizes, dx)]
    L = [n * d for n, d in zip(sizes, dx)]
    amp = rng.uniform(-1.0, 1.0, size=32)
    wid = rng.uniform(0.5, 2.0, size=32)
    cen = np.stack([rng.uniform(-La / 4, La / 4, size=32) for La in L], axis=1)
    V = np.zeros(sizes)
    for a, w, r0 in zip(amp, wid, cen):
        # separable Gaussian: outer product of three 1D factors
        g = [np.exp(-((ax - c0) ** 2) / (2.0 * w**2)) for ax, c0 in zip(axes, r0)]
        V += a * g[0][:, None, None] * g[1][None, :, None] * g[2][None, None, :]
    p0 = rng.uniform(-1.0, 1.0, size=3)
    psi = gaussian_packet(sizes, dx, (0.0, 0.0, 0.0), p0, 2.0)[None]
    return Workload("cfg3_schroedinger3d", tuple(sizes), dx, 0.01, 1, nsteps, psi, V=V,
                    note="32 random Gaussians, centred packet sigma=2")


def config4(sizes=(1024, 1024), nsteps=200) -> Workload:
    """2D Dirac, 2 components, soft-core Z=1 (zeta=0.791), A(t)=5 sin(t) along axis 0 in the kinetic factor (G16, G27)."""
    rng = np.random.default_rng(SEED0 + 4)
    dx = (0.1, 0.1)
    dt = 1e-4
    X, Y = mesh(sizes, dx)
    V = -1.0 / np.sqrt(X**2 + Y**2 + 0.791**2)
    kbar = rng.uniform(-5.0, 5.0, size=2)
    psi = dirac_packet(sizes, dx, kbar, 1.0, 2, 1.0, C_LIGHT)
    avg = np.zeros((nsteps + 8, 2))
    avg[:, 0] = sinus_step_average(5.0, 1.0, dt, nsteps + 8)
    return Workload("cfg4_dirac2d", tuple(sizes), dx, dt, 2, nsteps, psi, V=V,
                    field_kind=FIELD_A, step_avg=avg, note="soft-core zeta=0.791, A0=5, w=1")


def config5(sizes=(256, 256, 256), nsteps=100) -> Workload:
    """3D Dirac, 4 components, static soft-core Coulomb, no field."""
    rng = np.random.default_rng(SEED0 + 5)
    dx = (0.1, 0.1, 0.1)
    X, Y, Z = mesh(sizes, dx)
    V = -1.0 / np.sqrt(X**2 + Y**2 + Z**2 + 1.0)
    del X, Y, Z
    kbar = rng.uniform(-5.0, 5.0, size=3)
    psi = dirac_packet(sizes, dx, kbar, 1.0, 4, 1.0, C_LIGHT)
    return Workload("cfg5_dirac3d", tuple(sizes), dx, 1e-4, 4, nsteps, psi, V=V, note="soft-core zeta=1")


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def dirac1d(sizes=(1024,), nsteps=100, ncomp=2) -> Workload:
    """1D Dirac (eq. 17/35): positive-energy packet in a soft-core well, zeta=1.4133."""
    rng = np.random.default_rng(SEED0 + 6)
    dx = (0.1,)
    x = axis_r(sizes[0], dx[0])
    V = -1.0 / np.sqrt(x**2 + 1.4133**2)
    kbar = rng.uniform(-5.0, 5.0, size=1)
    psi = dirac_packet(sizes, dx, kbar, 1.0, ncomp, 1.0, C_LIGHT)
    return Workload("dirac1d", tuple(sizes), dx, 1e-4, ncomp, nsteps, psi, V=V)


def dirac2d4(sizes=(1024, 1024), nsteps=128) -> Workload:
    """2D Dirac with all FOUR components, the shape of the paper's own 2D code and benchmark (PAPER.md:115, 284, 310:
    "Gaussian wave packets in a harmonic potential"): harmonic well, positive-energy spin-up packet, no field."""
    rng = np.random.default_rng(SEED0 + 7)
    dx = (0.1, 0.1)
    X, Y = mesh(sizes, dx)
    V = 0.5 * (X**2 + Y**2)
    kbar = rng.uniform(-5.0, 5.0, size=2)
    psi = dirac_packet(sizes, dx, kbar, 1.0, 4, 1.0, C_LIGHT)
    return Workload("dirac2d_4comp", tuple(sizes), dx, 1e-4, 4, nsteps, psi, V=V, note="harmonic well, 4 components")


def dirac2d_magnetic(sizes=(1024, 1024), nsteps=128) -> Workload:
    """2D Dirac, 2 components, with a POSITION-DEPENDENT vector potential applied in position space as the paper does
    (eq. 18a, 188-198 eq. 26): homogeneous magnetic field B = 50 a.u. in the symmetric gauge
    A = (B/2)(-y, x), soft-core well, positive-energy packet.  extra["A"] holds A(r), shape (2, *sizes)."""
    rng = np.random.default_rng(SEED0 + 8)
    dx = (0.1, 0.1)
    X, Y = mesh(sizes, dx)
    V = -1.0 / np.sqrt(X**2 + Y**2 + 0.791**2)
    kbar = rng.uniform(-5.0, 5.0, size=2)
    psi = dirac_packet(sizes, dx, kbar, 1.0, 2, 1.0, C_LIGHT)
    B = 50.0
    A = np.stack([-0.5 * B * Y, 0.5 * B * X])
    return Workload("dirac2d_magnetic", tuple(sizes), dx, 1e-4, 2, nsteps, psi, V=V, note="B = 50 a.u., symmetric gauge", extra={"A": A})


# ---------------------------------------------------------------------------------------------------------
# the laser pulse of PAPER.md:400-412 (eq. 46a-c): inputs for the position-space vector-potential factor
# ---------------------------------------------------------------------------------------------------------
def pulse_envelope(eta, j: int, l: int):
    """f_{j,l}(eta) of eq. 46c: j half cycles in all, linear turn-on and turn-off ramps of l half cycles each, plateau
    in between, zero outside -j pi <= eta <= 0."""
    eta = np.asarray(eta, dtype=np.float64)
    x = eta / np.pi
    f = np.zeros_like(eta)
    on = (x >= -j) & (x <= -j + l)
    flat = (x > -j + l) & (x < -l)
    off = (x >= -l) & (x <= 0)
    f[on] = (eta[on] + j * np.pi) / (l * np.pi)
    f[flat] = 1.0
    f[off] = -eta[off] / (l * np.pi)
    return f


def pulse_field(eta, E0: float, j: int, l: int):
    """E(eta) = E0 sin(eta) f_{j,l}(eta), eta = k.x - omega t (eq. 46a); B = E / c (eq. 46b)."""
    return E0 * np.sin(eta) * pulse_envelope(eta, j, l)


def pulse_vector_potential(eta, E0: float, omega: float, j: int, l: int):
    """A(eta) with E = -dA/dt = omega dA/deta and A = 0 ahead of the pulse (eta >= 0): A(eta) = -(1/omega) int_eta^0 E.
    Closed form on each piece of the envelope: int sin(e) (a e + b) de = -(a e + b) cos(e) + a sin(e)."""
    eta = np.asarray(eta, dtype=np.float64)

    def F(e, a, b):  # antiderivative of sin(e) (a e + b)
        return -(a * e + b) * np.cos(e) + a * np.sin(e)

    pieces = [(-j * np.pi, (-j + l) * np.pi, 1.0 / (l * np.pi), j / l), ((-j + l) * np.pi, -l * np.pi, 0.0, 1.0),
              (-l * np.pi, 0.0, -1.0 / (l * np.pi), 0.0)]
    total = np.zeros_like(eta)  # int_eta^0 sin f
    for lo, hi, a, b in pieces:
        if hi <= lo:
            continue
        e0 = np.clip(eta, lo, hi)
        total += F(hi, a, b) - F(e0, a, b)
    return -(E0 / omega) * total


def pulse_step_average(x, t: float, tau: float, E0: float, omega: float, j: int, l: int, kx: float):
    """(1/tau) int_t^{t+tau} A(kx x - omega t') dt' by 8-point Gauss-Legendre quadrature (reading G12: the library and the
    oracle are handed the same step average)."""
    nodes, weights = np.polynomial.legendre.leggauss(8)
    acc = np.zeros_like(np.asarray(x, dtype=np.float64))
    for xi, wi in zip(nodes, weights):
        tt = t + 0.5 * tau * (xi + 1.0)
        acc += 0.5 * wi * pulse_vector_potential(kx * x - omega * tt, E0, omega, j, l)
    return acc


def random_state(sizes, ncomp, seed, dx=None) -> np.ndarray:
    """Unstructured complex Gaussian noise, normalised: the harshest parity input (all k populated)."""
    rng = np.random.default_rng(seed)
    shape = (ncomp,) + tuple(sizes)
    psi = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    return normalise(psi, dx if dx is not None else (1.0,) * len(sizes))
