"""GPU parity: the CUDA path (through the C ABI of include/sso.h) against the CPU oracle, element by element,
on the same seeded inputs (workloads.py).  Metric and bars (BASELINE.json north_star, G19):
relative L2 error over all components  <= 1e-11 (complex128) / <= 2e-5 (complex64)  after 100 steps.
For complex64 the oracle starts from the complex64-rounded psi0 promoted to double.
"""
import ctypes

import numpy as np
import pytest

import oracle
import paper_1012_3911_b200 as sso
import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {sso.C128: 1e-11, sso.C64: 2e-5}


@pytest.fixture(scope="module")
def torch():
    import torch as t

    assert t.cuda.is_available()
    t.cuda.set_device(0)
    sso.lib()  # fails loudly if libsso.so is missing: there is no fallback
    return t


def rel_l2(got, want):
    return float(np.linalg.norm((got - want).ravel()) / np.linalg.norm(want.ravel()))


def make_plan(w, prec=sso.C128):
    p = sso.Plan(w.sizes, w.dx, w.dt, w.ncomp, prec)
    p.set_constants(w.mass, w.c, w.charge)
    p.set_potential(w.V)
    if w.field_kind:
        p.set_field(w.field_kind, np.ascontiguousarray(w.step_avg))
    return p


def make_oracle(w):
    o = oracle.Solver(w.sizes, w.dx, w.dt, w.ncomp, w.mass, w.c, w.charge)
    o.set_potential(w.V)
    if w.field_kind:
        o.set_field(w.field_kind, w.step_avg)
    return o


def start_state(w, prec):
    return w.psi0.astype(np.complex128 if prec == sso.C128 else np.complex64)


def gpu_steps(torch, w, nsteps, prec=sso.C128, chunks=None, psi0=None, options=()):
    p = make_plan(w, prec)
    for o, v in options:
        p.set_option(o, v)
    if options:
        p.set_potential(w.V)
    psi = torch.from_numpy(start_state(w, prec) if psi0 is None else psi0).cuda()
    for c in chunks or [nsteps]:
        p.step(psi, c)
    torch.cuda.synchronize()
    nrm = p.norm(psi)
    p.destroy()
    return psi.cpu().numpy(), nrm


def oracle_steps(w, nsteps, prec=sso.C128, psi0=None):
    o = make_oracle(w)
    s = (start_state(w, prec) if psi0 is None else psi0).astype(np.complex128)
    return o.step(s, nsteps)


# ---------------------------------------------------------------------------------------------------------
# 100-step parity on reduced grids of every config: several tiles per pass, non-square shapes
# ---------------------------------------------------------------------------------------------------------
REDUCED = [
    ("cfg1", lambda: wl.config1(sizes=(1024,), nsteps=100), sso.C128),
    ("cfg2a", lambda: wl.config2(sizes=(256, 512), nsteps=100), sso.C128),
    ("cfg2b", lambda: wl.config2(sizes=(256, 512), nsteps=100), sso.C64),
    ("cfg2a_tall", lambda: wl.config2(sizes=(1024, 64), nsteps=100), sso.C128),
    ("cfg3", lambda: wl.config3(sizes=(32, 64, 128), nsteps=100), sso.C128),
    ("cfg4", lambda: wl.config4(sizes=(256, 128), nsteps=100), sso.C128),
    ("cfg5", lambda: wl.config5(sizes=(32, 16, 64), nsteps=100), sso.C128),
    ("dirac1d_c2", lambda: wl.dirac1d(sizes=(512,), nsteps=100, ncomp=2), sso.C128),
    ("dirac1d_c4", lambda: wl.dirac1d(sizes=(512,), nsteps=100, ncomp=4), sso.C128),
    ("cfg4_c64", lambda: wl.config4(sizes=(128, 128), nsteps=100), sso.C64),
    ("cfg3_c64", lambda: wl.config3(sizes=(32, 32, 64), nsteps=100), sso.C64),
]


@pytest.mark.parametrize("name,make,prec", REDUCED, ids=[r[0] for r in REDUCED])
def test_parity_100_steps_reduced(torch, name, make, prec):
    w = make()
    got, nrm = gpu_steps(torch, w, 100, prec)
    want = oracle_steps(w, 100, prec)
    err = rel_l2(got.astype(np.complex128), want)
    assert err <= TOL[prec], (name, err)
    # element by element as well: no single point may be off by more than the bar times the peak amplitude
    peak = np.abs(want).max()
    assert np.abs(got - want).max() <= 5 * TOL[prec] * peak
    assert abs(nrm - 1.0) < (1e-11 if prec == sso.C128 else 1e-4)


def test_config1_full_size_100_and_1000_steps(torch):
    """BASELINE config 1 at its full size, parity recorded at 100 and 1000 steps."""
    w = wl.config1()
    o = make_oracle(w)
    p = make_plan(w)
    psi = torch.from_numpy(w.psi0.copy()).cuda()
    ref = w.psi0
    for upto, n in ((100, 100), (1000, 900)):
        p.step(psi, n)
        ref = o.step(ref, n)
        torch.cuda.synchronize()
        err = rel_l2(psi.cpu().numpy(), ref)
        assert err <= 1e-11, (upto, err)
    assert p.get_time_index() == 1000
    p.destroy()


def test_random_state_all_axis_lengths(torch):
    """Every supported line length, noise input (all k populated), contiguous and strided passes."""
    for n in (16, 32, 64, 128, 256, 512, 1024, 2048, 4096):
        for sizes in ((n,), (n, 16), (16, n)):
            dx = (0.1,) * len(sizes)
            psi0 = wl.random_state(sizes, 1, seed=n + len(sizes), dx=dx)
            rng = np.random.default_rng(n)
            V = rng.uniform(-1, 1, size=sizes)
            w = wl.Workload("rand", sizes, dx, 0.01, 1, 3, psi0, V=V)
            got, _ = gpu_steps(torch, w, 3)
            want = oracle_steps(w, 3)
            assert rel_l2(got, want) <= 1e-13, (sizes, rel_l2(got, want))


def test_random_state_all_axis_lengths_complex64(torch):
    """The complex64 instantiation of every line length: a 1D line, contiguous and strided passes, noise input."""
    for n in (16, 32, 64, 128, 256, 512, 1024, 2048, 4096):
        for sizes in ((n,), (n, 16), (16, n)):
            dx = (0.1,) * len(sizes)
            psi0 = wl.random_state(sizes, 1, seed=n + len(sizes), dx=dx).astype(np.complex64)
            rng = np.random.default_rng(n)
            V = rng.uniform(-1, 1, size=sizes)
            w = wl.Workload("rand", sizes, dx, 0.01, 1, 3, psi0, V=V)
            got, _ = gpu_steps(torch, w, 3, sso.C64, psi0=psi0)
            want = oracle_steps(w, 3, psi0=psi0)
            err = rel_l2(got.astype(np.complex128), want)
            assert err <= 2e-6, (sizes, err)


def test_complex64_dirac_1d_and_3d(torch):
    """complex64 Dirac: a 1D line (2 and 4 components) and a 3D lattice with A(t), noise input."""
    for ncomp, sizes in ((2, (512,)), (4, (256,)), (4, (32, 16, 64)), (2, (64, 128))):
        dx = (0.05,) * len(sizes)
        psi0 = wl.random_state(sizes, ncomp, seed=17 * ncomp + len(sizes), dx=dx).astype(np.complex64)
        rng = np.random.default_rng(ncomp + 40)
        V = rng.uniform(-50, 50, size=sizes)
        avg = rng.uniform(-3, 3, size=(8, len(sizes)))
        w = wl.Workload("rand", sizes, dx, 2e-4, ncomp, 4, psi0, V=V, field_kind=wl.FIELD_A, step_avg=avg)
        got, _ = gpu_steps(torch, w, 4, sso.C64, psi0=psi0)
        want = oracle_steps(w, 4, psi0=psi0)
        err = rel_l2(got.astype(np.complex128), want)
        assert err <= 2e-6, (ncomp, sizes, err)


def test_random_state_3d_and_dirac(torch):
    for ncomp, sizes in ((1, (16, 32, 64)), (4, (64, 16, 32)), (2, (128, 64)), (4, (64, 128)), (4, (2048,)), (2, (4096,))):
        dx = (0.05,) * len(sizes)
        psi0 = wl.random_state(sizes, ncomp, seed=7 * ncomp + len(sizes), dx=dx)
        rng = np.random.default_rng(ncomp)
        V = rng.uniform(-50, 50, size=sizes)
        nd = len(sizes)
        avg = rng.uniform(-3, 3, size=(8, nd))
        w = wl.Workload("rand", sizes, dx, 2e-4, ncomp, 4, psi0, V=V, field_kind=wl.FIELD_A, step_avg=avg)
        got, _ = gpu_steps(torch, w, 4)
        want = oracle_steps(w, 4)
        assert rel_l2(got, want) <= 1e-13, (ncomp, sizes, rel_l2(got, want))


def test_position_space_vector_potential(torch):
    """The paper's own Dirac interaction factor (eq. 18a, 23-26, 34): A(r) applied in position space, merged between
    steps, together with V, with and without a homogeneous A(t) in the kinetic factor, all lattice dimensions."""
    cases = [(2, (256,), None), (4, (128,), wl.FIELD_A), (2, (64, 128), wl.FIELD_A), (4, (32, 64), None), (4, (16, 32, 32), None)]
    for ncomp, sizes, kind in cases:
        nd = len(sizes)
        dx = (0.1,) * nd
        rng = np.random.default_rng(100 * ncomp + nd)
        psi0 = wl.random_state(sizes, ncomp, seed=5 * ncomp + nd, dx=dx)
        R = wl.mesh(sizes, dx)
        A = np.stack([40.0 * np.sin(0.7 * R[(a + 1) % nd] + a) + rng.uniform(-5, 5) for a in range(nd)])  # smooth, a.u.
        w = wl.Workload("apos", sizes, dx, 1e-4, ncomp, 6, psi0, V=rng.uniform(-2000, 2000, size=sizes),
                        field_kind=kind or wl.FIELD_NONE, step_avg=rng.uniform(-3, 3, size=(8, nd)) if kind else None)
        for prec, tol in ((sso.C128, 1e-13), (sso.C64, 2e-6)):
            p = make_plan(w, prec)
            p.set_vector_potential(A)
            s0 = psi0.astype(np.complex128 if prec == sso.C128 else np.complex64)
            psi = torch.from_numpy(s0).cuda()
            p.step(psi, 2)
            p.step(psi, 4)
            torch.cuda.synchronize()
            o = make_oracle(w)
            o.set_vector_potential(A)
            want = o.step(s0.astype(np.complex128), 6)
            err = rel_l2(psi.cpu().numpy().astype(np.complex128), want)
            assert err <= tol, (ncomp, sizes, kind, prec, err)
            assert p.launch_count(3) > 0
            # switching the factor off again gives the plain step
            p.set_vector_potential(None)
            p.set_time_index(0)
            psi = torch.from_numpy(s0).cuda()
            p.step(psi, 2)
            torch.cuda.synchronize()
            assert rel_l2(psi.cpu().numpy().astype(np.complex128), oracle_steps(w, 2, psi0=s0)) <= tol
            p.destroy()
    with pytest.raises(sso.SsoError) as e:
        sso.Plan((64,), (0.1,), 0.01, 1).set_vector_potential(np.ones((1, 64)))
    assert e.value.code == sso.ERR_UNSUPPORTED
    # a host array with a NaN or an Inf is refused like the rows of sso_set_field (it would end up in psi otherwise)
    p = sso.Plan((32, 32), (0.1, 0.1), 0.01, 2)
    for bad in (np.nan, np.inf):
        A = np.zeros((2, 32, 32))
        A[1, 7, 5] = bad
        with pytest.raises(sso.SsoError) as e:
            p.set_vector_potential(A)
        assert e.value.code == sso.ERR_INVALID
    p.destroy()


def test_field_e_on_every_axis(torch):
    """Length-gauge field with components along all axes (the last axis uses the per-step line phase table)."""
    for sizes in ((64,), (32, 64), (16, 32, 64)):
        nd = len(sizes)
        dx = (0.2,) * nd
        rng = np.random.default_rng(nd)
        psi0 = wl.random_state(sizes, 1, seed=nd, dx=dx)
        w = wl.Workload("e", sizes, dx, 0.01, 1, 5, psi0, V=rng.uniform(-1, 1, size=sizes), field_kind=wl.FIELD_E,
                        step_avg=rng.uniform(-0.5, 0.5, size=(6, nd)))
        got, _ = gpu_steps(torch, w, 5)
        assert rel_l2(got, oracle_steps(w, 5)) <= 1e-13
        got2, _ = gpu_steps(torch, w, 5, chunks=[2, 1, 2])
        assert rel_l2(got2, got) <= 1e-14  # merged potential phases equal unmerged ones up to rounding


def test_schroedinger_with_vector_potential(torch):
    """SSO_FIELD_A for ncomp = 1: kinetic tables rebuilt per step (eq. 13 with the shift, reading G17)."""
    for sizes in ((128,), (32, 64)):
        nd = len(sizes)
        dx = (0.1,) * nd
        rng = np.random.default_rng(3 + nd)
        psi0 = wl.random_state(sizes, 1, seed=11 + nd, dx=dx)
        w = wl.Workload("a", sizes, dx, 0.01, 1, 4, psi0, V=rng.uniform(-1, 1, size=sizes), field_kind=wl.FIELD_A,
                        step_avg=rng.uniform(-2, 2, size=(4, nd)))
        got, _ = gpu_steps(torch, w, 4)
        assert rel_l2(got, oracle_steps(w, 4)) <= 1e-13


# ---------------------------------------------------------------------------------------------------------
# every pipeline variant computes the same step: direct kernel, forced/disabled TMA ring, group and buffer counts
# ---------------------------------------------------------------------------------------------------------
OPT_TL_STRIDED, OPT_GROUPS, OPT_RING, OPT_THREADS, OPT_SRING, OPT_DIRAC_TABLE = 2, 4, 5, 6, 7, 8
VARIANTS = [
    ("direct_strided", [(OPT_SRING, 2)]),
    ("ring_forced", [(OPT_SRING, 1)]),
    ("ring_rows32B", [(OPT_SRING, 1), (OPT_TL_STRIDED, 2)]),
    ("one_group", [(OPT_GROUPS, 1)]),
    ("two_groups_single_buffer", [(OPT_GROUPS, 2), (OPT_RING, 1)]),
    ("three_buffers", [(OPT_GROUPS, 2), (OPT_RING, 3)]),
    ("cta384", [(OPT_THREADS, 384)]),
    ("cta512", [(OPT_THREADS, 512)]),
    ("dirac_table", [(OPT_DIRAC_TABLE, 1)]),
    ("rows64B_one_spare_buffer", [(OPT_TL_STRIDED, 4), (OPT_GROUPS, 1), (OPT_RING, 2)]),
    ("many_buffers_one_group", [(OPT_GROUPS, 1), (OPT_RING, 6)]),
]


@pytest.mark.parametrize("name,options", VARIANTS, ids=[v[0] for v in VARIANTS])
def test_pipeline_variants_agree_with_oracle(torch, name, options):
    cases = [
        wl.config2(sizes=(256, 256), nsteps=6),        # Schroedinger 2D with E(t)
        wl.config3(sizes=(64, 128, 64), nsteps=4),     # 3D: middle-axis DIF/DIT passes
        wl.config4(sizes=(128, 256), nsteps=4),        # Dirac 2 components with A(t)
        wl.config5(sizes=(64, 32, 64), nsteps=3),      # Dirac 4 components
    ]
    for w in cases:
        n = w.nsteps
        got, nrm = gpu_steps(torch, w, n, options=options)
        want = oracle_steps(w, n)
        assert rel_l2(got, want) <= 1e-13, (name, w.name, rel_l2(got, want))
        assert abs(nrm - 1.0) < 1e-12


def test_many_tiles_per_group_large_lattice(torch):
    """A lattice large enough that every group of the ring refills its buffers many times (the failure mode of a
    ring shared between groups showed only beyond 128 MB): F then F^-1 along every axis must return N psi."""
    sizes = (128, 256, 256)
    p = sso.Plan(sizes, (0.1, 0.1, 0.1), 0.01, 1, sso.C128)   # V = 0, no field: the step is F^-1 K F
    g = torch.Generator(device="cuda")
    g.manual_seed(5)
    psi0 = torch.randn(sizes, dtype=torch.complex128, device="cuda", generator=g)
    psi = psi0.clone()
    p.step(psi, 1)
    p2 = sso.Plan(sizes, (0.1, 0.1, 0.1), -0.01, 1, sso.C128)
    p2.step(psi, 1)
    torch.cuda.synchronize()
    err = float((psi - psi0).abs().max() / psi0.abs().max())
    assert err < 1e-13, err
    p.destroy()
    p2.destroy()


LONG_AXIS = [
    ("2d-8192x32-c128", (8192, 32), sso.C128), ("2d-32x8192-c128", (32, 8192), sso.C128),
    ("2d-8192x64-c64", (8192, 64), sso.C64), ("2d-16x8192-c64", (16, 8192), sso.C64),
    ("3d-16x8192x16-c128", (16, 8192, 16), sso.C128),
]


@pytest.mark.parametrize("name,sizes,prec", LONG_AXIS, ids=[c[0] for c in LONG_AXIS])
def test_axis_of_8192_points(torch, name, sizes, prec):
    """SSO_MAX_AXIS = 8192: the longest line one CTA holds (512 threads x 16 points; the complex128 kernels read its
    twiddles from global memory).  Schroedinger with a field on the long axis, unstructured noise, 6 steps."""
    nd = len(sizes)
    rng = np.random.default_rng(8192 + nd + sizes[0])
    w = wl.config2(sizes=sizes[:2], nsteps=6) if nd == 2 else wl.config3(sizes=sizes, nsteps=6)
    psi0 = wl.random_state(sizes, 1, 8192, w.dx)
    avg = np.zeros((6, nd))
    avg[:, int(np.argmax(sizes))] = rng.uniform(-0.05, 0.05, size=6)
    w.field_kind, w.step_avg = sso.FIELD_E, avg
    got, nrm = gpu_steps(torch, w, 6, prec, psi0=psi0.astype(np.complex128 if prec == sso.C128 else np.complex64))
    want = oracle_steps(w, 6, prec, psi0=psi0.astype(np.complex128 if prec == sso.C128 else np.complex64))
    assert rel_l2(got, want) <= TOL[prec] * 0.1
    assert abs(nrm - 1.0) < (1e-11 if prec == sso.C128 else 1e-4)


LONG_DIRAC = [
    ("2d-4096x16-4comp-c128", 4, (4096, 16), sso.C128, False), ("2d-8192x16-2comp-c128", 2, (8192, 16), sso.C128, True),
    ("3d-4096x16x16-4comp-c64", 4, (4096, 16, 16), sso.C64, False), ("2d-2048x32-4comp-c128", 4, (2048, 32), sso.C128, True),
]


@pytest.mark.parametrize("name,ncomp,sizes,prec,field", LONG_DIRAC, ids=[c[0] for c in LONG_DIRAC])
def test_dirac_lines_longer_than_one_cta_holds(torch, name, ncomp, sizes, prec, field):
    """ncomp * n_0 > 8192: the components of a k point no longer meet in one CTA; the kinetic sandwich runs as
    transform, pointwise Dirac kernel, transform.  (The last case, 4 x 2048, is the longest that still runs fused.)"""
    nd = len(sizes)
    rng = np.random.default_rng(4096 + ncomp + nd)
    dx = (0.1,) * nd
    grids = np.meshgrid(*[wl.axis_r(n, d) for n, d in zip(sizes, dx)], indexing="ij")
    V = -1.0 / np.sqrt(sum(g * g for g in grids) + 1.0)
    psi0 = wl.random_state(sizes, ncomp, 4096 + ncomp, dx)
    nsteps = 5
    w = wl.Workload(name, tuple(sizes), dx, 1e-4, ncomp, nsteps, psi0, V=V)
    if field:
        avg = np.zeros((nsteps, nd))
        avg[:, 0] = rng.uniform(-5.0, 5.0, size=nsteps)
        avg[:, nd - 1] = rng.uniform(-5.0, 5.0, size=nsteps)
        w.field_kind, w.step_avg = sso.FIELD_A, avg
    cdt = np.complex128 if prec == sso.C128 else np.complex64
    got, nrm = gpu_steps(torch, w, nsteps, prec, psi0=psi0.astype(cdt))
    want = oracle_steps(w, nsteps, prec, psi0=psi0.astype(cdt))
    assert rel_l2(got, want) <= TOL[prec] * 0.1
    assert abs(nrm - 1.0) < (1e-11 if prec == sso.C128 else 1e-4)


def test_free_packet_in_the_laser_pulse_of_equation_46(torch):
    """PAPER.md:400-412 (section V.3): a free 2D Dirac packet in a pulse travelling along x with E along y, the
    vector potential A_y(k x - omega t) of eq. 46 applied in position space (eq. 26) and replaced every step by its
    step average (sso_set_vector_potential); 2 and 4 components against the oracle."""
    sizes, dx, tau, nsteps = (256, 64), (0.05, 0.05), 2e-5, 12
    c, omega = wl.C_LIGHT, 2 * np.pi * wl.C_LIGHT / 8.0   # wavelength 8 a.u. so that the grid sees several half cycles
    E0, j, l = 3000.0, 8, 2
    X, Y = wl.mesh(sizes, dx)
    for ncomp in (2, 4):
        psi0 = wl.dirac_packet(sizes, dx, np.array([0.0, 0.0]), 2.0, ncomp, 1.0, c)
        p = sso.Plan(sizes, dx, tau, ncomp, sso.C128)
        o = oracle.Solver(sizes, dx, tau, ncomp)
        psi = torch.from_numpy(psi0).cuda()
        ref = psi0.copy()
        for n in range(nsteps):
            t = 4e-3 + n * tau  # the pulse front has reached the packet
            A = np.zeros((2,) + sizes)
            A[1] = wl.pulse_step_average(X, t, tau, E0, omega, j, l, omega / c)
            assert np.abs(A[1]).max() > 1.0
            p.set_vector_potential(np.ascontiguousarray(A))
            o.set_vector_potential(A)
            p.step(psi, 1)
            ref = o.step(ref, 1)
        torch.cuda.synchronize()
        got = psi.cpu().numpy()
        assert rel_l2(got, ref) <= 1e-12
        assert abs(p.norm(psi) - 1.0) < 1e-12
        assert rel_l2(got, psi0) > 1e-3  # the pulse did act on the packet
        p.destroy()
