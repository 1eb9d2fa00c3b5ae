"""Randomised GPU parity: seeded random lattices (1D/2D/3D, every axis length from 16 to 1024, Schroedinger and Dirac, both
precisions), random fields and random settings of the tuning knobs (tile widths, groups, buffers of the tile pool, tile
order, thread count, potential representation), a few steps each, against the CPU oracle.  The knobs must never change
the result; a knob value that does not fit a shape must fall back, not fail."""
import numpy as np
import pytest

import oracle
import paper_1012_3911_b200 as sso
import workloads as wl

pytestmark = pytest.mark.gpu
TOL = {sso.C128: 1e-12, sso.C64: 2e-5}


@pytest.fixture(scope="module")
def torch():
    import torch as t

    assert t.cuda.is_available()
    t.cuda.set_device(0)
    sso.lib()
    return t


def random_case(rng):
    nd = int(rng.integers(1, 4))
    lgs = [int(rng.integers(4, 14 if nd < 3 else 9)) for _ in range(nd)]
    while sum(lgs) > 18:  # at most 2^18 lattice points: the oracle stays fast
        lgs[int(np.argmax(lgs))] -= 1
    sizes = [1 << lg for lg in lgs]
    ncomp = int(rng.choice([1, 1, 2, 4])) if nd < 3 else int(rng.choice([1, 1, 4]))
    if nd == 1 and ncomp * sizes[0] > 8192:
        ncomp = 1
    apos = ncomp > 1 and rng.random() < 0.25  # the position-space vector-potential factor
    prec = sso.C128 if rng.random() < 0.7 else sso.C64
    kinds = [sso.FIELD_NONE, sso.FIELD_E, sso.FIELD_A]
    kind = int(rng.choice(kinds))
    opts = []
    if rng.random() < 0.7:
        for opt, values in ((sso.OPT_LINES_PER_TILE_CONTIG, [0, 1, 2, 4, 8]), (sso.OPT_LINES_PER_TILE_STRIDED, [0, 1, 2, 4, 8]),
                            (sso.OPT_LINES_PER_TILE_MIDDLE, [0, 2, 4, 8, 16]), (sso.OPT_GROUPS_PER_CTA, [0, 1, 2, 3, 5]),
                            (sso.OPT_RING_BUFFERS, [0, 1, 2, 3, 5, 7, 12]), (sso.OPT_TILE_ORDER, [0, 1, 2, 6, 16]),
                            (sso.OPT_THREADS_PER_CTA, [0, 384, 512]), (sso.OPT_STRIDED_RING, [0, 0, 2]),
                            (sso.OPT_POTENTIAL_PHASE, [0, 0, 1]), (sso.OPT_DIRAC_TABLE, [0, 1]), (sso.OPT_CLUSTER_1D, [0, 1, 4, 8])):
            if rng.random() < 0.4:
                opts.append((opt, int(rng.choice(values))))
    return nd, tuple(sizes), ncomp, prec, kind, opts, apos


@pytest.mark.parametrize("seed", range(int(__import__("os").environ.get("SSO_FUZZ_SEEDS", "96"))))
def test_random_lattice_fields_and_knobs(torch, seed):
    rng = np.random.default_rng(77000 + seed)
    nd, sizes, ncomp, prec, kind, opts, apos = random_case(rng)
    dx = tuple(float(x) for x in rng.uniform(0.05, 0.3, size=nd))
    tau = 0.01 if ncomp == 1 else 1e-4
    nsteps = int(rng.integers(1, 5))
    V = rng.uniform(-1.0, 1.0, size=sizes) * (1.0 if ncomp == 1 else 100.0)
    psi0 = wl.random_state(sizes, ncomp, 1000 + seed, dx)
    cdt = np.complex128 if prec == sso.C128 else np.complex64
    psi0 = psi0.astype(cdt)
    avg = rng.uniform(-0.3, 0.3, size=(nsteps, nd)) * (1.0 if kind == sso.FIELD_E else 3.0)
    p = sso.Plan(sizes, dx, tau, ncomp, prec)
    o = oracle.Solver(sizes, dx, tau, ncomp)
    for opt, val in opts:
        p.set_option(opt, val)
    p.set_potential(V)
    o.set_potential(V)
    if kind != sso.FIELD_NONE:
        p.set_field(kind, np.ascontiguousarray(avg))
        o.set_field(kind, avg)
    if apos:
        A = rng.uniform(-30.0, 30.0, size=(nd,) + tuple(sizes))
        p.set_vector_potential(np.ascontiguousarray(A))
        o.set_vector_potential(A)
    psi = torch.from_numpy(psi0).cuda()
    ref = psi.clone()
    label = (nd, sizes, ncomp, prec, kind, opts, apos, nsteps)
    nrm, chi, r = p.step_observe(psi, nsteps, ref)
    torch.cuda.synchronize()
    want = o.step(psi0.astype(np.complex128), nsteps)
    got = psi.cpu().numpy()
    err = float(np.linalg.norm((got - want).ravel()) / np.linalg.norm(want.ravel()))
    assert err <= TOL[prec], (label, err)
    assert abs(nrm - o.norm(want)) <= 100 * TOL[prec], label
    assert abs(chi - o.overlap(psi0.astype(np.complex128), want)) <= 100 * TOL[prec], label
    np.testing.assert_allclose(r, o.expect_r(want), atol=1000 * TOL[prec] * max(n * d for n, d in zip(sizes, dx)), err_msg=str(label))
    p.destroy()
