"""GPU parity of the 1D Schroedinger steps on a thread-block cluster (sso_line1d_cluster.cuh: the line spread over
4 or 8 SMs, exchanges through distributed shared memory; SURVEY 8(f) NEXT-3 (i) and NEXT-4 "lines longer than one
CTA") against the CPU oracle, through the C ABI."""
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
    sso.lib()
    return t


def rel_l2(got, want):
    return float(np.linalg.norm((got - want).ravel()) / np.linalg.norm(want.ravel()))


def run_gpu(torch, w, nsteps, prec, cluster, chunks=None, field=None):
    p = sso.Plan(w.sizes, w.dx, w.dt, 1, prec)
    p.set_option(sso.OPT_CLUSTER_1D, cluster)
    p.set_potential(w.V)
    if field is not None:
        p.set_field(*field)
    psi0 = w.psi0.astype(np.complex128 if prec == sso.C128 else np.complex64)
    psi = torch.from_numpy(psi0).cuda()
    for c in chunks or [nsteps]:
        p.step(psi, c)
    torch.cuda.synchronize()
    nrm = p.norm(psi)
    p.destroy()
    return psi.cpu().numpy(), nrm, psi0


def run_oracle(w, nsteps, psi0, field=None):
    o = oracle.Solver(w.sizes, w.dx, w.dt, 1)
    o.set_potential(w.V)
    if field is not None:
        o.set_field(*field)
    return o.step(psi0.astype(np.complex128), nsteps)


CASES = [
    ("4096-cs8-c128", 4096, 8, sso.C128), ("4096-cs4-c128", 4096, 4, sso.C128), ("2048-cs4-c128", 2048, 4, sso.C128),
    ("8192-auto-c128", 8192, 0, sso.C128), ("16384-cs4-c128", 16384, 4, sso.C128), ("32768-auto-c128", 32768, 0, sso.C128),
    ("4096-cs8-c64", 4096, 8, sso.C64), ("32768-auto-c64", 32768, 0, sso.C64),
]


@pytest.mark.parametrize("name,n,cluster,prec", CASES, ids=[c[0] for c in CASES])
def test_cluster_line_100_steps_vs_oracle(torch, name, n, cluster, prec):
    """config 1 (harmonic well, coherent state with phase noise) on lattices of 2048 .. 32768 points, 100 steps."""
    w = wl.config1(sizes=(n,), nsteps=100)
    got, nrm, psi0 = run_gpu(torch, w, 100, prec, cluster)
    want = run_oracle(w, 100, psi0)
    err = rel_l2(got, want)
    assert err <= TOL[prec], err
    assert np.abs(got - want).max() <= 5 * TOL[prec] * np.abs(want).max()
    assert abs(nrm - 1.0) < (1e-11 if prec == sso.C128 else 1e-4)


def test_cluster_and_single_cta_agree_and_chunking(torch):
    w = wl.config1(sizes=(4096,), nsteps=64)
    a, _, _ = run_gpu(torch, w, 64, sso.C128, 8)
    b, _, _ = run_gpu(torch, w, 64, sso.C128, 1)
    c, _, _ = run_gpu(torch, w, 64, sso.C128, 8, chunks=[1, 30, 33])
    assert rel_l2(a, b) < 1e-13
    assert rel_l2(c, a) < 1e-13


def test_cluster_line_random_state_and_vector_potential(torch):
    """unstructured noise (all k populated) with SSO_FIELD_A: the kinetic table is rebuilt every step."""
    n, nsteps = 8192, 12
    rng = np.random.default_rng(8192)
    w = wl.config1(sizes=(n,), nsteps=nsteps)
    w.psi0 = wl.random_state((n,), 1, 77, w.dx)
    avg = rng.uniform(-2.0, 2.0, size=(nsteps, 1))
    got, nrm, psi0 = run_gpu(torch, w, nsteps, sso.C128, 0, field=(sso.FIELD_A, np.ascontiguousarray(avg)))
    want = run_oracle(w, nsteps, psi0, field=(oracle.FIELD_A, avg))
    assert rel_l2(got, want) <= 1e-12


def test_long_line_needs_the_cluster_path(torch):
    w = wl.config1(sizes=(16384,), nsteps=4)
    p = sso.Plan(w.sizes, w.dx, w.dt, 1, sso.C128)
    p.set_potential(w.V)
    psi = torch.from_numpy(w.psi0.astype(np.complex128)).cuda()
    p.set_option(sso.OPT_CLUSTER_1D, 1)  # off: no single CTA holds 16384 points
    with pytest.raises(sso.SsoError) as e:
        p.step(psi, 1)
    assert e.value.code == sso.ERR_UNSUPPORTED
    p.set_option(sso.OPT_CLUSTER_1D, 0)
    p.set_field(sso.FIELD_E, np.zeros((4, 1)))  # length-gauge field: not on the cluster path
    with pytest.raises(sso.SsoError) as e:
        p.step(psi, 1)
    assert e.value.code == sso.ERR_UNSUPPORTED
    p.destroy()


def test_8192_point_line_on_one_cta(torch):
    """8192 points are the most one CTA holds (512 threads x 16 points, twiddles read from global memory for
    complex128): with the cluster switched off, or with a length-gauge field, the direct kernel takes the line."""
    w = wl.config1(sizes=(8192,), nsteps=20)
    got, nrm, psi0 = run_gpu(torch, w, 20, sso.C128, 1)
    want = run_oracle(w, 20, psi0)
    assert rel_l2(got, want) <= 1e-12
    rng = np.random.default_rng(81)
    avg = rng.uniform(-0.2, 0.2, size=(6, 1))
    got, nrm, psi0 = run_gpu(torch, w, 6, sso.C64, 0, field=(sso.FIELD_E, np.ascontiguousarray(avg)))
    want = run_oracle(w, 6, psi0, field=(oracle.FIELD_E, avg))
    assert rel_l2(got, want) <= 2e-5


def test_first_call_can_be_captured(torch):
    """sso.h: sso_step only enqueues kernels from the first call on.  The tables of the cluster kernel (n = 4096 picks 8
    CTAs by default) are made by sso_plan_create / sso_set_option, so the very first sso_step of a plan, and the first
    one after the cluster choice changed, can sit inside a stream capture (cudaMalloc / cudaFree there would end it)."""
    w = wl.config1(sizes=(4096,), nsteps=6)
    want = run_oracle(w, 6, w.psi0)
    for cluster in (0, 4, 1):
        p = sso.Plan(w.sizes, w.dx, w.dt, 1, sso.C128)
        p.set_potential(w.V)
        p.set_option(sso.OPT_CLUSTER_1D, cluster)
        psi = torch.from_numpy(w.psi0.copy()).cuda()
        st = torch.cuda.Stream()
        st.wait_stream(torch.cuda.current_stream())
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            p.step(psi, 3, stream=torch.cuda.current_stream())  # no warm-up call before the capture
        g.replay()
        g.replay()
        torch.cuda.synchronize()
        assert rel_l2(psi.cpu().numpy(), want) < TOL[sso.C128], cluster
        p.destroy()


def test_momentum_of_a_long_line_is_refused_up_front(torch):
    """sso_expect_momentum has no transform beyond 8192 points: SSO_ERR_UNSUPPORTED, stated in sso.h, before any work."""
    w = wl.config1(sizes=(16384,), nsteps=1)
    p = sso.Plan(w.sizes, w.dx, w.dt, 1, sso.C128)
    psi = torch.from_numpy(w.psi0.copy()).cuda()
    with pytest.raises(sso.SsoError) as ei:
        p.expect_momentum(psi)
    assert ei.value.code == sso.ERR_UNSUPPORTED
    assert abs(p.norm(psi) - 1.0) < 1e-12  # the plan is still usable
    p.destroy()
