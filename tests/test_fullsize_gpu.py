"""BASELINE.json's configs at their FULL sizes, in the launch configuration bench.py times (default options):
a few oracle steps element by element where the oracle finishes in seconds, one-by-one sampled outputs
through the O(N) definition sum, and the size-independent properties (unitarity, reversibility).  Plus the
boundary's edge cases on the GPU.
"""
import ctypes

import numpy as np
import pytest

import oracle
import paper_1012_3911_b200 as sso
import workloads as wl
from test_parity_gpu import TOL, gpu_steps, make_oracle, make_plan, oracle_steps, rel_l2, start_state, torch  # noqa: F401

pytestmark = pytest.mark.gpu

FULL = [
    ("cfg2a", lambda: wl.config2(nsteps=8), sso.C128, 3),
    ("cfg2b", lambda: wl.config2(nsteps=8), sso.C64, 3),
    ("cfg4", lambda: wl.config4(nsteps=8), sso.C128, 3),
    ("cfg3", lambda: wl.config3(nsteps=4), sso.C128, 2),
    ("cfg5", lambda: wl.config5(nsteps=2), sso.C128, 1),
]


@pytest.mark.parametrize("name,make,prec,nsteps", FULL, ids=[f[0] for f in FULL])
def test_full_size_first_steps_and_samples(torch, name, make, prec, nsteps):
    w = make()
    got, nrm = gpu_steps(torch, w, nsteps, prec)
    want = oracle_steps(w, nsteps, prec)
    err = rel_l2(got.astype(np.complex128), want)
    assert err <= TOL[prec] * 0.1, (name, err)
    assert abs(nrm - 1.0) < (1e-12 if prec == sso.C128 else 1e-5)
    # sampled outputs of step `nsteps`, each computed on its own from the definition (O(N) sum per sample):
    # oracle state after nsteps-1 steps -> V/2, forward DFT -> K -> one inverse-DFT sum + V/2 per sample
    o = make_oracle(w)
    prev = o.step(start_state(w, prec).astype(np.complex128), nsteps - 1) if nsteps > 1 else start_state(w, prec).astype(np.complex128)
    psik = o.half_step_to_k(prev, nsteps - 1)
    rng = np.random.default_rng(99)
    centre = int(np.ravel_multi_index([n // 2 for n in w.sizes], w.sizes))
    idx = [centre, 0, w.npoints - 1] + [int(i) for i in rng.integers(0, w.npoints, size=5)]
    flat = got.reshape(w.ncomp, -1)
    scale = np.abs(want).max()
    for i in idx:
        s = o.inverse_sample(psik, nsteps - 1, i)
        assert np.abs(flat[:, i] - s).max() <= TOL[prec] * scale, (name, i)


FULL100 = [
    ("cfg2a", lambda: wl.config2(nsteps=100), sso.C128),
    ("cfg2b", lambda: wl.config2(nsteps=100), sso.C64),
    ("cfg4", lambda: wl.config4(nsteps=100), sso.C128),
    ("cfg3", lambda: wl.config3(nsteps=100), sso.C128),
    ("cfg5", lambda: wl.config5(nsteps=100), sso.C128),
]


@pytest.mark.parametrize("name,make,prec", FULL100, ids=[f[0] for f in FULL100])
def test_full_size_100_steps(torch, name, make, prec):
    """north_star's bar as stated: relative L2 error <= 1e-11 (complex128) / 2e-5 (complex64) after 100 steps, at
    BASELINE.json's full sizes, default options (the launch configuration bench.py times), element-wise bound too.
    The oracle needs about 4 / 2 / 16 / 110 s for configs 2 / 4 / 3 / 5 on 16 host cores."""
    w = make()
    got, nrm = gpu_steps(torch, w, 100, prec)
    want = oracle_steps(w, 100, prec)
    err = rel_l2(got.astype(np.complex128), want)
    assert err <= TOL[prec], (name, err)
    peak = np.abs(want).max()
    assert np.abs(got - want).max() <= 5 * TOL[prec] * peak, name
    assert abs(nrm - 1.0) < (1e-11 if prec == sso.C128 else 1e-4)


@pytest.mark.parametrize("cfg,nsteps", [(2, 300), (3, 80), (5, 24)])
def test_full_size_runs_are_bitwise_reproducible(torch, cfg, nsteps):
    """Many tiles per ring buffer, many steps, twice: the two results must be bit-identical.  A buffer handed back to
    the copy engine before every thread is done with it (the cross-proxy ordering the refill relies on) shows up as
    run-to-run differences long before it shows up as a parity failure."""
    w = wl.CONFIGS[cfg](nsteps=nsteps)
    a, _ = gpu_steps(torch, w, nsteps)
    b, _ = gpu_steps(torch, w, nsteps)
    assert np.array_equal(a.view(np.float64), b.view(np.float64))


@pytest.mark.parametrize("cfg,prec", [(2, sso.C128), (2, sso.C64), (3, sso.C128), (4, sso.C128), (5, sso.C128)])
def test_full_size_unitarity_and_reversibility(torch, cfg, prec):
    """Strang step is unitary and symmetric: the norm stays 1 and stepping with -dt (fields replayed
    backwards) returns psi0 (eq. 7).  Holds at any size; run at BASELINE's sizes."""
    nsteps = {2: 20, 3: 6, 4: 20, 5: 4}[cfg]
    w = wl.CONFIGS[cfg](nsteps=nsteps)
    p = make_plan(w, prec)
    s0 = start_state(w, prec)
    psi = torch.from_numpy(s0).cuda()
    p.step(psi, nsteps)
    n1 = p.norm(psi)
    assert abs(n1 - 1.0) < (1e-12 if prec == sso.C128 else 2e-5), n1
    moved = rel_l2(psi.cpu().numpy(), s0)
    assert moved > 1e-4  # the step did something
    back = sso.Plan(w.sizes, w.dx, -w.dt, w.ncomp, prec)
    back.set_constants(w.mass, w.c, w.charge)
    back.set_potential(w.V)
    if w.field_kind:
        back.set_field(w.field_kind, np.ascontiguousarray(w.step_avg[:nsteps][::-1]))
    back.step(psi, nsteps)
    torch.cuda.synchronize()
    err = rel_l2(psi.cpu().numpy(), s0)
    assert err <= (1e-12 if prec == sso.C128 else 2e-5), err
    p.destroy()
    back.destroy()


# ---------------------------------------------------------------------------------------------------------
# edge cases of the boundary
# ---------------------------------------------------------------------------------------------------------

def test_zero_steps_and_chunking(torch):
    w = wl.config2(sizes=(64, 128), nsteps=12)
    p = make_plan(w)
    psi = torch.from_numpy(w.psi0.copy()).cuda()
    p.step(psi, 0)
    torch.cuda.synchronize()
    assert np.array_equal(psi.cpu().numpy(), w.psi0)
    assert p.get_time_index() == 0 and p.launch_count(0) == 0
    one, _ = gpu_steps(torch, w, 12)
    many, _ = gpu_steps(torch, w, 12, chunks=[1] * 12)
    assert rel_l2(many, one) < 1e-14
    want = oracle_steps(w, 12)
    assert rel_l2(one, want) < 1e-13 and rel_l2(many, want) < 1e-13
    p.destroy()


def test_time_index_selects_the_field_row(torch):
    w = wl.config4(sizes=(64, 64), nsteps=10)
    p = make_plan(w)
    psi = torch.from_numpy(w.psi0.copy()).cuda()
    p.set_time_index(5)
    p.step(psi, 3)
    torch.cuda.synchronize()
    o = make_oracle(w)
    o.set_time_index(5)
    assert rel_l2(psi.cpu().numpy(), o.step(w.psi0, 3)) < 1e-13
    assert p.get_time_index() == 8
    p.destroy()


def test_error_paths_on_device(torch):
    w = wl.config2(sizes=(32, 32), nsteps=4)
    p = make_plan(w)
    psi = torch.from_numpy(w.psi0.copy()).cuda()
    before = psi.clone()
    with pytest.raises(sso.SsoError) as e:
        p.step(psi, w.step_avg.shape[0] + 1)  # field table too short
    assert e.value.code == sso.ERR_STATE
    with pytest.raises(sso.SsoError) as e:
        p.step(psi.data_ptr() + 8, 1)  # misaligned
    assert e.value.code == sso.ERR_INVALID
    with pytest.raises(sso.SsoError) as e:
        p.step(psi, -1)
    assert e.value.code == sso.ERR_INVALID
    with pytest.raises(sso.SsoError):
        p.step(None, 1)
    with pytest.raises(sso.SsoError):
        p.set_field(7, w.step_avg)
    with pytest.raises(sso.SsoError):
        p.set_field(sso.FIELD_E, np.full((2, 2), np.nan))
    with pytest.raises(sso.SsoError):
        p.set_constants(-1.0, 1.0, 1.0)
    with pytest.raises(sso.SsoError):
        p.set_option(sso.OPT_LINES_PER_TILE_CONTIG, 3)
    with pytest.raises(sso.SsoError):
        p.set_time_index(-1)
    torch.cuda.synchronize()
    assert torch.equal(psi, before)  # failed calls touched nothing
    p.destroy()
    p.destroy()  # idempotent


def test_binding_rejects_mismatched_buffers(torch):
    """The C ABI takes bare pointers; the Python binding refuses buffers that do not match the plan."""
    w = wl.config2(sizes=(32, 64), nsteps=2)
    p = make_plan(w)
    good = torch.from_numpy(w.psi0.copy()).cuda()
    with pytest.raises(ValueError):
        p.step(good.to(torch.complex64), 1)           # element width
    with pytest.raises(ValueError):
        p.step(good[:, :16], 1)                        # size
    with pytest.raises(ValueError):
        p.step(good.transpose(1, 2), 1)                # contiguity
    with pytest.raises(ValueError):
        p.step(torch.from_numpy(w.psi0.copy()), 1)     # host tensor for a device argument
    with pytest.raises(ValueError):
        p.step_host(good, 1)                           # device tensor for a host argument
    with pytest.raises(ValueError):
        p.set_potential(w.V.astype(np.float32))        # V must be float64
    with pytest.raises(ValueError):
        p.norm(good[:, :16])
    p.step(good, 1)
    p.destroy()


def test_changing_the_potential_representation_invalidates_the_potential(torch):
    w = wl.config2(sizes=(32, 64), nsteps=2)
    p = make_plan(w)
    psi = torch.from_numpy(w.psi0.copy()).cuda()
    p.set_option(sso.OPT_POTENTIAL_PHASE, 1)
    with pytest.raises(sso.SsoError) as e:
        p.step(psi, 1)
    assert e.value.code == sso.ERR_STATE
    p.set_potential(w.V)
    p.step(psi, 2)
    torch.cuda.synchronize()
    assert rel_l2(psi.cpu().numpy(), oracle_steps(w, 2)) < 1e-13
    p.destroy()


def test_profile_step_reports_every_pass(torch):
    w = wl.config3(sizes=(32, 32, 64), nsteps=4)
    p = make_plan(w)
    psi = torch.from_numpy(w.psi0.copy()).cuda()
    rows = p.profile_step(psi, 4)
    torch.cuda.synchronize()
    names = {r[0].split(" [")[0]: r[1] for r in rows}
    assert names["opening"] == 1 and names["closing"] == 1 and names["potential"] == 3 and names["kinetic"] == 4
    assert sum(r[1] for r in rows if r[0].startswith("middle axis")) == 8
    assert all(r[2] > 0.0 for r in rows)
    assert rel_l2(psi.cpu().numpy(), oracle_steps(w, 4)) < 1e-13  # the profiled call is a real step
    p.destroy()


def test_potential_sources_agree(torch):
    """Host V, device V and V = NULL (zero) through sso_set_potential."""
    w = wl.config3(sizes=(16, 32, 32), nsteps=3)
    a, _ = gpu_steps(torch, w, 3)
    p = make_plan(w)
    p.set_potential(torch.from_numpy(w.V).cuda(), on_device=True)
    psi = torch.from_numpy(w.psi0.copy()).cuda()
    p.step(psi, 3)
    torch.cuda.synchronize()
    assert np.array_equal(psi.cpu().numpy(), a)
    p.set_potential(None)
    p.set_time_index(0)
    psi = torch.from_numpy(w.psi0.copy()).cuda()
    p.step(psi, 3)
    torch.cuda.synchronize()
    w0 = wl.Workload("free", w.sizes, w.dx, w.dt, 1, 3, w.psi0, V=None)
    assert rel_l2(psi.cpu().numpy(), oracle_steps(w0, 3)) < 1e-13
    p.destroy()


def test_tile_options_and_angle_table_do_not_change_results(torch):
    w = wl.config2(sizes=(128, 256), nsteps=6)
    want = oracle_steps(w, 6)
    for opts in (((sso.OPT_LINES_PER_TILE_CONTIG, 1), (sso.OPT_LINES_PER_TILE_STRIDED, 1)),
                 ((sso.OPT_LINES_PER_TILE_CONTIG, 4), (sso.OPT_LINES_PER_TILE_STRIDED, 8)),
                 ((sso.OPT_POTENTIAL_PHASE, 1),)):
        got, _ = gpu_steps(torch, w, 6, options=opts)
        assert rel_l2(got, want) < 1e-13, opts


def test_step_host_matches_device_path(torch):
    w = wl.config4(sizes=(64, 128), nsteps=5)
    dev, _ = gpu_steps(torch, w, 5)
    p = make_plan(w)
    host = torch.from_numpy(w.psi0.copy()).pin_memory()
    p.step_host(host, 5)
    assert np.array_equal(host.numpy(), dev)
    p.destroy()


def test_norm_matches_oracle(torch):
    for prec in (sso.C128, sso.C64):
        w = wl.config5(sizes=(16, 16, 32), nsteps=1)
        s = start_state(w, prec)
        p = make_plan(w, prec)
        got = p.norm(torch.from_numpy(s).cuda())
        want = make_oracle(w).norm(s.astype(np.complex128))
        assert abs(got - want) <= 1e-14 * want
        p.destroy()


def test_steps_on_a_side_stream_and_graph_capture(torch):
    """sso_step only enqueues kernels on the caller's stream, so it can be captured into a CUDA graph."""
    w = wl.config2(sizes=(64, 64), nsteps=8)
    p = make_plan(w)
    psi = torch.from_numpy(w.psi0.copy()).cuda()
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        p.step(psi, 2, stream=st)
    st.synchronize()
    g = torch.cuda.CUDAGraph()
    p.set_time_index(2)
    with torch.cuda.graph(g, stream=st):
        p.step(psi, 3, stream=torch.cuda.current_stream())
    g.replay()
    torch.cuda.synchronize()
    assert rel_l2(psi.cpu().numpy(), oracle_steps(w, 5)) < 1e-13
    p.destroy()


def test_first_step_of_a_dirac_table_plan_can_be_captured(torch):
    """SSO_OPT_DIRAC_TABLE = 1: the table is allocated by sso_set_option, not by the first sso_step, which therefore
    can sit inside a stream capture without a warm-up call (only the kernel that fills the table is enqueued)."""
    w = wl.config4(sizes=(64, 64), nsteps=4)
    p = make_plan(w)
    p.set_option(sso.OPT_DIRAC_TABLE, 1)
    psi = torch.from_numpy(w.psi0.copy()).cuda()
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=st):
        p.step(psi, 4, stream=torch.cuda.current_stream())
    g.replay()
    torch.cuda.synchronize()
    assert rel_l2(psi.cpu().numpy(), oracle_steps(w, 4)) < 1e-12
    p.destroy()


BENCH_ONLY = [
    ("d1", lambda: wl.dirac1d(sizes=(4096,), nsteps=100, ncomp=2), 100),
    ("d2x4", lambda: wl.dirac2d4(nsteps=20), 20),
    ("d2A", lambda: wl.dirac2d_magnetic(nsteps=20), 20),
]


@pytest.mark.parametrize("name,make,nsteps", BENCH_ONLY, ids=[b[0] for b in BENCH_ONLY])
def test_bench_only_workloads_at_full_size(torch, name, make, nsteps):
    """The three workloads bench.py times besides BASELINE.json's configs (the paper's 1D Dirac line, its 4-component
    2D Dirac shape, and 2D Dirac with A(r) applied in position space, eq. 26), at the size and in the launch
    configuration of the bench (default options, one call), element by element against the oracle."""
    w = make()
    p = make_plan(w)
    o = make_oracle(w)
    if "A" in w.extra:
        p.set_vector_potential(np.ascontiguousarray(w.extra["A"]))
        o.set_vector_potential(w.extra["A"])
    psi = torch.from_numpy(w.psi0.copy()).cuda()
    p.step(psi, nsteps)
    torch.cuda.synchronize()
    nrm = p.norm(psi)
    p.destroy()
    got = psi.cpu().numpy()
    want = o.step(w.psi0.astype(np.complex128), nsteps)
    assert rel_l2(got, want) <= TOL[sso.C128], (name, rel_l2(got, want))
    assert np.abs(got - want).max() <= 5 * TOL[sso.C128] * np.abs(want).max(), name
    assert abs(nrm - 1.0) < 1e-11
