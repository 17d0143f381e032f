"""GPU leapfrog stepper (etics_stepper_*) against oracle.leapfrog with the oracle's forces.

Tolerance: each force evaluation agrees with the oracle to 1e-10 (tests/parity.py); over n steps of length dt a relative
force error e moves x by at most ~ (n dt)^2 |a| e / 2 and v by ~ n dt |a| e, and with n dt = 0.12 << the dynamical time of
all but a handful of particles nothing is amplified, so 1e-9 on x (relative) and on v (relative to |v| + n dt |a|) has
an order of magnitude of head-room.  Graph replay and plain launches must agree bit for bit.
"""
import numpy as np
import pytest

import oracle
from paper_1406_4254_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
STEP_TOL = 1e-9


@pytest.fixture(scope="module")
def E():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1406_4254_b200 import binding
    binding.lib()
    binding.etics_init()
    return binding


def initial_conditions(n, seed):
    pos, mass = W.particles("hernquist", n, seed=seed)
    # seeded isotropic velocities of the order of the circular speed at r = 1 (not an equilibrium: any smooth state will do)
    vel = 0.3 * np.stack([W.uniforms(seed, n, 3 + k) - 0.5 for k in range(3)])
    return pos, vel, mass


def run_gpu(E, method, pos, vel, mass, dt, nsteps, nmax, lmax, graph, chunks=(None,)):
    dpos, dvel, dmass = (torch.from_numpy(a.copy()).cuda() for a in (pos, vel, mass))
    s = E.Stepper(method, dpos, dvel, dmass, dt, nmax=nmax, lmax=lmax, use_graph=graph)
    for c in chunks:
        s.step(nsteps if c is None else c)
    torch.cuda.synchronize()
    out = dpos.cpu().numpy(), dvel.cpu().numpy(), s.acc.cpu().numpy(), s.pot.cpu().numpy()
    s.close()
    return out


def check(x, v, a, x0, v0, a0, ndt):
    ex = np.max(np.linalg.norm(x - x0, axis=0) / np.linalg.norm(x0, axis=0))
    ev = np.max(np.linalg.norm(v - v0, axis=0) / (np.linalg.norm(v0, axis=0) + ndt * np.linalg.norm(a0, axis=0)))
    ea = np.max(np.linalg.norm(a - a0, axis=0) / np.linalg.norm(a0, axis=0))
    assert ex <= STEP_TOL and ev <= STEP_TOL and ea <= 10 * STEP_TOL, (ex, ev, ea)


@pytest.mark.parametrize("graph", [False, True])
def test_scf_leapfrog_12_steps(E, graph):
    n, dt, nsteps, nmax, lmax = 3_000, 0.01, 12, 10, 6
    pos, vel, mass = initial_conditions(n, 11)
    x, v, a, pot = run_gpu(E, 0, pos, vel, mass, dt, nsteps, nmax, lmax, graph)
    x0, v0, a0 = oracle.leapfrog(oracle.scf_acceleration(mass, nmax, lmax), pos, vel, dt, nsteps)
    check(x, v, a, x0, v0, a0, nsteps * dt)
    A, B = oracle.scf_coeffs(x0, mass, nmax, lmax)
    pot0 = oracle.scf_force(x0, nmax, lmax, A, B)[1]
    assert np.max(np.abs(pot - pot0) / np.abs(pot0)) <= 10 * STEP_TOL


@pytest.mark.parametrize("graph", [False, True])
def test_mex_leapfrog_12_steps(E, graph):
    n, dt, nsteps, lmax = 3_000, 0.01, 12, 4
    pos, vel, mass = initial_conditions(n, 12)
    x, v, a, pot = run_gpu(E, 1, pos, vel, mass, dt, nsteps, 0, lmax, graph)
    x0, v0, a0 = oracle.leapfrog(oracle.mex_acceleration(mass, lmax), pos, vel, dt, nsteps)
    check(x, v, a, x0, v0, a0, nsteps * dt)


@pytest.mark.parametrize("method,nmax,lmax", [(0, 10, 6), (1, 0, 6)])
def test_graph_replay_is_bit_identical_and_steps_compose(E, method, nmax, lmax):
    pos, vel, mass = initial_conditions(20_011, 13)
    plain = run_gpu(E, method, pos, vel, mass, 0.005, 6, nmax, lmax, False)
    graph = run_gpu(E, method, pos, vel, mass, 0.005, 6, nmax, lmax, True)
    split = run_gpu(E, method, pos, vel, mass, 0.005, 6, nmax, lmax, True, chunks=(1, 2, 0, 3))
    for p, g, s in zip(plain, graph, split):
        assert np.array_equal(p, g) and np.array_equal(p, s)


def test_graph_replay_large_sort_path(E):
    """N above one sort tile per resident block: the step's graph holds the one-kernel-per-phase sort (20 MEX launches)."""
    pos, vel, mass = initial_conditions(1_300_003, 16)
    plain = run_gpu(E, 1, pos, vel, mass, 0.002, 3, 0, 2, False)
    graph = run_gpu(E, 1, pos, vel, mass, 0.002, 3, 0, 2, True)
    for p, g in zip(plain, graph):
        assert np.array_equal(p, g)
    assert np.all(np.isfinite(graph[0])) and np.all(np.isfinite(graph[2]))


def test_stepper_argument_errors(E):
    import ctypes as C
    pos, vel, mass = initial_conditions(100, 1)
    d = [torch.from_numpy(a.copy()).cuda() for a in (pos, vel, mass)]
    acc = torch.empty((3, 100), dtype=torch.float64, device="cuda"); pot = torch.empty(100, dtype=torch.float64, device="cuda")
    ws = torch.empty(E.lib().etics_stepper_workspace_bytes(1, 100, 0, 4), dtype=torch.uint8, device="cuda")
    h = C.c_void_p()
    args = lambda method, n, lmax, wsb: (C.byref(h), method, d[0].data_ptr(), d[1].data_ptr(), d[2].data_ptr(), n, 0, lmax, 0.01,
                                          acc.data_ptr(), pot.data_ptr(), ws.data_ptr(), wsb, 0, 0)
    assert E.lib().etics_stepper_create(*args(2, 100, 4, ws.numel())) == E.ETICS_ERR_ARG
    assert E.lib().etics_stepper_create(*args(1, 0, 4, ws.numel())) == E.ETICS_ERR_ARG
    assert E.lib().etics_stepper_create(*args(1, 100, 11, ws.numel())) == E.ETICS_ERR_LIMIT
    assert E.lib().etics_stepper_create(*args(1, 100, 4, 16)) == E.ETICS_ERR_WORKSPACE
    assert h.value is None
    assert E.lib().etics_stepper_step(None, 1) == E.ETICS_ERR_ARG
    assert E.lib().etics_stepper_destroy(None) == E.ETICS_OK


@pytest.mark.parametrize("graph", [False, True])
def test_scf_temporal_softening(E, graph):
    """coefficients refreshed every 4th force evaluation, held in between."""
    n, dt, nsteps, nmax, lmax, every = 2_000, 0.01, 10, 8, 5, 4
    pos, vel, mass = initial_conditions(n, 14)
    dpos, dvel, dmass = (torch.from_numpy(a.copy()).cuda() for a in (pos, vel, mass))
    s = E.Stepper(0, dpos, dvel, dmass, dt, nmax=nmax, lmax=lmax, use_graph=graph)
    s.set_coefficient_interval(every)
    s.step(3); s.step(nsteps - 3)
    torch.cuda.synchronize()
    x0, v0, a0 = oracle.leapfrog(oracle.scf_acceleration(mass, nmax, lmax, every=every), pos, vel, dt, nsteps)
    check(dpos.cpu().numpy(), dvel.cpu().numpy(), s.acc.cpu().numpy(), x0, v0, a0, nsteps * dt)
    assert E.lib().etics_stepper_set_coefficient_interval(s._h, 2) == E.ETICS_ERR_ARG   # only before the first step
    s.close()
