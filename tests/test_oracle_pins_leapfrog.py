"""Pins of oracle.leapfrog (the kick-drift-kick integrator of PAPER.md:257 that SURVEY.md §8(f)1 asks for).

None of them re-types the update formula: the harmonic oscillator has a closed-form DISCRETE solution under
kick-drift-kick, the scheme is time-reversible, it is second-order accurate on a Kepler orbit, and it conserves linear
momentum exactly for pairwise forces.  A dropped half kick, a swapped kick/drift order, dt in place of dt/2 or a stale
acceleration each fail at least one of them.
"""
import numpy as np

import oracle


def harmonic(omega):
    return lambda x: -(omega ** 2) * x


def test_harmonic_oscillator_closed_form():
    # KDK on x'' = -w^2 x is the linear map (x, v) -> M (x, v) with trace 2 - (w dt)^2: a rotation by theta with
    # cos(theta) = 1 - (w dt)^2 / 2 in the variables (x, v / (w sqrt(1 - (w dt)^2 / 4))): a textbook result.
    w, dt, n = 1.7, 0.05, 200
    x0 = np.array([[0.3, -1.0], [0.0, 0.2], [1.1, 0.0]]); v0 = np.array([[0.1, 0.0], [0.5, -0.3], [0.0, 0.9]])
    x, v, a = oracle.leapfrog(harmonic(w), x0, v0, dt, n)
    h = w * dt
    theta = np.arccos(1.0 - 0.5 * h * h)
    wp = w * np.sqrt(1.0 - 0.25 * h * h)
    xe = x0 * np.cos(n * theta) + (v0 / wp) * np.sin(n * theta)
    ve = v0 * np.cos(n * theta) - (x0 * wp) * np.sin(n * theta)
    assert np.max(np.abs(x - xe)) < 1e-12 and np.max(np.abs(v - ve)) < 1e-12
    assert np.array_equal(a, harmonic(w)(x))          # the returned acceleration belongs to the final positions


def kepler(x):
    r3 = np.sum(x * x, axis=0) ** 1.5
    return -x / r3


def test_time_reversible():
    x0 = np.array([[1.0], [0.0], [0.0]]); v0 = np.array([[0.0], [0.9], [0.2]])
    x1, v1, _ = oracle.leapfrog(kepler, x0, v0, 0.01, 300)
    x2, v2, _ = oracle.leapfrog(kepler, x1, -v1, 0.01, 300)
    assert np.max(np.abs(x2 - x0)) < 1e-11 and np.max(np.abs(v2 + v0)) < 1e-11


def test_second_order_on_a_circular_kepler_orbit():
    x0 = np.array([[1.0], [0.0], [0.0]]); v0 = np.array([[0.0], [1.0], [0.0]])
    T = 1.0
    errs = []
    for n in (100, 200, 400):
        x, v, _ = oracle.leapfrog(kepler, x0, v0, T / n, n)
        errs.append(np.linalg.norm(x[:, 0] - np.array([np.cos(T), np.sin(T), 0.0])))
    assert 3.7 < errs[0] / errs[1] < 4.3 and 3.7 < errs[1] / errs[2] < 4.3
    # energy error stays bounded and small (symplectic): |dE/E| = O(dt^2)
    x, v, _ = oracle.leapfrog(kepler, x0, v0, 0.01, 2000)
    E = 0.5 * np.sum(v * v) - 1.0 / np.linalg.norm(x)
    assert abs(E + 0.5) < 1e-4


def test_zero_steps_and_inputs_untouched():
    x0 = np.array([[1.0], [0.0], [0.0]]); v0 = np.array([[0.0], [1.0], [0.0]])
    xc, vc = x0.copy(), v0.copy()
    x, v, a = oracle.leapfrog(kepler, x0, v0, 0.1, 0)
    assert np.array_equal(x, x0) and np.array_equal(v, v0) and np.array_equal(a, kepler(x0))
    oracle.leapfrog(kepler, x0, v0, 0.1, 3)
    assert np.array_equal(x0, xc) and np.array_equal(v0, vc)


def test_mex_leapfrog_energy_and_two_body_radial_fall():
    # MEX lmax = 0 with two particles is Gauss's law: the inner one feels nothing, the outer one falls radially towards
    # the origin under m_inner / r^2 — a 1-D Kepler fall whose energy v^2/2 - m/r the leapfrog conserves to O(dt^2).
    pos = np.array([[0.1, 2.0], [0.0, 0.0], [0.0, 0.0]]); vel = np.zeros((3, 2)); mass = np.array([1.0, 1e-3])
    f = oracle.mex_acceleration(mass, 0)
    x, v, _ = oracle.leapfrog(f, pos, vel, 0.01, 100)
    assert np.array_equal(x[:, 0], pos[:, 0]) and np.all(v[:, 0] == 0.0)
    E0 = -1.0 / 2.0
    E1 = 0.5 * v[0, 1] ** 2 - 1.0 / x[0, 1]
    assert x[0, 1] < 2.0 and v[0, 1] < 0.0 and abs(E1 - E0) < 1e-6
    assert np.all(x[1:, 1] == 0.0)


def test_temporal_softening_static_field_conserves_particle_energies():
    # coefficients held over many steps = motion in a STATIC potential, in which the energy of every particle,
    # v^2/2 + Phi(x) with Phi from the held coefficients, is conserved by the leapfrog to O(dt^2); with every = 1 the helper
    # is the plain force.  (A wrong refresh schedule moves the potential under the particles and breaks the first part;
    # a stale acceleration breaks the second.)
    from paper_1406_4254_b200 import workloads as W
    pos, mass = W.particles("hernquist", 400, seed=21)
    vel = 0.3 * np.stack([W.uniforms(21, 400, 3 + k) - 0.5 for k in range(3)])
    f = oracle.scf_acceleration(mass, 6, 4, every=10_000)
    x, v, _ = oracle.leapfrog(f, pos, vel, 0.002, 50)
    A, B = f.state["AB"]
    assert f.state["calls"] == 51
    A0, B0 = oracle.scf_coeffs(pos, mass, 6, 4)
    assert np.array_equal(A, A0) and np.array_equal(B, B0)          # still the coefficients of x_0
    E0 = 0.5 * np.sum(vel ** 2, axis=0) + oracle.scf_force(pos, 6, 4, A, B)[1]
    E1 = 0.5 * np.sum(v ** 2, axis=0) + oracle.scf_force(x, 6, 4, A, B)[1]
    assert np.max(np.abs(E1 - E0) / np.abs(E0)) < 2e-4
    x1, v1, _ = oracle.leapfrog(oracle.scf_acceleration(mass, 6, 4, every=1), pos, vel, 0.002, 5)
    x2, v2, _ = oracle.leapfrog(oracle.scf_acceleration(mass, 6, 4), pos, vel, 0.002, 5)
    assert np.array_equal(x1, x2) and np.array_equal(v1, v2)
    # the schedule: every = 3 refreshes at evaluations 0, 3, 6 -> after 7 steps the held table belongs to x_6
    f3 = oracle.scf_acceleration(mass, 6, 4, every=3)
    xs = []
    g = lambda xx: (xs.append(xx.copy()), f3(xx))[1]
    oracle.leapfrog(g, pos, vel, 0.002, 7)
    A6, _ = oracle.scf_coeffs(xs[6], mass, 6, 4)
    assert np.array_equal(f3.state["AB"][0], A6)
