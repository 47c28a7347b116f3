"""Pins for the oracle's Vay pusher ("conventional particle pusher algorithms, (e.g., Boris 1970; Vay 2008)").

What fixes it without reference to its own formulas:
  * the defining property of Vay's scheme: when E + v x B = 0 (a particle moving with the E x B drift velocity) the momentum does
    not change, for ANY time step -- Boris does not have it;
  * pure B: |u| is conserved exactly, and the motion is a rotation about B;
  * E parallel to B: u_par grows by (q/m) E dt per step exactly;
  * it solves the same equation (Eq. 3) as Boris: the two agree to O(dt^3) per step, and both converge to the exact relativistic
    cyclotron motion in uniform B (closed form) at second order.
"""
import numpy as np
import pytest

from helpers import cart_grid, make_particles, uniform_fields


def test_vay_keeps_a_drifting_particle_force_free(orc):
    rng = np.random.default_rng(11)
    for _ in range(20):
        B = rng.standard_normal(3)
        vd = rng.standard_normal(3); vd -= (vd @ B) / (B @ B) * B                 # drift velocity, perpendicular to B
        vd *= rng.uniform(0.05, 0.6) / np.linalg.norm(vd)
        E = -np.cross(vd, B)                                                      # E + vd x B = 0
        vd = vd + rng.uniform(-0.7, 0.7) * B / np.linalg.norm(B)                  # plus any velocity along B: still force free
        u = vd / np.sqrt(1.0 - vd @ vd)
        for dt in (0.01, 0.5, 5.0):
            assert np.allclose(orc.vay(u, E, B, -1.7, dt), u, rtol=0, atol=1e-13 * max(1.0, np.linalg.norm(u)))
        assert not np.allclose(orc.boris(u, E, B, -1.7, 5.0), u, atol=1e-3)      # Boris drifts off at large dt: the pin discriminates


def test_vay_pure_B_is_a_rotation_and_E_parallel_B_is_exact(orc):
    u = np.array([0.3, -1.2, 0.7]); B = np.array([0.4, 0.1, -0.9])
    n0 = np.linalg.norm(u); par0 = u @ B / np.linalg.norm(B)
    for _ in range(300):
        u = orc.vay(u, [0, 0, 0], B, 2.0, 0.2)
    assert np.linalg.norm(u) == pytest.approx(n0, rel=1e-13)
    assert u @ B / np.linalg.norm(B) == pytest.approx(par0, rel=1e-12)
    u = np.array([0.3, 0.1, -0.2]); qm, E, Bz, dt = -2.0, 0.7, 1.3, 0.05
    for n in range(1, 200):
        u = orc.vay(u, [0, 0, E], [0, 0, Bz], qm, dt)
        assert u[2] == pytest.approx(-0.2 + n * qm * E * dt, abs=1e-13)


def test_vay_and_boris_solve_the_same_equation(orc):
    """one step: |u_vay - u_boris| = O(dt^3); cyclotron motion in uniform B against the closed form u(t) = R(omega t) u0, omega = qB/(gamma m)"""
    u0 = np.array([0.8, 0.3, -0.5]); E = np.array([0.2, -0.1, 0.3]); B = np.array([0.1, 0.9, -0.4])
    d = [np.linalg.norm(orc.vay(u0, E, B, 1.0, dt) - orc.boris(u0, E, B, 1.0, dt)) for dt in (0.08, 0.04, 0.02)]
    assert 6.5 < d[0] / d[1] < 9.5 and 6.5 < d[1] / d[2] < 9.5, d
    gam = np.sqrt(1 + 0.25)
    errs = []
    for dt in (0.1, 0.05):
        u = np.array([0.5, 0.0, 0.0]); n = int(round(4.0 / dt))
        for _ in range(n):
            u = orc.vay(u, [0, 0, 0], [0, 0, 1.0], 1.0, dt)
        ang = -4.0 / gam                                                          # q > 0, B = +z: clockwise
        errs.append(np.linalg.norm(u - 0.5 * np.array([np.cos(ang), np.sin(ang), 0.0])))
    assert 3.5 < errs[0] / errs[1] < 4.5 and errs[1] < 5e-4


def test_gather_push_uses_the_selected_pusher(orc):
    g = cart_grid(orc, 3, (8, 8, 8), (4.0, 4.0, 4.0))
    F = uniform_fields(orc, g, E=(0.4, 0.0, 0.0), B=(0.0, 0.0, 2.0))           # contravariant: physical E_x = 0.2, B_z = 1
    p = make_particles(orc, [[3, 3, 3]], [[0.5, 0.5, 0.5]], [[0.3, 0.1, 0.2]])
    try:
        assert orc.set_pusher(1) == 0
        out = orc.gather_push(g, F, p, 1.0, 0.1)
        want = orc.vay([0.3, 0.1, 0.2], [0.2, 0, 0], [0, 0, 1.0], 1.0, 0.1)
        assert np.allclose([out.u[0][0], out.u[1][0], out.u[2][0]], want, atol=1e-15)
    finally:
        orc.set_pusher(0)
    out = orc.gather_push(g, F, p, 1.0, 0.1)
    assert np.allclose([out.u[0][0], out.u[1][0], out.u[2][0]], orc.boris([0.3, 0.1, 0.2], [0.2, 0, 0], [0, 0, 1.0], 1.0, 0.1), atol=1e-15)
