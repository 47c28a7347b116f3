"""Pins for the TIME LEVELS and EVALUATION POINTS of the oracle (readings G3, G4, G8, G11 of DESIGN.md): the places where a
plausible misreading survives the other pin files because their test particles have E = 0, constant gamma, or old = new.

Each test fixes the result by something other than the oracle's own formula:
  * Eq. 3 is time reversible: pushing with -dt undoes the push, for any E and B;
  * a charge starting at rest in a uniform E follows the hyperbola x(t) = (sqrt(1 + (a t)^2) - 1) / a exactly, and the
    leap-frog of P:141-149 (u at half steps, x^(n+1) = x^n + u^(n+1/2)/gamma^(n+1/2) dt) converges to it at second order;
  * the out-of-plane current is a rate at n+1/2 (step 8 deposits between x^n and x^(n+1)): its nodal sum is
    q w v^3 with the NEW momentum, v^3 = v^phihat / sqrt(h33) taken at the midpoint of the move, the azimuth midpoint along
    the shorter arc; sqrt(h33) = the cylindrical radius of the forward map, not the oracle's metric routine;
  * theta = pi exactly is clamped into the last cell (0 <= delta < 1 is an invariant of the particle format).
tests/oracle_mutants.py lists the one-line mutations of orc.c each of these kills.
"""
import numpy as np
import pytest

from helpers import cart_grid, make_particles, sph_grid, qsph_grid, uniform_fields


def test_boris_is_time_reversible_with_E_and_B(orc):
    """Eq. 3: u -> boris(dt) -> boris(-dt) returns u to round-off.  Holds only if the rotation uses gamma of u^- = u + eps E
    (the value the rotation conserves); gamma of the incoming u breaks it at first order in E."""
    rng = np.random.default_rng(3)
    for _ in range(50):
        u = rng.standard_normal(3) * rng.choice([0.1, 1.0, 10.0])
        E = rng.standard_normal(3) * 0.8
        B = rng.standard_normal(3) * 1.5
        qm, dt = rng.choice([-1.0, 1.0, 30.0]), rng.uniform(0.01, 0.3)
        back = orc.boris(orc.boris(u, E, B, qm, dt), E, B, qm, -dt)
        assert np.allclose(back, u, rtol=0, atol=1e-13 * max(1.0, np.abs(u).max()))
    # and the forward push is not the identity in these cases (the test is not vacuous)
    assert not np.allclose(orc.boris([0.1, 0.2, 0.3], [0.5, 0, 0], [0, 0, 1.0], 1.0, 0.1), [0.1, 0.2, 0.3])


def _hyperbola_error(orc, dt, T=6.0):
    """steps 3-7 through orc_gather_push on a 3D Cartesian grid (dx = 0.5) with uniform E along x; the particle starts at
    rest at t = 0, i.e. u^(-1/2) = -a dt / 2; returns max |x_n - x_exact(t_n)| in physical units."""
    g = cart_grid(orc, 3, (64, 4, 4), (32.0, 2.0, 2.0))
    Ex, qm = 0.75, 1.0                                                  # E^1 = 1.5 is exact in the fp32 field arrays
    a = qm * Ex
    F = uniform_fields(orc, g, E=(Ex / 0.5, 0, 0))                      # contravariant E^1 = E^xhat / sqrt(h11)
    p = make_particles(orc, [[2, 1, 1]], [[0.0, 0.5, 0.5]], [[-0.5 * a * dt, 0.0, 0.0]])
    x0 = 2 * 0.5
    worst, prev, unwrapped = 0.0, x0, x0
    for n in range(1, int(round(T / dt)) + 1):
        p = orc.gather_push(g, F, p, qm, dt)
        x = (p.i[0][0] + p.d[0][0]) * 0.5
        step = x - (prev % 32.0)
        step -= 32.0 * np.round(step / 32.0)
        unwrapped += step
        prev = unwrapped
        t = n * dt
        worst = max(worst, abs(unwrapped - x0 - (np.sqrt(1.0 + (a * t) ** 2) - 1.0) / a))
        assert p.u[0][0] == pytest.approx(a * (t - 0.5 * dt), rel=1e-12)      # u^(n-1/2) exactly linear in t (E only)
    return worst


def test_hyperbolic_motion_converges_at_second_order(orc):
    """P:141-149 (reading G4): x advances with u^(n+1/2) / gamma^(n+1/2).  Against the exact hyperbola the error falls 4x
    when dt halves; with gamma taken at the old time level it would be first order (2x)."""
    e1, e2, e3 = _hyperbola_error(orc, 0.1), _hyperbola_error(orc, 0.05), _hyperbola_error(orc, 0.025)
    assert e1 < 3e-3
    assert 3.6 < e1 / e2 < 4.4 and 3.6 < e2 / e3 < 4.4, (e1, e2, e3)


def test_out_of_plane_current_2d_uses_the_new_momentum(orc):
    """J^3 is the rate q w v^3 at n+1/2: the block at n+1 carries u^(n+1/2), the old block u^(n-1/2)."""
    g = cart_grid(orc, 2, (6, 6), (3.0, 3.0))
    u_old = np.array([0.1, 0.4, -0.7]); u_new = np.array([0.3, -0.2, 0.9])
    po = make_particles(orc, [[2, 3]], [[0.8, 0.4]], [u_old], w=1.5)
    pn = make_particles(orc, [[3, 3]], [[0.1, 0.2]], [u_new], w=1.5)
    J = orc.zeros_current(g)
    orc.deposit(g, po, pn, J, -1.0, 0.2)
    assert J[2].sum() == pytest.approx(-1.0 * 1.5 * u_new[2] / np.sqrt(1 + u_new @ u_new), rel=1e-14)


@pytest.mark.parametrize("mk", ["sph", "qsph"])
def test_out_of_plane_current_axisymmetric_midpoint_and_shorter_arc(orc, mk):
    """A particle that moves in x1, x2 AND phi, across phi = 2 pi, with u_old != u_new.  Nodal sum of J^3 = q w v^phihat / rho_cyl
    with v^phihat = (-u_x sin phi_m + u_y cos phi_m) / gamma from the NEW momentum, phi_m = the midpoint along the shorter arc,
    rho_cyl = cylindrical radius of the midpoint of the move in code coordinates, from the forward map."""
    g = sph_grid(orc, (20, 20), 1.0, 11.0) if mk == "sph" else qsph_grid(orc, (20, 20), 1.0, 11.0, 0.2, 0.4)
    u_old = np.array([0.5, 0.1, -0.3]); u_new = np.array([-0.4, 0.8, 0.25])
    phi0, phi1 = 6.20, 0.07                                   # moves forward through 2 pi: shorter arc = +0.153...
    po = make_particles(orc, [[7, 10]], [[0.9, 0.2]], [u_old], w=2.0, phi=phi0)
    pn = make_particles(orc, [[8, 9]], [[0.3, 0.7]], [u_new], w=2.0, phi=phi1)
    J = orc.zeros_current(g)
    orc.deposit(g, po, pn, J, 1.0, 0.1)
    dphi = (phi1 - phi0 + np.pi) % (2 * np.pi) - np.pi
    assert 0.1 < dphi < 0.2
    phm = phi0 + 0.5 * dphi
    xm = [0.5 * (7.9 + 8.3), 0.5 * (10.2 + 9.7), 0.0]
    X = orc.code_to_cart(g, xm)                               # phi = 0: rho_cyl = X[0]
    assert X[1] == pytest.approx(0.0, abs=1e-15)
    gam = np.sqrt(1 + u_new @ u_new)
    vphi = (-u_new[0] * np.sin(phm) + u_new[1] * np.cos(phm)) / gam
    want = 1.0 * 2.0 * vphi / X[0]
    assert J[2].sum() == pytest.approx(want, rel=1e-13)
    # sensitivity: the old azimuth, the arithmetic mean of the azimuths, the old position or the old momentum all differ visibly
    for wrong in (np.sin(phi0), np.sin(0.5 * (phi0 + phi1))):
        assert abs(np.sin(phm) - wrong) > 1e-2


def _exact_landing_u(X0, dt):
    """u (< 0) with fl(fl(u / sqrt(1 + u u)) * dt) == -X0 exactly, found by stepping through neighbouring doubles"""
    v = -X0 / dt
    u = v / np.sqrt(1.0 - v * v)
    for _ in range(4000):
        got = (u / np.sqrt(1.0 + u * u)) * dt
        if got == -X0:
            return u
        u = np.nextafter(u, -np.inf if got > -X0 else np.inf)
    return None


def test_landing_on_theta_equals_pi_is_clamped_into_the_last_cell(orc):
    """G11: a particle that lands on the lower polar axis to the last bit (rho = 0, theta = pi, x2 = N_theta) must come out
    in cell N_theta - 1 with delta < 1: 0 <= delta < 1 and 0 <= i < N are invariants of the particle format."""
    g = sph_grid(orc, (16, 16), 1.0, 9.0)                     # N_theta = 16: pi / (pi/16) == 16 exactly
    F = uniform_fields(orc, g)
    dt = 0.5
    hit = 0
    for d2 in (0.45, 0.50, 0.55, 0.60, 0.70, 0.80):             # cylindrical radius 4 sin((1 - d2) pi / 16) < dt
        x = [6.0, 15.0 + d2, 0.0]
        X = orc.code_to_cart(g, x)                            # phi = 0: Y = 0, X[0] = cylindrical radius > 0, X[2] < 0
        assert X[1] == 0.0 and X[0] > 0 and X[2] < 0
        u = _exact_landing_u(X[0], dt)
        if u is None:
            continue
        out = orc.gather_push(g, F, make_particles(orc, [[6, 15]], [[0.0, d2]], [[u, 0.0, 0.0]], phi=0.0), 1.0, dt)
        back = orc.code_to_cart(g, [out.i[0][0] + out.d[0][0], out.i[1][0] + out.d[1][0], out.phi[0]])
        assert abs(back[0]) < 1e-14 and abs(back[1]) < 1e-14 and back[2] == pytest.approx(X[2], rel=1e-14)
        assert out.tag[0] == 1
        assert out.i[1][0] == 15, "theta = pi must be clamped into the last theta-cell"
        assert 0.0 <= out.d[1][0] < 1.0 and out.d[1][0] > 1.0 - 1e-15
        hit += 1
    assert hit >= 2, "no start point lands on the axis exactly: the pin is vacuous"


def test_the_listed_mutants_of_the_oracle_are_killed_by_their_pins():
    """tests/oracle_mutants.py: every listed one-line misreading of orc.c fails the pin named beside it (and the unmutated
    oracle passes those pins: they are part of this suite)."""
    import oracle_mutants as M
    survivors = [name for k in range(len(M.MUTANTS)) for name, killed in [M.check(k)] if not killed]
    assert not survivors, f"mutants that pass every designated pin: {survivors}"
