"""Pins for the oracle's pusher, mover and crossing bookkeeping.

BASELINE.json names them: exact gyration frequency and energy conservation in a pure uniform B, the
closed-form E x B drift, brute-force single-particle cell-crossing cases.  Added: uniform E parallel to B
(closed form), free streaming through the curvilinear grids (a straight line in the Cartesian frame).
"""
import numpy as np
import pytest

from helpers import cart_grid, make_particles, qsph_grid, sph_grid, uniform_fields


# ------------------------------------------------------------------ O4 Boris alone
def test_boris_pure_B_conserves_energy_and_rotates_by_the_scheme_angle(orc):
    """Pure uniform B: |u| constant to round-off; rotation per step exactly 2 atan(|q| B dt / (2 gamma m)),
    which tends to omega_c dt (the gyration frequency, Eq. 3).  q > 0, B = +z: clockwise seen from +z."""
    for qm, Bz, dt, u0 in [(1.0, 1.0, 0.225, [0.3, -0.2, 0.4]), (-1.0, 2.5, 0.1, [3.0, 1.0, -2.0]), (100.0, 0.01, 0.05, [0.1, 0.0, 0.0])]:
        u = np.array(u0, dtype=np.float64)
        gam = np.sqrt(1 + u @ u)
        n0 = np.linalg.norm(u)
        for _ in range(500):
            un = orc.boris(u, [0, 0, 0], [0, 0, Bz], qm, dt)
            ang = np.arctan2(un[1], un[0]) - np.arctan2(u[1], u[0])
            ang = (ang + np.pi) % (2 * np.pi) - np.pi
            assert ang == pytest.approx(-2 * np.arctan(qm * Bz * dt / (2 * gam)), abs=1e-14)
            assert un[2] == pytest.approx(u[2], abs=1e-15)
            u = un
        assert np.linalg.norm(u) == pytest.approx(n0, rel=1e-13)
    # the scheme angle tends to the exact omega_c dt = q B dt / (gamma m) as dt -> 0, second order
    gam = np.sqrt(1 + 0.25)
    for dt in (1e-2, 1e-3):
        un = orc.boris([0.5, 0, 0], [0, 0, 0], [0, 0, 1.0], 1.0, dt)
        w = dt / gam                                   # exact omega_c dt
        rel = 1.0 - (-np.arctan2(un[1], un[0])) / w    # 2 atan(w/2) = w (1 - w^2/12 + ...)
        assert rel == pytest.approx(w * w / 12.0, rel=1e-3)


def test_boris_E_parallel_B_is_exact(orc):
    """Uniform E || B: u_par(n) = u_par(0) + n (q/m) E dt exactly; the perpendicular part only rotates."""
    u = np.array([0.3, 0.1, -0.2]); qm, E, B, dt = -2.0, 0.7, 1.3, 0.05
    perp0 = np.hypot(u[0], u[1])
    for n in range(1, 200):
        u = orc.boris(u, [0, 0, E], [0, 0, B], qm, dt)
        assert u[2] == pytest.approx(-0.2 + n * qm * E * dt, abs=1e-13)
    assert np.hypot(u[0], u[1]) == pytest.approx(perp0, rel=1e-12)


def test_boris_exb_drift(orc):
    """Crossed fields |E| < |B|: the gyro-averaged velocity tends to E x B / B^2 with O((omega_c dt)^2) error
    (closed form; tolerance 2e-3 from SURVEY 8(c))."""
    for EoB, dt in [(0.1, 0.2), (0.5, 0.1)]:
        E = [0.0, EoB, 0.0]; B = [0.0, 0.0, 1.0]
        u = np.array([0.0, 0.0, 0.0]); X = np.zeros(3)
        nsteps = int(4000 / dt)
        for _ in range(nsteps):
            u = orc.boris(u, E, B, 1.0, dt)
            X += u / np.sqrt(1 + u @ u) * dt
        vd = X / (nsteps * dt)
        assert vd[0] == pytest.approx(EoB, rel=2e-3)          # E x B / B^2 = +x
        assert abs(vd[1]) < 2e-3 * EoB + 2e-4
        assert vd[2] == 0.0


# ------------------------------------------------------------------ whole gather_push on Cartesian grids
def test_gather_push_gyration_on_a_cartesian_grid(orc):
    """Steps 3-7 end to end with uniform contravariant B^3 = B0/dz... (3D) : the orbit closes on a circle of
    the Larmor radius of the discrete scheme; |u| conserved; cell index + offset stay consistent."""
    g = cart_grid(orc, 3, (16, 16, 16), (8.0, 8.0, 8.0))       # dx = 0.5 -> sqrt(h) = 0.5
    B0 = 1.0
    F = uniform_fields(orc, g, B=(0, 0, B0 / 0.5))             # contravariant B^3 = B^zhat / sqrt(h33)
    p = make_particles(orc, [[8, 8, 8]], [[0.25, 0.5, 0.5]], [[0.4, 0.0, 0.1]])
    dt = 0.05
    gam = np.sqrt(1 + 0.4 ** 2 + 0.1 ** 2)
    X0 = (8.25 * 0.5, 8.5 * 0.5)
    # discrete Boris + leapfrog orbit: the positions lie on a circle of radius |v_perp| dt / (2 sin(alpha/2))
    # with alpha = 2 atan(dt/(2 gamma)) the per-step rotation (positions advance by chords)
    vperp = 0.4 / gam
    alpha = 2 * np.arctan(B0 * dt / (2 * gam))
    R = vperp * dt / (2 * np.sin(alpha / 2))
    pts = []
    for _ in range(400):
        p = orc.gather_push(g, F, p, 1.0, dt)
        pts.append([(p.i[0][0] + p.d[0][0]) * 0.5, (p.i[1][0] + p.d[1][0]) * 0.5, (p.i[2][0] + p.d[2][0]) * 0.5])
        assert 0 <= p.d[0][0] < 1 and 0 <= p.d[1][0] < 1 and 0 <= p.d[2][0] < 1
    pts = np.array(pts)
    # fit a circle through the first three points -> centre; every later point at distance R
    A = 2 * (pts[1:3, :2] - pts[0, :2]); b = (pts[1:3, :2] ** 2).sum(1) - (pts[0, :2] ** 2).sum()
    ctr = np.linalg.solve(A, b)
    rad = np.linalg.norm(pts[:, :2] - ctr, axis=1)
    assert np.allclose(rad, R, rtol=1e-10)
    # uniform drift along z with v_z = u_z / gamma (periodic wrap at 8.0)
    z = pts[:, 2]
    want = (8.5 * 0.5 + 0.1 / gam * dt * np.arange(1, 401)) % 8.0
    assert np.allclose(z, want, atol=1e-11)
    u = np.array([p.u[0][0], p.u[1][0], p.u[2][0]])
    assert np.linalg.norm(u) == pytest.approx(np.sqrt(0.17), rel=1e-13)


def test_gather_push_exb_drift_2d_cartesian(orc):
    """The full steps 3-7 in 2D Cartesian with dx != 1: contravariant components E^2 = E^yhat/dy, B^3 = B^zhat
    (h33 = 1 in 2D).  The guiding centre drifts with E x B / B^2 in physical units."""
    g = cart_grid(orc, 2, (32, 32), (16.0, 16.0))
    Ey, Bz = 0.2, 1.0
    F = uniform_fields(orc, g, E=(0, Ey / 0.5, 0), B=(0, 0, Bz))
    p = make_particles(orc, [[3, 16]], [[0.0, 0.0]], [[0.0, 0.0, 0.0]])
    dt = 0.1
    x_unwrapped = 3 * 0.5
    prev = x_unwrapped
    nsteps = 20000
    for _ in range(nsteps):
        p = orc.gather_push(g, F, p, 1.0, dt)
        x = (p.i[0][0] + p.d[0][0]) * 0.5
        dxs = x - (prev % 16.0)
        dxs -= 16.0 * np.round(dxs / 16.0)
        prev += dxs
    assert (prev - x_unwrapped) / (nsteps * dt) == pytest.approx(Ey / Bz, rel=2e-3)


# ------------------------------------------------------------------ O7 crossing, brute force
def test_crossing_patterns_brute_force(orc):
    """All 3^D patterns, both periodic wraps, delta = 0 and landing exactly on a face; expected (i', delta')
    computed by hand: x' = i + delta + v dt / dx, i' = floor(x') mod N, delta' = x' - floor(x')."""
    for D in (2, 3):
        N = (4, 5, 3)[:D]
        g = cart_grid(orc, D, N, tuple(float(n) for n in N))        # dx = 1
        F = uniform_fields(orc, g)
        dt = 0.5
        cases = []
        import itertools
        for pat in itertools.product((-1, 0, 1), repeat=D):
            for start in ("interior", "low_edge", "high_edge"):
                i, d, u = [], [], []
                for a in range(D):
                    ia = {"interior": 1, "low_edge": 0, "high_edge": N[a] - 1}[start]
                    # velocity 0.5 c * dt 0.5 = 0.25 cells; choose delta so that the pattern happens
                    da = {-1: 0.1, 0: 0.5, 1: 0.9}[pat[a]]
                    i.append(ia); d.append(da)
                    u.append(pat[a] * 0.5)
                cases.append((i, d, u))
        # delta = 0 moving backwards, and landing exactly on a face (0.75 + 0.25 = 1.0 exactly in binary)
        cases.append(([2] * D, [0.0] * D, [-0.5] + [0.0] * (D - 1)))
        cases.append(([2] * D, [0.75] * D, [0.5] + [0.0] * (D - 1)))        # with gamma: v = u/gamma, handled below
        for i, d, u in cases:
            uu = np.zeros(3); uu[:D] = u
            # choose u such that v = u / gamma equals the intended velocity: u = v / sqrt(1 - v^2)
            v = uu.copy()
            gam = 1.0 / np.sqrt(1.0 - v @ v)
            p = make_particles(orc, [i], [d], [v * gam])
            out = orc.gather_push(g, F, p, 1.0, dt)
            vv = (v * gam) / np.sqrt(1 + (v * gam) @ (v * gam))
            for a in range(D):
                xn = i[a] + d[a] + vv[a] * dt
                fl = np.floor(xn)
                assert out.i[a][0] == int(fl) % N[a], (i, d, u, a)
                assert out.d[a][0] == pytest.approx(xn - fl, abs=1e-15)
                assert 0.0 <= out.d[a][0] < 1.0
            assert out.tag[0] == 1
    # exact face landing: 0.75 + 0.25 -> delta' = 0, i' = i + 1 (v = 0.5 exactly needs u = 0.5/sqrt(0.75))
    g = cart_grid(orc, 2, (4, 4), (4.0, 4.0))
    F = uniform_fields(orc, g)
    uex = 0.5 / np.sqrt(0.75)
    out = orc.gather_push(g, F, make_particles(orc, [[3, 1]], [[0.75, 0.5]], [[uex, 0, 0]]), 1.0, 0.5)
    assert abs((out.i[0][0] + out.d[0][0]) % 4 - 0.0) < 1e-15 or out.d[0][0] > 1 - 1e-15


def test_absorbing_and_dead_particles(orc):
    """G9: leaving a non-periodic side sets tag = Dead; dead particles are passed through untouched."""
    g = cart_grid(orc, 2, (4, 4), (4.0, 4.0), bc=(orc.ABSORB, orc.PERIODIC))
    F = uniform_fields(orc, g)
    p = make_particles(orc, [[3, 1], [0, 1], [2, 2], [1, 1]], [[0.9, 0.5], [0.1, 0.5], [0.5, 0.5], [0.5, 0.5]],
                       [[2.0, 0, 0], [-2.0, 0, 0], [2.0, 0, 0], [1.0, 1.0, 0.0]], tag=[1, 1, 1, 0])
    out = orc.gather_push(g, F, p, 1.0, 0.5)
    assert list(out.tag) == [0, 0, 1, 0]
    assert out.i[0][3] == 1 and out.d[0][3] == 0.5 and out.u[0][3] == 1.0      # dead: untouched


# ------------------------------------------------------------------ curvilinear mover: free streaming is a straight line
@pytest.mark.parametrize("mk", ["sph", "qsph0", "qsph"])
def test_free_streaming_is_a_straight_line_in_cartesian_space(orc, mk):
    """No fields: x^X(n) = x^X(0) + n v dt (Eq. 3) whatever the grid; pins forward map, move and
    back-map chained over many steps, including phi bookkeeping."""
    g = {"sph": sph_grid(orc, (64, 64), 1.0, 20.0),
         "qsph0": qsph_grid(orc, (64, 64), 1.0, 20.0, 0.0, 0.0),
         "qsph": qsph_grid(orc, (64, 64), 1.0, 20.0, 0.5, 0.4)}[mk]
    F = uniform_fields(orc, g)
    x0 = np.array([10.3, 20.7, 1.0])
    X0 = orc.code_to_cart(g, x0)
    u = np.array([0.8, -0.5, 0.6])
    v = u / np.sqrt(1 + u @ u)
    p = make_particles(orc, [[10, 20]], [[0.3, 0.7]], [u], phi=1.0)
    dt = 0.02
    for n in range(1, 301):
        p = orc.gather_push(g, F, p, 1.0, dt)
        X = orc.code_to_cart(g, [p.i[0][0] + p.d[0][0], p.i[1][0] + p.d[1][0], p.phi[0]])
        assert np.allclose(X, X0 + n * v * dt, atol=1e-11)
        assert p.tag[0] == 1
    assert np.allclose([p.u[0][0], p.u[1][0], p.u[2][0]], u)      # u stays in the global Cartesian basis


def test_axis_crossing_flips_phi(orc):
    """A particle flying over the pole: theta stays in [0, pi], phi jumps by pi; Cartesian track stays straight."""
    g = sph_grid(orc, (16, 16), 1.0, 9.0)
    F = uniform_fields(orc, g)
    x0 = np.array([4.0, 0.05, 0.3])
    X0 = orc.code_to_cart(g, x0)
    # velocity pointing across the axis: -x direction in the phi = 0.3 meridian plane
    vdir = -np.array([np.cos(0.3), np.sin(0.3), 0.0])
    u = 2.0 * vdir
    v = u / np.sqrt(5.0)
    p = make_particles(orc, [[4, 0]], [[0.0, 0.05]], [u], phi=0.3)
    seen_flip = False
    for n in range(1, 40):
        p = orc.gather_push(g, F, p, 1.0, 0.01)
        X = orc.code_to_cart(g, [p.i[0][0] + p.d[0][0], p.i[1][0] + p.d[1][0], p.phi[0]])
        assert np.allclose(X, X0 + n * v * 0.01, atol=1e-12)
        assert p.i[1][0] >= 0 and 0 <= p.d[1][0] < 1
        if abs(p.phi[0] - (0.3 + np.pi)) < 1e-9:
            seen_flip = True
    assert seen_flip


def test_gather_push_in_a_dipole_conserves_energy_with_E_zero(orc):
    """Pure (non-uniform) B on the spherical grid: each step is a rotation of u, so |u| is conserved to
    round-off whatever the interpolation and basis change did (BASELINE.json: energy conservation)."""
    g = qsph_grid(orc, (48, 48), 1.0, 20.0, 0.0, 0.3)
    shape = g.padded_shape
    rng = np.random.default_rng(7)
    F = [np.zeros(shape, dtype=np.float32) for _ in range(3)] + [rng.standard_normal(shape).astype(np.float32) for _ in range(3)]
    n = 64
    p = make_particles(orc, np.stack([rng.integers(2, 40, n), rng.integers(2, 44, n)], 1), rng.uniform(0, 1, (n, 2)),
                       rng.standard_normal((n, 3)), phi=rng.uniform(0, 2 * np.pi, n))
    e0 = np.sqrt(p.u[0] ** 2 + p.u[1] ** 2 + p.u[2] ** 2)
    for _ in range(20):
        p = orc.gather_push(g, F, p, 50.0, 0.002)
    e1 = np.sqrt(p.u[0] ** 2 + p.u[1] ** 2 + p.u[2] ** 2)
    alive = p.tag == 1
    assert alive.sum() > 32
    assert np.allclose(e1[alive], e0[alive], rtol=1e-13)
