"""Pins of the hybrid pusher (N3, "Boris,GCA" / "Vay,GCA", reading G26) against what the paper's two sentences fix:
the switch on |E|/|B| and on the nominal gyroradius rho_L = gamma beta m c^2 / (q |B|) of the momentum the particle has at that
time step, and, in the guiding-centre regime, zero momentum perpendicular to the local B with the parallel momentum following
du_par/dt = (q/m) E_par (closed form).  Everything beyond those sentences is a reading ("parity unpinned", G26)."""
import numpy as np
import pytest

from helpers import cart_grid, make_particles, uniform_fields


@pytest.fixture()
def gca(orc):
    prev = orc.set_pusher(2)
    yield orc
    orc.set_pusher(prev)
    orc.set_gca(0.0, 0.0)


def _push_one(orc, g, E, B, u, qm, dt):
    """one particle through orc_gather_push in uniform fields (dx = 1: contravariant = orthonormal)"""
    F = uniform_fields(orc, g, E=E, B=B)
    p = make_particles(orc, [[3, 3, 3]], [[0.5, 0.5, 0.5]], [u])
    out = orc.gather_push(g, F, p, qm, dt)
    return np.array([out.u[a][0] for a in range(3)]), np.array([out.i[a][0] + out.d[a][0] for a in range(3)])


def test_guiding_centre_regime_kills_u_perp_and_follows_E_par(gca):
    orc = gca
    g = cart_grid(orc, 3, 8, 8.0)
    b = np.array([1.0, 2.0, -2.0]) / 3.0
    B = 5.0 * b
    Epar, Eperp = 0.3, 0.4 * np.cross(b, [0.0, 0.0, 1.0])
    E = Epar * b + Eperp
    qm, dt = -1.5, 0.2
    u0 = 0.3 * b + 0.2 * np.cross(b, [1.0, 0.0, 0.0])
    orc.set_gca(1.0, 0.9)                       # rho_L = |u| / (1.5 * 5) = 0.05 < 1; |E|/|B| = 0.1 < 0.9
    u1, x1 = _push_one(orc, g, E.astype(np.float32), B.astype(np.float32), u0, qm, dt)
    B32, E32 = B.astype(np.float32).astype(np.float64), E.astype(np.float32).astype(np.float64)
    b32 = B32 / np.linalg.norm(B32)
    assert np.linalg.norm(np.cross(u1, b32)) < 1e-15                       # no perpendicular momentum
    want_par = u0 @ b32 + qm * (E32 @ b32) * dt                            # du_par/dt = (q/m) E_par, exact for uniform fields
    assert abs(u1 @ b32 - want_par) < 1e-14
    gam = np.sqrt(1.0 + want_par ** 2)
    assert np.allclose(x1, 3.5 + want_par * b32 / gam * dt, atol=1e-14)    # sub-step 6 unchanged: the particle slides along the field line


def test_switch_on_the_gyroradius_of_the_momentum_before_the_push(gca):
    orc = gca
    g = cart_grid(orc, 3, 8, 8.0)
    B, E = np.array([0.0, 0.0, 2.0]), np.array([0.05, 0.0, 0.01])
    qm, dt = 2.0, 0.1
    rho_crit = 0.25                              # |u| m / (|q| |B|) < 0.25  <=>  |u| < 1.0
    orc.set_gca(rho_crit, 0.9)
    for umag, regime in ((0.999, "gca"), (1.001, "boris")):
        u0 = umag * np.array([0.6, 0.0, 0.8])
        u1, _ = _push_one(orc, g, E.astype(np.float32), B.astype(np.float32), u0, qm, dt)
        ub = orc.boris(u0, E.astype(np.float32).astype(np.float64), B, qm, dt)
        if regime == "boris":
            assert np.allclose(u1, ub, rtol=0, atol=1e-15)
        else:
            assert abs(u1[0]) < 1e-15 and abs(u1[1]) < 1e-15 and abs(u1[2] - ub[2]) < 1e-15
    # the criterion uses the momentum BEFORE the push: a strong parallel E that lifts |u| above the threshold during this very step
    orc.set_gca(rho_crit, 0.9)
    Ebig = np.array([0.0, 0.0, 1.5])
    u0 = 0.9 * np.array([0.6, 0.0, 0.8])
    u1, _ = _push_one(orc, g, Ebig.astype(np.float32), B.astype(np.float32), u0, qm, dt)
    assert np.linalg.norm(u1) > 1.0 and abs(u1[0]) < 1e-15               # still the guiding-centre step


def test_switch_on_E_over_B_and_degenerate_B(gca):
    orc = gca
    g = cart_grid(orc, 3, 8, 8.0)
    B = np.array([0.0, 1.0, 0.0])
    qm, dt = 1.0, 0.05
    u0 = np.array([0.01, 0.02, 0.0])
    orc.set_gca(10.0, 0.9)
    for e, regime in ((0.89, "gca"), (0.91, "boris")):
        E = np.array([e, 0.0, 0.0])
        u1, _ = _push_one(orc, g, E.astype(np.float32), B.astype(np.float32), u0, qm, dt)
        ub = orc.boris(u0, E.astype(np.float32).astype(np.float64), B, qm, dt)
        if regime == "boris":
            assert np.allclose(u1, ub, rtol=0, atol=1e-15)
        else:
            assert abs(u1[0]) < 1e-15 and abs(u1[2]) < 1e-15 and abs(u1[1] - ub[1]) < 1e-15
    u1, _ = _push_one(orc, g, np.float32([0.3, 0, 0]), np.float32([0, 0, 0]), u0, qm, dt)      # B = 0: conventional push
    assert np.allclose(u1, orc.boris(u0, np.float64(np.float32([0.3, 0, 0])), np.zeros(3), qm, dt), atol=1e-15)


def test_vay_gca_uses_vay_outside_the_regime(orc):
    prev = orc.set_pusher(3)
    try:
        g = cart_grid(orc, 3, 8, 8.0)
        E, B = np.array([0.1, 0.0, 0.02]), np.array([0.0, 0.3, 0.4])
        qm, dt = -1.0, 0.1
        orc.set_gca(0.5, 0.9)
        u0 = np.array([2.0, -1.0, 0.5])                                      # rho_L = 2.29 / 0.5 > 0.5: conventional
        u1, _ = _push_one(orc, g, E.astype(np.float32), B.astype(np.float32), u0, qm, dt)
        E64, B64 = E.astype(np.float32).astype(np.float64), B.astype(np.float32).astype(np.float64)
        assert np.allclose(u1, orc.vay(u0, E64, B64, qm, dt), rtol=0, atol=1e-15)
        u0 = 0.05 * u0                                                        # rho_L small: Vay, then the projection on b
        u1, _ = _push_one(orc, g, E.astype(np.float32), B.astype(np.float32), u0, qm, dt)
        b = B64 / np.linalg.norm(B64)
        uv = orc.vay(u0, E64, B64, qm, dt)
        assert np.allclose(u1, (uv @ b) * b, rtol=0, atol=1e-15)
    finally:
        orc.set_pusher(prev); orc.set_gca(0.0, 0.0)
