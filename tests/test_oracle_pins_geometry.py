"""Pins for the oracle's metric, coordinate maps, gather and basis change.

Each test checks the oracle against something the paper or the mathematics fixes, never against a
retyped copy of its own formula: the metric must be the one induced by the embedding code->Cartesian
(finite-difference Jacobian of the forward map), the basis change must be that Jacobian applied to the
contravariant components, maps must round-trip, the cubic inverse must agree with a bisection root.
"""
import numpy as np
import pytest

from helpers import cart_grid, qsph_grid, sph_grid


def _grids(orc):
    return [
        cart_grid(orc, 2, (16, 24), (8.0, 6.0)),
        cart_grid(orc, 3, (8, 12, 10), (4.0, 3.0, 7.5)),
        sph_grid(orc, (32, 48), 1.0, 10.0),
        qsph_grid(orc, (32, 48), 1.0, 20.0, 0.0, 0.0),
        qsph_grid(orc, (32, 48), 1.5, 50.0, 1.0, 0.4),       # Fig. 2 parameters r0 = (2/3) rmin, vartheta = 0.4
        qsph_grid(orc, (32, 48), 1.0, 50.0, 0.0, 0.9),
    ]


def _random_code_point(g, rng):
    x = np.array([rng.uniform(0.05, g.N[0] - 0.05), rng.uniform(0.05, g.N[1] - 0.05), 0.0])
    if g.axisym:
        x[2] = rng.uniform(0, 2 * np.pi)
    elif g.D == 3:
        x[2] = rng.uniform(0.05, g.N[2] - 0.05)
    return x


def _jacobian(orc, g, x, eps=1e-5):
    Jm = np.zeros((3, 3))
    for a in range(3):
        xp = x.copy(); xm = x.copy(); xp[a] += eps; xm[a] -= eps
        Jm[:, a] = (orc.code_to_cart(g, xp) - orc.code_to_cart(g, xm)) / (2 * eps)
    return Jm


def test_metric_is_induced_by_the_embedding(orc):
    """h_ij = dX/dx^i . dX/dx^j for the forward maps of P:271-315; diagonal."""
    rng = np.random.default_rng(1)
    for g in _grids(orc):
        for _ in range(25):
            x = _random_code_point(g, rng)
            Jm = _jacobian(orc, g, x)
            G = Jm.T @ Jm
            h = orc.metric_h(g, x)
            for a in range(3):
                if g.kind == orc.CART and a >= g.D:
                    assert h[a] == 1.0            # P:229 "1 for 1D/2D"
                    continue
                assert G[a, a] == pytest.approx(h[a], rel=2e-7), (g.kind, a)
                for b in range(a):
                    assert abs(G[a, b]) <= 1e-6 * np.sqrt(G[a, a] * G[b, b]) + 1e-12


def test_qsph_reduces_to_log_spherical(orc):
    """R = log(r - r0); with r0 = 0, vartheta = 0 the grid is r = rmin (rmax/rmin)^(x1/N), theta = pi x2/N."""
    g = qsph_grid(orc, (40, 20), 1.0, 20.0, 0.0, 0.0)
    for x1, x2 in [(0.0, 10.0), (13.25, 3.5), (40.0, 19.0)]:
        X = orc.code_to_cart(g, [x1, x2, 0.0])
        r = np.hypot(X[0], X[2])
        assert r == pytest.approx(20.0 ** (x1 / 40.0), rel=1e-13)
        assert np.arctan2(X[0], X[2]) == pytest.approx(np.pi * x2 / 20.0, rel=1e-13)
        h = orc.metric_h(g, [x1, x2, 0.0])
        assert np.sqrt(h[0]) == pytest.approx(r * np.log(20.0) / 40.0, rel=1e-13)     # dr/dx1 = r dR
        assert np.sqrt(h[1]) == pytest.approx(r * np.pi / 20.0, rel=1e-13)


def test_dtheta_dT_is_the_derivative_of_theta(orc):
    for vt in [0.0, 0.1, 0.4, 0.9]:
        for T in np.linspace(0.05, 3.09, 17):
            fd = (orc.theta_of_T(vt, T + 1e-6) - orc.theta_of_T(vt, T - 1e-6)) / 2e-6
            assert orc.dtheta_dT(vt, T) == pytest.approx(fd, abs=1e-9)
    # end points and equator are fixed points of the stretch: theta(0)=0, theta(pi/2)=pi/2, theta(pi)=pi
    for vt in [0.1, 0.4]:
        assert orc.theta_of_T(vt, 0.0) == 0.0
        assert orc.theta_of_T(vt, np.pi / 2) == pytest.approx(np.pi / 2, abs=1e-15)
        assert orc.theta_of_T(vt, np.pi) == pytest.approx(np.pi, abs=1e-15)


def test_dx_min_matches_the_paper_statement(orc):
    """2D Cartesian with dx = dy gives dx_min = dx / sqrt(2); 3D gives dx / sqrt(3)."""
    assert orc.dx_min(cart_grid(orc, 2, (8, 8), (4.0, 4.0))) == pytest.approx(0.5 / np.sqrt(2), rel=1e-14)
    assert orc.dx_min(cart_grid(orc, 3, (4, 4, 4), (2.0, 2.0, 2.0))) == pytest.approx(0.5 / np.sqrt(3), rel=1e-14)
    # spherical: "determined by the size of the smallest cell" -> innermost ring next to the axis
    g = sph_grid(orc, (16, 16), 1.0, 5.0)
    h = orc.metric_h(g, [0.5, 0.5, 0.0])
    assert orc.dx_min(g) == pytest.approx((1 / h[0] + 1 / h[1]) ** -0.5, rel=1e-14)


def test_maps_round_trip(orc):
    """forward o backward = identity, phi in [0, 2 pi), theta in [0, pi]."""
    rng = np.random.default_rng(2)
    for g in _grids(orc):
        for _ in range(200):
            x = _random_code_point(g, rng)
            X = orc.code_to_cart(g, x)
            x2 = orc.cart_to_code(g, X)
            assert np.allclose(x2, x, rtol=0, atol=2e-12 * max(1.0, np.abs(x).max()))
            if g.axisym:
                assert 0.0 <= x2[2] < 2 * np.pi
                assert 0.0 <= x2[1] <= g.N[1]


def test_backward_map_special_directions(orc):
    g = sph_grid(orc, (10, 10), 1.0, 11.0)
    # on the +z axis theta = 0, on -z theta = pi; +x axis phi = 0, +y phi = pi/2, -x phi = pi, -y phi = 3 pi / 2
    assert orc.cart_to_code(g, [0, 0, 2.0])[1] == pytest.approx(0.0, abs=1e-15)
    assert orc.cart_to_code(g, [0, 0, -2.0])[1] == pytest.approx(10.0, abs=1e-14)
    for X, phi in [([2, 0, 0], 0.0), ([0, 2, 0], np.pi / 2), ([-2, 0, 0], np.pi), ([0, -2, 0], 1.5 * np.pi)]:
        x = orc.cart_to_code(g, X)
        assert x[2] == pytest.approx(phi, abs=1e-15)
        assert x[0] == pytest.approx(1.0, abs=1e-14)      # r = 2 -> (2 - 1) / 1
        assert x[1] == pytest.approx(5.0, abs=1e-14)


def test_cubic_inverse_against_bisection_and_B3(orc):
    """App. B: T(theta).  Brute-force bisection root of theta(T) - theta; B3 with the corrected radicand
    agrees, B3 exactly as extracted does not."""
    for vt in [0.01, 0.1, 0.4, 0.9]:
        worst_printed = 0.0
        for theta in np.linspace(0.0, np.pi, 41):
            lo, hi = 0.0, np.pi
            for _ in range(200):
                mid = 0.5 * (lo + hi)
                if orc.theta_of_T(vt, mid) < theta: lo = mid
                else: hi = mid
            root = 0.5 * (lo + hi)
            assert orc.T_of_theta(vt, theta) == pytest.approx(root, abs=5e-15 * np.pi + 1e-15)
            assert orc.T_of_theta_printed_B3(vt, theta) == pytest.approx(root, abs=1e-11)
            p = orc.T_of_theta_printed_B3(-vt, theta)
            worst_printed = max(worst_printed, 9.0 if np.isnan(p) else abs(p - root))
        assert worst_printed > 1e-2          # the printed radicand is not the inverse
    assert orc.T_of_theta(0.0, 1.234) == 1.234   # identity when vartheta = 0


# ------------------------------------------------------------------ gather (O2)
def _padded(orc, g, fn, stag):
    """Fill a padded fp32 array with fn evaluated at the component's own lattice points (index + stagger)."""
    shape = g.padded_shape
    D = g.D
    idx = np.meshgrid(*[np.arange(s, dtype=np.float64) - orc.NGHOST for s in shape], indexing="ij")   # slowest..fastest
    coords = list(reversed(idx))       # coords[0] is x1 (fastest)
    pos = [coords[a] + 0.5 * stag[a] for a in range(D)]
    return np.ascontiguousarray(fn(*pos), dtype=np.float32)


STAG = [(1, 0, 0), (0, 1, 0), (0, 0, 1), (0, 1, 1), (1, 0, 1), (1, 1, 0)]    # Yee


@pytest.mark.parametrize("D", [2, 3])
def test_gather_reproduces_linear_fields_exactly(orc, D):
    """Multilinear interpolation on each component's own staggered lattice reproduces any field that is
    linear in code coordinates (and constants: the weights sum to one)."""
    g = cart_grid(orc, D, (6, 5, 4)[:D], (6.0, 5.0, 4.0)[:D])
    rng = np.random.default_rng(3)
    coef = rng.integers(-4, 5, size=(6, 4)).astype(np.float64) / 4.0        # exactly representable in fp32
    F = []
    for c in range(6):
        a = coef[c]
        if D == 3:
            F.append(_padded(orc, g, lambda x, y, z: a[0] + a[1] * x + a[2] * y + a[3] * z, STAG[c]))
        else:
            F.append(_padded(orc, g, lambda x, y: a[0] + a[1] * x + a[2] * y, STAG[c]))
    for _ in range(200):
        i = [int(rng.integers(0, g.N[a])) for a in range(D)]
        d = rng.uniform(0, 1, size=D)
        if rng.uniform() < 0.3:
            d[rng.integers(0, D)] = rng.choice([0.0, 0.5, 0.25])
        out = orc.gather(g, F, i, d)
        for c in range(6):
            a = coef[c]
            x = [i[k] + d[k] for k in range(D)]
            want = a[0] + sum(a[1 + k] * x[k] for k in range(D))
            assert out[c] == pytest.approx(want, abs=1e-13)


def test_gather_on_a_stagger_point_returns_the_element(orc):
    g = cart_grid(orc, 3, (5, 5, 5), (5.0, 5.0, 5.0))
    rng = np.random.default_rng(4)
    F = [rng.standard_normal(g.padded_shape).astype(np.float32) for _ in range(6)]
    i = [2, 3, 1]
    for c in range(6):
        d = [0.5 if STAG[c][a] else 0.0 for a in range(3)]
        out = orc.gather(g, F, i, d)
        assert out[c] == float(F[c][i[2] + 2, i[1] + 2, i[0] + 2])
    # 2D: no third index at all
    g2 = cart_grid(orc, 2, (5, 4), (5.0, 4.0))
    F2 = [rng.standard_normal(g2.padded_shape).astype(np.float32) for _ in range(6)]
    for c in range(6):
        d = [0.5 if STAG[c][a] else 0.0 for a in range(2)]
        assert orc.gather(g2, F2, [1, 2], d)[c] == float(F2[c][2 + 2, 1 + 2])


def test_gather_stencil_footprint(orc):
    """A delta function at one lattice point is seen only by particles within one lattice spacing of it, with
    the tent weight: pins base-index and weight selection per stagger."""
    g = cart_grid(orc, 2, (8, 8), (8.0, 8.0))
    for c in range(6):
        F = [np.zeros(g.padded_shape, dtype=np.float32) for _ in range(6)]
        F[c][3 + 2, 4 + 2] = 1.0                # lattice point (i=4, j=3) + stagger
        px, py = 4 + 0.5 * STAG[c][0], 3 + 0.5 * STAG[c][1]
        for x, y in [(4.2, 3.1), (3.6, 3.9), (4.9, 2.7), (5.6, 3.0), (4.0, 4.6), (2.9, 3.0)]:
            i = [int(np.floor(x)), int(np.floor(y))]
            out = orc.gather(g, F, i, [x - i[0], y - i[1]])
            want = max(0.0, 1 - abs(x - px)) * max(0.0, 1 - abs(y - py))
            assert out[c] == pytest.approx(want, abs=1e-15)


# ------------------------------------------------------------------ basis change (O3)
def test_basis_change_is_the_jacobian_of_the_forward_map(orc):
    """A contravariant vector transforms with dX/dx^i: A^X = sum_i A^i dX/dx^i (P:76-81 + P:287-289)."""
    rng = np.random.default_rng(5)
    for g in _grids(orc):
        for _ in range(20):
            x = _random_code_point(g, rng)
            A = rng.standard_normal(3)
            Jm = _jacobian(orc, g, x)
            want = Jm @ A
            got = orc.to_cartesian_basis(g, x, A)
            assert np.allclose(got, want, rtol=0, atol=3e-7 * np.linalg.norm(want) + 1e-12)


def test_basis_change_preserves_invariants(orc):
    rng = np.random.default_rng(6)
    g = qsph_grid(orc, (32, 32), 1.0, 30.0, 0.5, 0.3)
    for _ in range(20):
        x = _random_code_point(g, rng)
        E, B = rng.standard_normal(3), rng.standard_normal(3)
        h = orc.metric_h(g, x)
        Eo, Bo = np.sqrt(h) * E, np.sqrt(h) * B
        Ec, Bc = orc.to_cartesian_basis(g, x, E), orc.to_cartesian_basis(g, x, B)
        assert Ec @ Ec == pytest.approx(Eo @ Eo, rel=1e-13)
        assert Bc @ Bc == pytest.approx(Bo @ Bo, rel=1e-13)
        assert Ec @ Bc == pytest.approx(Eo @ Bo, rel=1e-12, abs=1e-14)
    gc = cart_grid(orc, 2, (10, 10), (5.0, 2.5))
    assert np.allclose(orc.to_cartesian_basis(gc, [1.0, 1.0, 0.0], [1.0, 1.0, 1.0]), [0.5, 0.25, 1.0])   # E^xhat = dx E^1
