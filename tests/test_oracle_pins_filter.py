"""Pins for the oracle's current filter + J = conformal J / sqrt(h) (Eqs. 9-11).

What fixes the result independently of the oracle's loops:
  * Eqs. 9-11 are the tensor product of the 1D kernel (1/4, 1/2, 1/4): a constant is invariant, the sum over a periodic box is
    preserved, a Fourier mode cos(k.x) is multiplied by prod_d cos^2(k_d / 2) per pass (the transfer function of that kernel);
  * the axis rules of P:386 on a hand-computed 1D-in-theta example (even J^1, odd J^2, J^3 = 0 on the axis);
  * J^i = conformal J^i / sqrt(h) with sqrt(h) = |det of the Jacobian of the forward map| by finite differences.
"""
import numpy as np
import pytest

from helpers import cart_grid, sph_grid, qsph_grid


def test_constant_is_invariant_and_sum_is_preserved_periodic(orc):
    for D, N in ((2, (6, 5)), (3, (5, 4, 6))):
        g = cart_grid(orc, D, N, tuple(float(n) for n in N))
        rng = np.random.default_rng(50 + D)
        J = [np.full(g.padded_shape, 1.7) for _ in range(3)]
        orc.filter_current(g, J, 3)
        act = tuple([slice(2, -2)] * D)
        for c in range(3):
            assert np.allclose(J[c][act], 1.7, atol=1e-14)
        J = [rng.standard_normal(g.padded_shape) for _ in range(3)]
        s0 = [j[act].sum() for j in J]
        orc.filter_current(g, J, 2)
        for c in range(3):
            assert J[c][act].sum() == pytest.approx(s0[c], abs=1e-12)


def test_fourier_mode_is_damped_by_cos2_of_half_k_per_pass(orc):
    N = (16, 12, 8)
    g = cart_grid(orc, 3, N, tuple(float(n) for n in N))
    m = (3, 2, 1)
    k = [2 * np.pi * m[a] / N[a] for a in range(3)]
    z, y, x = np.meshgrid(np.arange(N[2]), np.arange(N[1]), np.arange(N[0]), indexing="ij")
    mode = np.cos(k[0] * x + k[1] * y + k[2] * z + 0.3)
    for npass in (1, 4):
        J = [np.zeros(g.padded_shape) for _ in range(3)]
        for c in range(3):
            J[c][2:-2, 2:-2, 2:-2] = (c + 1) * mode
        orc.filter_current(g, J, npass)
        fac = np.prod([np.cos(0.5 * kk) ** 2 for kk in k]) ** npass
        for c in range(3):
            assert np.allclose(J[c][2:-2, 2:-2, 2:-2], (c + 1) * fac * mode, atol=1e-13)


def test_axis_rules_hand_example(orc):
    """SPH grid, currents uniform in x1 far from the radial edges, so that the x1 convolution is the identity there and the
    theta convolution can be written by hand: J^1(j=0) -> 1/2 J^1(0) + 1/4 (J^1(1) + J^1(1)) (even image), J^2(j=1/2) ->
    1/2 J^2(1/2) + 1/4 (J^2(3/2) - J^2(1/2)) (odd image), J^3(j=0) = 0 and J^3(1) -> 1/2 J^3(1) + 1/4 (0 + J^3(2))."""
    g = sph_grid(orc, (12, 6), 1.0, 7.0)
    N1, N2 = 12, 6
    a1 = np.array([3.0, 1.0, 4.0, 1.0, 5.0, 9.0, 2.0])       # J^1 at nodes j = 0..6
    a2 = np.array([2.0, 7.0, 1.0, 8.0, 2.0, 8.0])            # J^2 at j + 1/2, j = 0..5
    a3 = np.array([5.0, 6.0, 5.0, 3.0, 5.0, 8.0, 9.0])       # J^3 at nodes j = 0..6 (axis values must be zeroed)
    J = [np.zeros(g.padded_shape) for _ in range(3)]
    J[0][2:2 + N2 + 1, 2:2 + N1] = a1[:, None]
    J[1][2:2 + N2, 2:2 + N1 + 1] = a2[:, None]
    J[2][2:2 + N2 + 1, 2:2 + N1 + 1] = a3[:, None]
    orc.filter_current(g, J, 1)
    col = 2 + 6                                              # x1 index 6: three cells from either radial edge
    e1 = np.concatenate([[a1[1]], a1, [a1[-2]]])             # even images at both axes
    want1 = 0.25 * e1[:-2] + 0.5 * e1[1:-1] + 0.25 * e1[2:]
    assert np.allclose(J[0][2:2 + N2 + 1, col], want1, atol=1e-14)
    e2 = np.concatenate([[-a2[0]], a2, [-a2[-1]]])           # odd images
    want2 = 0.25 * e2[:-2] + 0.5 * e2[1:-1] + 0.25 * e2[2:]
    assert np.allclose(J[1][2:2 + N2, col], want2, atol=1e-14)
    b3 = a3.copy(); b3[0] = b3[-1] = 0.0                     # J^3 = 0 on the axis: as input of the stencil and as result
    want3 = np.zeros(N2 + 1)
    want3[1:-1] = 0.25 * b3[:-2] + 0.5 * b3[1:-1] + 0.25 * b3[2:]
    assert np.allclose(J[2][2:2 + N2 + 1, col], want3, atol=1e-14)
    # absorbing radial side: values beyond the lattice count as zero (reading G20): first J^3 column keeps 1/2 + 1/4 of a uniform row
    assert J[2][2 + 3, 2] == pytest.approx((0.5 + 0.25) * want3[3], rel=1e-14)


@pytest.mark.parametrize("mk", ["cart", "sph", "qsph"])
def test_division_by_sqrt_h_at_each_component_position(orc, mk):
    """J^i = conformal J^i / sqrt(h) at the component's own Yee position; sqrt(h) = |det d(X,Y,Z)/d(x1,x2,phi)| of the
    forward map by central differences (Cartesian 3D: the cell volume)."""
    if mk == "cart":
        g = cart_grid(orc, 3, (4, 5, 3), (2.0, 10.0, 0.75))
        J = [np.ones(g.padded_shape) for _ in range(3)]
        orc.filter_current(g, J, 0, divide=True)
        vol = 0.5 * 2.0 * 0.25
        for c in range(3):
            assert np.allclose(J[c][2:-2, 2:-2, 2:-2], 1.0 / vol, rtol=1e-14)
        return
    g = sph_grid(orc, (8, 8), 1.0, 5.0) if mk == "sph" else qsph_grid(orc, (8, 8), 1.0, 9.0, 0.3, 0.4)
    J = [np.ones(g.padded_shape) for _ in range(3)]
    orc.filter_current(g, J, 0, divide=True)

    def sqrt_h_fd(x1, x2):
        eps = 1e-6
        cols = []
        for a in range(3):
            xp = np.array([x1, x2, 0.4]); xm = xp.copy()
            xp[a] += eps; xm[a] -= eps
            cols.append((orc.code_to_cart(g, xp) - orc.code_to_cart(g, xm)) / (2 * eps))
        return abs(np.linalg.det(np.stack(cols, 1)))
    for (c, i, j, x1, x2) in [(0, 3, 2, 3.5, 2.0), (1, 3, 2, 3.0, 2.5), (2, 3, 2, 3.0, 2.0), (0, 7, 7, 7.5, 7.0), (1, 0, 0, 0.0, 0.5)]:
        assert J[c][2 + j, 2 + i] == pytest.approx(1.0 / sqrt_h_fd(x1, x2), rel=1e-7)
    # on the axis sqrt(h) = 0: the conformal value is kept (J^3 = 0 by Eq. 12; E^1 uses Eq. 13 with the conformal current)
    assert J[0][2 + 0, 2 + 3] == 1.0 and J[0][2 + 8, 2 + 3] == 1.0
