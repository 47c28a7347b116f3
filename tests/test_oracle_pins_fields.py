"""Pins of the oracle's field solver (N2: orc_faraday / orc_ampere, Eqs. A1, A2, 12, 13; P:127-129, P:160-167, P:360-382,
P:1040-1068) against things other than itself:
  * the exact eigenmode of the Yee leap-frog scheme in vacuum (numerical dispersion relation, textbook) on a 3D Cartesian grid
    with three different cell sizes: signs, staggering, h_ii, sqrt(h), time levels;
  * the textbook curl in spherical coordinates of analytic fields, second-order convergence, linear-r and quasi-spherical
    metrics, including the integrated form of Eq. 13 on both poles;
  * a hand value of Eq. 13 (uniform curl), A(x1) against a quadrature of sqrt(h) from the metric;
  * div B unchanged to round-off (div curl = 0 on the lattice, any metric);
  * Gauss's law carried by the charge-conserving deposit (Eq. 5 + Eq. 6): div(sqrt(h) E) - jc * conformal charge is invariant;
  * a physical one: cold-plasma oscillation of the closed loop at omega_p (sign and size of the current term, sqrt(h) != 1).
"""
import numpy as np
import pytest

from helpers import cart_grid, sph_grid, qsph_grid, make_particles

NG = 2
STAG_E = [(1, 0, 0), (0, 1, 0), (0, 0, 1)]
STAG_B = [(0, 1, 1), (1, 0, 1), (1, 1, 0)]


def zeros3(g):
    return [np.zeros(g.padded_shape, dtype=np.float64) for _ in range(3)]


def coords(g, stag):
    """code coordinates (x1, x2[, x3]) of every element of a padded array of a component with stagger `stag`, broadcastable"""
    D = g.D
    ax = []
    for d in range(D):
        a = np.arange(-NG, g.N[d] + NG, dtype=np.float64) + 0.5 * stag[d]
        shape = [1] * D
        shape[D - 1 - d] = a.size                      # x1 fastest = last numpy axis
        ax.append(a.reshape(shape))
    return ax


def lattice_slices(orc, g, stag):
    """numpy slices of the lattice points of a component (periodic: 0..N-1; otherwise N points if staggered, N+1 if not)"""
    sl = []
    for d in range(g.D):
        n = g.N[d] if g.bc[d] == orc.PERIODIC else (g.N[d] if stag[d] else g.N[d] + 1)
        sl.append(slice(NG, NG + n))
    return tuple(reversed(sl))


# ------------------------------------------------------------------------------------------------------------------
def test_vacuum_plane_wave_follows_the_yee_dispersion_relation_exactly(orc):
    """Leap-frog Yee eigenmode (textbook): with K_d = (2/dx_d) sin(k_d dx_d / 2), W = (2/dt) sin(w dt / 2): W^2 = |K|^2,
    W B0 = K x E0, K.E0 = 0; E lives at integer, B at half-integer time levels.  After M steps the oracle must sit on the
    analytic mode to round-off."""
    N, L = (12, 10, 8), (6.0, 7.0, 3.2)                 # dx = 0.5, 0.7, 0.4
    g = cart_grid(orc, 3, N, L)
    dx = np.array([L[d] / N[d] for d in range(3)])
    m = np.array([2, -1, 1])
    k = 2 * np.pi * m / np.array(L)
    K = 2.0 / dx * np.sin(0.5 * k * dx)
    dt = 0.45 * dx.min()
    W = np.sqrt((K ** 2).sum())
    w = 2.0 / dt * np.arcsin(0.5 * W * dt)
    E0 = np.cross(K, [0.3, -0.2, 0.9]); E0 /= np.linalg.norm(E0)
    B0 = np.cross(K, E0) / W

    def mode(stag, amp, t):
        x = coords(g, stag)
        ph = sum(k[d] * x[d] * dx[d] for d in range(3)) - w * t
        return amp * np.cos(ph)

    E = [mode(STAG_E[c], E0[c], 0.0) / dx[c] for c in range(3)]           # contravariant: F^c = F^hat_c / dx_c
    B = [mode(STAG_B[c], B0[c], -0.5 * dt) / dx[c] for c in range(3)]
    M = 7
    for _ in range(M):
        orc.faraday(g, E, B, dt)
        orc.fill_field_ghosts(g, E + B)
        orc.ampere(g, E, B, None, dt, 4 * np.pi)
        orc.fill_field_ghosts(g, E + B)
    for c in range(3):
        sl = lattice_slices(orc, g, STAG_E[c])
        assert np.abs(E[c] * dx[c] - mode(STAG_E[c], E0[c], M * dt))[sl].max() < 1e-12
        sl = lattice_slices(orc, g, STAG_B[c])
        assert np.abs(B[c] * dx[c] - mode(STAG_B[c], B0[c], (M - 0.5) * dt))[sl].max() < 1e-12


def test_ghost_fill_is_periodic_image_and_axis_mirror(orc):
    g = cart_grid(orc, 2, (6, 5), (3.0, 2.5))
    rng = np.random.default_rng(3)
    F = [rng.standard_normal(g.padded_shape) for _ in range(6)]
    ref = [f.copy() for f in F]
    orc.fill_field_ghosts(g, F)
    for c in range(6):
        act = ref[c][NG:-NG, NG:-NG]
        assert np.array_equal(F[c], np.pad(act, NG, mode="wrap"))
    g = sph_grid(orc, (5, 6), 1.0, 4.0)
    F = [rng.standard_normal(g.padded_shape) for _ in range(6)]
    ref = [f.copy() for f in F]
    orc.fill_field_ghosts(g, F)
    N2 = 6
    for c6 in range(6):
        stag2 = (STAG_E + STAG_B)[c6][1]
        sign = 1.0 if c6 % 3 == 0 else -1.0                                   # reading G10: r even, theta and phi odd
        col = slice(0, g.padded_shape[1])
        for gi in (1, 2):
            if stag2:      # points j + 1/2: -1/2 <-> +1/2, N2 + 1/2 <-> N2 - 1/2
                assert np.array_equal(F[c6][NG - gi, col], sign * ref[c6][NG + gi - 1, col])
                assert np.array_equal(F[c6][NG + N2 - 1 + gi, col], sign * ref[c6][NG + N2 - gi, col])
            else:          # nodes: -j <-> +j, N2 + j <-> N2 - j
                assert np.array_equal(F[c6][NG - gi, col], sign * ref[c6][NG + gi, col])
                if gi == 1:
                    assert np.array_equal(F[c6][NG + N2 + gi, col], sign * ref[c6][NG + N2 - gi, col])
        assert np.array_equal(F[c6][NG:NG + N2, :], ref[c6][NG:NG + N2, :])   # radial ghosts (ABSORB) and the lattice are left alone


# ------------------------------------------------------------------------------------------------------------------
def _geom(orc, g, stag):
    """r, theta and sqrt(h_ii) at every element of a component's padded array (2D axisymmetric)"""
    x1, x2 = coords(g, stag)
    X1, X2 = np.broadcast_arrays(x1, x2)
    h = orc.metric_h_many(g, X1.ravel(), X2.ravel()).reshape(X1.shape + (3,))
    # r and theta from the forward map of the oracle's maps module (pinned separately in test_oracle_pins_geometry)
    pts = np.stack([X1.ravel(), X2.ravel(), np.zeros(X1.size)], axis=1)
    XYZ = np.array([orc.code_to_cart(g, p) for p in pts])
    r = np.sqrt((XYZ ** 2).sum(axis=1)).reshape(X1.shape)
    th = np.arctan2(np.sqrt(XYZ[:, 0] ** 2 + XYZ[:, 1] ** 2), XYZ[:, 2]).reshape(X1.shape)
    th = np.where(X2 < 0, -th, th)
    return r, th, np.sqrt(h)


# analytic axisymmetric test fields (orthonormal components) and their textbook curl in spherical coordinates:
#   (curl F)_r = 1/(r sin th) d_th(sin th F_ph),  (curl F)_th = -1/r d_r(r F_ph),  (curl F)_ph = 1/r [d_r(r F_th) - d_th F_r]
def _F(r, th):
    return np.cos(th) / r ** 2, np.sin(th) / r, np.sin(th) / r ** 2


def _curlF(r, th):
    return 2 * np.cos(th) / r ** 3, np.sin(th) / r ** 3, np.sin(th) / r ** 3


def _curl_error(orc, g, law, skip_axis_rows=0):
    """max error of the oracle's discrete curl (orthonormal components) against the analytic one, per component"""
    src_stag, dst_stag = (STAG_E, STAG_B) if law == "faraday" else (STAG_B, STAG_E)
    src = []
    for c in range(3):
        r, th, sh = _geom(orc, g, src_stag[c])
        with np.errstate(divide="ignore", invalid="ignore"):
            v = _F(r, th)[c] / sh[..., c]
        src.append(np.ascontiguousarray(np.where(sh[..., c] > 0, v, 0.0)))
    dst = zeros3(g)
    dt = 1e-3
    if law == "faraday":
        orc.faraday(g, src, dst, dt)
        sgn = -1.0
    else:
        orc.ampere(g, dst, src, None, dt, 4 * np.pi)
        sgn = 1.0
    err = []
    N1, N2 = g.N
    for c in range(3):
        r, th, sh = _geom(orc, g, dst_stag[c])
        got = dst[c] * sh[..., c] / (sgn * dt)
        want = _curlF(r, th)[c]
        sl = list(lattice_slices(orc, g, dst_stag[c]))           # (x2 slice, x1 slice)
        if law == "ampere" and c != 0:
            sl[1] = slice(NG + 1, NG + N1)                       # tangential E on the two radial faces is not advanced
        if c == 2 and law == "ampere" or c == 1 and law == "faraday":
            sl[0] = slice(NG + 1, NG + N2)                       # E^3 / B^2 on the axis are set to zero (Eq. 12)
        if skip_axis_rows:
            sl[0] = slice(NG + skip_axis_rows, NG + N2 - skip_axis_rows)
        err.append(np.abs(got - want)[tuple(sl)].max())
    return np.array(err), dst


@pytest.mark.parametrize("kind", ["sph", "qsph-log", "qsph-stretched"])
@pytest.mark.parametrize("law", ["faraday", "ampere"])
def test_curvilinear_curl_converges_to_the_textbook_curl_at_second_order(orc, kind, law):
    """linear-r and log-r grids: second order everywhere, the E^1 axis points (Eq. 13) included.  With the theta stretch
    (vartheta != 0) the map theta(T) has theta'' != 0 at the poles, so the scheme itself is only first-order accurate in the
    rows next to the axis (a property of the discretisation, not of this code); there the test asks for second order away from
    the axis and for plain convergence next to it."""
    mk = {"sph": lambda n: sph_grid(orc, (n, n), 1.0, 3.0), "qsph-log": lambda n: qsph_grid(orc, (n, n), 1.0, 3.0, 0.3, 0.0),
          "qsph-stretched": lambda n: qsph_grid(orc, (n, n), 1.0, 3.0, 0.3, 0.35)}[kind]
    skip = 3 if kind == "qsph-stretched" else 0
    e1, _ = _curl_error(orc, mk(24), law, skip)
    e2, _ = _curl_error(orc, mk(48), law, 2 * skip)
    print(kind, law, e1, e2, e1 / e2)
    assert (e2 < 2e-2).all()
    assert (e1 / e2 > 3.0).all() and (e1 / e2 < 4.8).all()
    if skip:
        a1, _ = _curl_error(orc, mk(24), law)
        a2, _ = _curl_error(orc, mk(48), law)
        print("  with the axis rows:", a1, a2, a1 / a2)
        assert (a1 / a2 > 1.7).all()


def test_axis_rules_eq12_and_eq13_hand_values(orc):
    """B_phi = B0 r sin(theta) (curl = 2 B0 z): Eq. 13 gives dE^1 = dt B0 (1 + cos(dtheta/2)) / dr at theta = 0, minus that at
    theta = pi (hand calculation: B_3 = B0 r^2 sin^2(dtheta/2), A = r^2 dr (1 - cos(dtheta/2))); the current term is
    -dt (jc/2) J^1 / A with A checked against a quadrature of sqrt(h) from the metric; Eq. 12 zeroes E^3 and B^2 on the axis."""
    N1, N2 = 6, 8
    g = sph_grid(orc, (N1, N2), 2.0, 5.0)
    dr, dth = 3.0 / N1, np.pi / N2
    B0, dt, jc = 0.7, 0.01, 4 * np.pi
    r, th, sh = _geom(orc, g, STAG_B[2])
    B = zeros3(g)
    B[2] = np.ascontiguousarray(B0 * r * np.sin(th) / sh[..., 2])
    B[1][...] = 0.123                                                     # B^2 is not used by E^1 in 2D; Eq. 12 must zero it on the axis
    E = zeros3(g)
    E[2][...] = 5.0
    orc.ampere(g, E, B, None, dt, jc)
    want = dt * B0 * (1 + np.cos(0.5 * dth)) / dr
    assert np.allclose(E[0][NG, NG:NG + N1], want, rtol=1e-13)
    assert np.allclose(E[0][NG + N2, NG:NG + N1], -want, rtol=1e-13)
    assert np.all(E[2][NG, NG:NG + N1 + 1] == 0.0) and np.all(E[2][NG + N2, NG:NG + N1 + 1] == 0.0)
    Bz = [b.copy() for b in B]
    orc.faraday(g, zeros3(g), Bz, dt)
    assert np.all(Bz[1][NG, NG:NG + N1] == 0.0) and np.all(Bz[1][NG + N2, NG:NG + N1] == 0.0)
    assert np.all(Bz[1][NG + 1:NG + N2, NG:NG + N1] == 0.123)
    # the current term and A(x1) for both metrics
    for gg in (g, qsph_grid(orc, (N1, N2), 2.0, 5.0, 0.5, 0.4)):
        J = zeros3(gg); J[0][...] = 1.0
        E = zeros3(gg)
        orc.ampere(gg, E, zeros3(gg), J, dt, jc)
        for i in (0, 3):
            xs = (np.arange(4000) + 0.5) / 8000.0                         # midpoint rule on x2 in [0, 1/2]
            h = orc.metric_h_many(gg, np.full(xs.size, i + 0.5), xs)
            A = np.sqrt(h.prod(axis=1)).sum() / 8000.0
            assert abs(orc.axis_area(gg, i + 0.5) / A - 1) < 1e-6
            assert np.isclose(E[0][NG, NG + i], -dt * 0.5 * jc / A, rtol=1e-6)
            assert np.isclose(E[0][NG + N2, NG + i], -dt * 0.5 * jc / A, rtol=1e-6)
            # next to the axis the plain form of A2: -dt jc J / sqrt(h)
            hh = orc.metric_h(gg, [i + 0.5, 1.0, 0.0])
            assert np.isclose(E[0][NG + 1, NG + i], -dt * jc / np.sqrt(hh.prod()), rtol=1e-13)


@pytest.mark.parametrize("kind", ["cart3", "sph", "qsph"])
def test_div_B_is_unchanged_by_faraday(orc, kind):
    """div curl = 0 on the lattice for any diagonal metric: sum_d Delta_d(sqrt(h) B^d) at the cell centres keeps its value"""
    rng = np.random.default_rng(11)
    if kind == "cart3":
        g = cart_grid(orc, 3, (6, 5, 7), (3.0, 2.0, 4.2))
    else:
        g = sph_grid(orc, (7, 9), 1.0, 4.0) if kind == "sph" else qsph_grid(orc, (7, 9), 1.0, 6.0, 0.2, 0.4)
    E = [rng.standard_normal(g.padded_shape) for _ in range(3)]
    B = [rng.standard_normal(g.padded_shape) for _ in range(3)]
    if g.kind == orc.CART:
        orc.fill_field_ghosts(g, E + B)

    def sqrth(stag):
        if g.kind == orc.CART:
            return np.prod([(g.xmax[d] - g.xmin[d]) / g.N[d] for d in range(3)])
        return _geom(orc, g, stag)[2].prod(axis=-1)

    def div(Bv):
        tot = 0.0
        for d in range(g.D):
            f = sqrth(STAG_B[d]) * Bv[d]
            ax = g.D - 1 - d
            inner = tuple(slice(NG, NG + g.N[a]) for a in reversed(range(g.D)))
            tot = tot + (np.roll(f, -1, axis=ax) - f)[inner]
        return tot

    if g.kind != orc.CART:                       # Eq. 12 first, so that the comparison is between two admissible states
        orc.faraday(g, zeros3(g), B, 0.0)
    d0 = div(B)
    orc.faraday(g, E, B, 0.37)
    if g.kind == orc.CART:
        orc.fill_field_ghosts(g, E + B)
    d1 = div(B)
    scale = max(np.abs(sqrth(STAG_B[d]) * B[d]).max() for d in range(g.D))
    assert np.abs(d1 - d0).max() < 1e-12 * scale
    assert np.abs(d0).max() > 1e-3 * scale       # the check is not vacuous


@pytest.mark.parametrize("kind", ["cart3", "cart2", "sph"])
def test_gauss_law_is_carried_by_the_deposited_current(orc, kind):
    """Eq. 5 + Eq. 6: sum_d Delta_d(sqrt(h) E^d) - jc * (conformal nodal charge) is invariant under orc_ampere fed with the
    conformal currents of orc_deposit (any B: div curl = 0)."""
    rng = np.random.default_rng(5)
    n = 400
    if kind == "cart3":
        g = cart_grid(orc, 3, (6, 5, 4), (3.0, 3.5, 1.6)); D = 3
    elif kind == "cart2":
        g = cart_grid(orc, 2, (8, 6), (4.0, 4.2)); D = 2
    else:
        g = sph_grid(orc, (10, 12), 1.0, 6.0); D = 2
    lo = 2 if kind == "sph" else 0
    i0 = np.stack([rng.integers(lo, g.N[a] - lo, n) for a in range(D)], axis=1)
    d0 = rng.random((n, D))
    x1 = i0 + d0 + rng.uniform(-0.9, 0.9, (n, D))
    i1 = np.floor(x1).astype(np.int64); d1 = x1 - i1
    if kind != "sph":
        i1 = np.mod(i1, np.array(g.N[:D]))
    u = rng.standard_normal((n, 3))
    wq = rng.uniform(0.5, 2.0, n)
    phi = rng.uniform(0, 2 * np.pi, n) if kind == "sph" else None
    po = make_particles(orc, i0, d0, u, w=wq, phi=phi)
    pn = make_particles(orc, i1, d1, u, w=wq, phi=phi)
    q, dt, jc = -1.3, 0.21, 4 * np.pi
    J = orc.zeros_current(g)
    orc.deposit(g, po, pn, J, q, dt)
    orc.fold_current(g, J)
    rho0 = orc.charge_density(g, po, q); orc.fold_scalar(g, rho0)
    rho1 = orc.charge_density(g, pn, q); orc.fold_scalar(g, rho1)
    E = [rng.standard_normal(g.padded_shape) for _ in range(3)]
    B = [rng.standard_normal(g.padded_shape) for _ in range(3)]
    if kind != "sph":
        orc.fill_field_ghosts(g, E + B)

    def sqrth(stag):
        if g.kind == orc.CART:
            return np.prod([(g.xmax[d] - g.xmin[d]) / g.N[d] for d in range(D)])
        return _geom(orc, g, stag)[2].prod(axis=-1)

    def divE(Ev):
        tot = 0.0
        for d in range(D):
            f = sqrth(STAG_E[d]) * Ev[d]
            tot = tot + f - np.roll(f, 1, axis=D - 1 - d)
        return tot

    g0 = divE(E) - jc * rho0
    orc.ampere(g, E, B, J, dt, jc)
    if kind != "sph":
        orc.fill_field_ghosts(g, E + B)
    g1 = divE(E) - jc * rho1
    inner = tuple(slice(NG + 1, NG + g.N[a] - 1) for a in reversed(range(D))) if kind == "sph" else \
        tuple(slice(NG, NG + g.N[a]) for a in reversed(range(D)))
    scale = jc * np.abs(rho1).max()
    assert np.abs(g1 - g0)[inner].max() < 1e-11 * scale
    assert np.abs(jc * (rho1 - rho0))[inner].max() > 1e-2 * scale       # the charge did move


# ------------------------------------------------------------------------------------------------------------------
def test_cold_plasma_oscillates_at_the_plasma_frequency(orc):
    """The closed loop (sub-steps 2-11 of P:127-167) on a 2D Cartesian box with dx = 0.5: cold electrons on a neutralising
    background, velocity perturbation u_x = u0 sin(k x).  E_x must oscillate at omega_p^2 = jc n0 q^2 / m with
    n0 = (particles per cell * w) / (dx dy) -- the sign of the current term, its size and the 1/sqrt(h) in front of it.
    Leap-frog: sin(w dt / 2) = w_p dt / 2 up to O((k dx)^2) grid corrections."""
    N, dx = (32, 4), 0.5
    g = cart_grid(orc, 2, N, (N[0] * dx, N[1] * dx))
    ppc_side = 4
    sub = (np.arange(ppc_side) + 0.5) / ppc_side
    ii, jj, a, b = np.meshgrid(np.arange(N[0]), np.arange(N[1]), sub, sub, indexing="ij")
    n = ii.size
    i = np.stack([ii.ravel(), jj.ravel()], axis=1)
    d = np.stack([a.ravel(), b.ravel()], axis=1)
    q, m, w, jc = -1.0, 1.0, 0.002, 4 * np.pi
    n0 = ppc_side ** 2 * w / dx ** 2
    wp = np.sqrt(jc * n0 * q * q / m)
    dt = 0.1 / wp * 2.0                                   # w_p dt = 0.2
    assert dt < 0.45 * dx
    k = 2 * np.pi / (N[0] * dx)
    u = np.zeros((n, 3)); u[:, 0] = 1e-3 * np.sin(k * (i[:, 0] + d[:, 0]) * dx)
    p = make_particles(orc, i, d, u, w=w)
    E, B = zeros3(g), zeros3(g)
    amp = []
    x_e1 = (np.arange(N[0]) + 0.5) * dx
    steps = int(round(2.5 * 2 * np.pi / (wp * dt)))
    for _ in range(steps):
        orc.faraday(g, E, B, 0.5 * dt)
        orc.fill_field_ghosts(g, E + B)
        F = [np.ascontiguousarray(f.astype(np.float32)) for f in E + B]
        J = orc.zeros_current(g)
        orc.step(g, F, p, J, q, m, dt)
        orc.fold_current(g, J)
        orc.faraday(g, E, B, 0.5 * dt)
        orc.ampere(g, E, B, J, dt, jc)
        ex = E[0][NG:NG + N[1], NG:NG + N[0]].mean(axis=0) * dx          # orthonormal E_x(x)
        amp.append(2.0 * (ex * np.sin(k * x_e1)).mean())
    amp = np.array(amp)
    t = (np.arange(steps) + 1) * dt
    # frequency from the zero crossings of the mode amplitude
    s = np.sign(amp)
    zc = np.where(s[1:] * s[:-1] < 0)[0]
    tz = t[zc] - amp[zc] * (t[zc + 1] - t[zc]) / (amp[zc + 1] - amp[zc])
    assert len(tz) >= 4
    w_meas = np.pi / np.diff(tz).mean()
    w_scheme = 2.0 / dt * np.arcsin(0.5 * wp * dt)
    print("omega_p", wp, "scheme", w_scheme, "measured", w_meas, "amplitude", np.abs(amp).max())
    assert abs(w_meas / w_scheme - 1) < 0.02
    # bounded oscillation (a wrong sign of the current term grows exponentially): last maximum ~ first maximum
    half = len(amp) // 2
    assert np.abs(amp[half:]).max() < 1.2 * np.abs(amp[:half]).max()
    # and the size: E_max = u0 m w_p / |q| (energy exchange between the flow and the field)
    assert abs(np.abs(amp).max() / (1e-3 * m * w_scheme / abs(q)) - 1) < 0.05
