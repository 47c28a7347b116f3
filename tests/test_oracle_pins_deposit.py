"""Pins for the oracle's current deposit, fold and continuity checker.

What fixes the result without reference to the oracle's own formulas:
  * Eq. 6: div J + d(rho)/dt = 0 at every node, to round-off, for any move with |delta i| <= 1;
  * the geometric definition of the current of a cloud-in-cell particle: the charge that the unit cloud sweeps
    through each dual-cell face along Umeda's two straight segments (numerical quadrature, brute force);
  * sum rule sum_nodes J^d = q w dx^d / dt; time-reversal antisymmetry; additivity (no-crossing move = one
    Villasenor-Buneman segment).
"""
import itertools

import numpy as np
import pytest

from helpers import cart_grid, make_particles, qsph_grid, sph_grid, uniform_fields


def _move(orc, g, i0, d0, x_new, w=1.0, u_new=None, phi=None, phi_new=None):
    """old block at (i0, d0); new block at absolute code position x_new (periodic wrap applied)."""
    i0 = np.atleast_2d(i0); d0 = np.atleast_2d(d0); x_new = np.atleast_2d(x_new)
    n, D = i0.shape
    i1 = np.floor(x_new).astype(np.int64)
    d1 = x_new - i1
    for a in range(D):
        if g.bc[a] == orc.PERIODIC:
            i1[:, a] %= g.N[a]
    u = np.zeros((n, 3)) if u_new is None else np.atleast_2d(u_new)
    po = make_particles(orc, i0, d0, u, w=w, phi=phi)
    pn = make_particles(orc, i1, d1, u, w=w, phi=phi_new if phi_new is not None else phi)
    return po, pn


def _residual(orc, g, po, pn, q, dt):
    J = orc.zeros_current(g)
    orc.deposit(g, po, pn, J, q, dt)
    orc.fold_current(g, J)
    r0 = orc.charge_density(g, po, q); orc.fold_scalar(g, r0)
    r1 = orc.charge_density(g, pn, q); orc.fold_scalar(g, r1)
    return orc.continuity_residual(g, J, r0, r1, dt), J


@pytest.mark.parametrize("D", [2, 3])
def test_continuity_holds_to_roundoff_for_random_moves(orc, D):
    N = (6, 5, 4)[:D]
    g = cart_grid(orc, D, N, tuple(float(n) for n in N))
    rng = np.random.default_rng(10 + D)
    n = 4000
    i0 = np.stack([rng.integers(0, N[a], n) for a in range(D)], 1)
    d0 = rng.uniform(0, 1, (n, D))
    disp = rng.uniform(-0.999, 0.999, (n, D))
    xn = i0 + d0 + disp
    # keep |delta i| <= 1: always true for |disp| < 1
    w = rng.uniform(0.5, 2.0, n)
    po, pn = _move(orc, g, i0, d0, xn, w=w, u_new=rng.standard_normal((n, 3)))
    worst, J = _residual(orc, g, po, pn, -1.0, 0.37)
    scale = np.abs(w).sum() / 0.37 / np.prod(N)
    assert worst <= 1e-13 * scale * 50
    # every one of the 3^D crossing patterns occurred
    pats = set(map(tuple, (np.floor(d0 + disp)).astype(int)))
    assert len(pats) == 3 ** D


def test_continuity_single_particle_all_patterns_and_wraps(orc):
    g = cart_grid(orc, 3, (3, 3, 3), (3.0, 3.0, 3.0))
    for pat in itertools.product((-1, 0, 1), repeat=3):
        for cell in [(0, 0, 0), (2, 2, 2), (1, 0, 2)]:
            d0 = np.array([0.3, 0.6, 0.45])
            disp = np.array([{-1: -0.5, 0: 0.2, 1: 0.9}[p] for p in pat])
            po, pn = _move(orc, g, [cell], [d0], [np.array(cell) + d0 + disp], w=1.7)
            worst, J = _residual(orc, g, po, pn, 2.0, 0.5)
            assert worst < 1e-13
            # sum rule: total conformal current = q w dx / dt
            for a in range(3):
                act = J[a][2:-2, 2:-2, 2:-2]
                assert act.sum() == pytest.approx(2.0 * 1.7 * disp[a] / 0.5, abs=1e-13)


# ---------------------------------------------------------------- brute force: geometric flux through dual faces
def _tent(s):
    return np.maximum(0.0, 1.0 - np.abs(s))


def _flux_brute_force(xa, xb, shape_nodes, q_over_dt, D, nsub=64):
    """Current of a unit-cloud (CIC) particle moving xa -> relay -> xb along two straight segments (Umeda's zig-zag
    relay point in absolute coordinates).  J^a at (n_a + 1/2, n_b, n_c) = charge crossing the plane x_a = n_a + 1/2
    inside the dual-cell face of the transverse node: q * dx_a * [plane inside the cloud] * overlap(transverse).
    Integrated with 2-point Gauss on nsub sub-intervals per segment."""
    xa = np.asarray(xa, float); xb = np.asarray(xb, float)
    ia, ib = np.floor(xa), np.floor(xb)
    xr = np.minimum(np.minimum(ia, ib) + 1.0, np.maximum(np.maximum(ia, ib), 0.5 * (xa + xb)))
    J = [np.zeros(shape_nodes) for _ in range(D)]
    gp = np.array([-1.0, 1.0]) / np.sqrt(3.0)
    for (p0, p1) in ((xa, xr), (xr, xb)):
        dseg = p1 - p0
        for s in range(nsub):
            for t in ((s + 0.5 + 0.5 * gp[0]) / nsub, (s + 0.5 + 0.5 * gp[1]) / nsub):
                x = p0 + dseg * t
                wt = 0.5 / nsub
                for a in range(D):
                    if dseg[a] == 0.0:
                        continue
                    na = int(np.floor(x[a]))              # plane x_a = na + 1/2 lies inside the cloud [x-1/2, x+1/2)
                    others = [b for b in range(D) if b != a]
                    for node in itertools.product(*[range(shape_nodes[b]) for b in others]):
                        ov = 1.0
                        for b, nb in zip(others, node):
                            ov *= _tent(x[b] - nb)
                        if ov == 0.0:
                            continue
                        idx = [0] * D
                        idx[a] = na
                        for b, nb in zip(others, node):
                            idx[b] = nb
                        J[a][tuple(idx)] += q_over_dt * dseg[a] * wt * ov
    return J


@pytest.mark.parametrize("D", [2, 3])
def test_deposit_equals_the_geometric_flux_of_a_cic_cloud(orc, D):
    N = (5,) * D
    g = cart_grid(orc, D, N, tuple(float(n) for n in N), bc=(orc.ABSORB,) * D)    # no wrap: compare raw arrays
    rng = np.random.default_rng(20 + D)
    q, w, dt = -1.0, 1.3, 0.4
    for trial in range(30 if D == 3 else 60):
        i0 = rng.integers(1, 4, D)
        d0 = rng.uniform(0, 1, D)
        disp = rng.uniform(-0.95, 0.95, D)
        if trial % 5 == 0:
            disp[rng.integers(0, D)] = 0.0
        xa = i0 + d0; xb = xa + disp
        po, pn = _move(orc, g, [i0], [d0], [xb], w=w)
        J = orc.zeros_current(g)
        orc.deposit(g, po, pn, J, q, dt)
        Jb = _flux_brute_force(xa, xb, (6,) * D, q * w / dt, D)
        for a in range(D):
            got = J[a][tuple([slice(2, 8)] * D)]              # active nodes 0..5, numpy order slowest..fastest
            want = np.transpose(Jb[a])                        # brute force indexed [x1, x2, (x3)] -> transpose
            assert np.allclose(got, want, rtol=0, atol=2e-14 * abs(q * w / dt)), (trial, a)


def test_no_crossing_move_is_one_villasenor_buneman_segment(orc):
    """Additivity: with the relay at the midpoint the two half-segments add up to the single straight segment
    formula J1[s2,s3] = Q D1 [omega(W2,s2) omega(W3,s3) +- D2 D3 / 12] (textbook Villasenor-Buneman 1992)."""
    g = cart_grid(orc, 3, (4, 4, 4), (4.0, 4.0, 4.0))
    a = np.array([0.2, 0.7, 0.4]); b = np.array([0.9, 0.1, 0.55])
    po, pn = _move(orc, g, [[1, 2, 1]], [a], [np.array([1, 2, 1]) + b], w=1.0)
    J = orc.zeros_current(g)
    orc.deposit(g, po, pn, J, 1.0, 1.0)
    Dv = b - a; W = 0.5 * (a + b)
    for comp in range(3):
        t1, t2 = (comp + 1) % 3, (comp + 2) % 3
        for s1 in range(2):
            for s2 in range(2):
                om = (W[t1] if s1 else 1 - W[t1]) * (W[t2] if s2 else 1 - W[t2])
                want = Dv[comp] * (om + (1 if s1 == s2 else -1) * Dv[t1] * Dv[t2] / 12.0)
                n = [1, 2, 1]; n[t1] += s1; n[t2] += s2
                assert J[comp][n[2] + 2, n[1] + 2, n[0] + 2] == pytest.approx(want, abs=1e-15)


def test_time_reversal_antisymmetry(orc):
    g = cart_grid(orc, 3, (4, 4, 4), (4.0, 4.0, 4.0))
    rng = np.random.default_rng(31)
    n = 200
    i0 = rng.integers(0, 4, (n, 3)); d0 = rng.uniform(0, 1, (n, 3)); xn = i0 + d0 + rng.uniform(-0.9, 0.9, (n, 3))
    po, pn = _move(orc, g, i0, d0, xn)
    J1 = orc.zeros_current(g); orc.deposit(g, po, pn, J1, 1.0, 1.0); orc.fold_current(g, J1)
    J2 = orc.zeros_current(g); orc.deposit(g, pn, po, J2, 1.0, 1.0); orc.fold_current(g, J2)
    for a in range(3):
        assert np.allclose(J1[a], -J2[a], atol=1e-13)


def test_fold_is_a_periodic_sum(orc):
    """what landed in ghosts is added to the opposite active layer; afterwards ghosts mirror the active image."""
    g = cart_grid(orc, 2, (4, 3), (4.0, 3.0))
    rng = np.random.default_rng(32)
    J = [rng.standard_normal(g.padded_shape) for _ in range(3)]
    J0 = [a.copy() for a in J]
    orc.fold_current(g, J)
    for c in range(3):
        want = np.zeros((3, 4))
        for jj in range(7):
            for ii in range(8):
                want[(jj - 2) % 3, (ii - 2) % 4] += J0[c][jj, ii]
        assert np.allclose(J[c][2:5, 2:6], want, atol=1e-14)
        for jj in range(7):
            for ii in range(8):
                assert J[c][jj, ii] == pytest.approx(want[(jj - 2) % 3, (ii - 2) % 4], abs=1e-14)


def test_absorbed_and_dead_particles_deposit_nothing(orc):
    g = cart_grid(orc, 2, (4, 4), (4.0, 4.0), bc=(orc.ABSORB, orc.PERIODIC))
    po = make_particles(orc, [[3, 1], [1, 1]], [[0.9, 0.5], [0.5, 0.5]], [[0, 0, 0], [0, 0, 0]], tag=[1, 0])
    pn = make_particles(orc, [[4, 1], [1, 1]], [[0.2, 0.5], [0.7, 0.5]], [[0, 0, 0], [0, 0, 0]], tag=[0, 0])
    J = orc.zeros_current(g)
    orc.deposit(g, po, pn, J, 1.0, 1.0)
    assert all(np.all(a == 0.0) for a in J)


def test_out_of_plane_current_2d(orc):
    """G8 (unpinned by the paper beyond this): sum over nodes of J^3 = q w v3_code; equal halves on the two
    segments, bilinear weights at the segment midpoints."""
    g = cart_grid(orc, 2, (6, 6), (3.0, 3.0))
    u = np.array([0.3, -0.2, 0.9]); gam = np.sqrt(1 + u @ u)
    po, pn = _move(orc, g, [[2, 3]], [[0.8, 0.4]], [[3.1, 3.2]], w=1.5, u_new=u)
    J = orc.zeros_current(g)
    orc.deposit(g, po, pn, J, -1.0, 0.2)
    assert J[2].sum() == pytest.approx(-1.0 * 1.5 * u[2] / gam, rel=1e-14)          # h33 = 1 in 2D Cartesian
    # segment 1: (0.8,0.4)->(1.0, 0.3) in cell (2,3), midpoint (0.9, 0.35); segment 2 in cell (3,3): (0,0.3)->(0.1,0.2), midpoint (0.05,0.25)
    half = 0.5 * -1.0 * 1.5 * u[2] / gam
    assert J[2][3 + 2, 2 + 2] == pytest.approx(half * 0.1 * 0.65, rel=1e-12)
    assert J[2][3 + 2, 4 + 2] == pytest.approx(half * 0.05 * 0.75, rel=1e-12)      # node (4,3): segment 2 only
    # node (3,3) receives from both segments: seg1 weight 0.9*0.65, seg2 weight 0.95*0.75
    assert J[2][3 + 2, 3 + 2] == pytest.approx(half * (0.9 * 0.65 + 0.95 * 0.75), rel=1e-12)


def test_out_of_plane_current_axisymmetric(orc):
    """v3_code = v^phihat / sqrt(h33) at the midpoint: a particle moving purely in phi at radius r, theta:
    J^3 total = q w (v_phi / (r sin theta))."""
    g = sph_grid(orc, (20, 20), 1.0, 11.0)
    r, th = 1.0 + 7.5 * 0.5, 10.5 * np.pi / 20
    phi = 0.7
    vphi = 0.6
    gam = 1 / np.sqrt(1 - vphi ** 2)
    u = gam * vphi * np.array([-np.sin(phi), np.cos(phi), 0.0])
    po = make_particles(orc, [[7, 10]], [[0.5, 0.5]], [u], w=2.0, phi=phi)
    pn = make_particles(orc, [[7, 10]], [[0.5, 0.5]], [u], w=2.0, phi=phi)       # same place: isolates the J^3 formula
    J = orc.zeros_current(g)
    orc.deposit(g, po, pn, J, 1.0, 0.1)
    assert J[2].sum() == pytest.approx(2.0 * vphi / (r * np.sin(th)), rel=1e-13)
    assert np.all(J[0] == 0) and np.all(J[1] == 0)


@pytest.mark.parametrize("mk", ["sph", "qsph"])
def test_continuity_is_metric_free_on_curvilinear_grids(orc, mk):
    """Eq. 6 holds for the conformal current whatever the metric: full step (gather, push, move,
    back-map, deposit) of a random plasma on an axisymmetric grid, including absorbed particles."""
    g = sph_grid(orc, (24, 24), 1.0, 6.0) if mk == "sph" else qsph_grid(orc, (24, 24), 1.0, 12.0, 0.3, 0.4)
    rng = np.random.default_rng(40)
    n = 3000
    shape = g.padded_shape
    F = [0.2 * rng.standard_normal(shape).astype(np.float32) for _ in range(6)]
    i0 = np.stack([rng.integers(0, 24, n), rng.integers(0, 24, n)], 1)
    p = make_particles(orc, i0, rng.uniform(0, 1, (n, 2)), 0.8 * rng.standard_normal((n, 3)), w=rng.uniform(0.1, 3.0, n),
                       phi=rng.uniform(0, 2 * np.pi, n))
    p.tag = np.ones(n, dtype=np.int8)
    dt = 0.5 * orc.dx_min(g)
    old = p.copy()
    J = orc.zeros_current(g)
    orc.step(g, F, p, J, -1.0, 1.0, dt)
    assert (p.tag == 0).sum() > 0                 # some left through r_min / r_max
    assert (p.i[1] == 0).sum() > 0
    orc.fold_current(g, J)
    both = ((old.tag == 1) & (p.tag == 1)).astype(np.int8)
    r0 = orc.charge_density(g, old, -1.0, mask=both)
    r1 = orc.charge_density(g, p, -1.0, mask=both)
    worst = orc.continuity_residual(g, J, r0, r1, dt)
    norm = orc.charge_density(g, old, 1.0, mask=both).max() / dt
    assert worst <= 1e-12 * norm


def test_full_step_continuity_3d_cartesian(orc):
    g = cart_grid(orc, 3, (8, 8, 8), (4.0, 4.0, 4.0))
    rng = np.random.default_rng(41)
    n = 4096
    F = [0.5 * rng.standard_normal(g.padded_shape).astype(np.float32) for _ in range(6)]
    p = make_particles(orc, rng.integers(0, 8, (n, 3)), rng.uniform(0, 1, (n, 3)), rng.standard_normal((n, 3)))
    old = p.copy()
    J = orc.zeros_current(g)
    dt = 0.225
    orc.step(g, F, p, J, 1.0, 1.0, dt)
    orc.fold_current(g, J)
    r0 = orc.charge_density(g, old, 1.0); orc.fold_scalar(g, r0)
    r1 = orc.charge_density(g, p, 1.0); orc.fold_scalar(g, r1)
    worst = orc.continuity_residual(g, J, r0, r1, dt)
    assert worst <= 1e-12 * r0.max() / dt


def test_sort_check(orc):
    keys = np.array([0, 0, 1, 3, 3, 3, 5], dtype=np.int32)
    offs = np.array([0, 2, 3, 3, 6, 6, 7], dtype=np.int32)
    assert orc.sort_check(keys, 6, offs) == 0
    assert orc.sort_check(keys[::-1].copy(), 6) == 1
    bad = offs.copy(); bad[3] = 4
    assert orc.sort_check(keys, 6, bad) == 3
    assert orc.sort_check(np.array([0, 7], dtype=np.int32), 6) == 2


def test_tag_sort_is_a_stable_partition(orc):
    """N4: after the tag sort the alive particles come first and npart counts them; hand example + the properties that
    define a stable partition (same multiset, both groups in their original order)."""
    i = [[3, 1], [0, 2], [5, 5], [4, 4], [1, 1], [2, 0]]
    p = make_particles(orc, i, np.arange(12).reshape(6, 2) / 20.0, np.arange(18).reshape(6, 3) * 0.1, w=[1, 2, 3, 4, 5, 6],
                       tag=[1, 0, 0, 1, 1, 0])
    out, na = orc.compact(p)
    assert na == 3
    assert list(out.w) == [1, 4, 5, 2, 3, 6] and list(out.tag) == [1, 1, 1, 0, 0, 0]
    assert list(out.i[0]) == [3, 4, 1, 0, 5, 2] and list(out.i[1]) == [1, 4, 1, 2, 5, 0]
    assert np.allclose(out.u[2], [0.2, 1.1, 1.4, 0.5, 0.8, 1.7]) and np.allclose(out.d[1], [0.05, 0.35, 0.45, 0.15, 0.25, 0.55])
    rng = np.random.default_rng(60)
    n = 500
    tag = (rng.uniform(size=n) < 0.7).astype(np.int8)
    p = make_particles(orc, rng.integers(0, 9, (n, 3)), rng.uniform(0, 1, (n, 3)), rng.standard_normal((n, 3)), w=np.arange(n) + 1.0, tag=tag)
    out, na = orc.compact(p)
    assert na == int(tag.sum())
    assert np.array_equal(out.w[:na], p.w[tag == 1]) and np.array_equal(out.w[na:], p.w[tag == 0])
    assert np.all(out.tag[:na] == 1) and np.all(out.tag[na:] == 0)
