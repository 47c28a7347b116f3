"""Physics pins of the oracle's closed loop (sub-steps 2-11 of P:127-167) against linear theory the paper itself quotes
(sect. 5.1.1): the growth rate of the relativistic two-stream instability, Eq. 14, and of the current-filamentation
(Weibel) mode whose short-wavelength limit is P:849.  A wrong time level in the push, move or deposit, a missing gamma^3, a wrong
sign or factor between deposit and Ampere, or a wrong out-of-plane current (reading G8) moves these rates by far more than the bars.

Small boxes (two / three wavelengths of the seeded mode, quiet start on a regular lattice) keep the runs at a few seconds each."""
import math

import numpy as np

from helpers import cart_grid, make_particles

NG = 2


def _beams(orc, N, dx, ub, eps, k, w, side, axis):
    sub = (np.arange(side) + 0.5) / side
    ii, jj, a, b = np.meshgrid(np.arange(N[0]), np.arange(N[1]), sub, sub, indexing="ij")
    i = np.stack([ii.ravel(), jj.ravel()], axis=1)
    d = np.stack([a.ravel(), b.ravel()], axis=1)
    x = (i[:, 0] + d[:, 0]) * dx
    out = []
    for sign in (+1.0, -1.0):
        u = np.zeros((i.shape[0], 3))
        u[:, axis] = sign * ub + eps * np.sin(k * x)
        out.append(make_particles(orc, i, d, u, w=w))
    return out


def _loop(orc, g, beams, dt, jc, steps, comp, mode):
    N = g.N
    E = [np.zeros(g.padded_shape) for _ in range(3)]
    B = [np.zeros(g.padded_shape) for _ in range(3)]
    amp = np.zeros(steps)
    for s in range(steps):
        orc.faraday(g, E, B, 0.5 * dt)
        orc.fill_field_ghosts(g, E + B)
        F = [np.ascontiguousarray(f.astype(np.float32)) for f in E + B]
        J = orc.zeros_current(g)
        for p in beams:
            orc.step(g, F, p, J, -1.0, 1.0, dt)
        orc.fold_current(g, J)
        orc.faraday(g, E, B, 0.5 * dt)
        orc.ampere(g, E, B, J, dt, jc)
        row = (E + B)[comp][NG:NG + N[1], NG:NG + N[0]].mean(axis=0)
        amp[s] = np.abs(np.fft.rfft(row)[mode]) * 2.0 / N[0]
    return amp


def _rate(A, t):
    isat = int(np.argmax(A))
    lo = np.where(A[:isat] >= 1e-3 * A[isat])[0][0]
    hi = np.where(A[:isat] >= 1e-1 * A[isat])[0][0]
    assert hi - lo > 50, "no clean linear phase"
    return np.polyfit(t[lo:hi], np.log(A[lo:hi]), 1)[0]


def test_two_stream_instability_grows_at_the_rate_of_eq14(orc):
    """Eq. 14: 1 = a [ (w - k v)^-2 + (w + k v)^-2 ], a = w_p^2 / (2 gamma_b^3)  =>  (w^2 - K)^2 = 2 a (w^2 + K), K = k^2 v_b^2,
    Gamma^2 = sqrt(a^2 + 4 a K) - a - K; the seeded mode sits at the maximum Gamma_max = w_p / (2 gamma_b)^(3/2)."""
    N, dx, mode = (108, 2), 1.0, 2
    g = cart_grid(orc, 2, N, (N[0] * dx, N[1] * dx))
    wp, ub, jc, side = 0.1, 0.5, 4.0 * math.pi, 4
    gam = math.sqrt(1.0 + ub * ub); vb = ub / gam
    dt = 0.45 * dx
    w = wp * wp * dx * dx / (jc * 2 * side * side)          # w_p^2 = jc n q^2 / m with n = 2 side^2 w / dx^2
    k = 2.0 * math.pi * mode / (N[0] * dx)
    a = wp * wp / (2.0 * gam ** 3); K = (k * vb) ** 2
    Gamma = math.sqrt(math.sqrt(a * a + 4.0 * a * K) - a - K)
    assert abs(Gamma / (wp / (2.0 * gam) ** 1.5) - 1.0) < 0.01
    steps = int(round(70.0 / (wp * dt)))
    A = _loop(orc, g, _beams(orc, N, dx, ub, 1e-5, k, w, side, 0), dt, jc, steps, 0, mode)
    slope = _rate(A, (np.arange(steps) + 1) * dt)
    print(f"oracle two-stream: Gamma(Eq. 14) = {Gamma:.5f}, measured {slope:.5f} ({slope / Gamma - 1:+.2%})")
    assert abs(slope / Gamma - 1.0) < 0.02
    assert 0.02 < A.max() / wp < 2.0                        # trapping amplitude e E / (m w_p c) = O(0.1 .. 1)


def test_filamentation_instability_grows_at_the_linear_rate(orc):
    """beams along +-z, k along x: w^4 - w^2 (k^2 + w_p^2 / gamma_b^3) - w_p^2 k^2 v_b^2 / gamma_b = 0 (cold two-beam linear theory;
    its k -> infinity limit is the paper's Gamma_max = v_b w_p / gamma_b^(1/2)), k taken as the Yee curl sees it."""
    N, dx, mode = (132, 2), 1.0, 3
    g = cart_grid(orc, 2, N, (N[0] * dx, N[1] * dx))
    wp, ub, jc, side = 0.1, 0.5, 4.0 * math.pi, 4
    gam = math.sqrt(1.0 + ub * ub); vb = ub / gam
    dt = 0.45 * dx
    w = wp * wp * dx * dx / (jc * 2 * side * side)
    k = 2.0 * math.pi * mode / (N[0] * dx)
    kg = 2.0 / dx * math.sin(0.5 * k * dx)
    b = kg * kg + wp * wp / gam ** 3
    Gamma = math.sqrt(0.5 * (math.sqrt(b * b + 4.0 * wp * wp * kg * kg * vb * vb / gam) - b))
    assert 0.8 < Gamma / (vb * wp / math.sqrt(gam)) < 1.0
    steps = int(round(50.0 / (wp * dt)))
    A = _loop(orc, g, _beams(orc, N, dx, ub, 1e-5, k, w, side, 2), dt, jc, steps, 4, mode)
    slope = _rate(A, (np.arange(steps) + 1) * dt)
    print(f"oracle filamentation: Gamma(linear theory) = {Gamma:.5f}, measured {slope:.5f} ({slope / Gamma - 1:+.2%})")
    assert abs(slope / Gamma - 1.0) < 0.03
