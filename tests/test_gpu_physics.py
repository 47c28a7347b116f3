"""Physics check of the closed loop on the GPU (no oracle involved): the relativistic two-stream instability of sect. 5.1.1.

Two cold counter-streaming electron beams (u_b = +-0.5, densities n_b / 2) on a neutralising background, quasi-1D (2D box, 16 cells in
y), every call of the loop through the C ABI: ent_faraday (half), ent_step_pair on re-binned blocks, ent_fold_current, ent_faraday
(half), ent_ampere, ghost fill.  The mode that is seeded must grow at the rate Eq. 14 gives for its wavenumber,

    (w^2 - k^2 v_b^2)^2 = 2 a (w^2 + k^2 v_b^2),   a = w_p^2 / (2 gamma_b^3)
    =>  Gamma^2 = sqrt(a^2 + 4 a k^2 v_b^2) - a - k^2 v_b^2,      Gamma_max = w_p / (2 gamma_b)^(3/2)

which is sensitive to everything the parity tests check piecewise: the sign and size of the current term, the time centring of push,
move and deposit, the relativistic factor in the push (gamma_b^3), the gather, the field solver and the unit conventions between
them (w_p^2 = j_coeff n q^2 / m)."""
import math

import numpy as np
import pytest
import torch

import parity as P

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    from paper_2511_17710_b200 import binding as bind, synth
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: there is no CPU fallback for the product path")
    ctx = bind.ent_create(0, None)
    yield bind, synth, ctx
    bind.ent_destroy(ctx)


def _beam(synth, g, sign, ub, eps, k, w, side, axis=0):
    """quiet start: side x side particles on a regular lattice in every cell, u_axis = sign u_b + eps sin(k x)"""
    Nx, Ny = g.N
    sub = (torch.arange(side, dtype=torch.float64) + 0.5) / side
    ii, jj, a, b = torch.meshgrid(torch.arange(Nx, dtype=torch.float64), torch.arange(Ny, dtype=torch.float64), sub, sub, indexing="ij")
    ii, jj, a, b = ii.reshape(-1), jj.reshape(-1), a.reshape(-1), b.reshape(-1)
    n = ii.numel()
    dx = (g.xmax[0] - g.xmin[0]) / Nx
    x = (ii + a) * dx
    u = [torch.zeros(n, dtype=torch.float32) for _ in range(3)]
    u[axis] = (sign * ub + eps * torch.sin(k * x)).to(torch.float32)
    return synth.Species(q=-1.0, m=1.0, i=[ii.to(torch.int32), jj.to(torch.int32)], d=[a.to(torch.float32), b.to(torch.float32)],
                         u=u, w=torch.full((n,), w, dtype=torch.float32))


def _run_loop(bind, synth, ctx, g, beams, dt, jc, steps, comp, mode):
    """the closed loop of P:127-167 through the C ABI; returns the amplitude of Fourier mode `mode` (along x, mean over y) of field
    component `comp` after every step"""
    eg = P.grid_to_ent(bind, g)
    bind.ent_set_option(ctx, bind.OPT_STEP_IMPL, 0)
    bind.ent_set_option(ctx, bind.OPT_PUSHER, 0)
    bind.ent_set_grid(ctx, eg)
    Nx, Ny = g.N
    F = [torch.zeros(eg.padded_shape, dtype=torch.float32, device="cuda") for _ in range(6)]
    J = bind.zeros_current(eg, "cuda")
    pes = []
    bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 1)
    for sp in beams:
        pe = P.species_to_ent(bind, synth, g, sp, "cuda")
        ps = pe.empty_like()
        bind.ent_sort(ctx, pe, ps, None)
        pes.append(ps)
    bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 0)
    NG = bind.NGHOST
    amp = torch.zeros(steps, dtype=torch.float64, device="cuda")
    for s in range(steps):
        if s > 0 and s % 3 == 0:
            for b in range(2):
                ps = pes[b].empty_like()
                bind.ent_sort(ctx, pes[b], ps, None)
                pes[b] = ps
        bind.ent_faraday(ctx, F, 0.5 * dt)
        bind.ent_fill_field_ghosts(ctx, F)
        bind.ent_zero_current(ctx, J)
        bind.ent_step_pair(ctx, F, pes[0], pes[1], J, dt)
        bind.ent_fold_current(ctx, J)
        bind.ent_faraday(ctx, F, 0.5 * dt)
        bind.ent_ampere(ctx, F, J, dt, jc)
        bind.ent_fill_field_ghosts(ctx, F)
        row = F[comp][NG:NG + Ny, NG:NG + Nx].to(torch.float64).mean(dim=0)
        amp[s] = torch.fft.rfft(row)[mode].abs() * (2.0 / Nx)
    torch.cuda.synchronize()
    assert bind.ent_get_stat(ctx, bind.STAT_LAST_STEP_TILED) == 1
    assert bind.ent_get_stat(ctx, bind.STAT_BAD_MOVES) == 0
    return amp.cpu().numpy()


def _fitted_rate(A, t):
    """slope of log A over the two decades that end one decade below the maximum (the linear phase)"""
    isat = int(np.argmax(A))
    lo = np.where(A[:isat] >= 1e-3 * A[isat])[0][0]
    hi = np.where(A[:isat] >= 1e-1 * A[isat])[0][0]
    assert hi - lo > 50, "no clean linear phase: the seeded mode did not grow over two decades"
    return np.polyfit(t[lo:hi], np.log(A[lo:hi]), 1)[0], isat, lo, hi


def test_two_stream_growth_rate_follows_eq14(env):
    bind, synth, ctx = env
    Nx, Ny, dx, mode = 432, 16, 1.0, 8
    g = synth.GridSpec(D=2, N=(Nx, Ny), bc=(synth.PERIODIC, synth.PERIODIC), kind=synth.CART, xmin=(0.0, 0.0, 0.0),
                       xmax=(Nx * dx, Ny * dx, 1.0))
    wp, ub, jc, side = 0.1, 0.5, 4.0 * math.pi, 4
    gam = math.sqrt(1.0 + ub * ub); vb = ub / gam
    dt = 0.45 * dx
    w = wp * wp * dx * dx / (jc * 2 * side * side)             # w_p^2 = jc n q^2 / m,  n = 2 side^2 w / dx^2 (both beams)
    k = 2.0 * math.pi * mode / (Nx * dx)
    a = wp * wp / (2.0 * gam ** 3); K = (k * vb) ** 2
    Gamma = math.sqrt(math.sqrt(a * a + 4.0 * a * K) - a - K)
    assert abs(Gamma / (wp / (2.0 * gam) ** 1.5) - 1.0) < 0.01  # the seeded mode sits at the maximum of Eq. 14
    beams = [_beam(synth, g, s, ub, 1e-5, k, w, side) for s in (+1.0, -1.0)]
    steps = int(round(75.0 / (wp * dt)))                      # 75 / w_p: the seed (1e-5 u_b) saturates after ~ 60 / w_p
    A = _run_loop(bind, synth, ctx, g, beams, dt, jc, steps, 0, mode)
    t = (np.arange(steps) + 1) * dt
    slope, isat, lo, hi = _fitted_rate(A, t)
    print(f"two-stream: Gamma(Eq. 14) = {Gamma:.5f}, measured {slope:.5f} ({slope / Gamma - 1:+.2%}), saturation |E_x| = {A[isat]:.3e} "
          f"at w_p t = {wp * t[isat]:.1f}, fit window w_p t = {wp * t[lo]:.1f} .. {wp * t[hi]:.1f}")
    assert abs(slope / Gamma - 1.0) < 0.02
    # the field saturates when the beams trap: e E / (m w_p c) of order 0.1 .. 1 (a wrong charge-to-current factor moves it)
    assert 0.02 < A[isat] / wp < 2.0


def test_weibel_filamentation_growth_rate(env):
    """Same beams along +-z, wavevector along x (sect. 5.1.1, second half): the current-filamentation mode (E_z, B_y).  Linearising
    the cold two-beam system for k perpendicular to v_b (momentum gamma^3 m dv_z/dt = q E_z, gamma m dv_x/dt = -q v_z B_y, continuity,
    Faraday, Ampere) gives  w^4 - w^2 (k^2 + w_p^2 / gamma_b^3) - w_p^2 k^2 v_b^2 / gamma_b = 0,  so
    Gamma^2 = ( sqrt(b^2 + 4 w_p^2 k^2 v_b^2 / gamma_b) - b ) / 2,  b = k^2 + w_p^2 / gamma_b^3,  which tends to the paper's
    Gamma_max = v_b w_p / gamma_b^(1/2) for k >> w_p.  Exercises what the two-stream run does not: the out-of-plane current
    (reading G8), the magnetic force of the push, the transverse part of the field solver."""
    bind, synth, ctx = env
    Nx, Ny, dx, mode = 432, 16, 1.0, 10
    g = synth.GridSpec(D=2, N=(Nx, Ny), bc=(synth.PERIODIC, synth.PERIODIC), kind=synth.CART, xmin=(0.0, 0.0, 0.0),
                       xmax=(Nx * dx, Ny * dx, 1.0))
    wp, ub, jc, side = 0.1, 0.5, 4.0 * math.pi, 4
    gam = math.sqrt(1.0 + ub * ub); vb = ub / gam
    dt = 0.45 * dx
    w = wp * wp * dx * dx / (jc * 2 * side * side)
    k = 2.0 * math.pi * mode / (Nx * dx)
    kg = 2.0 / dx * math.sin(0.5 * k * dx)                     # the wavenumber the Yee curl sees
    b = kg * kg + wp * wp / gam ** 3
    Gamma = math.sqrt(0.5 * (math.sqrt(b * b + 4.0 * wp * wp * kg * kg * vb * vb / gam) - b))
    assert 0.8 < Gamma / (vb * wp / math.sqrt(gam)) < 1.0       # below the asymptotic maximum of P:849, as it must be at c k = 1.45 w_p
    beams = [_beam(synth, g, s, ub, 1e-5, k, w, side, axis=2) for s in (+1.0, -1.0)]
    steps = int(round(75.0 / (wp * dt)))
    A = _run_loop(bind, synth, ctx, g, beams, dt, jc, steps, 4, mode)        # B_y
    t = (np.arange(steps) + 1) * dt
    slope, isat, lo, hi = _fitted_rate(A, t)
    print(f"Weibel: Gamma(linear theory) = {Gamma:.5f}, measured {slope:.5f} ({slope / Gamma - 1:+.2%}), saturation |B_y| = {A[isat]:.3e} "
          f"at w_p t = {wp * t[isat]:.1f}, fit window w_p t = {wp * t[lo]:.1f} .. {wp * t[hi]:.1f}")
    assert abs(slope / Gamma - 1.0) < 0.02
