"""Parity at BASELINE.json's FULL size, in the launch configuration bench.py times (C3: 256^3, 67,108,864 particles per
species; C4: 512^3, 268,435,456 per species; block sorted, tiled kernel, incremental re-sort every 3 steps).  The oracle cannot follow 67 M particles for many
steps in seconds, so the last step is checked
  * on a seeded SAMPLE of particles, advanced one by one by the oracle from the GPU's own state before the step
    (positions, cell indices, momenta: the bars of tests/parity.py),
  * on the CURRENT in two sub-boxes (one interior, one wrapped around the periodic corner): the oracle deposits every
    particle that can reach the box and the nodes of the box are compared element by element,
  * through the property that holds at any size: discrete charge continuity (Eq. 6) of the GPU's own output over the WHOLE
    grid, with the oracle's checker.
"""
import numpy as np
import pytest
import torch

import parity as P

pytestmark = pytest.mark.gpu

NSAMPLE = 200_000
BOX = 16


def _subset(bind, p, idx):
    s = lambda t: None if t is None else t[idx].contiguous()
    return bind.Particles(cell=s(p.cell), d=[s(t) for t in p.d], u=[s(t) for t in p.u], w=s(p.w), phi=s(p.phi), tag=s(p.tag), q=p.q, m=p.m)


def _in_box_periodic(i, lo, width, N):
    """mask of cells with (i - lo) mod N < width, per dimension (all dimensions periodic)"""
    m = None
    for a in range(len(i)):
        r = torch.remainder(i[a].to(torch.int64) - lo[a], N[a]) < width
        m = r if m is None else (m & r)
    return m


@pytest.mark.parametrize("name", ["C3", "C4"])
def test_full_size_last_step(orc, name):
    from paper_2511_17710_b200 import binding as bind, synth
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    if torch.cuda.mem_get_info()[1] < 100e9:
        pytest.skip("needs a GPU with > 100 GB for the full-size workloads")
    wl = synth.CONFIGS[name](1, device="cuda")
    g = wl.grid
    sp = wl.species[0]                                      # the electrons; the positrons run the same kernel
    wl.species = None
    eg, og = P.grid_to_ent(bind, g), P.grid_to_orc(orc, g)
    ctx = bind.ent_create(0, None)
    try:
        bind.ent_set_grid(ctx, eg)
        F = wl.fields
        pe = bind.Particles(cell=synth.pack_cell(g, sp.i), d=sp.d, u=sp.u, w=sp.w, q=sp.q, m=sp.m)
        del sp
        spare = pe.empty_like()
        bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 1)
        bind.ent_sort(ctx, pe, spare, None)                 # full sort, as bench.py does before its warm-up
        bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 0)
        pe, spare = spare, pe
        J = bind.zeros_current(eg, "cuda")
        for s in range(5):                                  # steps 0-2, re-bin, steps 3-4; step 4 is checked
            if s == 3:
                bind.ent_sort(ctx, pe, spare, None)
                assert bind.ent_get_stat(ctx, bind.STAT_LAST_SORT_REBIN) == 1
                pe, spare = spare, pe
            if s == 4:
                before = pe.clone()
            bind.ent_zero_current(ctx, J)
            bind.ent_step(ctx, F, pe, J, wl.dt)
            assert bind.ent_get_stat(ctx, bind.STAT_LAST_STEP_TILED) == 1
        bind.ent_fold_current(ctx, J)
        torch.cuda.synchronize()
        assert bind.ent_get_stat(ctx, bind.STAT_STRAYS) == 0 and bind.ent_get_stat(ctx, bind.STAT_BAD_MOVES) == 0
        del spare
        F_orc = P.fields_to_orc(F)

        # ---- (1) sampled particles, one step of the oracle from the GPU's state before the step
        gen = torch.Generator(device="cuda"); gen.manual_seed(1234)
        idx = torch.randint(0, pe.n, (NSAMPLE,), device="cuda", generator=gen)
        pb = P.ent_to_orc(orc, g, _subset(bind, before, idx))
        po = orc.gather_push(og, F_orc, pb, before.q / before.m, wl.dt)
        stats = P.compare_particles(g, _subset(bind, pe, idx), po, steps=1, orc_metric=(orc, og))
        print("sample:", stats)

        # ---- (2) current in two sub-boxes: every particle that can reach a node of the box goes through the oracle
        Jscale = max(float(j.abs().max()) for j in J)
        ib = synth.unpack_cell(g, before.cell)
        N = [int(n) for n in g.N]
        for lo in ((40, 100, 200), (N[0] - 8, N[1] - 8, N[2] - 8)):       # interior; wrapped around the periodic corner
            m = _in_box_periodic(ib, [l - 2 for l in lo], BOX + 4, N)
            sel = torch.nonzero(m).squeeze(1)
            pbox = P.ent_to_orc(orc, g, _subset(bind, before, sel))
            Jo = orc.zeros_current(og)
            orc.step(og, F_orc, pbox, Jo, before.q, before.m, wl.dt)
            orc.fold_current(og, Jo)
            worst = 0.0
            ax = [np.array([(lo[a] + k) % N[a] for k in range(BOX)]) + 2 for a in range(3)]       # padded indices of the box nodes
            for c in range(3):
                jg = J[c].cpu().numpy().astype(np.float64)[np.ix_(ax[2], ax[1], ax[0])]
                jo = Jo[c][np.ix_(ax[2], ax[1], ax[0])]
                worst = max(worst, float(np.abs(jg - jo).max()))
            print(f"box at {lo}: {sel.numel()} particles, max|dJ|/max|J| = {worst / Jscale:.3e}")
            assert worst <= P.J_TOL * Jscale
        del ib, Jo

        # ---- (3) continuity of the GPU's own step over the whole grid (Eq. 6), oracle's checker
        c = P.continuity_of_gpu_step(orc, og, P.ent_to_orc(orc, g, before), P.ent_to_orc(orc, g, pe), J, before.q, wl.dt)
        print(f"continuity residual (whole grid): {c:.3e}")
        assert c <= P.CONT_TOL
    finally:
        bind.ent_destroy(ctx)


@pytest.mark.parametrize("name", ["C3", "C4"])
def test_full_size_pair_launch_last_step(orc, name):
    """The launch configuration bench.py times by default: BOTH species through ent_step_pair (one launch of the tiled kernel),
    blocks sorted, re-binned every 3 steps.  Sampled particles of each species, the summed current of the two species in two
    sub-boxes against the oracle, whole-grid continuity of the summed charge."""
    from paper_2511_17710_b200 import binding as bind, synth
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    if torch.cuda.mem_get_info()[1] < 100e9:
        pytest.skip("needs a GPU with > 100 GB for the full-size workloads")
    wl = synth.CONFIGS[name](1, device="cuda")
    g = wl.grid
    eg, og = P.grid_to_ent(bind, g), P.grid_to_orc(orc, g)
    ctx = bind.ent_create(0, None)
    try:
        bind.ent_set_grid(ctx, eg)
        F = wl.fields
        pes = [bind.Particles(cell=synth.pack_cell(g, sp.i), d=sp.d, u=sp.u, w=sp.w, q=sp.q, m=sp.m) for sp in wl.species]
        wl.species = None
        spares = [pe.empty_like() for pe in pes]
        bind.ent_reserve(ctx, max(pe.n for pe in pes))
        bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 1)
        for k in range(2):
            bind.ent_sort(ctx, pes[k], spares[k], None)
            pes[k], spares[k] = spares[k], pes[k]
        bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 0)
        J = bind.zeros_current(eg, "cuda")
        befores = None
        for s in range(5):                                  # steps 0-2, re-bin, steps 3-4; step 4 is checked
            if s == 3:
                for k in range(2):
                    bind.ent_sort(ctx, pes[k], spares[k], None)
                    assert bind.ent_get_stat(ctx, bind.STAT_LAST_SORT_REBIN) == 1
                    pes[k], spares[k] = spares[k], pes[k]
            if s == 4:
                del spares
                befores = [pe.clone() for pe in pes]
            bind.ent_zero_current(ctx, J)
            bind.ent_step_pair(ctx, F, pes[0], pes[1], J, wl.dt)
            assert bind.ent_get_stat(ctx, bind.STAT_LAST_STEP_TILED) == 1
        bind.ent_fold_current(ctx, J)
        torch.cuda.synchronize()
        assert bind.ent_get_stat(ctx, bind.STAT_STRAYS) == 0 and bind.ent_get_stat(ctx, bind.STAT_BAD_MOVES) == 0
        F_orc = P.fields_to_orc(F)
        gen = torch.Generator(device="cuda"); gen.manual_seed(4321)
        for k in range(2):
            idx = torch.randint(0, pes[k].n, (NSAMPLE // 2,), device="cuda", generator=gen)
            pb = P.ent_to_orc(orc, g, _subset(bind, befores[k], idx))
            po = orc.gather_push(og, F_orc, pb, befores[k].q / befores[k].m, wl.dt)
            print(f"species {k} sample:", P.compare_particles(g, _subset(bind, pes[k], idx), po, steps=1, orc_metric=(orc, og)))
        Jscale = max(float(j.abs().max()) for j in J)
        N = [int(n) for n in g.N]
        for lo in ((40, 100, 200), (N[0] - 8, N[1] - 8, N[2] - 8)):
            Jo = orc.zeros_current(og)
            npart = 0
            for k in range(2):
                ib = synth.unpack_cell(g, befores[k].cell)
                sel = torch.nonzero(_in_box_periodic(ib, [l - 2 for l in lo], BOX + 4, N)).squeeze(1)
                del ib
                npart += sel.numel()
                orc.step(og, F_orc, P.ent_to_orc(orc, g, _subset(bind, befores[k], sel)), Jo, befores[k].q, befores[k].m, wl.dt)
            orc.fold_current(og, Jo)
            ax = [np.array([(lo[a] + k) % N[a] for k in range(BOX)]) + 2 for a in range(3)]
            worst = max(float(np.abs(J[c].cpu().numpy().astype(np.float64)[np.ix_(ax[2], ax[1], ax[0])] - Jo[c][np.ix_(ax[2], ax[1], ax[0])]).max())
                        for c in range(3))
            print(f"box at {lo}: {npart} particles of both species, max|dJ|/max|J| = {worst / Jscale:.3e}")
            assert worst <= P.J_TOL * Jscale
        del Jo
        if name == "C3":                                      # host memory: the checker holds every particle of both species in fp64
            c = P.continuity_of_gpu_steps(orc, og, [P.ent_to_orc(orc, g, b) for b in befores], [P.ent_to_orc(orc, g, pe) for pe in pes], J,
                                          [b.q for b in befores], wl.dt)
            print(f"continuity residual (whole grid, both species): {c:.3e}")
            assert c <= P.CONT_TOL
    finally:
        bind.ent_destroy(ctx)


def test_c5_full_size_last_step(orc):
    """C5 at full size (quasi-spherical 2048^2, ~134 M particles per species, tiled axisymmetric kernel, heavy tiles split over
    several CTAs): sampled particles against the oracle, the current of an inner (dense) box, whole-grid continuity."""
    from paper_2511_17710_b200 import binding as bind, synth
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    if torch.cuda.mem_get_info()[1] < 100e9:
        pytest.skip("needs a GPU with > 100 GB for the full-size workloads")
    wl = synth.config5(1, device="cuda")
    g = wl.grid
    sp = wl.species[0]
    wl.species = None
    eg, og = P.grid_to_ent(bind, g), P.grid_to_orc(orc, g)
    ctx = bind.ent_create(0, None)
    try:
        bind.ent_set_grid(ctx, eg)
        F = wl.fields
        pe = bind.Particles(cell=synth.pack_cell(g, sp.i), d=sp.d, u=sp.u, w=sp.w, phi=sp.phi,
                            tag=torch.ones(sp.n, dtype=torch.uint8, device="cuda"), q=sp.q, m=sp.m)
        del sp
        spare = pe.empty_like()
        bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 1)
        bind.ent_sort(ctx, pe, spare, None)
        bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 0)
        pe, spare = spare, pe
        J = bind.zeros_current(eg, "cuda")
        for s in range(5):
            if s == 3:
                bind.ent_sort(ctx, pe, spare, None)
                assert bind.ent_get_stat(ctx, bind.STAT_LAST_SORT_REBIN) == 1
                pe, spare = spare, pe
            if s == 4:
                before = pe.clone()
            bind.ent_zero_current(ctx, J)
            bind.ent_step(ctx, F, pe, J, wl.dt)
            assert bind.ent_get_stat(ctx, bind.STAT_LAST_STEP_TILED) == 1
        bind.ent_fold_current(ctx, J)
        torch.cuda.synchronize()
        assert bind.ent_get_stat(ctx, bind.STAT_BAD_MOVES) == 0
        del spare
        F_orc = P.fields_to_orc(F)

        gen = torch.Generator(device="cuda"); gen.manual_seed(4321)
        idx = torch.randint(0, pe.n, (NSAMPLE,), device="cuda", generator=gen)
        pb = P.ent_to_orc(orc, g, _subset(bind, before, idx))
        po = orc.gather_push(og, F_orc, pb, before.q / before.m, wl.dt)
        stats = P.compare_particles(g, _subset(bind, pe, idx), po, steps=1, orc_metric=(orc, og))
        print("sample:", stats)

        Jscale = max(float(j.abs().max()) for j in J)
        ib = synth.unpack_cell(g, before.cell)
        lo = (8, 1000)                                       # dense inner radii, near the equator
        m = (ib[0] >= lo[0] - 2) & (ib[0] < lo[0] + BOX + 2) & (ib[1] >= lo[1] - 2) & (ib[1] < lo[1] + BOX + 2)
        sel = torch.nonzero(m).squeeze(1)
        pbox = P.ent_to_orc(orc, g, _subset(bind, before, sel))
        bound = P.offset_format_bound(orc, g, og, pbox, before.q, wl.dt)
        Jo = orc.zeros_current(og)
        orc.step(og, F_orc, pbox, Jo, before.q, before.m, wl.dt)
        orc.fold_current(og, Jo)
        worst = 0.0
        ax = [np.arange(lo[a], lo[a] + BOX) + 2 for a in range(2)]
        for c in range(3):
            e = np.abs(J[c].cpu().numpy().astype(np.float64)[np.ix_(ax[1], ax[0])] - Jo[c][np.ix_(ax[1], ax[0])])
            e = (e - bound[c][np.ix_(ax[1], ax[0])]).clip(min=0.0)
            worst = max(worst, float(e.max()))
        print(f"box at {lo}: {sel.numel()} particles, max|dJ|/max|J| = {worst / Jscale:.3e}")
        assert worst <= P.J_TOL * Jscale
        del ib, Jo

        c = P.continuity_of_gpu_step(orc, og, P.ent_to_orc(orc, g, before), P.ent_to_orc(orc, g, pe), J, before.q, wl.dt)
        print(f"continuity residual (whole grid): {c:.3e}")
        assert c <= P.CONT_TOL
    finally:
        bind.ent_destroy(ctx)


def test_c2_full_size_every_step(orc):
    """C2 at BASELINE.json's size (log-spherical 256 x 256, ~1 M particles per species, 20 steps): the oracle follows EVERY particle
    for all 20 steps; sorted block, tiled axisymmetric kernel, incremental re-sort every 3 steps; every step checks the current (end
    to end with the format allowance, raw value printed; strict deposit check without allowance) and continuity."""
    from paper_2511_17710_b200 import binding as bind, synth
    import test_gpu_parity as T
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    ctx = bind.ent_create(0, None)
    try:
        wl = synth.config2(1)
        assert tuple(wl.grid.N) == (256, 256) and wl.steps == 20
        stats = T._run_case((bind, synth, ctx, orc), wl, impl=0, sort_first=True, resort_every=3)
        print("C2 full size:", stats)
        assert all(st["tiled"] == 1 and st["strays"] == 0 for st in stats.values())
    finally:
        bind.ent_destroy(ctx)
