"""ent_step_host / ent_step_host_pair (host buffers in, host buffers out: the calls behind the `e2e` figure of bench.py) against the
oracle.  The calls return the blocks permuted (tile-sorted); the weights are made unique per particle so that the original order
can be restored, then positions, momenta and the summed current meet the same bars as the device-buffer calls."""
import numpy as np
import pytest
import torch

import parity as P

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name", ["C3/8", "C1", "C2/4"])
@pytest.mark.parametrize("pair", [False, True])
def test_host_calls_match_oracle(orc, name, pair):
    from paper_2511_17710_b200 import binding as bind, synth
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: there is no CPU fallback for the product path")
    base, _, shrink = name.partition("/")
    wl = synth.CONFIGS[base](int(shrink) if shrink else 1)
    g = wl.grid
    eg, og = P.grid_to_ent(bind, g), P.grid_to_orc(orc, g)
    ctx = bind.ent_create(0, None)
    try:
        bind.ent_set_grid(ctx, eg)
        for sp in wl.species:                                   # unique weights = particle labels (exact in fp32)
            lab = (1.0 + torch.arange(sp.n, dtype=torch.float64) * 2.0 ** -20).to(torch.float32)
            sp.w = (lab if eg.axisym else sp.w * lab).contiguous()      # (the sqrt(h) weights of the axisymmetric recipes would collide)
            assert torch.unique(sp.w).numel() == sp.n
        hF = [f.contiguous().pin_memory() for f in wl.fields]
        hJ = [torch.zeros(eg.padded_shape, dtype=torch.float32).pin_memory() for _ in range(3)]
        hps = [P.species_to_ent(bind, synth, g, sp, "cpu").to("cpu", pin=True) for sp in wl.species]
        pos = [P.species_to_orc(orc, sp) for sp in wl.species]
        Jo = orc.zeros_current(og)
        for sp, po in zip(wl.species, pos):
            orc.step(og, P.fields_to_orc(wl.fields), po, Jo, sp.q, sp.m, wl.dt)
        if pair:
            up, down = bind.ent_step_host_pair(ctx, hF, hps[0], hps[1], hJ, wl.dt, 1)
            Jg = [j.clone() for j in hJ]
        else:
            Jg = [torch.zeros_like(j) for j in hJ]
            up = down = 0
            for hp in hps:
                u_, d_ = bind.ent_step_host(ctx, hF, hp, hJ, wl.dt, 1)
                up += u_; down += d_
                for a, b in zip(Jg, hJ):
                    a += b                                       # every call returns the current of its own species
        assert up > 0 and down > 0
        for sp, hp, po in zip(wl.species, hps, pos):
            order = torch.argsort(hp.w)                          # back to the original order (weights increase with the index)
            assert torch.equal(hp.w[order], sp.w)
            back = bind.Particles(cell=hp.cell[order], d=[t[order] for t in hp.d], u=[t[order] for t in hp.u], w=hp.w[order],
                                  phi=None if hp.phi is None else hp.phi[order], tag=None if hp.tag is None else hp.tag[order], q=hp.q, m=hp.m)
            st = P.compare_particles(g, back, po, steps=1, orc_metric=(orc, og))
            print(name, "pair" if pair else "single", st)
        Jdev = [j.cuda() for j in Jg]
        bind.ent_fold_current(ctx, Jdev)
        torch.cuda.synchronize()
        orc.fold_current(og, Jo)
        if not eg.axisym:
            print(name, "J:", P.compare_current(Jdev, Jo))
    finally:
        bind.ent_destroy(ctx)
