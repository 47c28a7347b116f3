"""GPU parity of ent_filter_current (step 9: Eqs. 9-11 + J = conformal J / sqrt(h)) against orc_filter_current, element by
element on every lattice point, periodic / absorbing / axis rules, even and odd pass counts; ghost layers must stay untouched."""
import numpy as np
import pytest
import torch

import parity as P

pytestmark = pytest.mark.gpu

TOL = 2e-6          # fp32 (27-term convolution + one division) against fp64, relative to max |J|


@pytest.fixture(scope="module")
def env(orc):
    from paper_2511_17710_b200 import binding as bind, synth
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: there is no CPU fallback for the product path")
    ctx = bind.ent_create(0, None)
    yield bind, synth, ctx, orc
    bind.ent_destroy(ctx)


def _grids(synth):
    c = lambda D, N, bc: synth.GridSpec(D=D, N=N, bc=bc, kind=synth.CART, xmin=(0.0,) * 3, xmax=tuple(0.5 * n for n in N) + (1.0,) * (3 - D))
    a = lambda kind, N, rmax, vt: synth.GridSpec(D=2, N=N, bc=(synth.ABSORB, synth.AXIS), kind=kind, xmin=(1.0, 0.0, 0.0),
                                                  xmax=(rmax, np.pi, 1.0), r0=0.0, vartheta=vt)
    return {"cart3-periodic": c(3, (40, 24, 20), (0, 0, 0)), "cart2-periodic": c(2, (70, 36), (0, 0)),
            "cart3-absorb": c(3, (20, 16, 12), (1, 0, 1)), "sph": a(synth.SPH, (48, 40), 9.0, 0.0),
            "qsph": a(synth.QSPH, (64, 56), 30.0, 0.4)}


@pytest.mark.parametrize("name", ["cart3-periodic", "cart2-periodic", "cart3-absorb", "sph", "qsph"])
@pytest.mark.parametrize("npasses,divide", [(1, False), (2, True), (5, True), (0, True)])
def test_filter_matches_oracle(env, name, npasses, divide):
    bind, synth, ctx, orc = env
    g = _grids(synth)[name]
    eg, og = P.grid_to_ent(bind, g), P.grid_to_orc(orc, g)
    bind.ent_set_grid(ctx, eg)
    gen = torch.Generator().manual_seed(77)
    J32 = [torch.randn(g.padded_shape, generator=gen, dtype=torch.float32) for _ in range(3)]
    Jg = [j.cuda() for j in J32]
    Jo = [j.numpy().astype(np.float64) for j in J32]
    before = [j.copy() for j in Jo]
    bind.ent_filter_current(ctx, Jg, npasses, divide)
    torch.cuda.synchronize()
    orc.filter_current(og, Jo, npasses, divide)
    scale = max(np.abs(j).max() for j in Jo)
    worst = 0.0
    for c in range(3):
        got = Jg[c].cpu().numpy().astype(np.float64)
        worst = max(worst, np.abs(got - Jo[c]).max() / scale)
        # ghost layers are not written (include/ent.h): the outermost layer of the padded array keeps its input bits
        edge = np.ones(got.shape, dtype=bool)
        edge[tuple([slice(1, -1)] * got.ndim)] = False
        assert np.array_equal(got[edge], before[c][edge])
    print(name, npasses, divide, "max|dJ|/max|J| =", worst)
    assert worst <= TOL


def test_filter_error_paths(env):
    bind, synth, ctx, orc = env
    g = _grids(synth)["cart2-periodic"]
    eg = P.grid_to_ent(bind, g)
    bind.ent_set_grid(ctx, eg)
    J = bind.zeros_current(eg, "cuda")
    with pytest.raises(bind.EntError):
        bind.ent_filter_current(ctx, J, -1, False)
    bind.ent_filter_current(ctx, J, 0, False)              # nothing to do
    assert all(float(j.abs().max()) == 0.0 for j in J)
