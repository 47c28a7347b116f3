"""The input generators (paper_2511_17710_b200/synth.py) restate two pieces of the paper's geometry to lay out their inputs:
the spherical / quasi-spherical metric, used for fields, weights w = sqrt(h)/V0 and dt, and Eq. 8.
They must agree with the oracle's O1 functions, which are pinned against finite differences of the forward maps."""
import numpy as np
import pytest
import torch

from paper_2511_17710_b200 import synth


def _grids(orc):
    mk = lambda kind, N, rmin, rmax, r0, vt: (
        synth.GridSpec(D=2, N=N, bc=(synth.ABSORB, synth.AXIS), kind=kind, xmin=(rmin, 0.0, 0.0), xmax=(rmax, np.pi, 1.0), r0=r0, vartheta=vt),
        orc.Grid(D=2, N=N, bc=(orc.ABSORB, orc.AXIS), kind=kind, xmin=(rmin, 0.0), xmax=(rmax, np.pi), r0=r0, vartheta=vt))
    return [mk(synth.SPH, (48, 40), 1.0, 9.0, 0.0, 0.0), mk(synth.QSPH, (64, 64), 1.0, 20.0, 0.0, 0.0),
            mk(synth.QSPH, (40, 56), 1.0, 50.0, 0.0, 0.4), mk(synth.QSPH, (32, 32), 1.5, 12.0, 1.0, 0.7)]


def test_sph_geometry_equals_the_oracle_metric(orc):
    rng = np.random.default_rng(5)
    for sg, og in _grids(orc):
        x1 = rng.uniform(0, sg.N[0], 500); x2 = rng.uniform(0, sg.N[1], 500)
        r, th, h1, h2, h3 = synth.sph_geometry(sg, torch.from_numpy(x1), torch.from_numpy(x2))
        h = orc.metric_h_many(og, x1, x2)
        assert np.allclose(h1.numpy() ** 2, h[:, 0], rtol=1e-13)
        assert np.allclose(h2.numpy() ** 2, h[:, 1], rtol=1e-13)
        assert np.allclose(h3.numpy() ** 2, h[:, 2], rtol=1e-12, atol=1e-300)
        # (r, theta) against the oracle's forward map at phi = 0: X = r sin(theta), Z = r cos(theta)
        for k in range(0, 500, 50):
            X = orc.code_to_cart(og, [x1[k], x2[k], 0.0])
            assert X[0] == pytest.approx(float(r[k] * torch.sin(th[k])), rel=1e-13)
            assert X[2] == pytest.approx(float(r[k] * torch.cos(th[k])), rel=1e-13, abs=1e-13)


def test_cfl_dx_min_equals_eq8_of_the_oracle(orc):
    for sg, og in _grids(orc):
        assert synth.cfl_dx_min(sg) == pytest.approx(orc.dx_min(og), rel=1e-13)
    sg = synth.GridSpec(D=3, N=(8, 6, 4), bc=(0, 0, 0), kind=synth.CART, xmin=(0.0, 0.0, 0.0), xmax=(4.0, 6.0, 1.0))
    og = orc.Grid(D=3, N=(8, 6, 4), bc=(0, 0, 0), kind=orc.CART, xmin=(0.0, 0.0, 0.0), xmax=(4.0, 6.0, 1.0))
    assert synth.cfl_dx_min(sg) == pytest.approx(orc.dx_min(og), rel=1e-14)
